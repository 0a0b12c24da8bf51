// vn_log64.cuh -- -(1/2) ln(r2) and 1/r2 in double for the fp64 pair kernels (vn_farfield_f64.cu, vn_fmm.cu).
// There is no SFU logarithm or reciprocal in double on sm_100; this is the cheapest form found.
#pragma once

#include "vn_common.cuh"

namespace vn {

constexpr int kLogTab = 1024;                 // (1/2) ln of the 10-bit mantissas 1 + k/1024
constexpr int kExpTab = 2048;                 // (1/2) ln2 (E - 1023) for every exponent field

// -(1/2) ln(r2) and 1/r2 in double: 9 DP instructions + one MUFU.RCP64H + two 8-byte shared-memory loads,
// no exponent/mantissa surgery on r2 and no integer-to-double conversion (I2F.F64 occupies the FP64 pipe).
//   t0  = hardware reciprocal seed of r2 (2^-20 accurate, full exponent range)
//   1/r2 = t0 (1 + d + d^2), d = 1 - r2 t0                                     (one cubic step, 3 DP)
//   rc  = t0 truncated to 10 mantissa bits = 2^(E-1023) (1 + k/1024);  eps = r2 rc - 1 (one fma; 0 <= eps < 2^-10)
//   -(1/2) ln r2 = (1/2) ln rc - (1/2) log1p(eps),  log1p by its series through eps^4 (next term <= 1.8e-16), Horner
//   (1/2) ln rc = tabE[E] + tab[k]:  tab[k] = (1/2) ln(1 + k/1024), tabE[E] = (1/2) ln2 (E - 1023) for every
//   exponent field E = 0 .. 2047; both built by every block at start-up (24 KB of shared memory).
// r2 must be a positive normal double whose reciprocal is normal too (the header's precondition).
__device__ __forceinline__ void log_rcp_f64(double r2, const double *__restrict__ tab, double &mhalf_log, double &inv)
{
    double t0;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(t0) : "d"(r2));                // MUFU.RCP64H
    const int rch = __double2hiint(t0) & 0xfffffc00;                        // truncate to 10 mantissa bits
    const double rc = __hiloint2double(rch, 0);
    const int k = (rch >> 10) & 0x3ff;
    const double base = tab[kLogTab + (rch >> 20)] + tab[k];
    // reciprocal
    const double d = fma(-r2, t0, 1.0);
    const double p = fma(d, d, d);
    inv = fma(t0, p, t0);
    // logarithm
    const double eps = fma(r2, rc, -1.0);
    double q = 0.125;                                  // -(1/2) (1 - eps/2 + eps^2/3 - eps^3/4)
    q = fma(q, eps, -1.0 / 6.0);
    q = fma(q, eps, 0.25);
    q = fma(q, eps, -0.5);
    mhalf_log = fma(eps, q, base);
}

// the two tables of log_rcp_f64, consecutive in memory (shared, or the scratch copy the pair kernel loads from):
// tab[0 .. kLogTab) and tabE[0 .. kExpTab)
__device__ __forceinline__ void build_log_tables(double *tab, int tid, int nthreads)
{
    for (int k = tid; k < kLogTab; k += nthreads) tab[k] = 0.5 * log1p((double)k * (1.0 / 1024.0));
    for (int i = tid; i < kExpTab; i += nthreads) tab[kLogTab + i] = 0.34657359027997265471 * (double)(i - 1023);
}

}  // namespace vn

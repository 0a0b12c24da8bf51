// vn_log64.cuh -- -(1/2) ln(r2) and 1/r2 in double for the fp64 pair kernels (vn_farfield_f64.cu, vn_fmm.cu).
// There is no SFU logarithm or reciprocal in double on sm_100; this is the cheapest form found.
#pragma once

#include "vn_common.cuh"

namespace vn {

#ifndef VN_LOG_BITS
#define VN_LOG_BITS 11                        // mantissa bits of the table index
#endif
constexpr int kLogBits = VN_LOG_BITS;
constexpr int kLogTab = 1 << kLogBits;        // (1/2) ln of the mantissas 1 + k/2^kLogBits
constexpr int kExpTab = 2048;                 // (1/2) ln2 (E - 1023) for every exponent field
constexpr int kLogMask = ~((1 << (20 - kLogBits)) - 1);   // keeps kLogBits mantissa bits of a double's high word

// -(1/2) ln(r2) and 1/r2 in double: 8 DP instructions + one MUFU.RCP64H + two 8-byte shared-memory loads + five
// integer instructions, no exponent/mantissa surgery on r2 and no integer-to-double conversion (I2F.F64 occupies
// the FP64 pipe).
//   t0  = hardware reciprocal seed of r2 (2^-20 accurate, full exponent range)
//   1/r2 = t0 (1 + d + d^2), d = 1 - r2 t0                                     (one cubic step, 3 DP)
//   rc  = t0 truncated to kLogBits mantissa bits = 2^(E-1023) (1 + k/2^kLogBits);  eps = r2 rc - 1 (one fma;
//         0 <= eps < 2^-kLogBits (1 + 2^-19))
//   -(1/2) ln r2 = (1/2) ln rc - (1/2) log1p(eps),  log1p by its series through eps^3 (11-bit table: the next
//   term, eps^4/8 <= 2^-47 = 7e-15 absolute on a value of order one -- the tolerance of the path is 1e-12 relative
//   and the measured parity 3e-15 ... 6e-15) or through eps^4 (10-bit table), Horner.  The coefficient 1/6 is
//   rounded to its high word (relative 1.5e-8 on a term below 2^-34): a double whose low word is zero is an
//   immediate operand of DFMA, anything else costs two moves per use.
//   (1/2) ln rc = tabE[E] + tab[k]:  tab[k] = (1/2) ln(1 + k/2^kLogBits), tabE[E] = (1/2) ln2 (E - 1023) for every
//   exponent field E = 0 .. 2047 (16 KB + 16 KB of shared memory).
// r2 must be a positive normal double whose reciprocal is normal too (the header's precondition).
// (MUFU.RCP64H writes a high word only, so t0 and rc each cost one move that zeroes their low word; keeping
// dedicated register pairs with persistent zero low words was tried -- ptxas copies the zero into a fresh pair
// anyway.)
__device__ __forceinline__ void log_rcp_f64(double r2, const double *__restrict__ tab, double &mhalf_log, double &inv)
{
    double t0;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(t0) : "d"(r2));                // MUFU.RCP64H
    const int rch = __double2hiint(t0) & kLogMask;                          // truncate to kLogBits mantissa bits
    const double rc = __hiloint2double(rch, 0);
    const double base = *reinterpret_cast<const double *>(reinterpret_cast<const char *>(tab) + (kLogTab * 8) +
                                                          ((rch >> 17) & 0x3ff8)) +
                        *reinterpret_cast<const double *>(reinterpret_cast<const char *>(tab) +
                                                          ((rch >> (17 - kLogBits)) & ((kLogTab - 1) * 8)));
    // reciprocal
    const double d = fma(-r2, t0, 1.0);
    const double p = fma(d, d, d);
    inv = fma(t0, p, t0);
    // logarithm
    const double eps = fma(r2, rc, -1.0);
#if VN_LOG_BITS >= 11
    double q = fma(eps, __hiloint2double(0xbfc55555, 0), 0.25);        // -(1/2) (1 - eps/2 + eps^2/3)
#else
    double q = fma(eps, 0.125, __hiloint2double(0xbfc55555, 0));       // -(1/2) (1 - eps/2 + eps^2/3 - eps^3/4)
    q = fma(q, eps, 0.25);
#endif
    q = fma(q, eps, -0.5);
    mhalf_log = fma(eps, q, base);
}

// the two tables of log_rcp_f64, consecutive in memory (shared, or the scratch copy the kernels load from):
// tab[0 .. kLogTab) and tabE[0 .. kExpTab)
__device__ __forceinline__ void build_log_tables(double *tab, int tid, int nthreads)
{
    for (int k = tid; k < kLogTab; k += nthreads) tab[k] = 0.5 * log1p((double)k * (1.0 / (double)kLogTab));
    for (int i = tid; i < kExpTab; i += nthreads) tab[kLogTab + i] = 0.34657359027997265471 * (double)(i - 1023);
}

}  // namespace vn

// vn_farfield_small.cu -- vn_farfield for suspensions of at most kSmallPoints points: ONE launch, no scratch.
//
//   U_i = 1/(4 pi mu) sum_{j not in ves(i)} [ -log|r| g_j + (r.g_j)/|r|^2 r ],  r = x_i - y_j, g_j = f_j w_j
//   (PAPER.md:129-136 eqs 2.8/2.9, :173 trapezoid rule)
//
// The general path (vn_farfield_f32.cu / vn_farfield_f64.cu) spends a stream-ordered allocation, a memset and three
// launches around its pair kernel; at BASELINE.json configs[0] (16 x 32 = 512 points, 0.25 M interactions) those
// cost more than the sum itself (0.14 ms per step for a 0.06 ms kernel in round 1).  Below kSmallPoints the whole
// call is this kernel: a block owns kSmallTargets targets, the kSmallSplit threads of a warp share one target (each takes every
// kSmallSplit-th source of a staged chunk; g = F*W is formed while staging), own-vesicle sources are skipped by
// index, the partial sums meet in a fixed-order shuffle reduction, scaled and stored.  One-directional (the symmetric
// evaluation needs cross-block accumulators, i.e. the scratch this path exists to avoid), no atomics, bitwise
// reproducible.  fp32: SFU lg2 / rcp as in the general fp32 kernel, per-chunk partial sums folded into running sums.
// fp64: libdevice log and division (the table-driven log of the general kernel would cost a 32 KB table per block).
#include "vn_common.cuh"

namespace vn {

constexpr int kSmallThreads = 128;
constexpr int kSmallSplit = 32;                             // threads per target: a warp (at most 1,024 points: the kernel
                                                            // is latency-bound, so parallelism counts, not instruction count;
                                                            // measured at 16 x 32 points in double: 4 threads per target 42 us)
constexpr int kSmallTargets = kSmallThreads / kSmallSplit;  // targets per block: 4

template <typename real, typename real2>
__global__ void __launch_bounds__(kSmallThreads)
farfield_small_kernel(const real2 *__restrict__ X, const real2 *__restrict__ F, const real *__restrict__ W, int P,
                      int npts, double prefactor, real2 *__restrict__ U)
{
    __shared__ real sx[kSmallThreads], sy[kSmallThreads], gx[kSmallThreads], gy[kSmallThreads];
    const int tid = threadIdx.x, slot = tid / kSmallSplit, part = tid % kSmallSplit;
    const int i = blockIdx.x * kSmallTargets + slot;
    const bool live = i < P;
    const real2 xi = X[live ? i : P - 1];
    const int own = ((live ? i : P - 1) / npts) * npts;     // first point of the target's own vesicle
    real ux = 0, uy = 0;
    for (int s0 = 0; s0 < P; s0 += kSmallThreads) {
        __syncthreads();
        if (s0 + tid < P) {
            const real2 y = X[s0 + tid], f = F[s0 + tid];
            const real w = W[s0 + tid];
            sx[tid] = y.x;
            sy[tid] = y.y;
            gx[tid] = f.x * w;                              // product in the storage precision, as in the general path
            gy[tid] = f.y * w;
        }
        __syncthreads();
        const int cnt = min(kSmallThreads, P - s0);
        real px = 0, py = 0;                                // per-chunk partial sums (two-level accumulation)
        for (int j = part; j < cnt; j += kSmallSplit) {
            if ((unsigned)(s0 + j - own) < (unsigned)npts) continue;      // own vesicle: self term, not ours
            const real rx = xi.x - sx[j], ry = xi.y - sy[j];
            if (sizeof(real) == 4) {
                const float r2 = fmaf((float)rx, (float)rx, (float)ry * (float)ry);
                const float ml = -0.34657359027997264f * sfu_lg2(r2);
                const float qd = fmaf((float)rx, (float)gx[j], (float)ry * (float)gy[j]) * sfu_rcp(r2);
                px += fmaf(ml, (float)gx[j], qd * (float)rx);
                py += fmaf(ml, (float)gy[j], qd * (float)ry);
            } else {
                const double r2 = fma((double)rx, (double)rx, (double)ry * (double)ry);
                const double ml = -0.5 * log(r2);
                const double qd = fma((double)rx, (double)gx[j], (double)ry * (double)gy[j]) / r2;
                px += fma(ml, (double)gx[j], qd * (double)rx);
                py += fma(ml, (double)gy[j], qd * (double)ry);
            }
        }
        ux += px;
        uy += py;
    }
#pragma unroll
    for (int m = 1; m < kSmallSplit; m <<= 1) {
        ux += __shfl_xor_sync(0xffffffffu, ux, m);
        uy += __shfl_xor_sync(0xffffffffu, uy, m);
    }
    if (live && part == 0) {
        real2 o;
        o.x = (real)(prefactor * (double)ux);
        o.y = (real)(prefactor * (double)uy);
        U[i] = o;
    }
}

vn_status farfield_small(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu, void *U,
                         vn_precision prec, cudaStream_t st)
{
    const int P = (int)(nves * npts);
    const int grid = (P + kSmallTargets - 1) / kSmallTargets;
    const double pref = 1.0 / (4.0 * 3.14159265358979323846 * mu);
    profile_mark(st, true);
    if (prec == VN_F32)
        farfield_small_kernel<float, float2><<<grid, kSmallThreads, 0, st>>>((const float2 *)X, (const float2 *)F,
                                                                              (const float *)W, P, (int)npts, pref, (float2 *)U);
    else
        farfield_small_kernel<double, double2><<<grid, kSmallThreads, 0, st>>>((const double2 *)X, (const double2 *)F,
                                                                                (const double *)W, P, (int)npts, pref, (double2 *)U);
    profile_mark(st, false);
    count_launch(1);
    return cudaGetLastError() == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

}  // namespace vn

// vn_weights.cu -- step a-1: trapezoid arclength weights W[v,j] = (2 pi / N) |dX_v/dalpha (alpha_j)|
// (PAPER.md:163-169 spectral derivative, :173 trapezoid rule).
//
// The Fourier derivative with the unmatched k = N/2 mode dropped (reading A4) is the
// circulant matrix
//     D_jk = 1/2 (-1)^(j-k) cot((j-k) pi / N)   (N even),   1/2 (-1)^(j-k) csc((j-k) pi / N)   (N odd),
//     D_jj = 0,
// applied directly: O(N^2) per vesicle, 2.6e8 FMAs at 8,000 x 128 -- four orders of magnitude
// below the pair sum, so no FFT.  Arithmetic is double for both storage precisions: in fp32 the
// products c*x with box coordinates ~1e2 and cot ~ N/pi would lose the derivative to rounding.
#include "vn_common.cuh"

namespace vn {

// c[m] = D_{j, j-m}: first column of the circulant, m = 0 .. N-1.
__device__ __forceinline__ double weights_coeff(int m, int N)
{
    if (m == 0) return 0.0;
    const double a = (double)m / (double)N;              // angle / pi
    const double sn = sinpi(a), cs = cospi(a);
    const double sign = (m & 1) ? -1.0 : 1.0;
    return (N & 1) ? 0.5 * sign / sn : 0.5 * sign * cs / sn;
}
__global__ void weights_table(int N, double *__restrict__ c)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m < N) c[m] = weights_coeff(m, N);
}
// Up to kLocalTable points per vesicle every block builds the column itself, in shared memory (N / 128 coefficients
// per thread against 2 N FMAs of its own work): no table kernel and no scratch allocation around the call, which at
// 16 x 32 points cost more than the weights.
constexpr int kLocalTable = 1024;

template <typename real, typename real2, bool LOCAL>
__global__ void __launch_bounds__(128)
weights_kernel(const real2 *__restrict__ X, int N, const double *__restrict__ cg, real *__restrict__ W)
{
    __shared__ double sx[128], sy[128];
    __shared__ double sc[LOCAL ? kLocalTable : 1];
    const double *c = cg;
    if (LOCAL) {
        for (int m = threadIdx.x; m < N; m += 128) sc[m] = weights_coeff(m, N);
        c = sc;                                          // the first barrier of the loop below orders these writes
    }
    const int v = blockIdx.y;
    const int j = blockIdx.x * 128 + threadIdx.x;
    const real2 *Xv = X + (size_t)v * N;
    // differences to the vesicle's first point: D annihilates constants, and small numbers round less
    const double x0 = (double)Xv[0].x, y0 = (double)Xv[0].y;
    double dx = 0.0, dy = 0.0;
    for (int k0 = 0; k0 < N; k0 += 128) {
        const int k = k0 + threadIdx.x;
        __syncthreads();
        if (k < N) {
            const real2 p = Xv[k];
            sx[threadIdx.x] = (double)p.x - x0;
            sy[threadIdx.x] = (double)p.y - y0;
        }
        __syncthreads();
        if (j < N) {
            const int cnt = min(128, N - k0);
            int m = j - k0;                    // (j - k) mod N, walks down as k walks up
            if (m < 0) m += N;
            for (int q = 0; q < cnt; ++q) {
                const double cm = LOCAL ? c[m] : __ldg(c + m);
                dx = fma(cm, sx[q], dx);
                dy = fma(cm, sy[q], dy);
                m = (m == 0) ? N - 1 : m - 1;
            }
        }
    }
    if (j < N)
        W[(size_t)v * N + j] = (real)((2.0 * 3.14159265358979323846 / (double)N) * sqrt(dx * dx + dy * dy));
}

vn_status arclength_weights(const void *X, int64_t nves, int64_t npts, void *W, vn_precision prec, cudaStream_t st)
{
    const int N = (int)npts;
    const bool local = N <= kLocalTable;
    double *c = nullptr;
    if (!local) {
        VN_CUDA(cudaMallocAsync((void **)&c, sizeof(double) * (size_t)N, st));
        weights_table<<<(N + 127) / 128, 128, 0, st>>>(N, c);
        count_launch(1);
    }
    // grid.y is limited to 65535: walk the vesicles in slabs
    const int jb = (N + 127) / 128;
    for (int64_t v0 = 0; v0 < nves; v0 += 65535) {
        const int nv = (int)((nves - v0) < 65535 ? (nves - v0) : 65535);
        const dim3 grid(jb, nv);
        if (prec == VN_F32) {
            if (local) weights_kernel<float, float2, true><<<grid, 128, 0, st>>>((const float2 *)X + v0 * N, N, c, (float *)W + v0 * N);
            else weights_kernel<float, float2, false><<<grid, 128, 0, st>>>((const float2 *)X + v0 * N, N, c, (float *)W + v0 * N);
        } else {
            if (local) weights_kernel<double, double2, true><<<grid, 128, 0, st>>>((const double2 *)X + v0 * N, N, c, (double *)W + v0 * N);
            else weights_kernel<double, double2, false><<<grid, 128, 0, st>>>((const double2 *)X + v0 * N, N, c, (double *)W + v0 * N);
        }
        count_launch(1);
    }
    const cudaError_t e = cudaGetLastError();
    if (!local) VN_CUDA(cudaFreeAsync(c, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

}  // namespace vn

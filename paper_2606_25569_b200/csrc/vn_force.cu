// vn_force.cu -- row f-2 of DESIGN.md: the elastic membrane force, the producer of the density F that
// vn_farfield consumes (PAPER.md:123 eq 2.7, :319 Fig. 5b; evaluated twice per time step, :451):
//
//     f = -kappa_b X_ssss + (sigma X_s)_s ,      d/ds = |dX/dalpha|^-1 d/dalpha
//
// d/dalpha is the Fourier derivative with the unmatched k = N/2 mode dropped, applied as the circulant
// matrix of vn_weights.cu (same table kernel).  One block per vesicle, everything in shared memory:
// five applications of D to a two-component array (X -> X_alpha, three more for X_ssss, one for the
// tension term), 10 N^2 DFMA per vesicle -- 1.3e9 at 8,000 x 128, four orders of magnitude below the
// pair sum.  Arithmetic is double for both storage precisions: the fourth derivative amplifies
// rounding by (N/2)^4 / |X_alpha|^4 (~1e8 at N = 128), which fp32 arithmetic cannot afford.
#include "vn_common.cuh"

namespace vn {

__global__ void weights_table(int N, double *__restrict__ c);   // vn_weights.cu


// out = D in for both components; in/out are shared-memory arrays of N doubles each, c the first column of the
// circulant.  When N is a multiple of 4 a thread owns four consecutive outputs and walks the inputs four at a
// time over a sliding window of seven table entries (two aligned groups of four): 32 DFMA per six 16-byte
// shared-memory loads instead of 2 DFMA per three 8-byte loads.
template <int kForceThreads>
__device__ __forceinline__ void apply_D(const double *__restrict__ c, int N, const double *inx, const double *iny,
                                        double *outx, double *outy)
{
    if ((N & 3) == 0) {
        const int G = N >> 2;                       // groups of four
        for (int t = threadIdx.x; t < G; t += kForceThreads) {
            double dx[4] = {0.0, 0.0, 0.0, 0.0}, dy[4] = {0.0, 0.0, 0.0, 0.0};
            int u = t;                              // (t - g) mod G: c[4u + (r - s)] multiplies in[4g + s] into out[4t + r]
            double cA[4], cB[4];
            {
                const double2 a = ((const double2 *)(c + 4 * u))[0], b = ((const double2 *)(c + 4 * u))[1];
                cA[0] = a.x; cA[1] = a.y; cA[2] = b.x; cA[3] = b.y;
            }
            for (int g = 0; g < G; ++g) {
                const int um = (u == 0) ? G - 1 : u - 1;
                {
                    const double2 a = ((const double2 *)(c + 4 * um))[0], b = ((const double2 *)(c + 4 * um))[1];
                    cB[0] = a.x; cB[1] = a.y; cB[2] = b.x; cB[3] = b.y;
                }
                double vx[4], vy[4];
                {
                    const double2 a = ((const double2 *)(inx + 4 * g))[0], b = ((const double2 *)(inx + 4 * g))[1];
                    vx[0] = a.x; vx[1] = a.y; vx[2] = b.x; vx[3] = b.y;
                    const double2 e = ((const double2 *)(iny + 4 * g))[0], f = ((const double2 *)(iny + 4 * g))[1];
                    vy[0] = e.x; vy[1] = e.y; vy[2] = f.x; vy[3] = f.y;
                }
#pragma unroll
                for (int sidx = 0; sidx < 4; ++sidx)
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        const double cm = r >= sidx ? cA[r - sidx] : cB[4 + r - sidx];
                        dx[r] = fma(cm, vx[sidx], dx[r]);
                        dy[r] = fma(cm, vy[sidx], dy[r]);
                    }
#pragma unroll
                for (int r = 0; r < 4; ++r) cA[r] = cB[r];
                u = um;
            }
#pragma unroll
            for (int r = 0; r < 4; ++r) { outx[4 * t + r] = dx[r]; outy[4 * t + r] = dy[r]; }
        }
        return;
    }
    for (int j = threadIdx.x; j < N; j += kForceThreads) {
        double dx = 0.0, dy = 0.0;
        int m = j;                                  // (j - q) mod N for q = 0
        for (int q = 0; q < N; ++q) {
            const double cm = c[m];
            dx = fma(cm, inx[q], dx);
            dy = fma(cm, iny[q], dy);
            m = (m == 0) ? N - 1 : m - 1;
        }
        outx[j] = dx;
        outy[j] = dy;
    }
}

// kForceThreads = 32 for npts <= 256 (with four outputs per thread one warp covers 128 points; small blocks keep
// more vesicles in flight: 0.15 ms against 0.21 ms at 8,000 x 128), 128 otherwise (npts <= 1024: <= 8 points per thread)
template <typename real, typename real2, int kForceThreads>
__global__ void __launch_bounds__(kForceThreads)
elastic_force_kernel(const real2 *__restrict__ X, const real *__restrict__ sigma, int N, double kappa_b,
                     const double *__restrict__ ctab, real2 *__restrict__ F)
{
    extern __shared__ __align__(16) double sm[];
    double *c = sm, *sa = sm + N;
    double *ax = sm + 2 * N, *ay = sm + 3 * N, *bx = sm + 4 * N, *by = sm + 5 * N, *sx = sm + 6 * N, *sy = sm + 7 * N;
    const size_t v0 = (size_t)blockIdx.x * N;
    const double x0 = (double)X[v0].x, y0 = (double)X[v0].y;      // D annihilates constants
    for (int j = threadIdx.x; j < N; j += kForceThreads) {
        const real2 p = X[v0 + j];
        c[j] = ctab[j];
        ax[j] = (double)p.x - x0;
        ay[j] = (double)p.y - y0;
    }
    __syncthreads();
    apply_D<kForceThreads>(c, N, ax, ay, bx, by);                                 // X_alpha
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += kForceThreads) {
        const double s = sqrt(bx[j] * bx[j] + by[j] * by[j]);
        sa[j] = s;
        sx[j] = bx[j] / s;                                         // X_s
        sy[j] = by[j] / s;
        const double sg = (double)sigma[v0 + j];
        ax[j] = sg * sx[j];                                        // sigma X_s
        ay[j] = sg * sy[j];
    }
    __syncthreads();
    apply_D<kForceThreads>(c, N, ax, ay, bx, by);                                 // d/dalpha (sigma X_s)
    __syncthreads();
    double tx[8], ty[8];                                           // (sigma X_s)_s of this thread's points
    const int per = (N + kForceThreads - 1) / kForceThreads;       // <= 8: 32 threads up to npts 256, 128 threads up to 1024
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int j = threadIdx.x + k * kForceThreads;
        tx[k] = ty[k] = 0.0;
        if (k < per && j < N) { tx[k] = bx[j] / sa[j]; ty[k] = by[j] / sa[j]; }
    }
    // X_ss, X_sss, X_ssss
    const double *inx = sx, *iny = sy;
    for (int rep = 0; rep < 3; ++rep) {
        __syncthreads();
        apply_D<kForceThreads>(c, N, inx, iny, bx, by);
        __syncthreads();
        for (int j = threadIdx.x; j < N; j += kForceThreads) {
            ax[j] = bx[j] / sa[j];
            ay[j] = by[j] / sa[j];
        }
        inx = ax; iny = ay;
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int j = threadIdx.x + k * kForceThreads;
        if (k < per && j < N) {
            real2 o;
            o.x = (real)fma(-kappa_b, ax[j], tx[k]);
            o.y = (real)fma(-kappa_b, ay[j], ty[k]);
            F[v0 + j] = o;
        }
    }
}

vn_status elastic_force(const void *X, const void *sigma, int64_t nves, int64_t npts, double kappa_b, void *F,
                        vn_precision prec, cudaStream_t st)
{
    const int N = (int)npts;
    const size_t smem = sizeof(double) * 8 * (size_t)N;
    static bool attr_dev[kMaxDevices] = {false};
    bool &attr_set = attr_dev[current_device()];
    if (!attr_set) {
        VN_CUDA(cudaFuncSetAttribute(elastic_force_kernel<float, float2, 128>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
        VN_CUDA(cudaFuncSetAttribute(elastic_force_kernel<double, double2, 128>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
        attr_set = true;
    }
    double *c = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&c, sizeof(double) * (size_t)N, st));
    weights_table<<<(N + 127) / 128, 128, 0, st>>>(N, c);
    for (int64_t v0 = 0; v0 < nves; v0 += 1 << 30) {
        const int nv = (int)((nves - v0) < (1 << 30) ? (nves - v0) : (1 << 30));
        if (prec == VN_F32 && N <= 256)
            elastic_force_kernel<float, float2, 32><<<nv, 32, smem, st>>>(
                (const float2 *)X + v0 * N, (const float *)sigma + v0 * N, N, kappa_b, c, (float2 *)F + v0 * N);
        else if (prec == VN_F32)
            elastic_force_kernel<float, float2, 128><<<nv, 128, smem, st>>>(
                (const float2 *)X + v0 * N, (const float *)sigma + v0 * N, N, kappa_b, c, (float2 *)F + v0 * N);
        else if (N <= 256)
            elastic_force_kernel<double, double2, 32><<<nv, 32, smem, st>>>(
                (const double2 *)X + v0 * N, (const double *)sigma + v0 * N, N, kappa_b, c, (double2 *)F + v0 * N);
        else
            elastic_force_kernel<double, double2, 128><<<nv, 128, smem, st>>>(
                (const double2 *)X + v0 * N, (const double *)sigma + v0 * N, N, kappa_b, c, (double2 *)F + v0 * N);
        count_launch(1);
    }
    count_launch(1);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(c, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

}  // namespace vn

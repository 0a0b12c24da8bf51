// vn_redistribute.cu -- row f-3 of DESIGN.md: redistributing the points of every vesicle equally in
// arclength (PAPER.md:331-335 sec 4.2; called three times per time step, :451, :463) -- the "boundary
// reparameterization" module the abstract names beside the N-body sum.
//
// In the paper's order (readings R1-R5):
//   1. upsample by 6: trigonometric interpolant of X on M = 6 N nodes (an even N keeps its k = N/2 mode
//      as cos(N alpha / 2));
//   2. arclength at the fine nodes: sa = |dX/dalpha| (Fourier derivative, Nyquist mode dropped), then the
//      Fourier series of sa on the fine grid integrated term by term (its k = M/2 mode dropped);
//   3. for the equispaced targets l~_k = k L / N: search the increasing sequence l_0 .. l_M for the
//      interval, theta from its two endpoints, Xnew_k = Xup_m + theta (Xup_{m+1} - Xup_m).
// One block per vesicle, everything in shared memory, direct O(M^2) sums with a twiddle table
// (M = 768 at npts = 128: 1.6e6 DFMA per vesicle, 1.3e10 at 8,000 vesicles -- 1 % of one pair sum;
// 6 N is not a power of two and the size does not pay for a mixed-radix FFT).  Arithmetic is double for
// both storage precisions.
#include "vn_common.cuh"

namespace vn {

constexpr int kRedThreads = 256;
constexpr int kUp = 6;

__global__ void twiddle_table(int M, double2 *__restrict__ tw)   // (cos, sin)(2 pi m / M)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= M) return;
    double s, c;
    sincospi(2.0 * (double)m / (double)M, &s, &c);
    tw[m] = make_double2(c, s);
}

template <typename real, typename real2>
__global__ void __launch_bounds__(kRedThreads)
redistribute_kernel(const real2 *__restrict__ X, int N, const double2 *__restrict__ twg, real2 *__restrict__ Xnew)
{
    extern __shared__ __align__(16) double sm[];
    const int M = kUp * N, K = (N - 1) / 2, H = M / 2 - 1;      // H = highest mode of sa that is kept
    double2 *tw = (double2 *)sm;                                  // [M]
    double *cf = sm + 2 * M;                                      // [4 (K+1)]: (re_x, im_x, re_y, im_y), k = 0..K
    double *xu = cf + 4 * (K + 1), *yu = xu + M, *sa = yu + M, *l = sa + M;   // l: [M+1]
    double *p = l + M + 1, *q = p + (H + 1);                      // [H+1] each
    double *x0 = q + (H + 1), *y0 = x0 + N;                       // the vesicle, relative to its first point
    __shared__ double nyq[2], s0_sh;
    const int tid = threadIdx.x;
    const size_t v0 = (size_t)blockIdx.x * N;
    const double ox = (double)X[v0].x, oy = (double)X[v0].y;

    for (int m = tid; m < M; m += kRedThreads) tw[m] = twg[m];
    for (int j = tid; j < N; j += kRedThreads) {
        const real2 pt = X[v0 + j];
        x0[j] = (double)pt.x - ox;
        y0[j] = (double)pt.y - oy;
    }
    __syncthreads();

    // 1a. Fourier coefficients k = 0..K (the signal is real: k < 0 is the conjugate), and k = N/2
    for (int k = tid; k <= K; k += kRedThreads) {
        double rx = 0.0, ix = 0.0, ry = 0.0, iy = 0.0;
        int a = 0;                                               // (6 k j) mod M
        const int step = (kUp * k) % M;
        for (int j = 0; j < N; ++j) {
            const double2 t = tw[a];
            rx = fma(x0[j], t.x, rx); ix = fma(-x0[j], t.y, ix);
            ry = fma(y0[j], t.x, ry); iy = fma(-y0[j], t.y, iy);
            a += step; if (a >= M) a -= M;
        }
        const double inv = 1.0 / (double)N;
        cf[4 * k + 0] = rx * inv; cf[4 * k + 1] = ix * inv; cf[4 * k + 2] = ry * inv; cf[4 * k + 3] = iy * inv;
    }
    if (tid == kRedThreads - 1) {
        double nx = 0.0, ny = 0.0;
        if ((N & 1) == 0)
            for (int j = 0; j < N; ++j) { nx += (j & 1) ? -x0[j] : x0[j]; ny += (j & 1) ? -y0[j] : y0[j]; }
        nyq[0] = nx / (double)N; nyq[1] = ny / (double)N;
    }
    __syncthreads();

    // 1b / 2a. interpolant and |derivative| on the fine grid
    for (int m = tid; m < M; m += kRedThreads) {
        double x = cf[0], y = cf[2], dx = 0.0, dy = 0.0;
        int a = 0;                                               // (k m) mod M
        for (int k = 1; k <= K; ++k) {
            a += m; if (a >= M) a -= M;
            const double2 t = tw[a];
            const double rx = cf[4 * k + 0], ix = cf[4 * k + 1], ry = cf[4 * k + 2], iy = cf[4 * k + 3];
            const double ex = fma(rx, t.x, -ix * t.y), ey = fma(ry, t.x, -iy * t.y);        // Re(c e^{ik a})
            const double fx = fma(-ix, t.x, -rx * t.y), fy = fma(-iy, t.x, -ry * t.y);      // Re(i c e^{ik a})
            x = fma(2.0, ex, x); y = fma(2.0, ey, y);
            dx = fma(2.0 * (double)k, fx, dx); dy = fma(2.0 * (double)k, fy, dy);
        }
        if ((N & 1) == 0) {
            const double cn = tw[(int)(((long long)(N / 2) * m) % M)].x;
            x = fma(nyq[0], cn, x); y = fma(nyq[1], cn, y);
        }
        xu[m] = x; yu[m] = y;
        sa[m] = sqrt(dx * dx + dy * dy);
    }
    __syncthreads();

    // 2b. Fourier coefficients of sa: mean and modes 1..H
    for (int k = tid; k <= H; k += kRedThreads) {
        double pr = 0.0, qi = 0.0;
        int a = 0;
        for (int m = 0; m < M; ++m) {
            const double2 t = tw[a];
            pr = fma(sa[m], t.x, pr); qi = fma(-sa[m], t.y, qi);
            a += k; if (a >= M) a -= M;
        }
        p[k] = pr / (double)M; q[k] = qi / (double)M;
        if (k == 0) s0_sh = pr / (double)M;
    }
    __syncthreads();
    const double s0 = s0_sh;
    for (int k = tid + 1; k <= H; k += kRedThreads) {            // fold the 2/k of the integration in
        p[k] *= 2.0 / (double)k; q[k] *= 2.0 / (double)k;
    }
    __syncthreads();

    // 2c. l_m = s0 alpha'_m + sum_k [ p_k sin(k alpha'_m) - q_k (1 - cos(k alpha'_m)) ]
    const double two_pi = 6.283185307179586476925286766559;
    for (int m = tid; m < M; m += kRedThreads) {
        double acc = 0.0;
        int a = 0;
        for (int k = 1; k <= H; ++k) {
            a += m; if (a >= M) a -= M;
            const double2 t = tw[a];
            acc = fma(p[k], t.y, acc);
            acc = fma(-q[k], 1.0 - t.x, acc);
        }
        l[m] = fma(s0, two_pi * (double)m / (double)M, acc);
    }
    if (tid == 0) l[M] = two_pi * s0;
    __syncthreads();

    // 3. search and interpolate
    const double L = two_pi * s0;
    for (int k = tid; k < N; k += kRedThreads) {
        const double lt = (double)k * L / (double)N;
        int lo = 0, hi = M - 1;                                  // smallest m with l[m+1] > lt (l increasing)
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (l[mid + 1] > lt) hi = mid; else lo = mid + 1;
        }
        const int m = lo, m1 = (m + 1 == M) ? 0 : m + 1;
        const double theta = (lt - l[m]) / (l[m + 1] - l[m]);
        real2 o;
        o.x = (real)(ox + fma(theta, xu[m1] - xu[m], xu[m]));
        o.y = (real)(oy + fma(theta, yu[m1] - yu[m], yu[m]));
        Xnew[v0 + k] = o;
    }
}

static size_t redistribute_smem(int N)
{
    const int M = kUp * N, K = (N - 1) / 2, H = M / 2 - 1;
    return sizeof(double) * (size_t)(2 * M + 4 * (K + 1) + 3 * M + (M + 1) + 2 * (H + 1) + 2 * N);
}

vn_status redistribute(const void *X, int64_t nves, int64_t npts, void *Xnew, vn_precision prec, cudaStream_t st)
{
    const int N = (int)npts, M = kUp * N;
    const size_t smem = redistribute_smem(N);
    static bool attr_set = false;
    if (!attr_set) {
        const int cap = (int)redistribute_smem(512);
        VN_CUDA(cudaFuncSetAttribute(redistribute_kernel<float, float2>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap));
        VN_CUDA(cudaFuncSetAttribute(redistribute_kernel<double, double2>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap));
        attr_set = true;
    }
    double2 *tw = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&tw, sizeof(double2) * (size_t)M, st));
    twiddle_table<<<(M + 127) / 128, 128, 0, st>>>(M, tw);
    for (int64_t v0 = 0; v0 < nves; v0 += 1 << 30) {
        const int nv = (int)((nves - v0) < (1 << 30) ? (nves - v0) : (1 << 30));
        if (prec == VN_F32)
            redistribute_kernel<float, float2><<<nv, kRedThreads, smem, st>>>((const float2 *)X + v0 * N, N, tw,
                                                                               (float2 *)Xnew + v0 * N);
        else
            redistribute_kernel<double, double2><<<nv, kRedThreads, smem, st>>>((const double2 *)X + v0 * N, N, tw,
                                                                                 (double2 *)Xnew + v0 * N);
        count_launch(1);
    }
    count_launch(1);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(tw, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

}  // namespace vn

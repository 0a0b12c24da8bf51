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
// Every step is linear in its input and periodic, i.e. a circulant: the trigonometric interpolant and its
// derivative are  Xup_m = sum_j D0[(m - 6 j) mod M] X_j,  X'up_m = sum_j D1[(m - 6 j) mod M] X_j  (Dirichlet
// kernel and its derivative sampled on the fine grid), and the term-by-term integral of the Fourier series of sa
// is  prim_m = sum_n G[(m - n) mod M] sa_n,  G[d] = (1/M) sum_{k=1}^{M/2-1} (2/k) sin(2 pi k d / M), so that
// l_m = mean(sa) alpha'_m + prim_m - prim_0.  The three tables are built once per call; one block per vesicle
// then applies them from shared memory: thread c owns the six fine nodes 6c .. 6c+5 of coarse point c, all
// table reads are 16-byte loads at a 48-byte lane stride (conflict-free), inputs are broadcast, and the
// integration walks the sources six at a time over a sliding 12-entry window of G (36 DFMA per 6 loads).
// M = 768 at npts = 128: 0.98e6 DFMA per vesicle, 7.9e9 at 8,000 vesicles -- under 1 % of one pair sum; 6 N is
// not a power of two and the size does not pay for a mixed-radix FFT.  Arithmetic is double for both
// storage precisions.
#include "vn_common.cuh"

namespace vn {

constexpr int kRedThreads = 128;
constexpr int kUp = 6;

// D0, D1, G (M doubles each, consecutive) -- see the header comment.
__global__ void redistribute_tables(int N, double *__restrict__ tab)
{
    const int M = kUp * N, K = (N - 1) / 2, H = M / 2 - 1;
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= M) return;
    double d0 = 1.0, d1 = 0.0, g = 0.0;
    int a = 0;                                                   // (k d) mod M
    for (int k = 1; k <= H; ++k) {
        a += d; if (a >= M) a -= M;
        double sn, cs;
        sincospi(2.0 * (double)a / (double)M, &sn, &cs);
        if (k <= K) { d0 = fma(2.0, cs, d0); d1 = fma(-2.0 * (double)k, sn, d1); }
        g = fma(2.0 / (double)k, sn, g);
    }
    if ((N & 1) == 0) d0 += cospi(2.0 * (double)(((long long)(N / 2) * d) % M) / (double)M);
    tab[d] = d0 / (double)N;
    tab[M + d] = d1 / (double)N;
    tab[2 * M + d] = g / (double)M;
}

template <typename real, typename real2>
__global__ void __launch_bounds__(kRedThreads)
redistribute_kernel(const real2 *__restrict__ X, int N, const double *__restrict__ tabg, real2 *__restrict__ Xnew)
{
    extern __shared__ __align__(16) double sm[];
    const int M = kUp * N;
    double *D0 = sm, *D1 = sm + M, *G = sm + 2 * M;
    double *xu = sm + 3 * M, *yu = sm + 4 * M, *sa = sm + 5 * M;
    double2 *xy = (double2 *)(sm + 6 * M);                        // [N] the vesicle, relative to its first point
    double *l = sm + 6 * M + 2 * N;                               // [M+1]
    __shared__ double red[kRedThreads / 32], s0_sh, prim0_sh;
    const int tid = threadIdx.x;
    const size_t v0 = (size_t)blockIdx.x * N;
    const double ox = (double)X[v0].x, oy = (double)X[v0].y;

    for (int m = tid; m < 3 * M; m += kRedThreads) sm[m] = tabg[m];
    for (int j = tid; j < N; j += kRedThreads) {
        const real2 pt = X[v0 + j];
        xy[j] = make_double2((double)pt.x - ox, (double)pt.y - oy);
    }
    __syncthreads();

    // 1 / 2a. interpolant and |derivative| at the six fine nodes of every coarse point
    double part = 0.0;                                            // this thread's share of sum(sa)
    for (int c = tid; c < N; c += kRedThreads) {
        double ax[kUp], ay[kUp], bx[kUp], by[kUp];
#pragma unroll
        for (int r = 0; r < kUp; ++r) ax[r] = ay[r] = bx[r] = by[r] = 0.0;
        int u = c;                                                // (c - j) mod N
        for (int j = 0; j < N; ++j) {
            const double2 pj = xy[j];
            const double2 *e0 = (const double2 *)(D0 + kUp * u), *e1 = (const double2 *)(D1 + kUp * u);
#pragma unroll
            for (int h = 0; h < kUp / 2; ++h) {
                const double2 a0 = e0[h], a1 = e1[h];
                ax[2 * h] = fma(a0.x, pj.x, ax[2 * h]);         ay[2 * h] = fma(a0.x, pj.y, ay[2 * h]);
                ax[2 * h + 1] = fma(a0.y, pj.x, ax[2 * h + 1]); ay[2 * h + 1] = fma(a0.y, pj.y, ay[2 * h + 1]);
                bx[2 * h] = fma(a1.x, pj.x, bx[2 * h]);         by[2 * h] = fma(a1.x, pj.y, by[2 * h]);
                bx[2 * h + 1] = fma(a1.y, pj.x, bx[2 * h + 1]); by[2 * h + 1] = fma(a1.y, pj.y, by[2 * h + 1]);
            }
            u = (u == 0) ? N - 1 : u - 1;
        }
#pragma unroll
        for (int r = 0; r < kUp; ++r) {
            const double s = sqrt(bx[r] * bx[r] + by[r] * by[r]);
            xu[kUp * c + r] = ax[r];
            yu[kUp * c + r] = ay[r];
            sa[kUp * c + r] = s;
            part += s;
        }
    }
#pragma unroll
    for (int k = 16; k >= 1; k >>= 1) part += __shfl_xor_sync(0xffffffffu, part, k);
    if ((tid & 31) == 0) red[tid >> 5] = part;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
        for (int k = 0; k < kRedThreads / 32; ++k) t += red[k];
        s0_sh = t / (double)M;
    }

    // 2b. prim_m = sum_n G[(m - n) mod M] sa_n: sources six at a time, G window = groups u-1 and u
    const double two_pi = 6.283185307179586476925286766559;
    for (int c = tid; c < N; c += kRedThreads) {
        double acc[kUp];
#pragma unroll
        for (int r = 0; r < kUp; ++r) acc[r] = 0.0;
        int u = c;                                                // (c - q) mod N
        double gA[kUp], gB[kUp];                                  // G[6u .. 6u+5], G[6(u-1) .. 6(u-1)+5]
#pragma unroll
        for (int h = 0; h < kUp / 2; ++h) {
            const double2 t = ((const double2 *)(G + kUp * u))[h];
            gA[2 * h] = t.x; gA[2 * h + 1] = t.y;
        }
        for (int q = 0; q < N; ++q) {
            const int um = (u == 0) ? N - 1 : u - 1;
#pragma unroll
            for (int h = 0; h < kUp / 2; ++h) {
                const double2 t = ((const double2 *)(G + kUp * um))[h];
                gB[2 * h] = t.x; gB[2 * h + 1] = t.y;
            }
            double sn[kUp];
#pragma unroll
            for (int h = 0; h < kUp / 2; ++h) {
                const double2 t = ((const double2 *)(sa + kUp * q))[h];
                sn[2 * h] = t.x; sn[2 * h + 1] = t.y;
            }
#pragma unroll
            for (int sidx = 0; sidx < kUp; ++sidx)
#pragma unroll
                for (int r = 0; r < kUp; ++r)
                    acc[r] = fma(r >= sidx ? gA[r - sidx] : gB[kUp + r - sidx], sn[sidx], acc[r]);
#pragma unroll
            for (int r = 0; r < kUp; ++r) gA[r] = gB[r];
            u = um;
        }
#pragma unroll
        for (int r = 0; r < kUp; ++r) l[kUp * c + r] = acc[r];
        if (c == 0) prim0_sh = acc[0];
    }
    __syncthreads();
    const double s0 = s0_sh, prim0 = prim0_sh;
    for (int m = tid; m < M; m += kRedThreads) l[m] = fma(s0, two_pi * (double)m / (double)M, l[m] - prim0);
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
    const int M = kUp * N;
    return sizeof(double) * (size_t)(7 * M + 2 * N + 1);
}

vn_status redistribute(const void *X, int64_t nves, int64_t npts, void *Xnew, vn_precision prec, cudaStream_t st)
{
    const int N = (int)npts, M = kUp * N;
    const size_t smem = redistribute_smem(N);
    static bool attr_dev[kMaxDevices] = {false};
    bool &attr_set = attr_dev[current_device()];
    if (!attr_set) {
        const int cap = (int)redistribute_smem(512);
        VN_CUDA(cudaFuncSetAttribute(redistribute_kernel<float, float2>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap));
        VN_CUDA(cudaFuncSetAttribute(redistribute_kernel<double, double2>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap));
        attr_set = true;
    }
    double *tw = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&tw, sizeof(double) * 3 * (size_t)M, st));
    redistribute_tables<<<(M + 127) / 128, 128, 0, st>>>(N, tw);
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

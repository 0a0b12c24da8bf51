// vn_near.cu -- row f-1 of DESIGN.md: the near-field relation and the correction that turns the plain
// far-field sum into the paper's DirectSingleLayerIntegral.
//
//   near(t, v')  <=>  v' != ves(t)  and  min_j |x_t - X[v',j]| <= h_v',   h_v' = max_j W[v',j]
//   (PAPER.md:144 "distance of x to the vesicle <= the arclength spacing", :248 |d| <= h, :426
//    FindNearFieldPoints; reading N1 for h)
//   U_masked[t] = U[t] - 1/(4 pi mu) sum_{v' near t} sum_j K(x_t - X[v',j]) F[v',j] W[v',j]
//   (PAPER.md:329: "boolean masks to set neighboring vesicles' contribution to zero"; :425)
//
// The relation is sparse (a point has at most a handful of near vesicles), so nothing P x nves is ever
// formed: vesicle bounding boxes cull the vesicle pairs, the surviving pairs get the exact
// point-to-point test, and the result is a CSR list (near_ptr[P+1], near_ves[nnz]) in ascending
// (t, v') order.  The decision d^2 <= h^2 is taken in double for both storage precisions (inputs
// promoted), so that it does not depend on fp32 rounding of the distance.
#include "vn_common.cuh"

namespace vn {

constexpr int kNearThreads = 128;

// ------------------------------------------------------------------------------------------------
// per-vesicle bounding box (xmin, xmax, ymin, ymax) and spacing h = max_j W
template <typename real, typename real2>
__global__ void __launch_bounds__(kNearThreads)
vesicle_bounds(const real2 *__restrict__ X, const real *__restrict__ W, int npts, double4 *__restrict__ bb,
               double *__restrict__ h)
{
    __shared__ double red[5][kNearThreads / 32];
    const int v = blockIdx.x;
    const real2 *Xv = X + (size_t)v * npts;
    const real *Wv = W + (size_t)v * npts;
    double xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY, hm = 0.0;
    for (int j = threadIdx.x; j < npts; j += kNearThreads) {
        const real2 p = Xv[j];
        xmin = fmin(xmin, (double)p.x); xmax = fmax(xmax, (double)p.x);
        ymin = fmin(ymin, (double)p.y); ymax = fmax(ymax, (double)p.y);
        hm = fmax(hm, (double)Wv[j]);
    }
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
        xmin = fmin(xmin, __shfl_xor_sync(0xffffffffu, xmin, m));
        xmax = fmax(xmax, __shfl_xor_sync(0xffffffffu, xmax, m));
        ymin = fmin(ymin, __shfl_xor_sync(0xffffffffu, ymin, m));
        ymax = fmax(ymax, __shfl_xor_sync(0xffffffffu, ymax, m));
        hm = fmax(hm, __shfl_xor_sync(0xffffffffu, hm, m));
    }
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { red[0][w] = xmin; red[1][w] = xmax; red[2][w] = ymin; red[3][w] = ymax; red[4][w] = hm; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < kNearThreads / 32; ++k) {
            xmin = fmin(xmin, red[0][k]); xmax = fmax(xmax, red[1][k]);
            ymin = fmin(ymin, red[2][k]); ymax = fmax(ymax, red[3][k]);
            hm = fmax(hm, red[4][k]);
        }
        bb[v] = make_double4(xmin, xmax, ymin, ymax);
        h[v] = hm;
    }
}

// ------------------------------------------------------------------------------------------------
// Block v = target vesicle.  Source vesicles v' are scanned in ascending order, 128 at a time: each
// thread tests one bounding box against the block's own (gap between the boxes <= h_v', a necessary
// condition), the survivors are listed in order, and every survivor gets the exact test
// min_j |x_i - X[v',j]|^2 <= h_v'^2 for every target point i of v.
//   FILL = false: cnt[t] = number of near vesicles of point t.
//   FILL = true : near_ves[cursor[t]++] = v' (cursor starts at near_ptr[t]; entries at or beyond
//                 `capacity` are dropped).
template <typename real2, bool FILL>
__global__ void __launch_bounds__(kNearThreads)
near_kernel(const real2 *__restrict__ X, int nves, int npts, const double4 *__restrict__ bb,
            const double *__restrict__ h, int *__restrict__ cnt, long long *__restrict__ cursor,
            int *__restrict__ near_ves, long long capacity)
{
    __shared__ int cand[kNearThreads];
    __shared__ int warp_cnt[kNearThreads / 32];
    __shared__ double2 ys[kNearThreads];
    const int v = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const double4 me = bb[v];
    const real2 *Xv = X + (size_t)v * npts;

    if (!FILL)
        for (int i = tid; i < npts; i += kNearThreads) cnt[(size_t)v * npts + i] = 0;

    for (int c0 = 0; c0 < nves; c0 += kNearThreads) {
        const int vp = c0 + tid;
        bool hit = false;
        if (vp < nves && vp != v) {
            const double4 o = bb[vp];
            const double gx = fmax(0.0, fmax(o.x - me.y, me.x - o.y));
            const double gy = fmax(0.0, fmax(o.z - me.w, me.z - o.w));
            const double hv = h[vp];
            hit = gx * gx + gy * gy <= hv * hv * (1.0 + 1e-12);   // never rejects a true near pair
        }
        const unsigned b = __ballot_sync(0xffffffffu, hit);
        __syncthreads();                                  // previous round's cand / ys are drained
        if (lane == 0) warp_cnt[wid] = __popc(b);
        __syncthreads();
        int before = 0, total = 0;
#pragma unroll
        for (int k = 0; k < kNearThreads / 32; ++k) {
            if (k < wid) before += warp_cnt[k];
            total += warp_cnt[k];
        }
        if (hit) cand[before + __popc(b & ((1u << lane) - 1u))] = vp;
        __syncthreads();

        for (int q = 0; q < total; ++q) {
            const int sv = cand[q];
            const real2 *Xs = X + (size_t)sv * npts;
            const double hv = h[sv];
            const double h2 = hv * hv;
            for (int i0 = 0; i0 < npts; i0 += kNearThreads) {       // target points of v
                const int i = i0 + tid;
                double tx = 0.0, ty = 0.0;
                if (i < npts) { const real2 p = Xv[i]; tx = (double)p.x; ty = (double)p.y; }
                double dmin2 = INFINITY;
                for (int j0 = 0; j0 < npts; j0 += kNearThreads) {   // source points of v'
                    __syncthreads();
                    if (j0 + tid < npts) { const real2 p = Xs[j0 + tid]; ys[tid] = make_double2((double)p.x, (double)p.y); }
                    __syncthreads();
                    const int n = min(kNearThreads, npts - j0);
                    for (int j = 0; j < n; ++j) {
                        const double rx = tx - ys[j].x, ry = ty - ys[j].y;
                        dmin2 = fmin(dmin2, rx * rx + ry * ry);
                    }
                }
                if (i < npts && dmin2 <= h2) {
                    const size_t t = (size_t)v * npts + i;
                    if (!FILL) {
                        cnt[t] += 1;
                    } else {
                        const long long pos = cursor[t];
                        cursor[t] = pos + 1;
                        if (pos < capacity) near_ves[pos] = sv;
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// exclusive scan cnt[P] -> ptr[P+1] (64-bit), three small kernels: block sums, scan of the block sums
// by one block, rescan with the offsets.

__device__ __forceinline__ long long block_exclusive_scan(long long v, long long *total)
{
    __shared__ long long wsum[kScanThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    long long incl = v;
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {
        const long long o = __shfl_up_sync(0xffffffffu, incl, m);
        if (lane >= m) incl += o;
    }
    __syncthreads();
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    long long before = 0, all = 0;
#pragma unroll
    for (int k = 0; k < kScanThreads / 32; ++k) {
        if (k < wid) before += wsum[k];
        all += wsum[k];
    }
    *total = all;
    return before + incl - v;
}

__global__ void __launch_bounds__(kScanThreads) scan_block_sums(const int *__restrict__ cnt, int P, long long *__restrict__ bsum)
{
    const int base = blockIdx.x * kScanBlock + threadIdx.x * kScanItems;
    long long s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
        if (base + k < P) s += cnt[base + k];
    long long total;
    (void)block_exclusive_scan(s, &total);
    if (threadIdx.x == 0) bsum[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanThreads) scan_of_sums(long long *__restrict__ bsum, int nb)
{
    long long carry = 0;
    for (int b0 = 0; b0 < nb; b0 += kScanThreads) {
        const int b = b0 + threadIdx.x;
        const long long v = b < nb ? bsum[b] : 0;
        long long total;
        const long long ex = block_exclusive_scan(v, &total);
        if (b < nb) bsum[b] = carry + ex;
        carry += total;
    }
}

__global__ void __launch_bounds__(kScanThreads)
scan_apply(const int *__restrict__ cnt, int P, const long long *__restrict__ bsum, long long *__restrict__ ptr,
           long long *__restrict__ cursor)
{
    const int base = blockIdx.x * kScanBlock + threadIdx.x * kScanItems;
    int c[kScanItems];
    long long s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        c[k] = base + k < P ? cnt[base + k] : 0;
        s += c[k];
    }
    long long total;
    long long off = bsum[blockIdx.x] + block_exclusive_scan(s, &total);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < P) {
            ptr[base + k] = off;
            if (cursor) cursor[base + k] = off;
        }
        off += c[k];
        if (base + k == P - 1) ptr[P] = off;
    }
}

// ------------------------------------------------------------------------------------------------
vn_status near_pairs(const void *X, const void *W, int64_t nves, int64_t npts, int64_t *near_ptr,
                     int32_t *near_ves, int64_t capacity, vn_precision prec, cudaStream_t st)
{
    const int P = (int)(nves * npts);
    const int nb = (P + kScanBlock - 1) / kScanBlock;
    const bool fill = near_ves != nullptr && capacity > 0;
    // scratch: bb | h | cnt | bsum | cursor
    auto up = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t b_bb = up(sizeof(double4) * (size_t)nves), b_h = up(sizeof(double) * (size_t)nves);
    const size_t b_cnt = up(sizeof(int) * (size_t)P), b_bs = up(sizeof(long long) * (size_t)nb);
    const size_t b_cur = fill ? up(sizeof(long long) * (size_t)P) : 0;
    char *scratch = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scratch, b_bb + b_h + b_cnt + b_bs + b_cur, st));
    double4 *bb = (double4 *)scratch;
    double *h = (double *)(scratch + b_bb);
    int *cnt = (int *)(scratch + b_bb + b_h);
    long long *bsum = (long long *)(scratch + b_bb + b_h + b_cnt);
    long long *cursor = fill ? (long long *)(scratch + b_bb + b_h + b_cnt + b_bs) : nullptr;

    const int nv = (int)nves, np = (int)npts;
    if (prec == VN_F32) {
        vesicle_bounds<float, float2><<<nv, kNearThreads, 0, st>>>((const float2 *)X, (const float *)W, np, bb, h);
        near_kernel<float2, false><<<nv, kNearThreads, 0, st>>>((const float2 *)X, nv, np, bb, h, cnt, nullptr, nullptr, 0);
    } else {
        vesicle_bounds<double, double2><<<nv, kNearThreads, 0, st>>>((const double2 *)X, (const double *)W, np, bb, h);
        near_kernel<double2, false><<<nv, kNearThreads, 0, st>>>((const double2 *)X, nv, np, bb, h, cnt, nullptr, nullptr, 0);
    }
    scan_block_sums<<<nb, kScanThreads, 0, st>>>(cnt, P, bsum);
    scan_of_sums<<<1, kScanThreads, 0, st>>>(bsum, nb);
    scan_apply<<<nb, kScanThreads, 0, st>>>(cnt, P, bsum, (long long *)near_ptr, cursor);
    count_launch(5);
    if (fill) {
        if (prec == VN_F32)
            near_kernel<float2, true><<<nv, kNearThreads, 0, st>>>((const float2 *)X, nv, np, bb, h, nullptr, cursor,
                                                                   (int *)near_ves, (long long)capacity);
        else
            near_kernel<double2, true><<<nv, kNearThreads, 0, st>>>((const double2 *)X, nv, np, bb, h, nullptr, cursor,
                                                                    (int *)near_ves, (long long)capacity);
        count_launch(1);
    }
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scratch, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------------
// Correction: one warp per target.  sum = sum_{v' near t} sum_j [ -log|r| g + (r.g)/|r|^2 r ] in double
// (g = F*W formed in the storage precision, exactly as the packing step of the main kernels does),
// lanes stride over j, fixed-order shuffle reduction (deterministic).  `sink` adds -sum to the
// fixed-point accumulators of the pair kernel of that precision.
template <typename real, typename real2, typename Sink>
__global__ void __launch_bounds__(256)
near_correction(const real2 *__restrict__ X, const real2 *__restrict__ F, const real *__restrict__ W, int P,
                int npts, const long long *__restrict__ near_ptr, const int *__restrict__ near_ves, Sink sink)
{
    const int t = blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (t >= P) return;
    const long long k0 = near_ptr[t], k1 = near_ptr[t + 1];
    double sx = 0.0, sy = 0.0;
    if (k1 > k0) {
        const real2 xt = X[t];
        for (long long k = k0; k < k1; ++k) {
            const size_t s0 = (size_t)near_ves[k] * npts;
            for (int j = lane; j < npts; j += 32) {
                const real2 y = X[s0 + j];
                const real2 f = F[s0 + j];
                const real w = W[s0 + j];
                const double gx = (double)(f.x * w), gy = (double)(f.y * w);
                const double rx = (double)xt.x - (double)y.x, ry = (double)xt.y - (double)y.y;
                const double r2 = rx * rx + ry * ry;
                const double ml = -0.5 * log(r2);
                const double q = (rx * gx + ry * gy) / r2;
                sx += ml * gx + q * rx;
                sy += ml * gy + q * ry;
            }
        }
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) {
            sx += __shfl_xor_sync(0xffffffffu, sx, m);
            sy += __shfl_xor_sync(0xffffffffu, sy, m);
        }
    }
    if (lane == 0) sink(t, -sx, -sy);
}

struct SinkFixedF64 {
    long long *acc;
    const unsigned long long *gmax_bits;
    int P;
    __device__ void operator()(int t, double x, double y) const
    {
        if (x == 0.0 && y == 0.0) return;
        const Fixed2 f = fixed2_scale(*gmax_bits, P);
        red_fixed2(acc + 4 * (size_t)t + 0, x, f);
        red_fixed2(acc + 4 * (size_t)t + 2, y, f);
    }
};

struct SinkAccum {      // the fast multipole path: plain double accumulators in original point order, one writer per point
    double2 *accum;
    __device__ void operator()(int t, double x, double y) const
    {
        if (x == 0.0 && y == 0.0) return;
        accum[t] = make_double2(accum[t].x + x, accum[t].y + y);
    }
};

struct SinkFixedF32 {
    long long *acc;
    const unsigned *gmax_bits;
    int P;
    __device__ void operator()(int t, double x, double y) const
    {
        if (x == 0.0 && y == 0.0) return;
        const double scale = fixed_scale(*gmax_bits, P);
        atomicAdd((unsigned long long *)(acc + 2 * (size_t)t + 0), (unsigned long long)__double2ll_rn(x * scale));
        atomicAdd((unsigned long long *)(acc + 2 * (size_t)t + 1), (unsigned long long)__double2ll_rn(y * scale));
    }
};

vn_status near_correction_f64(const void *X, const void *F, const void *W, int P, int npts, const int64_t *near_ptr,
                              const int32_t *near_ves, long long *acc, const unsigned long long *gmax_bits,
                              cudaStream_t st)
{
    near_correction<double, double2, SinkFixedF64><<<(P + 7) / 8, 256, 0, st>>>(
        (const double2 *)X, (const double2 *)F, (const double *)W, P, npts, (const long long *)near_ptr,
        (const int *)near_ves, SinkFixedF64{acc, gmax_bits, P});
    count_launch(1);
    return cudaGetLastError() == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

vn_status near_correction_accum(const void *X, const void *F, const void *W, int P, int npts, const int64_t *near_ptr,
                                const int32_t *near_ves, double2 *accum, vn_precision prec, cudaStream_t st)
{
    if (prec == VN_F32)
        near_correction<float, float2, SinkAccum><<<(P + 7) / 8, 256, 0, st>>>(
            (const float2 *)X, (const float2 *)F, (const float *)W, P, npts, (const long long *)near_ptr,
            (const int *)near_ves, SinkAccum{accum});
    else
        near_correction<double, double2, SinkAccum><<<(P + 7) / 8, 256, 0, st>>>(
            (const double2 *)X, (const double2 *)F, (const double *)W, P, npts, (const long long *)near_ptr,
            (const int *)near_ves, SinkAccum{accum});
    count_launch(1);
    return cudaGetLastError() == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

vn_status near_correction_f32(const void *X, const void *F, const void *W, int P, int npts, const int64_t *near_ptr,
                              const int32_t *near_ves, long long *acc, const unsigned *gmax_bits, cudaStream_t st)
{
    near_correction<float, float2, SinkFixedF32><<<(P + 7) / 8, 256, 0, st>>>(
        (const float2 *)X, (const float2 *)F, (const float *)W, P, npts, (const long long *)near_ptr,
        (const int *)near_ves, SinkFixedF32{acc, gmax_bits, P});
    count_launch(1);
    return cudaGetLastError() == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

}  // namespace vn

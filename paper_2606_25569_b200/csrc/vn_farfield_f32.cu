// vn_farfield_f32.cu -- fp32 far-field Stokeslet sum for sm_100a (steps a-2 .. a-5 of DESIGN.md).
//
//   U_i = 1/(4 pi mu) sum_{j not in ves(i)} [ -log|r| g_j + (r.g_j)/|r|^2 r ],  r = x_i - y_j, g_j = f_j w_j
//   (PAPER.md:129-136 eqs 2.8/2.9, :173 trapezoid rule, :425 DirectSingleLayerIntegral)
//
// Per pair, in the order the inner loop does it (canonical count 2 FADD + 3 FMUL + 6 FFMA + rcp + lg2):
//   r = x - y; r2 = rx*rx + ry*ry; A += lg2(r2) * g; d = rx*gx + ry*gy; B += (d / r2) * r
//   U = 1/(4 pi mu) * ( -(ln 2 / 2) * A + B )
// Two targets share one packed register (FADD2/FMUL2/FFMA2) and one reciprocal:
//   t = rcp(a*b), 1/a = t*b, 1/b = t*a   (a, b = the two r2 of the packed pair; 1.5 SFU ops per pair).
#include "vn_common.cuh"

namespace vn {

// ------------------------------------------------------------------------------------------------
// a-2: g = F*W, packed with the position into one 32-byte record per source, every value
// duplicated so that one LDS.128 yields ready-made packed operands (yx,yx | yy,yy) and (gx,gx | gy,gy).
__global__ void pack_sources_f32(const float2 *__restrict__ X, const float2 *__restrict__ F,
                                 const float *__restrict__ W, int P, ulonglong2 *__restrict__ src)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P) return;
    const float2 y = X[s];
    const float2 f = F[s];
    const float w = W[s];
    const float gx = f.x * w, gy = f.y * w;
    src[2 * (size_t)s + 0] = make_ulonglong2(pk(y.x, y.x), pk(y.y, y.y));
    src[2 * (size_t)s + 1] = make_ulonglong2(pk(gx, gx), pk(gy, gy));
}

// ------------------------------------------------------------------------------------------------
// a-3 / a-4: pair kernel.  Block = (target block, source chunk).  Each thread owns T = 2*NP targets
// (NP packed pairs) in registers; source tiles of kTile points stream through a kStages-deep ring of
// shared-memory buffers filled by 1-D bulk async copies (TMA) that complete on mbarriers.
// A tile that cannot contain points of the block's own vesicles takes the fast path (no predicate
// at all); the few tiles that overlap them, and a ragged last tile, take the predicated slow path.
template <int NP>
__global__ void __launch_bounds__(kThreads, 4)
farfield_f32_kernel(const ulonglong2 *__restrict__ src, const float2 *__restrict__ X, int P, int npts,
                    int n_tiles, int n_chunks, float2 *__restrict__ part)
{
    constexpr int T = 2 * NP;
    __shared__ __align__(128) ulonglong2 tile[kStages][kTile * 2];
    __shared__ __align__(8) u64 full_bar[kStages];
    __shared__ __align__(8) u64 empty_bar[kStages];

    const int tid = threadIdx.x;
    const int tb = blockIdx.x / n_chunks;
    const int sc = blockIdx.x - tb * n_chunks;
    const int t_begin = chunk_tile_begin(n_tiles, n_chunks, sc);
    const int nt = chunk_tile_begin(n_tiles, n_chunks, sc + 1) - t_begin;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], kThreads / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();

    auto issue = [&](int i) {   // one thread: tile i of this chunk -> stage i % kStages
        const int s = i % kStages;
        const int first = (t_begin + i) * kTile;
        const int cnt = min(kTile, P - first);
        const uint32_t bytes = (uint32_t)cnt * 32u;
        mbar_expect_tx(&full_bar[s], bytes);
        bulk_g2s(&tile[s][0], src + 2 * (size_t)first, bytes, &full_bar[s]);
    };
    if (tid == 0) {
        const int pre = nt < kStages ? nt : kStages;
        for (int i = 0; i < pre; ++i) issue(i);
    }

    // targets: packed pair p holds points base + (2p)*kThreads + tid (low half) and
    // base + (2p+1)*kThreads + tid (high half); indices past the end are clamped (never stored).
    const int base = tb * (T * kThreads);
    u64 tx[NP], ty[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const float2 a = X[min(base + (2 * p) * kThreads + tid, P - 1)];
        const float2 b = X[min(base + (2 * p + 1) * kThreads + tid, P - 1)];
        tx[p] = pk(a.x, b.x);
        ty[p] = pk(a.y, b.y);
    }
    // source index range occupied by the vesicles this block's targets belong to
    const int last_target = min(base + T * kThreads, P) - 1;
    const int span_begin = (base / npts) * npts;
    const int span_end = (last_target / npts + 1) * npts;

    u64 Rx[NP], Ry[NP];   // running sums of  -(ln2/2) A + B  over the tiles of this chunk
#pragma unroll
    for (int p = 0; p < NP; ++p) Rx[p] = Ry[p] = 0ull;
    const u64 KA = pk(-0.34657359027997264f, -0.34657359027997264f);   // -(ln 2)/2

    for (int i = 0; i < nt; ++i) {
        const int s = i % kStages;
        if (tid == 0 && i >= 1 && i - 1 + kStages < nt) {   // refill the stage drained last iteration
            mbar_wait(&empty_bar[(i - 1) % kStages], ((i - 1) / kStages) & 1);
            issue(i - 1 + kStages);
        }
        mbar_wait(&full_bar[s], (i / kStages) & 1);

        const int first = (t_begin + i) * kTile;
        const ulonglong2 *ts = tile[s];
        const bool fast = (first >= span_end || first + kTile <= span_begin) && (first + kTile <= P);
        if (fast) {
            u64 Ax[NP], Ay[NP], Bx[NP], By[NP];   // per-tile partial sums (two-level accumulation)
#pragma unroll
            for (int p = 0; p < NP; ++p) Ax[p] = Ay[p] = Bx[p] = By[p] = 0ull;
#pragma unroll 2
            for (int j = 0; j < kTile; ++j) {
                const ulonglong2 yy = ts[2 * j + 0];   // (yx,yx) (yy,yy)
                const ulonglong2 gg = ts[2 * j + 1];   // (gx,gx) (gy,gy)
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    const u64 rx = sub2(tx[p], yy.x);
                    const u64 ry = sub2(ty[p], yy.y);
                    const u64 r2 = fma2(rx, rx, mul2(ry, ry));
                    float a, b;
                    upk(r2, a, b);
                    const float t = sfu_rcp(a * b);
                    const u64 inv = pk(t * b, t * a);
                    const u64 l = pk(sfu_lg2(a), sfu_lg2(b));
                    Ax[p] = fma2(l, gg.x, Ax[p]);
                    Ay[p] = fma2(l, gg.y, Ay[p]);
                    const u64 d = fma2(rx, gg.x, mul2(ry, gg.y));
                    const u64 q = mul2(d, inv);
                    Bx[p] = fma2(q, rx, Bx[p]);
                    By[p] = fma2(q, ry, By[p]);
                }
            }
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                Rx[p] = add2(Rx[p], fma2(KA, Ax[p], Bx[p]));
                Ry[p] = add2(Ry[p], fma2(KA, Ay[p], By[p]));
            }
        } else {
            // predicated path: own-vesicle sources and the ragged tail are skipped per pair
            const int cnt = min(kTile, P - first);
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                float x0, x1, y0, y1;
                upk(tx[p], x0, x1);
                upk(ty[p], y0, y1);
                const int own0 = (min(base + (2 * p) * kThreads + tid, P - 1) / npts) * npts;
                const int own1 = (min(base + (2 * p + 1) * kThreads + tid, P - 1) / npts) * npts;
                float ax0 = 0.f, ay0 = 0.f, bx0 = 0.f, by0 = 0.f, ax1 = 0.f, ay1 = 0.f, bx1 = 0.f, by1 = 0.f;
#pragma unroll 1
                for (int j = 0; j < cnt; ++j) {
                    const ulonglong2 yy = ts[2 * j + 0];
                    const ulonglong2 gg = ts[2 * j + 1];
                    float sx, sy, gx, gy, dum;
                    upk(yy.x, sx, dum);
                    upk(yy.y, sy, dum);
                    upk(gg.x, gx, dum);
                    upk(gg.y, gy, dum);
                    const int jg = first + j;
                    {
                        const float rx = x0 - sx, ry = y0 - sy;
                        const float r2 = fmaf(rx, rx, ry * ry);
                        const float l = sfu_lg2(r2);
                        const float q = fmaf(rx, gx, ry * gy) * sfu_rcp(r2);
                        if ((unsigned)(jg - own0) >= (unsigned)npts) {
                            ax0 = fmaf(l, gx, ax0); ay0 = fmaf(l, gy, ay0);
                            bx0 = fmaf(q, rx, bx0); by0 = fmaf(q, ry, by0);
                        }
                    }
                    {
                        const float rx = x1 - sx, ry = y1 - sy;
                        const float r2 = fmaf(rx, rx, ry * ry);
                        const float l = sfu_lg2(r2);
                        const float q = fmaf(rx, gx, ry * gy) * sfu_rcp(r2);
                        if ((unsigned)(jg - own1) >= (unsigned)npts) {
                            ax1 = fmaf(l, gx, ax1); ay1 = fmaf(l, gy, ay1);
                            bx1 = fmaf(q, rx, bx1); by1 = fmaf(q, ry, by1);
                        }
                    }
                }
                Rx[p] = add2(Rx[p], fma2(KA, pk(ax0, ax1), pk(bx0, bx1)));
                Ry[p] = add2(Ry[p], fma2(KA, pk(ay0, ay1), pk(by0, by1)));
            }
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty_bar[s]);
    }

    // per-chunk partial results; a-5 finishes them
    float2 *out = part + (size_t)sc * (size_t)P;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        float x0, x1, y0, y1;
        upk(Rx[p], x0, x1);
        upk(Ry[p], y0, y1);
        const int i0 = base + (2 * p) * kThreads + tid;
        const int i1 = base + (2 * p + 1) * kThreads + tid;
        if (i0 < P) out[i0] = make_float2(x0, y0);
        if (i1 < P) out[i1] = make_float2(x1, y1);
    }
}

// ------------------------------------------------------------------------------------------------
// a-5: sum the chunk partials in a fixed order (deterministic), scale by 1/(4 pi mu), store U.
__global__ void finish_f32(const float2 *__restrict__ part, int P, int n_chunks, double scale,
                           float2 *__restrict__ U)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P) return;
    double sx = 0.0, sy = 0.0;
    for (int c = 0; c < n_chunks; ++c) {
        const float2 v = part[(size_t)c * (size_t)P + i];
        sx += (double)v.x;
        sy += (double)v.y;
    }
    U[i] = make_float2((float)(scale * sx), (float)(scale * sy));
}

// ------------------------------------------------------------------------------------------------
constexpr int kNP32 = 4;   // 8 targets per thread

vn_status farfield_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                       void *U, cudaStream_t st)
{
    const int P = (int)(nves * npts);
    static int slots = 0;
    if (slots == 0) {
        int dev = 0, sms = 0, occ = 0;
        VN_CUDA(cudaGetDevice(&dev));
        VN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        VN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, farfield_f32_kernel<kNP32>, kThreads, 0));
        slots = sms * (occ > 0 ? occ : 1);
    }
    const Split sp = choose_split(P, 2 * kNP32 * kThreads, slots, 16);

    ulonglong2 *src = nullptr;
    float2 *part = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&src, (size_t)P * 32, st));
    VN_CUDA(cudaMallocAsync((void **)&part, (size_t)P * sizeof(float2) * (size_t)sp.n_chunks, st));

    pack_sources_f32<<<(P + 255) / 256, 256, 0, st>>>((const float2 *)X, (const float2 *)F, (const float *)W, P, src);
    profile_mark(st, true);
    farfield_f32_kernel<kNP32><<<sp.n_tb * sp.n_chunks, kThreads, 0, st>>>(src, (const float2 *)X, P, (int)npts,
                                                                          sp.n_tiles, sp.n_chunks, part);
    profile_mark(st, false);
    finish_f32<<<(P + 255) / 256, 256, 0, st>>>(part, P, sp.n_chunks, 1.0 / (4.0 * 3.14159265358979323846 * mu),
                                                 (float2 *)U);
    count_launch(3);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(src, st));
    VN_CUDA(cudaFreeAsync(part, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

}  // namespace vn

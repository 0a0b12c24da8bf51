// vn_farfield_f32.cu -- fp32 far-field Stokeslet sum for sm_100a (steps a-2 .. a-5 of DESIGN.md).
//
//   U_i = 1/(4 pi mu) sum_{j not in ves(i)} [ -log|r| g_j + (r.g_j)/|r|^2 r ],  r = x_i - y_j, g_j = f_j w_j
//   (PAPER.md:129-136 eqs 2.8/2.9, :173 trapezoid rule, :425 DirectSingleLayerIntegral)
//
// The kernel matrix K(r) = -log|r| I + r r^T/|r|^2 is even in r and symmetric, so the unordered pair
// {i, j} needs r, |r|^2, 1/|r|^2 and log|r|^2 ONCE and serves both U_i += K g_j and U_j += K g_i.
// The kernel walks unordered pairs of point tiles and applies every pair in both directions.  With
// KA = -(ln 2)/2 it builds M' = K / KA once per unordered pair,
//   r = x - y; r2 = rx*rx + ry*ry; inv = 1/(KA r2); l = lg2(r2);  u = r * inv
//   M'xx = l + ux*rx;  M'xy = ux*ry;  M'yy = l + uy*ry                                 (shared)
//   i <- j:  U'_i += M' g_j      j <- i:  U'_j += M' g_i                                (4 FP32 instr each)
//   U = 1/(4 pi mu) * KA * U'
// Two targets share one packed register (FADD2/FMUL2/FFMA2).  Per directed interaction this is 9.0 FP32
// lane-instructions and 1.0 SFU ops (two rcp, two lg2 per packed pair of unordered pairs) against the
// canonical 11 + 2 of a one-directional sum.  Build-time tunables (measured on
// B200): VN_F32_SHARED_RCP=1 lets the two r2 of a packed pair share one reciprocal
// (t = rcp(KA a b), 1/(KA a) = t b: 9.5 lane-instr + 0.75 SFU) -- 5 % slower here because the FMA pipe,
// not the SFU, is the bound; VN_F32_MINBLK (resident blocks per SM: 3 = 168 registers, more ILP, beats
// 4 = 128 registers), VN_F32_BATCH, VN_F32_NP, VN_F32_MINTILES.
//
// Cross-block accumulation goes through 64-bit fixed-point atomics (integer addition is associative, so
// the result is bitwise reproducible whatever the block order); see fixed_scale().
#include <mutex>

#include "vn_common.cuh"

namespace vn {

#ifndef VN_F32_NP
#define VN_F32_NP 4
#endif
constexpr int kNP32 = VN_F32_NP;                  // packed target pairs per thread (8 targets)
constexpr int kST32 = 2 * kNP32 * kThreads;       // points per super-tile (target block): 1024
constexpr int kSub32 = kST32 / kTile;             // source tiles per super-tile: 8
#ifndef VN_F32_BATCH
#define VN_F32_BATCH 8
#endif
#ifndef VN_F32_MINBLK
#define VN_F32_MINBLK 3
#endif
#ifndef VN_F32_MINTILES
#define VN_F32_MINTILES 1
#endif
#ifndef VN_F32_SHARED_RCP
#define VN_F32_SHARED_RCP 0                       // 1: the two r2 of a packed pair share one SFU reciprocal
#endif
constexpr int kBatch = VN_F32_BATCH;              // sources per cross-lane reduction batch
#ifndef VN_F32_RED_UNROLL
#define VN_F32_RED_UNROLL 1                       // batches per scheduling region of the deferred-reduction loop: 3, 5, 15 measured
#endif                                            // -10 %, -27 %, -36 % at 2000 x 128 (13 KB of SASS per batch: instruction cache)
constexpr int kRedUnroll = VN_F32_RED_UNROLL;
#ifndef VN_F32_DIAG_NOMUFU
#define VN_F32_DIAG_NOMUFU 0                      // DIAGNOSTIC builds only (wrong results): bit 0 drops the SFU operations of the
#endif                                            // fast loop, bit 1 its j <- i reduction; measured at 8000 x 128: 3240 / 3133 /
                                                  // 3327 GInt/s for 1 / 2 / 3 against 3079
#ifndef VN_F32_PREFETCH
#define VN_F32_PREFETCH 0                         // 1 (mode 2 only): the first source record of a batch is loaded a batch ahead;
                                                  // measured 3043 against 3079 GInt/s at 8000 x 128: off
#endif
#ifndef VN_F32_SMEMRED
#define VN_F32_SMEMRED 2                          // how the j <- i contributions of a batch are summed over the warp.
#endif                                            // 0: register transpose-reduce (16 shuffles); 1: transposed shared-memory
                                                  // buffer; 2: the same, summed while the NEXT batch is computed; 3: as 2 with
                                                  // the packed pairs parked as they are.  Measured at 8000 x 128 / 2000 x 128 /
                                                  // 256 x 128 (GInt/s): 0: 2942 / 2905 / 2203, 1: 2971 / 2938 / 2233,
                                                  // 2: 3078 / 3046 / 2295, 3: 2987 / 2955 / 2246

// ------------------------------------------------------------------------------------------------
// a-2: g = F*W, packed with the position into one 32-byte record per source, every value
// duplicated so that one LDS.128 yields ready-made packed operands (yx,yx | yy,yy) and (gx,gx | gy,gy).
// Also gmax (bit pattern of a non-negative float orders like the float).
__global__ void pack_sources_f32(const float2 *__restrict__ X, const float2 *__restrict__ F,
                                 const float *__restrict__ W, int P, ulonglong2 *__restrict__ src,
                                 unsigned *__restrict__ gmax_bits)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    float m = 0.f;
    if (s < P) {
        const float2 y = X[s];
        const float2 f = F[s];
        const float w = W[s];
        const float gx = f.x * w, gy = f.y * w;
        src[2 * (size_t)s + 0] = make_ulonglong2(pk(y.x, y.x), pk(y.y, y.y));
        src[2 * (size_t)s + 1] = make_ulonglong2(pk(gx, gx), pk(gy, gy));
        m = fabsf(gx) + fabsf(gy);
        // a non-finite density or position cannot be carried through the integer accumulators point by point:
        // flag it (gmax = +Inf) and finish_f32 answers NaN everywhere
        if (!(m <= 3.4028234e38f) || !(fabsf(y.x) + fabsf(y.y) <= 3.4028234e38f)) m = __int_as_float(0x7f800000);
    }
    const unsigned wm = __reduce_max_sync(0xffffffffu, __float_as_uint(m));
    if ((threadIdx.x & 31) == 0 && wm != 0u) atomicMax(gmax_bits, wm);
}

// ------------------------------------------------------------------------------------------------
// a-3 / a-4: pair kernel.  Points are cut into super-tiles of kST32 = 1024 points.  Block (I, c) owns
// super-tile I as targets (each thread 8 points in 4 packed register pairs, with their densities) and
// walks chunk c of the source-tile list of I:
//   s = 0            the 8 tiles of super-tile I itself: one-directional, own vesicle predicated out;
//   s = 1 .. S_I     the tiles of super-tile (I + s) mod n_st: both directions.
// With S_I = floor((n_st-1)/2) (+1 for I < n_st/2 when n_st is even) every unordered pair of super-tiles
// is visited exactly once and every block has the same amount of work.
// Source tiles of kTile points stream through a kStages-deep ring of shared-memory buffers filled by
// 1-D bulk async copies (TMA) that complete on mbarriers.  A tile that cannot contain points of the
// block's own vesicles takes the fast path (no predicate); tiles that overlap them and a ragged last
// tile take the predicated path.
// CHECK = true (vn_selfcheck): every record read from the ring is compared with its original in global memory and
// mismatches are counted -- a stage refilled while a warp still reads it, or read before its copy has landed, shows
// up as a non-zero count (the tool this replaces, compute-sanitizer's racecheck, is not available on the pool).
template <int NP, bool CHECK>
__global__ void __launch_bounds__(kThreads, VN_F32_MINBLK)
farfield_f32_kernel(const ulonglong2 *__restrict__ src, const float2 *__restrict__ X, int P, int npts,
                    int n_tiles, int n_st, int n_chunks, const unsigned *__restrict__ gmax_bits,
                    long long *__restrict__ acc, int part, int nparts, unsigned long long *__restrict__ mismatches)
{
    constexpr int T = 2 * NP;
    __shared__ __align__(128) ulonglong2 tile[kStages][kTile * 2];
    __shared__ __align__(8) u64 full_bar[kStages];
    __shared__ int drained[kStages];                 // warps that have left each stage (stage_last_out)
#if VN_F32_SMEMRED == 3
    constexpr int kRedRow = 72, kRedHalf = 36;       // 64 floats per row (both halves of every lane's packed pair)
    __shared__ __align__(16) float red[kThreads / 32][2 * kBatch * kRedRow];
#elif VN_F32_SMEMRED
#ifndef VN_F32_REDROW
#define VN_F32_REDROW 40          // row stride and half-row offset in floats.  40 / 20: the 16-byte loads of half rows are
#define VN_F32_REDHALF 20         // conflict-free, the 4-byte stores of lanes 16-19 share banks with lanes 0-3 (2-way, 20 %
#endif                            // of the kernel's shared-memory wavefronts are replays); 36 / 16 is conflict-free for both
                                  // and measured 0.5 % SLOWER (3063 against 3079 GInt/s at 8000 x 128), as was a double-buffered
                                  // variant with one __syncwarp per batch (2991): the kernel's speed follows ptxas's schedule,
                                  // not the shared-memory traffic (8 % of the LSU pipe)
    constexpr int kRedRow = VN_F32_REDROW, kRedHalf = VN_F32_REDHALF;
    __shared__ __align__(16) float red[kThreads / 32][2 * kBatch * kRedRow];
#endif

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int bid = blockIdx.x * nparts + part;      // blocks are dealt round-robin to the parts (one part per GPU)
    const int I = bid / n_chunks;
    const int sc = bid - I * n_chunks;
    int S = (n_st - 1) / 2;
    if ((n_st & 1) == 0 && I < n_st / 2) S += 1;
    const int nu = kSub32 * (S + 1);
    const int u_begin = chunk_tile_begin(nu, n_chunks, sc);
    const int nt = chunk_tile_begin(nu, n_chunks, sc + 1) - u_begin;

    auto tile_of = [&](int u) {        // source tile index of list entry u (may be >= n_tiles: empty)
        const int s = u / kSub32;
        int J = I + s;
        if (J >= n_st) J -= n_st;
        return J * kSub32 + (u - s * kSub32);
    };

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full_bar[s], 1);
            drained[s] = 0;
        }
        mbar_fence_init();
    }
    __syncthreads();

    auto issue = [&](int i) {   // one thread: list entry u_begin + i -> stage i % kStages
        const int s = i % kStages;
        const int first = tile_of(u_begin + i) * kTile;
        const int cnt = min(kTile, P - first);
        if (cnt > 0) {
            const uint32_t bytes = (uint32_t)cnt * 32u;
            mbar_expect_tx(&full_bar[s], bytes);
            bulk_g2s(&tile[s][0], src + 2 * (size_t)first, bytes, &full_bar[s]);
        } else {
            mbar_arrive(&full_bar[s]);      // empty entry: complete the phase without a copy
        }
    };
    if (tid == 0) {
        const int pre = nt < kStages ? nt : kStages;
        for (int i = 0; i < pre; ++i) issue(i);
    }

    const double scale = fixed_scale(*gmax_bits, P);

    // targets: packed pair p holds points base + (2p)*kThreads + tid (low half) and
    // base + (2p+1)*kThreads + tid (high half); indices past the end are clamped to P-1 and carry a
    // zero density (their results are never stored, their contributions to others vanish).
    const int base = I * kST32;
    u64 tx[NP], ty[NP], hx[NP], hy[NP];          // positions and densities g_i of the targets
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const int i0 = base + (2 * p) * kThreads + tid, i1 = i0 + kThreads;
        const int c0 = min(i0, P - 1), c1 = min(i1, P - 1);
        const float2 a = X[c0], b = X[c1];
        tx[p] = pk(a.x, b.x);
        ty[p] = pk(a.y, b.y);
        float g0x, g0y, g1x, g1y, dum;
        const ulonglong2 ga = src[2 * (size_t)c0 + 1], gb = src[2 * (size_t)c1 + 1];
        upk(ga.x, g0x, dum); upk(ga.y, g0y, dum);
        upk(gb.x, g1x, dum); upk(gb.y, g1y, dum);
        if (i0 >= P) g0x = g0y = 0.f;
        if (i1 >= P) g1x = g1y = 0.f;
        hx[p] = pk(g0x, g1x);
        hy[p] = pk(g0y, g1y);
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
        mbar_wait(&full_bar[s], (i / kStages) & 1);

        const int u = u_begin + i;
        const bool both = u >= kSub32;                    // s >= 1: another super-tile, both directions
        const int first = tile_of(u) * kTile;
        const int cnt = min(kTile, P - first);
        const ulonglong2 *ts = tile[s];
        auto verify = [&](int j, const ulonglong2 &yy, const ulonglong2 &gg) {      // CHECK builds only
            const ulonglong2 oy = __ldcg(src + 2 * (size_t)(first + j)), og = __ldcg(src + 2 * (size_t)(first + j) + 1);
            if (oy.x != yy.x || oy.y != yy.y || og.x != gg.x || og.y != gg.y) atomicAdd(mismatches, 1ull);
        };
        const bool fast = both && (first >= span_end || first + kTile <= span_begin) && (cnt == kTile);
        if (fast) {
            // per-tile partial sums (two-level accumulation), in units of -(ln2/2): U' = U / KA
            u64 Ux[NP], Uy[NP];
#pragma unroll
            for (int p = 0; p < NP; ++p) Ux[p] = Uy[p] = 0ull;
            constexpr int kDup = 32 / (2 * kBatch);       // lanes that end a batch with the same warp total
            long long *accj = acc + 2 * (size_t)first + lane / kDup;
            // this thread's contributions c[2 jj], c[2 jj + 1] to the sources jb .. jb + kBatch - 1 (and its own sums Ux, Uy)
#if VN_F32_PREFETCH
            ulonglong2 pre_y = ts[0], pre_g = ts[1];      // the first source of the next batch, loaded a batch ahead
#endif
            auto batch = [&](int jb, u64 (&cp)[2 * kBatch]) {
#pragma unroll
                for (int jj = 0; jj < kBatch; ++jj) {
#if VN_F32_PREFETCH
                    const ulonglong2 yy = jj == 0 ? pre_y : ts[2 * (jb + jj) + 0];
                    const ulonglong2 gg = jj == 0 ? pre_g : ts[2 * (jb + jj) + 1];
#else
                    const ulonglong2 yy = ts[2 * (jb + jj) + 0];   // (yx,yx) (yy,yy)
                    const ulonglong2 gg = ts[2 * (jb + jj) + 1];   // (gx,gx) (gy,gy)
#endif
                    if (CHECK) verify(jb + jj, yy, gg);
                    u64 rx[NP], ry[NP], l[NP], inv[NP];
#pragma unroll
                    for (int p = 0; p < NP; ++p) {
                        rx[p] = sub2(tx[p], yy.x);
                        ry[p] = sub2(ty[p], yy.y);
                        const u64 r2 = fma2(rx[p], rx[p], mul2(ry[p], ry[p]));
                        float a, b;
                        upk(r2, a, b);
#if VN_F32_SHARED_RCP
                        const float t = sfu_rcp((a * b) * -0.34657359027997264f);   // 1/(KA a b)
                        inv[p] = pk(t * b, t * a);                                   // 1/(KA r2)
#else
                        float ka, kb;
                        upk(mul2(r2, KA), ka, kb);
#if VN_F32_DIAG_NOMUFU & 1   // diagnostic build only (wrong results): how fast is the loop without its SFU operations?
                        inv[p] = pk(ka, kb);
#else
                        inv[p] = pk(sfu_rcp(ka), sfu_rcp(kb));                       // 1/(KA r2)
#endif
#endif
#if VN_F32_DIAG_NOMUFU & 1
                        l[p] = r2;
#else
                        l[p] = pk(sfu_lg2(a), sfu_lg2(b));
#endif
                    }
                    u64 cUx = 0ull, cUy = 0ull;
#pragma unroll
                    for (int p = 0; p < NP; ++p) {
                        // M' = K / KA = lg2(r2) I + r r^T / (KA r2)
                        const u64 ux = mul2(rx[p], inv[p]);
                        const u64 uy = mul2(ry[p], inv[p]);
                        const u64 Mxy = mul2(ux, ry[p]);
                        const u64 Mxx = fma2(ux, rx[p], l[p]);
                        const u64 Myy = fma2(uy, ry[p], l[p]);
                        // one chain through all eight products: neighbours share an operand slot
                        Ux[p] = fma2(Mxx, gg.x, Ux[p]);
                        cUx = fma2(Mxx, hx[p], cUx);
                        cUy = fma2(Mxy, hx[p], cUy);
                        cUx = fma2(Mxy, hy[p], cUx);
                        cUy = fma2(Myy, hy[p], cUy);
                        Uy[p] = fma2(Myy, gg.y, Uy[p]);
                        Ux[p] = fma2(Mxy, gg.y, Ux[p]);
                        Uy[p] = fma2(Mxy, gg.x, Uy[p]);
                    }
                    cp[2 * jj + 0] = cUx;       // both targets of the packed pair still side by side
                    cp[2 * jj + 1] = cUy;
                }
            };
            auto fold = [&](const u64 (&cp)[2 * kBatch], float (&c)[2 * kBatch]) {
#pragma unroll
                for (int v = 0; v < 2 * kBatch; ++v) {
                    float lo, hi;
                    upk(cp[v], lo, hi);
                    c[v] = lo + hi;
                }
            };
#if VN_F32_SMEMRED == 3
            // As mode 2, but the packed pairs are parked as they are (STS.64): the lo + hi additions move out of the
            // batch's arithmetic into the deferred sum (32 floats per lane instead of 16).
            static_assert(kDup == 2, "shared-memory reduction assumes 16 values per batch");
            float *rw = red[tid >> 5];
            const int col = 2 * lane + (lane >= 16 ? kRedHalf - 32 : 0);
            const float4 *row = reinterpret_cast<const float4 *>(rw + (lane >> 1) * kRedRow + (lane & 1) * kRedHalf);
            auto park = [&](const u64 (&cp)[2 * kBatch]) {
                __syncwarp();                                       // every lane has read the previous batch's rows
#pragma unroll
                for (int v = 0; v < 2 * kBatch; ++v) *reinterpret_cast<u64 *>(rw + v * kRedRow + col) = cp[v];
            };
            auto sum4 = [](const float4 &q) { return (q.x + q.y) + (q.z + q.w); };
            auto total = [&](const float4 (&q)[8]) {
                float t = ((sum4(q[0]) + sum4(q[1])) + (sum4(q[2]) + sum4(q[3]))) +
                          ((sum4(q[4]) + sum4(q[5])) + (sum4(q[6]) + sum4(q[7])));
                t += __shfl_xor_sync(0xffffffffu, t, 1);
                return t;
            };
            {
                u64 cp[2 * kBatch];
                batch(0, cp);
                park(cp);
            }
#pragma unroll kRedUnroll
            for (int jb = kBatch; jb < kTile; jb += kBatch) {
                __syncwarp();                                       // the parked rows are complete
                float4 q[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) q[e] = row[e];
                u64 cp[2 * kBatch];
                batch(jb, cp);
                const float t = total(q);
                if (lane % kDup == 0) red_fixed(accj + 2 * (jb - kBatch), t * -0.34657359027997264f, scale);
                park(cp);
            }
            {
                __syncwarp();
                float4 q[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) q[e] = row[e];
                const float t = total(q);
                if (lane % kDup == 0) red_fixed(accj + 2 * (kTile - kBatch), t * -0.34657359027997264f, scale);
            }
#elif VN_F32_SMEMRED == 2
            // The c values of a batch are parked in a transposed shared-memory buffer and summed over the warp
            // while the NEXT batch is computed: the loads are issued before that batch's arithmetic and nothing
            // of it depends on them, so the reduction's latency chain hides behind 576 packed instructions
            // instead of ending every batch.
            static_assert(kDup == 2, "shared-memory reduction assumes 16 values per batch");
            float *rw = red[tid >> 5];
            const int col = lane + (lane >= 16 ? kRedHalf - 16 : 0);
            const float4 *row = reinterpret_cast<const float4 *>(rw + (lane >> 1) * kRedRow + (lane & 1) * kRedHalf);
            auto park = [&](const float (&c)[2 * kBatch]) {
                __syncwarp();                                       // every lane has read the previous batch's rows
#pragma unroll
                for (int v = 0; v < 2 * kBatch; ++v) rw[v * kRedRow + col] = c[v];
            };
            auto total = [&](const float4 &q0, const float4 &q1, const float4 &q2, const float4 &q3) {
                float t = ((q0.x + q0.y) + (q0.z + q0.w)) + ((q1.x + q1.y) + (q1.z + q1.w)) +
                          (((q2.x + q2.y) + (q2.z + q2.w)) + ((q3.x + q3.y) + (q3.z + q3.w)));
                t += __shfl_xor_sync(0xffffffffu, t, 1);
                return t;
            };
            {
                u64 cp[2 * kBatch];
                float c[2 * kBatch];
                batch(0, cp);
#if VN_F32_PREFETCH
                pre_y = ts[2 * kBatch + 0];
                pre_g = ts[2 * kBatch + 1];
#endif
                fold(cp, c);
                park(c);
            }
#pragma unroll kRedUnroll
            for (int jb = kBatch; jb < kTile; jb += kBatch) {
                __syncwarp();                                       // the parked rows are complete
                const float4 q0 = row[0], q1 = row[1], q2 = row[2], q3 = row[3];
                u64 cp[2 * kBatch];
                float c[2 * kBatch];
                batch(jb, cp);
#if VN_F32_PREFETCH
                {
                    const int jn = min(jb + kBatch, kTile - 1);     // (the last batch of a tile prefetches a record it will not use)
                    pre_y = ts[2 * jn + 0];
                    pre_g = ts[2 * jn + 1];
                }
#endif
#if VN_F32_DIAG_NOMUFU & 2       // diagnostic build only (wrong results): the loop without the j <- i reduction
#pragma unroll
                for (int v = 0; v < 2 * kBatch; ++v) Ux[v % NP] = add2(Ux[v % NP], cp[v]);
                (void)q0; (void)q1; (void)q2; (void)q3; (void)c;
#else
                fold(cp, c);
                const float t = total(q0, q1, q2, q3);
                if (lane % kDup == 0) red_fixed(accj + 2 * (jb - kBatch), t * -0.34657359027997264f, scale);
                park(c);
#endif
            }
            {
                __syncwarp();
                const float4 q0 = row[0], q1 = row[1], q2 = row[2], q3 = row[3];
                const float t = total(q0, q1, q2, q3);
                if (lane % kDup == 0) red_fixed(accj + 2 * (kTile - kBatch), t * -0.34657359027997264f, scale);
            }
#else
#pragma unroll 1
            for (int jb = 0; jb < kTile; jb += kBatch) {
                u64 cp[2 * kBatch];
                float c[2 * kBatch];              // this thread's contributions to the batch's sources
                batch(jb, cp);
                fold(cp, c);
#if VN_F32_SMEMRED == 1
                static_assert(kDup == 2, "shared-memory reduction assumes 16 values per batch");
                {
                    float *rw = red[tid >> 5];
                    const int col = lane + (lane >= 16 ? kRedHalf - 16 : 0);
                    __syncwarp();                                   // the previous batch's reads are done
#pragma unroll
                    for (int v = 0; v < 2 * kBatch; ++v) rw[v * kRedRow + col] = c[v];
                    __syncwarp();
                    const float4 *row = reinterpret_cast<const float4 *>(rw + (lane >> 1) * kRedRow + (lane & 1) * kRedHalf);
                    const float4 q0 = row[0], q1 = row[1], q2 = row[2], q3 = row[3];
                    c[0] = ((q0.x + q0.y) + (q0.z + q0.w)) + ((q1.x + q1.y) + (q1.z + q1.w)) +
                           (((q2.x + q2.y) + (q2.z + q2.w)) + ((q3.x + q3.y) + (q3.z + q3.w)));
                    c[0] += __shfl_xor_sync(0xffffffffu, c[0], 1);
                }
#else
                // transpose-reduce over the warp: 16 values per lane -> lane L ends with the warp
                // total of value L / kDup; 16 shuffles instead of 16 x 5 at kBatch = 8.
                int m = 16;
#pragma unroll
                for (int w = kBatch; w >= 1; w >>= 1, m >>= 1) {
                    const bool up = (lane & m) != 0;
#pragma unroll
                    for (int k = 0; k < w; ++k) {
                        const float send = up ? c[k] : c[k + w];
                        const float keep = up ? c[k + w] : c[k];
                        c[k] = keep + __shfl_xor_sync(0xffffffffu, send, m);
                    }
                }
#pragma unroll
                for (; m >= 1; m >>= 1) c[0] += __shfl_xor_sync(0xffffffffu, c[0], m);
#endif
                if (lane % kDup == 0) red_fixed(accj + 2 * jb, c[0] * -0.34657359027997264f, scale);
            }
#endif
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                Rx[p] = fma2(KA, Ux[p], Rx[p]);
                Ry[p] = fma2(KA, Uy[p], Ry[p]);
            }
        } else if (!both && cnt == kTile && npts % kTile == 0 && base + kST32 <= P) {
            // a tile of the block's OWN super-tile when vesicles are whole tiles (npts a multiple of 128, the
            // paper's N = 128): target k of a thread lies in tile k of the super-tile, so its own vesicle is
            // excluded for ALL lanes alike.  One-directional, unpredicated, packed; the excluded halves (which
            // also hold the r = 0 self pairs) are discarded after the tile.
            u64 Ux[NP], Uy[NP];
#pragma unroll
            for (int p = 0; p < NP; ++p) Ux[p] = Uy[p] = 0ull;
#pragma unroll 2
            for (int j = 0; j < kTile; ++j) {
                const ulonglong2 yy = ts[2 * j + 0];
                const ulonglong2 gg = ts[2 * j + 1];
                if (CHECK) verify(j, yy, gg);
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    const u64 rx = sub2(tx[p], yy.x);
                    const u64 ry = sub2(ty[p], yy.y);
                    const u64 r2 = fma2(rx, rx, mul2(ry, ry));
                    float a, b, ka, kb;
                    upk(r2, a, b);
                    upk(mul2(r2, KA), ka, kb);
                    const u64 inv = pk(sfu_rcp(ka), sfu_rcp(kb));
                    const u64 l = pk(sfu_lg2(a), sfu_lg2(b));
                    const u64 ux = mul2(rx, inv);
                    const u64 uy = mul2(ry, inv);
                    const u64 Mxy = mul2(ux, ry);
                    const u64 Mxx = fma2(ux, rx, l);
                    const u64 Myy = fma2(uy, ry, l);
                    Ux[p] = fma2(Mxx, gg.x, fma2(Mxy, gg.y, Ux[p]));
                    Uy[p] = fma2(Mxy, gg.x, fma2(Myy, gg.y, Uy[p]));
                }
            }
            const int vs_src = first / npts;
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                float x0, x1, y0, y1;
                upk(Ux[p], x0, x1);
                upk(Uy[p], y0, y1);
                if ((base + (2 * p) * kThreads) / npts == vs_src) x0 = y0 = 0.f;
                if ((base + (2 * p + 1) * kThreads) / npts == vs_src) x1 = y1 = 0.f;
                Rx[p] = fma2(KA, pk(x0, x1), Rx[p]);
                Ry[p] = fma2(KA, pk(y0, y1), Ry[p]);
            }
        } else if (cnt > 0) {
            // predicated path: own-vesicle sources and the ragged tail are skipped per pair
            float ux[T], uy[T];
            int own[T];
#pragma unroll
            for (int k = 0; k < T; ++k) {
                ux[k] = uy[k] = 0.f;
                own[k] = (min(base + k * kThreads + tid, P - 1) / npts) * npts;
            }
#pragma unroll 1
            for (int j = 0; j < cnt; ++j) {
                const ulonglong2 yy = ts[2 * j + 0];
                const ulonglong2 gg = ts[2 * j + 1];
                if (CHECK) verify(j, yy, gg);
                float sx, sy, gx, gy, dum;
                upk(yy.x, sx, dum);
                upk(yy.y, sy, dum);
                upk(gg.x, gx, dum);
                upk(gg.y, gy, dum);
                const int jg = first + j;
                float cx = 0.f, cy = 0.f;
#pragma unroll
                for (int k = 0; k < T; ++k) {
                    float x0, x1, y0, y1, h0x, h1x, h0y, h1y;
                    upk(tx[k >> 1], x0, x1);
                    upk(ty[k >> 1], y0, y1);
                    upk(hx[k >> 1], h0x, h1x);
                    upk(hy[k >> 1], h0y, h1y);
                    const float xk = (k & 1) ? x1 : x0, yk = (k & 1) ? y1 : y0;
                    const float hkx = (k & 1) ? h1x : h0x, hky = (k & 1) ? h1y : h0y;
                    if ((unsigned)(jg - own[k]) >= (unsigned)npts) {
                        const float rx = xk - sx, ry = yk - sy;
                        const float r2 = fmaf(rx, rx, ry * ry);
                        const float l = -0.34657359027997264f * sfu_lg2(r2);
                        const float inv = sfu_rcp(r2);
                        const float q = fmaf(rx, gx, ry * gy) * inv;
                        ux[k] += fmaf(l, gx, q * rx);
                        uy[k] += fmaf(l, gy, q * ry);
                        const float w = fmaf(rx, hkx, ry * hky) * inv;
                        cx += fmaf(l, hkx, w * rx);
                        cy += fmaf(l, hky, w * ry);
                    }
                }
                if (both) {
#pragma unroll
                    for (int m = 16; m >= 1; m >>= 1) {
                        cx += __shfl_xor_sync(0xffffffffu, cx, m);
                        cy += __shfl_xor_sync(0xffffffffu, cy, m);
                    }
                    if (lane == 0) {
                        red_fixed(acc + 2 * (size_t)jg + 0, cx, scale);
                        red_fixed(acc + 2 * (size_t)jg + 1, cy, scale);
                    }
                }
            }
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                Rx[p] = add2(Rx[p], pk(ux[2 * p], ux[2 * p + 1]));
                Ry[p] = add2(Ry[p], pk(uy[2 * p], uy[2 * p + 1]));
            }
        }
        __syncwarp();
        if (lane == 0 && stage_last_out(&drained[s], kThreads / 32) && i + kStages < nt)
            issue(i + kStages);                      // the last warp out of the stage refills it
    }

    // this block's one-directional sums for its own targets
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        float x0, x1, y0, y1;
        upk(Rx[p], x0, x1);
        upk(Ry[p], y0, y1);
        const int i0 = base + (2 * p) * kThreads + tid;
        const int i1 = i0 + kThreads;
        if (i0 < P) {
            red_fixed(acc + 2 * (size_t)i0 + 0, x0, scale);
            red_fixed(acc + 2 * (size_t)i0 + 1, y0, scale);
        }
        if (i1 < P) {
            red_fixed(acc + 2 * (size_t)i1 + 0, x1, scale);
            red_fixed(acc + 2 * (size_t)i1 + 1, y1, scale);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a-5: fixed point -> float, scale by 1/(4 pi mu), store U.
__global__ void finish_f32(const long long *__restrict__ acc, int n, int P, const unsigned *__restrict__ gmax_bits,
                           double prefactor, float2 *__restrict__ U)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (*gmax_bits == 0x7f800000u) {                      // non-finite input somewhere: see pack_sources_f32
        U[i] = make_float2(__int_as_float(0x7fc00000), __int_as_float(0x7fc00000));
        return;
    }
    const double f = prefactor / fixed_scale(*gmax_bits, P);
    const longlong2 v = *reinterpret_cast<const longlong2 *>(acc + 2 * (size_t)i);
    U[i] = make_float2((float)(f * (double)v.x), (float)(f * (double)v.y));
}

// ------------------------------------------------------------------------------------------------
// pack + pair kernel for the blocks of one part: acc (P x 2 words) and gmax are the caller's, already zeroed
static vn_status accumulate_f32(const void *X, const void *F, const void *W, int P, int npts, int part, int nparts,
                                ulonglong2 *src, long long *acc, unsigned *gmax, cudaStream_t st,
                                unsigned long long *mismatches = nullptr)
{
    static int slots_dev[kMaxDevices] = {0};
    int &slots = slots_dev[current_device()];
    if (slots == 0) {
        int dev = 0, sms = 0, occ = 0;
        VN_CUDA(cudaGetDevice(&dev));
        VN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        VN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, farfield_f32_kernel<kNP32, false>, kThreads, 0));
        slots = sms * (occ > 0 ? occ : 1);
    }
    // the grid is the single-device grid whatever nparts is: the blocks' own roundings are then the same and the
    // summed accumulators bit for bit those of vn_farfield (the chunk length tuned for one device costs 0.3 % on 8)
    const SymSplit sp = choose_sym_split(P, kST32, slots, VN_F32_MINTILES, 0);
    const long long blocks = (long long)sp.n_st * sp.n_chunks;
    const int mine = (int)((blocks - part + nparts - 1) / nparts);
    pack_sources_f32<<<(P + 255) / 256, 256, 0, st>>>((const float2 *)X, (const float2 *)F, (const float *)W, P, src, gmax);
    profile_mark(st, true);
    if (mine > 0 && !mismatches)
        farfield_f32_kernel<kNP32, false><<<mine, kThreads, 0, st>>>(src, (const float2 *)X, P, npts, sp.n_tiles, sp.n_st,
                                                                     sp.n_chunks, gmax, acc, part, nparts, nullptr);
    else if (mine > 0)
        farfield_f32_kernel<kNP32, true><<<mine, kThreads, 0, st>>>(src, (const float2 *)X, P, npts, sp.n_tiles, sp.n_st,
                                                                    sp.n_chunks, gmax, acc, part, nparts, mismatches);
    profile_mark(st, false);
    count_launch(mine > 0 ? 2 : 1);
    return VN_OK;
}

vn_status farfield_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                       void *U, cudaStream_t st, const int64_t *near_ptr, const int32_t *near_ves)
{
    const int P = (int)(nves * npts);
    // scratch: packed sources | fixed-point accumulators | gmax
    const size_t b_src = (size_t)P * 32, b_acc = (size_t)P * 16;
    char *scratch = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scratch, b_src + b_acc + 16, st));
    ulonglong2 *src = (ulonglong2 *)scratch;
    long long *acc = (long long *)(scratch + b_src);
    unsigned *gmax = (unsigned *)(scratch + b_src + b_acc);
    VN_CUDA(cudaMemsetAsync(acc, 0, b_acc + 16, st));
    vn_status rc = accumulate_f32(X, F, W, P, (int)npts, 0, 1, src, acc, gmax, st);
    if (rc == VN_OK && near_ptr)   // row f-1: take the near vesicles' contributions out again before the final rounding
        rc = near_correction_f32(X, F, W, P, (int)npts, near_ptr, near_ves, acc, gmax, st);
    if (rc != VN_OK) { (void)cudaFreeAsync(scratch, st); return rc; }
    finish_f32<<<(P + 255) / 256, 256, 0, st>>>(acc, P, P, gmax, 1.0 / (4.0 * 3.14159265358979323846 * mu), (float2 *)U);
    count_launch(1);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scratch, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// vn_selfcheck: the general path with poisoned scratch (every byte 0xFF before use: a read of scratch that nothing
// wrote shows up in the result) and the ring verification of the CHECK kernel; *mismatches (device) is incremented.
vn_status farfield_selfcheck_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                                 void *U, unsigned long long *mismatches, cudaStream_t st)
{
    const int P = (int)(nves * npts);
    const size_t b_src = (size_t)P * 32, b_acc = (size_t)P * 16;
    char *scratch = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scratch, b_src + b_acc + 16, st));
    VN_CUDA(cudaMemsetAsync(scratch, 0xFF, b_src + b_acc + 16, st));
    ulonglong2 *src = (ulonglong2 *)scratch;
    long long *acc = (long long *)(scratch + b_src);
    unsigned *gmax = (unsigned *)(scratch + b_src + b_acc);
    VN_CUDA(cudaMemsetAsync(acc, 0, b_acc + 16, st));
    const vn_status rc = accumulate_f32(X, F, W, P, (int)npts, 0, 1, src, acc, gmax, st, mismatches);
    if (rc != VN_OK) { (void)cudaFreeAsync(scratch, st); return rc; }
    finish_f32<<<(P + 255) / 256, 256, 0, st>>>(acc, P, P, gmax, 1.0 / (4.0 * 3.14159265358979323846 * mu), (float2 *)U);
    count_launch(1);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scratch, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// Section 8e building blocks: the accumulators of the blocks of part `part` of `nparts` (all sources known to the
// caller), and the final step on any contiguous range of (summed) accumulators.
vn_status farfield_partial_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, int part,
                               int nparts, void *acc, void *gmax, cudaStream_t st)
{
    const int P = (int)(nves * npts);
    ulonglong2 *src = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&src, (size_t)P * 32, st));
    VN_CUDA(cudaMemsetAsync(acc, 0, (size_t)P * 16, st));
    VN_CUDA(cudaMemsetAsync(gmax, 0, 8, st));
    const vn_status rc = accumulate_f32(X, F, W, P, (int)npts, part, nparts, src, (long long *)acc, (unsigned *)gmax, st);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(src, st));
    return rc != VN_OK ? rc : (e == cudaSuccess ? VN_OK : VN_ERR_CUDA);
}

vn_status farfield_finish_f32(const void *acc, const void *gmax, int64_t P_total, int64_t count, double mu, void *U,
                              cudaStream_t st)
{
    finish_f32<<<(int)((count + 255) / 256), 256, 0, st>>>((const long long *)acc, (int)count, (int)P_total,
                                                           (const unsigned *)gmax,
                                                           1.0 / (4.0 * 3.14159265358979323846 * mu), (float2 *)U);
    count_launch(1);
    return cudaGetLastError() == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------------
// vn_farfield_noalloc_f32: the general fp32 path (pack, symmetric pair kernel, finish -- the same kernels, the same
// grid, hence bit for bit the same U as farfield_f32) for callers that may not allocate: code under stream capture,
// tight serving loops, harnesses that forbid cudaMalloc.  farfield_f32 takes 48 bytes of scratch per point from the
// stream-ordered allocator; here the scratch is the static device array below, 12 MiB + 256 B that EVERY device
// which loads the library holds until the process exits -- which is why the limit is modest: kStaticMaxPoints =
// 262,144 points (BASELINE.json configs[0..3]; configs[4], 1.02 M points, needs 47 MiB and stays with vn_farfield).
//   layout:  [0, 32 maxP)  packed sources (ulonglong2 pairs, written by pack_sources_f32 before anything reads them)
//            [32 maxP, 32 maxP + 16 P)  fixed-point accumulators, then 16 bytes holding gmax: cleared by every call
// All calls on a device share the array and it keeps the last call's contents; two calls whose kernels overlap on the
// GPU (different streams, or graphs replayed concurrently) race on it.  Calls on one stream are ordered and safe.
// In host code the array's name is a host-side stand-in, not a device address: the address is asked for once per
// device, with that device current, by cudaGetSymbolAddress, and only that pointer is handed to the kernels.
constexpr int kStaticMaxPoints = 1 << 18;
constexpr size_t kStaticSrcBytes = (size_t)kStaticMaxPoints * 32;
constexpr size_t kStaticAccBytes = (size_t)kStaticMaxPoints * 16;
constexpr size_t kStaticScratchBytes = kStaticSrcBytes + kStaticAccBytes + 256;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

int64_t farfield_static_max_points() { return kStaticMaxPoints; }

// device address of g_static_scratch on the CURRENT device (cached per device ordinal)
static vn_status static_scratch_base(unsigned char **base)
{
    static std::mutex lock;
    static unsigned char *base_dev[kMaxDevices] = {nullptr};
    int dev = -1;
    VN_CUDA(cudaGetDevice(&dev));
    const bool cached = dev >= 0 && dev < kMaxDevices;
    std::lock_guard<std::mutex> guard(lock);
    if (cached && base_dev[dev]) {
        *base = base_dev[dev];
        return VN_OK;
    }
    void *p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p) {
        (void)cudaGetLastError();
        return VN_ERR_CUDA;
    }
    if (cached) base_dev[dev] = (unsigned char *)p;
    *base = (unsigned char *)p;
    return VN_OK;
}

vn_status farfield_static_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                              void *U, cudaStream_t st)
{
    if (nves * npts > (int64_t)kStaticMaxPoints) return VN_ERR_TOO_LARGE;
    const int P = (int)(nves * npts);
    unsigned char *base = nullptr;
    const vn_status rb = static_scratch_base(&base);
    if (rb != VN_OK) return rb;
    ulonglong2 *src = (ulonglong2 *)base;
    long long *acc = (long long *)(base + kStaticSrcBytes);
    unsigned *gmax = (unsigned *)(base + kStaticSrcBytes + (size_t)P * 16);
    VN_CUDA(cudaMemsetAsync(acc, 0, (size_t)P * 16 + 16, st));      // what must start at zero: accumulators, gmax
    const vn_status rc = accumulate_f32(X, F, W, P, (int)npts, 0, 1, src, acc, gmax, st);
    if (rc != VN_OK) return rc;
    finish_f32<<<(P + 255) / 256, 256, 0, st>>>(acc, P, P, gmax, 1.0 / (4.0 * 3.14159265358979323846 * mu), (float2 *)U);
    count_launch(1);
    return cudaGetLastError() == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------------
// Row f-4: free targets.  Velocity induced at nt points that lie on no membrane by ALL vesicles
// (eq 2.8 summed over every vesicle, trapezoid rule; the velocity-field
// evaluation behind the streamline plots).  Targets and sources are different sets, so
// there is no symmetry to use: one-directional sum, per pair
//   r = x - y; r2 = rx*rx + ry*ry; A += lg2(r2) * g; d = rx*gx + ry*gy; B += (d / r2) * r
// (2 FADD + 3 FMUL + 6 FFMA + 1.5 MUFU with the shared reciprocal), 8 targets per thread as packed
// pairs, the same tile ring, per-tile partial sums folded into running sums, fixed-point atomics out.
#ifndef VN_TGT32_LASTOUT
#define VN_TGT32_LASTOUT 0         // 1: stage hand-back by the last warp out as in the pair kernel; measured
#endif                             // 2008 against 2178 GInt/s at 2000 x 128 sources, 512 x 512 targets: off
#ifndef VN_TGT32_LOCAL_FIX
#define VN_TGT32_LOCAL_FIX 1       // a bad distance spoils its own target only (one check per tile, see the kernel)
#endif
#ifndef VN_F32_TGT_MINBLK
#define VN_F32_TGT_MINBLK 3       // measured at 2000 x 128 sources, 512 x 512 targets: 2245 GInt/s against 2229 with 4
#endif
template <int NP>
__global__ void __launch_bounds__(kThreads, VN_F32_TGT_MINBLK)
targets_f32_kernel(const ulonglong2 *__restrict__ src, const float2 *__restrict__ Xt, int nt_pts, int P,
                   int n_tiles, int n_chunks, const unsigned *__restrict__ gmax_bits, long long *__restrict__ acc)
{
    constexpr int T = 2 * NP;
    __shared__ __align__(128) ulonglong2 tile[kStages][kTile * 2];
    __shared__ __align__(8) u64 full_bar[kStages];
#if VN_TGT32_LASTOUT
    __shared__ int drained[kStages];                 // warps that have left each stage (stage_last_out)
#else
    __shared__ __align__(8) u64 empty_bar[kStages];
#endif

    const int tid = threadIdx.x;
    const int tb = blockIdx.x / n_chunks;
    const int sc = blockIdx.x - tb * n_chunks;
    const int t_begin = chunk_tile_begin(n_tiles, n_chunks, sc);
    const int nt = chunk_tile_begin(n_tiles, n_chunks, sc + 1) - t_begin;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full_bar[s], 1);
#if VN_TGT32_LASTOUT
            drained[s] = 0;
#else
            mbar_init(&empty_bar[s], kThreads / 32);
#endif
        }
        mbar_fence_init();
    }
    __syncthreads();

    auto issue = [&](int i) {
        const int s = i % kStages;
        const int first = (t_begin + i) * kTile;
        const uint32_t bytes = (uint32_t)min(kTile, P - first) * 32u;
        mbar_expect_tx(&full_bar[s], bytes);
        bulk_g2s(&tile[s][0], src + 2 * (size_t)first, bytes, &full_bar[s]);
    };
    if (tid == 0) {
        const int pre = nt < kStages ? nt : kStages;
        for (int i = 0; i < pre; ++i) issue(i);
    }

    const int base = tb * (T * kThreads);
    u64 tx[NP], ty[NP], Rx[NP], Ry[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const float2 a = Xt[min(base + (2 * p) * kThreads + tid, nt_pts - 1)];
        const float2 b = Xt[min(base + (2 * p + 1) * kThreads + tid, nt_pts - 1)];
        tx[p] = pk(a.x, b.x);
        ty[p] = pk(a.y, b.y);
        Rx[p] = Ry[p] = 0ull;
    }
    const u64 KA = pk(-0.34657359027997264f, -0.34657359027997264f);   // -(ln 2)/2

    for (int i = 0; i < nt; ++i) {
        const int s = i % kStages;
#if !VN_TGT32_LASTOUT
        if (tid == 0 && i >= 1 && i - 1 + kStages < nt) {
            mbar_wait(&empty_bar[(i - 1) % kStages], ((i - 1) / kStages) & 1);
            issue(i - 1 + kStages);
        }
#endif
        mbar_wait(&full_bar[s], (i / kStages) & 1);

        const int cnt = min(kTile, P - (t_begin + i) * kTile);
        const ulonglong2 *ts = tile[s];
        u64 Ax[NP], Ay[NP], Bx[NP], By[NP];   // per-tile partial sums (two-level accumulation)
#pragma unroll
        for (int p = 0; p < NP; ++p) Ax[p] = Ay[p] = Bx[p] = By[p] = 0ull;
        auto pair = [&](int j) {
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
                const u64 inv = mul2(pk(t, t), pk(b, a));   // (1/a, 1/b): one packed multiply on the swapped pair
                                                            // (the swap is register allocation, no instruction)
                const u64 l = pk(sfu_lg2(a), sfu_lg2(b));
                Ax[p] = fma2(l, gg.x, Ax[p]);
                Ay[p] = fma2(l, gg.y, Ay[p]);
                const u64 d = fma2(rx, gg.x, mul2(ry, gg.y));
                const u64 q = mul2(d, inv);
                Bx[p] = fma2(q, rx, Bx[p]);
                By[p] = fma2(q, ry, By[p]);
            }
        };
        if (cnt == kTile) {
#pragma unroll 2
            for (int j = 0; j < kTile; ++j) pair(j);
        } else {
#pragma unroll 1
            for (int j = 0; j < cnt; ++j) pair(j);
        }
#if VN_TGT32_LOCAL_FIX
        {   // The shared reciprocal t = rcp(a b) turns into Inf or 0 when a*b leaves the fp32 normal range (a target on
            // top of a source, |r| beyond 1e-9 .. 1e9) and then spoils BOTH targets of the packed pair.  One sum over
            // the tile's partial sums detects it (NaN / Inf is sticky); the warp then redoes this tile with one
            // reciprocal per pair, so that only the target that owns the bad distance keeps a non-finite value.
            u64 chk = add2(add2(Ax[0], Ay[0]), add2(Bx[0], By[0]));
#pragma unroll
            for (int p = 1; p < NP; ++p) chk = add2(chk, add2(add2(Ax[p], Ay[p]), add2(Bx[p], By[p])));
            float c0, c1;
            upk(chk, c0, c1);
            if (__any_sync(0xffffffffu, !(fabsf(c0 + c1) <= 3.4028234e38f))) {
#pragma unroll
                for (int p = 0; p < NP; ++p) {        // unrolled: a dynamic index would move the arrays to local memory
                    float x0, x1, y0, y1;
                    upk(tx[p], x0, x1);
                    upk(ty[p], y0, y1);
                    float a[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};      // (Ax, Ay, Bx, By) of the two targets
#pragma unroll 1
                    for (int j = 0; j < cnt; ++j) {
                        float sx, sy, gx, gy, dum;
                        upk(ts[2 * j + 0].x, sx, dum);
                        upk(ts[2 * j + 0].y, sy, dum);
                        upk(ts[2 * j + 1].x, gx, dum);
                        upk(ts[2 * j + 1].y, gy, dum);
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const float rx = (h ? x1 : x0) - sx, ry = (h ? y1 : y0) - sy;
                            const float r2 = fmaf(rx, rx, ry * ry);
                            const float l = sfu_lg2(r2);
                            const float q = fmaf(rx, gx, ry * gy) * sfu_rcp(r2);
                            a[h][0] = fmaf(l, gx, a[h][0]);
                            a[h][1] = fmaf(l, gy, a[h][1]);
                            a[h][2] = fmaf(q, rx, a[h][2]);
                            a[h][3] = fmaf(q, ry, a[h][3]);
                        }
                    }
                    Ax[p] = pk(a[0][0], a[1][0]);
                    Ay[p] = pk(a[0][1], a[1][1]);
                    Bx[p] = pk(a[0][2], a[1][2]);
                    By[p] = pk(a[0][3], a[1][3]);
                }
            }
        }
#endif
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            Rx[p] = add2(Rx[p], fma2(KA, Ax[p], Bx[p]));
            Ry[p] = add2(Ry[p], fma2(KA, Ay[p], By[p]));
        }
        __syncwarp();
#if VN_TGT32_LASTOUT
        if ((tid & 31) == 0 && stage_last_out(&drained[s], kThreads / 32) && i + kStages < nt)
            issue(i + kStages);                      // the last warp out of the stage refills it
#else
        if ((tid & 31) == 0) mbar_arrive(&empty_bar[s]);
#endif
    }

    const double scale = fixed_scale(*gmax_bits, P);
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        float x0, x1, y0, y1;
        upk(Rx[p], x0, x1);
        upk(Ry[p], y0, y1);
        const int i0 = base + (2 * p) * kThreads + tid;
        const int i1 = i0 + kThreads;
        if (i0 < nt_pts) {
            red_fixed(acc + 2 * (size_t)i0 + 0, x0, scale);
            red_fixed(acc + 2 * (size_t)i0 + 1, y0, scale);
        }
        if (i1 < nt_pts) {
            red_fixed(acc + 2 * (size_t)i1 + 0, x1, scale);
            red_fixed(acc + 2 * (size_t)i1 + 1, y1, scale);
        }
    }
}

vn_status farfield_targets_f32(const void *Xt, int64_t nt, const void *X, const void *F, const void *W,
                               int64_t nves, int64_t npts, double mu, void *Ut, cudaStream_t st)
{
    const int P = (int)(nves * npts), n = (int)nt;
    static int slots_dev[kMaxDevices] = {0};
    int &slots = slots_dev[current_device()];
    if (slots == 0) {
        int dev = 0, sms = 0, occ = 0;
        VN_CUDA(cudaGetDevice(&dev));
        VN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        VN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, targets_f32_kernel<kNP32>, kThreads, 0));
        slots = sms * (occ > 0 ? occ : 1);
    }
    // target blocks come from the free targets, chunks from the sources
    const Split sp = choose_split_for((n + kST32 - 1) / kST32, (P + kTile - 1) / kTile, slots, 16);

    const size_t b_src = (size_t)P * 32, b_acc = (size_t)n * 16;
    char *scratch = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scratch, b_src + b_acc + 16, st));
    ulonglong2 *src = (ulonglong2 *)scratch;
    long long *acc = (long long *)(scratch + b_src);
    unsigned *gmax = (unsigned *)(scratch + b_src + b_acc);
    VN_CUDA(cudaMemsetAsync(acc, 0, b_acc + 16, st));

    pack_sources_f32<<<(P + 255) / 256, 256, 0, st>>>((const float2 *)X, (const float2 *)F, (const float *)W, P, src, gmax);
    profile_mark(st, true);
    targets_f32_kernel<kNP32><<<sp.n_tb * sp.n_chunks, kThreads, 0, st>>>(src, (const float2 *)Xt, n, P, sp.n_tiles,
                                                                         sp.n_chunks, gmax, acc);
    profile_mark(st, false);
    finish_f32<<<(n + 255) / 256, 256, 0, st>>>(acc, n, P, gmax, 1.0 / (4.0 * 3.14159265358979323846 * mu), (float2 *)Ut);
    count_launch(3);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scratch, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// host-only: the decomposition vn_farfield (fp32) would use with `slots` resident blocks (vn_plan_farfield)
void plan_f32(long long P, int slots, int *super_tile, int *sub, SymSplit *sp)
{
    *super_tile = kST32;
    *sub = kSub32;
    *sp = choose_sym_split(P, kST32, slots, VN_F32_MINTILES, 0);
}

}  // namespace vn

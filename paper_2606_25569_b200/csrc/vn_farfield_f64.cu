// vn_farfield_f64.cu -- fp64 far-field Stokeslet sum for sm_100a (parity-grade variant, steps a-2 .. a-5).
//
//   U_i = 1/(4 pi mu) sum_{j not in ves(i)} [ -log|r| g_j + (r.g_j)/|r|^2 r ],  r = x_i - y_j, g_j = f_j w_j
//   (PAPER.md:129-136 eqs 2.8/2.9, :173 trapezoid rule, :425 DirectSingleLayerIntegral)
//
// Same decomposition as the fp32 kernel (vn_farfield_f32.cu): K(r) = -log|r| I + r r^T/|r|^2 is even
// and symmetric, so every unordered pair of points is evaluated once,
//   r = x - y; r2 = rx*rx + ry*ry; ml = -(1/2) ln r2; inv = 1/r2; u = r * inv
//   Kxx = ml + ux*rx;  Kxy = ux*ry;  Kyy = ml + uy*ry
// and applied in both directions, U_i += K g_j and U_j += K g_i: 28 DP instructions per unordered pair
// (14 per directed interaction) instead of about 36 per directed pair of a one-directional sum.
// The FP64 pipe (64 lanes/clk/SM) is the bound, so the instruction count is what matters: there is no
// SFU log or reciprocal in double, see log_rcp_f64().
// Cross-block accumulation goes through 2 x 64-bit fixed-point atomics per value (Fixed2 in
// vn_common.cuh): exact to 2^-102 of the term bound and bitwise reproducible.
#include "vn_common.cuh"
#include "vn_log64.cuh"

namespace vn {

#ifndef VN_F64_T
#define VN_F64_T 6                // measured at 2000 x 128 with 2 blocks/SM: 4 targets 1057, 6 targets 1091, 8 targets 1090 GInt/s
#endif
constexpr int kT64 = VN_F64_T;                // targets per thread
constexpr int kST64 = kT64 * kThreads;        // points per super-tile (target block): 512
constexpr int kSub64 = kST64 / kTile;         // source tiles per super-tile: 4
#ifndef VN_F64_BATCH
#define VN_F64_BATCH 8
#endif
#ifndef VN_F64_MINBLK
#define VN_F64_MINBLK 2           // 2 blocks/SM (up to 255 registers, no spills) beat 3 (168 registers): more independent
#endif                            // pairs in flight per warp matter more to the FP64 pipe than more warps
#ifndef VN_F64_GTAB
#define VN_F64_GTAB 1             // the pair kernel's blocks copy the log tables from scratch (built once per call by
#endif                            // pack_sources_f64 with the same code) instead of building them: +1 % at 2000 x 128,
                                  // +2.4 % at 256 x 128 (one-tile blocks)
#ifndef VN_F64_LASTOUT
#define VN_F64_LASTOUT 0          // 1: stage hand-back by the last warp out (as in the fp32 kernel); costs 28 bytes of
                                  // spills at 3 blocks/SM and measured 965 against 1000 GInt/s at 2000 x 128: off
#endif
#ifndef VN_F64_MAXTILES
#define VN_F64_MAXTILES kStages   // cap of the chunk length (0: none)
#endif
#ifndef VN_F64_SMEMRED
#define VN_F64_SMEMRED 1          // 1: the j <- i contributions of a batch are summed over the warp through a transposed
#endif                            // shared-memory buffer (16 STS.64 + 8 LDS.128 + 2 SHFL) instead of the register
                                  // transpose-reduce (0: 32 SHFL + 60 FSEL + 45 MOV for 64-bit values); 2, 3: the sum
                                  // deferred behind the next batch as in the fp32 kernel -- no gain here (pair kernel at
                                  // 2000 x 128: 59.93 ms with 1, 62.05 with 2 (two call sites of the batch cost an address
                                  // add per table lookup), 60.12 with 3): the FP64 pipe, not the reduction chain, is what
                                  // the two warps per scheduler wait for
#ifndef VN_TGT64_LASTOUT
#define VN_TGT64_LASTOUT 1         // free-target kernel: the last warp out of a ring stage refills it (stage_last_out);
#endif                             // measured 719 against 696 GInt/s at 2000 x 128 sources, 512 x 512 targets
#ifndef VN_F64_MINTILES
#define VN_F64_MINTILES 1
#endif
constexpr int kBatch64 = VN_F64_BATCH;        // sources per cross-lane reduction batch
// shared-memory layout of the fp64 kernels (dynamic)
constexpr int kPairTileBytes = kStages * kTile * 32;
constexpr int kTabBytes = (kLogTab + kExpTab) * 8;
constexpr int kRedRow = 36, kRedHalf = 18;
constexpr int kRedBytes = VN_F64_SMEMRED ? (kThreads / 32) * 2 * kBatch64 * kRedRow * 8 : 0;
constexpr int kPairSmem = kPairTileBytes + kRedBytes;      // dynamic part; the tables (kTabBytes) are static
constexpr int kTgtSmem = kPairTileBytes;

// a-2: one 32-byte record (yx, yy, gx, gy) per source, g = F*W; also gmax = max_j (|gx| + |gy|)
// (the bit pattern of a non-negative double orders like the double).
__global__ void pack_sources_f64(const double2 *__restrict__ X, const double2 *__restrict__ F,
                                 const double *__restrict__ W, int P, double4 *__restrict__ src,
                                 unsigned long long *__restrict__ gmax_bits, double *__restrict__ gtab)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (gtab) build_log_tables(gtab, s, gridDim.x * blockDim.x);   // once per call, for the pair kernel's blocks
    double m = 0.0;
    if (s < P) {
        const double2 y = X[s];
        const double2 f = F[s];
        const double w = W[s];
        const double gx = f.x * w, gy = f.y * w;
        src[s] = make_double4(y.x, y.y, gx, gy);
        m = fabs(gx) + fabs(gy);
        // a non-finite density or position cannot be carried through the integer accumulators point by point:
        // flag it (gmax = +Inf) and finish_f64 answers NaN everywhere
        if (!(m <= 1.7976931348623157e308) || !(fabs(y.x) + fabs(y.y) <= 1.7976931348623157e308))
            m = __longlong_as_double(0x7ff0000000000000ll);
    }
#pragma unroll
    for (int k = 16; k >= 1; k >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, k));
    if ((threadIdx.x & 31) == 0 && m != 0.0) atomicMax(gmax_bits, (unsigned long long)__double_as_longlong(m));
}

// a-3 / a-4: pair kernel; block (I, c) = super-tile I as targets x chunk c of I's list of source tiles
// (own super-tile one-directional with the own vesicle predicated out, then the tiles of super-tiles
// I+1 .. I+S_I in both directions) -- the same walk as farfield_f32_kernel.
// CHECK = true (vn_selfcheck): ring verification as in farfield_f32_kernel.
template <bool CHECK>
__global__ void __launch_bounds__(kThreads, VN_F64_MINBLK)
farfield_f64_kernel(const double4 *__restrict__ src, const double2 *__restrict__ X, int P, int npts,
                    int n_tiles, int n_st, int n_chunks, const unsigned long long *__restrict__ gmax_bits,
                    long long *__restrict__ acc, const double2 *__restrict__ gtab, int part, int nparts,
                    unsigned long long *__restrict__ mismatches)
{
    constexpr int T = kT64;
    constexpr int B = kBatch64;
    constexpr int kDup = 32 / (2 * B);              // lanes that end up with the same reduced value
    // the log tables are static shared memory (their addresses fold into the lookups as immediates); the tile ring
    // and the reduction buffer are dynamic (together with the tables more than the 48 KB a kernel may declare)
    extern __shared__ __align__(128) unsigned char smem_f64[];
    double4 (*tile)[kTile] = reinterpret_cast<double4 (*)[kTile]>(smem_f64);
    __shared__ __align__(16) double tab[kLogTab + kExpTab];
    __shared__ __align__(8) u64 full_bar[kStages];
#if VN_F64_LASTOUT
    __shared__ int drained[kStages];                 // warps that have left each stage (stage_last_out)
#else
    __shared__ __align__(8) u64 empty_bar[kStages];
#endif
#if VN_F64_SMEMRED
    // per warp: 2B rows (values) of 32 lanes; 16-byte loads of half rows are conflict-free with a half offset of
    // 18 doubles and a row stride of 36 (bank shifts of 4 and 8 words)
    double (*red)[2 * B * kRedRow] = reinterpret_cast<double (*)[2 * B * kRedRow]>(smem_f64 + kPairTileBytes);
#endif

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int bid = blockIdx.x * nparts + part;      // blocks are dealt round-robin to the parts (one part per GPU)
    const int I = bid / n_chunks;
    const int sc = bid - I * n_chunks;
    int S = (n_st - 1) / 2;
    if ((n_st & 1) == 0 && I < n_st / 2) S += 1;
    const int nu = kSub64 * (S + 1);
    const int u_begin = chunk_tile_begin(nu, n_chunks, sc);
    const int nt = chunk_tile_begin(nu, n_chunks, sc + 1) - u_begin;

    auto tile_of = [&](int u) {        // source tile index of list entry u (may be >= n_tiles: empty)
        const int s = u / kSub64;
        int J = I + s;
        if (J >= n_st) J -= n_st;
        return J * kSub64 + (u - s * kSub64);
    };

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full_bar[s], 1);
#if VN_F64_LASTOUT
            drained[s] = 0;
#else
            mbar_init(&empty_bar[s], kThreads / 32);
#endif
        }
        mbar_fence_init();
    }
#if VN_F64_GTAB
    static_assert((kLogTab + kExpTab) % (2 * kThreads) == 0, "table copy assumes whole rounds");
#pragma unroll
    for (int k = 0; k < (kLogTab + kExpTab) / (2 * kThreads); ++k)
        reinterpret_cast<double2 *>(tab)[k * kThreads + tid] = __ldg(gtab + k * kThreads + tid);
#else
    build_log_tables(tab, tid, kThreads);
#endif
    __syncthreads();

    auto issue = [&](int i) {   // one thread: list entry u_begin + i -> stage i % kStages
        const int s = i % kStages;
        const int first = tile_of(u_begin + i) * kTile;
        const int cnt = min(kTile, P - first);
        if (cnt > 0) {
            const uint32_t bytes = (uint32_t)cnt * 32u;
            mbar_expect_tx(&full_bar[s], bytes);
            bulk_g2s(&tile[s][0], src + first, bytes, &full_bar[s]);
        } else {
            mbar_arrive(&full_bar[s]);      // empty entry: complete the phase without a copy
        }
    };
    if (tid == 0) {
        const int pre = nt < kStages ? nt : kStages;
        for (int i = 0; i < pre; ++i) issue(i);
    }

    const Fixed2 fx = fixed2_scale(*gmax_bits, P);

    // targets: point base + k*kThreads + tid; indices past the end are clamped to P-1 and carry a zero
    // density (their results are never stored, their contributions to others vanish).
    const int base = I * kST64;
    double tx[T], ty[T], hx[T], hy[T], Ux[T], Uy[T];
#pragma unroll
    for (int k = 0; k < T; ++k) {
        const int i0 = base + k * kThreads + tid;
        const double4 a = src[min(i0, P - 1)];
        tx[k] = a.x;
        ty[k] = a.y;
        hx[k] = i0 < P ? a.z : 0.0;
        hy[k] = i0 < P ? a.w : 0.0;
        Ux[k] = Uy[k] = 0.0;
    }
    const int last_target = min(base + T * kThreads, P) - 1;
    const int span_begin = (base / npts) * npts;
    const int span_end = (last_target / npts + 1) * npts;

    for (int i = 0; i < nt; ++i) {
        const int s = i % kStages;
#if !VN_F64_LASTOUT
        if (tid == 0 && i >= 1 && i - 1 + kStages < nt) {   // refill the stage drained last iteration
            mbar_wait(&empty_bar[(i - 1) % kStages], ((i - 1) / kStages) & 1);
            issue(i - 1 + kStages);
        }
#endif
        mbar_wait(&full_bar[s], (i / kStages) & 1);

        const int u = u_begin + i;
        const bool both = u >= kSub64;                    // another super-tile: both directions
        const int first = tile_of(u) * kTile;
        const int cnt = min(kTile, P - first);
        const double4 *ts = tile[s];
        auto verify = [&](int j, const double4 &sj) {                                // CHECK builds only
            const double2 *o = reinterpret_cast<const double2 *>(src + first + j);
            const double2 oa = __ldcg(o), ob = __ldcg(o + 1);
            if (__double_as_longlong(oa.x) != __double_as_longlong(sj.x) || __double_as_longlong(oa.y) != __double_as_longlong(sj.y) ||
                __double_as_longlong(ob.x) != __double_as_longlong(sj.z) || __double_as_longlong(ob.y) != __double_as_longlong(sj.w))
                atomicAdd(mismatches, 1ull);
        };
        const bool fast = both && (first >= span_end || first + kTile <= span_begin) && (cnt == kTile);
        if (fast) {
            // lane L ends a batch holding the warp total of value L / kDup (value = 2*source + component);
            // sub-lane 0 adds its high word, sub-lane 1 its low word
            long long *accj = acc + 4 * (size_t)first + 2 * (lane / kDup) + (lane % kDup);
            // this thread's contributions c[2 jj], c[2 jj + 1] to the sources jb .. jb + B - 1 (and its own sums Ux, Uy)
            auto batch = [&](int jb, double (&c)[2 * B]) {
#pragma unroll
                for (int jj = 0; jj < B; ++jj) {
                    const double4 sj = ts[jb + jj];
                    if (CHECK) verify(jb + jj, sj);
                    double cx = 0.0, cy = 0.0;
#pragma unroll
                    for (int k = 0; k < T; ++k) {
                        const double rx = tx[k] - sj.x, ry = ty[k] - sj.y;
                        const double r2 = fma(rx, rx, ry * ry);
                        double ml, inv;
                        log_rcp_f64(r2, tab, ml, inv);
                        const double ux = rx * inv, uy = ry * inv;
                        const double Kxy = ux * ry;
                        const double Kxx = fma(ux, rx, ml);
                        const double Kyy = fma(uy, ry, ml);
                        Ux[k] = fma(Kxx, sj.z, fma(Kxy, sj.w, Ux[k]));
                        Uy[k] = fma(Kxy, sj.z, fma(Kyy, sj.w, Uy[k]));
                        cx = fma(Kxx, hx[k], fma(Kxy, hy[k], cx));
                        cy = fma(Kxy, hx[k], fma(Kyy, hy[k], cy));
                    }
                    c[2 * jj + 0] = cx;
                    c[2 * jj + 1] = cy;
                }
            };
#if VN_F64_SMEMRED == 3
            // as mode 2, with ONE call site of the batch arithmetic (the first trip has nothing parked yet)
            static_assert(kDup == 2, "shared-memory reduction assumes 16 values per batch");
            double *rw = red[tid >> 5];
            const int col = lane + (lane >= 16 ? kRedHalf - 16 : 0);
            const double2 *row = reinterpret_cast<const double2 *>(rw + (lane >> 1) * kRedRow + (lane & 1) * kRedHalf);
#pragma unroll 1
            for (int jb = 0; jb <= kTile; jb += B) {
                __syncwarp();                                       // the parked rows are complete
                double2 q[8];
                if (jb > 0) {
#pragma unroll
                    for (int e = 0; e < 8; ++e) q[e] = row[e];
                }
                double c[2 * B];
                if (jb < kTile) batch(jb, c);
                if (jb > 0) {
                    double t = (((q[0].x + q[0].y) + (q[1].x + q[1].y)) + ((q[2].x + q[2].y) + (q[3].x + q[3].y))) +
                               (((q[4].x + q[4].y) + (q[5].x + q[5].y)) + ((q[6].x + q[6].y) + (q[7].x + q[7].y)));
                    t += __shfl_xor_sync(0xffffffffu, t, 1);
                    if ((lane % kDup) < 2)
                        atomicAdd((unsigned long long *)(accj + 4 * (jb - B)), (unsigned long long)fixed2_word(t, fx, lane % kDup));
                }
                if (jb < kTile) {
                    __syncwarp();                                   // every lane has read the previous batch's rows
#pragma unroll
                    for (int v = 0; v < 2 * B; ++v) rw[v * kRedRow + col] = c[v];
                }
            }
#elif VN_F64_SMEMRED == 2
            // The c values of a batch are parked in the transposed shared-memory buffer and summed over the warp while
            // the NEXT batch is computed (loads issued before that batch's arithmetic, nothing of it depends on them).
            static_assert(kDup == 2, "shared-memory reduction assumes 16 values per batch");
            double *rw = red[tid >> 5];
            const int col = lane + (lane >= 16 ? kRedHalf - 16 : 0);
            const double2 *row = reinterpret_cast<const double2 *>(rw + (lane >> 1) * kRedRow + (lane & 1) * kRedHalf);
            auto park = [&](const double (&c)[2 * B]) {
                __syncwarp();                                       // every lane has read the previous batch's rows
#pragma unroll
                for (int v = 0; v < 2 * B; ++v) rw[v * kRedRow + col] = c[v];
            };
            auto total = [&](const double2 (&q)[8]) {
                double t = (((q[0].x + q[0].y) + (q[1].x + q[1].y)) + ((q[2].x + q[2].y) + (q[3].x + q[3].y))) +
                           (((q[4].x + q[4].y) + (q[5].x + q[5].y)) + ((q[6].x + q[6].y) + (q[7].x + q[7].y)));
                t += __shfl_xor_sync(0xffffffffu, t, 1);
                return t;
            };
            {
                double c[2 * B];
                batch(0, c);
                park(c);
            }
#pragma unroll 1
            for (int jb = B; jb < kTile; jb += B) {
                __syncwarp();                                       // the parked rows are complete
                double2 q[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) q[e] = row[e];
                double c[2 * B];
                batch(jb, c);
                const double t = total(q);
                if ((lane % kDup) < 2)
                    atomicAdd((unsigned long long *)(accj + 4 * (jb - B)), (unsigned long long)fixed2_word(t, fx, lane % kDup));
                park(c);
            }
            {
                __syncwarp();
                double2 q[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) q[e] = row[e];
                const double t = total(q);
                if ((lane % kDup) < 2)
                    atomicAdd((unsigned long long *)(accj + 4 * (kTile - B)), (unsigned long long)fixed2_word(t, fx, lane % kDup));
            }
#else
#pragma unroll 1
            for (int jb = 0; jb < kTile; jb += B) {
                double c[2 * B];
                batch(jb, c);
#if VN_F64_SMEMRED == 1
                // sum over the warp through shared memory: lane L stores value v at row v, column L; then lane L
                // adds up half (L & 1) of row L >> 1 and the two halves meet in one shuffle: lane L ends with the
                // warp total of value L / 2 (kDup = 2 at B = 8)
                static_assert(kDup == 2, "shared-memory reduction assumes 16 values per batch");
                {
                    double *rw = red[tid >> 5];
                    const int col = lane + (lane >= 16 ? kRedHalf - 16 : 0);
                    __syncwarp();                                   // the previous batch's reads are done
#pragma unroll
                    for (int v = 0; v < 2 * B; ++v) rw[v * kRedRow + col] = c[v];
                    __syncwarp();
                    const double2 *row = reinterpret_cast<const double2 *>(rw + (lane >> 1) * kRedRow + (lane & 1) * kRedHalf);
                    double s0 = 0.0, s1 = 0.0;
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        const double2 v = row[q];
                        s0 += v.x;
                        s1 += v.y;
                    }
                    c[0] = s0 + s1;
                    c[0] += __shfl_xor_sync(0xffffffffu, c[0], 1);
                }
#else
                // transpose-reduce over the warp: 2B values per lane -> one warp total per lane
                int m = 16;
#pragma unroll
                for (int w = B; w >= 1; w >>= 1, m >>= 1) {
                    const bool up = (lane & m) != 0;
#pragma unroll
                    for (int k = 0; k < w; ++k) {
                        const double send = up ? c[k] : c[k + w];
                        const double keep = up ? c[k + w] : c[k];
                        c[k] = keep + __shfl_xor_sync(0xffffffffu, send, m);
                    }
                }
#pragma unroll
                for (; m >= 1; m >>= 1) c[0] += __shfl_xor_sync(0xffffffffu, c[0], m);
#endif
                if ((lane % kDup) < 2)
                    atomicAdd((unsigned long long *)(accj + 4 * jb),
                              (unsigned long long)fixed2_word(c[0], fx, lane % kDup));
            }
#endif
        } else if (!both && cnt == kTile && npts % kTile == 0 && base + kST64 <= P) {
            // a tile of the block's OWN super-tile when vesicles are whole tiles (npts a multiple of 128): target k
            // of every thread lies in tile k, so "own vesicle" is the same decision for the whole block -- a uniform
            // skip instead of a per-pair predicate.  One-directional.
            const int vs_src = first / npts;
            bool skip[T];
#pragma unroll
            for (int k = 0; k < T; ++k) skip[k] = (base + k * kThreads) / npts == vs_src;
#pragma unroll 2
            for (int j = 0; j < kTile; ++j) {
                const double4 sj = ts[j];
                if (CHECK) verify(j, sj);
#pragma unroll
                for (int k = 0; k < T; ++k) {
                    if (skip[k]) continue;
                    const double rx = tx[k] - sj.x, ry = ty[k] - sj.y;
                    const double r2 = fma(rx, rx, ry * ry);
                    double ml, inv;
                    log_rcp_f64(r2, tab, ml, inv);
                    const double qd = fma(rx, sj.z, ry * sj.w) * inv;
                    Ux[k] = fma(ml, sj.z, fma(qd, rx, Ux[k]));
                    Uy[k] = fma(ml, sj.w, fma(qd, ry, Uy[k]));
                }
            }
        } else if (cnt > 0) {
            // predicated path: own-vesicle sources and the ragged tail are skipped per pair
            int own[T];
#pragma unroll
            for (int k = 0; k < T; ++k) own[k] = (min(base + k * kThreads + tid, P - 1) / npts) * npts;
#pragma unroll 1
            for (int j = 0; j < cnt; ++j) {
                const double4 sj = ts[j];
                if (CHECK) verify(j, sj);
                const int jg = first + j;
                double cx = 0.0, cy = 0.0;
#pragma unroll
                for (int k = 0; k < T; ++k) {
                    if ((unsigned)(jg - own[k]) >= (unsigned)npts) {
                        const double rx = tx[k] - sj.x, ry = ty[k] - sj.y;
                        const double r2 = fma(rx, rx, ry * ry);
                        double ml, inv;
                        log_rcp_f64(r2, tab, ml, inv);
                        const double ux = rx * inv, uy = ry * inv;
                        const double Kxy = ux * ry;
                        const double Kxx = fma(ux, rx, ml);
                        const double Kyy = fma(uy, ry, ml);
                        Ux[k] = fma(Kxx, sj.z, fma(Kxy, sj.w, Ux[k]));
                        Uy[k] = fma(Kxy, sj.z, fma(Kyy, sj.w, Uy[k]));
                        cx = fma(Kxx, hx[k], fma(Kxy, hy[k], cx));
                        cy = fma(Kxy, hx[k], fma(Kyy, hy[k], cy));
                    }
                }
                if (both) {
#pragma unroll
                    for (int m = 16; m >= 1; m >>= 1) {
                        cx += __shfl_xor_sync(0xffffffffu, cx, m);
                        cy += __shfl_xor_sync(0xffffffffu, cy, m);
                    }
                    if (lane < 4) {   // lanes 0..3: x hi, x lo, y hi, y lo
                        const double v = (lane & 2) ? cy : cx;
                        atomicAdd((unsigned long long *)(acc + 4 * (size_t)jg + lane),
                                  (unsigned long long)fixed2_word(v, fx, lane & 1));
                    }
                }
            }
        }
        __syncwarp();
#if VN_F64_LASTOUT
        if (lane == 0 && stage_last_out(&drained[s], kThreads / 32) && i + kStages < nt)
            issue(i + kStages);                      // the last warp out of the stage refills it
#else
        if (lane == 0) mbar_arrive(&empty_bar[s]);
#endif
    }

    // this block's sums for its own targets
#pragma unroll
    for (int k = 0; k < T; ++k) {
        const int i0 = base + k * kThreads + tid;
        if (i0 < P) {
            red_fixed2(acc + 4 * (size_t)i0 + 0, Ux[k], fx);
            red_fixed2(acc + 4 * (size_t)i0 + 2, Uy[k], fx);
        }
    }
}

// a-5: fixed point -> double, scale by 1/(4 pi mu), store U.
__global__ void finish_f64(const long long *__restrict__ acc, int n, int P, const unsigned long long *__restrict__ gmax_bits,
                           double prefactor, double2 *__restrict__ U)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (*gmax_bits == 0x7ff0000000000000ull) {            // non-finite input somewhere: see pack_sources_f64
        const double qnan = __longlong_as_double(0x7ff8000000000000ll);
        U[i] = make_double2(qnan, qnan);
        return;
    }
    const Fixed2 fx = fixed2_scale(*gmax_bits, P);
    const longlong2 a = *reinterpret_cast<const longlong2 *>(acc + 4 * (size_t)i);
    const longlong2 b = *reinterpret_cast<const longlong2 *>(acc + 4 * (size_t)i + 2);
    U[i] = make_double2(prefactor * fixed2_value(a.x, a.y, fx), prefactor * fixed2_value(b.x, b.y, fx));
}

// pack + pair kernel for the blocks of one part: acc (P x 4 words) and gmax are the caller's, already zeroed;
// scratch holds the packed sources and, behind them, the log tables
static vn_status accumulate_f64(const void *X, const void *F, const void *W, int P, int npts, int part, int nparts,
                                char *scratch, long long *acc, unsigned long long *gmax, cudaStream_t st,
                                unsigned long long *mismatches = nullptr)
{
    static int slots_dev[kMaxDevices] = {0};
    int &slots = slots_dev[current_device()];
    if (slots == 0) {
        int dev = 0, sms = 0, occ = 0;
        VN_CUDA(cudaGetDevice(&dev));
        VN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        VN_CUDA(cudaFuncSetAttribute(farfield_f64_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPairSmem));
        VN_CUDA(cudaFuncSetAttribute(farfield_f64_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPairSmem));
        VN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, farfield_f64_kernel<false>, kThreads, kPairSmem));
        slots = sms * (occ > 0 ? occ : 1);
    }
    const SymSplit sp = choose_sym_split(P, kST64, slots, VN_F64_MINTILES, VN_F64_MAXTILES);   // see accumulate_f32
    const long long blocks = (long long)sp.n_st * sp.n_chunks;
    const int mine = (int)((blocks - part + nparts - 1) / nparts);
    double4 *src = (double4 *)scratch;
    double *gtab = VN_F64_GTAB ? (double *)(scratch + (size_t)P * 32) : nullptr;   // 16-byte aligned
    pack_sources_f64<<<(P + 255) / 256, 256, 0, st>>>((const double2 *)X, (const double2 *)F, (const double *)W, P, src, gmax, gtab);
    profile_mark(st, true);
    if (mine > 0 && !mismatches)
        farfield_f64_kernel<false><<<mine, kThreads, kPairSmem, st>>>(src, (const double2 *)X, P, npts, sp.n_tiles, sp.n_st,
                                                                      sp.n_chunks, gmax, acc, (const double2 *)gtab, part, nparts, nullptr);
    else if (mine > 0)
        farfield_f64_kernel<true><<<mine, kThreads, kPairSmem, st>>>(src, (const double2 *)X, P, npts, sp.n_tiles, sp.n_st,
                                                                     sp.n_chunks, gmax, acc, (const double2 *)gtab, part, nparts, mismatches);
    profile_mark(st, false);
    count_launch(mine > 0 ? 2 : 1);
    return VN_OK;
}
static size_t scratch_f64_bytes(int P) { return (size_t)P * 32 + (VN_F64_GTAB ? (size_t)kTabBytes : 0); }

vn_status farfield_f64(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                       void *U, cudaStream_t st, const int64_t *near_ptr, const int32_t *near_ves)
{
    const int P = (int)(nves * npts);
    // scratch: packed sources | log tables | fixed-point accumulators (hi, lo per component) | gmax
    const size_t b_src = scratch_f64_bytes(P), b_acc = (size_t)P * 32;
    char *scratch = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scratch, b_src + b_acc + 16, st));
    long long *acc = (long long *)(scratch + b_src);
    unsigned long long *gmax = (unsigned long long *)(scratch + b_src + b_acc);
    VN_CUDA(cudaMemsetAsync(acc, 0, b_acc + 16, st));
    vn_status rc = accumulate_f64(X, F, W, P, (int)npts, 0, 1, scratch, acc, gmax, st);
    if (rc == VN_OK && near_ptr)   // row f-1: take the near vesicles' contributions out again before the final rounding
        rc = near_correction_f64(X, F, W, P, (int)npts, near_ptr, near_ves, acc, gmax, st);
    if (rc != VN_OK) { (void)cudaFreeAsync(scratch, st); return rc; }
    finish_f64<<<(P + 255) / 256, 256, 0, st>>>(acc, P, P, gmax, 1.0 / (4.0 * 3.14159265358979323846 * mu), (double2 *)U);
    count_launch(1);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scratch, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// vn_selfcheck (see farfield_selfcheck_f32)
vn_status farfield_selfcheck_f64(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                                 void *U, unsigned long long *mismatches, cudaStream_t st)
{
    const int P = (int)(nves * npts);
    const size_t b_src = scratch_f64_bytes(P), b_acc = (size_t)P * 32;
    char *scratch = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scratch, b_src + b_acc + 16, st));
    VN_CUDA(cudaMemsetAsync(scratch, 0xFF, b_src + b_acc + 16, st));
    long long *acc = (long long *)(scratch + b_src);
    unsigned long long *gmax = (unsigned long long *)(scratch + b_src + b_acc);
    VN_CUDA(cudaMemsetAsync(acc, 0, b_acc + 16, st));
    const vn_status rc = accumulate_f64(X, F, W, P, (int)npts, 0, 1, scratch, acc, gmax, st, mismatches);
    if (rc != VN_OK) { (void)cudaFreeAsync(scratch, st); return rc; }
    finish_f64<<<(P + 255) / 256, 256, 0, st>>>(acc, P, P, gmax, 1.0 / (4.0 * 3.14159265358979323846 * mu), (double2 *)U);
    count_launch(1);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scratch, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// Section 8e building blocks (see vn_farfield_f32.cu)
vn_status farfield_partial_f64(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, int part,
                               int nparts, void *acc, void *gmax, cudaStream_t st)
{
    const int P = (int)(nves * npts);
    char *scratch = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scratch, scratch_f64_bytes(P), st));
    VN_CUDA(cudaMemsetAsync(acc, 0, (size_t)P * 32, st));
    VN_CUDA(cudaMemsetAsync(gmax, 0, 8, st));
    const vn_status rc = accumulate_f64(X, F, W, P, (int)npts, part, nparts, scratch, (long long *)acc,
                                        (unsigned long long *)gmax, st);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scratch, st));
    return rc != VN_OK ? rc : (e == cudaSuccess ? VN_OK : VN_ERR_CUDA);
}

vn_status farfield_finish_f64(const void *acc, const void *gmax, int64_t P_total, int64_t count, double mu, void *U,
                              cudaStream_t st)
{
    finish_f64<<<(int)((count + 255) / 256), 256, 0, st>>>((const long long *)acc, (int)count, (int)P_total,
                                                           (const unsigned long long *)gmax,
                                                           1.0 / (4.0 * 3.14159265358979323846 * mu), (double2 *)U);
    count_launch(1);
    return cudaGetLastError() == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------------
// Row f-4: free targets in double (see targets_f32_kernel): one-directional sum over ALL vesicles,
// 4 targets per thread, per pair  acc += ml * g + ((r.g) inv) * r  (22 DP instructions).
#ifndef VN_F64_TGT_MINBLK
#define VN_F64_TGT_MINBLK 4
#endif
#ifndef VN_F64_TGT_T
#define VN_F64_TGT_T 4
#endif
constexpr int kT64T = VN_F64_TGT_T;            // targets per thread of the free-target kernel
__global__ void __launch_bounds__(kThreads, VN_F64_TGT_MINBLK)
targets_f64_kernel(const double4 *__restrict__ src, const double2 *__restrict__ Xt, int nt_pts, int P,
                   int n_tiles, int n_chunks, const unsigned long long *__restrict__ gmax_bits,
                   long long *__restrict__ acc)
{
    constexpr int T = kT64T;
    extern __shared__ __align__(128) unsigned char smem_f64[];
    double4 (*tile)[kTile] = reinterpret_cast<double4 (*)[kTile]>(smem_f64);
    __shared__ __align__(16) double tab[kLogTab + kExpTab];
    __shared__ __align__(8) u64 full_bar[kStages];
#if VN_TGT64_LASTOUT
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
#if VN_TGT64_LASTOUT
            drained[s] = 0;
#else
            mbar_init(&empty_bar[s], kThreads / 32);
#endif
        }
        mbar_fence_init();
    }
    build_log_tables(tab, tid, kThreads);
    __syncthreads();

    auto issue = [&](int i) {
        const int s = i % kStages;
        const int first = (t_begin + i) * kTile;
        const uint32_t bytes = (uint32_t)min(kTile, P - first) * 32u;
        mbar_expect_tx(&full_bar[s], bytes);
        bulk_g2s(&tile[s][0], src + first, bytes, &full_bar[s]);
    };
    if (tid == 0) {
        const int pre = nt < kStages ? nt : kStages;
        for (int i = 0; i < pre; ++i) issue(i);
    }

    const int base = tb * (T * kThreads);
    double tx[T], ty[T], ux[T], uy[T];
#pragma unroll
    for (int k = 0; k < T; ++k) {
        const double2 a = Xt[min(base + k * kThreads + tid, nt_pts - 1)];
        tx[k] = a.x;
        ty[k] = a.y;
        ux[k] = uy[k] = 0.0;
    }

    for (int i = 0; i < nt; ++i) {
        const int s = i % kStages;
#if !VN_TGT64_LASTOUT
        if (tid == 0 && i >= 1 && i - 1 + kStages < nt) {
            mbar_wait(&empty_bar[(i - 1) % kStages], ((i - 1) / kStages) & 1);
            issue(i - 1 + kStages);
        }
#endif
        mbar_wait(&full_bar[s], (i / kStages) & 1);
        const int cnt = min(kTile, P - (t_begin + i) * kTile);
        const double4 *ts = tile[s];
#pragma unroll 2
        for (int j = 0; j < cnt; ++j) {
            const double4 sj = ts[j];
#pragma unroll
            for (int k = 0; k < T; ++k) {
                const double rx = tx[k] - sj.x, ry = ty[k] - sj.y;
                const double r2 = fma(rx, rx, ry * ry);
                double ml, inv;
                log_rcp_f64(r2, tab, ml, inv);
                const double q = fma(rx, sj.z, ry * sj.w) * inv;
                ux[k] = fma(ml, sj.z, fma(q, rx, ux[k]));
                uy[k] = fma(ml, sj.w, fma(q, ry, uy[k]));
            }
        }
        __syncwarp();
#if VN_TGT64_LASTOUT
        if ((tid & 31) == 0 && stage_last_out(&drained[s], kThreads / 32) && i + kStages < nt)
            issue(i + kStages);                      // the last warp out of the stage refills it
#else
        if ((tid & 31) == 0) mbar_arrive(&empty_bar[s]);
#endif
    }

    const Fixed2 fx = fixed2_scale(*gmax_bits, P);
#pragma unroll
    for (int k = 0; k < T; ++k) {
        const int i0 = base + k * kThreads + tid;
        if (i0 < nt_pts) {
            red_fixed2(acc + 4 * (size_t)i0 + 0, ux[k], fx);
            red_fixed2(acc + 4 * (size_t)i0 + 2, uy[k], fx);
        }
    }
}

vn_status farfield_targets_f64(const void *Xt, int64_t nt, const void *X, const void *F, const void *W,
                               int64_t nves, int64_t npts, double mu, void *Ut, cudaStream_t st)
{
    const int P = (int)(nves * npts), n = (int)nt;
    static int slots_dev[kMaxDevices] = {0};
    int &slots = slots_dev[current_device()];
    if (slots == 0) {
        int dev = 0, sms = 0, occ = 0;
        VN_CUDA(cudaGetDevice(&dev));
        VN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        VN_CUDA(cudaFuncSetAttribute(targets_f64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTgtSmem));
        VN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, targets_f64_kernel, kThreads, kTgtSmem));
        slots = sms * (occ > 0 ? occ : 1);
    }
    const Split sp = choose_split_for((n + kT64T * kThreads - 1) / (kT64T * kThreads), (P + kTile - 1) / kTile, slots, 8);

    const size_t b_src = (size_t)P * 32, b_acc = (size_t)n * 32;
    char *scratch = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scratch, b_src + b_acc + 16, st));
    double4 *src = (double4 *)scratch;
    long long *acc = (long long *)(scratch + b_src);
    unsigned long long *gmax = (unsigned long long *)(scratch + b_src + b_acc);
    VN_CUDA(cudaMemsetAsync(acc, 0, b_acc + 16, st));

    pack_sources_f64<<<(P + 255) / 256, 256, 0, st>>>((const double2 *)X, (const double2 *)F, (const double *)W, P, src, gmax, nullptr);
    profile_mark(st, true);
    targets_f64_kernel<<<sp.n_tb * sp.n_chunks, kThreads, kTgtSmem, st>>>(src, (const double2 *)Xt, n, P, sp.n_tiles,
                                                                  sp.n_chunks, gmax, acc);
    profile_mark(st, false);
    finish_f64<<<(n + 255) / 256, 256, 0, st>>>(acc, n, P, gmax, 1.0 / (4.0 * 3.14159265358979323846 * mu), (double2 *)Ut);
    count_launch(3);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scratch, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// host-only: the decomposition vn_farfield (fp64) would use with `slots` resident blocks (vn_plan_farfield)
void plan_f64(long long P, int slots, int *super_tile, int *sub, SymSplit *sp)
{
    *super_tile = kST64;
    *sub = kSub64;
    *sp = choose_sym_split(P, kST64, slots, VN_F64_MINTILES, VN_F64_MAXTILES);
}

}  // namespace vn

// vn_fmm.cu -- row f-4 (second half) of DESIGN.md: the far-field sum by a fast multipole method, O(P) instead
// of O(P^2).  The paper names it as the missing piece: "Applying the fast multipole method will significantly
// reduce the cost and make it scale as O(M), but an applicable GPU implementation is beyond the scope of this
// paper" (PAPER.md:451; :173 for the trapezoid rule + FMM setting).  It is an APPROXIMATION of vn_farfield
// with a controlled truncation error (expansion order p), not a replacement of the exact path.
//
// In complex notation z = x + i y, g = gx + i gy, r = z - zeta_j, the 2-D Stokeslet sum is
//   u(z) = sum_j [ -log|r| g_j + g_j/2 + (r / conj r) conj(g_j) / 2 ]
//        = -( Re Phi1 + i Re Phi2 ) + (z/2) conj( Phi1' + i Phi2' ) - (1/2) conj( psi ),
//   Phi_m(z) = sum_j g_{m,j} log(z - zeta_j)  (m = 1, 2: the real and imaginary parts of g as real charges),
//   psi(z)   = sum_j ( conj(zeta_j) g_j / (z - zeta_j) - conj(g_j) ),
// i.e. two complex logarithmic potentials and one Cauchy sum, all analytic away from the sources, so the classic
// 2-D FMM applies (Greengard & Rokhlin 1987, cited PAPER.md:173): uniform quadtree with L levels over the bounding
// square, power moments about box centres scaled by the box size, M2M / M2L / L2L in scaled variables, local
// expansions evaluated at the targets, direct sums over the 3 x 3 neighbour boxes.  The target's own vesicle is
// excluded as in vn_farfield: the direct part skips it, and what the expansions included of it (own-vesicle
// points in non-neighbour boxes) is subtracted by a short direct sum.  The expansions are double for both storage
// precisions, so the accuracy of the far part is set by p alone (truncation error about 0.45^p relative, measured);
// the direct part runs in the storage precision (fp32: the SFU pair arithmetic of the exact fp32 kernel).
#ifdef VN_FMM_TIMING
#include <cstdio>
#endif

#include "vn_common.cuh"
#include "vn_log64.cuh"

namespace vn {

// scan kernels of vn_near.cu (exclusive scan of int counts into 64-bit offsets)
__global__ void scan_block_sums(const int *__restrict__ cnt, int P, long long *__restrict__ bsum);
__global__ void scan_of_sums(long long *__restrict__ bsum, int nb);
__global__ void scan_apply(const int *__restrict__ cnt, int P, const long long *__restrict__ bsum,
                           long long *__restrict__ ptr, long long *__restrict__ cursor);

// ------------------------------------------------------------------------------------------------
// complex helpers (double2 = re, im)
typedef double2 cplx;
__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x)); }
__device__ __forceinline__ cplx cfma(cplx a, cplx b, cplx c)   // a*b + c
{
    return make_double2(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y)));
}
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx cscale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }
__device__ __forceinline__ cplx crcp(cplx a) { const double d = 1.0 / (a.x * a.x + a.y * a.y); return make_double2(a.x * d, -a.y * d); }

// ------------------------------------------------------------------------------------------------
// geometry: bounding square of all points, kept on the device as four order-preserving encodings
// (xmin, ymin, xmax, ymax) so that no host synchronisation is needed
__device__ __forceinline__ unsigned long long enc_f64(double v)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double dec_f64(unsigned long long e)
{
    return __longlong_as_double((long long)((e >> 63) ? (e & 0x7fffffffffffffffull) : ~e));
}
// Everything after the binning works in coordinates relative to the CENTRE of the root square (fmm_choose_level
// fixes it, fmm_bin subtracts it from the internal copies of the points): the moments conj(zeta) g and the term
// z conj(Phi') of the evaluation are each of size |z| / |r| times the result, so with absolute coordinates a
// suspension far from the origin would lose digits that the translation-invariant exact path keeps.
struct Geom {
    double x0, y0, size;     // lower-left corner and edge of the root square
};
__device__ __forceinline__ Geom load_geom(const unsigned long long *__restrict__ enc)
{
    Geom g;
    g.x0 = dec_f64(enc[0]);
    g.y0 = dec_f64(enc[1]);
    const double ex = dec_f64(enc[2]) - g.x0, ey = dec_f64(enc[3]) - g.y0;
    g.size = fmax(fmax(ex, ey) * (1.0 + 1e-9), 1e-300);
    return g;
}
__device__ __forceinline__ cplx box_centre(const Geom &g, int level, int ix, int iy)
{
    const double s = g.size / (double)(1 << level);
    return make_double2(fma((double)ix + 0.5, s, g.x0), fma((double)iy + 0.5, s, g.y0));
}

// enc[0..3] while the bounding box is being collected: ~enc(xmin), ~enc(ymin), enc(xmax), enc(ymax), all four
// growing under atomicMax from ZERO, so that the one memset that clears the counters initialises them too;
// enc[8] counts the blocks of the load kernels that have committed their box.  fmm_choose_level (run by the last of
// those blocks) turns them into the final form: plain encodings relative to the centre of the root square.
// Depth of the tree, chosen ON THE DEVICE once the bounding box is known (no host synchronisation): leaves of
// about kLeafTarget points, where the points are assumed to fill the bounding RECTANGLE evenly, i.e. a
// fraction 1/aspect of the root square (a 4:1 channel leaves three quarters of the leaves empty).  The host
// sizes scratch and grids for L_hi (two levels deeper than a full square needs); kernels of unused levels
// and leaves return at once.  enc[4] holds the level.
constexpr double kLeafTarget = 64.0;
__device__ void fmm_choose_level(volatile unsigned long long *enc, int P, int L_hi)
{
    if (enc[2] == 0ull) {                               // no finite point at all: an empty box, as before
        enc[0] = ~0ull;
        enc[1] = ~0ull;
    } else {
        enc[0] = ~enc[0];
        enc[1] = ~enc[1];
    }
    const double ex = dec_f64(enc[2]) - dec_f64(enc[0]), ey = dec_f64(enc[3]) - dec_f64(enc[1]);
    const double lo = fmin(ex, ey), hi = fmax(ex, ey);
    double occ = (hi > 0.0 && lo > 0.0) ? lo / hi : 1.0;
    occ = fmax(occ, 1.0 / 16.0);
    int L = 2;
    while (L < L_hi && (double)P / (occ * (double)(1ll << (2 * L))) > kLeafTarget) ++L;
#ifdef VN_FMM_LEVEL_SHIFT                               // build-time experiment: coarser (-1) or finer (+1) tree
    L += VN_FMM_LEVEL_SHIFT;
    L = L < 2 ? 2 : (L > L_hi ? L_hi : L);
#endif
    enc[4] = (unsigned long long)L;
    // centre of the root square; the bounds are re-encoded relative to it (every later kernel reads these)
    const double x0 = dec_f64(enc[0]), y0 = dec_f64(enc[1]), x1 = dec_f64(enc[2]), y1 = dec_f64(enc[3]);
    if (x0 <= x1) {
        const double half = 0.5 * fmax(fmax(x1 - x0, y1 - y0) * (1.0 + 1e-9), 1e-300);
        const double cx = x0 + half, cy = y0 + half;
        enc[5] = (unsigned long long)__double_as_longlong(cx);
        enc[6] = (unsigned long long)__double_as_longlong(cy);
        enc[0] = enc_f64(x0 - cx);
        enc[1] = enc_f64(y0 - cy);
        enc[2] = enc_f64(x1 - cx);
        enc[3] = enc_f64(y1 - cy);
    } else {
        enc[5] = 0ull;
        enc[6] = 0ull;
    }
}
__device__ __forceinline__ int load_level(const unsigned long long *__restrict__ enc) { return (int)enc[4]; }

// bounding box of a block's points: per-thread extremes -> warp shuffles -> shared memory -> FOUR atomics per block
// (one set per warp was 128 K serialised 64-bit atomics on four addresses at a million points: 80 of the kernel's 96 us)
__device__ __forceinline__ void bounds_commit(double x, double y, double X1, double Y1, unsigned long long *enc,
                                              unsigned tickets, int P_level, int L_hi)
{   // tickets: blocks of ALL load kernels of the call (sources, and targets where they are a separate set); the block
    // that draws the last one knows the whole box and fixes level and centre (no launch of its own for that)
    __shared__ double red[4][32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
        x = fmin(x, __shfl_xor_sync(0xffffffffu, x, m));
        y = fmin(y, __shfl_xor_sync(0xffffffffu, y, m));
        X1 = fmax(X1, __shfl_xor_sync(0xffffffffu, X1, m));
        Y1 = fmax(Y1, __shfl_xor_sync(0xffffffffu, Y1, m));
    }
    if (lane == 0) { red[0][warp] = x; red[1][warp] = y; red[2][warp] = X1; red[3][warp] = Y1; }
    __syncthreads();
    if (warp != 0) return;
    x = lane < nw ? red[0][lane] : INFINITY;
    y = lane < nw ? red[1][lane] : INFINITY;
    X1 = lane < nw ? red[2][lane] : -INFINITY;
    Y1 = lane < nw ? red[3][lane] : -INFINITY;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
        x = fmin(x, __shfl_xor_sync(0xffffffffu, x, m));
        y = fmin(y, __shfl_xor_sync(0xffffffffu, y, m));
        X1 = fmax(X1, __shfl_xor_sync(0xffffffffu, X1, m));
        Y1 = fmax(Y1, __shfl_xor_sync(0xffffffffu, Y1, m));
    }
    if (lane != 0) return;
    if (x <= X1) {
        atomicMax(enc + 0, ~enc_f64(x));
        atomicMax(enc + 1, ~enc_f64(y));
        atomicMax(enc + 2, enc_f64(X1));
        atomicMax(enc + 3, enc_f64(Y1));
    }
    __threadfence();
    if (atomicAdd(enc + 8, 1ull) == (unsigned long long)tickets - 1ull) {
        __threadfence();
        fmm_choose_level(enc, P_level, L_hi);
    }
}
constexpr int kLoadBlocks = 148 * 8;      // grid-stride: at most this many blocks commit a bounding box

__device__ void fmm_build_tables(int block, int q, double *base, double *logtab);

// positions and densities g = F*W promoted to double (original order), and the bounding box
template <typename real, typename real2>
__global__ void __launch_bounds__(256)
fmm_load(const real2 *__restrict__ X, const real2 *__restrict__ F, const real *__restrict__ W, int P,
         cplx *__restrict__ z, cplx *__restrict__ g, unsigned long long *enc, unsigned tickets, int P_level, int L_hi,
         int load_blocks, int q, double *tab, double *logtab)
{   // blocks load_blocks .. gridDim.x - 1 build the translation tables (fmm_build_tables) and touch no point
    if ((int)blockIdx.x >= load_blocks) {
        fmm_build_tables((int)blockIdx.x - load_blocks, q, tab, logtab);
        return;
    }
    double x = INFINITY, y = INFINITY, X1 = -INFINITY, Y1 = -INFINITY;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P; i += load_blocks * blockDim.x) {
        const real2 p = X[i];
        const real2 f = F[i];
        const real w = W[i];
        const double px = (double)p.x, py = (double)p.y;
        x = fmin(x, px);
        y = fmin(y, py);
        X1 = fmax(X1, px);
        Y1 = fmax(Y1, py);
        z[i] = make_double2(px, py);
        g[i] = make_double2((double)(f.x * w), (double)(f.y * w));   // product in the storage precision, as in the exact path
    }
    bounds_commit(x, y, X1, Y1, enc, tickets, P_level, L_hi);
}

// moves every point into the root square's frame (in place, see Geom), then: leaf box of every point and the
// population count of the leaves
__global__ void __launch_bounds__(256)
fmm_bin(cplx *__restrict__ z, int P, const unsigned long long *__restrict__ enc, int *__restrict__ cell,
        int *__restrict__ cnt)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P) return;
    const Geom gm = load_geom(enc);
    const int n = 1 << load_level(enc);
    const double inv = (double)n / gm.size;
    const cplx zc = make_double2(z[i].x - __longlong_as_double((long long)enc[5]), z[i].y - __longlong_as_double((long long)enc[6]));
    z[i] = zc;
    const int ix = min(max((int)((zc.x - gm.x0) * inv), 0), n - 1);
    const int iy = min(max((int)((zc.y - gm.y0) * inv), 0), n - 1);
    const int c = ix * n + iy;
    cell[i] = c;
    atomicAdd(cnt + c, 1);
}

__global__ void __launch_bounds__(256)
fmm_scatter(const int *__restrict__ cell, int P, long long *__restrict__ cursor, int *__restrict__ perm)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P) return;
    const long long pos = (long long)atomicAdd((unsigned long long *)(cursor + cell[i]), 1ull);
    perm[pos] = i;                                     // arbitrary order inside a leaf; fmm_sort_cells fixes it
}

// the atomic scatter leaves every leaf's points in arbitrary order: order each segment by point index so that
// every later sum runs in a fixed order (bitwise reproducible results).  One warp per leaf, rank sort: the
// indices of a segment are distinct, so the rank of an entry is the number of smaller ones.
// ... and the leaf's points are gathered into the sorted arrays by the warp that has just sorted them (no launch of
// its own, no second pass over perm): sources (z, g -> zs, gs, vesicle index vs, float record srcf) or free targets.
struct GatherArgs {
    const cplx *z, *g;          // original order (g == nullptr: free targets, positions only)
    cplx *zs, *gs;
    int *vs;
    float4 *srcf;               // nullable
    int npts;
};
__device__ __forceinline__ void gather_one(const GatherArgs &ga, long long pos, int i)
{
    const cplx zi = ga.z[i];
    ga.zs[pos] = zi;
    if (ga.g) {
        const cplx gi = ga.g[i];
        ga.gs[pos] = gi;
        ga.vs[pos] = i / ga.npts;
        if (ga.srcf) ga.srcf[pos] = make_float4((float)zi.x, (float)zi.y, (float)gi.x, (float)gi.y);
    }
}
__global__ void __launch_bounds__(128)
fmm_sort_cells(const long long *__restrict__ start, const unsigned long long *__restrict__ enc,
               const int *unsorted, int *__restrict__ perm, GatherArgs ga)
{   // the leaves of the level the device chose, walked with a grid stride: a grid sized for the deepest admissible
    // tree is mostly blocks without a leaf (61 K of 65 K at a million points), and scheduling those cost 40 us.
    // `unsorted` may be ga.vs (the sources' scatter buffer): a leaf's entries are all read before any is written.
    constexpr int kBuf = 256;                          // leaves up to this size are sorted in shared memory
    __shared__ int buf[4][kBuf];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ncell = 1 << (2 * load_level(enc));
    for (int c = blockIdx.x * 4 + w; c < ncell; c += gridDim.x * 4) {
    const long long a = start[c], b = start[c + 1];
    const int m = (int)(b - a);
    if (m <= 1) {
        if (m == 1 && lane == 0) {
            const int v = unsorted[a];
            perm[a] = v;
            gather_one(ga, a, v);
        }
        continue;
    }
    __syncwarp();                                      // the previous leaf's buffer is written out
    if (m <= kBuf) {                                   // bitonic network in the warp's shared memory (indices are distinct)
        int n2 = 2;
        while (n2 < m) n2 <<= 1;
        for (int i = lane; i < n2; i += 32) buf[w][i] = i < m ? unsorted[a + i] : 0x7fffffff;
        __syncwarp();
        for (int k = 2; k <= n2; k <<= 1)
            for (int j = k >> 1; j > 0; j >>= 1) {
                for (int t = lane; t < (n2 >> 1); t += 32) {
                    const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));      // lower index of pair t at distance j
                    const int x = buf[w][i], y = buf[w][i + j];
                    if ((x > y) == ((i & k) == 0)) {
                        buf[w][i] = y;
                        buf[w][i + j] = x;
                    }
                }
                __syncwarp();
            }
        for (int i = lane; i < m; i += 32) {
            const int v = buf[w][i];
            perm[a + i] = v;
            gather_one(ga, a + i, v);
        }
        continue;
    }
    for (long long i = a + lane; i < b; i += 32) {
        const int v = unsorted[i];
        int rank = 0;
        for (long long j = a; j < b; ++j) rank += unsorted[j] < v;
        perm[a + rank] = v;
    }
    __syncwarp();                                      // the leaf's perm is complete (and `unsorted` no longer read)
    for (long long i = a + lane; i < b; i += 32) gather_one(ga, i, perm[i]);
    }   // leaves
}


// ------------------------------------------------------------------------------------------------
// translation tables for order p (q = p + 1 coefficients), built once per call on the device:
//   Cb[n][l]   = C(n + l, l)                                    (real, q x q)          -- M2L
//   S(c; k, m) = C(k, m) delta_c^(k-m) 2^-m   (m <= k, else 0)  (complex, 4 x q x q)   -- M2M, child c -> parent, output k
//   T(c; k, m) = 2^-k C(m, k) delta_c^(m-k)   (m >= k, else 0)  (complex, 4 x q x q)   -- L2L, parent -> child c, output k
//   both stored [c][m][k], the OUTPUT index fastest: the lanes of a warp own consecutive k and read consecutive words
//   rho[t][n]  = tau_t^-n, n = 0 .. q;  lrho[t] = log(1/tau_t)  (complex, 49 offsets tau = dx + i dy, |dx|,|dy| <= 3)
//   coef[t][5][q]: the per-offset factors of fmm_m2l_half, one load each instead of a few operations per source:
//     [0][k] = rho^k / k (k >= 1), 1 (k = 0)   [1][k] = rho^k        (scaling of the source's moments)
//     [2][l] = -(-1)^l rho^l (l >= 1), -1 (l = 0)      [3][l] = [2][l] / l (l >= 1), -lrho (l = 0)      [4][l] = (-1)^l rho^(l+1)
// delta_c = ((a - 1/2) + i (b - 1/2)) / 2 is the child's centre in the parent's scaled variable, c = 2 a + b.
constexpr int kTableBlocks = 32;        // of 256 threads (fmm_load's block size)
constexpr int kLogTabBlocks = 4;
struct FmmTables {
    double *Cb;
    cplx *S, *T, *rho, *lrho, *coef;
};
__host__ __device__ inline size_t fmm_tables_doubles(int q) { return (((size_t)q * q + 1) & ~(size_t)1) + 2 * (size_t)(8 * q * q) + 2 * (size_t)(49 * (q + 1)) + 2 * 49 + 2 * (size_t)(49 * 5 * q); }
__host__ __device__ inline FmmTables fmm_tables_at(double *base, int q)
{
    FmmTables t;
    t.Cb = base;
    t.S = (cplx *)(base + (((size_t)q * q + 1) & ~(size_t)1));   // 16-byte aligned
    t.T = t.S + 4 * q * q;
    t.rho = t.T + 4 * q * q;
    t.lrho = t.rho + 49 * (q + 1);
    t.coef = t.lrho + 49;
    return t;
}
__device__ __forceinline__ double binom(int n, int l)
{
    if (l < 0 || l > n) return 0.0;
    double r = 1.0;
    for (int i = 1; i <= l; ++i) r = r * (double)(n - l + i) / (double)i;
    return r;
}
__device__ __forceinline__ cplx cpowi(cplx a, int n)
{
    cplx r = make_double2(1.0, 0.0);
    for (int i = 0; i < n; ++i) r = cmul(r, a);
    return r;
}
// Run by kTableBlocks (+ kLogTabBlocks) extra blocks of fmm_load -- the tables depend on the order only, so they
// are built beside the first pass over the points instead of in a launch of their own; `block` counts from 0.
// Blocks beyond kTableBlocks (present only when logtab is wanted: double-precision storage) build the two tables
// of log_rcp_f64 in global memory, which every block of the direct part copies to its shared memory.
__device__ void fmm_build_tables(int block, int q, double *base, double *logtab)
{
    if (block >= kTableBlocks) {
        build_log_tables(logtab, (block - kTableBlocks) * blockDim.x + threadIdx.x, kLogTabBlocks * blockDim.x);
        return;
    }
    const FmmTables t = fmm_tables_at(base, q);
    const int nthreads = kTableBlocks * blockDim.x, tid = block * blockDim.x + threadIdx.x;
    for (int e = tid; e < q * q; e += nthreads) {
        const int n = e / q, l = e % q;
        t.Cb[e] = binom(n + l, l);
    }
    for (int e = tid; e < 4 * q * q; e += nthreads) {
        const int c = e / (q * q), k = (e / q) % q, m = e % q;
        const cplx d = make_double2(0.5 * ((double)(c >> 1) - 0.5), 0.5 * ((double)(c & 1) - 0.5));
        cplx s = make_double2(0.0, 0.0), u = make_double2(0.0, 0.0);
        if (m <= k) s = cscale(cpowi(d, k - m), binom(k, m) * exp2(-(double)m));       // S[c][k][m]
        if (k <= m) u = cscale(cpowi(d, m - k), binom(m, k) * exp2(-(double)k));       // T[c][k][m]: row = child index k
        t.S[((size_t)c * q + m) * q + k] = s;
        t.T[((size_t)c * q + m) * q + k] = u;
    }
    for (int e = tid; e < 49 * (q + 1); e += nthreads) {
        const int o = e / (q + 1), n = e % (q + 1);
        const cplx tau = make_double2((double)(o / 7 - 3), (double)(o % 7 - 3));
        cplx r = make_double2(0.0, 0.0);
        if (tau.x != 0.0 || tau.y != 0.0) r = cpowi(crcp(tau), n);
        t.rho[e] = r;
        cplx lr = make_double2(0.0, 0.0);
        if (tau.x != 0.0 || tau.y != 0.0) lr = make_double2(-0.5 * log(tau.x * tau.x + tau.y * tau.y), -atan2(tau.y, tau.x));
        if (n == 0) t.lrho[o] = lr;
        if (n < q) {
            const double sg = (n & 1) ? -1.0 : 1.0, in = n > 0 ? 1.0 / (double)n : 0.0;
            cplx rn1 = make_double2(0.0, 0.0);                      // rho^(n+1)
            if (tau.x != 0.0 || tau.y != 0.0) rn1 = cmul(r, crcp(tau));
            cplx *c = t.coef + (size_t)o * 5 * q;
            c[0 * q + n] = n > 0 ? cscale(r, in) : make_double2(1.0, 0.0);
            c[1 * q + n] = r;
            c[2 * q + n] = n > 0 ? cscale(r, -sg) : make_double2(-1.0, 0.0);
            c[3 * q + n] = n > 0 ? cscale(r, -sg * in) : make_double2(-lr.x, -lr.y);
            c[4 * q + n] = cscale(rn1, sg);
        }
    }
}

// expansions: [box][3][q] complex, boxes of level l start at (4^l - 1)/3; index inside a level ix * 2^l + iy
__host__ __device__ inline long long level_offset(int l) { return ((1ll << (2 * l)) - 1) / 3; }

// ------------------------------------------------------------------------------------------------
// P2M: moments about the box centre in the scaled variable w = (zeta - c)/s:
//   A1_k = sum g_x w^k,  A2_k = sum g_y w^k,  B_k = sum conj(zeta) g w^k.
constexpr int kFmmMaxQ = 49;          // p <= 48
// One warp per leaf box, no shuffles (a reduction of every power over the lanes costs 60 shuffles per coefficient and
// 32 sources): the sum runs the other way round: for 32 sources at a time lane j writes 16 consecutive powers of
// ITS source into the warp's shared memory (row stride 17 sixteen-byte words: conflict-free both ways), then lane
// (half, k) adds up coefficient 16 g + k over the sources j = half, half + 2, ... -- a 16-byte load of the power and
// two broadcasts (g, conj(zeta) g) per 8 DFMA -- group g = 0 .. ceil(q / 16) - 1 after group, the power recurrence
// carried on in a register; the two halves meet once per leaf.
constexpr int kP2MWarps = 4;
constexpr int kP2MGroups = (kFmmMaxQ + 15) / 16;       // 4
__global__ void __launch_bounds__(32 * kP2MWarps)
fmm_p2m(const cplx *__restrict__ zs, const cplx *__restrict__ gs, const long long *__restrict__ start, int q,
             const unsigned long long *__restrict__ enc, cplx *__restrict__ mult, int *__restrict__ boxcnt)
{
    const int L = load_level(enc);
    constexpr int stride = 17;
    __shared__ cplx pws[kP2MWarps][32 * stride + 64];                 // [32][17] powers | [32] g | [32] conj(zeta) g
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, half = lane >> 4, k = lane & 15;
    cplx *pw = pws[warp], *sg = pw + 32 * stride, *sh = sg + 32;
    const int n = 1 << L, ncell = n * n;
    const Geom gm = load_geom(enc);
    const double s = gm.size / (double)n, inv_s = 1.0 / s;
    const int ng = (q + 15) >> 4;
    for (int c = blockIdx.x * kP2MWarps + warp; c < ncell; c += gridDim.x * kP2MWarps) {
        const long long a = start[c], b = start[c + 1];
        if (lane == 0) boxcnt[level_offset(L) + c] = (int)(b - a);
        cplx *out = mult + (level_offset(L) + c) * (long long)(3 * q);
        if (a == b) {                                                // the upper levels read the moments of empty leaves too
            for (int e = lane; e < 3 * q; e += 32) out[e] = make_double2(0.0, 0.0);
            continue;
        }
        const cplx ctr = box_centre(gm, L, c / n, c % n);
        cplx a1[kP2MGroups], a2[kP2MGroups], bb[kP2MGroups];         // A1, A2, B of coefficient 16 g + k (this half's sources)
#pragma unroll
        for (int g = 0; g < kP2MGroups; ++g) a1[g] = a2[g] = bb[g] = make_double2(0.0, 0.0);
        for (long long base = a; base < b; base += 32) {
            const long long idx = base + lane;
            const int cnt = (int)min(32ll, b - base);
            cplx w = make_double2(0.0, 0.0), p = make_double2(1.0, 0.0);
            __syncwarp();                                            // the previous 32 sources are consumed
            if (idx < b) {
                const cplx zt = zs[idx], g = gs[idx];
                w = make_double2((zt.x - ctr.x) * inv_s, (zt.y - ctr.y) * inv_s);
                sg[lane] = g;
                sh[lane] = cmul(make_double2(zt.x, -zt.y), g);      // conj(zeta) g
            }
#pragma unroll
            for (int g = 0; g < kP2MGroups; ++g) {
                if (g < ng) {
                    if (g > 0) __syncwarp();                         // the previous group's powers are consumed
                    cplx *row = pw + lane * stride;
#pragma unroll 4
                    for (int kk = 0; kk < 16; ++kk) {
                        row[kk] = p;
                        p = cmul(p, w);
                    }
                    __syncwarp();
                    if (16 * g + k < q) {
#pragma unroll 4
                        for (int j = half; j < cnt; j += 2) {
                            const cplx pp = pw[j * stride + k], g2 = sg[j], h = sh[j];
                            a1[g].x = fma(g2.x, pp.x, a1[g].x); a1[g].y = fma(g2.x, pp.y, a1[g].y);
                            a2[g].x = fma(g2.y, pp.x, a2[g].x); a2[g].y = fma(g2.y, pp.y, a2[g].y);
                            bb[g] = cfma(h, pp, bb[g]);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int g = 0; g < kP2MGroups; ++g) {
            if (g < ng) {
                cplx x1 = a1[g], x2 = a2[g], xb = bb[g];
                x1.x += __shfl_xor_sync(0xffffffffu, x1.x, 16); x1.y += __shfl_xor_sync(0xffffffffu, x1.y, 16);
                x2.x += __shfl_xor_sync(0xffffffffu, x2.x, 16); x2.y += __shfl_xor_sync(0xffffffffu, x2.y, 16);
                xb.x += __shfl_xor_sync(0xffffffffu, xb.x, 16); xb.y += __shfl_xor_sync(0xffffffffu, xb.y, 16);
                const int kq = 16 * g + k;
                if (kq < q && half == 0) {
                    out[kq] = x1;
                    out[q + kq] = x2;
                    out[2 * q + kq] = xb;
                }
            }
        }
    }
}

// M2M: parent moments from its four children, levels L-1 down to 2.  One BLOCK per parent box (grid-stride): the
// children's moments are staged in shared memory with coalesced loads (one round trip to L2 instead of one per term),
// then thread (c, a, k) -- child c, expansion a, output coefficient k: 12 q work items -- sums S(c; k, m) A_c,a[m]
// over m <= k, and q threads per expansion add the four children's parts.  The upper levels have a handful of boxes:
// what counts there is how little one thread does in a row, not the instruction total.
constexpr int kShiftThreads = 192;        // 12 q = 180 work items at q = 15
constexpr int kShiftStageQ = 49;     // = kFmmMaxQ: always (172 KB of dynamic shared memory at the largest order, opted into below)
#ifndef VN_FMM_SHIFT_WAVE
#define VN_FMM_SHIFT_WAVE 4
#endif
constexpr unsigned kShiftWave = VN_FMM_SHIFT_WAVE;   // blocks per SM of the single-level launches (grid-stride over the boxes)
// dst[e] = src[e], e = first, first + stride, ... < count, with eight loads in flight per thread: written as
// dst[e] = src[e] in a loop, every load waits for the previous store (the compiler cannot rule out aliasing), and
// the kernels of the small upper levels are nothing but such latencies in a row
// (loads go to L2, not through L1: the multi-level launches read what other blocks wrote earlier in the same launch)
__device__ __forceinline__ cplx ldcg_cplx(const cplx *p) { return __ldcg(p); }
__device__ __forceinline__ void stage_cplx(cplx *dst, const cplx *src, int first, int stride, int count)
{
    for (int e0 = first; e0 < count; e0 += 8 * stride) {
        cplx tmp[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int e = e0 + i * stride;
            if (e < count) tmp[i] = ldcg_cplx(src + e);
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int e = e0 + i * stride;
            if (e < count) dst[e] = tmp[i];
        }
    }
}
// Several levels in ONE launch: the levels below the top two have a few hundred boxes at most, a launch each is mostly
// launch latency.  All blocks of the grid meet at a counter between two levels; the host sizes such a grid so that
// every block is resident (occupancy query), otherwise the blocks that spin would wait for blocks that cannot start.
__device__ __forceinline__ void grid_barrier(unsigned long long *counter, unsigned long long target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(counter, 1ull);
        while (*(volatile unsigned long long *)counter < target) { }
        __threadfence();
    }
    __syncthreads();
}
constexpr int kM2MPre = (12 * kFmmMaxQ + kShiftThreads - 1) / kShiftThreads;   // children's coefficients per thread
__device__ __forceinline__ void m2m_prefetch(cplx (&pre)[kM2MPre], int &pre_cnt, int box, int nn, int n, int level, int q,
                                             int tid, const cplx *mult, const int *boxcnt)
{
    if (box >= nn) return;
    const int ix = box / n, iy = box % n;
    const long long child0 = level_offset(level + 1) + (long long)(2 * ix) * (2 * n) + 2 * iy;   // child c = 2 a + b at child0 + a * 2n + b
#pragma unroll
    for (int r = 0; r < kM2MPre; ++r) {
        const int e = min(tid + r * kShiftThreads, 12 * q - 1);     // surplus slots reload the last element (never stored)
        const int c = e / (3 * q);
        pre[r] = ldcg_cplx(mult + (child0 + (long long)(c >> 1) * (2 * n) + (c & 1)) * (long long)(3 * q) + (e - c * 3 * q));
    }
    if (tid < 4) pre_cnt = __ldcg(boxcnt + child0 + (long long)(tid >> 1) * (2 * n) + (tid & 1));
}
__device__ __forceinline__ void m2m_commit(const cplx (&pre)[kM2MPre], int pre_cnt, int q, int tid, cplx *ch, int *scnt)
{   // the prefetched box becomes the current one
#pragma unroll
    for (int r = 0; r < kM2MPre; ++r) {
        const int e = tid + r * kShiftThreads;
        if (e < 12 * q) ch[e] = pre[r];
    }
    if (tid < 4) scnt[tid] = pre_cnt;
}
// levels L - d_first, L - d_first - 1, ..., max(L - d_last, 2)  (L = the tree's depth, chosen on the device)
__global__ void __launch_bounds__(kShiftThreads)
fmm_m2m(int d_first, int d_last, int q, const double *__restrict__ tab, unsigned long long *enc,
        cplx *mult, int *boxcnt)
{
    const int L = load_level(enc);
    extern __shared__ __align__(16) double sm[];
    cplx *ch = (cplx *)sm;                                           // [4][3][q] children's moments
    cplx *part = ch + 12 * q;                                        // [4][3][q] their contributions to the parent
    __shared__ int scnt[4];
    const FmmTables t = fmm_tables_at(const_cast<double *>(tab), q);
    if (L - d_first < 2) return;                                     // nothing to do (uniform over the grid)
    // the table: in shared memory up to kShiftStageQ (every launch starts with a cold L1: read through it, the
    // loads of a work item would each wait for L2), straight from global memory above
    const cplx *Stab = t.S;
    if (q <= kShiftStageQ) {
        cplx *st = part + 12 * q;
        stage_cplx(st, t.S, threadIdx.x, blockDim.x, 4 * q * q);
        Stab = st;
    }
    const int tid = threadIdx.x;
    unsigned long long arrivals = 0;
    for (int level = L - d_first; level >= 2 && level >= L - d_last; --level) {
    if (level != L - d_first) grid_barrier(enc + 9, arrivals += gridDim.x);   // the level below is complete
    const int n = 1 << level, nn = n * n;
    // The block's boxes one after the other, the NEXT box's children (and their counts) in flight while this one is
    // computed: per box two barriers and no exposed round trip to L2 (the first version waited for the counts, then
    // for the children, then wrote: 2.6 us per box, 18 us for the 4,096 parents above a million points' leaves).
    // Children without sources hold zero moments (fmm_p2m and this kernel write them): all four are always loaded.
    cplx pre[kM2MPre] = {};
    int pre_cnt = 0;
    __syncthreads();                                                 // the previous level's last box is written out
    m2m_prefetch(pre, pre_cnt, blockIdx.x, nn, n, level, q, tid, mult, boxcnt);
    m2m_commit(pre, pre_cnt, q, tid, ch, scnt);
    __syncthreads();
    for (int box = blockIdx.x; box < nn; box += gridDim.x) {
        m2m_prefetch(pre, pre_cnt, box + gridDim.x, nn, n, level, q, tid, mult, boxcnt);
        for (int w = tid; w < 12 * q; w += kShiftThreads) {
            const int c = w / (3 * q), k = w % q;                    // w = (c * 3 + a) * q + k
            cplx s0 = make_double2(0.0, 0.0), s1 = s0;               // two chains: even and odd m
            if (scnt[c] != 0) {                                      // a child without sources adds nothing (a 4:1 channel: most)
                const cplx *A = ch + (w - k);
                const cplx *col = Stab + (size_t)c * q * q + k;
                int m = 0;
                for (; m + 1 <= k; m += 2) {
                    s0 = cfma(col[(size_t)m * q], A[m], s0);
                    s1 = cfma(col[(size_t)(m + 1) * q], A[m + 1], s1);
                }
                if (m <= k) s0 = cfma(col[(size_t)m * q], A[m], s0);
            }
            part[w] = cadd(s0, s1);
        }
        const int cnt_box = scnt[0] + scnt[1] + scnt[2] + scnt[3];
        __syncthreads();                                             // part is complete, ch and scnt are consumed
        cplx *out = mult + (level_offset(level) + box) * (long long)(3 * q);
        for (int e = tid; e < 3 * q; e += kShiftThreads)
            out[e] = cadd(cadd(part[e], part[3 * q + e]), cadd(part[6 * q + e], part[9 * q + e]));
        if (tid == 0) boxcnt[level_offset(level) + box] = cnt_box;
        m2m_commit(pre, pre_cnt, q, tid, ch, scnt);
        __syncthreads();                                             // ch holds the next box, part is consumed
    }
    }   // levels
}
static size_t shift_smem(int q);
__global__ void fmm_l2l(int d_hi, int d_lo, int q, const double *__restrict__ tab, unsigned long long *enc,
                        const int *__restrict__ tboxcnt, cplx *loc);
// blocks of the multi-level launches of fmm_m2m / fmm_l2l: all resident at once (see grid_barrier), at most two per SM
static int shift_resident_blocks(int q)
{
    static int q_dev[kMaxDevices] = {0}, blocks_dev[kMaxDevices] = {0};
    const int d = current_device();
    if (q_dev[d] != q || blocks_dev[d] == 0) {
        int dev = 0, sms = 0, o1 = 0, o2 = 0;
        const int max_smem = (int)shift_smem(kFmmMaxQ);              // the table in shared memory at any order: beyond 48 KB
        if (cudaFuncSetAttribute(fmm_m2m, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem) != cudaSuccess ||
            cudaFuncSetAttribute(fmm_l2l, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem) != cudaSuccess ||
            cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o1, fmm_m2m, kShiftThreads, shift_smem(q)) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o2, fmm_l2l, kShiftThreads, shift_smem(q)) != cudaSuccess) {
            (void)cudaGetLastError();
            return 1;                                  // a single block needs nobody else to be resident
        }
        const int occ = o1 < o2 ? o1 : o2;
        blocks_dev[d] = occ < 1 ? 1 : sms * (occ < 2 ? occ : 2);
        q_dev[d] = q;
    }
    return blocks_dev[d];
}
// The multi-level launches go through the cooperative-launch attribute: the driver then starts the grid only when all
// of its blocks fit at once -- also next to kernels of other streams -- which is what grid_barrier needs (a plain
// launch of a correctly sized grid is safe only as long as nothing else occupies the device).
template <typename... Params, typename... Args>
static cudaError_t launch_resident(void (*kernel)(Params...), int blocks, size_t smem, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks);
    cfg.blockDim = dim3(kShiftThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<Params>(args)...);
}
static size_t shift_smem(int q) { return sizeof(cplx) * (size_t)(24 * q + (q <= kShiftStageQ ? 4 * q * q : 0)); }

// ------------------------------------------------------------------------------------------------
// M2L: one WARP per target box of `level` (four boxes per block), no block barrier inside the loop.  Lane `ln` owns
// the coefficients l = ln and ln + 32 of all three local expansions (0, 1: the logarithmic potentials Phi1, Phi2;
// 2: the Cauchy sum psi).  For every box of the interaction list (children of the parent's neighbours that are
// not neighbours of the target; offset tau = target - source in box units, rho = 1/tau):
//   Ahat_k = A_k rho^k / k (k >= 1, log type)      Bhat_k = B_k rho^k (k >= 0)        (staged in the warp's shared memory)
//   b_l += (-1)^(l+1) rho^l ( A_0 / l + sum_{k>=1} C(k+l-1, l) Ahat_k )          l >= 1
//   b_0 += A_0 (log s - log rho) - sum_{k>=1} Ahat_k
//   d_l += (-1)^l rho^(l+1) / s * sum_{k>=0} C(k+l, l) Bhat_k ;   d_0 -= conj(A1_0 + i A2_0)   (the g/2 of each source)
// so the inner loop is a REAL binomial matrix (shared memory, same for every offset and level) times complex
// vectors: one matrix entry serves all three expansions (6 DFMA per 8-byte load + 3 broadcasts).
constexpr int kM2LWarps = 4;
__global__ void __launch_bounds__(32 * kM2LWarps)
fmm_m2l(int q, const double *__restrict__ tab, const unsigned long long *__restrict__ enc,
        const cplx *__restrict__ mult, const int *__restrict__ boxcnt, const int *__restrict__ tboxcnt,
        cplx *__restrict__ loc)
{   // tboxcnt: population of the TARGET boxes (the sources' own counts for vn_farfield_fmm; nullptr when the targets
    // are a separate set and every box may hold some): a box without targets needs no local expansion -- in a 4:1
    // channel three quarters of the root square's boxes are empty.
    // The boxes of ALL levels 2 .. L in one launch, deepest level first, and the interaction list built by the lanes
    // in parallel, as in fmm_m2l_half below.  Coefficients 32 .. q - 1 (q > 32: a few lanes' second coefficient) are
    // not carried through the loop by every lane -- half of its DFMAs would multiply padding -- but summed afterwards
    // by (coefficient, quarter of the k range) work items and met through shared memory.
    const int L = load_level(enc);
    extern __shared__ __align__(16) double sm[];
    double *Cb = sm;                                                  // [q][q]
    const int warp = threadIdx.x >> 5, ln = threadIdx.x & 31;
    cplx *hat = (cplx *)(sm + ((q * q + 1) & ~1)) + warp * (3 * (q + 1) + 96);   // [3][q+1] per warp; hat[a][q] = 0 pads the shifted read
    cplx *red = hat + 3 * (q + 1);                                    // [32][3] partial sums of the coefficients >= 32
    int *list = (int *)((cplx *)(sm + ((q * q + 1) & ~1)) + kM2LWarps * (3 * (q + 1) + 96)) + warp * 32;
    const FmmTables t = fmm_tables_at(const_cast<double *>(tab), q);
    for (int e = threadIdx.x; e < q * q; e += blockDim.x) Cb[e] = t.Cb[e];
    __syncthreads();
    const Geom gm = load_geom(enc);
    const double log_size = log(gm.size);
    const int l0 = ln, l1 = ln + 32;
    const bool v0 = l0 < q, v1 = l1 < q;
    const int nb = q > 32 ? q - 32 : 0, nchunk = nb ? 32 / nb : 0, kper = nb ? (q + nchunk - 1) / nchunk : 0;
    const long long total = level_offset(L + 1) - level_offset(2);
    for (long long gi = (long long)blockIdx.x * kM2LWarps + warp; gi < total; gi += (long long)gridDim.x * kM2LWarps) {
    int level = L;
    long long rem = gi;
    while (rem >= (1ll << (2 * level))) { rem -= 1ll << (2 * level); --level; }
    const int box = (int)rem, n = 1 << level;
    const double s = gm.size / (double)n, log_s = fma(-(double)level, 0.693147180559945309417, log_size);
    const long long lev0 = level_offset(level);
    if (tboxcnt && tboxcnt[lev0 + box] == 0) continue;
    const int ix = box / n, iy = box % n, px = ix >> 1, py = iy >> 1;
    __syncwarp();
    int nlist = 0;
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int e = ln + 32 * r;
        bool ok = false;
        int entry = 0;
        if (e < 36) {
            const int sx = 2 * (px - 1) + e / 6, sy = 2 * (py - 1) + e % 6;
            if (sx >= 0 && sx < n && sy >= 0 && sy < n && !(abs(sx - ix) <= 1 && abs(sy - iy) <= 1)) {
                const int src = sx * n + sy;
                ok = boxcnt[lev0 + src] != 0;
                entry = src | (((ix - sx + 3) * 7 + (iy - sy + 3)) << 24);
            }
        }
        const unsigned m = __ballot_sync(0xffffffffu, ok);
        if (ok) list[nlist + __popc(m & ((1u << ln) - 1u))] = entry;
        nlist += __popc(m);
    }
    __syncwarp();
    cplx acc[3][2];
#pragma unroll
    for (int a = 0; a < 3; ++a) acc[a][0] = acc[a][1] = make_double2(0.0, 0.0);
    const cplx *Mlev = mult + lev0 * (long long)(3 * q);
    for (int i = 0; i < nlist; ++i) {
            const int entry = list[i];
            const int o = entry >> 24;
            const cplx *rho = t.rho + (size_t)o * (q + 1);
            const cplx *A = Mlev + (long long)(entry & 0xffffff) * (3 * q);
            __syncwarp();                                             // the previous source's hat and red are consumed
            for (int k = ln; k <= q; k += 32) {
                cplx h0 = make_double2(0.0, 0.0), h1 = h0, h2 = h0;
                if (k < q) {
                    const cplx r = rho[k];
                    h0 = cmul(A[k], r);
                    h1 = cmul(A[q + k], r);
                    h2 = cmul(A[2 * q + k], r);
                    if (k >= 1) { const double ik = 1.0 / (double)k; h0 = cscale(h0, ik); h1 = cscale(h1, ik); }
                }
                hat[k] = h0;
                hat[(q + 1) + k] = h1;
                hat[2 * (q + 1) + k] = h2;
            }
            __syncwarp();
            const cplx A10 = A[0], A20 = A[q];                       // raw zeroth moments (real charges: imaginary part 0)
            cplx S[3][2];
#pragma unroll
            for (int a = 0; a < 3; ++a) S[a][0] = S[a][1] = make_double2(0.0, 0.0);
            const cplx *h0p = hat + 1, *h1p = hat + (q + 1) + 1, *h2p = hat + 2 * (q + 1);   // log arrays read k + 1
            {
                const double *Cl = Cb + (v0 ? l0 : 0);
#pragma unroll 4
                for (int k = 0; k < q; ++k) {
                    const double c0 = Cl[k * q];
                    const cplx e0 = h0p[k], e1 = h1p[k], e2 = h2p[k];     // Ahat1_{k+1}, Ahat2_{k+1}, Bhat_k
                    S[0][0].x = fma(c0, e0.x, S[0][0].x); S[0][0].y = fma(c0, e0.y, S[0][0].y);
                    S[1][0].x = fma(c0, e1.x, S[1][0].x); S[1][0].y = fma(c0, e1.y, S[1][0].y);
                    S[2][0].x = fma(c0, e2.x, S[2][0].x); S[2][0].y = fma(c0, e2.y, S[2][0].y);
                }
            }
            if (nb) {                                                 // coefficients 32 .. q - 1: item (coefficient j, chunk c of the k range)
                cplx T0 = make_double2(0.0, 0.0), T1 = T0, T2 = T0;
                if (ln < nchunk * nb) {
                    const int c = ln / nb, j = ln - c * nb;
                    const double *Cl = Cb + 32 + j;
                    const int k1 = min(q, (c + 1) * kper);
                    for (int k = c * kper; k < k1; ++k) {
                        const double c1 = Cl[k * q];
                        const cplx e0 = h0p[k], e1 = h1p[k], e2 = h2p[k];
                        T0.x = fma(c1, e0.x, T0.x); T0.y = fma(c1, e0.y, T0.y);
                        T1.x = fma(c1, e1.x, T1.x); T1.y = fma(c1, e1.y, T1.y);
                        T2.x = fma(c1, e2.x, T2.x); T2.y = fma(c1, e2.y, T2.y);
                    }
                }
                red[ln * 3 + 0] = T0;
                red[ln * 3 + 1] = T1;
                red[ln * 3 + 2] = T2;
                __syncwarp();
                if (v1)
                    for (int c = 0; c < nchunk; ++c) {
                        const cplx *pr = red + (ln + c * nb) * 3;
                        S[0][1] = cadd(S[0][1], pr[0]);
                        S[1][1] = cadd(S[1][1], pr[1]);
                        S[2][1] = cadd(S[2][1], pr[2]);
                    }
            }
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int l = j ? l1 : l0;
                if (!(j ? v1 : v0)) continue;
                const double sgn = (l & 1) ? -1.0 : 1.0;              // (-1)^l
                if (l == 0) {
                    const cplx lr = t.lrho[o];
                    acc[0][j] = cadd(acc[0][j], make_double2(A10.x * (log_s - lr.x) + A10.y * lr.y - S[0][j].x,
                                                             -A10.x * lr.y + A10.y * (log_s - lr.x) - S[0][j].y));
                    acc[1][j] = cadd(acc[1][j], make_double2(A20.x * (log_s - lr.x) + A20.y * lr.y - S[1][j].x,
                                                             -A20.x * lr.y + A20.y * (log_s - lr.x) - S[1][j].y));
                } else {
                    const double il = 1.0 / (double)l;
                    acc[0][j] = cadd(acc[0][j], cscale(cmul(rho[l], cadd(cscale(A10, il), S[0][j])), -sgn));
                    acc[1][j] = cadd(acc[1][j], cscale(cmul(rho[l], cadd(cscale(A20, il), S[1][j])), -sgn));
                }
                acc[2][j] = cadd(acc[2][j], cscale(cmul(rho[l + 1], S[2][j]), sgn / s));
                if (l == 0) acc[2][j] = cadd(acc[2][j], make_double2(-(A10.x - A20.y), A10.y + A20.x));   // -conj(A1_0 + i A2_0)
            }
        }
    cplx *out = loc + (lev0 + box) * (long long)(3 * q);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (v0) out[a * q + l0] = acc[a][0];
        if (v1) out[a * q + l1] = acc[a][1];
    }
    __syncwarp();
    }   // boxes
}
static size_t m2l_smem(int q)
{
    return sizeof(double) * (size_t)((q * q + 1) & ~1) + sizeof(cplx) * (size_t)(kM2LWarps * (3 * (q + 1) + 96)) +
           sizeof(int) * (size_t)(kM2LWarps * 32);
}

// M2L for q <= 16 (orders up to 15: the defaults, 12 in double and 14 in single precision, live here).  fmm_m2l gives
// a lane the coefficients l and l + 32: with q = 15 half of its DFMAs multiply padding and 17 of 32 lanes carry
// none.  Here a HALF-warp owns a source box -- lane = (half, l), two sources of the interaction list in flight per warp --
// and three more things change: the list (up to 27 non-empty boxes of the 6 x 6 parent-neighbour region) is built by the
// lanes in parallel (one round of boxcnt loads instead of 27 dependent ones), the next pair's moments are fetched into
// registers before the current pair's matrix-vector loop (the L2 latency of a source box hides behind the previous
// one's arithmetic), and the two halves' sums meet in one shuffle at the end.  Same formulas as fmm_m2l; the order in
// which the sources are added differs (fixed, so the result is still reproducible run to run).
constexpr int kM2LHalfQ = 16;
#ifndef VN_FMM_M2L_MINBLK
#define VN_FMM_M2L_MINBLK 4
#endif
__global__ void __launch_bounds__(32 * kM2LWarps, VN_FMM_M2L_MINBLK)
fmm_m2l_half(int q, const double *__restrict__ tab, const unsigned long long *__restrict__ enc,
             const cplx *__restrict__ mult, const int *__restrict__ boxcnt, const int *__restrict__ tboxcnt,
             cplx *__restrict__ loc)
{
    const int L = load_level(enc);
    extern __shared__ __align__(16) double sm[];
    double *Cb = sm;                                                  // [q][q]
    const int warp = threadIdx.x >> 5, ln = threadIdx.x & 31, half = ln >> 4, l = ln & 15;
    const int hstride = 3 * (q + 1) + 1;                              // odd number of 16-byte words: the halves' broadcasts fall in different banks
    cplx *hat = (cplx *)(sm + ((q * q + 1) & ~1)) + (warp * 2 + half) * hstride;   // [3][q+1] per half; hat[a][q] = 0 pads the shifted read
    int *list = (int *)((cplx *)(sm + ((q * q + 1) & ~1)) + kM2LWarps * 2 * hstride) + warp * 32;
    const FmmTables t = fmm_tables_at(const_cast<double *>(tab), q);
    for (int e = threadIdx.x; e < q * q; e += blockDim.x) Cb[e] = t.Cb[e];
    if (l < 3) hat[l * (q + 1) + q] = make_double2(0.0, 0.0);
    __syncthreads();
    const Geom gm = load_geom(enc);
    const double log_size = log(gm.size);
    const bool v = l < q;
    const int lv = v ? l : 0;                                        // lanes beyond q compute column 0 and store nothing
    // the boxes of ALL levels 2 .. L in one launch, deepest level first (M2L of a level needs the multipoles only, not
    // the other levels' local expansions; L2L adds the parents' afterwards): the small upper levels overlap with the
    // tail of the deepest one instead of costing a launch each
    const long long total = level_offset(L + 1) - level_offset(2);
    for (long long gi = (long long)blockIdx.x * kM2LWarps + warp; gi < total; gi += (long long)gridDim.x * kM2LWarps) {
        int level = L;
        long long rem = gi;
        while (rem >= (1ll << (2 * level))) { rem -= 1ll << (2 * level); --level; }
        const int box = (int)rem, n = 1 << level;
        const double s = gm.size / (double)n, inv_s = 1.0 / s, log_s = fma(-(double)level, 0.693147180559945309417, log_size);
        const long long lev0 = level_offset(level);
        const cplx *Mlev = mult + lev0 * (long long)(3 * q);
        if (tboxcnt && tboxcnt[lev0 + box] == 0) continue;
        const int ix = box / n, iy = box % n, px = ix >> 1, py = iy >> 1;
        // interaction list: children of the parent's neighbours that are not neighbours of the box and hold sources
        __syncwarp();
        int nlist = 0;
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            const int e = ln + 32 * r;
            bool ok = false;
            int entry = 0;
            if (e < 36) {
                const int sx = 2 * (px - 1) + e / 6, sy = 2 * (py - 1) + e % 6;
                if (sx >= 0 && sx < n && sy >= 0 && sy < n && !(abs(sx - ix) <= 1 && abs(sy - iy) <= 1)) {
                    const int src = sx * n + sy;
                    ok = boxcnt[lev0 + src] != 0;
                    entry = src | (((ix - sx + 3) * 7 + (iy - sy + 3)) << 24);
                }
            }
            const unsigned m = __ballot_sync(0xffffffffu, ok);
            if (ok) list[nlist + __popc(m & ((1u << ln) - 1u))] = entry;
            nlist += __popc(m);
        }
        __syncwarp();
        cplx acc0 = make_double2(0.0, 0.0), acc1 = acc0, acc2 = acc0;
        cplx sumA1 = acc0, sumA2 = acc0;                               // zeroth moments of the half's sources, for the l = 0 terms
        // the half's next source: coefficient l of its three expansions and the two factors that scale them
        cplx a0, a1, a2, cpre, cpreB;
        const cplx *cf;
        auto fetch = [&](int idx) {
            a0 = a1 = a2 = make_double2(0.0, 0.0);
            int o = 24;                                                // tau = 0: all factors 0 or harmless, an absent source adds nothing
            const cplx *A = Mlev;
            if (idx < nlist) {
                const int entry = list[idx];
                o = entry >> 24;
                A = Mlev + (long long)(entry & 0xffffff) * (3 * q);
            }
            cf = t.coef + (size_t)o * 5 * q + lv;
            if (v && idx < nlist) {
                a0 = A[l];
                a1 = A[q + l];
                a2 = A[2 * q + l];
            }
            cpre = __ldg(cf);
            cpreB = __ldg(cf + q);
        };
        fetch(half);
        for (int i = 0; i < nlist; i += 2) {
            __syncwarp();                                             // the previous pair's hat is consumed
            if (v) {
                hat[l] = cmul(a0, cpre);                               // Ahat1_k = A1_k rho^k / k
                hat[(q + 1) + l] = cmul(a1, cpre);
                hat[2 * (q + 1) + l] = cmul(a2, cpreB);                // Bhat_k = B_k rho^k
            }
            const cplx cS = __ldg(cf + 2 * q), cA = __ldg(cf + 3 * q), c2 = __ldg(cf + 4 * q);   // used after the loop below
            fetch(i + 2 + half);                                      // in flight during the loop below
            __syncwarp();
            const cplx A10 = hat[0], A20 = hat[q + 1];                // rho^0 = 1: the raw zeroth moments
            cplx S0 = make_double2(0.0, 0.0), S1 = S0, S2 = S0;
            const cplx *h0p = hat + 1, *h1p = hat + (q + 1) + 1, *h2p = hat + 2 * (q + 1);   // log arrays read k + 1
            const double *Cl = Cb + lv;
#pragma unroll 5
            for (int k = 0; k < q; ++k) {
                const double c0 = Cl[k * q];
                const cplx e0 = h0p[k], e1 = h1p[k], e2 = h2p[k];     // Ahat1_{k+1}, Ahat2_{k+1}, Bhat_k
                S0.x = fma(c0, e0.x, S0.x); S0.y = fma(c0, e0.y, S0.y);
                S1.x = fma(c0, e1.x, S1.x); S1.y = fma(c0, e1.y, S1.y);
                S2.x = fma(c0, e2.x, S2.x); S2.y = fma(c0, e2.y, S2.y);
            }
            // b_l += cS (A_0 / l + S) for l >= 1, b_0 += A_0 (log s - log rho) - S: cA = cS / l resp. -log rho, the log s
            // part and the -conj(A1_0 + i A2_0) of d_0 follow from the sums of the zeroth moments once per box
            acc0 = cfma(cS, S0, cfma(cA, A10, acc0));
            acc1 = cfma(cS, S1, cfma(cA, A20, acc1));
            acc2 = cfma(c2, S2, acc2);
            sumA1 = cadd(sumA1, A10);
            sumA2 = cadd(sumA2, A20);
        }
        {
            const double z0 = l == 0 ? 1.0 : 0.0;                     // the l = 0 terms, without a branch
            acc0 = make_double2(fma(z0 * log_s, sumA1.x, acc0.x), fma(z0 * log_s, sumA1.y, acc0.y));
            acc1 = make_double2(fma(z0 * log_s, sumA2.x, acc1.x), fma(z0 * log_s, sumA2.y, acc1.y));
            acc2 = make_double2(fma(acc2.x, inv_s, -z0 * (sumA1.x - sumA2.y)), fma(acc2.y, inv_s, z0 * (sumA1.y + sumA2.x)));
        }
        // the two halves' sums
        acc0.x += __shfl_xor_sync(0xffffffffu, acc0.x, 16); acc0.y += __shfl_xor_sync(0xffffffffu, acc0.y, 16);
        acc1.x += __shfl_xor_sync(0xffffffffu, acc1.x, 16); acc1.y += __shfl_xor_sync(0xffffffffu, acc1.y, 16);
        acc2.x += __shfl_xor_sync(0xffffffffu, acc2.x, 16); acc2.y += __shfl_xor_sync(0xffffffffu, acc2.y, 16);
        if (v && half == 0) {
            cplx *out = loc + (lev0 + box) * (long long)(3 * q);
            out[l] = acc0;
            out[q + l] = acc1;
            out[2 * q + l] = acc2;
        }
    }   // boxes
}
static size_t m2l_half_smem(int q)
{
    return sizeof(double) * (size_t)((q * q + 1) & ~1) + sizeof(cplx) * (size_t)(kM2LWarps * 2 * (3 * (q + 1) + 1)) +
           sizeof(int) * (size_t)(kM2LWarps * 32);
}

// L2L: child local expansions inherit the parent's; child level = `level`.  One BLOCK per PARENT box (grid-stride):
// the parent's expansion is staged once for its four children, thread (c, a, k) -- child c, expansion a, output
// coefficient k -- adds sum_{m >= k} T(c; k, m) par_a[m] to the child's own M2L part.
// child levels max(3, L - d_hi), ..., L - d_lo  top-down, a grid barrier between two of them
__global__ void __launch_bounds__(kShiftThreads)
fmm_l2l(int d_hi, int d_lo, int q, const double *__restrict__ tab, unsigned long long *enc,
        const int *__restrict__ tboxcnt, cplx *loc)
{
    const int L = load_level(enc);
    const int l_first = max(3, L - d_hi), l_end = L - d_lo;
    if (l_first > l_end) return;
    extern __shared__ __align__(16) double sm[];
    cplx *par = (cplx *)sm;                                          // [3][q]
    __shared__ int scnt[4];
    const FmmTables t = fmm_tables_at(const_cast<double *>(tab), q);
    const cplx *Ttab = t.T;                                          // staged like the table of fmm_m2m
    if (q <= kShiftStageQ) {
        cplx *st = par + 24 * q;
        stage_cplx(st, t.T, threadIdx.x, blockDim.x, 4 * q * q);
        Ttab = st;
    }
    const int tid = threadIdx.x;
    unsigned long long arrivals = 0;
    for (int level = l_first; level <= l_end; ++level) {
    if (level != l_first) grid_barrier(enc + 10, arrivals += gridDim.x);      // the level above is complete
    const int n = 1 << level, np = n >> 1;
    for (int pbox = blockIdx.x; pbox < np * np; pbox += gridDim.x) {
        if (tboxcnt && tboxcnt[level_offset(level - 1) + pbox] == 0) continue;   // no targets below the parent (see fmm_m2l)
        const int px = pbox / np, py = pbox % np;
        const long long child0 = level_offset(level) + (long long)(2 * px) * n + 2 * py;
        __syncthreads();
        if (tid < 4) scnt[tid] = tboxcnt ? tboxcnt[child0 + (long long)(tid >> 1) * n + (tid & 1)] : 1;
        stage_cplx(par, loc + (level_offset(level - 1) + pbox) * (long long)(3 * q), tid, kShiftThreads, 3 * q);
        __syncthreads();
        for (int w = tid; w < 12 * q; w += kShiftThreads) {
            const int c = w / (3 * q), r = w - c * 3 * q, k = r % q;  // r = a * q + k
            if (scnt[c] == 0) continue;
            cplx *out = loc + (child0 + (long long)(c >> 1) * n + (c & 1)) * (long long)(3 * q) + r;
            cplx s0 = ldcg_cplx(out), s1 = make_double2(0.0, 0.0);    // the child's own M2L part, in flight during the sum
            const cplx *A = par + (r - k);
            const cplx *col = Ttab + (size_t)c * q * q + k;
            int m = k;
            for (; m + 1 < q; m += 2) {
                s0 = cfma(col[(size_t)m * q], A[m], s0);
                s1 = cfma(col[(size_t)(m + 1) * q], A[m + 1], s1);
            }
            if (m < q) s0 = cfma(col[(size_t)m * q], A[m], s0);
            *out = cadd(s0, s1);
        }
    }
    }   // levels
}

// ------------------------------------------------------------------------------------------------
// ------------------------------------------------------------------------------------------------
// L2P + P2P: one block of 128 threads per leaf box (grid-stride).
//   far  = -(Re Phi1 + i Re Phi2) + (z/2) conj(Phi1' + i Phi2') - (1/2) conj(psi)   from the box's local expansions
//   near = direct sum over the points of the 3 x 3 neighbour boxes that belong to OTHER vesicles
// The sum goes to accum[original point index] (still without the 1/(4 pi mu)).  Targets (tz, tvs, tperm, tstart) are
// the sorted sources themselves for vn_farfield_fmm, a separate sorted set (tvs == nullptr: no vesicle to exclude)
// for the free-target variant.  The shape of the work:
//  * a thread owns TWO targets.  Single-precision storage: as the halves of packed fp32 pairs (FADD2 / FMUL2 / FFMA2
//    and the SFU lg2 / rcp, the arithmetic of the exact fp32 kernels on the stored floats): per source and target pair
//    11 packed instructions + 4 MUFU; per-chunk float partial sums folded into double accumulators;
//  * the own-vesicle exclusion costs no branch: the two SFU results of an excluded pair are replaced by zeros (a
//    select each), which removes both of its terms -- also for the self pair, whose lg2 / rcp are infinite;
//  * the leaf's n targets are dealt out evenly: rounds of at most 128 targets, ceil(n_r / 2) slots of two targets,
//    floor(128 / slots) threads per slot each taking every split-th source (n = 62: 31 slots x 4 threads; n = 100:
//    50 x 2), the partial sums meeting in a fixed order through shared memory -- no power-of-two quantisation;
//  * the three columns of the 3 x 3 neighbourhood are three contiguous index ranges (leaves are stored column by
//    column): they are staged as ONE list in chunks of 1,024 sources (a typical neighbourhood in one: measured 3.5 %
//    faster than 512), two barriers per chunk instead of two per box;
//  * the far field (Horner of the three local expansions, double) is evaluated by one thread per target, all
//    threads busy.
#ifndef VN_FMM_P2P_CHUNK
#define VN_FMM_P2P_CHUNK 1024
#endif
constexpr int kP2PChunk = VN_FMM_P2P_CHUNK;
#ifndef VN_FMM_P2P_CHUNK64
#define VN_FMM_P2P_CHUNK64 256
#endif
constexpr int kP2PChunk64 = VN_FMM_P2P_CHUNK64;
// F64 = true: the same deal of the work for double-precision storage -- a thread's two targets are two independent
// scalar chains through log_rcp_f64 (its 32 KB of tables in front of the source records, records of (x, y) and
// (gx, gy) doubles, 512 per chunk), the exclusion again a select on (log, 1 / r^2); sums run in double throughout.
template <bool F64> __host__ __device__ constexpr int p2p_chunk() { return F64 ? kP2PChunk64 : kP2PChunk; }
template <bool F64> __host__ __device__ constexpr size_t p2p_smem() { return (F64 ? sizeof(double) * (kLogTab + kExpTab) : 0) + (size_t)p2p_chunk<F64>() * 36; }
template <bool F64>
__global__ void __launch_bounds__(128)
fmm_l2p_p2p_packed(const float4 *__restrict__ srcf, const cplx *__restrict__ zs, const cplx *__restrict__ gs,
                   const double *__restrict__ logtab, const int *__restrict__ vs,
                   const long long *__restrict__ start, const cplx *__restrict__ tz, const int *__restrict__ tvs,
                   const int *__restrict__ tperm, const long long *__restrict__ tstart, int q,
                   const unsigned long long *__restrict__ enc, const cplx *__restrict__ loc, cplx *__restrict__ accum)
{
    constexpr int kT = 128, kChunk = p2p_chunk<F64>();
    __shared__ cplx lc[3 * kFmmMaxQ];
    extern __shared__ __align__(16) unsigned char p2p_sm[];
    double *tab = reinterpret_cast<double *>(p2p_sm);                                  // F64 only
    float4 *sxy = reinterpret_cast<float4 *>(p2p_sm + (F64 ? sizeof(double) * (kLogTab + kExpTab) : 0));
    float4 *sgg = sxy + kChunk;                        // fp32: (x, x, y, y) and (gx, gx, gy, gy), both halves of a packed operand
    int *sves = reinterpret_cast<int *>(sgg + kChunk); // fp64: the same 16 bytes hold (x, y) and (gx, gy) as doubles
    __shared__ cplx far[kT];
    __shared__ double4 red[kT];
    const int L = load_level(enc);
    const int n = 1 << L;
    const int tid = threadIdx.x;
    if (F64)
        for (int e = tid; e < kLogTab + kExpTab; e += kT) tab[e] = logtab[e];      // ordered by the barriers of the first leaf
    const Geom gm = load_geom(enc);
    const double s = gm.size / (double)n, inv_s = 1.0 / s;
    for (int c = blockIdx.x; c < n * n; c += gridDim.x) {
        const long long a = tstart[c], b = tstart[c + 1];
        if (a == b) continue;
        const int ix = c / n, iy = c % n;
        __syncthreads();                               // the previous leaf's lc is consumed
        for (int e = tid; e < 3 * q; e += kT) lc[e] = loc[(level_offset(L) + c) * (long long)(3 * q) + e];
        const cplx ctr = box_centre(gm, L, ix, iy);
        // the neighbourhood's sources: one contiguous index range per column
        long long cs[3];
        int clen[3];
        const int by0 = max(iy - 1, 0), by1 = min(iy + 1, n - 1);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int bx = ix - 1 + k;
            cs[k] = 0;
            clen[k] = 0;
            if (bx >= 0 && bx < n) {
                cs[k] = start[bx * n + by0];
                clen[k] = (int)(start[bx * n + by1 + 1] - cs[k]);
            }
        }
        const int total = clen[0] + clen[1] + clen[2];
        const int nt = (int)(b - a);
        const int rounds = (nt + kT - 1) / kT, per_round = (nt + rounds - 1) / rounds;
        for (int r = 0; r < rounds; ++r) {
            const long long t0 = a + (long long)r * per_round;
            const int cnt_t = (int)min((long long)per_round, b - t0);
            const int slots = (cnt_t + 1) >> 1;
            const int split = kT / slots;
            const int slot = tid / split, part = tid - slot * split;
            const bool active = slot < slots;
            const bool has_b = active && slot + slots < cnt_t;
            __syncthreads();                           // lc is loaded; the previous round's far / red are consumed
            if (tid < cnt_t) {
                // far field: Horner for value and derivative of the three local expansions
                const cplx z = tz[t0 + tid];
                const cplx t = make_double2((z.x - ctr.x) * inv_s, (z.y - ctr.y) * inv_s);
                cplx p1 = lc[q - 1], p2 = lc[2 * q - 1], p3 = lc[3 * q - 1];
                cplx d1 = make_double2(0.0, 0.0), d2 = d1;
                for (int l = q - 2; l >= 0; --l) {
                    d1 = cfma(d1, t, p1);
                    d2 = cfma(d2, t, p2);
                    p1 = cfma(p1, t, lc[l]);
                    p2 = cfma(p2, t, lc[q + l]);
                    p3 = cfma(p3, t, lc[2 * q + l]);
                }
                // phi = (Phi1' + i Phi2') = (d1 + i d2)/s ;  z conj(phi)
                const cplx phi = make_double2((d1.x - d2.y) * inv_s, (d1.y + d2.x) * inv_s);
                const cplx zc = cmul(z, make_double2(phi.x, -phi.y));
                far[tid] = make_double2(-p1.x + 0.5 * zc.x - 0.5 * p3.x, -p2.x + 0.5 * zc.y + 0.5 * p3.y);
            }
            // the slot's two targets (a dead second half repeats the first and is never stored)
            u64 zx2 = 0, zy2 = 0;
            cplx za = make_double2(0.0, 0.0), zb = za;
            int va = -2, vb = -2;
            if (active) {
                za = tz[t0 + slot];
                zb = tz[t0 + (has_b ? slot + slots : slot)];
                zx2 = pk((float)za.x, (float)zb.x);
                zy2 = pk((float)za.y, (float)zb.y);
                va = tvs ? tvs[t0 + slot] : -1;
                vb = has_b ? (tvs ? tvs[t0 + slot + slots] : -1) : -2;
            }
            double uxa = 0.0, uya = 0.0, uxb = 0.0, uyb = 0.0;
            for (int f0 = 0; f0 < total; f0 += kChunk) {
                __syncthreads();
                const int cnt = min(kChunk, total - f0);
                for (int e = tid; e < cnt; e += kT) {
                    int f = f0 + e;
                    long long idx;
                    if (f < clen[0]) idx = cs[0] + f;
                    else if (f < clen[0] + clen[1]) idx = cs[1] + (f - clen[0]);
                    else idx = cs[2] + (f - clen[0] - clen[1]);
                    if (F64) {
                        reinterpret_cast<cplx *>(sxy)[e] = zs[idx];
                        reinterpret_cast<cplx *>(sgg)[e] = gs[idx];
                    } else {
                        const float4 v = srcf[idx];                  // (x, y, gx, gy): the stored values, floats to begin with
                        sxy[e] = make_float4(v.x, v.x, v.y, v.y);
                        sgg[e] = make_float4(v.z, v.z, v.w, v.w);
                    }
                    sves[e] = vs[idx];
                }
                __syncthreads();
                if (active && F64) {
                    for (int j = part; j < cnt; j += split) {
                        const cplx pz = reinterpret_cast<const cplx *>(sxy)[j], pg = reinterpret_cast<const cplx *>(sgg)[j];
                        const int sv = sves[j];
                        {
                            const double rx = za.x - pz.x, ry = za.y - pz.y;
                            double ml, inv;
                            log_rcp_f64(fma(rx, rx, ry * ry), tab, ml, inv);
                            if (sv == va) { ml = 0.0; inv = 0.0; }
                            const double qd = fma(rx, pg.x, ry * pg.y) * inv;
                            uxa = fma(ml, pg.x, fma(qd, rx, uxa));
                            uya = fma(ml, pg.y, fma(qd, ry, uya));
                        }
                        {
                            const double rx = zb.x - pz.x, ry = zb.y - pz.y;
                            double ml, inv;
                            log_rcp_f64(fma(rx, rx, ry * ry), tab, ml, inv);
                            if (sv == vb) { ml = 0.0; inv = 0.0; }
                            const double qd = fma(rx, pg.x, ry * pg.y) * inv;
                            uxb = fma(ml, pg.x, fma(qd, rx, uxb));
                            uyb = fma(ml, pg.y, fma(qd, ry, uyb));
                        }
                    }
                }
                if (active && !F64) {
                    u64 fxl = 0, fyl = 0, fxq = 0, fyq = 0;           // packed (a, b): sum lg2 g  and  sum qd r
#pragma unroll 2
                    for (int j = part; j < cnt; j += split) {
                        const ulonglong2 pxy = *reinterpret_cast<const ulonglong2 *>(&sxy[j]);
                        const ulonglong2 pgg = *reinterpret_cast<const ulonglong2 *>(&sgg[j]);
                        const int sv = sves[j];
                        const u64 rx = sub2(zx2, pxy.x), ry = sub2(zy2, pxy.y);
                        const u64 r2 = fma2(rx, rx, mul2(ry, ry));
                        float r2a, r2b;
                        upk(r2, r2a, r2b);
                        const float lga = sv != va ? sfu_lg2(r2a) : 0.f, lgb = sv != vb ? sfu_lg2(r2b) : 0.f;
                        const float iva = sv != va ? sfu_rcp(r2a) : 0.f, ivb = sv != vb ? sfu_rcp(r2b) : 0.f;
                        const u64 lg = pk(lga, lgb);
                        const u64 qd = mul2(fma2(rx, pgg.x, mul2(ry, pgg.y)), pk(iva, ivb));
                        fxl = fma2(lg, pgg.x, fxl);
                        fyl = fma2(lg, pgg.y, fyl);
                        fxq = fma2(qd, rx, fxq);
                        fyq = fma2(qd, ry, fyq);
                    }
                    float la, lb, qa, qb;
                    upk(fxl, la, lb);
                    upk(fxq, qa, qb);
                    uxa += (double)fmaf(-0.34657359027997264f, la, qa);     // -ln(r) = -(ln 2 / 2) lg2(r^2)
                    uxb += (double)fmaf(-0.34657359027997264f, lb, qb);
                    upk(fyl, la, lb);
                    upk(fyq, qa, qb);
                    uya += (double)fmaf(-0.34657359027997264f, la, qa);
                    uyb += (double)fmaf(-0.34657359027997264f, lb, qb);
                }
            }
            red[tid] = make_double4(uxa, uya, uxb, uyb);
            __syncthreads();
            if (active && part == 0) {
                double4 u = red[tid];
                for (int p = 1; p < split; ++p) {
                    const double4 w = red[tid + p];
                    u.x += w.x; u.y += w.y; u.z += w.z; u.w += w.w;
                }
                const cplx fa = far[slot];
                accum[tperm[t0 + slot]] = make_double2(u.x + fa.x, u.y + fa.y);
                if (has_b) {
                    const cplx fb = far[slot + slots];
                    accum[tperm[t0 + slot + slots]] = make_double2(u.z + fb.x, u.w + fb.y);
                }
            }
        }
    }   // leaves
}

// own-vesicle points that sit in NON-neighbour leaf boxes of the target went through the expansions: take their
// contribution out again, scale by 1/(4 pi mu) and store.  One block per vesicle: its points (position, density, leaf)
// are staged in shared memory once and every thread walks them for its own point -- consecutive points of a membrane
// sit in the same or adjacent leaves, so a warp's neighbour tests agree and the few direct terms are not divergent.
// F32 (single-precision storage): the terms are evaluated with the SFU pair arithmetic of the fp32 kernels (the
// positions and densities are floats; the correction is a small part of the sum); double: libm log and a division.
constexpr int kFinThreads = 128;
constexpr int kFinChunk = 256;
template <typename real2, bool F32>
__global__ void __launch_bounds__(kFinThreads)
fmm_finish(const cplx *__restrict__ z, const cplx *__restrict__ g, const int *__restrict__ cell, int nves, int npts,
           const unsigned long long *__restrict__ enc, const cplx *__restrict__ accum, double prefactor,
           real2 *__restrict__ U)
{
    __shared__ cplx sz[kFinChunk], sg[kFinChunk];
    __shared__ int sc[kFinChunk];
    __shared__ int box[4];                              // leaf bounding box of the vesicle: min ix, min iy, max ix, max iy
    const int L = load_level(enc);
    const int n = 1 << L, tid = threadIdx.x;
    for (int ves = blockIdx.x; ves < nves; ves += gridDim.x) {
        const long long v0 = (long long)ves * npts;
        // a point has something to take out only if some point of its vesicle lies two or more leaves away: most
        // vesicles fit in 2 x 2 leaves, and in a wider one only the points of the outer leaves qualify
        __syncthreads();
        if (tid < 2) box[tid] = n;
        else if (tid < 4) box[tid] = -1;
        __syncthreads();
        {
            int x0 = n, y0 = n, x1 = -1, y1 = -1;
            for (int e = tid; e < npts; e += kFinThreads) {
                const int cj = cell[v0 + e], jx = cj >> L, jy = cj & (n - 1);
                x0 = min(x0, jx); y0 = min(y0, jy); x1 = max(x1, jx); y1 = max(y1, jy);
            }
#pragma unroll
            for (int m = 16; m >= 1; m >>= 1) {
                x0 = min(x0, __shfl_xor_sync(0xffffffffu, x0, m));
                y0 = min(y0, __shfl_xor_sync(0xffffffffu, y0, m));
                x1 = max(x1, __shfl_xor_sync(0xffffffffu, x1, m));
                y1 = max(y1, __shfl_xor_sync(0xffffffffu, y1, m));
            }
            if ((tid & 31) == 0) {
                atomicMin(&box[0], x0); atomicMin(&box[1], y0); atomicMax(&box[2], x1); atomicMax(&box[3], y1);
            }
        }
        __syncthreads();
        const int bx0 = box[0], by0 = box[1], bx1 = box[2], by1 = box[3];
        const bool compact = bx1 - bx0 <= 1 && by1 - by0 <= 1;      // every pair of its points is a neighbour pair
        for (int t0 = 0; t0 < npts; t0 += kFinThreads) {
            const bool live = t0 + tid < npts;
            const long long i = v0 + (live ? t0 + tid : 0);
            const cplx zi = z[i];
            const int ci = cell[i], ix = ci >> L, iy = ci & (n - 1);
            const bool mine = live && (ix - bx0 > 1 || bx1 - ix > 1 || iy - by0 > 1 || by1 - iy > 1);
            double cx = 0.0, cy = 0.0;
            for (int s0 = 0; s0 < npts && !compact; s0 += kFinChunk) {
                const int cnt = min(kFinChunk, npts - s0);
                __syncthreads();
                for (int e = tid; e < cnt; e += kFinThreads) {
                    sz[e] = z[v0 + s0 + e];
                    sg[e] = g[v0 + s0 + e];
                    sc[e] = cell[v0 + s0 + e];
                }
                __syncthreads();
                if (!mine) continue;
                float fx = 0.f, fy = 0.f;
                for (int j = 0; j < cnt; ++j) {
                    const int cj = sc[j];
                    if (abs((cj >> L) - ix) <= 1 && abs((cj & (n - 1)) - iy) <= 1) continue;   // in the direct part: masked there
                    const cplx zj = sz[j], gj = sg[j];
                    if (F32) {
                        const float rx = (float)(zi.x - zj.x), ry = (float)(zi.y - zj.y);
                        const float gx = (float)gj.x, gy = (float)gj.y;
                        const float r2 = fmaf(rx, rx, ry * ry);
                        const float ml = -0.34657359027997264f * sfu_lg2(r2);
                        const float qd = fmaf(rx, gx, ry * gy) * sfu_rcp(r2);
                        fx += fmaf(ml, gx, qd * rx);
                        fy += fmaf(ml, gy, qd * ry);
                    } else {
                        const double rx = zi.x - zj.x, ry = zi.y - zj.y;
                        const double r2 = rx * rx + ry * ry;
                        const double ml = -0.5 * log(r2);
                        const double qd = (rx * gj.x + ry * gj.y) / r2;
                        cx += ml * gj.x + qd * rx;
                        cy += ml * gj.y + qd * ry;
                    }
                }
                cx += (double)fx;
                cy += (double)fy;
            }
            if (live) {
                const cplx u = accum[i];
                real2 o;
                o.x = (decltype(o.x))(prefactor * (u.x - cx));
                o.y = (decltype(o.y))(prefactor * (u.y - cy));
                U[i] = o;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// -DVN_FMM_TIMING (diagnostic builds only): device time of every phase of vn_farfield_fmm, printed to stderr per call
#ifdef VN_FMM_TIMING
struct FmmTimer {
    cudaStream_t st;
    cudaEvent_t ev[40];
    const char *name[40];
    int n = 0;
    explicit FmmTimer(cudaStream_t s) : st(s) { tick("start"); }
    void tick(const char *what)
    {
        if (n >= 40) return;
        cudaEventCreate(&ev[n]);
        cudaEventRecord(ev[n], st);
        name[n++] = what;
    }
    ~FmmTimer()
    {
        cudaEventSynchronize(ev[n - 1]);
        float total = 0.f;
        cudaEventElapsedTime(&total, ev[0], ev[n - 1]);
        fprintf(stderr, "fmm phases (us):");
        for (int i = 1; i < n; ++i) {
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ev[i - 1], ev[i]);
            fprintf(stderr, " %s %.1f", name[i], ms * 1e3f);
        }
        fprintf(stderr, " | total %.1f\n", total * 1e3f);
        for (int i = 0; i < n; ++i) cudaEventDestroy(ev[i]);
    }
};
#define FMM_TICK(what) fmm_timer.tick(what)
#else
#define FMM_TICK(what) ((void)0)
#endif

// the double-precision direct part keeps the 32 KB log tables next to its source records: beyond the 48 KB default
static vn_status p2p_f64_prepare()
{
    static bool done_dev[kMaxDevices] = {false};
    bool &done = done_dev[current_device()];
    if (!done) {
        VN_CUDA(cudaFuncSetAttribute(fmm_l2p_p2p_packed<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p2p_smem<true>()));
        done = true;
    }
    return VN_OK;
}

static int fmm_levels_max(long long P)
{
    // the deepest tree the device may choose: leaves of kLeafTarget points if only 1/16 of the root square is occupied
    int L = 2;
    while (L < 10 && 16.0 * (double)P / (double)(1ll << (2 * L)) > kLeafTarget) ++L;
    return L;
}

vn_status farfield_fmm(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu, int order,
                       const int64_t *near_ptr, const int32_t *near_ves, void *U, vn_precision prec, cudaStream_t st)
{
    const int P = (int)(nves * npts), q = order + 1;
    const int L = fmm_levels_max(P);                  // upper bound: the device picks the level (fmm_choose_level)
    const int n = 1 << L, ncell = n * n;
    const long long nbox = level_offset(L + 1);
    const int nb_scan = (ncell + kScanBlock - 1) / kScanBlock;
    auto up = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t b_pt = up(sizeof(cplx) * (size_t)P), b_int = up(sizeof(int) * (size_t)P);
    const size_t b_exp = up(sizeof(cplx) * (size_t)nbox * 3 * q), b_cnt = up(sizeof(int) * (size_t)nbox);
    const size_t b_start = up(sizeof(long long) * ((size_t)ncell + 1)), b_bs = up(sizeof(long long) * (size_t)nb_scan);
    const size_t b_tab = up(sizeof(double) * fmm_tables_doubles(q)), b_log = up(sizeof(double) * (kLogTab + kExpTab));
    const size_t b_leaf = up(sizeof(int) * (size_t)ncell);
    const size_t total = 6 * b_pt + 3 * b_int + 2 * b_exp + b_cnt + b_leaf + 2 * b_start + b_bs + b_tab + b_log + 256;
    char *scr = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scr, total, st));
#ifdef VN_FMM_POISON    // diagnostic builds: every byte of scratch 0xFF (NaN) before use -- a read of something no kernel wrote shows in U
    VN_CUDA(cudaMemsetAsync(scr, 0xFF, total, st));
#endif
    char *ptr = scr;
    auto take = [&](size_t b) { char *r = ptr; ptr += b; return r; };
    cplx *z = (cplx *)take(b_pt), *g = (cplx *)take(b_pt), *zs = (cplx *)take(b_pt), *gs = (cplx *)take(b_pt);
    cplx *accum = (cplx *)take(b_pt);
    float4 *srcf = (float4 *)take(b_pt);               // 16 bytes per point, like a cplx
    int *cell = (int *)take(b_int), *perm = (int *)take(b_int), *vs = (int *)take(b_int);
    cplx *mult = (cplx *)take(b_exp), *loc = (cplx *)take(b_exp);
    unsigned long long *enc = (unsigned long long *)take(256);
    int *boxcnt = (int *)take(b_cnt), *cnt = (int *)take(b_leaf);
    long long *start = (long long *)take(b_start), *cursor = (long long *)take(b_start), *bsum = (long long *)take(b_bs);
    double *tab = (double *)take(b_tab), *logtab = (double *)take(b_log);

#ifdef VN_FMM_TIMING
    FmmTimer fmm_timer(st);
#endif
    VN_CUDA(cudaMemsetAsync(enc, 0, 256 + b_cnt + b_leaf, st));   // the bounding box, boxcnt and the leaf counts are adjacent
    const int gp = (P + 255) / 256, gl = gp < kLoadBlocks ? gp : kLoadBlocks;
    if (prec == VN_F32)                                            // the last block to finish also fixes level and centre
        fmm_load<float, float2><<<gl + kTableBlocks, 256, 0, st>>>((const float2 *)X, (const float2 *)F, (const float *)W, P, z, g, enc, gl, P, L, gl, q, tab, nullptr);
    else                                                           // log tables: double only
        fmm_load<double, double2><<<gl + kTableBlocks + kLogTabBlocks, 256, 0, st>>>((const double2 *)X, (const double2 *)F, (const double *)W, P, z, g, enc, gl, P, L, gl, q, tab, logtab);
    FMM_TICK("load");
    fmm_bin<<<gp, 256, 0, st>>>(z, P, enc, cell, cnt);
    scan_block_sums<<<nb_scan, kScanThreads, 0, st>>>(cnt, ncell, bsum);
    scan_of_sums<<<1, kScanThreads, 0, st>>>(bsum, nb_scan);
    scan_apply<<<nb_scan, kScanThreads, 0, st>>>(cnt, ncell, bsum, start, cursor);
    FMM_TICK("bin+scan");
    fmm_scatter<<<gp, 256, 0, st>>>(cell, P, cursor, vs);                  // vs doubles as the unsorted buffer
    {
        const GatherArgs ga = {z, g, zs, gs, vs, prec == VN_F32 ? srcf : nullptr, (int)npts};
        fmm_sort_cells<<<(ncell + 3) / 4 < 148 * 16 ? (ncell + 3) / 4 : 148 * 16, 128, 0, st>>>(start, enc, vs, perm, ga);
    }
    FMM_TICK("sort+gather");
    int launches = 8;

    const int p2p_grid = ncell < 148 * 64 ? ncell : 148 * 64;      // grid-stride over the leaves the device chose
    FMM_TICK("tables");
    profile_mark(st, true);
    fmm_p2m<<<(ncell + kP2MWarps - 1) / kP2MWarps < 148 * 16 ? (ncell + kP2MWarps - 1) / kP2MWarps : 148 * 16, 32 * kP2MWarps, 0, st>>>(zs, gs, start, q, enc, mult, boxcnt);
    ++launches;
    FMM_TICK("p2m");
    const int resident = L >= 3 ? shift_resident_blocks(q) : 1;     // also opts the two kernels into their shared memory
    if (L >= 3) {     // the level above the leaves with a full grid, all levels above it in one launch of resident blocks
        const unsigned nb = 1u << (2 * (L - 1));
        fmm_m2m<<<nb < 148u * kShiftWave ? nb : 148u * kShiftWave, kShiftThreads, shift_smem(q), st>>>(1, 1, q, tab, enc, mult, boxcnt);
        ++launches;
        if (L >= 4) {
            (void)launch_resident(fmm_m2m, resident, shift_smem(q), st, 2, 99, q, tab, enc, mult, boxcnt);
            ++launches;
        }
    }
    FMM_TICK("m2m");
    if (q <= kM2LHalfQ) {              // all levels in one launch
        const long long nb = (level_offset(L + 1) - level_offset(2) + kM2LWarps - 1) / kM2LWarps;
        fmm_m2l_half<<<(unsigned)(nb < 148 * 16 ? nb : 148 * 16), 32 * kM2LWarps, m2l_half_smem(q), st>>>(q, tab, enc, mult, boxcnt, boxcnt, loc);
        ++launches;
    } else {
        const long long nb = (level_offset(L + 1) - level_offset(2) + kM2LWarps - 1) / kM2LWarps;
        fmm_m2l<<<(unsigned)(nb < 148 * 16 ? nb : 148 * 16), 32 * kM2LWarps, m2l_smem(q), st>>>(q, tab, enc, mult, boxcnt, boxcnt, loc);
        ++launches;
    }
    FMM_TICK("m2l");
    if (L >= 3) {     // levels 3 .. L - 1 in one launch of resident blocks, the leaf level with a full grid
        if (L >= 4) {
            (void)launch_resident(fmm_l2l, resident, shift_smem(q), st, 99, 1, q, tab, enc, boxcnt, loc);
            ++launches;
        }
        const unsigned nb = 1u << (2 * (L - 1));
        fmm_l2l<<<nb < 148u * kShiftWave ? nb : 148u * kShiftWave, kShiftThreads, shift_smem(q), st>>>(0, 0, q, tab, enc, boxcnt, loc);
        ++launches;
    }
    FMM_TICK("l2l");
    if (prec == VN_F32)
        fmm_l2p_p2p_packed<false><<<p2p_grid, 128, p2p_smem<false>(), st>>>(srcf, zs, gs, logtab, vs, start, zs, vs, perm, start, q, enc, loc, accum);
    else if (p2p_f64_prepare() == VN_OK)
        fmm_l2p_p2p_packed<true><<<p2p_grid, 128, p2p_smem<true>(), st>>>(srcf, zs, gs, logtab, vs, start, zs, vs, perm, start, q, enc, loc, accum);
    profile_mark(st, false);
    FMM_TICK("l2p+p2p");
    if (near_ptr) {   // row f-1 on top: take the near vesicles' contributions out (they are all in the direct part)
        const vn_status rc = near_correction_accum(X, F, W, P, (int)npts, near_ptr, near_ves, accum, prec, st);
        if (rc != VN_OK) { (void)cudaFreeAsync(scr, st); return rc; }
    }
    const double pref = 1.0 / (4.0 * 3.14159265358979323846 * mu);
    if (prec == VN_F32)
        fmm_finish<float2, true><<<(unsigned)(nves < 148 * 64 ? nves : 148 * 64), kFinThreads, 0, st>>>(z, g, cell, (int)nves, (int)npts, enc, accum, pref, (float2 *)U);
    else
        fmm_finish<double2, false><<<(unsigned)(nves < 148 * 64 ? nves : 148 * 64), kFinThreads, 0, st>>>(z, g, cell, (int)nves, (int)npts, enc, accum, pref, (double2 *)U);
    count_launch(launches + 2);
    FMM_TICK("finish");
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scr, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------------
// Free targets by the same method (row f-4, both halves together): the sources build the tree and the local
// expansions exactly as above, the nt targets are sorted into the same leaves, and every target gets its
// leaf's local expansions plus the direct sum over the 3 x 3 neighbour leaves.  No vesicle is excluded.
template <typename real2>
__global__ void __launch_bounds__(256)
fmm_load_targets(const real2 *__restrict__ Xt, int nt, cplx *__restrict__ zt, unsigned long long *enc, unsigned tickets,
                 int P_level, int L_hi)
{
    double x = INFINITY, y = INFINITY, X1 = -INFINITY, Y1 = -INFINITY;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nt; i += gridDim.x * blockDim.x) {
        const real2 p = Xt[i];
        const double px = (double)p.x, py = (double)p.y;
        x = fmin(x, px);
        y = fmin(y, py);
        X1 = fmax(X1, px);
        Y1 = fmax(Y1, py);
        zt[i] = make_double2(px, py);
    }
    bounds_commit(x, y, X1, Y1, enc, tickets, P_level, L_hi);
}


template <typename real2>
__global__ void __launch_bounds__(256)
fmm_finish_targets(const cplx *__restrict__ accum, int nt, double prefactor, real2 *__restrict__ Ut)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nt) return;
    real2 o;
    o.x = (decltype(o.x))(prefactor * accum[i].x);
    o.y = (decltype(o.y))(prefactor * accum[i].y);
    Ut[i] = o;
}

vn_status farfield_targets_fmm(const void *Xt, int64_t nt64, const void *X, const void *F, const void *W, int64_t nves,
                               int64_t npts, double mu, int order, void *Ut, vn_precision prec, cudaStream_t st)
{
    const int P = (int)(nves * npts), nt = (int)nt64, q = order + 1;
    const int L = fmm_levels_max(P > nt ? P : nt);    // upper bound: the device picks the level
    const int n = 1 << L, ncell = n * n;
    const long long nbox = level_offset(L + 1);
    const int nb_scan = (ncell + kScanBlock - 1) / kScanBlock;
    auto up = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t b_pt = up(sizeof(cplx) * (size_t)P), b_int = up(sizeof(int) * (size_t)P);
    const size_t b_tpt = up(sizeof(cplx) * (size_t)nt), b_tint = up(sizeof(int) * (size_t)nt);
    const size_t b_exp = up(sizeof(cplx) * (size_t)nbox * 3 * q), b_cnt = up(sizeof(int) * (size_t)nbox);
    const size_t b_ccnt = up(sizeof(int) * (size_t)ncell);
    const size_t b_start = up(sizeof(long long) * ((size_t)ncell + 1)), b_bs = up(sizeof(long long) * (size_t)nb_scan);
    const size_t b_tab = up(sizeof(double) * fmm_tables_doubles(q)), b_log = up(sizeof(double) * (kLogTab + kExpTab));
    const size_t total = 5 * b_pt + 3 * b_int + 3 * b_tpt + 2 * b_tint + 2 * b_exp + b_cnt + 2 * b_ccnt + 4 * b_start +
                         b_bs + b_tab + b_log + 256;
    char *scr = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&scr, total, st));
#ifdef VN_FMM_POISON    // diagnostic builds: every byte of scratch 0xFF (NaN) before use -- a read of something no kernel wrote shows in U
    VN_CUDA(cudaMemsetAsync(scr, 0xFF, total, st));
#endif
    char *ptr = scr;
    auto take = [&](size_t b) { char *r = ptr; ptr += b; return r; };
    cplx *z = (cplx *)take(b_pt), *g = (cplx *)take(b_pt), *zs = (cplx *)take(b_pt), *gs = (cplx *)take(b_pt);
    float4 *srcf = (float4 *)take(b_pt);               // 16 bytes per point, like a cplx
    int *cell = (int *)take(b_int), *perm = (int *)take(b_int), *vs = (int *)take(b_int);
    cplx *zt = (cplx *)take(b_tpt), *zts = (cplx *)take(b_tpt), *accum = (cplx *)take(b_tpt);
    int *tcell = (int *)take(b_tint), *tperm = (int *)take(b_tint);
    cplx *mult = (cplx *)take(b_exp), *loc = (cplx *)take(b_exp);
    unsigned long long *enc = (unsigned long long *)take(256);
    int *boxcnt = (int *)take(b_cnt), *cnt = (int *)take(b_ccnt), *tcnt = (int *)take(b_ccnt);
    long long *start = (long long *)take(b_start), *cursor = (long long *)take(b_start);
    long long *tstart = (long long *)take(b_start), *tcursor = (long long *)take(b_start), *bsum = (long long *)take(b_bs);
    double *tab = (double *)take(b_tab), *logtab = (double *)take(b_log);

    VN_CUDA(cudaMemsetAsync(enc, 0, 256 + b_cnt + 2 * b_ccnt, st));   // the bounding box, boxcnt, cnt and tcnt are adjacent
    const int gp = (P + 255) / 256, gt = (nt + 255) / 256;
    const int gl = gp < kLoadBlocks ? gp : kLoadBlocks, glt = gt < kLoadBlocks ? gt : kLoadBlocks;
    const int Plev = P > nt ? P : nt;
    // sources and targets share one box: the last block of the two kernels together fixes level and centre
    if (prec == VN_F32) {
        fmm_load<float, float2><<<gl + kTableBlocks, 256, 0, st>>>((const float2 *)X, (const float2 *)F, (const float *)W, P, z, g, enc, gl + glt, Plev, L, gl, q, tab, nullptr);
        fmm_load_targets<float2><<<glt, 256, 0, st>>>((const float2 *)Xt, nt, zt, enc, gl + glt, Plev, L);
    } else {
        fmm_load<double, double2><<<gl + kTableBlocks + kLogTabBlocks, 256, 0, st>>>((const double2 *)X, (const double2 *)F, (const double *)W, P, z, g, enc, gl + glt, Plev, L, gl, q, tab, logtab);
        fmm_load_targets<double2><<<glt, 256, 0, st>>>((const double2 *)Xt, nt, zt, enc, gl + glt, Plev, L);
    }
    // sources into leaves
    fmm_bin<<<gp, 256, 0, st>>>(z, P, enc, cell, cnt);
    scan_block_sums<<<nb_scan, kScanThreads, 0, st>>>(cnt, ncell, bsum);
    scan_of_sums<<<1, kScanThreads, 0, st>>>(bsum, nb_scan);
    scan_apply<<<nb_scan, kScanThreads, 0, st>>>(cnt, ncell, bsum, start, cursor);
    fmm_scatter<<<gp, 256, 0, st>>>(cell, P, cursor, vs);                  // vs doubles as the unsorted buffer
    {
        const GatherArgs ga = {z, g, zs, gs, vs, prec == VN_F32 ? srcf : nullptr, (int)npts};
        fmm_sort_cells<<<(ncell + 3) / 4 < 148 * 16 ? (ncell + 3) / 4 : 148 * 16, 128, 0, st>>>(start, enc, vs, perm, ga);
    }
    // targets into the same leaves
    fmm_bin<<<gt, 256, 0, st>>>(zt, nt, enc, tcell, tcnt);
    scan_block_sums<<<nb_scan, kScanThreads, 0, st>>>(tcnt, ncell, bsum);
    scan_of_sums<<<1, kScanThreads, 0, st>>>(bsum, nb_scan);
    scan_apply<<<nb_scan, kScanThreads, 0, st>>>(tcnt, ncell, bsum, tstart, tcursor);
    fmm_scatter<<<gt, 256, 0, st>>>(tcell, nt, tcursor, (int *)accum);     // accum doubles as the unsorted buffer
    {
        const GatherArgs ga = {zt, nullptr, zts, nullptr, nullptr, nullptr, 1};
        fmm_sort_cells<<<(ncell + 3) / 4 < 148 * 16 ? (ncell + 3) / 4 : 148 * 16, 128, 0, st>>>(tstart, enc, (const int *)accum, tperm, ga);
    }
    int launches = 15;

    const int p2p_grid = ncell < 148 * 64 ? ncell : 148 * 64;      // grid-stride over the leaves the device chose
    profile_mark(st, true);
    fmm_p2m<<<(ncell + kP2MWarps - 1) / kP2MWarps < 148 * 16 ? (ncell + kP2MWarps - 1) / kP2MWarps : 148 * 16, 32 * kP2MWarps, 0, st>>>(zs, gs, start, q, enc, mult, boxcnt);
    ++launches;
    const int resident = L >= 3 ? shift_resident_blocks(q) : 1;     // also opts the two kernels into their shared memory
    if (L >= 3) {     // the level above the leaves with a full grid, all levels above it in one launch of resident blocks
        const unsigned nb = 1u << (2 * (L - 1));
        fmm_m2m<<<nb < 148u * kShiftWave ? nb : 148u * kShiftWave, kShiftThreads, shift_smem(q), st>>>(1, 1, q, tab, enc, mult, boxcnt);
        ++launches;
        if (L >= 4) {
            (void)launch_resident(fmm_m2m, resident, shift_smem(q), st, 2, 99, q, tab, enc, mult, boxcnt);
            ++launches;
        }
    }
    if (q <= kM2LHalfQ) {              // all levels in one launch
        const long long nb = (level_offset(L + 1) - level_offset(2) + kM2LWarps - 1) / kM2LWarps;
        fmm_m2l_half<<<(unsigned)(nb < 148 * 16 ? nb : 148 * 16), 32 * kM2LWarps, m2l_half_smem(q), st>>>(q, tab, enc, mult, boxcnt, nullptr, loc);
        ++launches;
    } else {
        const long long nb = (level_offset(L + 1) - level_offset(2) + kM2LWarps - 1) / kM2LWarps;
        fmm_m2l<<<(unsigned)(nb < 148 * 16 ? nb : 148 * 16), 32 * kM2LWarps, m2l_smem(q), st>>>(q, tab, enc, mult, boxcnt, nullptr, loc);
        ++launches;
    }
    if (L >= 3) {     // levels 3 .. L - 1 in one launch of resident blocks, the leaf level with a full grid
        if (L >= 4) {
            (void)launch_resident(fmm_l2l, resident, shift_smem(q), st, 99, 1, q, tab, enc, (const int *)nullptr, loc);
            ++launches;
        }
        const unsigned nb = 1u << (2 * (L - 1));
        fmm_l2l<<<nb < 148u * kShiftWave ? nb : 148u * kShiftWave, kShiftThreads, shift_smem(q), st>>>(0, 0, q, tab, enc, nullptr, loc);
        ++launches;
    }
    if (prec == VN_F32)
        fmm_l2p_p2p_packed<false><<<p2p_grid, 128, p2p_smem<false>(), st>>>(srcf, zs, gs, logtab, vs, start, zts, nullptr, tperm, tstart, q, enc, loc, accum);
    else if (p2p_f64_prepare() == VN_OK)
        fmm_l2p_p2p_packed<true><<<p2p_grid, 128, p2p_smem<true>(), st>>>(srcf, zs, gs, logtab, vs, start, zts, nullptr, tperm, tstart, q, enc, loc, accum);
    profile_mark(st, false);
    const double pref = 1.0 / (4.0 * 3.14159265358979323846 * mu);
    if (prec == VN_F32)
        fmm_finish_targets<float2><<<gt, 256, 0, st>>>(accum, nt, pref, (float2 *)Ut);
    else
        fmm_finish_targets<double2><<<gt, 256, 0, st>>>(accum, nt, pref, (double2 *)Ut);
    count_launch(launches + 2);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(scr, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

}  // namespace vn

// vn_api.cu -- the extern "C" boundary declared in include/vesnet_farfield.h: argument checks
// (before any CUDA call), device check (sm_100 family only, no fallback), dispatch by precision,
// and the host-buffer entry point.
#include <math.h>

#include <mutex>
#include <vector>

#include "vn_common.cuh"

namespace vn {

unsigned long long g_launches = 0;

static bool g_profile = false;
static std::mutex g_profile_mtx;
static std::vector<cudaEvent_t> g_profile_events;   // begin, end, begin, end, ...

void profile_mark(cudaStream_t st, bool begin)
{
    if (!__atomic_load_n(&g_profile, __ATOMIC_RELAXED)) return;    // cheap test without the lock ...
    std::lock_guard<std::mutex> lock(g_profile_mtx);
    if (!g_profile) return;                                        // ... decided under it
    if (begin != (g_profile_events.size() % 2 == 0)) return;   // keep pairs well formed
    cudaEvent_t ev;
    if (cudaEventCreate(&ev) != cudaSuccess) return;
    cudaEventRecord(ev, st);
    g_profile_events.push_back(ev);
}

vn_status farfield_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                       void *U, cudaStream_t st, const int64_t *near_ptr, const int32_t *near_ves);
vn_status farfield_f64(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                       void *U, cudaStream_t st, const int64_t *near_ptr, const int32_t *near_ves);
vn_status farfield_targets_f32(const void *Xt, int64_t nt, const void *X, const void *F, const void *W,
                               int64_t nves, int64_t npts, double mu, void *Ut, cudaStream_t st);
vn_status farfield_targets_f64(const void *Xt, int64_t nt, const void *X, const void *F, const void *W,
                               int64_t nves, int64_t npts, double mu, void *Ut, cudaStream_t st);
vn_status elastic_force(const void *X, const void *sigma, int64_t nves, int64_t npts, double kappa_b, void *F,
                        vn_precision prec, cudaStream_t st);
vn_status redistribute(const void *X, int64_t nves, int64_t npts, void *Xnew, vn_precision prec, cudaStream_t st);
vn_status farfield_fmm(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu, int order,
                       const int64_t *near_ptr, const int32_t *near_ves, void *U, vn_precision prec, cudaStream_t st);
vn_status farfield_targets_fmm(const void *Xt, int64_t nt, const void *X, const void *F, const void *W, int64_t nves,
                               int64_t npts, double mu, int order, void *Ut, vn_precision prec, cudaStream_t st);
void plan_f32(long long P, int slots, int *super_tile, int *sub, SymSplit *sp);
void plan_f64(long long P, int slots, int *super_tile, int *sub, SymSplit *sp);
vn_status near_pairs(const void *X, const void *W, int64_t nves, int64_t npts, int64_t *near_ptr,
                     int32_t *near_ves, int64_t capacity, vn_precision prec, cudaStream_t st);
vn_status arclength_weights(const void *X, int64_t nves, int64_t npts, void *W, vn_precision prec, cudaStream_t st);
vn_status pipe_peaks(double *rates, cudaStream_t st);
vn_status farfield_selfcheck_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                                 void *U, unsigned long long *mismatches, cudaStream_t st);
vn_status farfield_selfcheck_f64(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                                 void *U, unsigned long long *mismatches, cudaStream_t st);
vn_status farfield_small(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu, void *U,
                         vn_precision prec, cudaStream_t st);
vn_status farfield_partial_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, int part,
                               int nparts, void *acc, void *gmax, cudaStream_t st);
vn_status farfield_partial_f64(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, int part,
                               int nparts, void *acc, void *gmax, cudaStream_t st);
vn_status farfield_finish_f32(const void *acc, const void *gmax, int64_t P_total, int64_t count, double mu, void *U,
                              cudaStream_t st);
vn_status farfield_static_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                              void *U, cudaStream_t st);
int64_t farfield_static_max_points();
vn_status farfield_finish_f64(const void *acc, const void *gmax, int64_t P_total, int64_t count, double mu, void *U,
                              cudaStream_t st);

Split choose_split_for(int n_tb, int n_tiles, int slots, int min_tiles)
{
    Split sp;
    sp.n_tb = n_tb;
    sp.n_tiles = n_tiles;
    int max_chunks = sp.n_tiles / min_tiles;
    if (max_chunks < 1) max_chunks = 1;
    if (max_chunks > 32) max_chunks = 32;
    double best = -1.0;
    sp.n_chunks = 1;
    for (int c = 1; c <= max_chunks; ++c) {
        const long long blocks = (long long)sp.n_tb * c;
        const long long waves = (blocks + slots - 1) / slots;
        const double eff = (double)blocks / (double)(waves * slots);
        if (eff > best + 1e-3) { best = eff; sp.n_chunks = c; }
        else if (eff > best - 1e-3 && c > sp.n_chunks) { sp.n_chunks = c; if (eff > best) best = eff; }
    }
    return sp;
}

// Grid of the symmetric kernels: every super-tile walks a list of about sub*(n_st/2 + 1) source tiles,
// cut into n_chunks chunks of t = list/n_chunks tiles.  With W = n_st*list/slots tiles of work per resident-block
// slot, the run time measured on B200 follows  W (1 + o/t) + b t  tile-times: o = 0.03 tile-times of set-up and
// flush per block, b = 0.25 for the ragged end of a grid whose blocks do not run in lockstep (the hardware hands
// out blocks as slots free up, so a multi-wave grid has no wave quantisation worth modelling).  The minimum is at
// t = sqrt(W o / b) = sqrt(0.12 W): 1 tile per block at 256 x 128 points, 8 at 2000 x 128, 33 at 8000 x 128.
// Measured, fp32: 256 x 128 0.41 ms with 1-tile blocks against 0.47 ms with 416 blocks of 10 tiles;
// 1000 x 128 5.66 ms (6 tiles) against 5.72 (13).  max_tiles > 0 caps t (fp64 kernel: its stage refill waits for
// the slowest warp, which costs about half a tile-time per block once a block has more tiles than stages).
SymSplit choose_sym_split(long long P, int super_tile, int slots, int min_tiles, int max_tiles)
{
    SymSplit sp;
    sp.n_st = (int)((P + super_tile - 1) / super_tile);
    sp.n_tiles = (int)((P + kTile - 1) / kTile);
    const int sub = super_tile / kTile;
    const long long list = (long long)sub * (sp.n_st / 2 + 1);     // longest list over the super-tiles
    const double W = (double)sp.n_st * (double)list / (double)(slots > 0 ? slots : 1);
    long long t = (long long)(sqrt(0.12 * W) + 0.5);
    if (t < min_tiles) t = min_tiles;
    if (t < 1) t = 1;
    if (max_tiles > 0 && t > max_tiles) t = max_tiles;
    if (t > list) t = list;
    long long c = (list + t - 1) / t;
    // keep the grid below 2^31 - 1 blocks
    const long long cmax = 2147483647ll / (sp.n_st > 0 ? sp.n_st : 1);
    if (c > cmax) c = cmax;
    if (c < 1) c = 1;
    sp.n_chunks = (int)c;
#ifdef VN_SYM_FORCE_CHUNKS
    sp.n_chunks = VN_SYM_FORCE_CHUNKS;    // tuning builds only
#endif
    return sp;
}

static vn_status check_device()
{
    static int state_dev[kMaxDevices] = {0};   // 0 unknown, 1 ok, 2 unsupported
    int &state = state_dev[current_device()];
    int ok = state == 0 ? -1 : (state == 1 ? 1 : 0);
    if (ok < 0) {
        int dev = 0, major = 0;
        VN_CUDA(cudaGetDevice(&dev));
        VN_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        ok = (major == 10) ? 1 : 0;
        if (ok) {
            // keep freed stream-ordered scratch cached in the pool instead of returning it to the OS
            cudaMemPool_t pool;
            if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
                unsigned long long thr = ~0ull;
                (void)cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
            }
        }
    }
    state = ok ? 1 : 2;
    return ok ? VN_OK : VN_ERR_UNSUPPORTED;
}

// vn_farfield proper: the single-launch kernel for tiny suspensions, the symmetric pair kernels otherwise
static vn_status farfield_dispatch(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                                   void *U, vn_precision prec, cudaStream_t st)
{
    if (nves * npts <= kSmallPoints) return farfield_small(X, F, W, nves, npts, mu, U, prec, st);
    return prec == VN_F32 ? farfield_f32(X, F, W, nves, npts, mu, U, st, nullptr, nullptr)
                          : farfield_f64(X, F, W, nves, npts, mu, U, st, nullptr, nullptr);
}

static bool misaligned(const void *p, size_t a) { return ((uintptr_t)p % a) != 0; }

static vn_status check_shape(int64_t nves, int64_t npts, vn_precision prec)
{
    if (prec != VN_F32 && prec != VN_F64) return VN_ERR_INVALID_ARG;
    if (nves < 1 || npts < 1) return VN_ERR_INVALID_ARG;
    if (npts >= (1ll << 31) || nves >= (1ll << 31) || nves * npts >= (1ll << 31)) return VN_ERR_INVALID_ARG;
    return VN_OK;
}

}  // namespace vn

using namespace vn;

extern "C" {

vn_status vn_farfield(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                      void *U, vn_precision precision, void *stream)
{
    if (!X || !F || !W || !U) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (!isfinite(mu) || !(mu > 0.0)) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(F, pair) || misaligned(U, pair) || misaligned(W, pair / 2))
        return VN_ERR_INVALID_ARG;
    if (U == X || U == F || U == W) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    return farfield_dispatch(X, F, W, nves, npts, mu, U, precision, (cudaStream_t)stream);
}

// no allocation: static scratch (vn_farfield_f32.cu), fp32, at most vn_noalloc_max_points() points
vn_status vn_farfield_noalloc_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                                  void *U, void *stream)
{
    if (!X || !F || !W || !U) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, VN_F32) != VN_OK) return VN_ERR_INVALID_ARG;
    if (!isfinite(mu) || !(mu > 0.0)) return VN_ERR_INVALID_ARG;
    if (misaligned(X, 8) || misaligned(F, 8) || misaligned(U, 8) || misaligned(W, 4)) return VN_ERR_INVALID_ARG;
    if (U == X || U == F || U == W) return VN_ERR_INVALID_ARG;
    if (nves * npts > farfield_static_max_points()) return VN_ERR_TOO_LARGE;
    int dev = 0, major = 0;                  // the device check of the other entry points without their pool set-up
    VN_CUDA(cudaGetDevice(&dev));
    VN_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return VN_ERR_UNSUPPORTED;
    return farfield_static_f32(X, F, W, nves, npts, mu, U, (cudaStream_t)stream);
}

int64_t vn_noalloc_max_points(void) { return farfield_static_max_points(); }

vn_status vn_near_pairs(const void *X, const void *W, int64_t nves, int64_t npts, int64_t *near_ptr,
                        int32_t *near_ves, int64_t capacity, vn_precision precision, void *stream)
{
    if (!X || !W || !near_ptr) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (capacity < 0 || (capacity > 0 && !near_ves)) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(W, pair / 2) || misaligned(near_ptr, 8) || misaligned(near_ves, 4))
        return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    return near_pairs(X, W, nves, npts, near_ptr, near_ves, capacity, precision, (cudaStream_t)stream);
}

vn_status vn_farfield_masked(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                             const int64_t *near_ptr, const int32_t *near_ves, void *U, vn_precision precision,
                             void *stream)
{
    if (!X || !F || !W || !U || !near_ptr) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (!isfinite(mu) || !(mu > 0.0)) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(F, pair) || misaligned(U, pair) || misaligned(W, pair / 2) ||
        misaligned(near_ptr, 8) || misaligned(near_ves, 4))
        return VN_ERR_INVALID_ARG;
    if (U == X || U == F || U == W) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    cudaStream_t st = (cudaStream_t)stream;
    return precision == VN_F32 ? farfield_f32(X, F, W, nves, npts, mu, U, st, near_ptr, near_ves)
                               : farfield_f64(X, F, W, nves, npts, mu, U, st, near_ptr, near_ves);
}

vn_status vn_farfield_targets(const void *Xt, int64_t nt, const void *X, const void *F, const void *W,
                              int64_t nves, int64_t npts, double mu, void *Ut, vn_precision precision, void *stream)
{
    if (!X || !F || !W) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (nt < 0 || nt >= (1ll << 31)) return VN_ERR_INVALID_ARG;
    if (!isfinite(mu) || !(mu > 0.0)) return VN_ERR_INVALID_ARG;
    if (nt == 0) return VN_OK;
    if (!Xt || !Ut) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(F, pair) || misaligned(Xt, pair) || misaligned(Ut, pair) ||
        misaligned(W, pair / 2))
        return VN_ERR_INVALID_ARG;
    if (Ut == X || Ut == F || Ut == W || Ut == Xt) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    cudaStream_t st = (cudaStream_t)stream;
    return precision == VN_F32 ? farfield_targets_f32(Xt, nt, X, F, W, nves, npts, mu, Ut, st)
                               : farfield_targets_f64(Xt, nt, X, F, W, nves, npts, mu, Ut, st);
}

vn_status vn_arclength_weights(const void *X, int64_t nves, int64_t npts, void *W, vn_precision precision,
                               void *stream)
{
    if (!X || !W) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(W, pair / 2) || W == X) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    return arclength_weights(X, nves, npts, W, precision, (cudaStream_t)stream);
}

vn_status vn_elastic_force(const void *X, const void *sigma, int64_t nves, int64_t npts, double kappa_b, void *F,
                           vn_precision precision, void *stream)
{
    if (!X || !sigma || !F) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (npts > 1024 || !isfinite(kappa_b)) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(F, pair) || misaligned(sigma, pair / 2) || F == X || F == sigma)
        return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    return elastic_force(X, sigma, nves, npts, kappa_b, F, precision, (cudaStream_t)stream);
}

vn_status vn_redistribute_arclength(const void *X, int64_t nves, int64_t npts, void *Xnew, vn_precision precision,
                                    void *stream)
{
    if (!X || !Xnew) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (npts < 3 || npts > 512) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(Xnew, pair) || Xnew == X) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    return redistribute(X, nves, npts, Xnew, precision, (cudaStream_t)stream);
}

vn_status vn_farfield_fmm(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                          int order, const int64_t *near_ptr, const int32_t *near_ves, void *U,
                          vn_precision precision, void *stream)
{
    if (misaligned(near_ptr, 8) || misaligned(near_ves, 4)) return VN_ERR_INVALID_ARG;
    if (order == 0) order = precision == VN_F32 ? 14 : 38;      // the orders that meet 2e-5 / 1e-12, point-wise too
    if (!X || !F || !W || !U) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (!isfinite(mu) || !(mu > 0.0) || order < 2 || order > 48) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(F, pair) || misaligned(U, pair) || misaligned(W, pair / 2))
        return VN_ERR_INVALID_ARG;
    if (U == X || U == F || U == W) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    return farfield_fmm(X, F, W, nves, npts, mu, order, near_ptr, near_ves, U, precision, (cudaStream_t)stream);
}

vn_status vn_farfield_targets_fmm(const void *Xt, int64_t nt, const void *X, const void *F, const void *W,
                                  int64_t nves, int64_t npts, double mu, int order, void *Ut,
                                  vn_precision precision, void *stream)
{
    if (!X || !F || !W) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (order == 0) order = precision == VN_F32 ? 14 : 38;
    if (nt < 0 || nt >= (1ll << 31) || order < 2 || order > 48) return VN_ERR_INVALID_ARG;
    if (!isfinite(mu) || !(mu > 0.0)) return VN_ERR_INVALID_ARG;
    if (nt == 0) return VN_OK;
    if (!Xt || !Ut) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(F, pair) || misaligned(Xt, pair) || misaligned(Ut, pair) ||
        misaligned(W, pair / 2))
        return VN_ERR_INVALID_ARG;
    if (Ut == X || Ut == F || Ut == W || Ut == Xt) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    return farfield_targets_fmm(Xt, nt, X, F, W, nves, npts, mu, order, Ut, precision, (cudaStream_t)stream);
}

vn_status vn_farfield_host(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                           void *U, vn_precision precision)
{
    if (!X || !F || !U) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (!isfinite(mu) || !(mu > 0.0)) return VN_ERR_INVALID_ARG;
    if (U == X || U == F || U == W) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;

    // cached device buffer and stream PER DEVICE, grown on demand, kept for the life of the process (a caller that
    // switches devices finds each device's own cache again; nothing is dropped or leaked on a switch)
    struct HostCache {
        cudaStream_t st = nullptr;
        char *buf = nullptr;
        size_t cap = 0;
    };
    static std::mutex mtx;
    static HostCache cache[kMaxDevices];
    std::lock_guard<std::mutex> lock(mtx);
    HostCache &hc = cache[current_device()];
    if (!hc.st) VN_CUDA(cudaStreamCreateWithFlags(&hc.st, cudaStreamNonBlocking));
    cudaStream_t st = hc.st;
    const size_t P = (size_t)(nves * npts);
    const size_t es = precision == VN_F32 ? 4 : 8;
    const size_t bX = 2 * es * P, bW = es * P;
    auto up = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t need = 3 * up(bX) + up(bW);
    if (need > hc.cap) {
        if (hc.buf) VN_CUDA(cudaFree(hc.buf));
        hc.buf = nullptr; hc.cap = 0;
        VN_CUDA(cudaMalloc((void **)&hc.buf, need));
        hc.cap = need;
    }
    char *dX = hc.buf, *dF = dX + up(bX), *dU = dF + up(bX), *dW = dU + up(bX);
    VN_CUDA(cudaMemcpyAsync(dX, X, bX, cudaMemcpyHostToDevice, st));
    VN_CUDA(cudaMemcpyAsync(dF, F, bX, cudaMemcpyHostToDevice, st));
    vn_status rc;
    if (W) {
        VN_CUDA(cudaMemcpyAsync(dW, W, bW, cudaMemcpyHostToDevice, st));
    } else {
        rc = arclength_weights(dX, nves, npts, dW, precision, st);
        if (rc != VN_OK) return rc;
    }
    rc = farfield_dispatch(dX, dF, dW, nves, npts, mu, dU, precision, st);
    if (rc != VN_OK) return rc;
    VN_CUDA(cudaMemcpyAsync(U, dU, bX, cudaMemcpyDeviceToHost, st));
    VN_CUDA(cudaStreamSynchronize(st));
    return VN_OK;
}

vn_status vn_plan_farfield(int64_t nves, int64_t npts, vn_precision precision, int32_t resident_blocks, int32_t *plan)
{
    if (!plan || resident_blocks < 1 || check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    int super_tile = 0, sub = 0;
    SymSplit sp;
    if (precision == VN_F32) plan_f32(nves * npts, resident_blocks, &super_tile, &sub, &sp);
    else plan_f64(nves * npts, resident_blocks, &super_tile, &sub, &sp);
    plan[0] = super_tile;
    plan[1] = sub;
    plan[2] = sp.n_st;
    plan[3] = sp.n_chunks;
    plan[4] = kTile;
    return VN_OK;
}

vn_status vn_farfield_partial(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, int32_t part,
                              int32_t nparts, void *acc, void *gmax, vn_precision precision, void *stream)
{
    if (!X || !F || !W || !acc || !gmax) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (nparts < 1 || part < 0 || part >= nparts) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(F, pair) || misaligned(W, pair / 2) || misaligned(acc, 16) || misaligned(gmax, 8))
        return VN_ERR_INVALID_ARG;
    if (acc == X || acc == F || acc == W || gmax == acc) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    cudaStream_t st = (cudaStream_t)stream;
    return precision == VN_F32 ? farfield_partial_f32(X, F, W, nves, npts, part, nparts, acc, gmax, st)
                               : farfield_partial_f64(X, F, W, nves, npts, part, nparts, acc, gmax, st);
}

vn_status vn_farfield_finish(const void *acc, const void *gmax, int64_t npoints_total, int64_t count, double mu, void *U,
                             vn_precision precision, void *stream)
{
    if (precision != VN_F32 && precision != VN_F64) return VN_ERR_INVALID_ARG;
    if (npoints_total < 1 || npoints_total >= (1ll << 31) || count < 0 || count > npoints_total) return VN_ERR_INVALID_ARG;
    if (!isfinite(mu) || !(mu > 0.0)) return VN_ERR_INVALID_ARG;
    if (count == 0) return VN_OK;
    if (!acc || !gmax || !U) return VN_ERR_INVALID_ARG;
    if (misaligned(acc, 16) || misaligned(gmax, 8) || misaligned(U, precision == VN_F32 ? 8 : 16) || U == acc)
        return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    cudaStream_t st = (cudaStream_t)stream;
    return precision == VN_F32 ? farfield_finish_f32(acc, gmax, npoints_total, count, mu, U, st)
                               : farfield_finish_f64(acc, gmax, npoints_total, count, mu, U, st);
}

vn_status vn_selfcheck(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu, void *U,
                       vn_precision precision, void *stream, int64_t *mismatches)
{
    if (!X || !F || !W || !U || !mismatches) return VN_ERR_INVALID_ARG;
    if (check_shape(nves, npts, precision) != VN_OK) return VN_ERR_INVALID_ARG;
    if (!isfinite(mu) || !(mu > 0.0)) return VN_ERR_INVALID_ARG;
    const size_t pair = precision == VN_F32 ? 8 : 16;
    if (misaligned(X, pair) || misaligned(F, pair) || misaligned(U, pair) || misaligned(W, pair / 2))
        return VN_ERR_INVALID_ARG;
    if (U == X || U == F || U == W) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long *d_count = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&d_count, 8, st));
    VN_CUDA(cudaMemsetAsync(d_count, 0, 8, st));
    const vn_status rc = precision == VN_F32 ? farfield_selfcheck_f32(X, F, W, nves, npts, mu, U, d_count, st)
                                             : farfield_selfcheck_f64(X, F, W, nves, npts, mu, U, d_count, st);
    unsigned long long h_count = 0;
    const cudaError_t e1 = cudaMemcpyAsync(&h_count, d_count, 8, cudaMemcpyDeviceToHost, st);
    const cudaError_t e2 = cudaStreamSynchronize(st);
    (void)cudaFreeAsync(d_count, st);
    if (rc != VN_OK) return rc;
    if (e1 != cudaSuccess || e2 != cudaSuccess) { (void)cudaGetLastError(); return VN_ERR_CUDA; }
    *mismatches = (int64_t)h_count;
    return VN_OK;
}

vn_status vn_pipe_peaks(double *rates, void *stream)
{
    if (!rates) return VN_ERR_INVALID_ARG;
    const vn_status ds = check_device();
    if (ds != VN_OK) return ds;
    return pipe_peaks(rates, (cudaStream_t)stream);
}

vn_status vn_profile_enable(int enable)
{
    std::lock_guard<std::mutex> lock(g_profile_mtx);
    __atomic_store_n(&g_profile, enable != 0, __ATOMIC_RELAXED);
    if (!enable) {                                  // recorded and never read: do not keep the events
        for (cudaEvent_t ev : g_profile_events) cudaEventDestroy(ev);
        g_profile_events.clear();
    }
    return VN_OK;
}

int64_t vn_profile_read(double *ms, int64_t max_entries)
{
    std::lock_guard<std::mutex> lock(g_profile_mtx);
    const int64_t pairs = (int64_t)(g_profile_events.size() / 2);
    int64_t n = 0;
    bool bad = false;
    for (int64_t i = 0; i < pairs; ++i) {
        cudaEvent_t a = g_profile_events[2 * i], b = g_profile_events[2 * i + 1];
        float t = 0.f;
        if (cudaEventSynchronize(b) != cudaSuccess || cudaEventElapsedTime(&t, a, b) != cudaSuccess) bad = true;
        if (ms && n < max_entries) ms[n++] = (double)t;
        cudaEventDestroy(a);
        cudaEventDestroy(b);
    }
    for (size_t i = 2 * (size_t)pairs; i < g_profile_events.size(); ++i) cudaEventDestroy(g_profile_events[i]);
    g_profile_events.clear();
    return bad ? -1 : n;
}

int64_t vn_launch_count(void) { return (int64_t)__atomic_load_n(&g_launches, __ATOMIC_RELAXED); }

const char *vn_status_string(vn_status s)
{
    switch (s) {
        case VN_OK: return "ok";
        case VN_ERR_INVALID_ARG: return "invalid argument";
        case VN_ERR_UNSUPPORTED: return "unsupported device (needs compute capability 10.x, sm_100a build)";
        case VN_ERR_CUDA: return "CUDA runtime error";
        case VN_ERR_TOO_LARGE:
            return "too many points for the static scratch of vn_farfield_noalloc_f32 (at most 262,144 = vn_noalloc_max_points(); use vn_farfield)";
    }
    return "unknown status";
}

int vn_version(void) { return VN_VERSION; }

}  // extern "C"

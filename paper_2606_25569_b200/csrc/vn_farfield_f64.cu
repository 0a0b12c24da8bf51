// vn_farfield_f64.cu -- fp64 far-field Stokeslet sum for sm_100a (parity-grade variant).
//
// Same decomposition as the fp32 kernel (vn_farfield_f32.cu): block = (target block, source chunk),
// source tiles through a ring of shared-memory stages filled by bulk async copies, own-vesicle
// tiles on a predicated path.  Arithmetic is plain double: per pair
//   r = x - y; r2 = rx*rx + ry*ry; acc += -(1/2) log(r2) * g + ((r.g)/r2) * r
// (eqs 2.8/2.9).  There is no SFU log/rcp in double; see pair_f64().
#include "vn_common.cuh"

namespace vn {

constexpr int kT64 = 4;   // targets per thread

// a-2: one 32-byte record (yx, yy, gx, gy) per source, g = F*W.
__global__ void pack_sources_f64(const double2 *__restrict__ X, const double2 *__restrict__ F,
                                 const double *__restrict__ W, int P, double4 *__restrict__ src)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P) return;
    const double2 y = X[s];
    const double2 f = F[s];
    const double w = W[s];
    src[s] = make_double4(y.x, y.y, f.x * w, f.y * w);
}

// -(1/2) log(r2) and 1/r2 in double.  One reciprocal serves both: with r2 = m * 2^e, m in
// [sqrt(1/2), sqrt(2)), s = (m-1)/(m+1) and log m = 2 atanh(s); 1/(m (m+1)) gives 1/m and 1/(m+1)
// (same trick as the packed fp32 pair).  Series error < 2e-17 for |s| <= 0.1716.
__device__ __forceinline__ void log_rcp_f64(double r2, double &mhalf_log, double &inv)
{
    int hi = __double2hiint(r2);
    const int lo = __double2loint(r2);
    int e = (hi >> 20) - 1023;                      // r2 is a positive normal number (precondition)
    hi = (hi & 0x000fffff) | 0x3ff00000;            // mantissa in [1, 2)
    if (hi >= 0x3ff6a09f) { hi -= 0x00100000; e += 1; }   // -> [sqrt(1/2), sqrt(2))
    const double m = __hiloint2double(hi, lo);
    const double mp1 = m + 1.0;
    const double prod = m * mp1;
    // reciprocal of prod: hardware seed + two Newton steps
    double t;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(t) : "d"(prod));
    t = fma(fma(-prod, t, 1.0), t, t);
    t = fma(fma(-prod, t, 1.0), t, t);
    t = fma(fma(-prod, t, 1.0), t, t);
    const double inv_m = t * mp1;                   // 1/m
    const double s = (m - 1.0) * (t * m);           // (m-1)/(m+1)
    const double z = s * s;
    // atanh(s)/s = 1 + z/3 + z^2/5 + ... + z^10/21
    double p = 1.0 / 21.0;
    p = fma(p, z, 1.0 / 19.0);
    p = fma(p, z, 1.0 / 17.0);
    p = fma(p, z, 1.0 / 15.0);
    p = fma(p, z, 1.0 / 13.0);
    p = fma(p, z, 1.0 / 11.0);
    p = fma(p, z, 1.0 / 9.0);
    p = fma(p, z, 1.0 / 7.0);
    p = fma(p, z, 1.0 / 5.0);
    p = fma(p, z, 1.0 / 3.0);
    p = fma(p, z, 1.0);
    // -(1/2) log(r2) = -(1/2) e ln2 - s p
    mhalf_log = fma((double)e, -0.34657359027997265471, -(s * p));
    // 1/r2 = 2^-e / m
    inv = __hiloint2double(__double2hiint(inv_m) - (e << 20), __double2loint(inv_m));
}

__global__ void __launch_bounds__(kThreads, 4)
farfield_f64_kernel(const double4 *__restrict__ src, const double2 *__restrict__ X, int P, int npts,
                    int n_tiles, int n_chunks, double2 *__restrict__ part)
{
    constexpr int T = kT64;
    __shared__ __align__(128) double4 tile[kStages][kTile];
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

    auto issue = [&](int i) {
        const int s = i % kStages;
        const int first = (t_begin + i) * kTile;
        const int cnt = min(kTile, P - first);
        const uint32_t bytes = (uint32_t)cnt * 32u;
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
        const double2 a = X[min(base + k * kThreads + tid, P - 1)];
        tx[k] = a.x;
        ty[k] = a.y;
        ux[k] = uy[k] = 0.0;
    }
    const int last_target = min(base + T * kThreads, P) - 1;
    const int span_begin = (base / npts) * npts;
    const int span_end = (last_target / npts + 1) * npts;

    for (int i = 0; i < nt; ++i) {
        const int s = i % kStages;
        if (tid == 0 && i >= 1 && i - 1 + kStages < nt) {
            mbar_wait(&empty_bar[(i - 1) % kStages], ((i - 1) / kStages) & 1);
            issue(i - 1 + kStages);
        }
        mbar_wait(&full_bar[s], (i / kStages) & 1);

        const int first = (t_begin + i) * kTile;
        const double4 *ts = tile[s];
        const bool fast = (first >= span_end || first + kTile <= span_begin) && (first + kTile <= P);
        if (fast) {
            double px[T], py[T];
#pragma unroll
            for (int k = 0; k < T; ++k) px[k] = py[k] = 0.0;
#pragma unroll 2
            for (int j = 0; j < kTile; ++j) {
                const double4 sj = ts[j];
#pragma unroll
                for (int k = 0; k < T; ++k) {
                    const double rx = tx[k] - sj.x, ry = ty[k] - sj.y;
                    const double r2 = fma(rx, rx, ry * ry);
                    double ml, inv;
                    log_rcp_f64(r2, ml, inv);
                    const double q = fma(rx, sj.z, ry * sj.w) * inv;
                    px[k] = fma(ml, sj.z, fma(q, rx, px[k]));
                    py[k] = fma(ml, sj.w, fma(q, ry, py[k]));
                }
            }
#pragma unroll
            for (int k = 0; k < T; ++k) { ux[k] += px[k]; uy[k] += py[k]; }
        } else {
            const int cnt = min(kTile, P - first);
#pragma unroll
            for (int k = 0; k < T; ++k) {
                const int own = (min(base + k * kThreads + tid, P - 1) / npts) * npts;
                double px = 0.0, py = 0.0;
#pragma unroll 1
                for (int j = 0; j < cnt; ++j) {
                    const double4 sj = ts[j];
                    const double rx = tx[k] - sj.x, ry = ty[k] - sj.y;
                    const double r2 = fma(rx, rx, ry * ry);
                    if ((unsigned)(first + j - own) >= (unsigned)npts) {
                        double ml, inv;
                        log_rcp_f64(r2, ml, inv);
                        const double q = fma(rx, sj.z, ry * sj.w) * inv;
                        px = fma(ml, sj.z, fma(q, rx, px));
                        py = fma(ml, sj.w, fma(q, ry, py));
                    }
                }
                ux[k] += px;
                uy[k] += py;
            }
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty_bar[s]);
    }

    double2 *out = part + (size_t)sc * (size_t)P;
#pragma unroll
    for (int k = 0; k < T; ++k) {
        const int i0 = base + k * kThreads + tid;
        if (i0 < P) out[i0] = make_double2(ux[k], uy[k]);
    }
}

__global__ void finish_f64(const double2 *__restrict__ part, int P, int n_chunks, double scale,
                           double2 *__restrict__ U)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P) return;
    double sx = 0.0, sy = 0.0;
    for (int c = 0; c < n_chunks; ++c) {
        const double2 v = part[(size_t)c * (size_t)P + i];
        sx += v.x;
        sy += v.y;
    }
    U[i] = make_double2(scale * sx, scale * sy);
}

vn_status farfield_f64(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                       void *U, cudaStream_t st)
{
    const int P = (int)(nves * npts);
    static int slots = 0;
    if (slots == 0) {
        int dev = 0, sms = 0, occ = 0;
        VN_CUDA(cudaGetDevice(&dev));
        VN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        VN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, farfield_f64_kernel, kThreads, 0));
        slots = sms * (occ > 0 ? occ : 1);
    }
    const Split sp = choose_split(P, kT64 * kThreads, slots, 8);

    double4 *src = nullptr;
    double2 *part = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&src, (size_t)P * sizeof(double4), st));
    VN_CUDA(cudaMallocAsync((void **)&part, (size_t)P * sizeof(double2) * (size_t)sp.n_chunks, st));

    pack_sources_f64<<<(P + 255) / 256, 256, 0, st>>>((const double2 *)X, (const double2 *)F, (const double *)W, P, src);
    profile_mark(st, true);
    farfield_f64_kernel<<<sp.n_tb * sp.n_chunks, kThreads, 0, st>>>(src, (const double2 *)X, P, (int)npts, sp.n_tiles,
                                                                   sp.n_chunks, part);
    profile_mark(st, false);
    finish_f64<<<(P + 255) / 256, 256, 0, st>>>(part, P, sp.n_chunks, 1.0 / (4.0 * 3.14159265358979323846 * mu),
                                                 (double2 *)U);
    count_launch(3);
    const cudaError_t e = cudaGetLastError();
    VN_CUDA(cudaFreeAsync(src, st));
    VN_CUDA(cudaFreeAsync(part, st));
    return e == cudaSuccess ? VN_OK : VN_ERR_CUDA;
}

}  // namespace vn

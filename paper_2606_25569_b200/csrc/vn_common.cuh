// vn_common.cuh -- shared device helpers for the sm_100a far-field kernels.
// PTX wrappers only (mbarrier, 1-D bulk async copy, packed f32x2 math, SFU ops) plus the
// work decomposition used by both precisions.  No arithmetic of the method lives here.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/vesnet_farfield.h"

namespace vn {

typedef unsigned long long u64;

constexpr int kThreads = 128;      // threads per block in the pair kernels (4 warps)
constexpr int kTile = 128;         // sources per shared-memory tile
constexpr int kStages = 4;         // tiles in flight per block
constexpr int kSmallPoints = 1024; // vn_farfield of at most this many points is ONE launch (vn_farfield_small.cu)

// ---------------------------------------------------------------------------------------------
// launch bookkeeping (vn_launch_count)
extern unsigned long long g_launches;
inline void count_launch(int n = 1) { __atomic_fetch_add(&g_launches, (unsigned long long)n, __ATOMIC_RELAXED); }

// per-device caches (occupancy, function attributes, capability check) are indexed by the current device
constexpr int kMaxDevices = 64;
inline int current_device()
{
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= kMaxDevices) d = 0;
    return d;
}

// optional event pair around the pair kernel (vn_profile_enable / vn_profile_read)
void profile_mark(cudaStream_t st, bool begin);

#define VN_CUDA(call)                                   \
    do {                                                \
        cudaError_t e_ = (call);                        \
        if (e_ != cudaSuccess) { (void)cudaGetLastError(); return VN_ERR_CUDA; } \
    } while (0)

// ---------------------------------------------------------------------------------------------
// work decomposition: a block is (target block tb, source chunk sc); chunk sc covers tiles
// [tile_begin(sc), tile_begin(sc+1)).  Host and device use the same formula.
__host__ __device__ inline int chunk_tile_begin(int n_tiles, int n_chunks, int sc)
{
    return (int)(((long long)n_tiles * sc) / n_chunks);
}

struct Split {
    int n_tb;        // target blocks
    int n_tiles;     // source tiles of kTile points
    int n_chunks;    // source chunks (grid = n_tb * n_chunks)
};

// One-directional kernels (free targets): choose the number of source chunks so that the grid fills
// `slots` resident blocks in whole waves while each chunk keeps >= min_tiles tiles.
Split choose_split_for(int n_tb, int n_tiles, int slots, int min_tiles);

// Symmetric (both-direction) decomposition of the pair kernels of both precisions: block = (super-tile I,
// chunk c of I's source-tile list); see vn_farfield_f32.cu and choose_sym_split() in vn_api.cu.
struct SymSplit {
    int n_st;        // super-tiles (target blocks)
    int n_tiles;     // source tiles of kTile points
    int n_chunks;    // chunks of the per-super-tile list (grid = n_st * n_chunks)
};
SymSplit choose_sym_split(long long P, int super_tile, int slots, int min_tiles, int max_tiles);

// exclusive scan of int counts into 64-bit offsets (kernels in vn_near.cu, also used by vn_fmm.cu)
constexpr int kScanThreads = 256;
constexpr int kScanItems = 4;
constexpr int kScanBlock = kScanThreads * kScanItems;

// ---------------------------------------------------------------------------------------------
// shared-memory / mbarrier / bulk-copy PTX
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(u64 *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(u64 *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(u64 *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(u64 *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "VN_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra VN_DONE;\n"
        "bra VN_WAIT;\n"
        "VN_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// 1-D bulk asynchronous copy global -> shared (TMA engine, SASS UBLKCP); completes on `bar`.
// dst, src 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, u64 *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// Stage hand-back of the tile ring without anybody waiting: every warp counts itself out of stage s when it
// has read the tile; the warp that makes the count a multiple of the block's warp count was the last one out
// and refills the stage itself.  (A warp cannot run a whole ring ahead -- the refill it would need is only
// issued once all warps have left -- so the count identifies the last warp exactly.)  The fences order the
// warps' shared-memory reads before the bulk copy that overwrites the stage (generic -> async proxy).
__device__ __forceinline__ bool stage_last_out(int *drained, int warps)   // call from one lane per warp
{
    __threadfence_block();
    const int left = atomicAdd(drained, 1) + 1;
    if (left % warps != 0) return false;
    __threadfence_block();
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    return true;
}

// ---------------------------------------------------------------------------------------------
// 64-bit fixed-point accumulation of fp32 results across blocks (bitwise reproducible).
// Power-of-two scale of the fixed-point accumulators.  gmax = max_j (|g_jx| + |g_jy|).  Every term of
// the sum is bounded by (|ln2/2 * lg2 r2| + 1) |g_j| <= 64 gmax (|lg2| <= 150 over all positive fp32),
// so every partial sum of any subset is below bnd = 64 P gmax; 2^(61-e) with 2^e <= bnd < 2^(e+1)
// keeps |value * scale| < 2^62.
__device__ __forceinline__ double fixed_scale(unsigned gmax_bits, int P)
{
    const float gmax = __uint_as_float(gmax_bits);
    if (!(gmax > 0.f) || !(gmax <= 3.4028234e38f)) return 1.0;   // all-zero (or non-finite) density
    const double bnd = 64.0 * (double)P * (double)gmax;
    const int e = ((__double2hiint(bnd) >> 20) & 0x7ff) - 1023;
    return __hiloint2double((1023 + 61 - e) << 20, 0);
}

__device__ __forceinline__ void red_fixed(long long *addr, float v, double scale)
{
    const long long q = __double2ll_rn((double)v * scale);
    atomicAdd((unsigned long long *)addr, (unsigned long long)q);
}

// fp64 results: two 64-bit words per value.  The high word counts units of 1/s_hi (s_hi as above, with
// the term bound 512 gmax because |ln r2|/2 <= 355 over all positive doubles), the low word counts
// units of 2^-40/s_hi and receives the EXACT remainder v - hi/s_hi (an fma), rounded to that unit.
// A contribution therefore enters with an absolute error <= 2^-102 of the bound -- far below double
// rounding of the sum -- and, integer addition being associative, the total is bitwise reproducible.
// The remainder is below 2^39 units per contribution, so 2^23 contributions cannot overflow the low word.
struct Fixed2 {
    double s_hi, inv_s_hi, s_lo;
};
__device__ __forceinline__ Fixed2 fixed2_scale(unsigned long long gmax_bits, int P)
{
    const double gmax = __longlong_as_double((long long)gmax_bits);
    Fixed2 f;
    int ex = 1023 + 61;
    if (gmax > 0.0 && gmax <= 1.0e300) {
        const double bnd = 512.0 * (double)P * gmax;
        ex = 1023 + 61 - (((__double2hiint(bnd) >> 20) & 0x7ff) - 1023);
        ex = ex < 1 ? 1 : (ex > 2000 ? 2000 : ex);
    }
    f.s_hi = __hiloint2double(ex << 20, 0);
    f.inv_s_hi = __hiloint2double((2046 - ex) << 20, 0);
    f.s_lo = __hiloint2double((ex + 40) << 20, 0);
    return f;
}
// which = 0: the high word of v, which = 1: the low word
__device__ __forceinline__ long long fixed2_word(double v, const Fixed2 &f, int which)
{
    const long long qh = __double2ll_rn(v * f.s_hi);
    if (which == 0) return qh;
    const double rem = fma(-(double)qh, f.inv_s_hi, v);
    return __double2ll_rn(rem * f.s_lo);
}
__device__ __forceinline__ void red_fixed2(long long *addr, double v, const Fixed2 &f)   // addr[0] hi, addr[1] lo
{
    atomicAdd((unsigned long long *)addr + 0, (unsigned long long)fixed2_word(v, f, 0));
    atomicAdd((unsigned long long *)addr + 1, (unsigned long long)fixed2_word(v, f, 1));
}
__device__ __forceinline__ double fixed2_value(long long hi, long long lo, const Fixed2 &f)
{
    const long long carry = lo >> 40;               // move whole high units out of the low word
    hi += carry;
    lo -= carry << 40;
    return (double)hi * f.inv_s_hi + ((double)lo * f.inv_s_hi) * 9.094947017729282379e-13;   // 2^-40
}

// near-field correction (vn_near.cu), used by the masked variants of both precisions: subtracts the
// near vesicles' contributions from the fixed-point accumulators before the final rounding
vn_status near_correction_f32(const void *X, const void *F, const void *W, int P, int npts, const int64_t *near_ptr,
                              const int32_t *near_ves, long long *acc, const unsigned *gmax_bits, cudaStream_t st);
vn_status near_correction_accum(const void *X, const void *F, const void *W, int P, int npts, const int64_t *near_ptr,
                                const int32_t *near_ves, double2 *accum, vn_precision prec, cudaStream_t st);
vn_status near_correction_f64(const void *X, const void *F, const void *W, int P, int npts, const int64_t *near_ptr,
                              const int32_t *near_ves, long long *acc, const unsigned long long *gmax_bits,
                              cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// packed fp32 pairs (sm_100 FADD2 / FMUL2 / FFMA2) and single-instruction SFU ops
__device__ __forceinline__ u64 pk(float lo, float hi)
{
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk(u64 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 add2(u64 a, u64 b)
{
    u64 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 sub2(u64 a, u64 b)
{
    u64 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b)
{
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c)
{
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ float sfu_rcp(float x)   // MUFU.RCP
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float sfu_lg2(float x)   // MUFU.LG2
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

}  // namespace vn

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

// ---------------------------------------------------------------------------------------------
// launch bookkeeping (vn_launch_count)
extern unsigned long long g_launches;
inline void count_launch(int n = 1) { __atomic_fetch_add(&g_launches, (unsigned long long)n, __ATOMIC_RELAXED); }

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

// Choose the number of source chunks so that the grid fills `slots` resident blocks in whole
// waves (wave quantisation) while each chunk keeps >= min_tiles tiles.
Split choose_split(long long P, int targets_per_block, int slots, int min_tiles);

// Symmetric (both-direction) decomposition of the fp32 kernel: block = (super-tile I, chunk c of I's
// source-tile list); see vn_farfield_f32.cu.
struct SymSplit {
    int n_st;        // super-tiles (target blocks)
    int n_tiles;     // source tiles of kTile points
    int n_chunks;    // chunks of the per-super-tile list (grid = n_st * n_chunks)
};
SymSplit choose_sym_split(long long P, int super_tile, int slots, int min_tiles);

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

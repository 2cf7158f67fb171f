// Shared device helpers of the cc_ladder kernels (sm_100a).  Product code: nothing here is used by oracle/.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

namespace ccl {

// ------------------------------------------------------------------------------------------------ DMMA
// The only native FP64 tensor instruction on sm_100a: mma.sync m8n8k4 -> SASS DMMA.8x8x4
// (128 flop/clk/SM measured, profiles/round1_microbench.md).  Lane l: g = l>>2, q = l&3.
//   A (8x4, row):  a   = A[g][q]          B (4x8, col):  b   = B[q][g]
//   C/D (8x8):     c0  = C[g][2q]         c1 = C[g][2q+1]
__device__ __forceinline__ void dmma_8x8x4(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// ------------------------------------------------------------------------------------------------ cp.async
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// 16-byte global->shared copy; when !valid nothing is read and the 16 bytes are zero-filled.
__device__ __forceinline__ void cp_async_16(uint32_t dst, const void *src, bool valid)
{
    int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}

// 8-byte variant for operands whose rows are only 8-byte aligned (odd nvirt).
__device__ __forceinline__ void cp_async_8(uint32_t dst, const void *src, bool valid)
{
    int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}

__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }

template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

// ------------------------------------------------------------------------------------------------ mbarrier
// Shared-memory barriers used as "slab landed" flags: every thread's cp.async batch arrives on the barrier when its
// copies complete (no increment of the pending count: the barrier is initialised with the thread count).
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}

__device__ __forceinline__ void cp_async_mbar_arrive(uint32_t bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "CCL_MBAR_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra CCL_MBAR_DONE;\n"
        "bra CCL_MBAR_WAIT;\n"
        "CCL_MBAR_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

// Non-blocking probe of a phase (true: the phase with this parity has completed).  Issued a k-step ahead of the
// blocking wait, so that the barrier round trip overlaps the DMMA stream.
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}

// ------------------------------------------------------------------------------------------------ CTA pairs
// Split mode runs clusters of two CTAs that exchange their (ac|bd) / (ad|bc) tiles through distributed shared memory.
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(r));
    return r;
}

__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n"
                 "barrier.cluster.wait.acquire.aligned;\n" ::
                     : "memory");
}

__device__ __forceinline__ uint32_t map_to_cta(uint32_t smem_addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}

__device__ __forceinline__ void st_cluster_f64x2(uint32_t addr, double a, double b)
{
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};\n" ::"r"(addr), "d"(a), "d"(b) : "memory");
}

// ------------------------------------------------------------------------------------------------ reductions into R
// Fire-and-forget FP64 add performed by the L2 atomic unit (SASS RED.E.ADD.F64).
__device__ __forceinline__ void red_add_f64(double *p, double v)
{
    asm volatile("red.global.add.f64 [%0], %1;\n" ::"l"(p), "d"(v) : "memory");
}

// Same, predicated inside the instruction stream (no branch around it; nothing is accessed when !on).
__device__ __forceinline__ void red_add_f64_if(double *p, double v, bool on)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.s32 p, %2, 0;\n"
        "@p red.global.add.f64 [%0], %1;\n"
        "}\n" ::"l"(p),
        "d"(v), "r"((int)on)
        : "memory");
}

__host__ __device__ __forceinline__ int ceil_div(int a, int b) { return (a + b - 1) / b; }

// ------------------------------------------------------------------------------------------------ packed triangles
// Split (t+/t-) mode keeps T+-, W+- as row-major upper triangles (csrc/ladder_split.cuh) whose rows
// are aligned for 128-bit copies and full-sector reductions: element (c,d), d >= c, of a row-(i,j) triangle sits at
// tri_base(c) + d, where row c owns the slot d in [4*floor(c/4), v4), v4 = nvirt rounded up to a multiple of 4, and
// tri_base(c) is a multiple of 4.  The up to three slot entries left of the diagonal and the padding d >= nvirt hold
// zeros.  tri_size(v) doubles per (i,j): v^2/2 + O(v) instead of v^2.
__host__ __device__ __forceinline__ long long tri_v4(long long v) { return (v + 3) & ~3LL; }
__host__ __device__ __forceinline__ long long tri_base(long long c, long long v4)
{
    const long long m = c >> 2, r = c & 3;
    return 4 * m * v4 - 8 * m * (m - 1) + r * (v4 - 4 * m) - 4 * m;
}
__host__ __device__ __forceinline__ long long tri_size(long long v)      // = slot start of the (non-existent) row v
{
    const long long v4 = tri_v4(v);
    return tri_base(v, v4) + 4 * (v >> 2);
}

}  // namespace ccl

// Tensor memory (TMEM, 512 columns x 128 lanes x 32 bit per SM) used as a lane-private scratchpad.
//
// No tensor-core instruction is issued anywhere in this library (the path is not a contraction);
// what the warp kernels need is a second place, besides shared memory, to park data that a lane
// writes and later reads back ITSELF: the in-band spectrum E between the two inverse transforms (one
// per polarisation) and |z_theta|^2 of every sample until the phi pass adds |z_phi|^2 to it. With the .32x32b shape of
// tcgen05.ld/st, thread t of warp w owns TMEM lane 32 (w % 4) + t and reads/writes consecutive
// 32-bit columns of it: no bank conflicts by construction, a datapath separate from the LSU /
// shared-memory crossbar (measured on B200, 8 warps/SM: STTM.x2 1.05, LDTM.x2 1.5 cycles per
// 256-byte warp access against 2.0 for LDS.64/STS.64, and the two overlap), and it frees 17.5 KB of
// shared memory per warp. SASS: UTCALLOC / STTM / LDTM.
#pragma once
#include <cstdint>

namespace aera {

// One warp allocates all 512 columns (the kernels run one CTA per SM) and publishes the base
// address through shared memory; the caller follows with tmem_publish_sync().
__device__ __forceinline__ void tmem_alloc_all(uint32_t *base_in_smem)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"
                 ::"r"((uint32_t)__cvta_generic_to_shared(base_in_smem)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_free_all(uint32_t base)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(base) : "memory");
}

// Address of column `col` in the lane quarter that warp `warp` may access.
__device__ __forceinline__ uint32_t tmem_addr(uint32_t base, int warp, int col)
{
    return base + (((uint32_t)(warp & 3) * 32u) << 16) + (uint32_t)col;
}

// 64 bits per thread (two consecutive columns). The address must be warp-uniform.
__device__ __forceinline__ void tmem_st64(uint32_t addr, unsigned long long v)
{
    asm volatile("{\n.reg .b32 lo, hi;\nmov.b64 {lo, hi}, %1;\n"
                 "tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {lo, hi};\n}" ::"r"(addr), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long tmem_ld64(uint32_t addr)
{
    unsigned long long v;
    asm volatile("{\n.reg .b32 lo, hi;\n"
                 "tcgen05.ld.sync.aligned.32x32b.x2.b32 {lo, hi}, [%1];\nmov.b64 %0, {lo, hi};\n}" : "=l"(v) : "r"(addr) : "memory");
    return v;
}
// one 32-bit column per thread
__device__ __forceinline__ uint32_t tmem_ld32(uint32_t addr)
{
    uint32_t v;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void tmem_ld_dep32(uint32_t &a, uint32_t &b)
{
    asm volatile("" : "+r"(a), "+r"(b) :: "memory");
}
// Results of earlier tmem_ld64 calls may be used only after tmem_wait_ld(). The compiler does not
// know that, so each loaded value is then passed through tmem_ld_dep(): an empty volatile asm that
// "rewrites" it. Volatile asms keep their order, so no consumer can be scheduled above the wait.
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld_dep(unsigned long long &a, unsigned long long &b)
{
    asm volatile("" : "+l"(a), "+l"(b) :: "memory");
}
// Earlier tmem_st64 calls of this thread are complete (visible to its later tmem_ld64).
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

} // namespace aera

// umma.cuh -- sm_100a primitives of the tcgen05 GEMV / GEMM consumer (gemv_umma.cuh): tensor-map bulk copies
// (TMA, SASS UTMALDG), tensor memory allocation, tcgen05.mma with shared-memory descriptors (SASS UTCHMMA),
// tcgen05.ld (SASS LDTM), and the fences / commits that order them. No arithmetic of the method lives here.
#pragma once
#include <cuda.h>  // CUtensorMap (type only: the library does not link libcuda; the encoder is fetched at init)

#include "ptx.cuh"

namespace dvt {

// ---- tensor-map bulk copy global -> shared, 3 coordinates, completes on an mbarrier --------------------------
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint "
      "[%0], [%1, {%2, %3, %4}], [%5], %6;" ::"r"(smem_u32(dst)),
      "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}
// One lane of a converged warp. Branching on this (not on lane == 0) tells ptxas that a single thread is active,
// so the uniform-register operands of UTCHMMA / UTMALDG need no per-value waterfall loop.
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}

// ---- tensor memory -------------------------------------------------------------------------------------------
// One warp allocates `cols` columns (power of two >= 32) of the SM's 512 and owns the deallocation.
__device__ __forceinline__ void tmem_alloc(uint32_t* slot, uint32_t cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "r"(cols)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t addr, uint32_t cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// ---- tcgen05.mma, kind::f16 (bf16 x bf16 -> fp32), both operands in shared memory ----------------------------
// Shared-memory matrix descriptor of a K-major tile in the 128-byte swizzled canonical layout: rows of 64
// elements (128 bytes), 8-row groups of 1024 bytes `sbo` bytes apart. The tile base must be 1024-byte aligned;
// a step of 16 elements along K inside the 64-element row is +32 bytes on the start address. The 64-bit descriptor:
// start address >> 4 in bits [0, 14), leading byte offset (unused when swizzled) = 1 at bit 16, stride byte offset >> 4
// in bits [32, 46), descriptor version 1 at bit 46, layout type 2 (128-byte swizzle) at bits [61, 64); it is built as a
// low and a high 32-bit word (umma_desc_lo / umma_desc_hi_sw128 below).
// Instruction descriptor: D fp32, A and B bf16, both K-major, M x N tile (M = 64 or 128, N a multiple of 16).
__host__ __device__ __forceinline__ uint32_t umma_idesc_bf16(int m, int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | (static_cast<uint32_t>(n >> 3) << 17) | (static_cast<uint32_t>(m >> 4) << 24);
}
// D[tmem] (+)= A[smem] * B[smem]^T over 16 elements of K; issued by ONE thread for the CTA. The descriptors come
// as 32-bit halves: one thread issues every MMA of the CTA, so its instruction count per MMA is the tensor
// core's pace at small tiles (measured: building both 64-bit descriptors per MMA cost ~80 cycles each, five
// times the MMA itself); the caller keeps the constant high word and steps the low words (start address >> 4)
// by +2 per 16 k and +64 per slab.
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint32_t a_lo, uint32_t b_lo, uint32_t desc_hi, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t.reg .b64 da, db;\n\t"
      "setp.ne.b32 p, %5, 0;\n\t"
      "mov.b64 da, {%1, %3};\n\t"
      "mov.b64 db, {%2, %3};\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %4, p;\n\t}" ::"r"(tmem_d),
      "r"(a_lo), "r"(b_lo), "r"(desc_hi), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ uint32_t umma_desc_lo(uint32_t smem_addr) { return ((smem_addr & 0x3ffffu) >> 4) | (1u << 16); }
__device__ __forceinline__ uint32_t umma_desc_hi_sw128(uint32_t sbo) { return ((sbo >> 4) & 0x3fffu) | (1u << 14) | (2u << 29); }
// The mbarrier receives one arrival when every tcgen05.mma issued so far by this thread has completed
// (implies tcgen05.fence::before_thread_sync).
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// ---- tensor memory -> registers: lane (= this thread's lane of the warp's 32-lane quarter), 8 consecutive columns.
// The registers are defined only after tmem_ld_wait; tmem_ld_use ties them to it (volatile asm statements keep
// their order, so no use can be scheduled before the wait).
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr)
               : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld_use(uint32_t (&r)[8]) {
  asm volatile("" : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]));
}

}  // namespace dvt

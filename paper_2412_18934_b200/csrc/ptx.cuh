// ptx.cuh -- sm_100a primitives used by the draft-step kernels: mbarrier,
// 1-D bulk async copy (TMA, SASS UBLKCP), programmatic dependent launch,
// packed fp32 FMA, warp reductions. No arithmetic of the method lives here.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dvt {

constexpr int kConsumerWarps = 8;
constexpr int kConsumerThreads = kConsumerWarps * 32;  // 256
constexpr int kThreads = kConsumerThreads + 32;        // + one producer warp

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// ---- mbarrier ---------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
// Bounded wait: a protocol bug becomes a trap (a CUDA error the host reports)
// instead of a hung GPU.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t spins = 0;
  while (!mbar_try_wait(bar, parity)) {
    if (++spins > (1u << 24)) __trap();
  }
}

// ---- bulk async copy global -> shared (TMA 1-D), completes on an mbarrier ---
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
// dst, src and bytes must be multiples of 16.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar,
                                         uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint "
      "[%0], [%1], %2, [%3], %4;" ::"r"(smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}

// ---- programmatic dependent launch -----------------------------------------
// wait: all memory of the preceding kernels in the stream is visible after it.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// lets the next kernel in the stream start its weight prefetch early
__device__ __forceinline__ void pdl_launch_dependents() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// ---- per-launch time stamps (dovetail_hooks.h dovetail_trace_*): t[0] = earliest CTA start,
// t[1] = latest CTA end, in ns of %globaltimer. t == NULL (the default) costs one predicate.
__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ void trace_begin(unsigned long long* t) {
  if (t != nullptr && threadIdx.x == 0) atomicMin(t, globaltimer_ns());
}
__device__ __forceinline__ void trace_end(unsigned long long* t) {
  if (t != nullptr && threadIdx.x == 0) atomicMax(t + 1, globaltimer_ns());
}

// ---- grid-wide phase barrier of a persistent kernel (all CTAs resident: one per SM) -----------
// arrive: the calling thread's CTA has finished the phase; its global writes were made visible by
// __threadfence() of the writing threads + a CTA barrier before this call.
__device__ __forceinline__ void grid_arrive(int32_t* counter) {
  asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(counter) : "memory");
}
__device__ __forceinline__ int32_t ld_acquire_gpu(const int32_t* p) {
  int32_t v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// Bounded like mbar_wait: a protocol bug traps instead of hanging the GPU.
__device__ __forceinline__ void grid_wait(const int32_t* counter, int32_t target) {
  uint32_t spins = 0;
  while (ld_acquire_gpu(counter) < target) {
    if (++spins > (1u << 24)) __trap();
  }
}
// generic-proxy writes (st.global by other CTAs, observed through an acquire) before async-proxy reads
// (bulk copies) of the same global memory
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// ---- named barrier among the consumer warps only ---------------------------
__device__ __forceinline__ void consumer_sync() {
  asm volatile("bar.sync 1, %0;" ::"n"(kConsumerThreads) : "memory");
}

// ---- packed fp32 FMA: d.x += a.x*b.x, d.y += a.y*b.y ------------------------
__device__ __forceinline__ void ffma2(float2& d, const float2& a, const float2& b) {
#if defined(DVT_NO_FFMA2)
  d.x = fmaf(a.x, b.x, d.x);
  d.y = fmaf(a.y, b.y, d.y);
#else
  uint64_t& dd = reinterpret_cast<uint64_t&>(d);
  asm("fma.rn.f32x2 %0, %1, %2, %0;"
      : "+l"(dd)
      : "l"(reinterpret_cast<const uint64_t&>(a)), "l"(reinterpret_cast<const uint64_t&>(b)));
#endif
}

// two bf16 packed in a 32-bit word -> (low element, high element) as fp32, exact
__device__ __forceinline__ float2 bf16x2_to_f32x2(uint32_t w) {
  return make_float2(__uint_as_float(w << 16), __uint_as_float(w & 0xffff0000u));
}

// fp32 -> bf16 bits, round to nearest even (finite inputs)
__device__ __forceinline__ uint16_t f32_to_bf16_rn(float f) {
  uint32_t u = __float_as_uint(f);
  u += 0x7fffu + ((u >> 16) & 1u);
  return static_cast<uint16_t>(u >> 16);
}

// ---- warp reductions --------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Transposing reduction of V (power of two, <= 32) per-lane values over the 32
// lanes. On return v[0] of every lane holds the warp total of value index
// lane / (32 / V). Fixed order, V - 1 + log2(32 / V) shuffles.
template <int V>
__device__ __forceinline__ float warp_reduce_transpose(float (&v)[V], int lane) {
  static_assert(V >= 1 && V <= 32 && (V & (V - 1)) == 0, "V must be a power of two");
  int dist = 16;
#pragma unroll
  for (int h = V / 2; h >= 1; h >>= 1) {
    const bool up = (lane & dist) != 0;
#pragma unroll
    for (int i = 0; i < h; ++i) {
      const float send = up ? v[i] : v[i + h];
      const float keep = up ? v[i + h] : v[i];
      v[i] = keep + __shfl_xor_sync(0xffffffffu, send, dist);
    }
    dist >>= 1;
  }
  float r = v[0];
  for (; dist >= 1; dist >>= 1) r += __shfl_xor_sync(0xffffffffu, r, dist);
  return r;
}

}  // namespace dvt

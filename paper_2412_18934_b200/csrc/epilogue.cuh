// epilogue.cuh -- the fused epilogues shared by the two weight-streaming GEMV kernels (gemv.cuh: fp32 FMA,
// gemv_mma.cuh: bf16 tensor cores): what happens to a CTA's results Y[m, n] before they leave the SM
// (SURVEY.md 8a S1, S2, S4, S5, S6).
//
// Besides the fp32 result every epilogue that feeds a later GEMV also leaves the activation in the form the
// tensor-core kernel consumes as its B operand: each fp32 value split exactly into three bf16 terms
// x = x0 + x1 + x2 (all 24 mantissa bits), one plane per term, [plane][row][k] in global memory. The
// consumer copies K-chunks of those planes into its ring with bulk async copies; it converts nothing. Where
// the consumer applies RMSNorm the gain is folded into the planes here (x * g is split), and the sum of
// squares of the raw x over this CTA's columns goes to ssq_out[cta][row]; the consumer adds the partials
// of all CTAs in CTA order and scales its results by 1 / rms (pre-norm LLaMA block).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "ptx.cuh"
#include "state.cuh"

namespace dvt {

constexpr int kSplitPlanes = 3;

struct SplitOut {
  __nv_bfloat16* xs;  // [kSplitPlanes][rows][ld] or NULL: nothing to leave
  int64_t plane;      // elements between planes
  int64_t ld;         // elements between rows (>= K of the consumer, multiple of 8)
  int32_t perm;       // 1: int8 weights -- the terms are fp16 with rescaled remainders (store_split; the int8 consumer
                      // multiplies in fp16) and, within every aligned block of 32 k, stored in the order the
                      // consumer's fragments need (split_pos); 0: bf16 terms in natural order
};

// int8 weights (gemv_mma.cuh, WQ = 1): one ldmatrix gives a thread the weights k = 4t .. 4t + 3 and 16 + 4t .. 16 +
// 4t + 3 of a 32-block (t = lane & 3), i.e. the pairs (4t, 4t+1), (16+4t, ..) for the first mma and (4t+2, 4t+3),
// (18+4t, ..) for the second. The activation planes are stored so that a plain ldmatrix of B delivers exactly
// those pairs: k = 16a + 4t + 2b + e  ->  position 8(a + 2b) + 2t + e.
__device__ __forceinline__ int64_t split_pos(int64_t col, int perm) {
  if (!perm) return col;
  const int k = static_cast<int>(col & 31);
  const int a = k >> 4, t = (k >> 2) & 3, b = (k >> 1) & 1, e = k & 1;
  return (col & ~static_cast<int64_t>(31)) + 8 * (a + 2 * b) + 2 * t + e;
}

__device__ __forceinline__ void store_split(const SplitOut& o, int64_t row, int64_t col, float x) {
  if (o.perm) {
    // fp16 terms with rescaled remainders: x = h0 + 2^-11 h1 + 2^-22 h2, h1 = fp16((x - h0) 2^11), h2 likewise, so
    // that the remainders sit in fp16's normal range whatever the magnitude of x (a plain x - h0 of a small x is
    // subnormal: measured 9x the error on features of magnitude 1e-2). The consumer applies the powers of two when
    // it adds the terms' dot products. Needs |x| < 65504.
    const __half h0 = __float2half_rn(x);
    const float r1 = (x - __half2float(h0)) * 2048.0f;
    const __half h1 = __float2half_rn(r1);
    const __half h2 = __float2half_rn((r1 - __half2float(h1)) * 2048.0f);
    __half* dst = reinterpret_cast<__half*>(o.xs) + row * o.ld + split_pos(col, 1);
    dst[0] = h0;
    dst[o.plane] = h1;
    dst[2 * o.plane] = h2;
    return;
  }
  const uint16_t h0 = f32_to_bf16_rn(x);
  const float r1 = x - __uint_as_float(static_cast<uint32_t>(h0) << 16);
  const uint16_t h1 = f32_to_bf16_rn(r1);
  const float r2 = r1 - __uint_as_float(static_cast<uint32_t>(h1) << 16);
  uint16_t* dst = reinterpret_cast<uint16_t*>(o.xs) + row * o.ld + split_pos(col, o.perm);
  dst[0] = h0;
  dst[o.plane] = h1;
  dst[2 * o.plane] = f32_to_bf16_rn(r2);
}

// fp32 rows -> split-bf16 planes (epilogue.cuh). Batched loads, then the stores.
__device__ __forceinline__ void split_row(const SplitOut& so, int64_t row, const float* src, int d) {
  constexpr int B = 8;
  for (int k0 = threadIdx.x; k0 < d; k0 += blockDim.x * B) {
    float v[B];
#pragma unroll
    for (int i = 0; i < B; ++i) {
      const int k = k0 + i * blockDim.x;
      v[i] = k < d ? __ldg(src + k) : 0.f;
    }
#pragma unroll
    for (int i = 0; i < B; ++i) {
      const int k = k0 + i * blockDim.x;
      if (k < d) store_split(so, row, k, v[i]);
    }
  }
}

__device__ __forceinline__ float load_storage(const void* p, int64_t i, bool bf16) {
  return bf16 ? __bfloat162float(static_cast<const __nv_bfloat16*>(p)[i]) : static_cast<const float*>(p)[i];
}

__device__ __forceinline__ float sigmoidf_acc(float z) { return 1.0f / (1.0f + expf(-z)); }

// strict order of LM-head candidates: logit descending, token id ascending (reading A7)
__device__ __forceinline__ bool cand_before(float va, int ia, float vb, int ib) {
  return va > vb || (va == vb && ia < ib);
}

constexpr int kNoCand = 0x7fffffff;  // id of the "no candidate" entry (value -inf): after every real candidate
// A candidate (value, id) as an order-preserving pair of unsigned words: (key, lo) compares like cand_before
// (larger value first, then smaller id). key 0 = no candidate (below every real value, -inf included);
// -0 is canonicalised to +0 (cand_before treats them as equal). ids < 2^24 (dovetail_draft_init checks the vocabulary).
__device__ __forceinline__ uint32_t cand_key(float v, int id) {
  const uint32_t u = __float_as_uint(v + 0.f);
  return id == kNoCand ? 0u : ((u >> 31) ? ~u : (u | 0x80000000u));
}
__device__ __forceinline__ uint32_t cand_lo(int id, int cta) {
  return id == kNoCand ? 0u : ((static_cast<uint32_t>(0xffffff - id) << 8) | static_cast<uint32_t>(cta));
}
__device__ __forceinline__ float cand_key_value(uint32_t key) {
  return key == 0u ? -INFINITY : __uint_as_float((key >> 31) ? (key & 0x7fffffffu) : ~key);
}
__device__ __forceinline__ uint64_t umax64(uint64_t a, uint64_t b) { return a > b ? a : b; }

}  // namespace dvt

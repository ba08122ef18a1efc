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

#include "ptx.cuh"
#include "state.cuh"

namespace dvt {

constexpr int kSplitPlanes = 3;

struct SplitOut {
  __nv_bfloat16* xs;  // [kSplitPlanes][rows][ld] or NULL: nothing to leave
  int64_t plane;      // elements between planes
  int64_t ld;         // elements between rows (>= K of the consumer, multiple of 8)
};

__device__ __forceinline__ void store_split(const SplitOut& o, int64_t row, int64_t col, float x) {
  const uint16_t h0 = f32_to_bf16_rn(x);
  const float r1 = x - __uint_as_float(static_cast<uint32_t>(h0) << 16);
  const uint16_t h1 = f32_to_bf16_rn(r1);
  const float r2 = r1 - __uint_as_float(static_cast<uint32_t>(h1) << 16);
  uint16_t* dst = reinterpret_cast<uint16_t*>(o.xs) + row * o.ld + col;
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

}  // namespace dvt

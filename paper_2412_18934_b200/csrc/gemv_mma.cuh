// gemv_mma.cuh -- tensor-core consumer for the weight-streaming GEMV (bf16
// weights; S1 DGF, S2 QKV, S4 O-proj, S5 FFN, S6 LM head).
//
//   Y[m, n] = sum_k X[m, k] * W[n, k]      m < M <= 32 draft rows, W bf16 row-major [N, K]
//
// "Swap-AB": the weights are the 16 x 16 A operand of mma.sync.m16n8k16 (bf16 in,
// fp32 accumulate) and the draft rows are the 8 columns of B, so every weight
// byte is read from HBM once whatever M is. The fp32 activations are not
// rounded to bf16: each x is split exactly into S bf16 terms, x = x0 + x1 (+ x2)
// (S = 3 keeps all 24 mantissa bits, S = 2 keeps 16), one B column per term, and
// the S columns of a row are added in the epilogue. Products bf16 x bf16 are
// exact in fp32, so the result is an fp32-accumulated dot product of the fp32
// activations with the stored weights.
//
// The split is done ONCE, by the kernel that produced the activation
// (epilogue.cuh): this kernel finds the planes [s][row][k] in global memory (L2)
// and converts nothing. Shape of the kernel (one CTA per SM, 8 consumer warps +
// 4 weight-producer warps + 1 activation-producer warp):
//   * rows are dealt to the CTAs in contiguous ranges differing by <= 1 row
//     (same as k_gemv), and processed in super-blocks of RS <= 64 rows;
//   * a ring stage holds one K-chunk (KC elements) of every row of the
//     super-block (A part) and of every B column (B part), each row padded by
//     16 bytes, which makes the ldmatrix reads bank-conflict free. The weight
//     producers fill the A parts with 1-D bulk async copies (row-exact: no byte
//     of another CTA's rows is touched) and start before griddepcontrol.wait,
//     because weights never depend on activations; the activation producer
//     waits for the previous kernel, then copies the matching chunk of each
//     plane row (from L2) into the B part. Separate "full" barriers, one
//     "empty" barrier per stage;
//   * consumer warp w owns the k-units w, w + 8, ... (32 k each) of every
//     chunk, loads its B fragments once per unit (ldmatrix.x4) and reuses them
//     for all row blocks of the stage (ldmatrix.x4 of A + NT mma each);
//   * accumulators stay in registers for a whole super-block (all of K); only
//     then do the warps meet: partials go to shared memory, one named barrier,
//     and a fixed-order sum over the 8 warps and the S split columns
//     (deterministic);
//   * RMSNorm of the input costs nothing here: the gain is folded into the
//     planes and 1 / rms comes from the producers' partial sums of squares;
//   * the fused epilogues (gemv.cuh gemv_epilogue) run once over the CTA's
//     results and leave the planes for the next GEMV.
// There is no barrier inside the streaming loop and no prologue before it.
#pragma once
#include <cuda_bf16.h>

#include "gemv.cuh"
#include "ptx.cuh"
#include "state.cuh"

namespace dvt {

constexpr int kMmaMaxM = 32;
// A 1-D bulk copy costs its issuing warp ~35 ns whatever its size (measured: one producer warp
// moves 2.4 TB/s chip-wide with 512-byte copies, four move 7.2 TB/s), so four warps produce.
constexpr int kMmaProducerWarps = 4;
constexpr int kMmaThreads = kConsumerThreads + 32 * (kMmaProducerWarps + 1);

__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(addr)
               : "memory");
}

__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__device__ __forceinline__ uint32_t pack_bf16x2_rn(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}

// NT: 8-column tiles of B (columns = M * S <= 8 * NT); RBMAX: 16-row blocks per stage.
template <int NT, int RBMAX>
__global__ void __launch_bounds__(kMmaThreads, 1) k_gemv_mma(const GemvParams p) {
  extern __shared__ __align__(128) uint8_t smem[];
  const GemvGroup& G = p.g[blockIdx.y];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nct = gridDim.x, c = blockIdx.x;
  const int NS = p.n_stages, RS = p.rows_per_stage, KC = p.kc, K = p.K, M = p.M, S = G.S;
  const int ncols = M * S, PC = (ncols + 1) & ~1;
  const uint32_t b_off = static_cast<uint32_t>(RS) * p.seg_stride;  // B part of a stage

  uint8_t* ring = smem;
  uint64_t* full_a = reinterpret_cast<uint64_t*>(smem + static_cast<size_t>(NS) * p.stage_bytes);
  uint64_t* full_b = full_a + 8;
  uint64_t* empty = full_b + 8;
  uint32_t* zero16 = reinterpret_cast<uint32_t*>(empty + 8);  // B columns past ncols read these zeros
  float* rstd_s = reinterpret_cast<float*>(zero16 + 4);  // [32]
  float* part = rstd_s + kMmaMaxM;  // [warps][RS][PC]
  float* res = part + static_cast<size_t>(kConsumerWarps) * RS * PC;  // [cnt][M]

  const RowRange rr = cta_rows(G, c, nct);
  const int n_sb = (rr.cnt + RS - 1) / RS;
  trace_begin(p.trace);

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full_a[s], kMmaProducerWarps);
      mbar_init(&full_b[s], 1);
      mbar_init(&empty[s], kConsumerWarps);
    }
    mbar_fence_init();
  }
  if (tid < 4) zero16[tid] = 0u;
  __syncthreads();
  pdl_launch_dependents();

  if (warp >= kConsumerWarps + kMmaProducerWarps) {
    // ---------------- activation producer: one B column per lane (two when ncols > 32) -----------
    pdl_wait();  // the planes were written by the previous kernels
    const uint64_t pol = l2_policy_evict_last();
    const uint8_t* src[2] = {nullptr, nullptr};
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int col = lane + 32 * h;
      if (col < ncols) {
        const int m = col / S, s = col - m * S;
        if (G.xkind == X_ROWS) {
          const int64_t ri = G.xidx ? G.xidx[p.m0 + m] : p.m0 + m;
          src[h] = reinterpret_cast<const uint8_t*>(G.xs + s * G.xs_plane + ri * G.xs_ld);
        } else {  // embedding rows are bf16 already: one plane
          src[h] = reinterpret_cast<const uint8_t*>(static_cast<const __nv_bfloat16*>(G.embed) +
                                                    static_cast<size_t>(G.tokens[p.m0 + m]) * K);
        }
      }
    }
    int slot = 0, round = 0;
    for (int sb = 0; sb < n_sb; ++sb) {
      for (int k0 = 0; k0 < K; k0 += KC) {
        if (round > 0) mbar_wait(&empty[slot], (round & 1) ^ 1);
        const uint32_t segb = static_cast<uint32_t>(min(KC, K - k0)) * 2u;
        if (lane == 0) mbar_arrive_expect_tx(&full_b[slot], static_cast<uint32_t>(ncols) * segb);
        __syncwarp();
        uint8_t* dst = ring + static_cast<size_t>(slot) * p.stage_bytes + b_off;
#pragma unroll
        for (int h = 0; h < 2; ++h)
          if (src[h])
            bulk_g2s(dst + static_cast<size_t>(lane + 32 * h) * p.seg_stride, src[h] + static_cast<size_t>(k0) * 2, segb,
                     &full_b[slot], pol);
        if (++slot == NS) { slot = 0; ++round; }
      }
    }
    return;
  }

  if (warp >= kConsumerWarps) {
    // ---------------- weight producers: warp pw copies rows [16 pw, 16 pw + 16) of every stage ---
    const int pw = warp - kConsumerWarps;
    const uint64_t pol = l2_policy_evict_first();
    int slot = 0, round = 0;
    for (int sb = 0; sb < n_sb; ++sb) {
      const int v0 = sb * RS, nr = min(RS, rr.cnt - v0);
      const int r = pw * 16 + (lane & 15);  // this lane's row of the super-block (lanes 0..15)
      const bool mine = lane < 16 && r < nr;
      const int my_rows = max(0, min(16, nr - pw * 16));
      const uint8_t* src = nullptr;
      if (mine) {
        int j, n;
        locate_row(G, rr, v0 + r, j, n);
        src = static_cast<const uint8_t*>(G.w[j]) + static_cast<size_t>(n) * p.row_bytes;
      }
      for (int k0 = 0; k0 < K; k0 += KC) {
        if (round > 0) mbar_wait(&empty[slot], (round & 1) ^ 1);
        const uint32_t segb = static_cast<uint32_t>(min(KC, K - k0)) * 2u;
        if (lane == 0) mbar_arrive_expect_tx(&full_a[slot], static_cast<uint32_t>(my_rows) * segb);
        __syncwarp();
        uint8_t* dst = ring + static_cast<size_t>(slot) * p.stage_bytes;
        if (mine) bulk_g2s(dst + static_cast<size_t>(r) * p.seg_stride, src + static_cast<size_t>(k0) * 2, segb, &full_a[slot], pol);
        if (++slot == NS) { slot = 0; ++round; }
      }
    }
    return;
  }

  // ---------------- consumers -------------------------------------------------
  pdl_wait();  // residual stream, [h1 || h2], partial sums of squares: written by the previous kernels
  if (p.ssq_in) {  // RMSNorm: y = x / sqrt(mean(x^2) + eps) * g; g is in the planes, 1/rms is applied to the results
    for (int m = warp; m < M; m += kConsumerWarps) {  // partials of the producer's CTAs, fixed order
      float t = 0.f;
      for (int cc = lane; cc < p.ssq_nct; cc += 32) t += p.ssq_in[static_cast<int64_t>(cc) * kMaxRows + p.m0 + m];
      t = warp_sum(t);
      if (lane == 0) rstd_s[m] = 1.0f / sqrtf(t / static_cast<float>(K) + p.eps);
    }
  }
  // per-lane ldmatrix address pieces
  const uint32_t ring_u = smem_u32(ring);
  const uint32_t a_lane = static_cast<uint32_t>((lane & 7) + ((lane >> 3) & 1) * 8) * p.seg_stride + (lane >> 4) * 16;
  uint32_t b_lane[NT];   // offset within the B part of a stage, or ~0: the zero block
#pragma unroll
  for (int t = 0; t < NT; ++t) {
    const int col = t * 8 + (lane & 7);
    b_lane[t] = col < ncols ? static_cast<uint32_t>(col) * p.seg_stride + (lane >> 3) * 16 : 0xffffffffu;
  }
  const uint32_t zero_u = smem_u32(zero16);

  int slot = 0, round = 0;
  for (int sb = 0; sb < n_sb; ++sb) {
    const int v0 = sb * RS, nr = min(RS, rr.cnt - v0);
    const int rbs = (nr + 15) >> 4;
    float acc[RBMAX][NT][4];
#pragma unroll
    for (int rb = 0; rb < RBMAX; ++rb)
#pragma unroll
      for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[rb][t][e] = 0.f;

    for (int k0 = 0; k0 < K; k0 += KC) {
      const int n_units = min(KC, K - k0) >> 5;  // 32 k per unit
      mbar_wait(&full_a[slot], round & 1);
      mbar_wait(&full_b[slot], round & 1);
      const uint32_t sbase = ring_u + static_cast<uint32_t>(slot) * p.stage_bytes;
      for (int u = warp; u < n_units; u += kConsumerWarps) {
        uint32_t b[NT][4];
#pragma unroll
        for (int t = 0; t < NT; ++t) ldsm_x4(b[t], b_lane[t] == 0xffffffffu ? zero_u : sbase + b_off + b_lane[t] + u * 64);
#pragma unroll
        for (int rb = 0; rb < RBMAX; ++rb) {
          if (rb < rbs) {
            uint32_t a0[4], a1[4];
            const uint32_t aaddr = sbase + a_lane + static_cast<uint32_t>(rb * 16) * p.seg_stride + u * 64;
            ldsm_x4(a0, aaddr);
            ldsm_x4(a1, aaddr + 32);
#pragma unroll
            for (int t = 0; t < NT; ++t) {
              mma_bf16_16816(acc[rb][t], a0, b[t][0], b[t][1]);
              mma_bf16_16816(acc[rb][t], a1, b[t][2], b[t][3]);
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[slot]);  // this warp's share of the stage is in registers
      if (++slot == NS) { slot = 0; ++round; }
    }

    // ---- meet: partials -> shared memory, fixed-order sum over warps and split columns
    {
      const int g = lane >> 2, tq = lane & 3;
      float* pw = part + static_cast<size_t>(warp) * RS * PC;
#pragma unroll
      for (int rb = 0; rb < RBMAX; ++rb) {
        if (rb < rbs) {
#pragma unroll
          for (int t = 0; t < NT; ++t) {
            const int col = t * 8 + 2 * tq;
            if (col < PC) {
              *reinterpret_cast<float2*>(pw + (rb * 16 + g) * PC + col) = make_float2(acc[rb][t][0], acc[rb][t][1]);
              *reinterpret_cast<float2*>(pw + (rb * 16 + g + 8) * PC + col) = make_float2(acc[rb][t][2], acc[rb][t][3]);
            }
          }
        }
      }
    }
    consumer_sync();
    for (int idx = tid; idx < nr * M; idx += kConsumerThreads) {
      const int r = idx / M, m = idx - r * M;
      float t = 0.f;
      for (int w = 0; w < kConsumerWarps; ++w) {
        const float* q = part + (static_cast<size_t>(w) * RS + r) * PC + m * S;
        float tw = q[0];
        if (S >= 2) tw += q[1];
        if (S == 3) tw += q[2];
        t += tw;
      }
      res[static_cast<size_t>(v0 + r) * M + m] = t;
    }
    consumer_sync();  // part is reused by the next super-block
  }

  // ---- fused epilogue over the CTA's results: res[v * M + m] ---------------------
  const int nres = rr.cnt * M;
  if (p.ssq_in) {  // rstd_s was written before the streaming loop; the barriers of the meet order it
    for (int idx = tid; idx < nres; idx += kConsumerThreads) res[idx] *= rstd_s[idx % M];
    consumer_sync();
  }
  gemv_epilogue(p, G, rr, [&](int v, int m) -> float& { return res[static_cast<size_t>(v) * M + m]; }, M, p.m0, c, nct, true);
  trace_end(p.trace);
}

}  // namespace dvt

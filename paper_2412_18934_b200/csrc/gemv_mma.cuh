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
//   * a ring stage holds one K-chunk (KC elements) of every B column (B part)
//     and of every row of the super-block (A part), each row padded by
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

// A chain of up to kMaxChain GEMVs executed by ONE persistent launch (one CTA per SM, all resident): the
// weight producers roll from one matrix straight into the next -- weights never depend on activations, so the
// HBM stream does not stop at a GEMV boundary -- while the activation producer and the consumers of phase i + 1
// wait until every CTA has finished phase i (grid_arrive / grid_wait on a counter in global memory: the
// activations of phase i + 1 are the results of phase i from all CTAs). A single GEMV is a chain of one.
constexpr int kMaxChain = 4;

#ifdef DVT_CHAINDBG  // working builds only: per-CTA time stamps of the phases of a chain
#define DVT_DBG(ph, i) do { if (cp.dbg) cp.dbg[(static_cast<size_t>(blockIdx.x) * kMaxChain + (ph)) * 8 + (i)] = globaltimer_ns(); } while (0)
#else
#define DVT_DBG(ph, i) do { } while (0)
#endif

struct ChainParams {
  GemvParams ph[kMaxChain];
  int32_t n;
  int32_t stage_bytes, n_stages;  // ring geometry, common to the phases
  int32_t part_floats;            // floats of the partial buffer (largest phase)
  int32_t res_floats;             // floats of the result buffer (largest phase)
  int32_t* bar;                   // [n] phase counters, zeroed at the start of the step
  unsigned long long* dbg;        // DVT_CHAINDBG builds only
};

// The CTA's cnt rows are processed in n_sb super-blocks of nearly equal size (<= RS rows each), so that every
// ring stage carries about the same number of bytes (35 rows as 35, not as 32 + 3).
__device__ __forceinline__ void super_blocks(int cnt, int RS, int& n_sb, int& rsb) {
  n_sb = (cnt + RS - 1) / RS;
  rsb = n_sb > 0 ? (cnt + n_sb - 1) / n_sb : 0;
}

// which group of the phase this CTA works for, and its index within the group's CTAs (or -1: idle)
__device__ __forceinline__ int chain_cta(const GemvParams& p, int c, int& g) {
  g = c / p.ctas_per_group;
  if (g >= p.n_groups) { g = 0; return -1; }
  return c - g * p.ctas_per_group;
}

// four int8 (one 32-bit word, k ascending from the low byte) -> two fp16x2 words, exact: byte ^ 0x80 under the
// exponent byte 0x64 is the half 1024 + (q + 128); subtracting 1152 leaves q. Five instructions per four weights
// (the fp32 / bf16 route needs eleven, which made the int8 consumer instruction-bound: measured).
__device__ __forceinline__ void cvt_i8x4_f16x2(uint32_t r, uint32_t& lo, uint32_t& hi) {
  const uint32_t x = r ^ 0x80808080u;
  const uint32_t bias = 0x64806480u;  // (1152.0h, 1152.0h)
  uint32_t l = __byte_perm(x, 0x64646464u, 0x4140), h = __byte_perm(x, 0x64646464u, 0x4342);
  asm("sub.f16x2 %0, %0, %1;" : "+r"(l) : "r"(bias));
  asm("sub.f16x2 %0, %0, %1;" : "+r"(h) : "r"(bias));
  lo = l;
  hi = h;
}

__device__ __forceinline__ void mma_f16_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// NT: 8-column tiles of B (columns = M * S <= 8 * NT); RBMAX: 16-row blocks per stage; WQ: 1 = int8 weights with
// one fp32 scale per output row: half the bytes per weight, converted to fp16 in registers (exact),
// multiplied with fp16 activation terms (products exact in fp32), the scale applied to the row's result; the
// activation planes are stored in the matching k order (epilogue.cuh split_pos).
template <int NT, int RBMAX, int WQ>
__global__ void __launch_bounds__(kMmaThreads, 1) k_gemv_mma(const __grid_constant__ ChainParams cp) {
  constexpr int AES = WQ ? 1 : 2;  // bytes per weight
  extern __shared__ __align__(128) uint8_t smem[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int c_grid = blockIdx.x, n_grid = gridDim.x;
  const int NS = cp.n_stages;

  uint8_t* ring = smem;
  uint64_t* full_a = reinterpret_cast<uint64_t*>(smem + static_cast<size_t>(NS) * cp.stage_bytes);
  uint64_t* full_b = full_a + 8;
  uint64_t* empty = full_b + 8;
  uint32_t* zero16 = reinterpret_cast<uint32_t*>(empty + 8);  // B columns past ncols read these zeros
  float* rstd_s = reinterpret_cast<float*>(zero16 + 4);       // [2][32], alternating by phase
  float* part = rstd_s + 2 * kMmaMaxM;                        // [warps][RS][PC]
  float* res = part + cp.part_floats;                         // [cnt][M]
  float* wsc = res + cp.res_floats;                           // [cnt] row scales (int8 weights)

  trace_begin(cp.ph[0].trace);
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
    pdl_wait();  // the planes of the first phase were written by the previous kernels
    const uint64_t pol = l2_policy_evict_last();
    int slot = 0, round = 0;
    for (int ph = 0; ph < cp.n; ++ph) {
      const GemvParams& p = cp.ph[ph];
      int g;
      const int c = chain_cta(p, c_grid, g);
      const GemvGroup& G = p.g[g];
      const int K = p.K, KC = p.kc, M = p.M, S = G.S, RS = p.rows_per_stage, ncols = M * S;
      if (ph > 0) {  // the planes (and sums of squares) of this phase come from every CTA of the previous one
        if (lane == 0) grid_wait(cp.bar + ph - 1, n_grid);
        __syncwarp();
        fence_proxy_async();
        if (lane == 0) DVT_DBG(ph, 5);
      }
      if (lane == 0) DVT_DBG(ph, 6);
      if (c < 0) continue;
      const RowRange rr = cta_rows(G, c, p.ctas_per_group);
      int n_sb, rsb;
      super_blocks(rr.cnt, RS, n_sb, rsb);
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
      for (int sb = 0; sb < n_sb; ++sb) {
        for (int k0 = 0; k0 < K; k0 += KC) {
          if (round > 0) mbar_wait(&empty[slot], (round & 1) ^ 1);
          const uint32_t segb = static_cast<uint32_t>(min(KC, K - k0)) * 2u;
          if (lane == 0) mbar_arrive_expect_tx(&full_b[slot], static_cast<uint32_t>(ncols) * segb);
          __syncwarp();
          uint8_t* dst = ring + static_cast<size_t>(slot) * cp.stage_bytes;  // B columns first, then the A rows
#pragma unroll
          for (int h = 0; h < 2; ++h)
            if (src[h])
              bulk_g2s(dst + static_cast<size_t>(lane + 32 * h) * p.seg_stride, src[h] + static_cast<size_t>(k0) * 2, segb,
                       &full_b[slot], pol);
          if (++slot == NS) { slot = 0; ++round; }
        }
      }
    }
    return;
  }

  if (warp >= kConsumerWarps) {
    // ---------------- weight producers: warp pw copies rows [16 pw, 16 pw + 16) of every stage ---
    // They never wait for a phase boundary: only for ring slots.
    const int pw = warp - kConsumerWarps;
    const uint64_t pol = l2_policy_evict_first();
    int slot = 0, round = 0;
    for (int ph = 0; ph < cp.n; ++ph) {
      const GemvParams& p = cp.ph[ph];
      int g;
      const int c = chain_cta(p, c_grid, g);
      if (c < 0) continue;
      const GemvGroup& G = p.g[g];
      const int K = p.K, KC = p.kc, RS = p.rows_per_stage;
      const uint32_t a_off = static_cast<uint32_t>(p.M * G.S) * p.seg_stride;  // A rows follow the B columns
      const RowRange rr = cta_rows(G, c, p.ctas_per_group);
      int n_sb, rsb;
      super_blocks(rr.cnt, RS, n_sb, rsb);
      for (int sb = 0; sb < n_sb; ++sb) {
        const int v0 = sb * rsb, nr = min(rsb, rr.cnt - v0);
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
          if (pw == 0 && lane == 0 && sb == 0 && k0 == 0) DVT_DBG(ph, 7);
          const uint32_t segb = static_cast<uint32_t>(min(KC, K - k0)) * AES;
          if (lane == 0) mbar_arrive_expect_tx(&full_a[slot], static_cast<uint32_t>(my_rows) * segb);
          __syncwarp();
          uint8_t* dst = ring + static_cast<size_t>(slot) * cp.stage_bytes + a_off;
          if (mine) bulk_g2s(dst + static_cast<size_t>(r) * p.aseg_stride, src + static_cast<size_t>(k0) * AES, segb, &full_a[slot], pol);
          if (++slot == NS) { slot = 0; ++round; }
        }
      }
    }
    return;
  }

  // ---------------- consumers -------------------------------------------------
  pdl_wait();  // residual stream, [h1 || h2]: written by the previous kernels
  const uint32_t ring_u = smem_u32(ring);
  const uint32_t zero_u = smem_u32(zero16);
  int slot = 0, round = 0;
  for (int ph = 0; ph < cp.n; ++ph) {
    const GemvParams& p = cp.ph[ph];
    int g;
    const int c = chain_cta(p, c_grid, g);
    const GemvGroup& G = p.g[g];
    const int K = p.K, KC = p.kc, M = p.M, S = G.S, RS = p.rows_per_stage;
    const int ncols = M * S, PC = (ncols + 1) & ~1;
    if (ph > 0) trace_begin(p.trace);
    if (tid == 0) DVT_DBG(ph, 0);
    if (ph > 0) {
      // Results of the previous phase from every CTA ([h1 || h2], residual stream, sums of squares) are read
      // below: thread 0 acquires the phase counter, the barrier extends it to the CTA's consumers.
      if (tid == 0) grid_wait(cp.bar + ph - 1, n_grid);
      consumer_sync();
    }
    if (c >= 0 && p.ssq_in) {
      // RMSNorm: 1 / rms of each draft row from the producers' partial sums of squares, fixed order (lane l adds
      // CTAs l, l + 32, ...; then a butterfly). Overlaps the arrival of the phase's first activation chunk.
      float* rs = rstd_s + (ph & 1) * kMmaMaxM;
      for (int m = warp; m < M; m += kConsumerWarps) {
        float v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const int cc = lane + 32 * j;
          v[j] = cc < p.ssq_nct ? __ldcg(p.ssq_in + static_cast<int64_t>(cc) * kMaxRows + p.m0 + m) : 0.f;
        }
        float t = 0.f;
#pragma unroll
        for (int j = 0; j < 8; ++j) t += v[j];
        t = warp_sum(t);
        if (lane == 0) rs[m] = 1.0f / sqrtf(t / static_cast<float>(K) + p.eps);
      }
    }
    if (c >= 0) {
      const RowRange rr = cta_rows(G, c, p.ctas_per_group);
      EpiRegs pre;
      epi_prefetch(p, G, rr, M, p.m0, true, pre);  // in flight during the streaming loop
      if (WQ) {  // scale of each of the CTA's rows; read after the barriers of the first meet
        for (int v = tid; v < rr.cnt; v += kConsumerThreads) {
          int j, n;
          locate_row(G, rr, v, j, n);
          wsc[v] = __ldg(G.ws[j] + n);
        }
      }
      int n_sb, rsb;
      super_blocks(rr.cnt, RS, n_sb, rsb);
      const int RS16 = (RS + 15) & ~15;  // rows of the partial buffer: whole 16-row blocks
      // per-lane ldmatrix address pieces (a stage: the B columns, then the A rows)
      const int a_lrow = (lane & 7) + ((lane >> 3) & 1) * 8;  // this lane's row within a 16-row block
      const uint32_t a_lane = static_cast<uint32_t>(ncols) * p.seg_stride + (lane >> 4) * 16;
      uint32_t b_lane[NT];  // offset within the B part of a stage, or ~0: the zero block
#pragma unroll
      for (int t = 0; t < NT; ++t) {
        const int col = t * 8 + (lane & 7);
        b_lane[t] = col < ncols ? static_cast<uint32_t>(col) * p.seg_stride + (lane >> 3) * 16 : 0xffffffffu;
      }
      for (int sb = 0; sb < n_sb; ++sb) {
        const int v0 = sb * rsb, nr = min(rsb, rr.cnt - v0);
        const int rbs = (nr + 15) >> 4;
        uint32_t a_row[RBMAX];  // rows past the super-block's last one were never copied: read the last row instead
#pragma unroll
        for (int rb = 0; rb < RBMAX; ++rb) a_row[rb] = static_cast<uint32_t>(min(rb * 16 + a_lrow, nr - 1)) * p.aseg_stride;
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
          if (tid == 0 && sb == 0 && k0 == 0) DVT_DBG(ph, 1);
          const uint32_t sbase = ring_u + static_cast<uint32_t>(slot) * cp.stage_bytes;
          for (int u = warp; u < n_units; u += kConsumerWarps) {
            uint32_t b[NT][4];
#pragma unroll
            for (int t = 0; t < NT; ++t) ldsm_x4(b[t], b_lane[t] == 0xffffffffu ? zero_u : sbase + b_lane[t] + u * 64);
#pragma unroll
            for (int rb = 0; rb < RBMAX; ++rb) {
              if (rb < rbs) {
                uint32_t a0[4], a1[4];
                if (WQ) {  // 16 rows x 32 int8: one ldmatrix, then the exact conversion; pairs as split_pos orders B
                  uint32_t q[4];
                  ldsm_x4(q, sbase + a_lane + a_row[rb] + u * 32);
#pragma unroll
                  for (int e = 0; e < 4; ++e) cvt_i8x4_f16x2(q[e], a0[e], a1[e]);
                } else {
                  const uint32_t aaddr = sbase + a_lane + a_row[rb] + u * 64;
                  ldsm_x4(a0, aaddr);
                  ldsm_x4(a1, aaddr + 32);
                }
#pragma unroll
                for (int t = 0; t < NT; ++t) {
                  if (WQ) {
                    mma_f16_16816(acc[rb][t], a0, b[t][0], b[t][1]);
                    mma_f16_16816(acc[rb][t], a1, b[t][2], b[t][3]);
                  } else {
                    mma_bf16_16816(acc[rb][t], a0, b[t][0], b[t][1]);
                    mma_bf16_16816(acc[rb][t], a1, b[t][2], b[t][3]);
                  }
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
          const int gq = lane >> 2, tq = lane & 3;
          float* pw = part + static_cast<size_t>(warp) * RS16 * PC;
#pragma unroll
          for (int rb = 0; rb < RBMAX; ++rb) {
            if (rb < rbs) {
#pragma unroll
              for (int t = 0; t < NT; ++t) {
                const int col = t * 8 + 2 * tq;
                if (col < PC) {
                  *reinterpret_cast<float2*>(pw + (rb * 16 + gq) * PC + col) = make_float2(acc[rb][t][0], acc[rb][t][1]);
                  *reinterpret_cast<float2*>(pw + (rb * 16 + gq + 8) * PC + col) = make_float2(acc[rb][t][2], acc[rb][t][3]);
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
            const float* q = part + (static_cast<size_t>(w) * RS16 + r) * PC + m * S;
            float tw = q[0];
            if (WQ) {  // fp16 terms carry 2^-11 and 2^-22 (epilogue.cuh store_split)
              if (S >= 2) tw += q[1] * 4.8828125e-4f;
              if (S == 3) tw += q[2] * 2.384185791015625e-7f;
            } else {
              if (S >= 2) tw += q[1];
              if (S == 3) tw += q[2];
            }
            t += tw;
          }
          res[static_cast<size_t>(v0 + r) * M + m] = WQ ? t * wsc[v0 + r] : t;
        }
        consumer_sync();  // part is reused by the next super-block
      }

      if (tid == 0) DVT_DBG(ph, 2);
      // ---- fused epilogue over the CTA's results: res[v * M + m] ---------------------
      const int nres = rr.cnt * M;
      if (p.ssq_in) {  // rstd_s: written before the streaming loop; the barriers of the meet order it
        const float* rs = rstd_s + (ph & 1) * kMmaMaxM;
        for (int idx = tid; idx < nres; idx += kConsumerThreads) res[idx] *= rs[idx % M];
        consumer_sync();
      }
      gemv_epilogue(p, G, rr, [&](int v, int m) -> float& { return res[static_cast<size_t>(v) * M + m]; }, M, p.m0, c,
                    p.ctas_per_group, true, &pre);
    }
    if (tid == 0) DVT_DBG(ph, 3);
    if (ph + 1 < cp.n) {
      // This CTA's results of the phase are complete: count in. The writers order their generic-proxy stores
      // before the other CTAs' bulk copies (async proxy); the CTA barrier makes them happen before thread 0's
      // gpu-scope release, which is cumulative.
      fence_proxy_async();
      consumer_sync();
      if (tid == 0) grid_arrive(cp.bar + ph);
    }
    if (tid == 0) DVT_DBG(ph, 4);
    trace_end(p.trace);
  }
}

}  // namespace dvt

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

#ifdef DVT_CHAINDBG  // working builds only: per-CTA time stamps inside one launch
#define DVT_DBG(i) do { if (cp.dbg) cp.dbg[static_cast<size_t>(blockIdx.x) * 16 + (i)] = globaltimer_ns(); } while (0)
#else
#define DVT_DBG(i) do { } while (0)
#endif

struct MmaParams {
  GemvParams p;
  int32_t stage_bytes, n_stages;  // ring geometry
  int32_t part_floats;            // floats of the partial buffer
  int32_t res_floats;             // floats of the result buffer
  unsigned long long* dbg;        // DVT_CHAINDBG builds only
};

// The CTA's cnt rows are processed in n_sb super-blocks of nearly equal size (<= RS rows each), so that every
// ring stage carries about the same number of bytes (35 rows as 35, not as 32 + 3).
__device__ __forceinline__ void super_blocks(int cnt, int RS, int& n_sb, int& rsb) {
  n_sb = (cnt + RS - 1) / RS;
  rsb = n_sb > 0 ? (cnt + n_sb - 1) / n_sb : 0;
}

// Which rows this CTA works on: group g, index c within the group's CTAs (or c < 0: idle). Every role computes
// it BEFORE griddepcontrol.wait (it depends on the launch arguments only) and pins the results there. Measured:
// with 64-bit divisions in cta_rows this was a dependent chain of more than a microsecond that the consumers
// spent after the wait (ring full, HBM stream stopped) and the weight producers before their first copy; the
// host now supplies the quotients (GemvGroup::deal_base / deal_rem).
struct CtaGeom {
  int c, g, n_sb, rsb;
  RowRange rr;
};
__device__ __forceinline__ CtaGeom cta_geom(const GemvParams& p, int c_grid) {
  CtaGeom q;
  q.g = c_grid >= p.ctas_per_group ? 1 : 0;  // at most two groups
  q.c = c_grid - q.g * p.ctas_per_group;
  if (q.g >= p.n_groups) { q.g = 0; q.c = -1; }
  q.n_sb = q.rsb = 0;
  q.rr.cnt = q.rr.n0 = q.rr.cr = 0;
  q.rr.g0 = 0;
  if (q.c >= 0) {
    q.rr = cta_rows(p.g[q.g], q.c, p.ctas_per_group);
    super_blocks(q.rr.cnt, p.rows_per_stage, q.n_sb, q.rsb);
  }
  asm volatile("" : "+r"(q.c), "+r"(q.g), "+r"(q.n_sb), "+r"(q.rsb), "+r"(q.rr.cnt), "+r"(q.rr.n0), "+r"(q.rr.cr), "+l"(q.rr.g0));
  return q;
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

// four fp8 e4m3 bytes (k ascending from the low byte) -> two fp16x2 words, exact (every e4m3 value is an fp16 value):
// one cvt per pair of weights.
__device__ __forceinline__ void cvt_e4m3x4_f16x2(uint32_t r, uint32_t& lo, uint32_t& hi) {
  asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %2;\n\tcvt.rn.f16x2.e4m3x2 %0, l;\n\tcvt.rn.f16x2.e4m3x2 %1, h;\n\t}"
      : "=r"(lo), "=r"(hi)
      : "r"(r));
}

__device__ __forceinline__ void mma_f16_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// NT: 8-column tiles of B (columns = M * S <= 8 * NT); RBMAX: 16-row blocks per stage; WQ: 2 = fp8 e4m3 weights (as
// 1, with a hardware conversion per pair of weights); 1 = int8 weights with
// one fp32 scale per output row: half the bytes per weight, converted to fp16 in registers (exact),
// multiplied with fp16 activation terms (products exact in fp32), the scale applied to the row's result; the
// activation planes are stored in the matching k order (epilogue.cuh split_pos).
template <int NT, int RBMAX, int WQ>
__global__ void __launch_bounds__(kMmaThreads, 1) k_gemv_mma(const __grid_constant__ MmaParams cp) {
  constexpr int AES = WQ ? 1 : 2;  // bytes per weight
  extern __shared__ __align__(128) uint8_t smem[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int NS = cp.n_stages;
  const GemvParams& p = cp.p;

  uint8_t* ring = smem;
  uint64_t* full_a = reinterpret_cast<uint64_t*>(smem + static_cast<size_t>(NS) * cp.stage_bytes);
  uint64_t* full_b = full_a + 8;
  uint64_t* empty = full_b + 8;
  uint32_t* zero16 = reinterpret_cast<uint32_t*>(empty + 8);  // B columns past ncols read these zeros
  float* rstd_s = reinterpret_cast<float*>(zero16 + 4);       // [32]
  float* part = rstd_s + 2 * kMmaMaxM;                        // [warps][RS][PC]
  float* res = part + cp.part_floats;                         // [cnt][M]
  float* wsc = res + cp.res_floats;                           // [cnt] row scales (int8 weights)

  trace_begin(p.trace);
  if (tid == 0) DVT_DBG(0);
  if (tid < NS) {
    mbar_init(&full_a[tid], kMmaProducerWarps);
    mbar_init(&full_b[tid], 1);
    mbar_init(&empty[tid], kConsumerWarps);
    mbar_fence_init();
  }
  if (tid >= 32 && tid < 36) zero16[tid - 32] = 0u;
  __syncthreads();
  pdl_launch_dependents();

  const CtaGeom q = cta_geom(p, blockIdx.x);
  const int c = q.c;
  const GemvGroup& G = p.g[q.g];
  const RowRange rr = q.rr;
  const int n_sb = q.n_sb, rsb = q.rsb;
  const int K = p.K, KC = p.kc, M = p.M, S = G.S, ncols = M * S;

  if (warp >= kConsumerWarps + kMmaProducerWarps) {
    // ---------------- activation producer: one B column per lane (two when ncols > 32) -----------
    const uint64_t pol = l2_policy_evict_last();
    // everything that does not need the previous kernel's results is computed before the wait
    int64_t off[2];  // element offset of the column's plane row (X_ROWS without a row index: complete)
    int cm[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int col = lane + 32 * h;
      cm[h] = S == 1 ? col : (S == 2 ? col >> 1 : (col * 43) >> 7);  // col / S for col < 64, S <= 3
      const int s = col - cm[h] * S;
      off[h] = s * G.xs_plane + (G.xidx ? 0 : (p.m0 + cm[h]) * G.xs_ld);
    }
    asm volatile("" : "+l"(off[0]), "+l"(off[1]), "+r"(cm[0]), "+r"(cm[1]));
    pdl_wait();  // the planes were written by the previous kernels
    if (lane == 0) DVT_DBG(5);
    if (c < 0) return;
    const uint8_t* src[2] = {nullptr, nullptr};
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      if (lane + 32 * h < ncols) {
        if (G.xkind == X_ROWS) {
          const int64_t ro = G.xidx ? static_cast<int64_t>(G.xidx[p.m0 + cm[h]]) * G.xs_ld : 0;
          src[h] = reinterpret_cast<const uint8_t*>(G.xs + off[h] + ro);
        } else {  // embedding rows are bf16 already: one plane
          src[h] = reinterpret_cast<const uint8_t*>(static_cast<const __nv_bfloat16*>(G.embed) +
                                                    static_cast<size_t>(G.tokens[p.m0 + cm[h]]) * K);
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
        uint8_t* dst = ring + static_cast<size_t>(slot) * cp.stage_bytes;  // B columns first, then the A rows
#pragma unroll
        for (int h = 0; h < 2; ++h)
          if (src[h])
            bulk_g2s(dst + static_cast<size_t>(lane + 32 * h) * p.seg_stride, src[h] + static_cast<size_t>(k0) * 2, segb,
                     &full_b[slot], pol);
        if (lane == 0 && sb == 0 && k0 == 0) DVT_DBG(6);
        if (++slot == NS) { slot = 0; ++round; }
      }
    }
    return;
  }

  if (warp >= kConsumerWarps) {
    // ---------------- weight producers: warp pw copies rows [16 pw, 16 pw + 16) of every stage ---
    // They never wait for the previous kernel: weights do not depend on activations.
    if (c < 0) return;
    const int pw = warp - kConsumerWarps;
    const uint64_t pol = l2_policy_evict_first();
    const uint32_t a_off = static_cast<uint32_t>(ncols) * p.seg_stride;  // A rows follow the B columns
    int slot = 0, round = 0;
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
        if (pw == 0 && lane == 0 && sb == 0 && k0 == 0) DVT_DBG(7);
        const uint32_t segb = static_cast<uint32_t>(min(KC, K - k0)) * AES;
        if (lane == 0) mbar_arrive_expect_tx(&full_a[slot], static_cast<uint32_t>(my_rows) * segb);
        __syncwarp();
        uint8_t* dst = ring + static_cast<size_t>(slot) * cp.stage_bytes + a_off;
        if (mine) bulk_g2s(dst + static_cast<size_t>(r) * p.aseg_stride, src + static_cast<size_t>(k0) * AES, segb, &full_a[slot], pol);
        if (++slot == NS) { slot = 0; ++round; }
      }
    }
    return;
  }

  // ---------------- consumers -------------------------------------------------
  const int RS = p.rows_per_stage;
  const int PC = (ncols + 1) & ~1;
  const int RS16 = (RS + 15) & ~15;  // rows of the partial buffer: whole 16-row blocks
  const uint32_t ring_u = smem_u32(ring);
  const uint32_t zero_u = smem_u32(zero16);
  // per-lane ldmatrix address pieces (a stage: the B columns, then the A rows)
  const int a_lrow = (lane & 7) + ((lane >> 3) & 1) * 8;  // this lane's row within a 16-row block
  uint32_t a_lane = static_cast<uint32_t>(ncols) * p.seg_stride + (lane >> 4) * 16;
  uint32_t b_lane[NT];  // offset within the B part of a stage, or ~0: the zero block
#pragma unroll
  for (int t = 0; t < NT; ++t) {
    const int col = t * 8 + (lane & 7);
    b_lane[t] = col < ncols ? static_cast<uint32_t>(col) * p.seg_stride + (lane >> 3) * 16 : 0xffffffffu;
    asm volatile("" : "+r"(b_lane[t]));
  }
  asm volatile("" : "+r"(a_lane));
  pdl_wait();  // residual stream, [h1 || h2], sums of squares: written by the previous kernels
  if (tid == 0) DVT_DBG(1);
  if (c >= 0) {
    // RMSNorm: the partial sums of squares of draft row `warp` are requested now and added after the streaming
    // loop (their L2 round trip must not delay the first mma); rows >= 8 of a wide level are read there.
    float ssq_v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) ssq_v[j] = 0.f;
    if (p.ssq_in && warp < M) {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int cc = lane + 32 * j;
        if (cc < p.ssq_nct) ssq_v[j] = __ldcg(p.ssq_in + static_cast<int64_t>(cc) * kMaxRows + p.m0 + warp);
      }
    }
    EpiRegs pre;
    epi_prefetch(p, G, rr, M, p.m0, true, pre);  // in flight during the streaming loop
    if (WQ) {  // scale of each of the CTA's rows; read after the barriers of the first meet
      for (int v = tid; v < rr.cnt; v += kConsumerThreads) {
        int j, n;
        locate_row(G, rr, v, j, n);
        wsc[v] = __ldg(G.ws[j] + n);
      }
    }
    int slot = 0, round = 0;
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
        if (tid == 0 && sb == 0 && k0 == 0) DVT_DBG(2);
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
                uint32_t qw[4];
                ldsm_x4(qw, sbase + a_lane + a_row[rb] + u * 32);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                  if (WQ == 2) cvt_e4m3x4_f16x2(qw[e], a0[e], a1[e]);
                  else cvt_i8x4_f16x2(qw[e], a0[e], a1[e]);
                }
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

      if (sb == 0 && p.ssq_in) {
        // 1 / rms of each draft row from the producers' partial sums of squares, fixed order (lane l adds CTAs
        // l, l + 32, ...; then a butterfly); visible to the epilogue through the barriers of the meet
        for (int m = warp; m < M; m += kConsumerWarps) {
          if (m != warp) {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const int cc = lane + 32 * j;
              ssq_v[j] = cc < p.ssq_nct ? __ldcg(p.ssq_in + static_cast<int64_t>(cc) * kMaxRows + p.m0 + m) : 0.f;
            }
          }
          float t = 0.f;
#pragma unroll
          for (int j = 0; j < 8; ++j) t += ssq_v[j];
          t = warp_sum(t);
          if (lane == 0) rstd_s[m] = 1.0f / sqrtf(t / static_cast<float>(K) + p.eps);
        }
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
          const float* qp = part + (static_cast<size_t>(w) * RS16 + r) * PC + m * S;
          float tw = qp[0];
          if (WQ) {  // fp16 terms carry 2^-11 and 2^-22 (epilogue.cuh store_split)
            if (S >= 2) tw += qp[1] * 4.8828125e-4f;
            if (S == 3) tw += qp[2] * 2.384185791015625e-7f;
          } else {
            if (S >= 2) tw += qp[1];
            if (S == 3) tw += qp[2];
          }
          t += tw;
        }
        if (WQ) t *= wsc[v0 + r];
        if (p.ssq_in) t *= rstd_s[m];  // written before this super-block's barrier
        res[static_cast<size_t>(v0 + r) * M + m] = t;
      }
      consumer_sync();  // part is reused by the next super-block
    }

    if (tid == 0) DVT_DBG(3);
    // ---- fused epilogue over the CTA's results: res[v * M + m] ---------------------
    gemv_epilogue(p, G, rr, [&](int v, int m) -> float& { return res[static_cast<size_t>(v) * M + m]; }, M, p.m0, c,
                  p.ctas_per_group, true, &pre);
  }
  if (tid == 0) DVT_DBG(4);
  trace_end(p.trace);
}

}  // namespace dvt

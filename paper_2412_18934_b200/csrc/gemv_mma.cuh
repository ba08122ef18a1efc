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
// Shape of the kernel (one CTA per SM, 8 consumer warps + 4 producer warps):
//   * rows are dealt to the CTAs in contiguous ranges differing by <= 1 row
//     (same as k_gemv), and processed in super-blocks of RS <= 64 rows;
//   * the producer warps copy, per ring stage, one K-chunk (KC elements) of
//     every row of the super-block with 1-D bulk async copies (row-exact: no
//     byte of another CTA's rows is touched) into rows padded by 16 bytes, which
//     makes the ldmatrix reads of the consumers bank-conflict free; it starts
//     before griddepcontrol.wait because weights never depend on activations;
//   * the split activations of one K-panel live in shared memory as
//     [column][k] bf16 (column stride = 16 mod 128 bytes); consumer warp w owns
//     the k-units w, w + 8, ... (32 k each) of every chunk, loads its B
//     fragments once per unit (ldmatrix.x4) and reuses them for all row blocks
//     of the stage (ldmatrix.x4 of A + NT mma each);
//   * accumulators stay in registers for a whole (panel, super-block); only then
//     do the warps meet: partials go to shared memory, one named barrier, and a
//     fixed-order sum over the 8 warps and the S split columns (deterministic);
//   * the fused epilogues of k_gemv run once over the CTA's results.
// There is no barrier inside the streaming loop.
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
constexpr int kMmaThreads = kConsumerThreads + 32 * kMmaProducerWarps;

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
  const int NS = p.n_stages, RS = p.rows_per_stage, KC = p.kc, KP = p.kp, K = p.K, M = p.M, S = p.split;
  const int ncols = M * S, PC = (ncols + 1) & ~1;

  uint8_t* ring = smem;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + static_cast<size_t>(NS) * p.stage_bytes);
  uint64_t* empty = full + 8;
  uint64_t* xbar = empty + 8;  // consumers have issued their activation loads
  float* rstd_s = reinterpret_cast<float*>(xbar + 2);  // [32]
  const void** xptr_s = reinterpret_cast<const void**>(rstd_s + kMmaMaxM);  // [32] source row of each m
  float* ss_part = reinterpret_cast<float*>(xptr_s + kMmaMaxM);  // [warps][32] sum of squares
  uint8_t* bstore = reinterpret_cast<uint8_t*>(ss_part + kConsumerWarps * kMmaMaxM);  // [ncols][bs_stride] + 16 zero bytes
  float* part = reinterpret_cast<float*>(bstore + static_cast<size_t>(ncols) * p.bs_stride + 16);  // [warps][RS][PC]
  float* res = part + static_cast<size_t>(kConsumerWarps) * RS * PC;  // [cnt][M]

  const RowRange rr = cta_rows(G, c, nct);
  const int n_sb = (rr.cnt + RS - 1) / RS;
  const int n_panels = (K + KP - 1) / KP;
  trace_begin(p.trace);

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full[s], kMmaProducerWarps);
      mbar_init(&empty[s], kConsumerWarps);
    }
    mbar_init(xbar, kConsumerWarps);
    mbar_fence_init();
  }
  __syncthreads();
  pdl_launch_dependents();

  if (warp >= kConsumerWarps) {
    // ---------------- producers: warp pw copies rows [16 pw, 16 pw + 16) of every stage ---------
    const int pw = warp - kConsumerWarps;
    const uint64_t pol = l2_policy_evict_first();
    int slot = 0, round = 0;
    for (int pn = 0; pn < n_panels; ++pn) {
      const int k_begin = pn * KP, k_end = min(K, k_begin + KP);
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
        for (int k0 = k_begin; k0 < k_end; k0 += KC) {
          if (round > 0) mbar_wait(&empty[slot], (round & 1) ^ 1);
          // Only the first stage is requested before the consumers have issued their activation
          // loads, so that those do not queue behind a ring full of weights on this SM's return
          // path. Measured on the c3 step: gate before stage 1: 3080 us; before stage 0: 3125 us;
          // before stage 2: 3106 us; no gate: 3107 us.
          if (round == 0 && slot == 1) mbar_wait(xbar, 0);
          const uint32_t segb = static_cast<uint32_t>(min(KC, k_end - k0)) * 2u;
          if (lane == 0) mbar_arrive_expect_tx(&full[slot], static_cast<uint32_t>(my_rows) * segb);
          __syncwarp();
          uint8_t* dst = ring + static_cast<size_t>(slot) * p.stage_bytes;
          if (mine) bulk_g2s(dst + static_cast<size_t>(r) * p.seg_stride, src + static_cast<size_t>(k0) * 2, segb, &full[slot], pol);
          if (++slot == NS) { slot = 0; ++round; }
        }
      }
    }
    return;
  }

  // ---------------- consumers -------------------------------------------------
  pdl_wait();
  const StepDyn* dyn = p.dyn;
  const bool normed = G.gain != nullptr;
  const __nv_bfloat16* gain = static_cast<const __nv_bfloat16*>(G.gain);

  const bool x_embed = G.xkind != X_ROWS;
  if (tid < M && (x_embed || G.x_from_dyn || G.xidx)) {  // source row of each draft row (fp32 rows, or bf16 embedding rows)
    if (!x_embed) {
      const float* base = G.x_from_dyn ? dyn->feats : G.xsrc;
      const int64_t ri = G.xidx ? G.xidx[p.m0 + tid] : p.m0 + tid;
      xptr_s[tid] = base + ri * G.xld;
    } else {
      xptr_s[tid] = static_cast<const __nv_bfloat16*>(G.embed) + static_cast<size_t>(G.tokens[p.m0 + tid]) * K;
    }
  }
  ss_part[tid] = 0.f;  // kConsumerWarps * kMmaMaxM == kConsumerThreads
  if (tid < 4) reinterpret_cast<uint32_t*>(bstore + static_cast<size_t>(ncols) * p.bs_stride)[tid] = 0u;

  // per-lane ldmatrix address pieces
  const uint32_t ring_u = smem_u32(ring);
  const uint32_t a_lane = static_cast<uint32_t>((lane & 7) + ((lane >> 3) & 1) * 8) * p.seg_stride + (lane >> 4) * 16;
  uint32_t b_base[NT], b_kmul[NT];
#pragma unroll
  for (int t = 0; t < NT; ++t) {
    const int col = t * 8 + (lane & 7);
    const bool have = col < ncols;
    b_base[t] = smem_u32(bstore) + (have ? static_cast<uint32_t>(col) * p.bs_stride + (lane >> 3) * 16
                                         : static_cast<uint32_t>(ncols) * p.bs_stride);
    b_kmul[t] = have ? 2u : 0u;
  }

  int slot = 0, round = 0;
  for (int pn = 0; pn < n_panels; ++pn) {
    const int k_begin = pn * KP, k_end = min(K, k_begin + KP);
    const int kp_pairs = (k_end - k_begin) >> 1;
    // ---- split activations of this panel -> B store ---------------------------
    consumer_sync();  // every warp is done with the previous panel's B store
    {
      // Item idx = m * K8 + j covers k = k_begin + 8 j .. + 7 of row m: two 16-byte loads of
      // activations (one of gains), one 16-byte store per split column. The loads of a round are
      // issued before any is used (one L2 round trip per round of IB items per thread).
      constexpr int IB = 6;
      const int K8 = kp_pairs >> 2;
      const int n_items = M * K8;
      const bool direct = !x_embed && !G.x_from_dyn && !G.xidx;  // rows of a dense fp32 matrix
      bool signalled = pn > 0;
      for (int base = 0; base < n_items; base += kConsumerThreads * IB) {
        float4 va[IB], vb[IB];
        uint4 gq[IB];
        int mi[IB], ji[IB];
#pragma unroll
        for (int i = 0; i < IB; ++i) {
          const int idx = base + i * kConsumerThreads + tid;
          const bool valid = idx < n_items;
          const int m = valid ? idx / K8 : M;
          const int j = idx - m * K8;
          mi[i] = m;
          ji[i] = j;
          va[i] = vb[i] = make_float4(0.f, 0.f, 0.f, 0.f);
          gq[i] = make_uint4(0u, 0u, 0u, 0u);
          if (valid) {
            const int k = k_begin + 8 * j;
            if (!x_embed) {
              const float* xr = direct ? G.xsrc + static_cast<int64_t>(p.m0 + m) * G.xld : static_cast<const float*>(xptr_s[m]);
              va[i] = __ldg(reinterpret_cast<const float4*>(xr + k));
              vb[i] = __ldg(reinterpret_cast<const float4*>(xr + k + 4));
            } else {
              const uint4 e = __ldg(reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(xptr_s[m]) + k));
              const float2 e0 = bf16x2_to_f32x2(e.x), e1 = bf16x2_to_f32x2(e.y), e2 = bf16x2_to_f32x2(e.z), e3 = bf16x2_to_f32x2(e.w);
              va[i] = make_float4(e0.x, e0.y, e1.x, e1.y);
              vb[i] = make_float4(e2.x, e2.y, e3.x, e3.y);
            }
            if (normed) gq[i] = __ldg(reinterpret_cast<const uint4*>(gain + k));
          }
        }
        if (!signalled) {  // loads are in flight: let the producers fill the ring
          __syncwarp();
          if (lane == 0) mbar_arrive(xbar);
          signalled = true;
        }
#pragma unroll
        for (int i = 0; i < IB; ++i) {
          float x[8] = {va[i].x, va[i].y, va[i].z, va[i].w, vb[i].x, vb[i].y, vb[i].z, vb[i].w};
          const int m = mi[i];
          if (normed) {
            float ssq = 0.f;
#pragma unroll
            for (int e = 0; e < 8; ++e) ssq = fmaf(x[e], x[e], ssq);
            // segmented sum over the rows present in this warp's 32 items (usually one)
            const int m_lo = __shfl_sync(0xffffffffu, m, 0), m_hi = min(__shfl_sync(0xffffffffu, m, 31), M - 1);
            for (int mm = m_lo; mm <= m_hi; ++mm) {
              const float t = warp_sum(m == mm ? ssq : 0.f);
              if (lane == 0) ss_part[warp * kMmaMaxM + mm] += t;
            }
            const uint32_t gwv[4] = {gq[i].x, gq[i].y, gq[i].z, gq[i].w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const float2 g = bf16x2_to_f32x2(gwv[e]);
              x[2 * e] *= g.x;
              x[2 * e + 1] *= g.y;
            }
          }
          if (m < M) {
            uint32_t h0[4], h1[4], h2[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              h0[e] = pack_bf16x2_rn(x[2 * e], x[2 * e + 1]);
              const float2 f0 = bf16x2_to_f32x2(h0[e]);
              const float rx = x[2 * e] - f0.x, ry = x[2 * e + 1] - f0.y;
              h1[e] = pack_bf16x2_rn(rx, ry);
              const float2 f1 = bf16x2_to_f32x2(h1[e]);
              h2[e] = pack_bf16x2_rn(rx - f1.x, ry - f1.y);
            }
            uint8_t* col0 = bstore + static_cast<size_t>(m * S) * p.bs_stride + 16 * ji[i];
            *reinterpret_cast<uint4*>(col0) = make_uint4(h0[0], h0[1], h0[2], h0[3]);
            *reinterpret_cast<uint4*>(col0 + p.bs_stride) = make_uint4(h1[0], h1[1], h1[2], h1[3]);
            if (S == 3) *reinterpret_cast<uint4*>(col0 + 2 * p.bs_stride) = make_uint4(h2[0], h2[1], h2[2], h2[3]);
          }
        }
      }
      if (!signalled) {
        __syncwarp();
        if (lane == 0) mbar_arrive(xbar);
      }
    }
    consumer_sync();

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

      for (int k0 = k_begin; k0 < k_end; k0 += KC) {
        const int n_units = min(KC, k_end - k0) >> 5;  // 32 k per unit
        mbar_wait(&full[slot], round & 1);
        const uint32_t sbase = ring_u + static_cast<uint32_t>(slot) * p.stage_bytes + a_lane;
        for (int u = warp; u < n_units; u += kConsumerWarps) {
          uint32_t b[NT][4];
#pragma unroll
          for (int t = 0; t < NT; ++t) ldsm_x4(b[t], b_base[t] + static_cast<uint32_t>(k0 - k_begin + 32 * u) * b_kmul[t]);
#pragma unroll
          for (int rb = 0; rb < RBMAX; ++rb) {
            if (rb < rbs) {
              uint32_t a0[4], a1[4];
              const uint32_t aaddr = sbase + static_cast<uint32_t>(rb * 16) * p.seg_stride + u * 64;
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
          float tw = q[0] + q[1];
          if (S == 3) tw += q[2];
          t += tw;
        }
        float* dst = res + static_cast<size_t>(v0 + r) * M + m;
        *dst = pn == 0 ? t : *dst + t;
      }
      consumer_sync();  // part is reused by the next super-block
    }
  }
  // ---- fused epilogue over the CTA's results: res[v * M + m] ---------------------
  const int nres = rr.cnt * M;
  if (normed) {  // RMSNorm: y = x / sqrt(mean(x^2) + eps) * g; 1/rms is applied to the results
    if (tid < M) {
      float t = 0.f;
      for (int w = 0; w < kConsumerWarps; ++w) t += ss_part[w * kMmaMaxM + tid];
      rstd_s[tid] = 1.0f / sqrtf(t / static_cast<float>(K) + p.eps);
    }
    consumer_sync();
    for (int idx = tid; idx < nres; idx += kConsumerThreads) res[idx] *= rstd_s[idx % M];
    consumer_sync();
  }
  if (p.epi == EPI_STORE) {  // optional bias: the concat + Linear fusion
    const __nv_bfloat16* bias = static_cast<const __nv_bfloat16*>(p.bias);
    for (int idx = tid; idx < nres; idx += kConsumerThreads) {
      const int v2 = idx / M, mm = idx - v2 * M;
      const float bz = bias ? __bfloat162float(bias[rr.g0 + v2]) : 0.f;
      p.out[(p.m0 + mm) * p.out_ld + G.out_off + rr.g0 + v2] = res[idx] + bz;
    }
  } else if (p.epi == EPI_DGF) {
    // g = sigmoid(Wg [h1||h2] + bg); x = g*h1 + (1-g)*h2
    for (int idx = tid; idx < nres; idx += kConsumerThreads) {
      const int v2 = idx / M, mm = idx - v2 * M;
      const int64_t n = rr.g0 + v2;
      const float bz = __bfloat162float(static_cast<const __nv_bfloat16*>(p.bias)[n]);
      const float g = sigmoidf_acc(res[idx] + bz);
      const float h1 = p.hbuf[static_cast<int64_t>(p.m0 + mm) * 2 * p.d + n];
      const float h2 = p.hbuf[static_cast<int64_t>(p.m0 + mm) * 2 * p.d + p.d + n];
      p.out[(p.m0 + mm) * p.out_ld + n] = g * h1 + (1.0f - g) * h2;
    }
  } else if (p.epi == EPI_RESID) {
    for (int idx = tid; idx < nres; idx += kConsumerThreads) {
      const int v2 = idx / M, mm = idx - v2 * M;
      p.out[(p.m0 + mm) * p.out_ld + rr.g0 + v2] += res[idx];
    }
  } else if (p.epi == EPI_SWIGLU) {
    // act = SiLU(Wgate n) * (Wup n); gate rows are virtual rows [0, cr), up rows [cr, 2cr)
    for (int idx = tid; idx < rr.cr * M; idx += kConsumerThreads) {
      const int r = idx / M, mm = idx - r * M;
      const float gv = res[r * M + mm], uv = res[(rr.cr + r) * M + mm];
      p.out[(p.m0 + mm) * p.out_ld + rr.n0 + r] = gv * sigmoidf_acc(gv) * uv;
    }
  } else {  // EPI_LMHEAD: logits of rows [g0, g0 + cnt) of the vocabulary
    if (p.tap) {
      for (int idx = tid; idx < nres; idx += kConsumerThreads) {
        const int v2 = idx / M, mm = idx - v2 * M;
        p.tap[static_cast<int64_t>(p.m0 + mm) * p.vocab + rr.g0 + v2] = res[idx];
      }
    }
    for (int m = warp; m < M; m += kConsumerWarps) {
      float mx = -INFINITY;
      for (int v2 = lane; v2 < rr.cnt; v2 += 32) mx = fmaxf(mx, res[v2 * M + m]);
      mx = warp_max(mx);
      float se = 0.f;
      for (int v2 = lane; v2 < rr.cnt; v2 += 32) se += expf(res[v2 * M + m] - mx);
      se = warp_sum(se);
      const int64_t pc = static_cast<int64_t>(p.m0 + m) * nct + c;
      if (lane == 0) { p.stat[pc * 2] = mx; p.stat[pc * 2 + 1] = se; }
      // local top-b: b rounds of "best candidate strictly after the previous pick"
      float lv = INFINITY; int li = -1;
      for (int jb = 0; jb < p.b; ++jb) {
        float bv = -INFINITY; int bi = 0x7fffffff;
        for (int v2 = lane; v2 < rr.cnt; v2 += 32) {
          const float val = res[v2 * M + m];
          const int id = static_cast<int>(rr.g0) + v2;
          if (cand_before(lv, li, val, id) && cand_before(val, id, bv, bi)) { bv = val; bi = id; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
          const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
          if (cand_before(ov, oi, bv, bi)) { bv = ov; bi = oi; }
        }
        if (lane == 0) { p.cand_val[pc * kMaxBranch + jb] = bv; p.cand_id[pc * kMaxBranch + jb] = bi; }
        lv = bv; li = bi;
      }
    }
  }
  trace_end(p.trace);
}

}  // namespace dvt

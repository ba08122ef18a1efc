// gemv.cuh -- the weight-streaming GEMV that carries > 95 % of the step's HBM
// bytes (S1 DGF, S2 QKV, S4 O-proj, S5 FFN, S6 LM head).
//
//   Y[m, n] = sum_k X[m, k] * W[n, k]      m < M (draft rows, tiny), W row-major [N, K]
//
// Shape of the kernel (one CTA per SM, 8 consumer warps + 1 producer warp):
//   * the matrix rows are dealt to the CTAs in contiguous ranges whose sizes
//     differ by at most one row, so every SM streams the same number of bytes;
//   * the producer warp copies whole rows (1-D bulk async copies, one per row)
//     into a ring of shared-memory stages guarded by full/empty mbarriers; it
//     starts before griddepcontrol.wait because weights never depend on the
//     previous kernel (programmatic dependent launch hides ramp-up);
//   * consumer thread t keeps the activations of the 16-byte units t, t+256, ...
//     of K in registers (fp32) for MT rows and accumulates with packed fp32
//     FMAs; a transposing shuffle reduction and a fixed-order cross-warp sum
//     give one deterministic value per (row, m);
//   * results of the CTA's rows are kept in shared memory and the fused
//     epilogue (store / DGF gate+blend / residual add / SiLU*up / LM-head
//     top-b + softmax statistics) runs over them once per pass.
#pragma once
#include <cuda_bf16.h>

#include "epilogue.cuh"
#include "ptx.cuh"
#include "state.cuh"

namespace dvt {

enum XKind : int32_t { X_ROWS = 0, X_EMBED = 1 };
enum Epi : int32_t { EPI_STORE = 0, EPI_DGF = 1, EPI_RESID = 2, EPI_SWIGLU = 3, EPI_LMHEAD = 4, EPI_QKV = 5 };

constexpr int kRowsPerStageMax = 4;

struct GemvGroup {
  const void* w[3];      // up to three matrices sharing K and X
  const float* ws[3];    // int8 matrices (k_gemv_mma, WQ = 1): fp32 scale of every output row of w[j]
  int32_t rows[3];
  int32_t n_mat;
  int32_t paired;        // 1: the CTA's row range applies to each matrix (gate/up)
  int32_t pairperm;      // head_dim or 0. EPI_QKV: within every head of the concatenated [q | k | v] rows the virtual
                         // order is (0, dh/2, 1, dh/2 + 1, ...), and CTA ranges start on an even virtual row, so
                         // that the two rows of a rotary pair (i, i + dh/2) belong to the same CTA
  int32_t deal_base, deal_rem;  // dealing of the rows to the group's CTAs, set by the host: CTA c takes deal_base units
                         // (+ 1 for c < deal_rem) starting at unit c * deal_base + min(c, deal_rem); a unit is one row
                         // (of each matrix when paired) or one rotary pair. No division on the device: cta_rows sits
                         // on every role's start-up path.
  int32_t xkind;
  int32_t x_from_dyn;    // X_ROWS: source rows are the caller's hidden_feats
  const float* xsrc;     // X_ROWS: fp32 rows
  int64_t xld;           //         row stride in floats
  const int32_t* xidx;   //         source row of each m (NULL: m)
  const void* embed;     // X_EMBED: [vocab, K] in the storage dtype
  const int32_t* tokens; //          token of each m
  const void* gain;      // RMSNorm gain [K] (storage dtype) or NULL: no norm
  int32_t out_off;       // EPI_STORE: offset added to the output column
  // k_gemv_mma: the B operand of this group as split-bf16 planes (epilogue.cuh), left by the producer of
  // the activation. Row of draft row m: xidx ? xidx[m] : m. X_EMBED: the embedding table itself (one plane).
  const __nv_bfloat16* xs;
  int64_t xs_plane, xs_ld;
  int32_t S;             // planes read per draft row: 3 (all 24 mantissa bits), 2 (16 bits), 1 (bf16 source)
  int32_t S_fixed;       // != 0: S is this (1: the planes hold bf16 values, e.g. embedding rows), else chosen by M
};

struct GemvParams {
  GemvGroup g[2];        // blockIdx.y selects the group (DGF projections use two)
  const StepDyn* dyn;
  int32_t K, M;
  int32_t n_groups, ctas_per_group;  // k_gemv_mma (1-D grid): CTA c works for group c / ctas_per_group
  int32_t rows_per_stage, n_stages, stage_bytes, row_bytes;
  // k_gemv_mma only: K-chunk per stage, stride of a row / column within a stage (bytes)
  int32_t kc, seg_stride;
  int32_t aseg_stride;   // stride of a weight row within a stage (int8 weights: half of the bf16 stride)
  int32_t m0;            // k_gemv_mma: first draft row of this launch (levels wider than 32 rows run in row chunks)
  int32_t epi;
  float eps;
  float* out;            // STORE/SWIGLU: [M, out_ld]; DGF/RESID: residual stream rows x [M, out_ld]
  int64_t out_ld;
  const float* hbuf;     // DGF: [M, 2d] = [h1 || h2]
  const void* bias;      // DGF: gate bias [d]; STORE: optional bias added to the result (fusion linear)
  int32_t d;
  int32_t b;             // LMHEAD: candidates kept per row
  int32_t vocab;
  float* cand_val;       // LMHEAD: [kMaxRows][kMaxBranch][grid]
  int32_t* cand_id;
  float* stat;           // LMHEAD: [kMaxRows][grid][2] = (max, sum exp)
  float* tap;            // LMHEAD: optional logits tap rows [M, vocab]
  // k_gemv_mma, RMSNorm of the input: partial sums of squares of the raw x, [ssq_nct][kMaxRows], left by the
  // epilogue that produced x (the gain is already folded into the planes); NULL: no norm
  const float* ssq_in;
  int32_t ssq_nct;
  // what the epilogue leaves for the next GEMV (epilogue.cuh); all optional
  SplitOut so;           // planes of (result * gain_out)   [draft row][out_off + column]
  const void* gain_out;  // RMSNorm gain of the consumer [N] (storage dtype) or NULL
  SplitOut so_raw;       // planes of the raw result (the last block's x: next level's feature, LM-head input)
  float* ssq_out;        // [gridDim.x][kMaxRows] sum of squares of the raw result over this CTA's columns
  // EPI_QKV (S2 fused into the projection): rotary embedding, K / V append to the cache, rotated and scaled
  // queries as bf16 head + remainder planes for the tensor-core attention kernel
  const RowTables* rt;   // slot[] of this level's rows
  const float2* rope;    // [table rows][dh / 2] = (cos, sin)
  int32_t rope_row0, rope_per_row;
  int32_t Hq, Hkv, layer, level0;
  __nv_bfloat16* qs;     // [2][kMaxRows][Hq * dh]: plane 0 = bf16(q), plane 1 = bf16(q - plane 0)
  unsigned long long* trace;  // dovetail_trace_*: {first CTA start, last CTA end} of this launch, or NULL
};

template <typename WT>
struct Unit;  // one 16-byte unit of a weight row as fp32 pairs
template <>
struct Unit<__nv_bfloat16> {
  static constexpr int EPU = 8;
  __device__ static __forceinline__ void unpack(const uint4& w, float2 (&f)[4]) {
    f[0] = bf16x2_to_f32x2(w.x);
    f[1] = bf16x2_to_f32x2(w.y);
    f[2] = bf16x2_to_f32x2(w.z);
    f[3] = bf16x2_to_f32x2(w.w);
  }
};
template <>
struct Unit<float> {
  static constexpr int EPU = 4;
  __device__ static __forceinline__ void unpack(const uint4& w, float2 (&f)[2]) {
    f[0] = make_float2(__uint_as_float(w.x), __uint_as_float(w.y));
    f[1] = make_float2(__uint_as_float(w.z), __uint_as_float(w.w));
  }
};

struct RowRange {  // the CTA's share of the group's rows, as a list of "virtual rows"
  int32_t cnt;     // virtual rows of this CTA
  int32_t n0, cr;  // paired: first row and rows per matrix
  int64_t g0;      // linearised: first global row
};

__host__ __device__ __forceinline__ RowRange cta_rows(const GemvGroup& G, int c, int /*nct*/) {
  RowRange r;
  const int32_t u0 = c * G.deal_base + (c < G.deal_rem ? c : G.deal_rem), un = G.deal_base + (c < G.deal_rem ? 1 : 0);
  if (G.paired) {
    r.n0 = u0;
    r.cr = un;
    r.cnt = un * G.n_mat;
    r.g0 = 0;
  } else {
    const int32_t unit = G.pairperm ? 2 : 1;  // whole rotary pairs
    r.g0 = static_cast<int64_t>(u0) * unit;
    r.cnt = un * unit;
    r.n0 = 0;
    r.cr = 0;
  }
  return r;
}

// virtual row v -> matrix j, row n within it
__host__ __device__ __forceinline__ void locate_row(const GemvGroup& G, const RowRange& rr, int v, int& j,
                                           int& n) {
  if (G.paired) {
    j = (v >= rr.cr ? 1 : 0) + (v >= 2 * rr.cr ? 1 : 0);  // n_mat <= 3
    n = rr.n0 + (v - j * rr.cr);
  } else {
    int32_t g = static_cast<int32_t>(rr.g0) + v;
    if (G.pairperm) {  // virtual (0, 1, 2, 3, ...) of a head = rows (0, dh/2, 1, dh/2 + 1, ...); dh is a power of two
      const int32_t w = g & (G.pairperm - 1);
      g = g - w + (w >> 1) + (w & 1) * (G.pairperm >> 1);
    }
    j = 0;
    if (g >= G.rows[0]) {
      g -= G.rows[0];
      j = 1;
      if (g >= G.rows[1]) {
        g -= G.rows[1];
        j = 2;
      }
    }
    n = g;
  }
}

// ---- fused epilogue over the CTA's results --------------------------------------------------
// Operands of the epilogue that exist before the GEMV itself has run (residual stream, [h1 || h2], bias, the
// consumer's norm gain): loaded into registers at kernel start so that the epilogue does not wait for L2 after
// the last weight stage. Covers the first kEpiPre results of each thread; later ones are loaded late.
constexpr int kEpiPre = 2;
struct EpiRegs {
  float a[kEpiPre], b[kEpiPre], bz[kEpiPre], g[kEpiPre];
};

__device__ __forceinline__ void epi_load(const GemvParams& p, const GemvGroup& G, const RowRange& rr, int idx, int cnt,
                                         int mbase, bool bf16, float& a, float& b, float& bz, float& g) {
  const int m = idx / cnt, v = idx - m * cnt;
  const int64_t mm = mbase + m, n = rr.g0 + v;
  a = b = bz = 0.f;
  g = 1.f;
  if (p.epi == EPI_STORE) {
    if (p.bias) bz = load_storage(p.bias, n, bf16);
  } else if (p.epi == EPI_DGF) {
    bz = load_storage(p.bias, n, bf16);
    a = p.hbuf[mm * 2 * p.d + n];
    b = p.hbuf[mm * 2 * p.d + p.d + n];
  } else {
    a = p.out[mm * p.out_ld + G.out_off + n];  // residual stream
  }
  if (p.so.xs && p.gain_out) g = load_storage(p.gain_out, n, bf16);
}

__device__ __forceinline__ void epi_prefetch(const GemvParams& p, const GemvGroup& G, const RowRange& rr, int Mt, int mbase,
                                             bool bf16, EpiRegs& r) {
  if (p.epi != EPI_STORE && p.epi != EPI_DGF && p.epi != EPI_RESID) return;
#pragma unroll
  for (int i = 0; i < kEpiPre; ++i) {
    const int idx = threadIdx.x + i * kConsumerThreads;
    if (idx < rr.cnt * Mt) epi_load(p, G, rr, idx, rr.cnt, mbase, bf16, r.a[i], r.b[i], r.bz[i], r.g[i]);
  }
}

// res(v, m): result of the CTA's virtual row v for draft row mbase + m, m < Mt (already scaled by 1 / rms
// when the input is normed). Runs on the kConsumerThreads consumer threads of either GEMV kernel.
// pre: operands loaded by epi_prefetch, or NULL.
template <typename Res>
__device__ __forceinline__ void gemv_epilogue(const GemvParams& p, const GemvGroup& G, const RowRange& rr, Res res,
                                              int Mt, int mbase, int c, int nct, bool bf16, const EpiRegs* pre = nullptr) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int cnt = rr.cnt;
  if (p.epi == EPI_STORE || p.epi == EPI_DGF || p.epi == EPI_RESID) {
    int it = 0;
    for (int idx = tid; idx < cnt * Mt; idx += kConsumerThreads, ++it) {
      const int m = idx / cnt, v = idx - m * cnt;
      const int64_t mm = mbase + m, n = rr.g0 + v;
      float a, b, bz, g;
      if (pre != nullptr && it < kEpiPre) {
        a = pre->a[it < kEpiPre ? it : 0]; b = pre->b[it < kEpiPre ? it : 0];
        bz = pre->bz[it < kEpiPre ? it : 0]; g = pre->g[it < kEpiPre ? it : 0];
      } else {
        epi_load(p, G, rr, idx, cnt, mbase, bf16, a, b, bz, g);
      }
      float y = res(v, m);
      float* dst = p.out + mm * p.out_ld + G.out_off + n;
      if (p.epi == EPI_STORE) {  // optional bias: the concat + Linear fusion
        y += bz;
      } else if (p.epi == EPI_DGF) {
        // g = sigmoid(Wg [h1||h2] + bg); x = g*h1 + (1-g)*h2
        const float gt = sigmoidf_acc(y + bz);
        y = gt * a + (1.0f - gt) * b;
      } else {
        y += a;  // residual stream
      }
      *dst = y;
      res(v, m) = y;
      if (p.so.xs) store_split(p.so, mm, G.out_off + n, p.gain_out ? y * g : y);
      if (p.so_raw.xs) store_split(p.so_raw, mm, n, y);
    }
    if (p.ssq_out) {  // sum of squares of the raw result over this CTA's columns, fixed order
      consumer_sync();
      for (int m = warp; m < Mt; m += kConsumerWarps) {
        float t = 0.f;
        for (int v = lane; v < cnt; v += 32) t = fmaf(res(v, m), res(v, m), t);
        t = warp_sum(t);
        if (lane == 0) p.ssq_out[static_cast<int64_t>(c) * kMaxRows + mbase + m] = t;
      }
    }
  } else if (p.epi == EPI_QKV) {
    // S2 (reading A3): q, k of a head are rotated by the row's position, half-split pairing
    // (i, i + dh/2) = virtual rows (2i, 2i + 1) of the head; K (post-RoPE) and V are rounded to the cache dtype and
    // appended at cache row Lbase + slot[m]; q is scaled by 1 / sqrt(dh) and left as bf16 head + remainder.
    const int DH = G.pairperm, HALF = DH >> 1;
    const StepDyn* dyn = p.dyn;
    const int Lbase = p.level0 ? dyn->L : dyn->Lp;
    const int64_t cap = dyn->capacity;
    const float scale = 1.0f / sqrtf(static_cast<float>(DH));
    const int dq = p.Hq * DH;
    const int n_pairs = cnt >> 1;
    for (int idx = tid; idx < n_pairs * Mt; idx += kConsumerThreads) {
      const int m = idx / n_pairs, t = idx - m * n_pairs;
      const int mm = mbase + m;
      const int64_t g = rr.g0 + 2 * t;
      const int dsh = DH == 128 ? 7 : 6;  // head_dim is 64 or 128
      const int hh = static_cast<int>(g >> dsh), i = static_cast<int>(g & (DH - 1)) >> 1;
      const float a = res(2 * t, m), b = res(2 * t + 1, m);  // elements i and i + dh/2 of head hh
      if (hh < p.Hq + p.Hkv) {
        const float2 cs = p.rope[static_cast<size_t>(p.rope_row0 + (p.rope_per_row ? mm : 0)) * HALF + i];
        if (hh < p.Hq) {
          const float x[2] = {(a * cs.x - b * cs.y) * scale, (b * cs.x + a * cs.y) * scale};
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const uint16_t hi = f32_to_bf16_rn(x[h]);
            const float rem = x[h] - __uint_as_float(static_cast<uint32_t>(hi) << 16);
            uint16_t* dst = reinterpret_cast<uint16_t*>(p.qs) + static_cast<size_t>(mm) * dq + hh * DH + i + h * HALF;
            dst[0] = hi;
            dst[static_cast<size_t>(kMaxRows) * dq] = f32_to_bf16_rn(rem);
          }
        } else {
          uint16_t* dst = static_cast<uint16_t*>(dyn->kc) +
                          ((static_cast<size_t>(p.layer) * p.Hkv + (hh - p.Hq)) * cap + Lbase + p.rt->slot[mm]) * DH + i;
          dst[0] = f32_to_bf16_rn(a * cs.x - b * cs.y);
          dst[HALF] = f32_to_bf16_rn(b * cs.x + a * cs.y);
        }
      } else {
        uint16_t* dst = static_cast<uint16_t*>(dyn->vc) +
                        ((static_cast<size_t>(p.layer) * p.Hkv + (hh - p.Hq - p.Hkv)) * cap + Lbase + p.rt->slot[mm]) * DH + i;
        dst[0] = f32_to_bf16_rn(a);
        dst[HALF] = f32_to_bf16_rn(b);
      }
    }
  } else if (p.epi == EPI_SWIGLU) {
    // act = SiLU(Wgate n) * (Wup n); gate rows are virtual rows [0, cr), up rows [cr, 2cr)
    for (int idx = tid; idx < rr.cr * Mt; idx += kConsumerThreads) {
      const int m = idx / rr.cr, r = idx - m * rr.cr;
      const int64_t mm = mbase + m;
      const float gv = res(r, m), uv = res(rr.cr + r, m);
      const float y = gv * sigmoidf_acc(gv) * uv;
      p.out[mm * p.out_ld + rr.n0 + r] = y;
      if (p.so.xs) store_split(p.so, mm, rr.n0 + r, y);
    }
  } else {  // EPI_LMHEAD: logits of rows [g0, g0 + cnt) of the vocabulary
    if (p.tap) {
      for (int idx = tid; idx < cnt * Mt; idx += kConsumerThreads) {
        const int m = idx / cnt, v = idx - m * cnt;
        p.tap[static_cast<int64_t>(mbase + m) * p.vocab + rr.g0 + v] = res(v, m);
      }
    }
    for (int m = warp; m < Mt; m += kConsumerWarps) {
      float mx = -INFINITY;
      for (int v = lane; v < cnt; v += 32) mx = fmaxf(mx, res(v, m));
      mx = warp_max(mx);
      float se = 0.f;
      for (int v = lane; v < cnt; v += 32) se += expf(res(v, m) - mx);
      se = warp_sum(se);
      const int64_t pc = static_cast<int64_t>(mbase + m) * nct + c;
      if (lane == 0) { p.stat[pc * 2] = mx; p.stat[pc * 2 + 1] = se; }
      // local top-b: b rounds of "best candidate strictly after the previous pick", on order-preserving keys
      // (epilogue.cuh cand_key / cand_lo): a lane's best is a max over independent values and the warp's best two
      // redux.sync.max (chains of cand_before and five shuffle rounds cost ~5 us per row at 10 children).
      uint64_t bound = ~0ull;
      for (int jb = 0; jb < p.b; ++jb) {
        uint64_t best = 0ull;
#pragma unroll 4
        for (int v = lane; v < cnt; v += 32) {
          const int id = static_cast<int>(rr.g0) + v;
          const uint64_t key = (static_cast<uint64_t>(cand_key(res(v, m), id)) << 32) | cand_lo(id, 0);
          best = umax64(best, key < bound ? key : 0ull);
        }
        const uint32_t bh = static_cast<uint32_t>(best >> 32), bl = static_cast<uint32_t>(best);
        const uint32_t gh = __reduce_max_sync(0xffffffffu, bh);
        const uint32_t gl = __reduce_max_sync(0xffffffffu, bh == gh ? bl : 0u);
        bound = (static_cast<uint64_t>(gh) << 32) | gl;
        if (lane == 0) {  // entry-major: the heads (jb = 0) of a row's lists are contiguous for k_tree_level
          const int64_t o = (static_cast<int64_t>(mbase + m) * kMaxBranch + jb) * nct + c;
          p.cand_val[o] = cand_key_value(gh);
          p.cand_id[o] = gh != 0u ? static_cast<int>(0xffffffu - (gl >> 8)) : kNoCand;
        }
      }
    }
  }
}

template <typename WT, int MT, int NI>
__global__ void __launch_bounds__(kThreads, 1) k_gemv(const GemvParams p) {
  constexpr int EPU = Unit<WT>::EPU;
  constexpr int PAIRS = EPU / 2;
  constexpr int R = kRowsPerStageMax;
  constexpr int V = R * MT;
  extern __shared__ __align__(128) uint8_t smem[];

  const GemvGroup& G = p.g[blockIdx.y];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nct = gridDim.x, c = blockIdx.x;
  const int NS = p.n_stages, RS = p.rows_per_stage;

  uint8_t* ring = smem;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + static_cast<size_t>(NS) * p.stage_bytes);
  uint64_t* empty = full + 8;
  float* part = reinterpret_cast<float*>(empty + 8);  // [2][warps][V]
  float* rstd_s = part + 2 * kConsumerWarps * V;      // [4]
  float* red_s = rstd_s + 4;                          // [warps][4]
  float* res = red_s + kConsumerWarps * 4;            // [cnt][MT]

  const RowRange rr = cta_rows(G, c, nct);
  trace_begin(p.trace);
  const int spp = (rr.cnt + RS - 1) / RS;  // stages per pass over the CTA's rows
  const int m_tiles = (p.M + MT - 1) / MT;
  const int U = p.row_bytes >> 4;          // 16-byte units per row

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kConsumerWarps);
    }
    mbar_fence_init();
  }
  __syncthreads();
  pdl_launch_dependents();

  if (warp == kConsumerWarps) {
    // ---------------- producer: stream this CTA's rows, once per m-tile -----
    const uint64_t pol = l2_policy_evict_first();
    int it = 0;
    for (int mt = 0; mt < m_tiles; ++mt) {
      for (int s = 0; s < spp; ++s, ++it) {
        const int slot = it % NS;
        if (it >= NS) mbar_wait(&empty[slot], ((it / NS) & 1) ^ 1);
        const int nr = min(RS, rr.cnt - s * RS);
        if (lane == 0) mbar_arrive_expect_tx(&full[slot], static_cast<uint32_t>(nr) * p.row_bytes);
        __syncwarp();
        if (lane < nr) {
          int j, n;
          locate_row(G, rr, s * RS + lane, j, n);
          const uint8_t* src = static_cast<const uint8_t*>(G.w[j]) + static_cast<size_t>(n) * p.row_bytes;
          bulk_g2s(ring + static_cast<size_t>(slot) * p.stage_bytes + static_cast<size_t>(lane) * p.row_bytes,
                   src, p.row_bytes, &full[slot], pol);
        }
      }
    }
    return;
  }

  // ---------------- consumers -------------------------------------------------
  pdl_wait();  // activations of the previous kernel are visible from here on
  const StepDyn* dyn = p.dyn;
  const bool normed = G.gain != nullptr;

  for (int mt = 0; mt < m_tiles; ++mt) {
    const int m0 = mt * MT;
    // X slice of this thread: units tid, tid+256, ... of K, MT rows, fp32 pairs
    float2 xx[MT][NI][PAIRS];
    float ss[MT];
#pragma unroll
    for (int m = 0; m < MT; ++m) {
      ss[m] = 0.f;
      const int mm = m0 + m;
      const bool mvalid = mm < p.M;
      const float* xrow = nullptr;
      const WT* erow = nullptr;
      if (mvalid) {
        if (G.xkind == X_ROWS) {
          const float* base = G.x_from_dyn ? dyn->feats : G.xsrc;
          const int64_t ri = G.xidx ? G.xidx[mm] : mm;
          xrow = base + ri * G.xld;
        } else {
          erow = static_cast<const WT*>(G.embed) + static_cast<size_t>(G.tokens[mm]) * p.K;
        }
      }
#pragma unroll
      for (int i = 0; i < NI; ++i) {
        const int u = tid + i * kConsumerThreads;
        float xv[EPU];
#pragma unroll
        for (int e = 0; e < EPU; ++e) xv[e] = 0.f;
        if (mvalid && u < U) {
          if (xrow) {
#pragma unroll
            for (int q = 0; q < EPU / 4; ++q) {
              const float4 t4 = *reinterpret_cast<const float4*>(xrow + static_cast<size_t>(u) * EPU + q * 4);
              xv[q * 4 + 0] = t4.x; xv[q * 4 + 1] = t4.y; xv[q * 4 + 2] = t4.z; xv[q * 4 + 3] = t4.w;
            }
          } else {
            const uint4 w = *reinterpret_cast<const uint4*>(erow + static_cast<size_t>(u) * EPU);
            float2 f[PAIRS];
            Unit<WT>::unpack(w, f);
#pragma unroll
            for (int q = 0; q < PAIRS; ++q) { xv[2 * q] = f[q].x; xv[2 * q + 1] = f[q].y; }
          }
          if (normed) {
#pragma unroll
            for (int e = 0; e < EPU; ++e) ss[m] = fmaf(xv[e], xv[e], ss[m]);
            const uint4 gw = *reinterpret_cast<const uint4*>(static_cast<const WT*>(G.gain) + static_cast<size_t>(u) * EPU);
            float2 gf[PAIRS];
            Unit<WT>::unpack(gw, gf);
#pragma unroll
            for (int q = 0; q < PAIRS; ++q) { xv[2 * q] *= gf[q].x; xv[2 * q + 1] *= gf[q].y; }
          }
        }
#pragma unroll
        for (int q = 0; q < PAIRS; ++q) xx[m][i][q] = make_float2(xv[2 * q], xv[2 * q + 1]);
      }
    }
    if (normed) {  // RMSNorm: y = x / sqrt(mean(x^2) + eps) * g; 1/rms is applied to the results
#pragma unroll
      for (int m = 0; m < MT; ++m) {
        const float t = warp_sum(ss[m]);
        if (lane == 0) red_s[warp * 4 + m] = t;
      }
      consumer_sync();
      if (tid < MT) {
        float t = 0.f;
        for (int w = 0; w < kConsumerWarps; ++w) t += red_s[w * 4 + tid];
        rstd_s[tid] = 1.0f / sqrtf(t / static_cast<float>(p.K) + p.eps);
      }
      // visibility of rstd_s is ordered by the consumer_sync()s of the stage loop / epilogue
    }

    // ---- stream the rows ---------------------------------------------------
    for (int s = 0; s < spp; ++s) {
      const int it = mt * spp + s;
      const int slot = it % NS;
      const int nr = min(RS, rr.cnt - s * RS);
      mbar_wait(&full[slot], (it / NS) & 1);
      const uint8_t* sb = ring + static_cast<size_t>(slot) * p.stage_bytes;
      float2 acc[R][MT];
#pragma unroll
      for (int r = 0; r < R; ++r)
#pragma unroll
        for (int m = 0; m < MT; ++m) acc[r][m] = make_float2(0.f, 0.f);
#pragma unroll
      for (int i = 0; i < NI; ++i) {
        const int u = tid + i * kConsumerThreads;
        if (u < U) {
#pragma unroll
          for (int r = 0; r < R; ++r) {
            if (r < nr) {
              const uint4 w = *reinterpret_cast<const uint4*>(sb + static_cast<size_t>(r) * p.row_bytes + (static_cast<size_t>(u) << 4));
              float2 wf[PAIRS];
              Unit<WT>::unpack(w, wf);
#pragma unroll
              for (int q = 0; q < PAIRS; ++q)
#pragma unroll
                for (int m = 0; m < MT; ++m) ffma2(acc[r][m], wf[q], xx[m][i][q]);
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[slot]);  // the stage's bytes are in registers now

      float v[V];
#pragma unroll
      for (int r = 0; r < R; ++r)
#pragma unroll
        for (int m = 0; m < MT; ++m) v[r * MT + m] = acc[r][m].x + acc[r][m].y;
      const float tot = warp_reduce_transpose<V>(v, lane);
      float* pb = part + (it & 1) * (kConsumerWarps * V);
      if ((lane & (32 / V - 1)) == 0) pb[warp * V + lane / (32 / V)] = tot;
      consumer_sync();
      if (tid < nr * MT) {  // fixed-order sum over the warps: deterministic
        float t = 0.f;
#pragma unroll
        for (int w = 0; w < kConsumerWarps; ++w) t += pb[w * V + tid];
        res[(s * RS) * MT + tid] = t;
      }
    }
    consumer_sync();

    // ---- fused epilogue over the CTA's results -------------------------------
    const int nres = rr.cnt * MT;
    if (normed) {
      for (int idx = tid; idx < nres; idx += kConsumerThreads) res[idx] *= rstd_s[idx % MT];
      consumer_sync();
    }
    gemv_epilogue(p, G, rr, [&](int v, int m) -> float& { return res[v * MT + m]; }, min(MT, p.M - m0), m0, c, nct,
                  sizeof(WT) == 2);
    consumer_sync();  // res is reused by the next m-tile
  }
  trace_end(p.trace);
}

}  // namespace dvt

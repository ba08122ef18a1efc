// attention.cuh -- S2 (rotary embedding + KV append) and S3 (tree attention,
// the draft tree is built by autoregressive decoding, so every
// tree row attends the committed prefix, its tree ancestors and itself).
//
// Grid = (n_chunks, Hkv). CTA (c, hk) streams positions [c*PCH, (c+1)*PCH) of
// the prefix K/V of kv-head hk through a shared-memory ring (bulk async
// copies; the cache layout [layer][kv_head][capacity][head_dim] makes a run of
// positions one contiguous block) and keeps an fp32 online-softmax state for
// QT query vectors (rows x the q-heads of the GQA group). The CTA with c == 0
// also owns the "new region": it applies RoPE to this level's K, rounds K/V to
// the cache dtype, appends them, and attends the new-region slots each row's
// ancestor mask allows, reading the values as stored (the oracle attends the
// stored, rounded rows too). Partials (m, l, o) are merged in chunk order by
// the last CTA of a kv-head to finish: fixed order, deterministic.
#pragma once
#include <cuda_bf16.h>

#include "epilogue.cuh"
#include "ptx.cuh"
#include "state.cuh"

namespace dvt {


constexpr int kAttnStagePos = 32;  // positions per ring stage

struct AttnParams {
  const StepDyn* dyn;
  const float* qkv;        // [M][dq + 2*dkv] raw q, k, v of this level's rows (fp32)
  float* obuf;             // [M][dq]
  const __nv_bfloat16* qs; // k_tree_attention_mma with the S2 work fused into the QKV projection (gemv.cuh EPI_QKV):
                           // rotated, scaled queries [2][kMaxRows][dq] (bf16 head, remainder); K / V already appended
  SplitOut so;             // the same as split-bf16 planes for the O-projection GEMV (epilogue.cuh), or xs == NULL
  const RowTables* rows;
  const float2* rope;      // [table rows][dh/2] = (cos, sin) of the rotary angle
  int32_t rope_row0;       // table row of m = 0
  int32_t rope_per_row;    // 1: row m uses rope_row0 + m (level 0); 0: all rows share rope_row0
  int32_t M, Hq, Hkv, layer;
  int32_t level0;          // 1: Lbase = L (level-0 rows); 0: Lbase = L + n_new (tree rows)
  int32_t new_cnt;         // new-region slots that exist once this level's rows are appended
  int32_t n_stages;
  float* ws;               // partials [Hkv][n_chunks][qv_cap][dh + 2]
  int32_t qv_cap;
  int32_t* counters;       // [Hkv], zero between launches
  // k_tree_attention_mma: the cache of this step as launch arguments, so that the producers can
  // stream the prefix before griddepcontrol.wait (the prefix does not depend on this level)
  const void* kc;
  const void* vc;
  int32_t cap, Lbase;
  int32_t Lsafe;           // committed_len at step entry: rows below it are never written by the step
  unsigned long long* trace;  // dovetail_trace_*: {first CTA start, last CTA end} of this launch, or NULL
};

struct SoftState {  // running (max, sum) of one query vector
  float m, l;
};

// merge (m2, l2, o2) into (m1, l1, o1); -inf maxima mean "nothing seen yet"
template <int E>
__device__ __forceinline__ void softmax_merge(float& m1, float& l1, float (&o1)[E], float m2, float l2,
                                              const float (&o2)[E]) {
  const float mn = fmaxf(m1, m2);
  const float c1 = (m1 == -INFINITY) ? 0.f : expf(m1 - mn);
  const float c2 = (m2 == -INFINITY) ? 0.f : expf(m2 - mn);
  l1 = l1 * c1 + l2 * c2;
#pragma unroll
  for (int e = 0; e < E; ++e) o1[e] = o1[e] * c1 + o2[e] * c2;
  m1 = mn;
}

template <typename WT>
__device__ __forceinline__ void load_unit_f32(const void* p, float* f);
template <>
__device__ __forceinline__ void load_unit_f32<__nv_bfloat16>(const void* p, float* f) {
  const uint4 w = *reinterpret_cast<const uint4*>(p);
  float2 t;
  t = bf16x2_to_f32x2(w.x); f[0] = t.x; f[1] = t.y;
  t = bf16x2_to_f32x2(w.y); f[2] = t.x; f[3] = t.y;
  t = bf16x2_to_f32x2(w.z); f[4] = t.x; f[5] = t.y;
  t = bf16x2_to_f32x2(w.w); f[6] = t.x; f[7] = t.y;
}
template <>
__device__ __forceinline__ void load_unit_f32<float>(const void* p, float* f) {
  const float4 w = *reinterpret_cast<const float4*>(p);
  f[0] = w.x; f[1] = w.y; f[2] = w.z; f[3] = w.w;
}

__device__ __forceinline__ void store_cache(__nv_bfloat16* p, float v) {
  *reinterpret_cast<uint16_t*>(p) = f32_to_bf16_rn(v);
}
__device__ __forceinline__ void store_cache(float* p, float v) { *p = v; }

template <typename WT, int DH, int QT>
__global__ void __launch_bounds__(kThreads, 2) k_tree_attention(const AttnParams p) {
  constexpr int EPU = 16 / sizeof(WT);
  constexpr int ROWB = DH * sizeof(WT);          // bytes of one K (or V) row
  constexpr int LPR = ROWB / 16;                 // lanes that cover one row
  constexpr int GPW = 32 / LPR;                  // rows a warp handles at once
  constexpr int NG = kConsumerWarps * GPW;       // row groups of the CTA
  constexpr int PS = kAttnStagePos;
  constexpr int HALF = DH / 2;
  constexpr int STAGE_BYTES = 2 * PS * ROWB;
  constexpr int WSTR = DH + 2;                   // partial record: o[DH], m, l
  static_assert(LPR >= 1 && LPR <= 32, "head_dim / dtype not supported");
  extern __shared__ __align__(128) uint8_t smem[];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int c = blockIdx.x, hk = blockIdx.y, n_chunks = gridDim.x;
  const int NS = p.n_stages;
  const int grp = p.Hq / p.Hkv;
  const int qv_tot = p.M * grp;  // query vectors that share this kv-head
  const int n_qt = (qv_tot + QT - 1) / QT;
  const int dq = p.Hq * DH, dkv = p.Hkv * DH, ldq = dq + 2 * dkv;

  uint8_t* ring = smem;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + static_cast<size_t>(NS) * STAGE_BYTES);
  uint64_t* empty = full + 8;
  float* wsm = reinterpret_cast<float*>(empty + 8);           // [warps][QT][WSTR]
  int* flag_s = reinterpret_cast<int*>(wsm + kConsumerWarps * QT * WSTR);

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kConsumerWarps);
    }
    mbar_fence_init();
  }
  __syncthreads();
  pdl_launch_dependents();
  trace_begin(p.trace);
  pdl_wait();  // q/k/v of this level and the step's dynamic state are visible
  const StepDyn* dyn = p.dyn;
  const int Lbase = p.level0 ? dyn->L : dyn->Lp;
  const int cap = dyn->capacity;
  const WT* kc = static_cast<const WT*>(dyn->kc) + (static_cast<size_t>(p.layer) * p.Hkv + hk) * cap * DH;
  const WT* vc = static_cast<const WT*>(dyn->vc) + (static_cast<size_t>(p.layer) * p.Hkv + hk) * cap * DH;
  // this CTA's share of the prefix
  int pch = (Lbase + n_chunks - 1) / n_chunks;
  pch = (pch + PS - 1) / PS * PS;
  const int p_begin = min(Lbase, c * pch), p_end = min(Lbase, p_begin + pch);
  const int n_st = (p_end - p_begin + PS - 1) / PS;

  if (warp == kConsumerWarps) {
    // ---------------- producer ------------------------------------------------
    const uint64_t pol = l2_policy_evict_last();  // the prefix is re-read by every level
    int it = 0;
    for (int qt = 0; qt < n_qt; ++qt) {
      for (int s = 0; s < n_st; ++s, ++it) {
        const int slot = it % NS;
        if (it >= NS) mbar_wait(&empty[slot], ((it / NS) & 1) ^ 1);
        const int pos0 = p_begin + s * PS;
        const uint32_t bytes = static_cast<uint32_t>(min(PS, p_end - pos0)) * ROWB;
        if (lane == 0) mbar_arrive_expect_tx(&full[slot], 2 * bytes);
        __syncwarp();
        uint8_t* dst = ring + static_cast<size_t>(slot) * STAGE_BYTES;
        if (lane == 0) bulk_g2s(dst, kc + static_cast<size_t>(pos0) * DH, bytes, &full[slot], pol);
        if (lane == 1) bulk_g2s(dst + PS * ROWB, vc + static_cast<size_t>(pos0) * DH, bytes, &full[slot], pol);
      }
    }
    return;
  }

  // ---------------- consumers ---------------------------------------------------
  const RowTables* rows = p.rows;
  const int gl = lane % LPR;            // lane within its row group
  const int gid = warp * GPW + lane / LPR;
  const int d0 = gl * EPU;              // first head dimension this lane owns
  const float scale = 1.0f / sqrtf(static_cast<float>(DH));

  // S2: append this level's K/V rows of kv-head hk (c == 0 only). K is rotated
  // (half-split pairing (i, i + dh/2), reading A3) and both are rounded to the
  // cache dtype, as the oracle stores them.
  if (c == 0) {
    WT* kcw = const_cast<WT*>(kc);
    WT* vcw = const_cast<WT*>(vc);
    for (int idx = tid; idx < p.M * HALF; idx += kConsumerThreads) {
      const int m = idx / HALF, i = idx % HALF;
      const float* kr = p.qkv + static_cast<size_t>(m) * ldq + dq + hk * DH;
      const float2 cs = p.rope[static_cast<size_t>(p.rope_row0 + (p.rope_per_row ? m : 0)) * HALF + i];
      const float a = kr[i], b = kr[i + HALF];
      WT* dst = kcw + static_cast<size_t>(Lbase + rows->slot[m]) * DH;
      store_cache(dst + i, a * cs.x - b * cs.y);
      store_cache(dst + i + HALF, b * cs.x + a * cs.y);
    }
    for (int idx = tid; idx < p.M * DH; idx += kConsumerThreads) {
      const int m = idx / DH, i = idx % DH;
      const float* vr = p.qkv + static_cast<size_t>(m) * ldq + dq + dkv + hk * DH;
      store_cache(vcw + static_cast<size_t>(Lbase + rows->slot[m]) * DH + i, vr[i]);
    }
    __threadfence_block();
    consumer_sync();
  }

  for (int qt = 0; qt < n_qt; ++qt) {
    // rotated, scaled query slices of this lane
    float q[QT][EPU];
    int qm[QT];  // row of each query vector, -1 when past the end
#pragma unroll
    for (int t = 0; t < QT; ++t) {
      const int qv = qt * QT + t;
      qm[t] = qv < qv_tot ? qv / grp : -1;
      if (qm[t] >= 0) {
        const int hq = hk * grp + qv % grp;
        const float* qr = p.qkv + static_cast<size_t>(qm[t]) * ldq + hq * DH;
        const float2* cs = p.rope + static_cast<size_t>(p.rope_row0 + (p.rope_per_row ? qm[t] : 0)) * HALF;
#pragma unroll
        for (int e = 0; e < EPU; ++e) {
          const int dd = d0 + e;
          const int i = dd < HALF ? dd : dd - HALF;
          const float2 f = cs[i];
          const float a = qr[dd], b = qr[dd < HALF ? dd + HALF : dd - HALF];
          q[t][e] = (dd < HALF ? a * f.x - b * f.y : a * f.x + b * f.y) * scale;
        }
      } else {
#pragma unroll
        for (int e = 0; e < EPU; ++e) q[t][e] = 0.f;
      }
    }
    float mrun[QT], lrun[QT], o[QT][EPU];
#pragma unroll
    for (int t = 0; t < QT; ++t) {
      mrun[t] = -INFINITY;
      lrun[t] = 0.f;
#pragma unroll
      for (int e = 0; e < EPU; ++e) o[t][e] = 0.f;
    }

    // one position: scores of the QT queries against k, online-softmax update with v
    auto update = [&](const float (&kf)[EPU], const float (&vf)[EPU], const bool (&ok)[QT]) {
#pragma unroll
      for (int t = 0; t < QT; ++t) {
        float s = 0.f;
#pragma unroll
        for (int e = 0; e < EPU; ++e) s = fmaf(q[t][e], kf[e], s);
#pragma unroll
        for (int off = LPR / 2; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
        const float mn = ok[t] ? fmaxf(mrun[t], s) : mrun[t];
        const float corr = (mrun[t] == -INFINITY) ? 0.f : expf(mrun[t] - mn);
        const float pw = ok[t] ? expf(s - mn) : 0.f;
        lrun[t] = lrun[t] * corr + pw;
#pragma unroll
        for (int e = 0; e < EPU; ++e) o[t][e] = fmaf(pw, vf[e], o[t][e] * corr);
        mrun[t] = mn;
      }
    };

    // ---- the prefix chunk, from the ring ------------------------------------
    for (int s = 0; s < n_st; ++s) {
      const int it = qt * n_st + s;
      const int slot = it % NS;
      const int npos = min(PS, p_end - (p_begin + s * PS));
      mbar_wait(&full[slot], (it / NS) & 1);
      const uint8_t* sb = ring + static_cast<size_t>(slot) * STAGE_BYTES;
#pragma unroll
      for (int i = 0; i < PS / NG; ++i) {
        const int pl = gid + i * NG;
        const bool valid = pl < npos;
        float kf[EPU], vf[EPU];
        if (valid) {
          load_unit_f32<WT>(sb + pl * ROWB + gl * 16, kf);
          load_unit_f32<WT>(sb + PS * ROWB + pl * ROWB + gl * 16, vf);
        } else {
#pragma unroll
          for (int e = 0; e < EPU; ++e) { kf[e] = 0.f; vf[e] = 0.f; }
        }
        bool ok[QT];
#pragma unroll
        for (int t = 0; t < QT; ++t) ok[t] = valid && qm[t] >= 0;
        update(kf, vf, ok);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[slot]);
    }
    // ---- the new region: earlier rows of this step, masked per row ------------
    if (c == 0) {
      for (int j0 = 0; j0 < p.new_cnt; j0 += NG) {
        const int j = j0 + gid;
        const bool valid = j < p.new_cnt;
        float kf[EPU], vf[EPU];
        if (valid) {
          // stored (rounded) values, read back through L2: rows of this level were
          // written by this CTA above, older rows by earlier kernels
          const WT* kr = kc + static_cast<size_t>(Lbase + j) * DH + d0;
          const WT* vr = vc + static_cast<size_t>(Lbase + j) * DH + d0;
          const uint4 kw = __ldcg(reinterpret_cast<const uint4*>(kr));
          const uint4 vw = __ldcg(reinterpret_cast<const uint4*>(vr));
          load_unit_f32<WT>(&kw, kf);
          load_unit_f32<WT>(&vw, vf);
        } else {
#pragma unroll
          for (int e = 0; e < EPU; ++e) { kf[e] = 0.f; vf[e] = 0.f; }
        }
        bool ok[QT];
#pragma unroll
        for (int t = 0; t < QT; ++t)
          ok[t] = valid && qm[t] >= 0 && ((rows->mask[qm[t]][j >> 5] >> (j & 31)) & 1u);
        update(kf, vf, ok);
      }
    }
    // ---- merge the row groups of the warp, then the warps ---------------------
#pragma unroll
    for (int t = 0; t < QT; ++t) {
#pragma unroll
      for (int off = LPR; off < 32; off <<= 1) {
        const float m2 = __shfl_xor_sync(0xffffffffu, mrun[t], off);
        const float l2 = __shfl_xor_sync(0xffffffffu, lrun[t], off);
        float o2[EPU];
#pragma unroll
        for (int e = 0; e < EPU; ++e) o2[e] = __shfl_xor_sync(0xffffffffu, o[t][e], off);
        softmax_merge<EPU>(mrun[t], lrun[t], o[t], m2, l2, o2);
      }
      if (lane < LPR) {
        float* w = wsm + (warp * QT + t) * WSTR;
#pragma unroll
        for (int e = 0; e < EPU; ++e) w[d0 + e] = o[t][e];
        if (lane == 0) { w[DH] = mrun[t]; w[DH + 1] = lrun[t]; }
      }
    }
    consumer_sync();
    for (int idx = tid; idx < QT * DH; idx += kConsumerThreads) {
      const int t = idx / DH, dd = idx % DH;
      const int qv = qt * QT + t;
      if (qv >= qv_tot) continue;
      float mm = -INFINITY;
      for (int w = 0; w < kConsumerWarps; ++w) mm = fmaxf(mm, wsm[(w * QT + t) * WSTR + DH]);
      float ll = 0.f, oo = 0.f;
      for (int w = 0; w < kConsumerWarps; ++w) {
        const float* r = wsm + (w * QT + t) * WSTR;
        const float cw = (r[DH] == -INFINITY) ? 0.f : expf(r[DH] - mm);
        ll += r[DH + 1] * cw;
        oo += r[dd] * cw;
      }
      if (n_chunks == 1) {
        const int m = qv / grp, hq = hk * grp + qv % grp;
        {
          const float ov = oo / ll;
          p.obuf[static_cast<size_t>(m) * dq + hq * DH + dd] = ov;
          if (p.so.xs) store_split(p.so, m, hq * DH + dd, ov);
        }
      } else {
        float* r = p.ws + ((static_cast<size_t>(hk) * n_chunks + c) * p.qv_cap + qv) * WSTR;
        r[dd] = oo;
        if (dd == 0) { r[DH] = mm; r[DH + 1] = ll; }
      }
    }
    consumer_sync();  // wsm is reused by the next query tile
  }
  if (n_chunks > 1) {
    // the last CTA of this kv-head to arrive merges all chunks in chunk order
    __threadfence();
    consumer_sync();
    if (tid == 0) {
      const int old = atomicAdd(&p.counters[hk], 1);
      *flag_s = (old == n_chunks - 1);
    }
    consumer_sync();
    if (*flag_s) {
      __threadfence();
      for (int idx = tid; idx < qv_tot * DH; idx += kConsumerThreads) {
        const int qv = idx / DH, dd = idx % DH;
        const float* base = p.ws + (static_cast<size_t>(hk) * n_chunks * p.qv_cap + qv) * WSTR;
        const size_t cstride = static_cast<size_t>(p.qv_cap) * WSTR;
        float mm = -INFINITY;
        for (int cc = 0; cc < n_chunks; ++cc) mm = fmaxf(mm, __ldcg(base + cc * cstride + DH));
        float ll = 0.f, oo = 0.f;
        for (int cc = 0; cc < n_chunks; ++cc) {
          const float* r = base + cc * cstride;
          const float mc = __ldcg(r + DH);
          const float cw = (mc == -INFINITY) ? 0.f : expf(mc - mm);
          ll += __ldcg(r + DH + 1) * cw;
          oo += __ldcg(r + dd) * cw;
        }
        const int m = qv / grp, hq = hk * grp + qv % grp;
        {
          const float ov = oo / ll;
          p.obuf[static_cast<size_t>(m) * dq + hq * DH + dd] = ov;
          if (p.so.xs) store_split(p.so, m, hq * DH + dd, ov);
        }
      }
      if (tid == 0) p.counters[hk] = 0;
    }
  }
  trace_end(p.trace);
}

}  // namespace dvt

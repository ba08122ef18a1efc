// attention_mma.cuh -- tensor-core tree attention for bf16 caches (S2 append + S3,
// PAPER.md:94): same contract as k_tree_attention (attention.cuh), same grid
// (n_chunks, Hkv), same partial / merge protocol, but the per-position work runs on
// mma.sync.m16n8k16 the way flash-decoding kernels do:
//
//   S = Q K^T : A = 16 query vectors (rows of the level x q-heads of the GQA group,
//               zero padded) x head_dim, B = K rows as stored ([position][d] is the
//               "col" operand as it is);
//   O += P V  : A = P (the S accumulators re-used as the A fragment), B = V rows
//               through ldmatrix.trans.
// Neither the fp32 queries nor the probabilities are rounded to bf16: both are split
// into a bf16 head and a bf16 remainder (two mma per tile, 16 mantissa bits), the
// softmax statistics and the accumulators are fp32.
//
// CTA = 4 consumer warps + 2 producer warps, <= 2 CTAs per SM. The producers copy
// blocks of 64 positions (K and V rows, 16-byte cp.async with an XOR swizzle of the
// 16-byte chunk index by position & 7, which makes every ldmatrix conflict free; a
// 1-D bulk copy cannot swizzle) into a 3-deep ring signalled by mbarriers; each
// consumer warp owns one 16-position tile of every block and its own online-softmax
// state; warps, then chunks, are merged in fixed order (deterministic).
#pragma once
#include <cuda_bf16.h>

#include "attention.cuh"
#include "gemv_mma.cuh"
#include "ptx.cuh"
#include "state.cuh"

namespace dvt {


constexpr int kAmWarps = 4;                       // consumer warps
constexpr int kAmConsumers = kAmWarps * 32;       // 128
constexpr int kAmProducers = 64;                  // two producer warps
constexpr int kAmThreads = kAmConsumers + kAmProducers;
constexpr int kAmBlockPos = 64;                   // positions per ring block
constexpr int kAmStages = 3;
constexpr int kAmQRows = 16;                      // query vectors per pass

__device__ __forceinline__ void am_consumer_sync() {
  asm volatile("bar.sync 2, %0;" ::"n"(kAmConsumers) : "memory");
}

__device__ __forceinline__ void ldsm_x4_trans(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(addr)
               : "memory");
}

// 16-byte async copy global -> shared; src_bytes = 0 writes zeros without reading.
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, uint32_t src_bytes, uint64_t policy) {
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2, %3;" ::"r"(dst), "l"(src), "r"(src_bytes),
               "l"(policy)
               : "memory");
}
// arrives on the mbarrier once all prior cp.async of this thread have landed
__device__ __forceinline__ void cp_async_arrive(uint64_t* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// ---- thread-block cluster: the chunks of one kv-head merge through distributed shared memory
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
  return r;
}
// all threads of all CTAs of the cluster; release / acquire over shared::cluster
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ float ld_dsmem_f32(uint32_t local_addr, uint32_t rank) {
  uint32_t ra;
  float v;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(local_addr), "r"(rank));
  asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(ra) : "memory");
  return v;
}

// byte offset of 16-byte chunk `ch` of row `r` in a swizzled [rows][ROWB] tile
template <int ROWB>
__device__ __forceinline__ uint32_t am_swz(int r, int ch) {
  return static_cast<uint32_t>(r) * ROWB + static_cast<uint32_t>((ch ^ (r & 7)) << 4);
}

constexpr size_t am_smem_bytes(int DH, int QT = 1) {
  // q hi + lo tiles, ring of (K, V) blocks (the merge scratch aliases it), barriers
  return static_cast<size_t>(2 * QT * kAmQRows * DH * 2) + static_cast<size_t>(kAmStages) * 2 * kAmBlockPos * DH * 2 + 128;
}

// QT = 1: one tile of 16 query vectors per pass over the CTA's positions, the four consumer warps split the 64
// positions of a block (tree levels of a few rows: latency matters, every warp works on every block).
// QT = 2 (17 ... 32 query vectors): 32 per pass, warp w owns query tile w & 1 and the position half w >> 1 of every
// block; the two halves of a tile are merged like the four warps of QT = 1. One pass over the cache instead of two.
// QT = 4 ("wide": levels of many rows, level-0 batches of dovetail_draft_prefill): 64 query vectors per pass,
// consumer warp w owns query tile w and walks all 64 positions of every block with its own online-softmax state,
// the flash-attention arrangement -- the cache is streamed once per 64 query vectors instead of once per 16, and
// no merge over the warps is needed.
template <int DH, int QT>
__global__ void __launch_bounds__(kAmThreads, QT <= 2 ? 2 : 1) k_tree_attention_mma(const AttnParams p) {
  using WT = __nv_bfloat16;
  constexpr int ROWB = DH * 2;            // bytes of one K (or V) row
  constexpr int CPR = ROWB / 16;          // 16-byte chunks per row
  constexpr int KS = DH / 16;             // k-steps of S = Q K^T
  constexpr int DN = DH / 8;              // 8-wide d tiles of O
  constexpr int PB = kAmBlockPos;
  constexpr int BLK_BYTES = 2 * PB * ROWB;
  constexpr int HALF = DH / 2;
  constexpr int WSTR = DH + 4;            // partial record: o[DH], m, l (rows 16-byte aligned: the merges read float4)
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int QROWS = QT * kAmQRows;    // query vectors per pass
  uint8_t* q_hi = smem;                   // [QROWS][ROWB] swizzled bf16 heads of the rotated, scaled queries
  uint8_t* q_lo = q_hi + QROWS * ROWB;    // remainders
  uint8_t* ring = q_lo + QROWS * ROWB;
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + kAmStages * BLK_BYTES);
  uint64_t* empty = full + 4;
  uint64_t* tailbar = empty + 4;
  uint64_t* gatebar = tailbar + 1;  // a consumer has passed griddepcontrol.wait
  int* flag_s = reinterpret_cast<int*>(gatebar + 1);
  // The warp-merge scratch and this CTA's record alias the ring: when they are written every block of
  // the pass has been consumed, and the producers resume only after the pass's second cluster barrier.
  float* wsm = reinterpret_cast<float*>(ring);  // [warps][QR][WSTR]

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int c = blockIdx.x, hk = blockIdx.y, n_chunks = gridDim.x;
  const int grp = p.Hq / p.Hkv;
  const int qv_tot = p.M * grp;
  const int n_pass = (qv_tot + QROWS - 1) / QROWS;
  const int QR = min(QROWS, qv_tot);  // rows of the warp-merge scratch
  // [QR][WSTR] this CTA's record, read by the cluster ranks (wide: written by the warps directly, no warp merge)
  constexpr int NPART = QT == 1 ? kAmWarps : (QT == 2 ? 2 : 1);  // partial states per query vector inside the CTA
  float* crec = QT == 4 ? wsm : wsm + static_cast<size_t>(NPART) * QR * WSTR;
  // chunks [group * CS, (group + 1) * CS) of a kv-head form a cluster (CS = 1 without the launch attribute)
  const int CS = static_cast<int>(cluster_nctarank()), crank = static_cast<int>(cluster_ctarank());
  const int n_groups = n_chunks / CS, group = c / CS;
  const int dq = p.Hq * DH, dkv = p.Hkv * DH, ldq = dq + 2 * dkv;

  if (tid == 0) {
    for (int s = 0; s < kAmStages; ++s) {
      mbar_init(&full[s], kAmProducers);
      mbar_init(&empty[s], kAmWarps);
    }
    mbar_init(tailbar, kAmConsumers);
    mbar_init(gatebar, 1);
    mbar_fence_init();
  }
  __syncthreads();
  pdl_launch_dependents();
  trace_begin(p.trace);

  const int Lbase = p.Lbase, cap = p.cap;
  const WT* kc = static_cast<const WT*>(p.kc) + (static_cast<size_t>(p.layer) * p.Hkv + hk) * cap * DH;
  const WT* vc = static_cast<const WT*>(p.vc) + (static_cast<size_t>(p.layer) * p.Hkv + hk) * cap * DH;
  // blocks of PB positions are dealt to the chunks; the spare ones go to the LAST chunks because
  // chunk 0 also attends the new region
  const int n_blocks = (Lbase + PB - 1) / PB, bbase = n_blocks / n_chunks, brem = n_blocks % n_chunks;
  const int b_begin = c * bbase + max(0, c - (n_chunks - brem));
  const int b_end = b_begin + bbase + (c >= n_chunks - brem ? 1 : 0);
  const int p_begin = min(Lbase, b_begin * PB), p_end = min(Lbase, b_end * PB);
  const int n_blk = b_end - b_begin;
  const int n_tail = c == 0 ? (p.new_cnt + PB - 1) / PB : 0;  // the new region, chunk 0 only
  const int nb = n_blk + n_tail;

  if (warp >= kAmWarps) {
    // ---------------- producers ---------------------------------------------------
    const int ptid = tid - kAmConsumers;
    // the prefix is re-read by every level of the step and by the next steps (4 layers x 21 MB on the 13B shape
    // fit the 126 MB L2 next to the weight stream, which is evict_first): keep it
    const uint64_t pol = l2_policy_evict_last();
    // Invariant: before griddepcontrol.wait only cache rows below p.Lsafe -- the
    // prefix committed before this step, which no kernel of the step writes -- may be read. Rows
    // [Lsafe, Lbase) of a tree level were appended by this step's level-0 kernels, several launches
    // back; programmatic dependent launch orders a kernel only against its immediate predecessor and
    // only after the wait, so blocks that reach past Lsafe are gated on a consumer having waited.
    int slot = 0, round = 0;
    bool tail_ready = false, gate_open = false;
    for (int pass = 0; pass < n_pass; ++pass) {
      for (int b = 0; b < nb; ++b) {
        int pos0, cnt;
        if (b < n_blk) {
          pos0 = p_begin + b * PB;
          cnt = min(PB, p_end - pos0);
          if (!gate_open && pos0 + cnt > p.Lsafe) {
            mbar_wait(gatebar, 0);
            gate_open = true;
          }
        } else {
          if (!tail_ready) {  // this level's rows: appended by this CTA's consumers, or (fused S2) by the QKV kernel
            if (p.qs == nullptr) mbar_wait(tailbar, 0);
            else if (!gate_open) { mbar_wait(gatebar, 0); gate_open = true; }
            tail_ready = true;
          }
          pos0 = Lbase + (b - n_blk) * PB;
          cnt = min(PB, p.new_cnt - (b - n_blk) * PB);
        }
        if (round > 0) mbar_wait(&empty[slot], (round & 1) ^ 1);
        const uint32_t kdst = smem_u32(ring) + static_cast<uint32_t>(slot) * BLK_BYTES, vdst = kdst + PB * ROWB;
        const uint8_t* ksrc = reinterpret_cast<const uint8_t*>(kc + static_cast<size_t>(pos0) * DH);
        const uint8_t* vsrc = reinterpret_cast<const uint8_t*>(vc + static_cast<size_t>(pos0) * DH);
#pragma unroll 4
        for (int i = ptid; i < PB * CPR; i += kAmProducers) {
          const int r = i / CPR, ch = i % CPR;
          const bool valid = r < cnt;  // rows past the end are zero filled (0 * stale NaN would poison P V)
          const size_t so = valid ? static_cast<size_t>(r) * ROWB + ch * 16 : 0;
          const uint32_t d = am_swz<ROWB>(r, ch);
          cp_async16(kdst + d, ksrc + so, valid ? 16u : 0u, pol);
          cp_async16(vdst + d, vsrc + so, valid ? 16u : 0u, pol);
        }
        cp_async_arrive(&full[slot]);
        if (++slot == kAmStages) { slot = 0; ++round; }
      }
      cluster_sync_all();  // the two cluster barriers of the pass (see the consumers)
      cluster_sync_all();
    }
    return;
  }

  // ---------------- consumers -----------------------------------------------------
  pdl_wait();  // q/k/v of this level and the row tables are visible from here on
  if (tid == 0) mbar_arrive(gatebar);
  const RowTables* rows = p.rows;
  const int g = lane >> 2, tq = lane & 3;
  const float scale = 1.0f / sqrtf(static_cast<float>(DH));

  // S2: append this level's K/V rows of kv-head hk (chunk 0 only). K is rotated (half-split
  // pairing (i, i + dh/2), reading A3) and both are rounded to the cache dtype, as the oracle
  // stores them; the new region is then attended from the cache like the prefix.
  if (c == 0 && p.qs == nullptr) {
    WT* kcw = const_cast<WT*>(kc);
    WT* vcw = const_cast<WT*>(vc);
    for (int idx = tid; idx < p.M * HALF; idx += kAmConsumers) {
      const int m = idx / HALF, i = idx % HALF;
      const float* kr = p.qkv + static_cast<size_t>(m) * ldq + dq + hk * DH;
      const float2 cs = p.rope[static_cast<size_t>(p.rope_row0 + (p.rope_per_row ? m : 0)) * HALF + i];
      const float a = kr[i], b = kr[i + HALF];
      WT* dst = kcw + static_cast<size_t>(Lbase + rows->slot[m]) * DH;
      store_cache(dst + i, a * cs.x - b * cs.y);
      store_cache(dst + i + HALF, b * cs.x + a * cs.y);
    }
    for (int idx = tid; idx < p.M * DH; idx += kAmConsumers) {
      const int m = idx / DH, i = idx % DH;
      const float* vr = p.qkv + static_cast<size_t>(m) * ldq + dq + dkv + hk * DH;
      store_cache(vcw + static_cast<size_t>(Lbase + rows->slot[m]) * DH + i, vr[i]);
    }
    __threadfence();
    mbar_arrive(tailbar);
  }

  int slot = 0, round = 0;
  for (int pass = 0; pass < n_pass; ++pass) {
    const int qv0 = pass * QROWS;
    const int nq = min(QROWS, qv_tot - qv0);  // query vectors of this pass
    // ---- rotated, scaled queries -> bf16 head + remainder tiles ------------------
    if (p.qs != nullptr) {  // prepared by the QKV projection's epilogue: 16-byte copies into the swizzled tiles
      constexpr int NQ = kAmQRows * CPR * 2 / kAmConsumers;  // copies per thread and round, all loads issued before the stores
      static_assert(kAmQRows * CPR * 2 % kAmConsumers == 0, "query tile copies must divide among the consumers");
#pragma unroll 1
      for (int rd = 0; rd < QT; ++rd) {  // one round per 16-row tile
        uint4 v[NQ];
#pragma unroll
        for (int i = 0; i < NQ; ++i) {
          const int idx = tid + i * kAmConsumers;
          const int pl = idx / (kAmQRows * CPR), rem = idx - pl * (kAmQRows * CPR);
          const int r = rd * kAmQRows + rem / CPR, ch = rem % CPR;
          v[i] = make_uint4(0u, 0u, 0u, 0u);
          if (r < nq) {
            const int qv = qv0 + r, m = qv / grp, hq = hk * grp + qv % grp;
            v[i] = __ldcg(reinterpret_cast<const uint4*>(p.qs + (static_cast<size_t>(pl) * kMaxRows + m) * dq + hq * DH) + ch);
          }
        }
#pragma unroll
        for (int i = 0; i < NQ; ++i) {
          const int idx = tid + i * kAmConsumers;
          const int pl = idx / (kAmQRows * CPR), rem = idx - pl * (kAmQRows * CPR);
          const int r = rd * kAmQRows + rem / CPR, ch = rem % CPR;
          *reinterpret_cast<uint4*>((pl ? q_lo : q_hi) + am_swz<ROWB>(r, ch)) = v[i];
        }
      }
    } else
    for (int idx = tid; idx < QROWS * HALF; idx += kAmConsumers) {
      const int r = idx / HALF, i = idx % HALF;
      float x0 = 0.f, x1 = 0.f;
      if (r < nq) {
        const int qv = qv0 + r, m = qv / grp, hq = hk * grp + qv % grp;
        const float* qr = p.qkv + static_cast<size_t>(m) * ldq + hq * DH;
        const float2 cs = p.rope[static_cast<size_t>(p.rope_row0 + (p.rope_per_row ? m : 0)) * HALF + i];
        const float a = qr[i], b = qr[i + HALF];
        x0 = (a * cs.x - b * cs.y) * scale;
        x1 = (b * cs.x + a * cs.y) * scale;
      }
      const float xs[2] = {x0, x1};
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int d = i + h * HALF;
        const uint32_t off = am_swz<ROWB>(r, d >> 3) + (d & 7) * 2;
        const uint16_t hi = f32_to_bf16_rn(xs[h]);
        const float rem = xs[h] - __uint_as_float(static_cast<uint32_t>(hi) << 16);
        *reinterpret_cast<uint16_t*>(q_hi + off) = hi;
        *reinterpret_cast<uint16_t*>(q_lo + off) = f32_to_bf16_rn(rem);
      }
    }
    am_consumer_sync();

    // rows of this thread's accumulators: g and g + 8; their draft rows for the tail masks
    int mrow[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int r = (QT == 1 ? 0 : (QT == 2 ? (warp & 1) : warp) * kAmQRows) + g + 8 * h;  // QT > 1: this warp's own query tile
      mrow[h] = r < nq ? (qv0 + r) / grp : -1;
    }
    float mrun[2] = {-INFINITY, -INFINITY}, lrun[2] = {0.f, 0.f};
    float o[DN][4];
#pragma unroll
    for (int t = 0; t < DN; ++t)
#pragma unroll
      for (int e = 0; e < 4; ++e) o[t][e] = 0.f;

    // per-lane ldmatrix row / chunk pieces
    const int a_row = (lane & 7) + ((lane >> 3) & 1) * 8, a_ch = lane >> 4;          // A: q tiles
    const int k_row = (lane & 7) + (lane >> 4) * 8, k_ch = (lane >> 3) & 1;          // B of S: K rows
    const int v_row = (lane & 7) + ((lane >> 3) & 1) * 8, v_ch = lane >> 4;          // B of PV: V rows (.trans)

    for (int b = 0; b < nb; ++b) {
      const bool tail = b >= n_blk;
      const int cnt = tail ? min(PB, p.new_cnt - (b - n_blk) * PB) : min(PB, p_end - (p_begin + b * PB));
      mbar_wait(&full[slot], round & 1);
      if constexpr (QT == 1) {
      const int t0 = warp * 16;  // this warp's tile of the block
        if (t0 < cnt) {
          const uint32_t kb = smem_u32(ring) + static_cast<uint32_t>(slot) * BLK_BYTES, vb = kb + PB * ROWB;
          // four independent accumulation chains (head / remainder x two position tiles): a dependent
          // HMMA chain of 16 per tile was the longest latency of the block
          float s[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
          float sl[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
  #pragma unroll
          for (int ks = 0; ks < KS; ++ks) {
            uint32_t ah[4], al[4], kf[4];
            ldsm_x4(ah, smem_u32(q_hi) + am_swz<ROWB>(a_row, ks * 2 + a_ch));
            ldsm_x4(al, smem_u32(q_lo) + am_swz<ROWB>(a_row, ks * 2 + a_ch));
            ldsm_x4(kf, kb + am_swz<ROWB>(t0 + k_row, ks * 2 + k_ch));
            mma_bf16_16816(s[0], ah, kf[0], kf[1]);
            mma_bf16_16816(sl[0], al, kf[0], kf[1]);
            mma_bf16_16816(s[1], ah, kf[2], kf[3]);
            mma_bf16_16816(sl[1], al, kf[2], kf[3]);
          }
  #pragma unroll
          for (int nt = 0; nt < 2; ++nt)
  #pragma unroll
            for (int e = 0; e < 4; ++e) s[nt][e] += sl[nt][e];
          // masks: positions past the block's end, padded query rows, and (new region) the
          // ancestor mask of the row
          // (a full prefix block needs none: padded query rows are zero vectors, their scores are 0 and
          // their results are never read)
          float mx[2] = {-INFINITY, -INFINITY};
          const bool need_mask = tail || cnt < PB;  // uniform over the CTA
  #pragma unroll
          for (int nt = 0; nt < 2; ++nt)
  #pragma unroll
            for (int e = 0; e < 4; ++e) {
              const int h = e >> 1;
              if (need_mask) {
                const int pos = t0 + nt * 8 + 2 * tq + (e & 1);
                bool ok = pos < cnt && mrow[h] >= 0;
                if (ok && tail) {
                  const int j = (b - n_blk) * PB + pos;
                  ok = (rows->mask[mrow[h]][j >> 5] >> (j & 31)) & 1u;
                }
                s[nt][e] = ok ? s[nt][e] : -INFINITY;
              }
              mx[h] = fmaxf(mx[h], s[nt][e]);
            }
          float corr[2];
  #pragma unroll
          for (int h = 0; h < 2; ++h) {
            mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 1));
            mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 2));
            const float mn = fmaxf(mrun[h], mx[h]);
            corr[h] = (mrun[h] == -INFINITY) ? 0.f : __expf(mrun[h] - mn);
            mrun[h] = mn;
            lrun[h] *= corr[h];
          }
          uint32_t ph[4], pl[4];  // P as the A fragment of P V: head and remainder
  #pragma unroll
          for (int nt = 0; nt < 2; ++nt)
  #pragma unroll
            for (int h = 0; h < 2; ++h) {
              // ex2.approx of the difference to the running maximum (<= 0): relative error ~1e-6
              const float p0 = (s[nt][2 * h] == -INFINITY) ? 0.f : __expf(s[nt][2 * h] - mrun[h]);
              const float p1 = (s[nt][2 * h + 1] == -INFINITY) ? 0.f : __expf(s[nt][2 * h + 1] - mrun[h]);
              lrun[h] += p0 + p1;
              const uint32_t hi = pack_bf16x2_rn(p0, p1);
              const float2 hf = bf16x2_to_f32x2(hi);
              ph[nt * 2 + h] = hi;
              pl[nt * 2 + h] = pack_bf16x2_rn(p0 - hf.x, p1 - hf.y);
            }
          if (__any_sync(0xffffffffu, corr[0] != 1.f || corr[1] != 1.f)) {  // the maximum rarely moves after the first tiles
  #pragma unroll
            for (int t = 0; t < DN; ++t) {
              o[t][0] *= corr[0];
              o[t][1] *= corr[0];
              o[t][2] *= corr[1];
              o[t][3] *= corr[1];
            }
          }
  #pragma unroll
          for (int t = 0; t < DN; t += 2) {
            uint32_t vf[4];
            ldsm_x4_trans(vf, vb + am_swz<ROWB>(t0 + v_row, t + v_ch));
            mma_bf16_16816(o[t], ph, vf[0], vf[1]);
            mma_bf16_16816(o[t], pl, vf[0], vf[1]);
            mma_bf16_16816(o[t + 1], ph, vf[2], vf[3]);
            mma_bf16_16816(o[t + 1], pl, vf[2], vf[3]);
          }
        }
      } else if ((QT == 2 ? (warp & 1) : warp) * kAmQRows < nq) {
        // ---- QT = 4: this warp's 16 query vectors against all 64 positions of the block; QT = 2: against its half
        constexpr int NJ = QT == 2 ? 2 : 4;                  // 16-position tiles of the block this warp walks
        const int J0 = QT == 2 ? (warp >> 1) * 2 : 0;
        const int qtile = QT == 2 ? (warp & 1) : warp;
        const uint32_t kb = smem_u32(ring) + static_cast<uint32_t>(slot) * BLK_BYTES, vb = kb + PB * ROWB;
        const int q_row = qtile * kAmQRows + a_row;
        float s[2 * NJ][4];  // independent chains: head and remainder products share an accumulator
#pragma unroll
        for (int nt = 0; nt < 2 * NJ; ++nt)
#pragma unroll
          for (int e = 0; e < 4; ++e) s[nt][e] = 0.f;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
          uint32_t ah[4], al[4];
          ldsm_x4(ah, smem_u32(q_hi) + am_swz<ROWB>(q_row, ks * 2 + a_ch));
          ldsm_x4(al, smem_u32(q_lo) + am_swz<ROWB>(q_row, ks * 2 + a_ch));
#pragma unroll
          for (int j = 0; j < NJ; ++j) {
            uint32_t kf[4];
            ldsm_x4(kf, kb + am_swz<ROWB>((J0 + j) * 16 + k_row, ks * 2 + k_ch));
            mma_bf16_16816(s[2 * j], ah, kf[0], kf[1]);
            mma_bf16_16816(s[2 * j + 1], ah, kf[2], kf[3]);
            mma_bf16_16816(s[2 * j], al, kf[0], kf[1]);
            mma_bf16_16816(s[2 * j + 1], al, kf[2], kf[3]);
          }
        }
        float mx[2] = {-INFINITY, -INFINITY};
        const bool need_mask = tail || cnt < PB;  // uniform over the CTA
#pragma unroll
        for (int nt = 0; nt < 2 * NJ; ++nt)
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int h = e >> 1;
            if (need_mask) {
              const int pos = J0 * 16 + nt * 8 + 2 * tq + (e & 1);
              bool ok = pos < cnt && mrow[h] >= 0;
              if (ok && tail) {
                const int j = (b - n_blk) * PB + pos;
                ok = (rows->mask[mrow[h]][j >> 5] >> (j & 31)) & 1u;
              }
              s[nt][e] = ok ? s[nt][e] : -INFINITY;
            }
            mx[h] = fmaxf(mx[h], s[nt][e]);
          }
        float corr[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 1));
          mx[h] = fmaxf(mx[h], __shfl_xor_sync(0xffffffffu, mx[h], 2));
          const float mn = fmaxf(mrun[h], mx[h]);
          corr[h] = (mrun[h] == -INFINITY) ? 0.f : __expf(mrun[h] - mn);
          mrun[h] = mn;
          lrun[h] *= corr[h];
        }
        if (__any_sync(0xffffffffu, corr[0] != 1.f || corr[1] != 1.f)) {
#pragma unroll
          for (int t = 0; t < DN; ++t) {
            o[t][0] *= corr[0];
            o[t][1] *= corr[0];
            o[t][2] *= corr[1];
            o[t][3] *= corr[1];
          }
        }
#pragma unroll
        for (int j = 0; j < NJ; ++j) {  // 16 positions per step of P V
          uint32_t ph[4], pl[4];
#pragma unroll
          for (int n2 = 0; n2 < 2; ++n2)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const int nt = 2 * j + n2;
              const float p0 = (s[nt][2 * h] == -INFINITY || mrun[h] == -INFINITY) ? 0.f : __expf(s[nt][2 * h] - mrun[h]);
              const float p1 = (s[nt][2 * h + 1] == -INFINITY || mrun[h] == -INFINITY) ? 0.f : __expf(s[nt][2 * h + 1] - mrun[h]);
              lrun[h] += p0 + p1;
              const uint32_t hi = pack_bf16x2_rn(p0, p1);
              const float2 hf = bf16x2_to_f32x2(hi);
              ph[n2 * 2 + h] = hi;
              pl[n2 * 2 + h] = pack_bf16x2_rn(p0 - hf.x, p1 - hf.y);
            }
#pragma unroll
          for (int t = 0; t < DN; t += 2) {
            uint32_t vf[4];
            ldsm_x4_trans(vf, vb + am_swz<ROWB>((J0 + j) * 16 + v_row, t + v_ch));
            mma_bf16_16816(o[t], ph, vf[0], vf[1]);
            mma_bf16_16816(o[t], pl, vf[0], vf[1]);
            mma_bf16_16816(o[t + 1], ph, vf[2], vf[3]);
            mma_bf16_16816(o[t + 1], pl, vf[2], vf[3]);
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[slot]);
      if (++slot == kAmStages) { slot = 0; ++round; }
    }
    am_consumer_sync();  // every warp is done with the ring: the merge scratch aliases it

    if constexpr (QT != 4) {
    // ---- merge the partial states of a query vector (QT = 1: four warps, QT = 2: two position halves; fixed order)
      const int part = QT == 1 ? warp : (warp >> 1), rbase = QT == 1 ? 0 : (warp & 1) * kAmQRows;
  #pragma unroll
      for (int h = 0; h < 2; ++h) {
        lrun[h] += __shfl_xor_sync(0xffffffffu, lrun[h], 1);
        lrun[h] += __shfl_xor_sync(0xffffffffu, lrun[h], 2);
        const int r = rbase + g + 8 * h;
        if (r < nq) {
          float* w = wsm + (static_cast<size_t>(part) * QR + r) * WSTR;
  #pragma unroll
          for (int t = 0; t < DN; ++t)
            *reinterpret_cast<float2*>(w + t * 8 + 2 * tq) = make_float2(o[t][2 * h], o[t][2 * h + 1]);
          if (tq == 0) { w[DH] = mrun[h]; w[DH + 1] = lrun[h]; }
        }
      }
      am_consumer_sync();
      for (int idx = tid; idx < nq * (DH / 4); idx += kAmConsumers) {  // four d per thread: one set of weights per float4
        const int r = idx / (DH / 4), dd = (idx % (DH / 4)) * 4;
        float mm = -INFINITY;
#pragma unroll
        for (int w = 0; w < NPART; ++w) mm = fmaxf(mm, wsm[(w * QR + r) * WSTR + DH]);
        float ll = 0.f;
        float4 oo = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int w = 0; w < NPART; ++w) {
          const float* rr = wsm + (w * QR + r) * WSTR;
          const float cw = (rr[DH] == -INFINITY) ? 0.f : expf(rr[DH] - mm);
          const float4 ov = *reinterpret_cast<const float4*>(rr + dd);
          ll += rr[DH + 1] * cw;
          oo.x += ov.x * cw;
          oo.y += ov.y * cw;
          oo.z += ov.z * cw;
          oo.w += ov.w * cw;
        }
        float* rr = crec + static_cast<size_t>(r) * WSTR;
        *reinterpret_cast<float4*>(rr + dd) = oo;
        if (dd == 0) { rr[DH] = mm; rr[DH + 1] = ll; }
      }
    } else {
      // wide: every warp owns its query vectors; its state is this CTA's record of them
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        lrun[h] += __shfl_xor_sync(0xffffffffu, lrun[h], 1);
        lrun[h] += __shfl_xor_sync(0xffffffffu, lrun[h], 2);
        const int r = warp * kAmQRows + g + 8 * h;
        if (r < nq) {
          float* w = crec + static_cast<size_t>(r) * WSTR;
#pragma unroll
          for (int t = 0; t < DN; ++t)
            *reinterpret_cast<float2*>(w + t * 8 + 2 * tq) = make_float2(o[t][2 * h], o[t][2 * h + 1]);
          if (tq == 0) { w[DH] = mrun[h]; w[DH + 1] = lrun[h]; }
        }
      }
    }
    // ---- merge the chunks of the cluster in rank order through distributed shared memory ----
    cluster_sync_all();  // every CTA's record is complete and visible cluster-wide
    {  // every rank merges its slice of the head dimension (the work of the merge is spread over the cluster),
       // four consecutive d per thread and step: one 16-byte distributed-shared-memory load per rank
      const uint32_t crec_u = smem_u32(crec);
      const int slice4 = (DH / 4 + CS - 1) / CS;  // float4 groups per rank
      for (int idx = tid; idx < nq * slice4; idx += kAmConsumers) {
        const int r = idx / slice4, d4 = crank * slice4 + idx % slice4;
        if (d4 >= DH / 4) continue;
        const int dd = d4 * 4;
        const int qv = qv0 + r;
        const uint32_t ra = crec_u + static_cast<uint32_t>(r * WSTR) * 4;
        float mk[8], lk[8];
        float4 ok[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          mk[k] = -INFINITY;
          lk[k] = 0.f;
          ok[k] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (k < CS) {
            uint32_t rk;
            asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rk) : "r"(ra), "r"(static_cast<uint32_t>(k)));
            asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(mk[k]), "=f"(lk[k]) : "r"(rk + DH * 4) : "memory");
            asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];"
                         : "=f"(ok[k].x), "=f"(ok[k].y), "=f"(ok[k].z), "=f"(ok[k].w)
                         : "r"(rk + dd * 4)
                         : "memory");
          }
        }
        float mm = -INFINITY;
#pragma unroll
        for (int k = 0; k < 8; ++k) mm = fmaxf(mm, mk[k]);
        float ll = 0.f;
        float4 oo = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const float cw = (mk[k] == -INFINITY) ? 0.f : expf(mk[k] - mm);
          ll += lk[k] * cw;
          oo.x += ok[k].x * cw;
          oo.y += ok[k].y * cw;
          oo.z += ok[k].z * cw;
          oo.w += ok[k].w * cw;
        }
        if (n_groups == 1) {
          const int m = qv / grp, hq = hk * grp + qv % grp;
          const float4 ov = make_float4(oo.x / ll, oo.y / ll, oo.z / ll, oo.w / ll);
          *reinterpret_cast<float4*>(p.obuf + static_cast<size_t>(m) * dq + hq * DH + dd) = ov;
          if (p.so.xs) {
            store_split(p.so, m, hq * DH + dd, ov.x);
            store_split(p.so, m, hq * DH + dd + 1, ov.y);
            store_split(p.so, m, hq * DH + dd + 2, ov.z);
            store_split(p.so, m, hq * DH + dd + 3, ov.w);
          }
        } else {
          float* rr = p.ws + ((static_cast<size_t>(hk) * n_groups + group) * p.qv_cap + qv) * WSTR;
          *reinterpret_cast<float4*>(rr + dd) = oo;
          if (dd == 0) { rr[DH] = mm; rr[DH + 1] = ll; }
        }
      }
      if (n_groups > 1) __threadfence();  // the group's partial is complete in global memory before the leader counts in
    }
    cluster_sync_all();  // every rank has read the records: they (and the query tiles) may be reused
  }

  if (n_groups > 1 && crank == 0) {
    // the last cluster leader of this kv-head to arrive merges all groups in group order
    __threadfence();
    am_consumer_sync();
    if (tid == 0) {
      const int old = atomicAdd(&p.counters[hk], 1);
      *flag_s = (old == n_groups - 1);
    }
    am_consumer_sync();
    if (*flag_s) {
      __threadfence();
      // All blocks have been consumed, so the ring is free: the partial records are staged through
      // it with independent loads (one L2 round trip) instead of a chain of dependent ones.
      float* stg = reinterpret_cast<float*>(ring);
      const int rec = n_groups * WSTR;                       // floats of one query vector's records
      const int G = max(1, (kAmStages * BLK_BYTES / 4) / rec);  // query vectors per group
      for (int q0 = 0; q0 < qv_tot; q0 += G) {
        const int gq = min(G, qv_tot - q0);
        // 16-byte asynchronous copies straight into shared memory, all in flight at once, from a loop of a few
        // instructions: this code runs in one CTA per kv-head and launch, i.e. with a cold instruction cache --
        // an unrolled register-staged copy (8 loads per thread and round, 4 rounds) took 4.6 us, and unrolling it
        // further made it slower
        const int rec4 = rec / 4, w4n = WSTR / 4;  // 16-byte pieces per query vector / per record
        const uint32_t stg_u = smem_u32(stg);
        const uint64_t pol_m = l2_policy_evict_last();
        for (int e = tid; e < gq * rec4; e += kAmConsumers) {
          const int q = e / rec4, rem = e - q * rec4, cc = rem / w4n, w4 = rem - cc * w4n;
          cp_async16(stg_u + static_cast<uint32_t>(e) * 16u,
                     p.ws + ((static_cast<size_t>(hk) * n_groups + cc) * p.qv_cap + q0 + q) * WSTR + w4 * 4, 16u, pol_m);
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        am_consumer_sync();
        for (int idx = tid; idx < gq * (DH / 4); idx += kAmConsumers) {  // four d per thread: one set of weights per float4
          const int q = idx / (DH / 4), dd = (idx % (DH / 4)) * 4, qv = q0 + q;
          const float* base = stg + q * rec;
          float mm = -INFINITY;
          for (int cc = 0; cc < n_groups; ++cc) mm = fmaxf(mm, base[cc * WSTR + DH]);
          float ll = 0.f;
          float4 oo = make_float4(0.f, 0.f, 0.f, 0.f);
          for (int cc = 0; cc < n_groups; ++cc) {
            const float* rr = base + cc * WSTR;
            const float cw = (rr[DH] == -INFINITY) ? 0.f : expf(rr[DH] - mm);
            const float4 ov = *reinterpret_cast<const float4*>(rr + dd);
            ll += rr[DH + 1] * cw;
            oo.x += ov.x * cw;
            oo.y += ov.y * cw;
            oo.z += ov.z * cw;
            oo.w += ov.w * cw;
          }
          const int m = qv / grp, hq = hk * grp + qv % grp;
          const float4 ov = make_float4(oo.x / ll, oo.y / ll, oo.z / ll, oo.w / ll);
          *reinterpret_cast<float4*>(p.obuf + static_cast<size_t>(m) * dq + hq * DH + dd) = ov;
          if (p.so.xs) {
            store_split(p.so, m, hq * DH + dd, ov.x);
            store_split(p.so, m, hq * DH + dd + 1, ov.y);
            store_split(p.so, m, hq * DH + dd + 2, ov.z);
            store_split(p.so, m, hq * DH + dd + 3, ov.w);
          }
        }
        am_consumer_sync();
      }
      if (tid == 0) p.counters[hk] = 0;
    }
  }
  trace_end(p.trace);
}

}  // namespace dvt

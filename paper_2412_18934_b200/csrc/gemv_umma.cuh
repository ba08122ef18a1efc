// gemv_umma.cuh -- tcgen05 consumer for the weight-streaming GEMV at wide tree levels and level-0 catch-up
// rows (SURVEY.md 8a S1, S2, S4, S5, S6 at M = 9 ... 64 rows; 8(f4): PAPER.md:94 prompt rows).
//
//   Y[m, n] = sum_k X[m, k] * W[n, k]      m < M <= 64 draft rows, W bf16 row-major [N, K], K % 64 == 0
//
// Same work split, same activation planes, same fused epilogues as k_gemv_mma (gemv_mma.cuh); what changes is
// who multiplies. With mma.sync a warp keeps 16 weight rows x 8 columns per instruction in registers and the
// column tiles of a wide level multiply its instruction count and the re-reads of the activation operand
// (measured: 0.73 of the copy peak at M = 8, 0.45 at 16, 0.17 at 32). Here the 5th-generation tensor core reads
// both operands from shared memory and accumulates in tensor memory:
//   * swap-AB as before: the CTA's weight rows are the M side of tcgen05.mma (UMMA M = 64 or 128 tile rows), the
//     draft rows' split-bf16 planes are the N side (N = S * ceil8(M) columns, a multiple of 16), fp32
//     accumulators in TMEM, one column per (plane, draft row); the S planes of a row are added in the epilogue;
//   * both operands arrive by tensor-map bulk copies (cp.async.bulk.tensor, 128-byte swizzle): a box is 8 rows
//     x 64 k x nslab slabs, described by a 3-D map (k within slab, row, slab) so that one copy lands as nslab
//     swizzle atoms [slab][8 rows][128 B]. The CTA's rows stay row-exact: its virtual rows (gemv.cuh cta_rows /
//     locate_row) are grouped by the host into contiguous memory segments, each covered by 8-row boxes that
//     start at the segment's first row (a box may overhang into rows of a neighbour CTA: they are multiplied
//     and never read back; HBM still sees every row once, the overhang is an L2 hit);
//   * a stage of the ring = [weight groups][activation groups] of one K-chunk (64 * nslab elements); 8-row
//     groups are nslab KB apart (the descriptor's stride byte offset), a step of 16 k is +32 bytes;
//   * one thread issues the MMAs of a stage and commits them to the stage's "empty" barrier; after the last
//     chunk of a super-block (<= UMMA M tile rows) it commits to "tmem_full". Accumulators are double
//     buffered so that the next super-block's MMAs run under this one's drain;
//   * the 8 consumer warps only drain TMEM (tcgen05.ld, sum of the planes, 1 / rms) into the result buffer
//     and run the fused epilogue of gemv.cuh over it.
#pragma once
#include <cuda_bf16.h>

#include "attention_mma.cuh"  // thread-block cluster helpers (cluster rank, barrier, distributed shared memory loads)
#include "gemv.cuh"
#include "gemv_mma.cuh"
#include "ptx.cuh"
#include "state.cuh"
#include "umma.cuh"

namespace dvt {

constexpr int kUmmaMaxSb = 8;       // super-blocks per CTA (LM head of a 128k vocabulary: 867 rows)
constexpr int kUmmaMaxGroups = 16;  // 8-row groups per super-block: UMMA M = 128
constexpr int kUmmaMaxM = 64;
// warps: 8 consumers (TMEM drain + epilogue), weight producer, activation producer, MMA issuer
constexpr int kUmmaThreads = kConsumerThreads + 3 * 32;

// Built by the host for every CTA of a dealing (dovetail_draft.cu umma_tables): the 8-row boxes of each
// super-block. grp = (matrix j << 28) | first row of the box within w[j].
struct UmmaCtaTab {
  int32_t n_sb;
  int32_t n_grp[kUmmaMaxSb];
  int32_t grp[kUmmaMaxSb][kUmmaMaxGroups];
};

struct UmmaParams {
  GemvParams p;
  const CUtensorMap* wmap[2][3];  // weight matrices of each group: 3-D maps with nslab slabs per box
  const CUtensorMap* xmap[2];     // activation planes of each group (plane s = rows [s * x_cap, (s + 1) * x_cap))
  int32_t x_cap[2], x_row0[2];
  const UmmaCtaTab* tab[2];
  const uint16_t* vpos[2];        // [ctas][vpos_ld]: super-block * 128 + tile row of every virtual row
  int32_t vpos_ld;
  int32_t nslab, n_stages, stage_bytes;
  int32_t a_groups;               // 8-row groups reserved for the weight part of a stage; the activation part follows it,
                                  // so that what the tensor core reads past the CTA's last weight group (whole 64- /
                                  // 128-row tiles) is the activation part of the same stage, not foreign memory
  int32_t umma_m;                 // 64 or 128
  int32_t tmem_cols, acc_cols;    // allocation (2 buffers x k_split accumulators) and columns of one accumulator
  int32_t k_split;                // accumulators per super-block: K-chunk ch adds into accumulator ch % k_split. The tensor
                                  // core's fp32 accumulation rounds towards zero; chains of K / 16 steps into one
                                  // accumulator cost 3x the error of the mma.sync kernel's 8 shorter chains (measured),
                                  // so the chain is cut and the parts are added in fp32 by the epilogue
  int32_t ksplit;                 // 2: the CTAs of a cluster pair split K. Each multiplies the rows of BOTH over its half of K
                                  // (own rows = tile rows first, then the partner's), the partials of the partner's rows
                                  // go to an outbox the partner adds through distributed shared memory. A CTA with few rows
                                  // (O, down, DGF: 35 of a 64- / 128-row tile) then reads half of the activation operand
                                  // and issues half of the MMAs -- at 32-64 columns those, not HBM, bound it. 1: off
  int32_t cnt_pad;                // row stride of the result buffer res[m][v]
  int32_t ring_bytes;             // ring + the pad the tensor core may read past the last stage
};

__global__ void __launch_bounds__(kUmmaThreads, 1) k_gemv_umma(const __grid_constant__ UmmaParams cp) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~static_cast<uintptr_t>(1023));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const GemvParams& p = cp.p;
  const int NS = cp.n_stages, nslab = cp.nslab;
  const uint32_t GB = static_cast<uint32_t>(nslab) * 1024u;  // bytes of one 8-row group of a stage

  uint8_t* ring = smem;
  uint64_t* full_a = reinterpret_cast<uint64_t*>(smem + cp.ring_bytes);
  uint64_t* full_b = full_a + 8;
  uint64_t* empty = full_b + 8;
  uint64_t* tm_full = empty + 8;   // [2]
  uint64_t* tm_empty = tm_full + 2;  // [2]
  uint32_t* tslot = reinterpret_cast<uint32_t*>(tm_empty + 2);
  float* rstd_s = reinterpret_cast<float*>(tslot + 4);                // [kUmmaMaxM]
  int16_t* rmap = reinterpret_cast<int16_t*>(rstd_s + kUmmaMaxM);     // [kUmmaMaxSb][128]: virtual row of a tile row, or -1
  float* res = reinterpret_cast<float*>(rmap + kUmmaMaxSb * 128);     // [M][cnt_pad]
  float* outbox = res + static_cast<size_t>(p.M) * cp.cnt_pad;          // ksplit = 2: partials of the partner's rows, [M][cnt_pad]

  trace_begin(p.trace);
  if (tid < NS) {
    mbar_init(&full_a[tid], 1);
    mbar_init(&full_b[tid], 1);
    mbar_init(&empty[tid], 1);
  }
  if (tid >= 32 && tid < 34) {
    mbar_init(&tm_full[tid - 32], 1);
    mbar_init(&tm_empty[tid - 32], kConsumerWarps);
  }
  if (tid < 64) mbar_fence_init();
  if (warp == kConsumerWarps + 2) tmem_alloc(tslot, static_cast<uint32_t>(cp.tmem_cols));
  for (int i = tid; i < kUmmaMaxSb * 128; i += kUmmaThreads) rmap[i] = -1;
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_launch_dependents();
  const uint32_t tmem = *tslot;

  const CtaGeom q = cta_geom(p, blockIdx.x);
  const int c = q.c, gi = q.g;
  const GemvGroup& G = p.g[gi];
  const RowRange rr = q.rr;
  const int M = p.M, S = G.S, M8 = (M + 7) & ~7;
  const int nB = S * (M8 >> 3);             // activation groups really loaded
  const int N = (S * M8 + 15) & ~15;        // UMMA N
  const int n_chunks = p.K / (64 * nslab);
  const UmmaCtaTab* tab = c >= 0 ? cp.tab[gi] + c : nullptr;
  // K split over a cluster pair: this CTA's chunks, the partner's boxes appended to its own
  const bool ks2 = cp.ksplit == 2;
  const int krank = ks2 ? static_cast<int>(cluster_ctarank()) : 0;
  const int ch0 = ks2 && krank ? (n_chunks + 1) / 2 : 0, ch1 = ks2 && !krank ? (n_chunks + 1) / 2 : n_chunks;
  const UmmaCtaTab* ptab = ks2 ? cp.tab[gi] + (c ^ 1) : nullptr;
  const int png = ks2 ? ptab->n_grp[0] : 0;  // the partner's boxes (ksplit needs one super-block per CTA)

  if (warp == kConsumerWarps) {
    // ---------------- weight producer: one box per lane and stage; never waits for the previous kernel -------
    if (c >= 0) {
      const uint64_t pol = l2_policy_evict_first();
      const int n_sb = tab->n_sb;
      int slot = 0, round = 0;
      for (int sb = 0; sb < n_sb; ++sb) {
        const int ng0 = tab->n_grp[sb], ng = ng0 + png;
        const int gr = lane < ng ? (lane < ng0 ? tab->grp[sb][lane] : ptab->grp[0][lane - ng0]) : 0;
        const CUtensorMap* map = cp.wmap[gi][gr >> 28];
        const int row = gr & 0x0fffffff;
        for (int ch = ch0; ch < ch1; ++ch) {
          if (round > 0) mbar_wait(&empty[slot], (round & 1) ^ 1);
          if (lane == 0) mbar_arrive_expect_tx(&full_a[slot], static_cast<uint32_t>(ng) * GB);
          __syncwarp();
          if (lane < ng)
            tma_load_3d(ring + static_cast<size_t>(slot) * cp.stage_bytes + static_cast<uint32_t>(lane) * GB, map,
                        0, row, ch * nslab, &full_a[slot], pol);
          if (++slot == NS) { slot = 0; ++round; }
        }
      }
    }
  } else if (warp == kConsumerWarps + 1) {
    // ---------------- activation producer: planes left by the previous kernels (L2) ---------------------------
    pdl_wait();
    if (c >= 0) {
      const uint64_t pol = l2_policy_evict_last();
      const int n_sb = tab->n_sb;
      const CUtensorMap* map = cp.xmap[gi];
      const int mg = M8 >> 3;
      const int s = lane / mg, g8 = lane - s * mg;  // lane < nB <= 24: plane s, rows [8 g8, 8 g8 + 8) of the level
      const int row = s * cp.x_cap[gi] + cp.x_row0[gi] + p.m0 + g8 * 8;
      int slot = 0, round = 0;
      for (int sb = 0; sb < n_sb; ++sb) {
        for (int ch = ch0; ch < ch1; ++ch) {
          if (round > 0) mbar_wait(&empty[slot], (round & 1) ^ 1);
          if (lane == 0) mbar_arrive_expect_tx(&full_b[slot], static_cast<uint32_t>(nB) * GB);
          __syncwarp();
          if (lane < nB)
            tma_load_3d(ring + static_cast<size_t>(slot) * cp.stage_bytes + static_cast<uint32_t>(cp.a_groups + lane) * GB, map, 0, row,
                        ch * nslab, &full_b[slot], pol);
          if (++slot == NS) { slot = 0; ++round; }
        }
      }
    }
  } else if (warp == kConsumerWarps + 2) {
    // ---------------- MMA issuer ---------------------------------------------------------------------------
    if (c >= 0) {
      const int n_sb = tab->n_sb;
      const uint32_t idesc = umma_idesc_bf16(cp.umma_m, N);
      const uint32_t desc_hi = umma_desc_hi_sw128(GB);
      const uint32_t ring_u = smem_u32(ring);
      int slot = 0, round = 0;
      for (int sb = 0; sb < n_sb; ++sb) {
        const int buf = sb & 1;
        if (sb >= 2) mbar_wait(&tm_empty[buf], ((sb >> 1) & 1) ^ 1);  // drained by the consumers
        tc_fence_after();
        const uint32_t d_buf = tmem + static_cast<uint32_t>(buf * cp.k_split * cp.acc_cols);
        int ks = 0;
        for (int ch = ch0; ch < ch1; ++ch) {
          const uint32_t d_addr = d_buf + static_cast<uint32_t>(ks * cp.acc_cols);
          if (++ks == cp.k_split) ks = 0;
          mbar_wait(&full_a[slot], round & 1);
          mbar_wait(&full_b[slot], round & 1);
          tc_fence_after();
          if (elect_one()) {
            const uint32_t a_base = ring_u + static_cast<uint32_t>(slot) * cp.stage_bytes;
            uint32_t a_lo = umma_desc_lo(a_base), b_lo = umma_desc_lo(a_base + static_cast<uint32_t>(cp.a_groups) * GB);
            uint32_t accum = ch - ch0 >= cp.k_split ? 1u : 0u;
            for (int sl = 0; sl < nslab; ++sl) {  // one slab = 64 k = four MMAs
              umma_bf16(d_addr, a_lo, b_lo, desc_hi, idesc, accum);
              umma_bf16(d_addr, a_lo + 2, b_lo + 2, desc_hi, idesc, 1u);
              umma_bf16(d_addr, a_lo + 4, b_lo + 4, desc_hi, idesc, 1u);
              umma_bf16(d_addr, a_lo + 6, b_lo + 6, desc_hi, idesc, 1u);
              a_lo += 64;
              b_lo += 64;
              accum = 1u;
            }
            umma_commit(&empty[slot]);                       // the stage may be refilled once these MMAs have read it
            if (ch == ch1 - 1) umma_commit(&tm_full[buf]);  // the super-block's accumulators are complete
          }
          __syncwarp();
          if (++slot == NS) { slot = 0; ++round; }
        }
      }
    }
  } else {
    // ---------------- consumers: drain TMEM, fused epilogue --------------------------------------------------
    // tile row of every virtual row (static table) -> inverse map; nothing here depends on the previous kernel
    if (c >= 0) {
      const uint16_t* vp = cp.vpos[gi] + static_cast<size_t>(c) * cp.vpos_ld;
      for (int v = tid; v < rr.cnt; v += kConsumerThreads) rmap[vp[v]] = static_cast<int16_t>(v);
      if (ks2) {  // the partner's rows follow this CTA's boxes in the tile; marked by + 1024
        const uint16_t* vq = cp.vpos[gi] + static_cast<size_t>(c ^ 1) * cp.vpos_ld;
        const int pcnt = cta_rows(G, c ^ 1, p.ctas_per_group).cnt, shift = tab->n_grp[0] * 8;
        for (int v = tid; v < pcnt; v += kConsumerThreads) rmap[vq[v] + shift] = static_cast<int16_t>(1024 + v);
      }
    }
    pdl_wait();  // residual stream, [h1 || h2], sums of squares: written by the previous kernels
    if (c >= 0) {
      EpiRegs pre;
      epi_prefetch(p, G, rr, M, p.m0, true, pre);
      if (p.ssq_in) {
        // 1 / rms of each draft row from the producers' partial sums of squares, fixed order
        for (int m = warp; m < M; m += kConsumerWarps) {
          float t = 0.f;
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int cc = lane + 32 * j;
            if (cc < p.ssq_nct) t += __ldcg(p.ssq_in + static_cast<int64_t>(cc) * kMaxRows + p.m0 + m);
          }
          t = warp_sum(t);
          if (lane == 0) rstd_s[m] = 1.0f / sqrtf(t / static_cast<float>(p.K) + p.eps);
        }
      }
      consumer_sync();  // rmap, rstd_s
      const int n_sb = tab->n_sb;
      const int qd = warp & 3, half = warp >> 2;  // TMEM lane quarter of this warp; which half of the column chunks
      const bool row_ok = cp.umma_m == 128 || lane < 16;
      const int trow = cp.umma_m == 128 ? qd * 32 + lane : qd * 16 + lane;  // tile row held by this thread's TMEM lane
      const int cpad = cp.cnt_pad;
      for (int sb = 0; sb < n_sb; ++sb) {
        const int buf = sb & 1;
        mbar_wait(&tm_full[buf], (sb >> 1) & 1);
        tc_fence_after();
        const int v = row_ok ? rmap[sb * 128 + trow] : -1;
        const uint32_t t0 = tmem + (static_cast<uint32_t>(qd * 32) << 16) + static_cast<uint32_t>(buf * cp.k_split * cp.acc_cols);
        for (int c8 = half; c8 < (M8 >> 3); c8 += 2) {
          // sum over the K-split accumulators (fixed order), then over the planes of a row
          float acc[3][8];
#pragma unroll
          for (int s = 0; s < 3; ++s)
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[s][i] = 0.f;
          for (int ks = 0; ks < cp.k_split; ++ks) {
            uint32_t a0[8], a1[8] = {0, 0, 0, 0, 0, 0, 0, 0}, a2[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            const uint32_t tk = t0 + static_cast<uint32_t>(ks * cp.acc_cols + c8 * 8);
            tmem_ld8(tk, a0);
            if (S >= 2) tmem_ld8(tk + M8, a1);
            if (S == 3) tmem_ld8(tk + 2 * M8, a2);
            tmem_ld_wait();
            tmem_ld_use(a0);
            tmem_ld_use(a1);
            tmem_ld_use(a2);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              acc[0][i] += __uint_as_float(a0[i]);
              acc[1][i] += __uint_as_float(a1[i]);
              acc[2][i] += __uint_as_float(a2[i]);
            }
          }
          if (v >= 0) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const int m = c8 * 8 + i;
              if (m < M) {
                float t = acc[0][i];
                if (S >= 2) t += acc[1][i];
                if (S == 3) t += acc[2][i];
                if (p.ssq_in) t *= rstd_s[m];
                if (v >= 1024) outbox[m * cpad + (v - 1024)] = t;
                else res[m * cpad + v] = t;
              }
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&tm_empty[buf]);
      }
      if (ks2) {
        // both CTAs of the pair have drained: add the partner's partials of this CTA's rows (its outbox)
        cluster_sync_all();
        const uint32_t ob = smem_u32(outbox);
        for (int idx = tid; idx < M * rr.cnt; idx += kConsumerThreads) {
          const int m = idx / rr.cnt, v = idx - m * rr.cnt;
          res[m * cpad + v] += ld_dsmem_f32(ob + static_cast<uint32_t>(m * cpad + v) * 4u, static_cast<uint32_t>(krank ^ 1));
        }
      }
      consumer_sync();  // res complete
      gemv_epilogue(p, G, rr, [&](int v, int m) -> float& { return res[m * cpad + v]; }, M, p.m0, c, p.ctas_per_group, true, &pre);
    }
  }
  if (ks2) {
    if (warp >= kConsumerWarps) cluster_sync_all();  // the producer / MMA warps' share of the consumers' barrier above
    cluster_sync_all();                               // no CTA of the pair exits while its outbox may still be read
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kConsumerWarps + 2) {
    tc_fence_after();
    tmem_dealloc(tmem, static_cast<uint32_t>(cp.tmem_cols));
  }
  trace_end(p.trace);
}

}  // namespace dvt

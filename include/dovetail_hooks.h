/*
 * dovetail_hooks.h -- TEST AND MEASUREMENT HOOKS of libdovetail_draft.so.
 *
 * Not part of the product API of dovetail.h: nothing here changes what a draft
 * step computes; the hooks let the parity tests look at, and
 * teacher-force, the intermediate state of a step, and let bench.py attribute
 * device time to kernels. A handle with no hook set runs the plain step: the
 * launch sequence of dovetail_draft_step contains no hook code unless
 * dovetail_hooks_set() was called with a non-NULL argument (one flag test per
 * level on the host, nothing on the device).
 */
#ifndef DOVETAIL_HOOKS_H_
#define DOVETAIL_HOOKS_H_

#include "dovetail.h"

#ifdef __cplusplus
extern "C" {
#endif

/* All pointers are device pointers, borrowed until the next dovetail_hooks_set;
 * NULL disables the item.
 *
 * Taps (what the GPU computed):
 *   tap_logits [rows of the step, V] fp32: LM-head logits of every row whose LM head ran
 *              (step-row order: level-0 rows, then tree rows in cache-slot order).
 *   tap_hhat   [rows of the step, d] fp32: output hidden state of every row.
 *   tap_k/v    same dtype / layout / capacity as the KV cache: the K/V rows each level appended.
 *   tap_pool_token / tap_pool_cum [pool size]: token and cumulative log-probability of every
 *              candidate as the GPU computed them (before any forcing).
 *
 * Teacher forcing ("level-by-level with teacher forcing: after a logged tie,
 * continue the comparison from the oracle's frontier"). A step feeds every level with the
 * previous levels' results (parent hidden state, ancestors' K/V, candidate scores), so one
 * rounding-level difference or one flipped near-tie changes everything after it. With forcing,
 * after each level (and after its taps were taken) the step overwrites
 *   - the level's rows of its hidden-state buffer with force_hhat,
 *   - the K/V rows the level appended with the rows of force_k / force_v,
 *   - the level's candidates (pool token, cumulative score) with force_pool_token / _cum,
 * so that the next level (frontier, features, ancestors) starts from the caller's -- the
 * oracle's -- state, and every level's own arithmetic is compared in isolation. */
typedef struct {
  float* tap_logits;
  float* tap_hhat;
  void* tap_k;
  void* tap_v;
  int32_t* tap_pool_token;
  float* tap_pool_cum;
  const float* force_hhat;
  const void* force_k;
  const void* force_v;
  const int32_t* force_pool_token;
  const float* force_pool_cum;
} dovetail_hooks_t;

/* hooks == NULL (or all members NULL) removes every hook. */
int dovetail_hooks_set(dovetail_draft_t* h, const dovetail_hooks_t* hooks);

/* Per-kernel device time of the last step, for the roofline report.
 * dovetail_trace_enable(h, 1) makes every kernel of the following steps stamp %globaltimer at its
 * start (first CTA to start) and end (last CTA to finish) into a device buffer; the launches keep
 * their programmatic-dependent-launch overlap (nothing is serialised, unlike events around every
 * launch). After the caller has synchronised the stream, dovetail_trace_read returns one record per
 * launch of the last step, in launch order:
 *   kind[i]   0 step set-up, 1 DGF projections (or fusion linear), 2 DGF gate, 3 QKV, 4 tree attention,
 *             5 O-proj, 6 gate/up, 7 down, 8 LM head, 9 tree bookkeeping, 10 h fill
 *   level[i]  tree level of the launch (0 = the level-0 forward)
 *   bytes[i]  algorithmic HBM bytes of the launch (weights, prefix K/V)
 *   t0_ns[i], t1_ns[i]  first CTA start / last CTA end, ns of the GPU's global timer
 * Host arrays of capacity `cap`; *n = number of records written (<= cap). */
#define DOVETAIL_N_KINDS 11
int dovetail_trace_enable(dovetail_draft_t* h, int32_t enable);
int dovetail_trace_read(dovetail_draft_t* h, int32_t cap, int32_t* kind, int32_t* level, int64_t* bytes,
                        uint64_t* t0_ns, uint64_t* t1_ns, int32_t* n);

/* Design knobs for A/B measurements (bench.py --tune KEY=VALUE). They change how the step is launched, never
 * what it computes. Keys are listed here as they are added; an unknown key or a value out of range returns
 * EINVAL. */
int dovetail_hooks_tune(dovetail_draft_t* h, int32_t key, int32_t value);
/* key 1: tree levels (and level-0 row batches) of at least `value` rows run on the tcgen05 GEMV
 * (csrc/gemv_umma.cuh) instead of the mma.sync GEMV; 1 ... 64, 65 = never. Default 8. bf16 weights only. */
#define DOVETAIL_TUNE_UMMA_MIN_M 1
/* key 2: 1 (default) = dovetail_draft_step replays one CUDA graph per (tree_spec, n_new, attention geometry);
 * 0 = direct launches. Steps with test hooks or tracing set always launch directly. */
#define DOVETAIL_TUNE_GRAPHS 2
/* key 3: attention launches with more than `value` query vectors (rows of the level x q-heads per kv-head) use the
 * 64-vectors-per-pass kernel (csrc/attention_mma.cuh, QT = 4). Default 32 (measured on the 13B shape: at 32 vectors two
 * passes of the 16-vector kernel take 36 us against 43 us, at 48 vectors 38 against 30 us); 4096 = never, 0 = always. */
#define DOVETAIL_TUNE_ATTN_WIDE_MIN 3
/* key 4: 1 (default) = attention launches with 17 ... 32 query vectors use the 32-vectors-per-pass kernel (QT = 2: one
 * pass over the cache instead of two); 0 = two passes of the 16-vector kernel. */
#define DOVETAIL_TUNE_ATTN_QT2 4
/* key 5: the tcgen05 GEMVs whose CTAs hold one super-block (O, down, DGF) run with K split over CTA pairs
 * (csrc/gemv_umma.cuh UmmaParams::ksplit) at levels of at least `value` rows, and at any tcgen05 level when the boxes of a
 * pair fit a 64-row tile; default 48; 65 = never; 1 = always. */
#define DOVETAIL_TUNE_UMMA_KSPLIT_MIN_M 5

/* Host logic of the tcgen05 GEMV's row-exact work split (csrc/gemv_umma.cuh), callable without a GPU: for a group of
 * n_mat matrices with rows[] rows dealt to `ctas` CTAs (paired: gate / up; pairperm: head_dim of rotary-paired QKV
 * rows, else 0) returns per CTA the number of super-blocks n_sb[ctas], the 8-row boxes of each n_grp[ctas][8] and
 * grp[ctas][8][16] ((matrix << 28) | first row), its row count cnt[ctas] and the tile position of every virtual row
 * vpos[ctas][*vpos_ld] (super-block * 128 + tile row). Errors: EINVAL, ECAPACITY (more than 8 super-blocks per CTA or
 * vpos_cap too small). */
int dovetail_hooks_umma_tables(const int32_t rows[3], int32_t n_mat, int32_t paired, int32_t pairperm, int32_t ctas,
                               int32_t* n_sb, int32_t* n_grp, int32_t* grp, uint16_t* vpos, int32_t vpos_cap, int32_t* vpos_ld,
                               int32_t* cnt);

/* Counters of the last dovetail_draft_step, for tests that must know which kernel ran.
 *   key 1: launches of the tcgen05 GEMV (k_gemv_umma). Unknown key or NULL handle: -1. */
#define DOVETAIL_STAT_UMMA_LAUNCHES 1
/*   key 2: how the last step was launched: 0 direct launches, 1 graph replay, 2 graph captured and launched. */
#define DOVETAIL_STAT_GRAPH 2
/*   key 3: launches of the tcgen05 GEMV with K split over CTA pairs (direct launches only: a graph replay reports what its
 *          capture counted). */
#define DOVETAIL_STAT_KSPLIT_LAUNCHES 3
int dovetail_hooks_stat(const dovetail_draft_t* h, int32_t key);

/* Read-only HBM streaming ceilings, run by bench.py next to the step: reads `bytes`
 * bytes of `buf` (device, 16-byte aligned, larger than L2) exactly once on cuda_stream.
 *   mode 0: every thread sums 16-byte loads (grid-stride, 8 in flight per thread)
 *   mode 1: the GEMV's data path without arithmetic: one CTA per SM, bulk async copies of `seg`
 *           bytes (multiple of 16, 512 ... 8192) through a shared-memory ring of ~200 KB
 * Asynchronous; the caller times it with events. Errors: EINVAL, ECUDA. */
int dovetail_probe_stream(dovetail_draft_t* h, const void* buf, int64_t bytes, int32_t mode, int32_t seg,
                          void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* DOVETAIL_HOOKS_H_ */

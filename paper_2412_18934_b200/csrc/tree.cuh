// tree.cuh -- the integer side of the draft step:
//   S0  per-step set-up: level-0 row tables, rotary table
//   S7  merge of the LM-head partial top-b lists, log-softmax normaliser,
//       cumulative log-probability scores ("global acceptance probability"),
//       pool append, frontier selection, next level's row tables / ancestor masks
//   S8  final rerank to the top-gamma candidates, emitted in pool order
//   S9  KV commit of the accepted path
// Orders (reading A7): candidates of a row by (logit desc, token id asc);
// nodes by (cumulative score desc, pool index asc). Everything here is
// rank-by-counting on strict total orders, hence bit-exact by construction.
#pragma once
#include "gemv.cuh"
#include "ptx.cuh"
#include "state.cuh"

namespace dvt {

struct Pool {  // device arrays of capacity pool_cap
  int32_t* token;
  int32_t* parent;  // pool index or -1 (child of the root)
  int32_t* depth;   // 1-based level
  float* cum;       // sum of natural-log probabilities root -> node (reading A9)
  int32_t* row;     // step row that forwarded the node, or -1
};

// ---- S0 ---------------------------------------------------------------------
// grid = n_new + depth - 1 CTAs (one rotary-table row each) x 64 threads.
__global__ void k_step_begin(const StepDyn dynv, StepDyn* dyn, TreeState* ts, RowTables* rt0,
                             float2* rope, const double* inv_freq, int half, int vocab, int d, SplitOut feat_so,
                             unsigned long long* trace) {
  pdl_launch_dependents();
  trace_begin(trace);
  pdl_wait();
  const int r = blockIdx.x, n_new = dynv.n_new;
  // rotary angles in fp64: pos * theta^(-2i/dh) reaches thousands of radians
  const int pos = r < n_new ? dynv.L + r : dynv.Lp + (r - n_new);
  for (int i = threadIdx.x; i < half; i += blockDim.x) {
    double s, c;
    sincos(static_cast<double>(pos) * inv_freq[i], &s, &c);
    rope[static_cast<size_t>(r) * half + i] = make_float2(static_cast<float>(c), static_cast<float>(s));
  }
  // the caller's fp32 features as split-bf16 planes, the B operand of the DGF projection (epilogue.cuh)
  if (r < n_new && feat_so.xs != nullptr) split_row(feat_so, r, dynv.feats + static_cast<size_t>(r) * d, d);
  if (r == 0) {
    if (threadIdx.x == 0) {
      *dyn = dynv;  // ts->status is sticky until dovetail_draft_status / kv_commit reads it
      ts->pool_size = 0;
      ts->n_out = 0;
    }
    __syncthreads();
    for (int m = threadIdx.x; m < n_new; m += blockDim.x) {
      int t = dynv.tokens[m];
      if (t < 0 || t >= vocab) {
        t = min(max(t, 0), vocab - 1);
        atomicOr(&ts->status, 1);
      }
      rt0->token[m] = t;
      rt0->src[m] = m;
      rt0->slot[m] = m;  // cache row L + m
      rt0->pool[m] = -1;
      for (int w = 0; w < kMaskWords; ++w) {  // causal among the level-0 rows: bits 0..m
        const int lo = w * 32;
        rt0->mask[m][w] = m >= lo + 31 ? 0xffffffffu : (m < lo ? 0u : (0xffffffffu >> (31 - (m - lo))));
      }
    }
  }
  __syncthreads();
  trace_end(trace);
}

// Test hook (teacher forcing, dovetail_hooks.h): planes of M forced hidden-state rows. grid = M.
__global__ void k_resplit_rows(const float* x, int d, SplitOut so) {
  split_row(so, blockIdx.x, x + static_cast<size_t>(blockIdx.x) * d, d);
}

// int8 weights: the embedding row of each of the level's tokens as activation planes in the int8 consumer's
// format (fp16 terms, its k order). grid = M rows.
__global__ void k_embed_plane(const RowTables* rt, const __nv_bfloat16* embed, int d, SplitOut so, unsigned long long* trace) {
  pdl_launch_dependents();
  trace_begin(trace);
  pdl_wait();
  const int m = blockIdx.x;
  const __nv_bfloat16* src = embed + static_cast<size_t>(rt->token[m]) * d;
  constexpr int B = 8;  // loads of a round are issued before any store
  for (int k0 = threadIdx.x; k0 < d; k0 += blockDim.x * B) {
    float v[B];
#pragma unroll
    for (int i = 0; i < B; ++i) {
      const int k = k0 + i * blockDim.x;
      v[i] = k < d ? __bfloat162float(src[k]) : 0.f;
    }
#pragma unroll
    for (int i = 0; i < B; ++i) {
      const int k = k0 + i * blockDim.x;
      if (k < d) store_split(so, m, k, v[i]);
    }
  }
  __syncthreads();
  trace_end(trace);
}

// Wide levels (gemv_umma.cuh): the tensor-map copies of the tcgen05 GEMV read contiguous rows, so the level's
// gathered inputs are laid out first. grid = (M, kSplitPlanes + 1): y < kSplitPlanes copies plane y of the
// parent's hidden state (step row rt->src[m]) to row m of `par` (skipped when src == NULL: level 0 reads the
// caller's rows in place); y == kSplitPlanes copies the token's embedding row (bf16: one exact plane) to `emb`.
__global__ void k_gather_level(const RowTables* rt, const __nv_bfloat16* src, int64_t src_plane, __nv_bfloat16* par,
                               int64_t par_plane, const __nv_bfloat16* embed, __nv_bfloat16* emb, int64_t ld, int d,
                               unsigned long long* trace) {
  pdl_launch_dependents();
  trace_begin(trace);
  pdl_wait();
  const int m = blockIdx.x, y = blockIdx.y;
  const uint4* s4 = nullptr;
  uint4* d4 = nullptr;
  if (y < kSplitPlanes) {
    if (src != nullptr) {
      s4 = reinterpret_cast<const uint4*>(src + y * src_plane + static_cast<int64_t>(rt->src[m]) * ld);
      d4 = reinterpret_cast<uint4*>(par + y * par_plane + static_cast<int64_t>(m) * ld);
    }
  } else {
    s4 = reinterpret_cast<const uint4*>(embed + static_cast<size_t>(rt->token[m]) * d);
    d4 = reinterpret_cast<uint4*>(emb + static_cast<int64_t>(m) * ld);
  }
  if (s4 != nullptr)
    for (int i = threadIdx.x; i < d / 8; i += blockDim.x) d4[i] = s4[i];
  __syncthreads();
  trace_end(trace);
}

// dgf_proj == 0: h1 = f, h2 = e (W1 = W2 = identity). grid-stride over M * 2d.
template <typename WT>
__global__ void k_fill_h(const StepDyn* dyn, int from_dyn, const float* xsrc, int64_t xld,
                         const RowTables* rt, int use_idx, const WT* embed, float* hbuf, int M, int d, SplitOut so,
                         unsigned long long* trace) {
  pdl_launch_dependents();
  trace_begin(trace);
  pdl_wait();
  const float* base = from_dyn ? dyn->feats : xsrc;
  for (int64_t idx = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; idx < static_cast<int64_t>(M) * 2 * d;
       idx += static_cast<int64_t>(gridDim.x) * blockDim.x) {
    const int m = static_cast<int>(idx / (2 * d)), k = static_cast<int>(idx % (2 * d));
    float v;
    if (k < d) v = base[static_cast<int64_t>(use_idx ? rt->src[m] : m) * xld + k];
    else {
      const WT e = embed[static_cast<size_t>(rt->token[m]) * d + (k - d)];
      if (sizeof(WT) == 2) v = __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(&e));
      else v = *reinterpret_cast<const float*>(&e);
    }
    hbuf[idx] = v;
    if (so.xs) store_split(so, m, k, v);
  }
  __syncthreads();
  trace_end(trace);
}

// ---- S7 / S8 -----------------------------------------------------------------
struct TreeLevelParams {
  const StepDyn* dyn;
  TreeState* ts;
  Pool pool;
  uint32_t* treemask;      // [kMaxTreeSlots][kMaskWords] ancestor mask of each tree row
  // LM-head partials of this level's rows ...
  const float* cand_val;
  const int32_t* cand_id;
  const float* stat;
  int32_t nct;
  // ... or (replay) caller-supplied lists
  const int32_t* rp_tokens;
  const float* rp_logp;
  int32_t rp_maxb, rp_row0;
  int32_t M, b;            // rows expanded at this level, children kept per row
  int32_t level;           // 0-based; children get depth level + 1
  int32_t pool_begin;      // pool index of this level's first child
  int32_t M_next;          // rows of the next level (0: this is the last level)
  int32_t next_row0;       // step row of the next level's first row
  int32_t cur_row0;        // step row of this level's first expanded row (level 0: unused, the root row is n_new - 1)
  int32_t next_t0;         // tree-row index (= new-region slot) of the next level's first row
  int32_t n_new;           // step rows before the first tree row; root row = n_new - 1
  const RowTables* cur;
  RowTables* next;
  // final rerank (last level only)
  int32_t gamma, pool_total;
  int32_t* out_pool_idx;   // [gamma] pool index of each emitted candidate (for kv_commit)
  int32_t* o_ids;          // explicit outputs (replay); NULL: take them from dyn
  float* o_scores;
  int32_t* o_parents;
  int32_t* o_depths;
  int32_t* o_n;
  // test hooks (dovetail_hooks.h): taps of this level's candidates as computed, then teacher forcing
  int32_t* tap_token;
  float* tap_cum;
  const int32_t* force_token;
  const float* force_cum;
  unsigned long long* trace;
};

__device__ __forceinline__ bool node_before(const float* cum, int a, int b) {
  const float ca = cum[a], cb = cum[b];
  return ca > cb || (ca == cb && a < b);
}

constexpr int kTreeThreads = 512;  // one warp per expanded row for levels of <= 16 rows (a row's merge is a serial chain)
constexpr int kPoolSmem = 4352;  // >= kMaxBranch + kMaxTreeSlots * kMaxBranch + slack

__global__ void __launch_bounds__(kTreeThreads) k_tree_level(const TreeLevelParams p) {
  // phases B / C: pool scores and keep flags
  __shared__ float s_raw[2 * kPoolSmem];
  __shared__ int32_t s_cnt[kTreeThreads + 1];
  __shared__ int32_t s_tok[kMaxRows * kMaxBranch];  // this level's children: tokens (scores in s_cum), row-major [row][rank]
  float* s_cum = s_raw;
  int32_t* s_new = reinterpret_cast<int32_t*>(s_raw + kPoolSmem);
  pdl_launch_dependents();
  trace_begin(p.trace);
  pdl_wait();
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const Pool& P = p.pool;

  // ---- phase A: children of each expanded row --------------------------------
  // One warp per row. The row's global top-b is a b-round merge of the per-CTA lists, each of which is sorted in the
  // strict candidate order (gemv.cuh EPI_LMHEAD). Lane l owns the lists of CTAs l, l + 32, ... and keeps a window
  // of two entries per list in registers: a round picks the best head of the warp, the owning lane shifts that
  // list's window and requests the entry after it -- needed only if the same list wins twice more, so its L2
  // round trip is off the critical path. (Staging whole lists through shared memory, two rows at a time, cost
  // 53 us per level at 10 rows x 10 children; this takes the lists where they are.)
  for (int m = warp; m < p.M; m += kTreeThreads / 32) {
    const int parent = p.cur->pool[m];
    const float pcum = parent < 0 ? 0.f : P.cum[parent];
    const int base = p.pool_begin + m * p.b;
    if (p.rp_tokens) {
      if (lane < p.b) {
        const size_t o = static_cast<size_t>(p.rp_row0 + m) * p.rp_maxb + lane;
        P.token[base + lane] = p.rp_tokens[o];
        P.parent[base + lane] = parent;
        P.depth[base + lane] = p.level + 1;
        P.cum[base + lane] = pcum + p.rp_logp[o];
        P.row[base + lane] = -1;
        s_tok[m * p.b + lane] = p.rp_tokens[o];
        s_cum[m * p.b + lane] = pcum + p.rp_logp[o];
      }
      continue;
    }
    const float* st = p.stat + static_cast<size_t>(m) * p.nct * 2;
    const float* cv = p.cand_val + static_cast<size_t>(m) * p.nct * kMaxBranch;
    const int32_t* ci = p.cand_id + static_cast<size_t>(m) * p.nct * kMaxBranch;
    constexpr int kLists = 8;  // lists per lane: nct <= 256 (host)
    float hv[kLists], nv[kLists], smx[kLists], sse[kLists];
    int hi[kLists], ni[kLists], hp[kLists];
#pragma unroll
    for (int k = 0; k < kLists; ++k) {  // every load of the row is issued before the first use
      const int c = lane + 32 * k;
      hp[k] = 0;
      hv[k] = nv[k] = smx[k] = -INFINITY;
      hi[k] = ni[k] = 0x7fffffff;
      sse[k] = 0.f;
      if (c < p.nct) {
        hv[k] = __ldcg(cv + c * kMaxBranch);
        hi[k] = __ldcg(ci + c * kMaxBranch);
        if (p.b > 1) { nv[k] = __ldcg(cv + c * kMaxBranch + 1); ni[k] = __ldcg(ci + c * kMaxBranch + 1); }
        smx[k] = __ldcg(st + c * 2);
        sse[k] = __ldcg(st + c * 2 + 1);
      }
    }
    // log-sum-exp over the vocabulary from the per-CTA (max, sum exp) pairs, fixed order (lane-major, then butterfly)
    float mg = -INFINITY;
#pragma unroll
    for (int k = 0; k < kLists; ++k) mg = fmaxf(mg, smx[k]);
    mg = warp_max(mg);
    float se = 0.f;
#pragma unroll
    for (int k = 0; k < kLists; ++k) se += (smx[k] == -INFINITY) ? 0.f : sse[k] * expf(smx[k] - mg);
    se = warp_sum(se);
    const float logz = mg + logf(se);
    for (int jb = 0; jb < p.b; ++jb) {
      float bv = -INFINITY;
      int bi = 0x7fffffff;
#pragma unroll
      for (int k = 0; k < kLists; ++k)
        if (cand_before(hv[k], hi[k], bv, bi)) { bv = hv[k]; bi = hi[k]; }
      const int mine = bi;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (cand_before(ov, oi, bv, bi)) { bv = ov; bi = oi; }
      }
      if (mine == bi && bi != 0x7fffffff) {  // token ids are unique across the lists: exactly one lane advances
#pragma unroll
        for (int k = 0; k < kLists; ++k) {
          if (hi[k] == bi) {
            const int c = lane + 32 * k;
            ++hp[k];
            hv[k] = nv[k];
            hi[k] = ni[k];
            if (hp[k] + 1 < p.b) { nv[k] = __ldcg(cv + c * kMaxBranch + hp[k] + 1); ni[k] = __ldcg(ci + c * kMaxBranch + hp[k] + 1); }
            else { nv[k] = -INFINITY; ni[k] = 0x7fffffff; }
          }
        }
      }
      if (lane == 0) {
        P.token[base + jb] = bi;
        P.parent[base + jb] = parent;
        P.depth[base + jb] = p.level + 1;
        P.cum[base + jb] = pcum + (bv - logz);  // cumulative log-probability
        P.row[base + jb] = -1;
        s_tok[m * p.b + jb] = bi;  // phase B works from shared memory: no round trip through the pool
        s_cum[m * p.b + jb] = pcum + (bv - logz);
      }
    }
  }
  __syncthreads();

  const int n = p.M * p.b;
  if (p.tap_token != nullptr || p.force_token != nullptr) {  // hooks: never set in a plain step
    for (int i = tid; i < n; i += kTreeThreads) {
      const int node = p.pool_begin + i;
      if (p.tap_token) { p.tap_token[node] = P.token[node]; p.tap_cum[node] = P.cum[node]; }
      if (p.force_token) {
        P.token[node] = p.force_token[node];
        P.cum[node] = p.force_cum[node];
        s_tok[i] = p.force_token[node];
        s_cum[i] = p.force_cum[node];
      }
    }
    __syncthreads();
  }

  // ---- phase B: frontier of the next level = top-M_next children by score -----
  if (p.M_next > 0) {
    // Everything a selected child needs is its parent's row of THIS level (m = i / b): the node forwarded there
    // (cur->pool[m]), that row's step row (cur_row0 + m) and its ancestor mask (cur->mask[m]) -- no dependent
    // loads through the pool arrays.
    for (int i = tid; i < n; i += kTreeThreads) {
      int rank = 0;
      for (int j = 0; j < n; ++j) rank += (j != i && node_before(s_cum, j, i)) ? 1 : 0;
      if (rank < p.M_next) {
        const int node = p.pool_begin + i, r = rank, m = i / p.b;
        const bool root = p.level == 0;
        const int t = p.next_t0 + r;  // tree-row index = new-region slot
        p.next->token[r] = s_tok[i];
        p.next->src[r] = root ? p.n_new - 1 : p.cur_row0 + m;
        p.next->slot[r] = t;
        p.next->pool[r] = node;
        P.row[node] = p.next_row0 + r;
        for (int w = 0; w < kMaskWords; ++w) {
          uint32_t mk = root ? 0u : p.cur->mask[m][w];
          if ((t >> 5) == w) mk |= 1u << (t & 31);
          p.treemask[t * kMaskWords + w] = mk;
          p.next->mask[r][w] = mk;
        }
      }
    }
    __syncthreads();
    trace_end(p.trace);
    return;
  }

  // ---- phase C (last level): S8, top-gamma of the whole pool, pool order ------
  const int Pn = p.pool_total;
  for (int i = tid; i < Pn; i += kTreeThreads) s_cum[i] = P.cum[i];
  __syncthreads();
  const int n_keep = min(p.gamma, Pn);
  for (int i = tid; i < Pn; i += kTreeThreads) {
    int rank = 0;
    for (int j = 0; j < Pn; ++j) rank += (j != i && node_before(s_cum, j, i)) ? 1 : 0;
    s_new[i] = rank < n_keep ? 1 : 0;
  }
  __syncthreads();
  // exclusive prefix count of the keep flags: contiguous chunk per thread
  const int chunk = (Pn + kTreeThreads - 1) / kTreeThreads;
  const int lo = min(Pn, tid * chunk), hi = min(Pn, lo + chunk);
  int cnt = 0;
  for (int i = lo; i < hi; ++i) cnt += s_new[i];
  s_cnt[tid + 1] = cnt;
  __syncthreads();
  if (warp == 0) {  // inclusive prefix over the per-thread counts: kTreeThreads / 32 entries per lane, then a warp scan
    constexpr int E = kTreeThreads / 32;
    int loc = 0;
    for (int j = 0; j < E; ++j) loc += s_cnt[1 + lane * E + j];
    int inc = loc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int v = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += v;
    }
    int run2 = inc - loc;
    for (int j = 0; j < E; ++j) {
      run2 += s_cnt[1 + lane * E + j];
      s_cnt[1 + lane * E + j] = run2;
    }
    if (lane == 0) s_cnt[0] = 0;
  }
  __syncthreads();
  int run = s_cnt[tid];
  for (int i = lo; i < hi; ++i) {
    const int k = s_new[i];
    s_new[i] = k ? run : -1;  // output index of node i, or -1
    run += k;
  }
  __syncthreads();
  const StepDyn* dyn = p.dyn;
  int32_t* o_ids = p.o_ids ? p.o_ids : dyn->out_ids;
  float* o_scores = p.o_ids ? p.o_scores : dyn->out_scores;
  int32_t* o_parents = p.o_ids ? p.o_parents : dyn->out_parents;
  int32_t* o_depths = p.o_ids ? p.o_depths : dyn->out_depths;
  int32_t* o_n = p.o_ids ? p.o_n : dyn->out_n;
  for (int i = tid; i < Pn; i += kTreeThreads) {
    const int o = s_new[i];
    if (o < 0) continue;
    const int parent = P.parent[i];
    o_ids[o] = P.token[i];
    o_scores[o] = s_cum[i];
    o_parents[o] = parent < 0 ? -1 : s_new[parent];  // kept set is ancestor-closed (A7)
    if (o_depths) o_depths[o] = P.depth[i];
    p.out_pool_idx[o] = i;
  }
  if (tid == 0) {
    *o_n = n_keep;
    p.ts->n_out = n_keep;
    p.ts->pool_size = Pn;
  }
  __syncthreads();
  trace_end(p.trace);
}

// ---- S9 ------------------------------------------------------------------------
struct CommitPath {
  int32_t n;
  int32_t idx[kMaxDepth + 1];
};

// Validates the accepted path against the last step's output (root first, each
// entry a child of the previous one) and lists the tree rows to move.
__global__ void k_commit_plan(const CommitPath path, TreeState* ts, Pool pool, const int32_t* out_pool_idx,
                              int n_new) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  int err = 0, n_mv = 0;
  bool run = true;
  int prev = -1;
  for (int i = 0; i < path.n && !err; ++i) {
    const int o = path.idx[i];
    if (o < 0 || o >= ts->n_out) { err = 1; break; }
    const int node = out_pool_idx[o];
    if (pool.parent[node] != prev) { err = 1; break; }
    prev = node;
    const int row = pool.row[node];
    if (run && row >= 0) ts->commit_src[n_mv++] = row - n_new;
    else run = false;
  }
  ts->commit_err = err;
  ts->commit_n = err ? 0 : n_mv;
}

// grid = (n_layers * Hkv, 2): moves the committed rows of one (layer, kv-head) of
// K (y = 0) or V (y = 1): cache row Lp + src[i] -> Lp + i. All sources are read
// before any destination is written (src[i] >= i, ranges may overlap).
__global__ void k_commit_move(const TreeState* ts, void* kc, void* vc, int capacity, int Lp, int row_bytes) {
  extern __shared__ __align__(16) uint8_t sm[];
  const int n = ts->commit_n;
  if (ts->commit_err || n == 0) return;
  uint8_t* base = static_cast<uint8_t*>(blockIdx.y ? vc : kc) +
                  static_cast<size_t>(blockIdx.x) * capacity * row_bytes;
  const int units = row_bytes / 16;
  for (int idx = threadIdx.x; idx < n * units; idx += blockDim.x) {
    const int i = idx / units, u = idx % units;
    reinterpret_cast<uint4*>(sm)[idx] =
        *reinterpret_cast<const uint4*>(base + static_cast<size_t>(Lp + ts->commit_src[i]) * row_bytes + u * 16);
  }
  __syncthreads();
  for (int idx = threadIdx.x; idx < n * units; idx += blockDim.x) {
    const int i = idx / units, u = idx % units;
    *reinterpret_cast<uint4*>(base + static_cast<size_t>(Lp + i) * row_bytes + u * 16) = reinterpret_cast<uint4*>(sm)[idx];
  }
}

}  // namespace dvt

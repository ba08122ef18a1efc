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
      rt0->cum[m] = 0.f;
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

// Pool::row of a child: >= 0 the step row it is forwarded at; -1 not forwarded; -2 not forwarded and outside its
// own level's top-gamma, hence outside the step's top-gamma (S8 does not look at it).
__global__ void __launch_bounds__(kTreeThreads) k_tree_level(const TreeLevelParams p) {
  __shared__ float s_raw[2 * kPoolSmem];
  __shared__ int32_t s_tok[kMaxRows * kMaxBranch];  // this level's children: tokens (scores in s_cum), row-major [row][rank]
  __shared__ uint32_t s_bits[kPoolSmem / 32];       // S8: kept nodes, one bit per pool index
  __shared__ int32_t s_nc;
  float* s_cum = s_raw;                 // phases A / B: this level's children; S8: candidate scores
  float* s_scr = s_raw + kPoolSmem;     // phase A: per-warp list tails; S8: candidate pool indices
  pdl_launch_dependents();
  trace_begin(p.trace);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const Pool& P = p.pool;
  // kernel parameters before the wait: their (cold) constant-bank misses overlap the LM head's tail
  const int b = p.b, nct = p.nct;
  const float* cv0 = p.cand_val;
  const int32_t* ci0 = p.cand_id;
  const float* st0 = p.stat;
  asm volatile("" ::"r"(b), "r"(nct), "l"(cv0), "l"(ci0), "l"(st0));
  pdl_wait();

  // ---- phase A: children of each expanded row --------------------------------
  // One warp per row. The per-CTA lists of the LM head are sorted in the strict candidate order (gemv.cuh
  // EPI_LMHEAD) and stored entry-major ([row][entry j][CTA c]): the heads of a row are contiguous.
  //  (1) the warp reads every head (coalesced) and the (max, sum exp) pairs;
  //  (2) b rounds of warp-argmax over the heads name the b lists with the best heads, in order (lane r keeps the
  //      r-th). No other list can contribute: b heads come before each of its entries. Entry j of the r-th list has
  //      r + j candidates before it, so only j < b - r matters;
  //  (3) the second entry of every list comes with the heads; the other tail entries of the b lists (b > 2) are
  //      fetched in one batch into shared memory;
  //  (4) b rounds merge the <= b lists, lane r owning the r-th, without touching global memory.
  // (A merge that fetched a list's next entry when its head won paid an L2 round trip per round -- the scoreboard
  // waits for the load even where the value is not needed yet -- and its 128-byte-strided head loads cost 32 tag
  // look-ups per instruction: 15 us at 10 rows x 10 children, 37 us at 32 rows x 2, 21 us at 1 row x 32.)
  const int per_row = 2 * b * b;  // words of scratch per warp
  const int n_act = max(1, min(kTreeThreads / 32, kPoolSmem / per_row));
  for (int m = warp; m < p.M && warp < n_act; m += n_act) {
    const int base = p.pool_begin + m * b;
    if (p.rp_tokens) {
      const int parent = p.cur->pool[m];
      const float pcum = parent < 0 ? 0.f : p.cur->cum[m];
      if (lane < b) {
        const size_t o = static_cast<size_t>(p.rp_row0 + m) * p.rp_maxb + lane;
        P.token[base + lane] = p.rp_tokens[o];
        P.parent[base + lane] = parent;
        P.depth[base + lane] = p.level + 1;
        P.cum[base + lane] = pcum + p.rp_logp[o];
        P.row[base + lane] = -1;
        s_tok[m * b + lane] = p.rp_tokens[o];
        s_cum[m * b + lane] = pcum + p.rp_logp[o];
      }
      continue;
    }
    const size_t rowoff = static_cast<size_t>(m) * kMaxBranch * nct;
    const float* cv = cv0 + rowoff;
    const int32_t* ci = ci0 + rowoff;
    const float2* st = reinterpret_cast<const float2*>(st0) + static_cast<size_t>(m) * nct;
    constexpr int kLists = 8;  // lists per lane: nct <= 256 (host)
    // A candidate as two words that compare like cand_before: hk = its value as an order-preserving unsigned key
    // (0 = no candidate), lo = (0xffffff - id) << 8 | CTA. The warp's best is then two redux.sync.max.
    uint64_t key[kLists];
    float smx[kLists], sse[kLists], v1[kLists];  // v1 / i1: every list's second entry, fetched with the heads
    int i1[kLists];
#pragma unroll
    for (int k = 0; k < kLists; ++k) {  // every load of the row is issued before the first use
      const int c = lane + 32 * k;
      key[k] = 0ull;
      smx[k] = v1[k] = -INFINITY;
      sse[k] = 0.f;
      i1[k] = kNoCand;
      if (c < nct) {
        const float v = __ldcg(cv + c);
        const int id = __ldcg(ci + c);
        const float2 s2 = __ldcg(st + c);
        if (b > 1) { v1[k] = __ldcg(cv + nct + c); i1[k] = __ldcg(ci + nct + c); }
        key[k] = (static_cast<uint64_t>(cand_key(v, id)) << 32) | cand_lo(id, c);
        smx[k] = s2.x;
        sse[k] = s2.y;
      }
    }
    const int parent = p.cur->pool[m];  // (after the loads above are in flight)
    const float pcum = parent < 0 ? 0.f : p.cur->cum[m];
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
    // (2) the b best heads: lane r keeps the r-th. The lane's best is a pairwise tree (a serial scan of the eight
    // is a chain of ~50 dependent instructions per round); the winner is cleared by value, ids being unique.
    uint32_t* sh = reinterpret_cast<uint32_t*>(s_scr) + warp * per_row;
    uint32_t* sl = sh + b * b;
    uint32_t th = 0u, tl = 0u;
    for (int r = 0; r < b; ++r) {
      const uint64_t m01 = umax64(key[0], key[1]), m23 = umax64(key[2], key[3]);
      const uint64_t m45 = umax64(key[4], key[5]), m67 = umax64(key[6], key[7]);
      const uint64_t best = umax64(umax64(m01, m23), umax64(m45, m67));
      const uint32_t bh = static_cast<uint32_t>(best >> 32), bl = static_cast<uint32_t>(best);
      const uint32_t gh = __reduce_max_sync(0xffffffffu, bh);
      const uint32_t gl = __reduce_max_sync(0xffffffffu, bh == gh ? bl : 0u);
      const uint64_t g = (static_cast<uint64_t>(gh) << 32) | gl;
#pragma unroll
      for (int k = 0; k < kLists; ++k)
        if (key[k] == g && gh != 0u) {  // the winner hands the list's second entry over: (r, 1)
          key[k] = 0ull;
          if (b > 1) { sh[r * b + 1] = cand_key(v1[k], i1[k]); sl[r * b + 1] = cand_lo(i1[k], 0); }
        }
      if (lane == r) { th = gh; tl = gl; }
    }
    const int tc = th != 0u ? static_cast<int>(tl & 255u) : -1;  // CTA of the r-th list
    // (3) tails of those lists: entry (r, j), 2 <= j < b - r, at scratch [r * b + j] (a second round trip, b > 2 only)
    constexpr int kU = 16;
    const int binv = (65536 + b - 1) / b;  // e / b == (e * binv) >> 16 for e < 1024, b <= 32
    for (int e0 = 0; e0 < b * b && b > 2; e0 += 32 * kU) {
      float v[kU];
      int id[kU];
      bool ok2[kU];
#pragma unroll
      for (int u = 0; u < kU; ++u) {
        const int e = e0 + 32 * u + lane;
        const int r = (e * binv) >> 16, j = e - r * b;
        const int cr = __shfl_sync(0xffffffffu, tc, r & 31);
        const bool ok = e < b * b && j >= 2 && j < b - r && cr >= 0;
        v[u] = -INFINITY;
        id[u] = kNoCand;
        ok2[u] = ok;
        if (ok) {
          v[u] = __ldcg(cv + j * nct + cr);
          id[u] = __ldcg(ci + j * nct + cr);
        }
      }
#pragma unroll
      for (int u = 0; u < kU; ++u) {
        const int e = e0 + 32 * u + lane;
        if (ok2[u]) { sh[e] = cand_key(v[u], id[u]); sl[e] = cand_lo(id[u], 0); }
      }
    }
    __syncwarp();
    // (4) merge: lane r owns the r-th list
    uint32_t lh = th, ll = tl & ~255u;
    int hp = 0;
    const int lim = tc >= 0 ? b - lane : 0;
    uint32_t oh = 0u, ol = 0u;
    for (int jb = 0; jb < b; ++jb) {
      const uint32_t gh = __reduce_max_sync(0xffffffffu, lh);
      const uint32_t gl = __reduce_max_sync(0xffffffffu, lh == gh ? ll : 0u);
      if (lh == gh && ll == gl && gh != 0u) {
        ++hp;
        if (hp < lim) { lh = sh[lane * b + hp]; ll = sl[lane * b + hp]; }
        else { lh = ll = 0u; }
      }
      if (lane == jb) { oh = gh; ol = gl; }
    }
    if (lane < b) {
      const float ov = cand_key_value(oh);
      const int oi = oh != 0u ? static_cast<int>(0xffffffu - (ol >> 8)) : kNoCand;
      const float cum = pcum + (ov - logz);  // cumulative log-probability
      P.token[base + lane] = oi;
      P.parent[base + lane] = parent;
      P.depth[base + lane] = p.level + 1;
      P.cum[base + lane] = cum;
      P.row[base + lane] = -1;
      s_tok[m * b + lane] = oi;  // phase B works from shared memory: no round trip through the pool
      s_cum[m * b + lane] = cum;
    }
    __syncwarp();
  }
  if (tid == 0) s_nc = 0;
  for (int i = tid; i < kPoolSmem / 32; i += kTreeThreads) s_bits[i] = 0u;
  __syncthreads();

  const int n = p.M * b;
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
  // Everything a selected child needs is its parent's row of THIS level (m = i / b): the node forwarded there
  // (cur->pool[m]), that row's step row (cur_row0 + m) and its ancestor mask (cur->mask[m]) -- no dependent
  // loads through the pool arrays. A child ranked gamma or later among its own level cannot be in the step's
  // top-gamma: it is marked, and S8 ranks only the others (<= depth x gamma instead of the whole pool).
  for (int i = tid; i < n; i += kTreeThreads) {
    int rank = 0;
    for (int j = 0; j < n; ++j) rank += (j != i && node_before(s_cum, j, i)) ? 1 : 0;
    const int node = p.pool_begin + i;
    if (rank < p.M_next) {
      const int r = rank, m = i / b;
      const bool root = p.level == 0;
      const int t = p.next_t0 + r;  // tree-row index = new-region slot
      p.next->token[r] = s_tok[i];
      p.next->src[r] = root ? p.n_new - 1 : p.cur_row0 + m;
      p.next->slot[r] = t;
      p.next->pool[r] = node;
      p.next->cum[r] = s_cum[i];
      P.row[node] = p.next_row0 + r;
      for (int w = 0; w < kMaskWords; ++w) {
        uint32_t mk = root ? 0u : p.cur->mask[m][w];
        if ((t >> 5) == w) mk |= 1u << (t & 31);
        p.treemask[t * kMaskWords + w] = mk;
        p.next->mask[r][w] = mk;
      }
    } else if (rank >= p.gamma) {
      P.row[node] = -2;
    }
  }
  __syncthreads();
  if (p.M_next > 0) {
    trace_end(p.trace);
    return;
  }

  // ---- S8 (last level): top-gamma of the whole pool, emitted in pool order ------
  const int Pn = p.pool_total;
  const int n_keep = min(p.gamma, Pn);
  float* s_cc = s_raw;                                            // candidate scores
  int32_t* s_ci = reinterpret_cast<int32_t*>(s_raw + kPoolSmem);  // candidate pool indices
  for (int i = tid; i < Pn; i += kTreeThreads) {
    const int row = P.row[i];
    const float cum = P.cum[i];  // unconditional: one round trip, not two
    if (row != -2) {
      const int k = atomicAdd(&s_nc, 1);
      s_ci[k] = i;
      s_cc[k] = cum;
    }
  }
  __syncthreads();
  const int C = s_nc;  // >= n_keep: every level contributes its min(gamma, size) best
  for (int a = tid; a < C; a += kTreeThreads) {
    const float ca = s_cc[a];
    const int ia = s_ci[a];
    int rank = 0;
    for (int j = 0; j < C; ++j) {
      const float cj = s_cc[j];
      rank += (cj > ca || (cj == ca && s_ci[j] < ia)) ? 1 : 0;
    }
    if (rank < n_keep) atomicOr(&s_bits[ia >> 5], 1u << (ia & 31));
  }
  __syncthreads();
  // output index of a kept node = kept nodes before it in the pool
  int32_t* s_map = reinterpret_cast<int32_t*>(s_raw);  // (scores are read again from the pool)
  for (int i = tid; i < Pn; i += kTreeThreads) {
    if ((s_bits[i >> 5] >> (i & 31)) & 1u) {
      int o = __popc(s_bits[i >> 5] & ((1u << (i & 31)) - 1u));
      for (int w = 0; w < (i >> 5); ++w) o += __popc(s_bits[w]);
      s_map[i] = o;
    }
  }
  __syncthreads();
  const StepDyn* dyn = p.dyn;
  int32_t* o_ids = p.o_ids ? p.o_ids : dyn->out_ids;
  float* o_scores = p.o_ids ? p.o_scores : dyn->out_scores;
  int32_t* o_parents = p.o_ids ? p.o_parents : dyn->out_parents;
  int32_t* o_depths = p.o_ids ? p.o_depths : dyn->out_depths;
  int32_t* o_n = p.o_ids ? p.o_n : dyn->out_n;
  for (int i = tid; i < Pn; i += kTreeThreads) {
    if (!((s_bits[i >> 5] >> (i & 31)) & 1u)) continue;
    const int o = s_map[i];
    const int parent = P.parent[i];
    o_ids[o] = P.token[i];
    o_scores[o] = P.cum[i];
    o_parents[o] = parent < 0 ? -1 : s_map[parent];  // kept set is ancestor-closed (A7)
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

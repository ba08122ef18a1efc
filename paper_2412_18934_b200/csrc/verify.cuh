// verify.cuh -- the step right after the draft step: what the target needs to verify the
// candidates in one forward (ancestor mask, position ids, root-to-leaf paths), and the acceptance rule that
// turns the target's answer into the accepted path for dovetail_kv_commit -- greedy (T = 0) or speculative
// sampling (T = 1; Table 3, evaluates both). Integer work and single fp32 compares: bit-exact
// against the oracle by construction (reading A18 in DESIGN.md).
//
// Verifier rows: row 0 = the root (last verified token), row i + 1 = candidate i of the step's output
// (pool order: parents precede children, siblings in rank order).
#pragma once
#include "ptx.cuh"
#include "state.cuh"

namespace dvt {

struct VerifyPlanParams {
  const int32_t* parents;  // step output [n]
  const int32_t* depths;   // step output [n] (1-based)
  const int32_t* n_out;    // device scalar n
  int32_t gamma;           // capacity of the arrays = row stride of the mask minus 1
  int32_t root_position, max_depth;
  uint8_t* mask;           // [(gamma + 1) x (gamma + 1)]
  int32_t* position_ids;   // [gamma + 1]
  int32_t* paths;          // [gamma x max_depth]
  int32_t* n_paths;        // [1]
};

// One CTA. Rows past n_out are zeroed (mask) / -1 (paths).
__global__ void __launch_bounds__(256) k_verify_plan(const VerifyPlanParams p) {
  __shared__ int32_t s_leaf_rank[kMaxTreeSlots * kMaxBranch + kMaxBranch];  // >= pool capacity >= gamma kept
  __shared__ int32_t s_n_paths;
  const int n = *p.n_out, R = p.gamma + 1, tid = threadIdx.x;
  for (int i = tid; i < R * R; i += blockDim.x) p.mask[i] = 0;
  for (int i = tid; i < p.gamma * p.max_depth; i += blockDim.x) p.paths[i] = -1;
  __syncthreads();
  for (int r = tid; r <= n; r += blockDim.x) {
    p.mask[static_cast<size_t>(r) * R] = 1;  // the root is everybody's ancestor (and its own row)
    if (r == 0) { p.position_ids[0] = p.root_position; continue; }
    const int i = r - 1;
    p.position_ids[r] = p.root_position + p.depths[i];
    for (int a = i; a >= 0; a = p.parents[a]) p.mask[static_cast<size_t>(r) * R + a + 1] = 1;
  }
  for (int r = n + 1 + tid; r < R; r += blockDim.x) p.position_ids[r] = 0;
  // leaves = candidates that are nobody's parent, ranked in candidate order
  for (int i = tid; i < n; i += blockDim.x) {
    int is_parent = 0;
    for (int j = i + 1; j < n; ++j) is_parent |= (p.parents[j] == i);  // children follow their parent
    s_leaf_rank[i] = is_parent ? -1 : 0;
  }
  __syncthreads();
  if (tid == 0) {
    int k = 0;
    for (int i = 0; i < n; ++i)
      if (s_leaf_rank[i] == 0) s_leaf_rank[i] = k++;
    s_n_paths = k;
    *p.n_paths = k;
  }
  __syncthreads();
  for (int i = tid; i < n; i += blockDim.x) {
    const int k = s_leaf_rank[i];
    if (k < 0) continue;
    int len = 0;
    for (int a = i; a >= 0; a = p.parents[a]) ++len;
    int32_t* row = p.paths + static_cast<size_t>(k) * p.max_depth;
    int pos = len - 1;
    for (int a = i; a >= 0; a = p.parents[a]) row[pos--] = a;
  }
}

struct VerifyAcceptParams {
  const int32_t* token_ids;   // step output [n]
  const int32_t* parents;
  const int32_t* n_out;
  int32_t gamma, mode, vocab;
  const int32_t* tgt_argmax;  // mode 0: [gamma + 1] the target's argmax token at every verifier row
  const float* p_cand;        // mode 1: [gamma] target probability of candidate i's token at its parent
  const float* uniforms;      // mode 1: [gamma + 1] U[0,1): one per candidate, the last one for the bonus token
  const float* p_full;        // mode 1: [gamma + 1][vocab] the target's distribution at every verifier row
  int32_t* accepted_path;     // [max_depth]
  int32_t* n_acc;             // [1]
  int32_t* bonus_token;       // [1]
  int32_t max_depth;
};

constexpr int kVerifyThreads = 512;
constexpr int kVerifyStage = 1024;  // candidates staged in shared memory for the walk (more: read from global memory)

__global__ void __launch_bounds__(kVerifyThreads) k_verify_accept(const VerifyAcceptParams p) {
  constexpr int NW = kVerifyThreads / 32;
  __shared__ int32_t s_cur, s_nrej, s_rej[kMaxBranch * 4];
  __shared__ unsigned long long s_sum[NW], s_W;
  __shared__ int32_t s_par[kVerifyStage], s_tok[kVerifyStage], s_arg[kVerifyStage + 1];
  __shared__ float s_pc[kVerifyStage], s_un[kVerifyStage];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n = *p.n_out;
  // The walk is one thread following parent links: out of shared memory (one coalesced round trip for everything it
  // may touch) instead of a dependent global load per candidate looked at (~0.5 us each: 8 us per accepted level).
  const bool staged = n <= kVerifyStage;
  if (staged) {
    for (int i = tid; i < n; i += kVerifyThreads) {
      s_par[i] = p.parents[i];
      s_tok[i] = p.token_ids[i];
      if (p.mode == 0) s_arg[i] = p.tgt_argmax[i];
      else { s_pc[i] = p.p_cand[i]; s_un[i] = p.uniforms[i]; }
    }
    if (p.mode == 0 && tid == 0) s_arg[n] = p.tgt_argmax[n];
    __syncthreads();
  }
  if (tid == 0) {
    int cur = -1, na = 0, n_rej = 0;
    for (;;) {
      float rem = 1.0f;
      int found = -1;
      n_rej = 0;
      for (int i = 0; i < n && found < 0; ++i) {
        if ((staged ? s_par[i] : p.parents[i]) != cur) continue;
        const int tok = staged ? s_tok[i] : p.token_ids[i];
        if (p.mode == 0) {
          if (tok == (staged ? s_arg[cur + 1] : p.tgt_argmax[cur + 1])) found = i;
        } else {
          const float pc = staged ? s_pc[i] : p.p_cand[i];
          const float lhs = __fmul_rn(staged ? s_un[i] : p.uniforms[i], rem);  // no contraction: one multiply, one compare
          if (lhs < pc) found = i;
          else {
            rem = __fsub_rn(rem, pc);
            if (n_rej < kMaxBranch * 4) s_rej[n_rej] = tok;
            ++n_rej;
          }
        }
      }
      if (found < 0 || na >= p.max_depth) break;
      p.accepted_path[na++] = found;
      cur = found;
    }
    *p.n_acc = na;
    s_cur = cur;
    s_nrej = min(n_rej, kMaxBranch * 4);
    if (p.mode == 0) *p.bonus_token = staged ? s_arg[cur + 1] : p.tgt_argmax[cur + 1];
  }
  __syncthreads();
  if (p.mode == 0) return;
  // bonus token: integer inverse CDF over the target's distribution at the stopping row, rejected tokens removed.
  // The weights are integers, so a sum does not depend on its order. One CTA streams the row, so what matters is
  // loads in flight: every sum below issues 16 independent loads per lane before it adds, and the rejected tokens
  // (distinct: they are children of one node) are subtracted per range instead of being tested per element.
  // Pass 1: each warp sums its contiguous range (coalesced). Then, in the one warp whose range holds the threshold,
  // the range is narrowed 32-fold per round -- each lane sums a contiguous piece, a warp scan names the lane --
  // until it is one element per lane. (One contiguous chunk per thread, read element by element and walked again
  // by one thread, took 53 us on a 32000-token vocabulary and 141 us on 128256.)
  const float* pr = p.p_full + static_cast<size_t>(s_cur + 1) * p.vocab;
  const int n_rej = s_nrej;
  auto raw = [&](int x) -> unsigned long long { return static_cast<unsigned long long>(__fmul_rn(pr[x], 4294967296.0f)); };
  auto rejected = [&](int x0, int x1) -> unsigned long long {  // weight of the rejected tokens inside [x0, x1)
    unsigned long long sub = 0;
    for (int k = 0; k < n_rej; ++k)
      if (s_rej[k] >= x0 && s_rej[k] < x1) sub += raw(s_rej[k]);
    return sub;
  };
  auto strided_sum = [&](int x0, int x1, int first, int stride) -> unsigned long long {  // this thread's share of [x0, x1)
    constexpr int U = 16;
    unsigned long long acc = 0;
    for (int x = x0 + first; x < x1; x += U * stride) {
      float v[U];
#pragma unroll
      for (int u = 0; u < U; ++u) v[u] = x + u * stride < x1 ? pr[x + u * stride] : 0.f;
#pragma unroll
      for (int u = 0; u < U; ++u) acc += static_cast<unsigned long long>(__fmul_rn(v[u], 4294967296.0f));
    }
    return acc;
  };
  const int cw = (((p.vocab + NW - 1) / NW) + 31) & ~31;  // tokens per warp, a multiple of 32
  const int w0 = min(p.vocab, warp * cw), w1 = min(p.vocab, w0 + cw);
  unsigned long long tot = strided_sum(w0, w1, lane, 32);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
  tot -= rejected(w0, w1);
  if (lane == 0) s_sum[warp] = tot;
  __syncthreads();
  if (tid == 0) {  // exclusive prefix over the warp sums
    unsigned long long run = 0;
    for (int t = 0; t < NW; ++t) {
      const unsigned long long v = s_sum[t];
      s_sum[t] = run;
      run += v;
    }
    if (run == 0) *p.bonus_token = -1;
    s_W = run;
  }
  __syncthreads();
  const unsigned long long W = s_W;
  if (W == 0) return;
  const unsigned long long r = static_cast<unsigned long long>(static_cast<double>(p.uniforms[n]) * static_cast<double>(W));
  unsigned long long base = s_sum[warp];
  if (!(r >= base && r < base + tot)) return;  // exactly one warp's range holds the threshold
  int a = w0, bnd = w1;  // invariant: weight before a = base, and base <= r < base + weight[a, bnd)
  while (bnd - a > 32) {
    const int per = (bnd - a + 31) / 32;
    const int l0 = min(bnd, a + lane * per), l1 = min(bnd, l0 + per);
    const unsigned long long ls = strided_sum(l0, l1, 0, 1) - rejected(l0, l1);
    unsigned long long inc = ls;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long v = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += v;
    }
    const unsigned long long lbase = base + inc - ls;
    const unsigned hit = __ballot_sync(0xffffffffu, r >= lbase && r < lbase + ls);  // exactly one lane
    const int src = __ffs(hit) - 1;
    a = __shfl_sync(0xffffffffu, l0, src);
    bnd = __shfl_sync(0xffffffffu, l1, src);
    base = __shfl_sync(0xffffffffu, lbase, src);
  }
  const int x = a + lane;
  unsigned long long wv = 0;
  if (x < bnd) {
    wv = raw(x);
    for (int k = 0; k < n_rej; ++k)
      if (s_rej[k] == x) wv = 0;
  }
  unsigned long long inc = wv;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  const unsigned first = __ballot_sync(0xffffffffu, base + inc > r);  // the first token whose inclusive prefix passes r
  if (first != 0u && lane == __ffs(first) - 1) *p.bonus_token = x;
}

}  // namespace dvt

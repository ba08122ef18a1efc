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

constexpr int kVerifyThreads = 256;

__global__ void __launch_bounds__(kVerifyThreads) k_verify_accept(const VerifyAcceptParams p) {
  __shared__ int32_t s_cur, s_nrej, s_rej[kMaxBranch * 4];
  __shared__ unsigned long long s_sum[kVerifyThreads], s_W;
  const int tid = threadIdx.x;
  const int n = *p.n_out;
  if (tid == 0) {
    int cur = -1, na = 0, n_rej = 0;
    for (;;) {
      float rem = 1.0f;
      int found = -1;
      n_rej = 0;
      for (int i = 0; i < n && found < 0; ++i) {
        if (p.parents[i] != cur) continue;
        if (p.mode == 0) {
          if (p.token_ids[i] == p.tgt_argmax[cur + 1]) found = i;
        } else {
          const float lhs = __fmul_rn(p.uniforms[i], rem);  // no contraction: one multiply, one compare
          if (lhs < p.p_cand[i]) found = i;
          else {
            rem = __fsub_rn(rem, p.p_cand[i]);
            if (n_rej < kMaxBranch * 4) s_rej[n_rej] = p.token_ids[i];
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
    if (p.mode == 0) *p.bonus_token = p.tgt_argmax[cur + 1];
  }
  __syncthreads();
  if (p.mode == 0) return;
  // bonus token: integer inverse CDF over the target's distribution at the stopping row, rejected tokens removed
  const float* pr = p.p_full + static_cast<size_t>(s_cur + 1) * p.vocab;
  const int n_rej = s_nrej;
  const int chunk = (p.vocab + kVerifyThreads - 1) / kVerifyThreads;
  const int x0 = min(p.vocab, tid * chunk), x1 = min(p.vocab, x0 + chunk);
  auto weight = [&](int x) -> unsigned long long {
    for (int k = 0; k < n_rej; ++k)
      if (s_rej[k] == x) return 0ull;
    return static_cast<unsigned long long>(__fmul_rn(pr[x], 4294967296.0f));
  };
  unsigned long long mine = 0;
  for (int x = x0; x < x1; ++x) mine += weight(x);
  s_sum[tid] = mine;
  __syncthreads();
  if (tid == 0) {  // exclusive prefix over the 256 chunk sums
    unsigned long long run = 0;
    for (int t = 0; t < kVerifyThreads; ++t) {
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
  const unsigned long long lo = s_sum[tid];
  if (r >= lo && r < lo + mine) {  // exactly one thread's chunk holds the threshold
    unsigned long long acc = lo;
    for (int x = x0; x < x1; ++x) {
      acc += weight(x);
      if (acc > r) { *p.bonus_token = x; break; }
    }
  }
}

}  // namespace dvt

// state.cuh -- device-resident state of one draft step: the per-call values
// (caller pointers, committed length) that kernels read from device memory so
// that the launch sequence itself depends only on (tree_spec, n_new), the row
// tables of the level being forwarded, and the candidate pool.
#pragma once
#include <stdint.h>

namespace dvt {

constexpr int kMaxRows = 64;        // rows of one forward (cfg.max_rows <= 64)
constexpr int kMaxTreeSlots = 128;  // tree rows of one step (cfg.max_tree_slots <= 128)
constexpr int kMaxBranch = 32;
constexpr int kMaskWords = 4;       // 128 bits >= max(kMaxRows, kMaxTreeSlots) new-region slots
constexpr int kMaxDepth = 16;

// Written by k_step_begin from its kernel arguments at the start of every step.
struct StepDyn {
  const float* feats;   // caller's hidden_feats [n_new, d]
  const int32_t* tokens;
  void* kc;             // caller's KV cache
  void* vc;
  int32_t capacity;
  int32_t L;            // committed_len at entry
  int32_t n_new;
  int32_t Lp;           // L + n_new
  int32_t* out_ids;
  float* out_scores;
  int32_t* out_parents;
  int32_t* out_depths;  // nullable
  int32_t* out_n;
};

// Row tables of one level (two sets, alternating by level parity).
struct RowTables {
  int32_t token[kMaxRows];  // token id of the row
  int32_t src[kMaxRows];    // step row whose output hidden state is this row's input feature
  int32_t slot[kMaxRows];   // new-region slot index j: cache row = Lbase + j
  int32_t pool[kMaxRows];   // pool index of the node forwarded at this row (-1 at level 0)
  float cum[kMaxRows];      // that node's cumulative log-probability (0 at level 0)
  uint32_t mask[kMaxRows][kMaskWords];  // new-region slots the row attends (incl. itself)
};

// Candidate pool (O6-O8) and what kv_commit needs from the last step.
struct TreeState {
  int32_t status;  // 0 ok; bit 0: token id out of range (clamped)
  int32_t pool_size;
  int32_t n_out;
  int32_t commit_err;
  int32_t commit_n;
  int32_t commit_src[kMaxDepth + 1];  // tree-row index of each committed path node
};

}  // namespace dvt

/*
 * dovetail.h -- C ABI of libdovetail_draft.so
 *
 * The GPU-side draft step of Dovetail heterogeneous speculative decoding
 * (arxiv 2412.18934), written from the paper for NVIDIA B200 (sm_100a).
 *
 * What the library computes (paper citations are PAPER.md line numbers):
 *   - Dynamic Gating Fusion of the target's hidden feature with the token
 *     embedding: h1 = W1 f, h2 = W2 e, g = sigmoid(Wg [h1 || h2] + bg),
 *     x = g * h1 + (1 - g) * h2                       (Fig. 5 :98)
 *   - the deepened draft decoder stack, n_layers LLaMA blocks, run over the
 *     rows of one level of a draft-token tree with tree attention against the
 *     committed prefix KV cache and the row's tree ancestors
 *
 *   - LM head, per-node top-k expansion, cumulative-probability scoring,
 *     frontier selection for the next round and the final rerank to the
 *     top-gamma candidate set
 *   - the KV bookkeeping after the target has verified the candidates
 *                                                      (last sentence)
 *   - next to the step: prompt / catch-up rows (dovetail_draft_prefill),
 *     the verifier's inputs and the acceptance rule (dovetail_verify_*)
 *
 * How a step is launched: the kernels of one step are captured once per (tree_spec,
 * n_new, attention geometry) into a CUDA graph and replayed on the caller's stream
 * with the per-call pointers and lengths patched in; nothing synchronises with the
 * host. Levels of 1-7 rows stream the weights through k_gemv_mma (mma.sync), levels
 * of 8-64 rows and prefill batches through k_gemv_umma (tcgen05, tensor memory).
 *
 * Conventions
 *   - All functions are extern "C", return 0 on success and a negative
 *     dovetail_status_t on failure. Nothing throws, aborts or calls exit().
 *   - "dev" pointers are CUDA device pointers on the current device of the
 *     calling thread; "host" pointers are ordinary host memory. The library
 *     never takes ownership of caller memory.
 *   - Matrices are row-major [out, in] (y = W x), dtype = cfg.dtype.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = default stream).
 *   - There is no CPU fallback: every entry point fails with DOVETAIL_ECUDA
 *     when no sm_100 device is usable.
 */
#ifndef DOVETAIL_H_
#define DOVETAIL_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DOVETAIL_MAX_DEPTH 16
#define DOVETAIL_MAX_LAYERS 16

typedef enum {
  DOVETAIL_OK = 0,
  DOVETAIL_EINVAL = -1,    /* null pointer, bad shape, bad tree spec, bad path */
  DOVETAIL_ECAPACITY = -2, /* KV cache / tree pool too small for this call     */
  DOVETAIL_ECUDA = -3,     /* CUDA error; text in dovetail_last_error()        */
  DOVETAIL_ENOMEM = -4
} dovetail_status_t;

typedef enum { DOVETAIL_F32 = 0, DOVETAIL_BF16 = 1 } dovetail_dtype_t;

/* Fusion of the target's hidden feature f with the token embedding e.
 *   DGF           the paper's Dynamic Gating Fusion: h1 = W1 f, h2 = W2 e,
 *                 g = sigmoid(Wg [h1 || h2] + bg), x = g * h1 + (1 - g) * h2.
 *   CONCAT_LINEAR the EAGLE-2 fusion DGF replaces ("simply concatenates the two and maps
 *                 them to the hidden state dimension through a single linear transformation",
 *                 PAPER.md:104; ablation row "w/o both", Table 6):
 *                 x = Wfc [f || e] + bfc, with Wfc [d, 2d] passed as dgf_wg and bfc [d] as
 *                 dgf_bg; dgf_w1 / dgf_w2 are ignored (dgf_proj must be 0). */
typedef enum { DOVETAIL_FUSION_DGF = 0, DOVETAIL_FUSION_CONCAT_LINEAR = 1 } dovetail_fusion_t;

/* Model shape. The block is the LLaMA-family decoder layer of the paper's
 * target models: pre-RMSNorm, rotary embedding with half-split
 * pairing (i, i + head_dim/2), grouped-query attention, SiLU-gated FFN, no
 * linear biases. */
typedef struct {
  int32_t hidden;       /* d                                              */
  int32_t n_q_heads;    /* Hq                                             */
  int32_t n_kv_heads;   /* Hkv, divides Hq                                */
  int32_t head_dim;     /* dh, 64 or 128                                  */
  int32_t n_layers;     /* draft Transformer blocks (the paper's M), <= DOVETAIL_MAX_LAYERS */
  int32_t ffn;          /* F                                              */
  int32_t vocab;        /* V <= 2^24 - 2 (token ids travel in 24 bits of a candidate key) */
  float rope_theta;
  float rms_eps;
  int32_t dtype;        /* dovetail_dtype_t of weights, norm gains, bias and KV cache */
  int32_t dgf_proj;     /* 1: W1, W2 present (paper). 0: W1 = W2 = identity          */
  int32_t first_layer_input_norm; /* 1: layer 0 applies its input RMSNorm; 0: skips it */
  int32_t final_norm;   /* 1: RMSNorm(g_final) before the LM head; 0: none           */
  int32_t max_rows;     /* largest n_new and largest beam[] a step may use (<= 64)   */
  int32_t max_tree_slots; /* largest sum over tree levels of forwarded rows (<= 128) */
  int32_t max_branch;   /* largest branch[] a step may use (<= 32)                   */
  int32_t fusion;       /* dovetail_fusion_t: how the feature and the embedding are fused */
  int32_t weight_quant; /* 0: matrices stored in dtype. 1: every weight MATRIX (DGF, blocks, LM head) is int8, row-major
                           [out, in], with one fp32 scale per output row: W[n,k] = scale[n] * q[n,k] ("it is advisable
                           to apply int8 quantization to the drafting model on the GPU"). Needs dtype =
                           BF16 (embedding, norm gains, gate bias, KV cache stay bf16) and every inner dimension a
                           multiple of 32. 2: the same with fp8 e4m3 bytes (the "fn" flavour: no infinities, largest
                           value 448; NaN bytes must not occur) instead of int8: W[n,k] = scale[n] * e4m3(q[n,k])
                           (SURVEY.md 8 f1). */
} dovetail_config_t;

/* Device pointers to one decoder layer's weights. */
typedef struct {
  const void* g_attn; /* [d]        input RMSNorm gain          */
  const void* wq;     /* [Hq*dh, d]                             */
  const void* wk;     /* [Hkv*dh, d]                            */
  const void* wv;     /* [Hkv*dh, d]                            */
  const void* wo;     /* [d, Hq*dh]                             */
  const void* g_ffn;  /* [d]        post-attention RMSNorm gain */
  const void* wgate;  /* [F, d]                                 */
  const void* wup;    /* [F, d]                                 */
  const void* wdown;  /* [d, F]                                 */
  /* weight_quant != 0: fp32 per-row scales of the seven matrices, [out] each; ignored otherwise */
  const float* sq;
  const float* sk;
  const float* sv;
  const float* so;
  const float* sgate;
  const float* sup;
  const float* sdown;
} dovetail_layer_weights_t;

/* Device pointers to all weights. BORROWED: the caller keeps them alive and
 * unchanged for the life of the handle. The struct itself (and layers[]) is
 * host memory and is copied by dovetail_draft_init. */
typedef struct {
  const void* embed;   /* [V, d]  token embedding E                      */
  const void* dgf_w1;  /* [d, d]  hidden-state branch; NULL iff dgf_proj == 0 */
  const void* dgf_w2;  /* [d, d]  embedding branch;    NULL iff dgf_proj == 0 */
  const void* dgf_wg;  /* [d, 2d] gate, input order [h1 || h2]           */
  const void* dgf_bg;  /* [d]     gate bias                              */
  const dovetail_layer_weights_t* layers; /* host array [n_layers]       */
  const void* g_final; /* [d] or NULL (required iff final_norm)          */
  const void* lm_head; /* [V, d]                                         */
  /* weight_quant != 0: fp32 per-row scales of dgf_w1, dgf_w2, dgf_wg, lm_head; ignored otherwise */
  const float* dgf_s1;
  const float* dgf_s2;
  const float* dgf_sg;
  const float* lm_head_s;
} dovetail_weights_t;

/* Draft KV cache, caller-owned device memory.
 *   k, v : [n_layers][n_kv_heads][capacity][head_dim], dtype = cfg.dtype,
 *          K stored AFTER rotary embedding.
 * Rows [0, committed_len) are the committed prefix; dovetail_draft_step writes
 * rows >= committed_len and advances committed_len (see below). The struct
 * lives in host memory. */
typedef struct {
  void* k;
  void* v;
  int32_t capacity;
  int32_t committed_len;
} dovetail_kv_cache_t;

/* Draft tree shape (settings :184).
 *   depth  D >= 1 : number of token levels below the root = number of draft
 *                   forwards per step.
 *   branch[l]     : children kept per expanded node of level l (l = 0 is the
 *                   root, i.e. the last verified token). 1 <= branch <= max_branch.
 *   beam[l], l>=1 : at most this many level-l nodes (best cumulative
 *                   log-probability first) are forwarded and expanded;
 *                   0 = all of them. beam[0] is ignored.
 *   gamma         : number of candidates returned (root excluded).
 * The paper's server preset is depth 7, branch = beam = 10, gamma = 16. */
typedef struct {
  int32_t depth;
  int32_t branch[DOVETAIL_MAX_DEPTH];
  int32_t beam[DOVETAIL_MAX_DEPTH];
  int32_t gamma;
} dovetail_tree_spec_t;

/* Device output buffers of one step, each of capacity >= gamma.
 * Candidates are emitted in pool (topological) order: parents[i] < i or -1
 * (child of the root). scores[i] is the cumulative natural-log probability
 * root -> node ("global acceptance probability"). */
typedef struct {
  int32_t* token_ids; /* dev [gamma]           */
  float* scores;      /* dev [gamma]           */
  int32_t* parents;   /* dev [gamma]           */
  int32_t* depths;    /* dev [gamma] or NULL; level of the node, 1-based */
  int32_t* n_out;     /* dev [1]; = min(gamma, pool size) */
} dovetail_draft_out_t;

typedef struct dovetail_draft dovetail_draft_t;

/* Create a handle: validates cfg, records the borrowed weight pointers and
 * allocates the scratch the step needs (activations in fp32, tree pool,
 * per-CTA partials). Errors: EINVAL, ENOMEM, ECUDA. *out is NULL on failure. */
int dovetail_draft_init(const dovetail_weights_t* w, const dovetail_config_t* cfg,
                        dovetail_draft_t** out);

/* One draft step: D forwards of the draft model and the
 * final rerank, enqueued asynchronously on cuda_stream, no host
 * synchronisation inside.
 *   hidden_feats : dev fp32 [n_new, d]  target hidden states of the n_new
 *                  newly verified tokens (the vector the target's LM head
 *                  consumes), row i paired with tokens[i].
 *   tokens       : dev int32 [n_new]
 *   n_new        : 1 <= n_new <= cfg.max_rows
 * Level 0 runs the n_new rows at positions committed_len + i with causal
 * attention and appends their K/V at those cache rows; the last row's
 * distribution seeds the tree. Tree level l >= 1 runs the selected frontier
 * nodes at position committed_len + n_new + l - 1, each attending the prefix,
 * its tree ancestors and itself; its input feature is the draft's own output
 * hidden state of its parent row. Tree K/V go to cache rows after the prefix.
 * On return (still asynchronous) kv->committed_len has been advanced by n_new.
 * Needs committed_len + n_new + (tree rows) <= capacity, else ECAPACITY.
 * Ties: top-k within a row by (logit desc, token id asc); frontier and final
 * selection by (cumulative score desc, pool index asc).
 * Errors: EINVAL (null pointers, n_new out of range, bad tree spec),
 * ECAPACITY, ECUDA. Every shape of the step (tree plan, GEMV and attention
 * geometry of every level) is checked before the first launch: on EINVAL /
 * ECAPACITY nothing was enqueued and kv is untouched. A token id outside
 * [0, vocab) cannot be seen without reading device memory: the step clamps it,
 * raises a device-side flag and dovetail_draft_status() reports EINVAL. */
int dovetail_draft_step(dovetail_draft_t* h, const float* hidden_feats, const int32_t* tokens,
                        int32_t n_new, dovetail_kv_cache_t* kv, const dovetail_tree_spec_t* tree,
                        const dovetail_draft_out_t* out, void* cuda_stream);

/* Prompt / catch-up rows (the target first processes the prompt and hands
 * its hidden states and tokens to the draft model, which has to build its own K/V over them before the
 * first tree; limitation :274). Runs the draft model over n_rows (feature, token) pairs exactly as
 * dovetail_draft_step runs its level-0 rows -- positions committed_len + i, causal among themselves after
 * the committed prefix -- appends their K/V rows and advances kv->committed_len by n_rows.
 * No LM head and no tree: prefill(rows 0 .. n-2) followed by step(row n-1) equals step(rows 0 .. n-1)
 * (oracle pin P8). n_rows >= 1 is not bounded by cfg.max_rows: the rows run in batches of cfg.max_rows, each
 * batch one pass over the weights (bf16 models: the tcgen05 GEMV, csrc/gemv_umma.cuh).
 *   hidden_feats : dev fp32 [n_rows, d];  tokens : dev int32 [n_rows]
 * Asynchronous on cuda_stream. Errors: EINVAL, ECAPACITY (committed_len + n_rows > capacity), ECUDA; shapes are
 * checked before the first launch. A later dovetail_kv_commit needs a dovetail_draft_step first. */
int dovetail_draft_prefill(dovetail_draft_t* h, const float* hidden_feats, const int32_t* tokens, int32_t n_rows,
                           dovetail_kv_cache_t* kv, void* cuda_stream);

/* After verification: tell the draft which candidates the
 * target accepted.
 *   accepted_path : HOST int32 [n_acc], indices into the last step's output,
 *                   root -> leaf (accepted_path[0] has parent -1, each next
 *                   entry is a child of the previous one). n_acc may be 0.
 *   mode 0 (the paper's flow): the tree K/V rows are discarded; committed_len
 *          is unchanged; the caller feeds the accepted tokens with their true
 *          target features to the next dovetail_draft_step.
 *   mode 1 (extra): the K/V rows of the accepted nodes that were forwarded
 *          during the step are moved to cache rows committed_len.. in path
 *          order and committed_len advances by their count (the leading nodes
 *          of the path; a leaf that was never forwarded has no K/V). The
 *          count is returned in *n_committed (host, may be NULL). This mode
 *          synchronises the stream once to read the device-side validation.
 * Errors: EINVAL (bad path: cache untouched), ECUDA. */
int dovetail_kv_commit(dovetail_draft_t* h, dovetail_kv_cache_t* kv, const int32_t* accepted_path,
                       int32_t n_acc, int32_t mode, int32_t* n_committed, void* cuda_stream);

/* ---- after the draft step: verification bookkeeping and the acceptance rule ----
 * "These candidates are then sent to the target model ... for parallel verification. The target model
 * computes the logits of the candidate tokens in a single forward pass and applies a speculative sampling
 * algorithm to determine the accepted tokens."
 * Verifier rows: row 0 is the root (the last verified token, which the target has not forwarded yet), row
 * i + 1 is candidate i of the step's output. gamma = capacity of the step's output arrays. */

/* Device buffers of what the verifier's single forward needs. */
typedef struct {
  uint8_t* mask;         /* dev [(gamma+1) x (gamma+1)] row-major; mask[r][c] = 1 iff row c is r or an ancestor of r */
  int32_t* position_ids; /* dev [gamma+1]; root_position + depth (root depth 0)                                    */
  int32_t* paths;        /* dev [gamma x max_depth]; candidate indices root -> leaf of every leaf, padded with -1   */
  int32_t* n_paths;      /* dev [1]                                                                                */
} dovetail_verify_plan_t;

/* Fills plan from the last step's output (token tree in pool order). Rows past n_out are zero / -1.
 * Asynchronous on cuda_stream. Errors: EINVAL (null pointers, gamma < 1, max_depth < 1), ECUDA. */
int dovetail_verify_plan(dovetail_draft_t* h, const dovetail_draft_out_t* out, int32_t gamma,
                         int32_t root_position, int32_t max_depth, const dovetail_verify_plan_t* plan,
                         void* cuda_stream);

/* The target's answer, device memory. mode 0 needs tgt_argmax; mode 1 the other three. */
typedef struct {
  const int32_t* tgt_argmax; /* dev [gamma+1] the target's argmax token at every verifier row              */
  const float* p_cand;       /* dev [gamma] target probability of candidate i's token at its parent's row  */
  const float* uniforms;     /* dev [gamma+1] U[0,1): one per candidate, then one for the bonus token      */
  const float* p_full;       /* dev [gamma+1][vocab] the target's distribution at every verifier row       */
} dovetail_verify_in_t;

typedef struct {
  int32_t* accepted_path; /* dev [max_depth] candidate indices root -> last accepted node (input of kv_commit) */
  int32_t* n_acc;         /* dev [1]                                                                          */
  int32_t* bonus_token;   /* dev [1] the target's own next token after the accepted path; -1: no mass left   */
} dovetail_verify_out_t;

/* The acceptance rule. Walks down from the root; at each node its children are tried in candidate order.
 *   mode 0, greedy (T = 0): a child is accepted iff its token is the target's argmax at the parent's row;
 *           bonus token = the argmax at the last accepted row.
 *   mode 1, speculative sampling (T = 1): the draft tree is a deterministic top-k expansion, so every child
 *           is a point-mass proposal: it is accepted with probability p_cand / rem, rem = 1 - the target
 *           probability of the siblings already rejected at that node (decision: uniforms[i] * rem < p_cand[i]
 *           in fp32); the bonus token is drawn with uniforms[n_out] from p_full at the last accepted row with
 *           the rejected children's tokens removed. The emitted tokens follow the target's distribution exactly.
 * Asynchronous on cuda_stream; copy accepted_path / n_acc to the host for dovetail_kv_commit.
 * Errors: EINVAL (null pointers for the chosen mode, bad mode, gamma < 1, max_depth < 1), ECUDA. */
int dovetail_verify_accept(dovetail_draft_t* h, const dovetail_draft_out_t* out, int32_t gamma, int32_t mode,
                           int32_t max_depth, const dovetail_verify_in_t* in, const dovetail_verify_out_t* res,
                           void* cuda_stream);

/* Tree bookkeeping alone, for bit-exact checks of the
 * integer path: replays expansion, scoring, frontier selection and the final
 * rerank from caller-supplied per-row top-k lists instead of LM-head results.
 *   cand_tokens, cand_logp : dev [n_rows, max_b] with max_b = max over levels
 *        of branch[l]; row 0 is the root's list, then the forwarded rows of
 *        level 1, level 2, ... in frontier order; entries sorted as the LM-head
 *        stage would emit them (log-prob desc, token id asc).
 * Writes out like dovetail_draft_step and, when non-NULL, the pool arrays
 * (dev, capacity >= pool size): token, parent pool index, depth, cumulative
 * score, and pool_size[1]. Asynchronous on cuda_stream. */
int dovetail_tree_replay(dovetail_draft_t* h, const dovetail_tree_spec_t* tree,
                         const int32_t* cand_tokens, const float* cand_logp, int32_t n_rows,
                         int32_t max_b, const dovetail_draft_out_t* out, int32_t* pool_token,
                         int32_t* pool_parent, int32_t* pool_depth, float* pool_cum,
                         int32_t* pool_size, void* cuda_stream);

/* The same tree bookkeeping (PAPER.md:94 expansion and cumulative scores, :100
 * reduction to the gamma candidates) for callers that cannot allocate: code
 * under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc. No handle, no dovetail_draft_init: the candidate pool, the row
 * tables, the ancestor masks and the bookkeeping state live in ONE file-scope
 * device array of DOVETAIL_STATIC_SCRATCH_BYTES inside the library (every GPU
 * that loads the library holds it until the process exits). The call itself
 * allocates nothing (no cudaMalloc / cudaFree / allocating library routine):
 * it enqueues two cudaMemsetAsync and one k_tree_level launch per level.
 *   cand_tokens, cand_logp, n_rows, max_b, out: as for dovetail_tree_replay
 *        (device memory, caller-owned; out->depths may be NULL).
 * Limits (beyond them: DOVETAIL_EINVAL and a message naming the limit, nothing
 * is enqueued): depth <= DOVETAIL_MAX_DEPTH, branch[l] <= 32, rows forwarded
 * per level <= 64, tree rows <= 128, candidate pool
 * sum_l rows_l * branch[l] <= DOVETAIL_STATIC_MAX_POOL (half of what a handle
 * can hold; the paper's own tree, width 10 / depth 7, needs 610).
 * The array is shared by every call on the device and keeps the previous call's
 * contents; the call clears what has to start clean (level-0 row table,
 * bookkeeping state) on cuda_stream before the first launch. Two calls that
 * overlap on the GPU (different streams, or graphs replayed concurrently) RACE
 * on it: serialise them. The device current at the call must be the stream's;
 * the array's address is resolved once per device, at the first call there
 * (make that call outside stream capture).
 * Asynchronous on cuda_stream. Errors: EINVAL (null pointers, limits, lists too
 * short), ECUDA (no device, symbol lookup or launch failure);
 * dovetail_last_error(NULL) holds the message. */
#define DOVETAIL_STATIC_MAX_POOL 2048
#define DOVETAIL_STATIC_SCRATCH_BYTES 65536
int dovetail_tree_replay_static(const dovetail_tree_spec_t* tree, const int32_t* cand_tokens,
                                const float* cand_logp, int32_t n_rows, int32_t max_b,
                                const dovetail_draft_out_t* out, void* cuda_stream);

/* Result of the device-side input checks of the steps enqueued so far on this
 * handle (the step consumes the accepted tokens; a token id outside
 * [0, vocab) has no embedding row). dovetail_draft_step itself never
 * synchronises, so the check is reported here: the call synchronises
 * cuda_stream, reads the device-side status word and clears it.
 * Returns OK, EINVAL (a token id of a step since the last call was out of
 * range: that step gathered a clamped embedding row and its candidates are
 * meaningless) or ECUDA. */
int dovetail_draft_status(dovetail_draft_t* h, void* cuda_stream);

/* Number of kernel launches the last dovetail_draft_step enqueued. */
int dovetail_last_launch_count(const dovetail_draft_t* h);

/* Algorithmic HBM bytes of one forward over the given prefix length: all
 * weight bytes + prefix K/V bytes. */
int64_t dovetail_forward_bytes(const dovetail_draft_t* h, int32_t prefix_len);

void dovetail_draft_destroy(dovetail_draft_t* h);

/* Text of the last error on this handle (or of the last failed init when
 * h == NULL). Never NULL; valid until the next call on the same handle. */
const char* dovetail_last_error(const dovetail_draft_t* h);

#ifdef __cplusplus
}
#endif
#endif /* DOVETAIL_H_ */

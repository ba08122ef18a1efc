// dovetail_draft.cu -- host side of libdovetail_draft.so: the C ABI declared in
// include/dovetail.h. It validates arguments, owns the scratch buffers and
// enqueues the kernels of one draft step on the caller's
// stream; every step of the method runs in the kernels of gemv.cuh,
// attention.cuh and tree.cuh. There is no CPU fallback.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>  // header-only; a no-op unless a profiler injects itself

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/dovetail.h"
#include "../../include/dovetail_hooks.h"
#include "attention.cuh"
#include "attention_mma.cuh"
#include "gemv.cuh"
#include "gemv_mma.cuh"
#include "gemv_umma.cuh"
#include "state.cuh"
#include "stream_probe.cuh"
#include "tree.cuh"
#include "verify.cuh"

using namespace dvt;

namespace {

constexpr int kSmemBudget = 200 * 1024;  // dynamic shared memory a GEMV CTA may use
constexpr int kSmemMax = 227 * 1024;
constexpr int kAttnStages = 4;

char g_init_error[512] = "no error";

// NVTX range over one entry point (traces of the step / prefill / commit in a timeline profiler).
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};

struct LevelPlan {
  int rows;        // rows forwarded at this level (level 0: n_new)
  int rows_lm;     // rows whose LM-head lists are expanded (level 0: 1)
  int row0;        // first step row
  int t0;          // first tree-row index (levels >= 1)
  int pool_begin;  // pool index of the level's first child
};

}  // namespace

struct dovetail_draft {
  dovetail_config_t cfg;
  dovetail_weights_t w;
  std::vector<dovetail_layer_weights_t> layers;
  int num_sms = 0, es = 2;
  int wq = 0;  // 1: int8, 2: fp8 e4m3 weight matrices with per-row scales (cfg.weight_quant)
  __nv_bfloat16* xs_emb = nullptr;  // int8: embedding rows of the level, as a (permuted) plane [1][rows][ld_d]
  int dq = 0, dkv = 0, ldq = 0;
  int max_step_rows = 0, pool_cap = 0, attn_chunks_cap = 1, qv_cap = 1;
  // device scratch (owned)
  StepDyn* dyn = nullptr;
  TreeState* ts = nullptr;
  RowTables* rt = nullptr;  // [2]
  float2* rope = nullptr;
  double* inv_freq = nullptr;
  float *hbuf = nullptr, *hhat = nullptr, *qkv = nullptr, *obuf = nullptr, *act = nullptr;
  // split-bf16 planes of the activations, the B operands of the tensor-core GEMV (epilogue.cuh): [3][rows][ld]
  __nv_bfloat16 *xs_feat = nullptr, *xs_hhat = nullptr, *xs_x = nullptr, *xs_h12 = nullptr, *xs_o = nullptr, *xs_act = nullptr;
  int ld_d = 0, ld_2d = 0, ld_dq = 0, ld_f = 0;  // row strides (elements, multiples of 8)
  float* ssq = nullptr;  // [num_sms][kMaxRows] partial sums of squares of the residual stream
  __nv_bfloat16* qs = nullptr;  // [2][kMaxRows][dq] rotated, scaled queries (bf16 head + remainder), gemv.cuh EPI_QKV
  float* attn_ws = nullptr;
  int32_t* attn_cnt = nullptr;
  float* cand_val = nullptr;
  int32_t* cand_id = nullptr;
  float* stat = nullptr;
  Pool pool{};
  uint32_t* treemask = nullptr;
  int32_t* out_pool_idx = nullptr;
  TreeState* ts_host = nullptr;  // pinned
  // test / measurement hooks (dovetail_hooks.h); never set in a plain step
  dovetail_hooks_t hooks{};
  bool hooks_on = false;
  // last step
  bool have_step = false;
  int last_n_new = 0, last_depth = 0, last_gamma = 0;
  int last_launches = 0;
  int launches = 0;
  int umma_launches = 0, last_umma_launches = 0;
  int ksplit_launches = 0, last_ksplit_launches = 0;
  bool dry = false;  // shape-checking pass of dovetail_draft_step: nothing is launched
  // GEMVs queued by run_gemv, launched by flush_gemv
  struct QueuedGemv { GemvParams p; int n_groups, ctas, kind, max_cnt; int64_t bytes; };
  std::vector<QueuedGemv> queue;
  // tcgen05 GEMV (gemv_umma.cuh): tensor maps of the weight matrices and activation planes (four box depths
  // each: 1, 2, 4, 8 slabs of 64 k), row tables of every dealing seen so far
  int umma_min_m = 8;               // levels of at least this many rows take the tcgen05 kernel (65: never)
  int attn_max_clusters[3][9] = {};  // [mode][cluster size]: clusters of the attention kernel resident at once
  int umma_ksplit_min_m = 48;       // levels of at least this many rows split K over CTA pairs whatever the tile (65: never)
  int attn_qt2 = 1;                 // 17 ... 32 query vectors take the 32-per-pass attention kernel
  int attn_wide_min = 32;           // levels with more query vectors (rows x q-heads per kv-head) take the wide attention kernel
  CUtensorMap* maps_dev = nullptr;  // [n_maps][4]
  std::map<const void*, int> wmap_of;  // weight matrix -> first map index
  struct PlaneBuf { const __nv_bfloat16* base; int64_t elems, ld; int cap, map; };
  std::vector<PlaneBuf> plane_bufs;
  struct UmmaTable { UmmaCtaTab* tab = nullptr; uint16_t* vpos = nullptr; int vpos_ld = 0, g_max = 0, g_min = 0; bool ok = false;
                     int pair_max = 0, pair_min = 0; };  // K split over CTA pairs: boxes of CTAs 2i and 2i + 1 together (0: not eligible)
  std::map<std::array<int, 8>, UmmaTable> umma_tabs;
  __nv_bfloat16* xs_par = nullptr;  // [3][max_rows][ld_d] parent hidden states of a wide level, gathered
  // One CUDA graph per (tree_spec, n_new, attention geometry): the step's launch sequence with its
  // programmatic edges, replayed with the per-call values patched into the nodes that take them as arguments
  // (k_step_begin: caller pointers and lengths; tensor-core attention: cache pointers and lengths).
  struct StepGraph {
    std::vector<int> key;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaGraphNode_t begin_node = nullptr;
    cudaKernelNodeParams begin_params{};
    std::vector<void*> begin_args;
    StepDyn begin_dv{};
    std::vector<cudaGraphNode_t> attn_nodes;
    std::vector<cudaKernelNodeParams> attn_node_params;
    std::vector<AttnParams> attn_params;
    int launches = 0, umma_launches = 0;
    unsigned long long used = 0;
  };
  bool graphs_on = true;
  std::vector<StepGraph> graphs;
  unsigned long long graph_clock = 0;
  cudaStream_t cap_stream = nullptr;
  int last_graph = 0;  // 1: the last step was a graph replay, 2: captured and launched, 0: direct launches
#ifdef DVT_CHAINDBG
  unsigned long long* dbg = nullptr;
  int dbg_launch = 0;
#endif
  // per-launch time stamps (dovetail_trace_*)
  bool trace_on = false;
  unsigned long long* trace_buf = nullptr;  // device [kMaxTraceLaunches][2]
  unsigned long long* trace_host = nullptr; // pinned
  int cur_kind = 0;
  int64_t cur_bytes = 0;
  int cur_level = 0;
  float* probe_sink = nullptr;
  std::vector<int> tr_kind, tr_level;
  std::vector<int64_t> tr_bytes;
  int tr_used = 0;
  char err[512] = "no error";
};

namespace {

int fail(dovetail_draft* h, int code, const char* fmt, ...) {
  char* dst = h ? h->err : g_init_error;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 512, fmt, ap);
  va_end(ap);
  return code;
}

// ---- launch helper: every kernel is launched with the programmatic-stream-
// serialization attribute so that its prologue / weight prefetch overlaps the
// tail of its predecessor; the kernels call griddepcontrol.wait themselves.
constexpr int kMaxTraceLaunches = 4096;

// Time-stamp slot of the launch about to be made (NULL unless tracing); records its kind / bytes.
unsigned long long* trace_slot(dovetail_draft* h) {
  if (!h->trace_on || h->dry || h->tr_used >= kMaxTraceLaunches) return nullptr;
  const int i = h->tr_used;
  if (static_cast<int>(h->tr_kind.size()) <= i) { h->tr_kind.resize(i + 1); h->tr_level.resize(i + 1); h->tr_bytes.resize(i + 1); }
  h->tr_kind[i] = h->cur_kind;
  h->tr_level[i] = h->cur_level;
  h->tr_bytes[i] = h->cur_bytes;
  h->tr_used = i + 1;
  return h->trace_buf + 2 * static_cast<size_t>(i);
}

template <typename... KArgs, typename... Args>
cudaError_t launch_c(dovetail_draft* h, int cluster_x, bool pdl, void (*kern)(KArgs...), dim3 grid, dim3 block,
                     size_t smem, cudaStream_t st, Args... args) {
  if (h->dry) return cudaSuccess;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  int na = 0;
  if (pdl) {
    attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
  }
  if (cluster_x > 1) {  // thread-block cluster along x (attention chunks)
    attr[na].id = cudaLaunchAttributeClusterDimension;
    attr[na].val.clusterDim.x = cluster_x;
    attr[na].val.clusterDim.y = 1;
    attr[na].val.clusterDim.z = 1;
    ++na;
  }
  cfg.attrs = attr;
  cfg.numAttrs = na;
  ++h->launches;
  return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

template <typename... KArgs, typename... Args>
cudaError_t launch(dovetail_draft* h, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem,
                   cudaStream_t st, Args... args) {
  return launch_c(h, 1, true, kern, grid, block, smem, st, args...);
}

using GemvKernel = void (*)(const GemvParams);
using MmaKernel = void (*)(const MmaParams);

template <typename WT>
GemvKernel pick_gemv(int MT, int NI) {
  if (NI == 3) {
    if (MT == 1) return k_gemv<WT, 1, 3>;
    if (MT == 2) return k_gemv<WT, 2, 3>;
    return k_gemv<WT, 4, 3>;
  }
  if (MT == 1) return k_gemv<WT, 1, 7>;
  return k_gemv<WT, 2, 7>;
}

MmaKernel pick_gemv_mma(int NT, int wq) {
  if (wq == 2) {
    if (NT == 1) return k_gemv_mma<1, 4, 2>;
    if (NT == 2) return k_gemv_mma<2, 4, 2>;
    if (NT == 4) return k_gemv_mma<4, 4, 2>;
    return k_gemv_mma<8, 2, 2>;
  }
  if (wq) {
    if (NT == 1) return k_gemv_mma<1, 4, 1>;
    if (NT == 2) return k_gemv_mma<2, 4, 1>;
    if (NT == 4) return k_gemv_mma<4, 4, 1>;
    return k_gemv_mma<8, 2, 1>;
  }
  if (NT == 1) return k_gemv_mma<1, 4, 0>;
  if (NT == 2) return k_gemv_mma<2, 4, 0>;
  if (NT == 4) return k_gemv_mma<4, 4, 0>;
  return k_gemv_mma<8, 2, 0>;
}

using AttnKernel = void (*)(const AttnParams);

template <typename WT, int DH>
AttnKernel pick_attn_qt(int QT) {
  if (QT == 1) return k_tree_attention<WT, DH, 1>;
  if (QT == 2) return k_tree_attention<WT, DH, 2>;
  return k_tree_attention<WT, DH, 4>;
}

AttnKernel pick_attn(int dtype, int dh, int QT) {
  if (dtype == DOVETAIL_BF16)
    return dh == 128 ? pick_attn_qt<__nv_bfloat16, 128>(QT) : pick_attn_qt<__nv_bfloat16, 64>(QT);
  return dh == 128 ? pick_attn_qt<float, 128>(QT) : pick_attn_qt<float, 64>(QT);
}

cudaError_t set_max_smem_all() {
  cudaError_t e = cudaSuccess;
  auto set = [&](const void* f) {
    cudaError_t r = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
    if (r != cudaSuccess) e = r;
  };
  for (int nt = 1; nt <= 8; nt *= 2)
    for (int wq = 0; wq < 3; ++wq) set(reinterpret_cast<const void*>(pick_gemv_mma(nt, wq)));
  set(reinterpret_cast<const void*>(k_gemv_umma));
  set(reinterpret_cast<const void*>(k_tree_attention_mma<64, 1>));
  set(reinterpret_cast<const void*>(k_tree_attention_mma<128, 1>));
  set(reinterpret_cast<const void*>(k_tree_attention_mma<64, 2>));
  set(reinterpret_cast<const void*>(k_tree_attention_mma<128, 2>));
  set(reinterpret_cast<const void*>(k_tree_attention_mma<64, 4>));
  set(reinterpret_cast<const void*>(k_tree_attention_mma<128, 4>));
  const int mts[3] = {1, 2, 4};
  for (int mt : mts) {
    set(reinterpret_cast<const void*>(pick_gemv<__nv_bfloat16>(mt, 3)));
    set(reinterpret_cast<const void*>(pick_gemv<float>(mt, 3)));
    if (mt <= 2) {
      set(reinterpret_cast<const void*>(pick_gemv<__nv_bfloat16>(mt, 7)));
      set(reinterpret_cast<const void*>(pick_gemv<float>(mt, 7)));
    }
    for (int dt = 0; dt < 2; ++dt)
      for (int dh = 64; dh <= 128; dh += 64) set(reinterpret_cast<const void*>(pick_attn(dt, dh, mt)));
  }
  return e;
}

// How the GEMV of a [N, K] matrix is staged: rows per stage, ring depth, tile of draft rows.
struct GemvShape {
  int row_bytes, rows_per_stage, stage_bytes, n_stages, MT, NI, smem;
  bool ok;
};

GemvShape gemv_shape(int K, int es, int M, int res_rows) {
  GemvShape s{};
  s.row_bytes = K * es;
  const int units = s.row_bytes / 16;
  const int ni = (units + kConsumerThreads - 1) / kConsumerThreads;
  s.ok = (s.row_bytes % 16 == 0) && ni <= 7;
  s.NI = ni <= 3 ? 3 : 7;
  s.MT = M == 1 ? 1 : (M == 2 ? 2 : (s.NI == 7 ? 2 : 4));
  s.rows_per_stage = 32768 / s.row_bytes;
  if (s.rows_per_stage < 1) s.rows_per_stage = 1;
  if (s.rows_per_stage > kRowsPerStageMax) s.rows_per_stage = kRowsPerStageMax;
  s.stage_bytes = s.rows_per_stage * s.row_bytes;
  const int fixed = 128 /*barriers*/ + 2 * kConsumerWarps * 16 * 4 /*part*/ + 16 + kConsumerWarps * 16 +
                    res_rows * s.MT * 4 + 128;
  s.n_stages = (kSmemBudget - fixed) / s.stage_bytes;
  if (s.n_stages > 8) s.n_stages = 8;
  if (s.n_stages < 2) s.ok = false;
  s.smem = s.n_stages * s.stage_bytes + fixed;
  return s;
}

int div_up(int a, int b) { return (a + b - 1) / b; }

// Geometry of one launch of the tensor-core GEMV kernel (gemv_mma.cuh).
struct MmaGeom {
  int NT, RBMAX, RS, stage_bytes, n_stages, part_floats, res_floats, smem;
  int S, KC, seg_stride, aseg_stride, RSp;
  bool ok;
};

int nt_for(int cols) {
  int t = (cols + 7) / 8, r = 1;
  while (r < t) r *= 2;
  return r;
}

// wq: int8 weights (one byte per element in the A part of a stage)
MmaGeom mma_geom(const dovetail_draft::QueuedGemv& q, int wq) {
  MmaGeom s{};
  const int aes = wq ? 1 : 2;
  const int K = q.p.K, M = q.p.M;
  s.ok = K % 32 == 0 && M >= 1 && M <= kMmaMaxM && q.max_cnt >= 1;
  if (!s.ok) return s;
  const int nt2 = nt_for(2 * M), nt3 = nt_for(3 * M);
  s.S = nt3 == nt2 ? 3 : 2;  // the exact 3-way split when it costs no extra column tile
  if (q.p.g[0].S_fixed) s.S = std::max(s.S, q.p.g[0].S_fixed);
  const int nt = nt2, max_cnt = q.max_cnt, res_floats = q.max_cnt * M;
  if (nt > 8) { s.ok = false; return s; }
  s.NT = nt;
  s.RBMAX = nt == 8 ? 2 : 4;
  // Rows per stage and K-chunk: the first candidate that leaves a ring of >= 3 stages or >= 120 KB (else the
  // deepest ring found). A stage holds RS weight rows and M * S activation columns of one K-chunk. Wide levels
  // take the smaller stages: their B columns and partial buffers use most of the shared memory.
  const int rs_max = std::min(16 * s.RBMAX, (max_cnt + 15) / 16 * 16);
  const int ncols = M * s.S, PC = (ncols + 1) & ~1;
  MmaGeom best{};
  for (int rs = rs_max; rs >= 16; rs -= 16) {
    // rows a stage really carries: the CTA's rows in balanced super-blocks of <= rs rows
    const int nsb = div_up(max_cnt, rs), rows_eff = std::min(rs, div_up(max_cnt, nsb));
    for (int kc0 : {wq ? 1024 : 512, wq ? 512 : 256, wq ? 256 : 128}) {
      MmaGeom c = s;
      c.RS = rs;
      c.KC = std::min(kc0, (K + 63) / 64 * 64);
      c.part_floats = kConsumerWarps * rs * PC;
      // matrices with few rows per CTA (O, down: 35 of 64) take longer K-chunks so that their stages are full too
      const int full_stage = rs * (c.KC * aes + 16) + ncols * (c.KC * 2 + 16);
      while (c.KC < 2048 * (wq ? 2 : 1) && c.KC * 2 <= (K + 63) / 64 * 64 &&
             rows_eff * (c.KC * 2 * aes + 16) + ncols * (c.KC * 4 + 16) <= full_stage + 4096)
        c.KC *= 2;
      c.seg_stride = c.KC * 2 + 16;
      c.aseg_stride = c.KC * aes + 16;
      c.stage_bytes = rows_eff * c.aseg_stride + ncols * c.seg_stride;
      c.RSp = rows_eff;
      if (c.part_floats * 4 > 32768 && rs > 16) continue;
      c.res_floats = res_floats;
      int fixed = 3 * 64 + 16 + 2 * 4 * kMmaMaxM + c.part_floats * 4 + res_floats * 4 + (wq ? max_cnt * 4 : 0);
      fixed = (fixed + 15) / 16 * 16;
      c.n_stages = std::min(8, (kSmemMax - fixed - 64) / c.stage_bytes);
      c.smem = c.n_stages * c.stage_bytes + fixed;
      c.ok = c.n_stages >= 2;
      if (!c.ok) continue;
      if (c.n_stages >= 3 || c.n_stages * c.stage_bytes >= 120 * 1024) return c;  // two 66 KB stages stream as well as four 33 KB ones
      if (!best.ok || c.n_stages * c.stage_bytes > best.n_stages * best.stage_bytes) best = c;
    }
  }
  return best;
}


// ---- tcgen05 GEMV (gemv_umma.cuh): tensor maps, row tables, launch geometry --------------------------------
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// The library links only the CUDA runtime; the driver's tensor-map encoder is fetched through it.
EncodeTiledFn tensor_map_encoder() {
  void* f = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
      q != cudaDriverEntryPointSuccess)
    return nullptr;
  return reinterpret_cast<EncodeTiledFn>(f);
}

// Four maps (boxes of 1, 2, 4, 8 slabs) of a bf16 matrix [rows][ld], ld a multiple of 64: dimensions (k within a
// 64-element slab, row, slab) with strides (2 ld, 128) bytes, box (64, 8, nslab), 128-byte swizzle: one copy
// lands as nslab swizzle atoms [slab][8 rows][128 B] (gemv_umma.cuh).
bool encode_maps(EncodeTiledFn enc, const void* base, int64_t rows, int64_t ld, std::vector<CUtensorMap>& out) {
  for (int i = 0; i < 4; ++i) {
    CUtensorMap m;
    memset(&m, 0, sizeof m);
    const int nslab = 1 << i;
    if ((ld / 64) % nslab == 0) {
      const cuuint64_t dims[3] = {64, static_cast<cuuint64_t>(rows), static_cast<cuuint64_t>(ld / 64)};
      const cuuint64_t strides[2] = {static_cast<cuuint64_t>(ld) * 2, 128};
      const cuuint32_t box[3] = {64, 8, static_cast<cuuint32_t>(nslab)};
      const cuuint32_t es[3] = {1, 1, 1};
      if (enc(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    }
    out.push_back(m);
  }
  return true;
}

// Called once by dovetail_draft_init (bf16 weights). On any failure the tcgen05 path stays off and every level
// runs on k_gemv_mma.
void umma_init(dovetail_draft* h) {
  h->umma_min_m = kUmmaMaxM + 1;
  EncodeTiledFn enc = tensor_map_encoder();
  if (!enc) return;
  const dovetail_config_t& c = h->cfg;
  std::vector<CUtensorMap> maps;
  bool ok = true;
  auto add_w = [&](const void* w, int rows, int K) {
    if (!w || K % 64 != 0 || h->wmap_of.count(w)) return;
    h->wmap_of[w] = static_cast<int>(maps.size());
    ok = ok && encode_maps(enc, w, rows, K, maps);
  };
  const int d = c.hidden;
  add_w(h->w.dgf_w1, d, d);
  add_w(h->w.dgf_w2, d, d);
  add_w(h->w.dgf_wg, d, 2 * d);
  add_w(h->w.lm_head, c.vocab, d);
  for (const dovetail_layer_weights_t& L : h->layers) {
    add_w(L.wq, h->dq, d); add_w(L.wk, h->dkv, d); add_w(L.wv, h->dkv, d); add_w(L.wo, d, h->dq);
    add_w(L.wgate, c.ffn, d); add_w(L.wup, c.ffn, d); add_w(L.wdown, d, c.ffn);
  }
  auto add_x = [&](const __nv_bfloat16* xs, int cap, int ld) {
    if (!xs || ld % 64 != 0) return;
    dovetail_draft::PlaneBuf b{xs, static_cast<int64_t>(kSplitPlanes) * cap * ld, ld, cap, static_cast<int>(maps.size())};
    ok = ok && encode_maps(enc, xs, static_cast<int64_t>(kSplitPlanes) * cap, ld, maps);
    h->plane_bufs.push_back(b);
  };
  const int R = c.max_rows;
  add_x(h->xs_feat, R, h->ld_d); add_x(h->xs_hhat, h->max_step_rows, h->ld_d); add_x(h->xs_x, R, h->ld_d);
  add_x(h->xs_h12, R, h->ld_2d); add_x(h->xs_o, R, h->ld_dq); add_x(h->xs_act, R, h->ld_f);
  add_x(h->xs_emb, R, h->ld_d); add_x(h->xs_par, R, h->ld_d);
  if (!ok || maps.empty()) return;
  if (cudaMalloc(reinterpret_cast<void**>(&h->maps_dev), maps.size() * sizeof(CUtensorMap)) != cudaSuccess) { cudaGetLastError(); return; }
  if (cudaMemcpy(h->maps_dev, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice) != cudaSuccess) { cudaGetLastError(); return; }
  h->umma_min_m = 8;  // measured on the 13B shape: 257 vs 263 us per forward at 8 rows, 296 vs 279 at 6
}

// Row tables of one dealing (gemv_umma.cuh UmmaCtaTab): the CTA's virtual rows sorted into contiguous memory
// segments, each cut into 8-row boxes; boxes dealt to balanced super-blocks of <= 16 boxes.
// Pure host logic (tested on the CPU through dovetail_hooks_umma_tables): fills tabs[ctas] and vpos[ctas * vpos_ld].
// Returns false when a CTA would need more than kUmmaMaxSb super-blocks.
bool build_umma_tables(const GemvGroup& G, int ctas, std::vector<UmmaCtaTab>& tabs, std::vector<uint16_t>& vpos, int& vpos_ld,
                       int& g_max, int& g_min) {
  int max_cnt = 0;
  for (int c = 0; c < ctas; ++c) max_cnt = std::max(max_cnt, static_cast<int>(cta_rows(G, c, ctas).cnt));
  vpos_ld = (max_cnt + 7) / 8 * 8;
  tabs.assign(ctas, UmmaCtaTab{});
  vpos.assign(static_cast<size_t>(ctas) * std::max(1, vpos_ld), 0);
  g_max = 0;
  g_min = kUmmaMaxGroups;
  if (max_cnt <= 0) return false;
  for (int c = 0; c < ctas; ++c) {
    const RowRange rr = cta_rows(G, c, ctas);
    UmmaCtaTab& T = tabs[c];
    if (rr.cnt == 0) continue;
    std::vector<std::array<int, 3>> rows(rr.cnt);
    for (int v = 0; v < rr.cnt; ++v) {
      int j, n;
      locate_row(G, rr, v, j, n);
      rows[v] = {j, n, v};
    }
    std::sort(rows.begin(), rows.end());
    std::vector<int> gcode;
    std::vector<std::pair<int, int>> pos(rr.cnt);
    for (int i = 0; i < rr.cnt;) {
      int e = i + 1;
      while (e < rr.cnt && rows[e][0] == rows[i][0] && rows[e][1] == rows[e - 1][1] + 1) ++e;
      for (int off = i; off < e; off += 8) {
        const int g = static_cast<int>(gcode.size());
        gcode.push_back((rows[off][0] << 28) | rows[off][1]);
        for (int r = 0; r < 8 && off + r < e; ++r) pos[rows[off + r][2]] = {g, r};
      }
      i = e;
    }
    const int Gt = static_cast<int>(gcode.size());
    const int n_sb = div_up(Gt, kUmmaMaxGroups), per = div_up(Gt, n_sb);
    if (n_sb > kUmmaMaxSb) return false;
    T.n_sb = n_sb;
    for (int g = 0; g < Gt; ++g) {
      T.grp[g / per][g % per] = gcode[g];
      T.n_grp[g / per] = g % per + 1;
    }
    for (int sb = 0; sb < n_sb; ++sb) { g_max = std::max(g_max, T.n_grp[sb]); g_min = std::min(g_min, T.n_grp[sb]); }
    for (int v = 0; v < rr.cnt; ++v)
      vpos[static_cast<size_t>(c) * vpos_ld + v] = static_cast<uint16_t>((pos[v].first / per) * 128 + (pos[v].first % per) * 8 + pos[v].second);
  }
  return true;
}

const dovetail_draft::UmmaTable& umma_table(dovetail_draft* h, const GemvGroup& G, int ctas) {
  const std::array<int, 8> key = {G.rows[0], G.n_mat > 1 ? G.rows[1] : 0, G.n_mat > 2 ? G.rows[2] : 0, G.n_mat, G.paired,
                                  G.pairperm, ctas, G.deal_base};
  auto it = h->umma_tabs.find(key);
  if (it != h->umma_tabs.end()) return it->second;
  dovetail_draft::UmmaTable t;
  std::vector<UmmaCtaTab> tabs;
  std::vector<uint16_t> vpos;
  bool ok = build_umma_tables(G, ctas, tabs, vpos, t.vpos_ld, t.g_max, t.g_min);
  if (ok && ctas % 2 == 0) {  // pairs (2i, 2i + 1) of single-super-block CTAs whose boxes fit one tile together
    t.pair_max = 0;
    t.pair_min = 2 * kUmmaMaxGroups;
    for (int c = 0; c < ctas; c += 2) {
      if (tabs[c].n_sb != 1 || tabs[c + 1].n_sb != 1) { t.pair_max = 0; break; }
      const int g2 = tabs[c].n_grp[0] + tabs[c + 1].n_grp[0];
      t.pair_max = std::max(t.pair_max, g2);
      t.pair_min = std::min(t.pair_min, g2);
    }
    if (t.pair_max > kUmmaMaxGroups) t.pair_max = 0;
  }
  if (ok) {
    ok = cudaMalloc(reinterpret_cast<void**>(&t.tab), tabs.size() * sizeof(UmmaCtaTab)) == cudaSuccess &&
         cudaMalloc(reinterpret_cast<void**>(&t.vpos), vpos.size() * sizeof(uint16_t)) == cudaSuccess &&
         cudaMemcpy(t.tab, tabs.data(), tabs.size() * sizeof(UmmaCtaTab), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(t.vpos, vpos.data(), vpos.size() * sizeof(uint16_t), cudaMemcpyHostToDevice) == cudaSuccess;
    if (!ok) cudaGetLastError();
  }
  t.ok = ok;
  return h->umma_tabs.emplace(key, t).first->second;
}

struct UmmaGeom {
  bool ok;
  int nslab, n_stages, stage_bytes, a_groups, b_groups, umma_m, tmem_cols, acc_cols, k_split, cnt_pad, ring_bytes, smem, ksplit;
};

// Ring of one launch: the deepest K-chunk (64 * nslab elements) that leaves >= 3 stages or >= 120 KB in flight.
// ks2 = true: K split over CTA pairs (gemv_umma.cuh UmmaParams::ksplit): g_max / g_min are the pair sums of boxes.
UmmaGeom umma_geom(int K, int M, int s_max, int g_max, int max_cnt, bool ks2 = false, int g_min_pair = 0) {
  UmmaGeom u{};
  u.ksplit = ks2 ? 2 : 1;
  const int M8 = (M + 7) / 8 * 8;
  u.acc_cols = (s_max * M8 + 15) / 16 * 16;
  u.b_groups = u.acc_cols / 8;
  u.a_groups = g_max;
  u.umma_m = g_max <= 8 ? 64 : 128;
  u.k_split = std::max(1, std::min(std::min(8, 256 / u.acc_cols), K / 512));  // K / 512: every part sees >= 1 chunk of any depth
  u.tmem_cols = 32;
  while (u.tmem_cols < 2 * u.k_split * u.acc_cols) u.tmem_cols *= 2;
  u.cnt_pad = (max_cnt + 3) / 4 * 4;
  const int tail = 2544 + M * u.cnt_pad * 4 * (ks2 ? 2 : 1);  // barriers, 1 / rms, row map, results (+ outbox) (gemv_umma.cuh)
  UmmaGeom best{};
  for (int nslab = 8; nslab >= 1; nslab >>= 1) {
    if (K % (64 * nslab) != 0) continue;
    UmmaGeom g = u;
    const int gb = nslab * 1024;
    g.nslab = nslab;
    g.stage_bytes = (g.b_groups + g_max) * gb;
    // the tensor core reads whole 64- / 128-row tiles: past the weight groups into the activation part, and past
    // the last stage only by what that part does not cover
    const int pad = std::max(0, g.umma_m / 8 - (ks2 ? g_min_pair : g_max) - g.b_groups) * gb;
    if (ks2) {  // every CTA of a pair needs >= k_split chunks of its own
      const int per_rank = K / (64 * nslab) / 2;
      if (per_rank < 1) continue;
      g.k_split = std::min(g.k_split, per_rank);
      g.tmem_cols = 32;
      while (g.tmem_cols < 2 * g.k_split * g.acc_cols) g.tmem_cols *= 2;
    }
    g.n_stages = std::min(8, (kSmemMax - 1024 - tail - pad) / g.stage_bytes);
    if (g.n_stages < 2) continue;
    g.ring_bytes = g.n_stages * g.stage_bytes + pad;
    g.smem = 1024 + g.ring_bytes + tail;
    g.ok = true;
    if (g.n_stages >= 3 || g.n_stages * g.stage_bytes >= 120 * 1024) return g;
    if (!best.ok || g.n_stages * g.stage_bytes > best.n_stages * best.stage_bytes) best = g;
  }
  return best;
}

// Launches q on k_gemv_umma (in row chunks when the result buffer of a whole level does not fit). *done = false:
// the GEMV does not fit the tcgen05 kernel and nothing was launched.
int run_umma(dovetail_draft* h, cudaStream_t st, dovetail_draft::QueuedGemv& q, bool* done) {
  *done = false;
  GemvParams& p = q.p;
  if (p.K % 64 != 0 || !h->maps_dev) return DOVETAIL_OK;
  UmmaParams up{};
  int s_max = 1, g_max = 0, pair_max = 0, pair_min = 2 * kUmmaMaxGroups;
  bool pair_ok = true;
  for (int gi = 0; gi < q.n_groups; ++gi) {
    GemvGroup& G = p.g[gi];
    if (G.xkind != X_ROWS || G.xidx != nullptr || !G.xs) return DOVETAIL_OK;
    G.S = G.S_fixed ? G.S_fixed : 2;
    s_max = std::max(s_max, G.S);
    const dovetail_draft::PlaneBuf* pb = nullptr;
    for (const auto& b : h->plane_bufs)
      if (G.xs >= b.base && G.xs < b.base + b.elems) pb = &b;
    if (!pb || pb->ld != G.xs_ld || G.xs_plane != static_cast<int64_t>(pb->cap) * pb->ld || pb->ld != p.K) return DOVETAIL_OK;
    up.x_cap[gi] = pb->cap;
    up.x_row0[gi] = static_cast<int32_t>((G.xs - pb->base) / pb->ld);
    up.xmap[gi] = h->maps_dev + pb->map;  // + box depth below
    for (int j = 0; j < G.n_mat; ++j) {
      auto it = h->wmap_of.find(G.w[j]);
      if (it == h->wmap_of.end()) return DOVETAIL_OK;
      up.wmap[gi][j] = h->maps_dev + it->second;
    }
    const dovetail_draft::UmmaTable& T = umma_table(h, G, q.ctas);
    if (!T.ok) return DOVETAIL_OK;
    up.tab[gi] = T.tab;
    up.vpos[gi] = T.vpos;
    if (gi > 0 && T.vpos_ld != up.vpos_ld) return DOVETAIL_OK;  // groups of one launch share the dealing shape
    up.vpos_ld = T.vpos_ld;
    g_max = std::max(g_max, T.g_max);
    pair_max = std::max(pair_max, T.pair_max);
    pair_min = std::min(pair_min, T.pair_min);
    if (T.pair_max == 0) pair_ok = false;
  }
  const int Mtot = p.M;
  int Mc = Mtot;
  // CTAs with few rows at wide levels: K split over CTA pairs (half the activation operand and half the MMAs per CTA)
  // Measured: at 64 rows per level it always pays (13B shape: down 59 -> 48 us, batch of 64 prompt rows 988 -> 925 us);
  // below that only when the pair's boxes fit a 64-row tile (7B shape, 28 rows per CTA: down 24.8 -> 19.5 us at 10 rows;
  // 13B shape, 35 rows per CTA and a 128-row tile: 679 -> 697 us per forward at 16 rows).
  const bool ks2 = pair_ok && (Mtot >= h->umma_ksplit_min_m || (pair_max <= 8 && h->umma_ksplit_min_m <= kUmmaMaxM));
  auto geom = [&](int m) {
    UmmaGeom x = ks2 ? umma_geom(p.K, m, s_max, pair_max, q.max_cnt, true, pair_min) : UmmaGeom{};
    return x.ok ? x : umma_geom(p.K, m, s_max, g_max, q.max_cnt);
  };
  UmmaGeom g = geom(Mc);
  while (!g.ok && Mc > 8) {
    Mc = (Mc / 2 + 7) / 8 * 8;
    g = geom(Mc);
  }
  if (!g.ok) return DOVETAIL_OK;
  int lg = 0;
  while ((1 << lg) < g.nslab) ++lg;
  for (int gi = 0; gi < q.n_groups; ++gi) {
    up.xmap[gi] += lg;
    for (int j = 0; j < p.g[gi].n_mat; ++j) up.wmap[gi][j] += lg;
  }
  up.nslab = g.nslab; up.n_stages = g.n_stages; up.stage_bytes = g.stage_bytes; up.a_groups = g.a_groups;
  up.umma_m = g.umma_m; up.tmem_cols = g.tmem_cols; up.acc_cols = g.acc_cols; up.k_split = g.k_split; up.ksplit = g.ksplit; up.cnt_pad = g.cnt_pad;
  up.ring_bytes = g.ring_bytes;
  p.n_groups = q.n_groups;
  p.ctas_per_group = q.ctas;
  p.row_bytes = p.K * 2;
  h->cur_kind = q.kind;
  *done = true;
  for (int m0 = 0; m0 < Mtot; m0 += Mc) {
    p.M = std::min(Mc, Mtot - m0);
    p.m0 = m0;
    h->cur_bytes = m0 == 0 ? q.bytes : 0;  // the algorithmic bytes are counted once
    p.trace = trace_slot(h);
    up.p = p;
    if (!h->dry) { ++h->umma_launches; if (g.ksplit == 2) ++h->ksplit_launches; }
    cudaError_t e = launch_c(h, g.ksplit, true, k_gemv_umma, dim3(q.n_groups * q.ctas), dim3(kUmmaThreads), g.smem, st, up);
    if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "GEMV (tcgen05) launch failed: %s", cudaGetErrorString(e));
  }
  p.M = Mtot;
  p.m0 = 0;
  return DOVETAIL_OK;
}

// One GEMV on the FMA kernel (fp32 models; bf16 matrices whose K is not a multiple of 32).
int run_gemv_fma(dovetail_draft* h, cudaStream_t st, dovetail_draft::QueuedGemv& q) {
  GemvParams& p = q.p;
  h->cur_kind = q.kind;
  h->cur_bytes = q.bytes;
  const GemvShape s = gemv_shape(p.K, h->es, p.M, q.max_cnt + 1);
  if (!s.ok) return fail(h, DOVETAIL_EINVAL, "GEMV with K = %d is not supported (K * elem size must be a multiple of 16 and <= 28672 bytes)", p.K);
  p.rows_per_stage = s.rows_per_stage;
  p.n_stages = s.n_stages;
  p.stage_bytes = s.stage_bytes;
  p.row_bytes = s.row_bytes;
  GemvKernel k = h->es == 2 ? pick_gemv<__nv_bfloat16>(s.MT, s.NI) : pick_gemv<float>(s.MT, s.NI);
  p.trace = trace_slot(h);
  cudaError_t e = launch(h, k, dim3(q.ctas, q.n_groups), dim3(kThreads), s.smem, st, p);
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "GEMV launch failed: %s", cudaGetErrorString(e));
  return DOVETAIL_OK;
}

// One launch of the tensor-core kernel.
int run_mma(dovetail_draft* h, cudaStream_t st, dovetail_draft::QueuedGemv& q, const MmaGeom& g) {
  MmaParams cp{};
  cp.stage_bytes = g.stage_bytes;
  cp.n_stages = g.n_stages;
  cp.part_floats = g.part_floats;
  cp.res_floats = g.res_floats;
  GemvParams& p = q.p;
  p.n_groups = q.n_groups;
  p.ctas_per_group = q.ctas;
  p.rows_per_stage = g.RSp;
  p.row_bytes = p.K * (h->wq ? 1 : 2);
  p.kc = g.KC;
  p.seg_stride = g.seg_stride;
  p.aseg_stride = g.aseg_stride;
  for (int gi = 0; gi < q.n_groups; ++gi)
    p.g[gi].S = p.g[gi].xkind == X_EMBED ? 1 : (p.g[gi].S_fixed ? p.g[gi].S_fixed : g.S);
  h->cur_kind = q.kind;
  h->cur_bytes = q.bytes;
  p.trace = trace_slot(h);
  cp.p = p;
#ifdef DVT_CHAINDBG
  if (!h->dry) {
    if (!h->dbg) { cudaMalloc(reinterpret_cast<void**>(&h->dbg), sizeof(unsigned long long) * 64 * 148 * 16); cudaMemset(h->dbg, 0, sizeof(unsigned long long) * 64 * 148 * 16); }
    if (h->dbg_launch < 64) cp.dbg = h->dbg + static_cast<size_t>(h->dbg_launch++) * 148 * 16;
  }
#endif
  cudaError_t e = launch(h, pick_gemv_mma(g.NT, h->wq), dim3(q.n_groups * q.ctas), dim3(kMmaThreads), g.smem, st, cp);
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "GEMV (mma) launch failed: %s", cudaGetErrorString(e));
  return DOVETAIL_OK;
}

// Launch everything queued: tensor-core-capable GEMVs on k_gemv_mma, the rest on the FMA kernel. (Running several
// GEMVs in one persistent launch with a grid barrier between them was built and measured slower than separate
// launches with programmatic dependent launch: DESIGN.md, negative results.)
int flush_gemv(dovetail_draft* h, cudaStream_t st) {
  auto& Q = h->queue;
  int rc = DOVETAIL_OK;
  for (size_t i = 0; i < Q.size() && rc == DOVETAIL_OK; ++i) {
    if (h->es == 2 && !h->wq && Q[i].p.M >= h->umma_min_m && Q[i].p.M <= kUmmaMaxM) {  // wide level: tcgen05 consumer
      bool done = false;
      rc = run_umma(h, st, Q[i], &done);
      if (done || rc != DOVETAIL_OK) continue;
    }
    const MmaGeom g = h->es == 2 ? mma_geom(Q[i], h->wq) : MmaGeom{};
    if (g.ok) {
      rc = run_mma(h, st, Q[i], g);
    } else if (h->es == 2 && Q[i].p.M > kMmaMaxM && Q[i].p.K % 32 == 0) {
      // a level wider than 32 rows: chunks of <= 32 rows (64 B columns), the weights are streamed once per chunk
      const int Mtot = Q[i].p.M;
      for (int m0 = 0; m0 < Mtot && rc == DOVETAIL_OK; m0 += kMmaMaxM) {
        dovetail_draft::QueuedGemv c = Q[i];
        c.p.M = std::min(kMmaMaxM, Mtot - m0);
        c.p.m0 = m0;
        if (m0 > 0) c.bytes = 0;  // the algorithmic bytes are counted once
        const MmaGeom gc = mma_geom(c, h->wq);
        rc = gc.ok ? run_mma(h, st, c, gc) : fail(h, DOVETAIL_EINVAL, "GEMV with K = %d does not fit the tensor-core kernel", c.p.K);
      }
    } else if (h->wq) {
      rc = fail(h, DOVETAIL_EINVAL, "int8 weights: GEMV with K = %d, M = %d does not fit the tensor-core kernel", Q[i].p.K, Q[i].p.M);
    } else {
      rc = run_gemv_fma(h, st, Q[i]);
    }
  }
  Q.clear();
  return rc;
}

// Queue one GEMV: group list, K, M rows, epilogue. It is launched by the next flush_gemv.
int run_gemv(dovetail_draft* h, cudaStream_t st, GemvParams& p, int n_groups, int ctas_per_group, int kind) {
  (void)st;
  dovetail_draft::QueuedGemv q{};
  q.n_groups = n_groups;
  q.ctas = ctas_per_group;
  q.kind = kind;
  for (int g = 0; g < n_groups; ++g) {
    const GemvGroup& G = p.g[g];
    for (int j = 0; j < G.n_mat; ++j)
      q.bytes += h->wq ? static_cast<int64_t>(G.rows[j]) * (p.K + 4) : static_cast<int64_t>(G.rows[j]) * p.K * h->es;
    // dealing of the group's rows (units: rows, rows of each paired matrix, or rotary pairs) to its CTAs
    long units;
    int per_unit;
    if (G.paired) { units = G.rows[0]; per_unit = G.n_mat; }
    else {
      long tot = 0;
      for (int j = 0; j < G.n_mat; ++j) tot += G.rows[j];
      per_unit = G.pairperm ? 2 : 1;  // rotary pairs are dealt whole (gemv.cuh cta_rows)
      units = tot / per_unit;
    }
    p.g[g].deal_base = static_cast<int32_t>(units / ctas_per_group);
    p.g[g].deal_rem = static_cast<int32_t>(units % ctas_per_group);
    const int mc = per_unit * (p.g[g].deal_base + (p.g[g].deal_rem > 0 ? 1 : 0));
    q.max_cnt = std::max(q.max_cnt, mc);
  }
  p.dyn = h->dyn;
  q.p = p;
  h->queue.push_back(q);
  return DOVETAIL_OK;
}

GemvGroup rows_group(const float* xsrc, int64_t xld, const int32_t* xidx, int from_dyn, const void* gain) {
  GemvGroup g{};
  g.xkind = X_ROWS;
  g.xsrc = xsrc;
  g.xld = xld;
  g.xidx = xidx;
  g.x_from_dyn = from_dyn;
  g.gain = gain;
  return g;
}

// split-bf16 planes of an activation buffer with `rows` rows of stride ld (epilogue.cuh), first row row0
SplitOut planes(const dovetail_draft* h, __nv_bfloat16* xs, int64_t rows, int64_t ld, int64_t row0 = 0) {
  SplitOut o{};
  if (xs) {
    o.xs = xs + row0 * ld;
    o.plane = rows * ld;
    o.ld = ld;
    o.perm = h->wq;  // int8 weights: the planes are stored in the consumer's k order (epilogue.cuh split_pos)
  }
  return o;
}

void with_planes(GemvGroup& g, const SplitOut& o) {
  g.xs = o.xs;
  g.xs_plane = o.plane;
  g.xs_ld = o.ld;
}

int validate_tree(dovetail_draft* h, const dovetail_tree_spec_t* t, int n_new, std::vector<LevelPlan>& plan,
                  int& tree_rows, int& pool_total) {
  const dovetail_config_t& c = h->cfg;
  if (t->depth < 1 || t->depth > DOVETAIL_MAX_DEPTH) return fail(h, DOVETAIL_EINVAL, "tree depth %d out of range", t->depth);
  if (t->gamma < 1) return fail(h, DOVETAIL_EINVAL, "gamma must be >= 1");
  plan.resize(t->depth);
  int m = 1, pool = 0;
  tree_rows = 0;
  for (int l = 0; l < t->depth; ++l) {
    if (t->branch[l] < 1 || t->branch[l] > c.max_branch || t->branch[l] > c.vocab)
      return fail(h, DOVETAIL_EINVAL, "branch[%d] = %d out of range [1, min(max_branch, vocab)]", l, t->branch[l]);
    if (l >= 1) {
      if (t->beam[l] < 0) return fail(h, DOVETAIL_EINVAL, "beam[%d] negative", l);
      const long n = static_cast<long>(m) * t->branch[l - 1];
      m = static_cast<int>((t->beam[l] > 0 && t->beam[l] < n) ? t->beam[l] : n);
      if (m > c.max_rows) return fail(h, DOVETAIL_EINVAL, "level %d forwards %d rows > max_rows %d", l, m, c.max_rows);
      plan[l].rows = m;
      plan[l].rows_lm = m;
      plan[l].t0 = tree_rows;
      plan[l].row0 = n_new + tree_rows;
      tree_rows += m;
    } else {
      plan[0].rows = n_new;
      plan[0].rows_lm = 1;
      plan[0].t0 = 0;
      plan[0].row0 = 0;
    }
    plan[l].pool_begin = pool;
    pool += plan[l].rows_lm * t->branch[l];
  }
  if (tree_rows > c.max_tree_slots) return fail(h, DOVETAIL_EINVAL, "tree forwards %d rows > max_tree_slots %d", tree_rows, c.max_tree_slots);
  if (pool > h->pool_cap) return fail(h, DOVETAIL_EINVAL, "candidate pool %d exceeds capacity %d", pool, h->pool_cap);
  pool_total = pool;
  return DOVETAIL_OK;
}

template <typename T>
cudaError_t dmalloc(T** p, size_t n) {
  return cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T));
}

void destroy_graph(dovetail_draft::StepGraph& g) {
  if (g.exec) cudaGraphExecDestroy(g.exec);
  if (g.graph) cudaGraphDestroy(g.graph);
  g.exec = nullptr;
  g.graph = nullptr;
}

void free_all(dovetail_draft* h) {
  cudaFree(h->dyn); cudaFree(h->ts); cudaFree(h->rt); cudaFree(h->rope); cudaFree(h->inv_freq);
  cudaFree(h->hbuf); cudaFree(h->hhat); cudaFree(h->qkv); cudaFree(h->obuf); cudaFree(h->act);
  cudaFree(h->xs_feat); cudaFree(h->xs_hhat); cudaFree(h->xs_x); cudaFree(h->xs_h12); cudaFree(h->xs_o); cudaFree(h->xs_act);
  cudaFree(h->ssq);
  cudaFree(h->qs);
  cudaFree(h->xs_emb);
  cudaFree(h->xs_par);
  for (auto& g : h->graphs) destroy_graph(g);
  h->graphs.clear();
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  cudaFree(h->maps_dev);
  for (auto& kv : h->umma_tabs) { cudaFree(kv.second.tab); cudaFree(kv.second.vpos); }
  cudaFree(h->attn_ws); cudaFree(h->attn_cnt); cudaFree(h->cand_val); cudaFree(h->cand_id); cudaFree(h->stat);
  cudaFree(h->pool.token); cudaFree(h->pool.parent); cudaFree(h->pool.depth); cudaFree(h->pool.cum);
  cudaFree(h->pool.row); cudaFree(h->treemask); cudaFree(h->out_pool_idx);
  if (h->ts_host) cudaFreeHost(h->ts_host);
  cudaFree(h->trace_buf);
  cudaFree(h->probe_sink);
  if (h->trace_host) cudaFreeHost(h->trace_host);
}

// Test hooks of one level (dovetail_hooks.h): taps of what the level computed, then teacher forcing.
int level_hooks(dovetail_draft* h, cudaStream_t st, const dovetail_kv_cache_t* kv, const LevelPlan& lp, int l, int L,
                int Lp) {
  const dovetail_config_t& c = h->cfg;
  const dovetail_hooks_t& k = h->hooks;
  const int d = c.hidden, dh = c.head_dim, M = lp.rows;
  cudaError_t e = cudaSuccess;
  const size_t xoff = static_cast<size_t>(lp.row0) * d, xbytes = static_cast<size_t>(M) * d * sizeof(float);
  if (k.tap_hhat) e = cudaMemcpyAsync(k.tap_hhat + xoff, h->hhat + xoff, xbytes, cudaMemcpyDeviceToDevice, st);
  if (k.force_hhat && e == cudaSuccess) {
    e = cudaMemcpyAsync(h->hhat + xoff, k.force_hhat + xoff, xbytes, cudaMemcpyDeviceToDevice, st);
    if (h->xs_hhat && e == cudaSuccess) {  // the children read the forced rows as split-bf16 planes
      k_resplit_rows<<<M, 256, 0, st>>>(h->hhat + xoff, d, planes(h, h->xs_hhat, h->max_step_rows, h->ld_d, lp.row0));
      e = cudaGetLastError();
    }
  }
  const size_t pitch = static_cast<size_t>(kv->capacity) * dh * h->es, width = static_cast<size_t>(M) * dh * h->es;
  const size_t off = static_cast<size_t>(l == 0 ? L : Lp + lp.t0) * dh * h->es;
  const size_t height = static_cast<size_t>(c.n_layers) * c.n_kv_heads;
  auto cp2 = [&](void* dst, const void* src) {
    if (dst && src && e == cudaSuccess)
      e = cudaMemcpy2DAsync(static_cast<uint8_t*>(dst) + off, pitch, static_cast<const uint8_t*>(src) + off, pitch, width,
                            height, cudaMemcpyDeviceToDevice, st);
  };
  cp2(k.tap_k, kv->k);
  cp2(k.tap_v, kv->v);
  cp2(kv->k, k.force_k);
  cp2(kv->v, k.force_v);
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "tap / forcing copy failed: %s", cudaGetErrorString(e));
  return DOVETAIL_OK;
}

// Chunks per kv-head of the tensor-core attention kernel (measured on C2 / C3 / C5): at least two 64-position
// blocks per chunk (a CTA's fixed cost is ~6 us), at most two CTAs per SM, and when a head needs more than one
// cluster of 8 no more than ~200 CTAs in all (larger grids of 8-clusters are placed in waves).
// wide: the 64-query-vector kernel (one CTA per SM).
// All clusters of a launch must be resident at once: a cluster is placed on one GPC, and the second wave of a grid
// that does not fit costs a whole kernel time (measured on the 13B shape, 40 heads, prefix 2048: 7 chunks per head
// 24.2 us, 6 chunks 14.0 us). attn_max_clusters[wide][cs] = cudaOccupancyMaxActiveClusters of the kernel at cluster
// size cs (dovetail_draft_init); 0 = unknown.
AttnKernel attn_mma_kernel(int dh, int qt) {
  if (qt == 4) return dh == 128 ? k_tree_attention_mma<128, 4> : k_tree_attention_mma<64, 4>;
  if (qt == 2) return dh == 128 ? k_tree_attention_mma<128, 2> : k_tree_attention_mma<64, 2>;
  return dh == 128 ? k_tree_attention_mma<128, 1> : k_tree_attention_mma<64, 1>;
}

// mode: 0 = QT 1 (16 query vectors per pass), 1 = QT 4 (64, one CTA per SM), 2 = QT 2 (32).
void attn_mma_geom(const dovetail_draft* h, int Lbase, int mode, int& n_chunks, int& cs) {
  const int n_blocks = std::max(1, div_up(Lbase, kAmBlockPos));
  const int Hkv = h->cfg.n_kv_heads;
  const int* maxc = h->attn_max_clusters[mode];
  n_chunks = std::max(1, std::min(mode == 1 ? std::max(1, h->attn_chunks_cap / 2) : h->attn_chunks_cap, n_blocks / 2));
  if (n_chunks <= 8) {
    while (n_chunks > 1 && maxc[n_chunks] > 0 && Hkv > maxc[n_chunks]) --n_chunks;
    n_chunks = div_up(n_blocks, div_up(n_blocks, n_chunks));  // fewest chunks with the same blocks per chunk
    cs = n_chunks;
  } else {
    int groups = std::max(1, std::min(n_chunks, 200 / Hkv) / 8);
    if (maxc[8] > 0) groups = std::max(1, std::min(groups, maxc[8] / Hkv));
    if (maxc[8] > 0 && Hkv > maxc[8]) {  // not even one 8-cluster per head fits: smaller clusters, one per head
      n_chunks = 7;
      while (n_chunks > 1 && maxc[n_chunks] > 0 && Hkv > maxc[n_chunks]) --n_chunks;
      cs = n_chunks;
    } else {
      n_chunks = 8 * groups;
      cs = 8;
    }
  }
}

// Enqueues (or, with h->dry, only shape-checks) the kernels of one draft step.
// prefill: only the level-0 forward of the block stack (dovetail_draft_prefill): no LM head, no tree.
int enqueue_step(dovetail_draft* h, cudaStream_t st, const float* hidden_feats, const int32_t* tokens, int n_new,
                 dovetail_kv_cache_t* kv, const dovetail_tree_spec_t* tree, const dovetail_draft_out_t* out,
                 const std::vector<LevelPlan>& plan, int pool_total, bool prefill = false) {
  const dovetail_config_t& c = h->cfg;
  const int L = kv->committed_len, Lp = L + n_new;
  int rc = DOVETAIL_OK;
  h->launches = 0;
  h->umma_launches = 0;
  h->ksplit_launches = 0;
  const int d = c.hidden, F = c.ffn, V = c.vocab, dh = c.head_dim, half = dh / 2;
  const int dq = h->dq, dkv = h->dkv, ldq = h->ldq, nsm = h->num_sms;
  const int grp = c.n_q_heads / c.n_kv_heads;
  const bool bf16 = c.dtype == DOVETAIL_BF16;
  // bf16 models whose QKV projection runs on the tensor-core GEMV: S2 (RoPE, append, query preparation) is done
  // by that GEMV's epilogue; otherwise by the attention kernel
  const bool fused_s2 = bf16 && d % 32 == 0;
  cudaError_t e;

  // S0: per-step state, level-0 row tables, rotary table
  StepDyn dv{};
  dv.feats = hidden_feats;
  dv.tokens = tokens;
  dv.kc = kv->k;
  dv.vc = kv->v;
  dv.capacity = kv->capacity;
  dv.L = L;
  dv.n_new = n_new;
  dv.Lp = Lp;
  dv.out_ids = out->token_ids;
  dv.out_scores = out->scores;
  dv.out_parents = out->parents;
  dv.out_depths = out->depths;
  dv.out_n = out->n_out;
  h->cur_kind = 0;
  h->cur_bytes = 0;
  h->cur_level = 0;
  h->tr_used = 0;
  h->queue.clear();
#ifdef DVT_CHAINDBG
  h->dbg_launch = 0;
#endif
  if (h->trace_on && !h->dry) {  // start = ~0 (atomicMin), end = 0 (atomicMax)
    e = cudaMemsetAsync(h->trace_buf, 0, sizeof(unsigned long long) * 2 * kMaxTraceLaunches, st);
    if (e == cudaSuccess) e = cudaMemset2DAsync(h->trace_buf, 16, 0xff, 8, kMaxTraceLaunches, st);
    if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "trace reset failed: %s", cudaGetErrorString(e));
  }
  // k_step_begin is launched WITHOUT programmatic serialization: it starts only once everything
  // enqueued before the step has completed, which is what lets later kernels read the committed
  // prefix (cache rows < L) before their griddepcontrol.wait.
  const int64_t R = c.max_rows, SR = h->max_step_rows;
  const int nct_d = std::min(nsm, d);  // CTAs of the GEMVs that produce the residual stream (and its sums of squares)
  e = launch_c(h, 1, false, k_step_begin, dim3(n_new + tree->depth - 1), dim3(512), 0, st, dv, h->dyn, h->ts, h->rt,
               h->rope, static_cast<const double*>(h->inv_freq), half, V, d, planes(h, h->xs_feat, R, h->ld_d), trace_slot(h));
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "launch failed: %s", cudaGetErrorString(e));

  for (int l = 0; l < tree->depth; ++l) {
    const LevelPlan& lp = plan[l];
    const int M = lp.rows;
    h->cur_level = l;
    RowTables* cur = h->rt + (l & 1);
    RowTables* nxt = h->rt + ((l + 1) & 1);
    float* x = h->hhat + static_cast<size_t>(lp.row0) * d;  // residual stream rows of this level

    // S0 + S1: gather, DGF projections h1 = W1 f, h2 = W2 e
    if (c.dgf_proj && h->wq) {  // int8 weights: the level's embedding rows as a plane in the consumer's k order
      rc = flush_gemv(h, st);
      if (rc) return rc;
      h->cur_kind = 10;
      h->cur_bytes = 0;
      e = launch(h, k_embed_plane, dim3(M), dim3(640), 0, st, static_cast<const RowTables*>(cur),
                 static_cast<const __nv_bfloat16*>(h->w.embed), d, planes(h, h->xs_emb, R, h->ld_d), trace_slot(h));
      if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "launch failed: %s", cudaGetErrorString(e));
    }
    // wide level on the tcgen05 GEMV (gemv_umma.cuh): its tensor-map copies read contiguous rows, so the parents'
    // hidden states and the tokens' embedding rows are gathered first
    const bool wide = bf16 && !h->wq && h->maps_dev && M >= h->umma_min_m && M <= kUmmaMaxM && d % 64 == 0;
    if (c.dgf_proj && wide) {
      rc = flush_gemv(h, st);
      if (rc) return rc;
      h->cur_kind = 10;
      h->cur_bytes = 0;
      e = launch(h, k_gather_level, dim3(M, kSplitPlanes + 1), dim3(256), 0, st, static_cast<const RowTables*>(cur),
                 static_cast<const __nv_bfloat16*>(l == 0 ? nullptr : h->xs_hhat), static_cast<int64_t>(SR) * h->ld_d, h->xs_par,
                 static_cast<int64_t>(R) * h->ld_d, static_cast<const __nv_bfloat16*>(h->w.embed), h->xs_emb,
                 static_cast<int64_t>(h->ld_d), d, trace_slot(h));
      if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "launch failed: %s", cudaGetErrorString(e));
    }
    if (c.dgf_proj) {
      GemvParams p{};
      p.g[0] = rows_group(h->hhat, d, (l == 0 || wide) ? nullptr : cur->src, l == 0, nullptr);
      with_planes(p.g[0], l == 0 ? planes(h, h->xs_feat, R, h->ld_d)
                                 : (wide ? planes(h, h->xs_par, R, h->ld_d) : planes(h, h->xs_hhat, SR, h->ld_d)));
      p.g[0].w[0] = h->w.dgf_w1;
      p.g[0].ws[0] = h->w.dgf_s1;
      p.g[0].rows[0] = d;
      p.g[0].n_mat = 1;
      p.g[0].out_off = 0;
      p.g[1] = GemvGroup{};
      p.g[1].xkind = X_EMBED;
      p.g[1].embed = h->w.embed;
      p.g[1].tokens = cur->token;
      p.g[1].w[0] = h->w.dgf_w2;
      p.g[1].ws[0] = h->w.dgf_s2;
      p.g[1].rows[0] = d;
      if (h->wq) {  // int8 consumer: the embedding rows come as a plane in its k order (k_embed_plane below)
        p.g[1].xkind = X_ROWS;
        with_planes(p.g[1], planes(h, h->xs_emb, R, h->ld_d));
        p.g[1].S_fixed = 2;  // bf16 value = two fp16 terms exactly
      } else if (wide) {  // the gathered embedding rows: one exact bf16 plane
        p.g[1].xkind = X_ROWS;
        with_planes(p.g[1], planes(h, h->xs_emb, R, h->ld_d));
        p.g[1].S_fixed = 1;
      }
      p.g[1].n_mat = 1;
      p.g[1].out_off = d;
      p.K = d;
      p.M = M;
      p.epi = EPI_STORE;
      p.out = h->hbuf;
      p.out_ld = 2 * d;
      p.so = planes(h, h->xs_h12, R, h->ld_2d);
      rc = run_gemv(h, st, p, 2, std::max(1, std::min(nsm / 2, d)), 1);
      if (rc) return rc;
    } else {
      const int blocks = std::min(nsm, div_up(M * 2 * d, 256));
      rc = flush_gemv(h, st);
      if (rc) return rc;
      h->cur_kind = 10;
      h->cur_bytes = 0;
      if (bf16)
        e = launch(h, k_fill_h<__nv_bfloat16>, dim3(blocks), dim3(256), 0, st, static_cast<const StepDyn*>(h->dyn), l == 0 ? 1 : 0,
                   static_cast<const float*>(h->hhat), static_cast<int64_t>(d), static_cast<const RowTables*>(cur), l == 0 ? 0 : 1,
                   static_cast<const __nv_bfloat16*>(h->w.embed), h->hbuf, M, d, planes(h, h->xs_h12, R, h->ld_2d), trace_slot(h));
      else
        e = launch(h, k_fill_h<float>, dim3(blocks), dim3(256), 0, st, static_cast<const StepDyn*>(h->dyn), l == 0 ? 1 : 0,
                   static_cast<const float*>(h->hhat), static_cast<int64_t>(d), static_cast<const RowTables*>(cur), l == 0 ? 0 : 1,
                   static_cast<const float*>(h->w.embed), h->hbuf, M, d, SplitOut{}, trace_slot(h));
      if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "launch failed: %s", cudaGetErrorString(e));
    }
    {  // S1: gate, sigmoid, blend; or the single Linear of the EAGLE-2 fusion (:104)
      GemvParams p{};
      p.g[0] = rows_group(h->hbuf, 2 * d, nullptr, 0, nullptr);
      with_planes(p.g[0], planes(h, h->xs_h12, R, h->ld_2d));
      p.g[0].w[0] = h->w.dgf_wg;
      p.g[0].ws[0] = h->w.dgf_sg;
      p.g[0].rows[0] = d;
      p.g[0].n_mat = 1;
      p.K = 2 * d;
      p.M = M;
      p.epi = c.fusion == DOVETAIL_FUSION_CONCAT_LINEAR ? EPI_STORE : EPI_DGF;
      p.out = x;
      p.out_ld = d;
      p.hbuf = h->hbuf;
      p.bias = h->w.dgf_bg;
      p.d = d;
      // x feeds the first block's QKV: planes of x * g_attn (raw x when the first input norm is skipped)
      p.so = planes(h, h->xs_x, R, h->ld_d);
      p.gain_out = c.first_layer_input_norm ? h->layers[0].g_attn : nullptr;
      p.ssq_out = h->ssq;
      rc = run_gemv(h, st, p, 1, nct_d, 2);
      if (rc) return rc;
    }

    for (int ly = 0; ly < c.n_layers; ++ly) {
      const dovetail_layer_weights_t& W = h->layers[ly];
      {  // S2: RMSNorm + Q, K, V projections
        GemvParams p{};
        const void* gain = (ly == 0 && !c.first_layer_input_norm) ? nullptr : W.g_attn;
        p.g[0] = rows_group(x, d, nullptr, 0, gain);
        with_planes(p.g[0], planes(h, h->xs_x, R, h->ld_d));
        p.ssq_in = gain ? h->ssq : nullptr;
        p.ssq_nct = nct_d;
        p.g[0].w[0] = W.wq; p.g[0].rows[0] = dq; p.g[0].ws[0] = W.sq;
        p.g[0].w[1] = W.wk; p.g[0].rows[1] = dkv; p.g[0].ws[1] = W.sk;
        p.g[0].w[2] = W.wv; p.g[0].rows[2] = dkv; p.g[0].ws[2] = W.sv;
        p.g[0].n_mat = 3;
        p.K = d;
        p.M = M;
        p.eps = c.rms_eps;
        p.epi = EPI_STORE;
        p.out = h->qkv;
        p.out_ld = ldq;
        if (fused_s2) {  // S2 in the projection's epilogue: RoPE, K / V append, queries ready for the attention kernel
          p.epi = EPI_QKV;
          p.g[0].pairperm = dh;
          p.rt = cur;
          p.rope = h->rope;
          p.rope_row0 = l == 0 ? 0 : n_new + l - 1;
          p.rope_per_row = l == 0 ? 1 : 0;
          p.Hq = c.n_q_heads;
          p.Hkv = c.n_kv_heads;
          p.layer = ly;
          p.level0 = l == 0 ? 1 : 0;
          p.qs = h->qs;
        }
        rc = run_gemv(h, st, p, 1, std::min(nsm, ldq / 2), 3);
        if (rc) return rc;
      }
      {  // S2 (RoPE, KV append) + S3 tree attention
        rc = flush_gemv(h, st);
        if (rc) return rc;
        AttnParams a{};
        a.dyn = h->dyn;
        a.qkv = h->qkv;
        a.obuf = h->obuf;
        a.rows = cur;
        a.rope = h->rope;
        a.rope_row0 = l == 0 ? 0 : n_new + l - 1;
        a.rope_per_row = l == 0 ? 1 : 0;
        a.M = M;
        a.Hq = c.n_q_heads;
        a.Hkv = c.n_kv_heads;
        a.layer = ly;
        a.level0 = l == 0 ? 1 : 0;
        a.new_cnt = l == 0 ? n_new : lp.t0 + M;
        a.n_stages = kAttnStages;
        a.ws = h->attn_ws;
        a.qv_cap = h->qv_cap;
        a.counters = h->attn_cnt;
        const int Lbase = l == 0 ? L : Lp;
        const int qv_tot = M * grp;
        h->cur_kind = 4;
        h->cur_bytes = static_cast<int64_t>(2) * Lbase * dkv * h->es;
        a.trace = trace_slot(h);
        a.so = planes(h, h->xs_o, R, h->ld_dq);
        a.qs = fused_s2 ? h->qs : nullptr;
        if (bf16) {  // tensor-core kernel, chunks of a kv-head merged in a cluster (attention_mma.cuh)
          a.kc = kv->k;
          a.vc = kv->v;
          a.cap = kv->capacity;
          a.Lbase = Lbase;
          a.Lsafe = L;
          // more than 32 query vectors: 64 per pass over the cache, one query tile per warp (attention_mma.cuh)
          // 17 ... 32 query vectors: 32 per pass (QT = 2); more: 64 per pass, one query tile per warp (QT = 4)
          const int mode = qv_tot > h->attn_wide_min ? 1 : (qv_tot > kAmQRows && h->attn_qt2 ? 2 : 0);
          int n_chunks, cs;
          attn_mma_geom(h, Lbase, mode, n_chunks, cs);
          const int qt = mode == 1 ? 4 : (mode == 2 ? 2 : 1);
          const size_t smem = am_smem_bytes(dh, qt);
          auto kern = attn_mma_kernel(dh, qt);
          e = launch_c(h, cs, true, kern, dim3(n_chunks, c.n_kv_heads), dim3(kAmThreads), smem, st, a);
        } else {
          int n_chunks = std::min(h->attn_chunks_cap, std::max(1, div_up(Lbase, 2 * kAttnStagePos)));
          const int QT = qv_tot == 1 ? 1 : (qv_tot == 2 ? 2 : 4);
          const int stage_bytes = 2 * kAttnStagePos * dh * h->es;
          const size_t smem = static_cast<size_t>(kAttnStages) * stage_bytes + 128 +
                              static_cast<size_t>(kConsumerWarps) * QT * (dh + 2) * 4 + 16;
          e = launch(h, pick_attn(c.dtype, dh, QT), dim3(n_chunks, c.n_kv_heads), dim3(kThreads), smem, st, a);
        }
        if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "attention launch failed: %s", cudaGetErrorString(e));
      }
      {  // S4: x += Wo o
        GemvParams p{};
        p.g[0] = rows_group(h->obuf, dq, nullptr, 0, nullptr);
        with_planes(p.g[0], planes(h, h->xs_o, R, h->ld_dq));
        p.g[0].w[0] = W.wo; p.g[0].rows[0] = d; p.g[0].n_mat = 1; p.g[0].ws[0] = W.so;
        p.K = dq;
        p.M = M;
        p.epi = EPI_RESID;
        p.out = x;
        p.out_ld = d;
        p.so = planes(h, h->xs_x, R, h->ld_d);  // feeds gate / up through the post-attention norm
        p.gain_out = W.g_ffn;
        p.ssq_out = h->ssq;
        rc = run_gemv(h, st, p, 1, nct_d, 5);
        if (rc) return rc;
      }
      {  // S5a: act = SiLU(Wgate n) * (Wup n), n = RMSNorm(x)
        GemvParams p{};
        p.g[0] = rows_group(x, d, nullptr, 0, W.g_ffn);
        with_planes(p.g[0], planes(h, h->xs_x, R, h->ld_d));
        p.ssq_in = h->ssq;
        p.ssq_nct = nct_d;
        p.g[0].w[0] = W.wgate; p.g[0].rows[0] = F; p.g[0].ws[0] = W.sgate;
        p.g[0].w[1] = W.wup; p.g[0].rows[1] = F; p.g[0].ws[1] = W.sup;
        p.g[0].n_mat = 2;
        p.g[0].paired = 1;
        p.K = d;
        p.M = M;
        p.eps = c.rms_eps;
        p.epi = EPI_SWIGLU;
        p.out = h->act;
        p.out_ld = F;
        p.so = planes(h, h->xs_act, R, h->ld_f);
        rc = run_gemv(h, st, p, 1, std::min(nsm, F), 6);
        if (rc) return rc;
      }
      {  // S5b: x += Wdown act
        GemvParams p{};
        p.g[0] = rows_group(h->act, F, nullptr, 0, nullptr);
        with_planes(p.g[0], planes(h, h->xs_act, R, h->ld_f));
        p.g[0].w[0] = W.wdown; p.g[0].rows[0] = d; p.g[0].n_mat = 1; p.g[0].ws[0] = W.sdown;
        p.K = F;
        p.M = M;
        p.epi = EPI_RESID;
        p.out = x;
        p.out_ld = d;
        if (ly + 1 < c.n_layers) {  // feeds the next block's QKV through its input norm
          p.so = planes(h, h->xs_x, R, h->ld_d);
          p.gain_out = h->layers[ly + 1].g_attn;
          p.ssq_out = h->ssq;
        } else {
          // the block stack's output: feature of this row's children (raw) and input of the LM head
          p.so_raw = planes(h, h->xs_hhat, SR, h->ld_d, lp.row0);
          if (c.final_norm) {
            p.so = planes(h, h->xs_x, R, h->ld_d);
            p.gain_out = h->w.g_final;
            p.ssq_out = h->ssq;
          }
        }
        rc = run_gemv(h, st, p, 1, nct_d, 7);
        if (rc) return rc;
      }
    }

    if (prefill) {  // the rows' K / V are in the cache: that is all a catch-up batch leaves
      rc = flush_gemv(h, st);
      if (rc) return rc;
      break;
    }
    const int lm_ctas = std::min(std::min(nsm, V), 256);  // k_tree_level merges at most 256 per-CTA lists per row
    {  // S6: LM head + per-CTA top-b + softmax statistics. Level 0: the last row seeds the tree.
      GemvParams p{};
      const float* xs = l == 0 ? x + static_cast<size_t>(n_new - 1) * d : x;
      p.g[0] = rows_group(xs, d, nullptr, 0, c.final_norm ? h->w.g_final : nullptr);
      const int lm_row = l == 0 ? n_new - 1 : 0;  // first row of the level whose list is expanded
      with_planes(p.g[0], c.final_norm ? planes(h, h->xs_x, R, h->ld_d, lm_row) : planes(h, h->xs_hhat, SR, h->ld_d, lp.row0 + lm_row));
      if (c.final_norm) {
        p.ssq_in = h->ssq + lm_row;
        p.ssq_nct = nct_d;
      }
      p.g[0].w[0] = h->w.lm_head; p.g[0].rows[0] = V; p.g[0].n_mat = 1; p.g[0].ws[0] = h->w.lm_head_s;
      p.K = d;
      p.M = lp.rows_lm;
      p.eps = c.rms_eps;
      p.epi = EPI_LMHEAD;
      p.b = tree->branch[l];
      p.vocab = V;
      p.cand_val = h->cand_val;
      p.cand_id = h->cand_id;
      p.stat = h->stat;
      p.tap = h->hooks.tap_logits ? h->hooks.tap_logits + static_cast<size_t>(lp.row0 + (l == 0 ? n_new - 1 : 0)) * V : nullptr;
      rc = run_gemv(h, st, p, 1, lm_ctas, 8);
      if (rc) return rc;
    }
    {  // S7 (+ S8 after the last level)
      rc = flush_gemv(h, st);
      if (rc) return rc;
      TreeLevelParams t{};
      t.dyn = h->dyn;
      t.ts = h->ts;
      t.pool = h->pool;
      t.treemask = h->treemask;
      t.cand_val = h->cand_val;
      t.cand_id = h->cand_id;
      t.stat = h->stat;
      t.nct = lm_ctas;
      t.M = lp.rows_lm;
      t.b = tree->branch[l];
      t.level = l;
      t.pool_begin = lp.pool_begin;
      const bool last = l + 1 == tree->depth;
      t.M_next = last ? 0 : plan[l + 1].rows;
      t.next_row0 = last ? 0 : plan[l + 1].row0;
      t.cur_row0 = lp.row0;
      t.next_t0 = last ? 0 : plan[l + 1].t0;
      t.n_new = n_new;
      t.cur = cur;
      t.next = nxt;
      t.gamma = tree->gamma;
      t.pool_total = pool_total;
      t.out_pool_idx = h->out_pool_idx;
      t.tap_token = h->hooks.tap_pool_token;
      t.tap_cum = h->hooks.tap_pool_cum;
      t.force_token = h->hooks.force_pool_token;
      t.force_cum = h->hooks.force_pool_cum;
      h->cur_kind = 9;
      h->cur_bytes = 0;
      t.trace = trace_slot(h);
      e = launch(h, k_tree_level, dim3(1), dim3(kTreeThreads), 0, st, t);
      if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "tree launch failed: %s", cudaGetErrorString(e));
    }
    if (h->hooks_on && !h->dry) {
      rc = level_hooks(h, st, kv, lp, l, L, Lp);
      if (rc) return rc;
    }
  }
  return DOVETAIL_OK;
}

// The step as one graph launch. Key: everything the launch SEQUENCE depends on -- the tree, n_new and the grids /
// cluster sizes of the attention kernels (functions of the prefix length in 64-position blocks). Per-call values
// that are kernel arguments are patched into the instantiated graph: k_step_begin's StepDyn (caller pointers,
// committed length, outputs) and the tensor-core attention kernels' cache pointers and lengths.
int step_by_graph(dovetail_draft* h, cudaStream_t st, const float* hidden_feats, const int32_t* tokens, int n_new,
                  dovetail_kv_cache_t* kv, const dovetail_tree_spec_t* tree, const dovetail_draft_out_t* out,
                  const std::vector<LevelPlan>& plan, int pool_total) {
  const dovetail_config_t& c = h->cfg;
  const int L = kv->committed_len, Lp = L + n_new;
  const bool bf16 = c.dtype == DOVETAIL_BF16;
  std::vector<int> key = {tree->depth, tree->gamma, n_new};
  for (int l = 0; l < tree->depth; ++l) { key.push_back(tree->branch[l]); key.push_back(tree->beam[l]); }
  int nc[2] = {0, 0}, cs[2] = {0, 0};
  if (bf16) {
    attn_mma_geom(h, L, 0, nc[0], cs[0]);
    attn_mma_geom(h, Lp, 0, nc[1], cs[1]);
    for (int mode = 1; mode <= 2; ++mode) {  // the other kernels' geometry (which levels take them follows from the tree and n_new)
      int wn[2], wc[2];
      attn_mma_geom(h, L, mode, wn[0], wc[0]);
      attn_mma_geom(h, Lp, mode, wn[1], wc[1]);
      key.insert(key.end(), {wn[0], wc[0], wn[1], wc[1]});
    }
    key.insert(key.end(), {h->attn_wide_min, h->attn_qt2, h->umma_ksplit_min_m});
  } else {
    nc[0] = std::min(h->attn_chunks_cap, std::max(1, div_up(L, 2 * kAttnStagePos)));
    nc[1] = std::min(h->attn_chunks_cap, std::max(1, div_up(Lp, 2 * kAttnStagePos)));
  }
  key.insert(key.end(), {nc[0], cs[0], nc[1], cs[1], h->umma_min_m});
  dovetail_draft::StepGraph* g = nullptr;
  for (auto& x : h->graphs)
    if (x.key == key) g = &x;
  cudaError_t e = cudaSuccess;
  if (!g) {
    // shape check without launching, then capture the real launch sequence on the handle's own stream
    h->dry = true;
    int rc = enqueue_step(h, st, hidden_feats, tokens, n_new, kv, tree, out, plan, pool_total);
    h->dry = false;
    if (rc != DOVETAIL_OK) return rc;
    if (!h->cap_stream && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess)
      return fail(h, DOVETAIL_ECUDA, "stream creation failed");
    dovetail_draft::StepGraph ng;
    ng.key = key;
    e = cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "graph capture failed: %s", cudaGetErrorString(e));
    rc = enqueue_step(h, h->cap_stream, hidden_feats, tokens, n_new, kv, tree, out, plan, pool_total);
    e = cudaStreamEndCapture(h->cap_stream, &ng.graph);
    if (rc != DOVETAIL_OK) { destroy_graph(ng); cudaGetLastError(); return rc; }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&ng.exec, ng.graph, 0);
    if (e != cudaSuccess) { destroy_graph(ng); cudaGetLastError(); return fail(h, DOVETAIL_ECUDA, "graph instantiation failed: %s", cudaGetErrorString(e)); }
    size_t n_nodes = 0;
    cudaGraphGetNodes(ng.graph, nullptr, &n_nodes);
    std::vector<cudaGraphNode_t> nodes(n_nodes);
    cudaGraphGetNodes(ng.graph, nodes.data(), &n_nodes);
    for (cudaGraphNode_t nd : nodes) {
      cudaGraphNodeType ty;
      if (cudaGraphNodeGetType(nd, &ty) != cudaSuccess || ty != cudaGraphNodeTypeKernel) continue;
      cudaKernelNodeParams kp{};
      if (cudaGraphKernelNodeGetParams(nd, &kp) != cudaSuccess) continue;
      if (kp.func == reinterpret_cast<void*>(k_step_begin)) {
        ng.begin_node = nd;
        ng.begin_params = kp;
        ng.begin_args.assign(kp.kernelParams, kp.kernelParams + 11);  // k_step_begin takes 11 arguments
        ng.begin_dv = *static_cast<const StepDyn*>(kp.kernelParams[0]);
      } else if (kp.func == reinterpret_cast<void*>(attn_mma_kernel(64, 1)) || kp.func == reinterpret_cast<void*>(attn_mma_kernel(128, 1)) ||
                 kp.func == reinterpret_cast<void*>(attn_mma_kernel(64, 2)) || kp.func == reinterpret_cast<void*>(attn_mma_kernel(128, 2)) ||
                 kp.func == reinterpret_cast<void*>(attn_mma_kernel(64, 4)) || kp.func == reinterpret_cast<void*>(attn_mma_kernel(128, 4))) {
        ng.attn_nodes.push_back(nd);
        ng.attn_node_params.push_back(kp);
        ng.attn_params.push_back(*static_cast<const AttnParams*>(kp.kernelParams[0]));
      }
    }
    cudaGetLastError();
    if (!ng.begin_node) { destroy_graph(ng); return fail(h, DOVETAIL_ECUDA, "graph capture: step-begin node not found"); }
    ng.launches = h->launches;
    ng.umma_launches = h->umma_launches;
    if (h->graphs.size() >= 8) {  // evict the least recently used
      size_t lru = 0;
      for (size_t i = 1; i < h->graphs.size(); ++i)
        if (h->graphs[i].used < h->graphs[lru].used) lru = i;
      destroy_graph(h->graphs[lru]);
      h->graphs.erase(h->graphs.begin() + lru);
    }
    h->graphs.push_back(std::move(ng));
    g = &h->graphs.back();
    h->last_graph = 2;
  } else {
    // patch the per-call values
    StepDyn& dv = g->begin_dv;
    dv.feats = hidden_feats; dv.tokens = tokens; dv.kc = kv->k; dv.vc = kv->v; dv.capacity = kv->capacity;
    dv.L = L; dv.n_new = n_new; dv.Lp = Lp;
    dv.out_ids = out->token_ids; dv.out_scores = out->scores; dv.out_parents = out->parents;
    dv.out_depths = out->depths; dv.out_n = out->n_out;
    g->begin_args[0] = &dv;
    g->begin_params.kernelParams = g->begin_args.data();
    e = cudaGraphExecKernelNodeSetParams(g->exec, g->begin_node, &g->begin_params);
    for (size_t i = 0; i < g->attn_nodes.size() && e == cudaSuccess; ++i) {
      AttnParams& a = g->attn_params[i];
      a.kc = kv->k; a.vc = kv->v; a.cap = kv->capacity;
      a.Lbase = a.level0 ? L : Lp;
      a.Lsafe = L;
      void* args[1] = {&a};
      cudaKernelNodeParams kp = g->attn_node_params[i];
      kp.kernelParams = args;
      e = cudaGraphExecKernelNodeSetParams(g->exec, g->attn_nodes[i], &kp);
    }
    if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "graph update failed: %s", cudaGetErrorString(e));
    h->launches = g->launches;
    h->umma_launches = g->umma_launches;
    h->last_graph = 1;
  }
  g->used = ++h->graph_clock;
  e = cudaGraphLaunch(g->exec, st);
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "graph launch failed: %s", cudaGetErrorString(e));
  return DOVETAIL_OK;
}

// ---- dovetail_tree_replay_static (include/dovetail.h): scratch that nobody allocates ---------------------------
// What dovetail_draft_init gets from cudaMalloc for the tree bookkeeping, laid out over ONE file-scope device
// array instead. Every GPU that loads the library holds these bytes until the process exits; every call on a
// device shares them and finds the previous call's contents (the entry point clears what must start clean).
struct ReplayScratch {
  int32_t pool_token[DOVETAIL_STATIC_MAX_POOL];
  int32_t pool_parent[DOVETAIL_STATIC_MAX_POOL];
  int32_t pool_depth[DOVETAIL_STATIC_MAX_POOL];
  float pool_cum[DOVETAIL_STATIC_MAX_POOL];
  int32_t pool_row[DOVETAIL_STATIC_MAX_POOL];
  int32_t out_pool_idx[DOVETAIL_STATIC_MAX_POOL];
  uint32_t treemask[kMaxTreeSlots * kMaskWords];
  RowTables rt[2];
  TreeState ts;
};
static_assert(sizeof(ReplayScratch) <= DOVETAIL_STATIC_SCRATCH_BYTES, "the stated scratch size must hold the layout");
static_assert(DOVETAIL_STATIC_MAX_POOL <= kPoolSmem, "k_tree_level stages the pool's scores in shared memory");
static __device__ __align__(256) unsigned char g_replay_scratch[DOVETAIL_STATIC_SCRATCH_BYTES];

// In host code `g_replay_scratch` is only a stand-in for the symbol, NOT a device address: a kernel handed it would
// fault (or, where the GPU can reach host memory, quietly use the wrong bytes). The device address is looked up
// once per device, with that device current, and kept.
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
ReplayScratch* g_static_ptr[kStaticMaxDevices] = {};

int replay_scratch(ReplayScratch** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(nullptr, DOVETAIL_ECUDA, "no CUDA device: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kStaticMaxDevices) return fail(nullptr, DOVETAIL_ECUDA, "device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (g_static_ptr[dev] == nullptr) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_replay_scratch);
    if (e != cudaSuccess || p == nullptr)
      return fail(nullptr, DOVETAIL_ECUDA, "cudaGetSymbolAddress(static scratch) failed on device %d: %s", dev,
                  cudaGetErrorString(e));
    g_static_ptr[dev] = static_cast<ReplayScratch*>(p);
  }
  *out = g_static_ptr[dev];
  return DOVETAIL_OK;
}

}  // namespace

extern "C" {

int dovetail_draft_init(const dovetail_weights_t* w, const dovetail_config_t* cfg, dovetail_draft_t** out) {
  if (out) *out = nullptr;
  if (!w || !cfg || !out) return fail(nullptr, DOVETAIL_EINVAL, "null argument");
  const dovetail_config_t& c = *cfg;
  if (c.hidden < 8 || c.n_q_heads < 1 || c.n_kv_heads < 1 || c.n_q_heads % c.n_kv_heads != 0 ||
      (c.head_dim != 64 && c.head_dim != 128) || c.n_layers < 1 || c.n_layers > DOVETAIL_MAX_LAYERS ||
      c.ffn < 8 || c.vocab < 1 || c.vocab > (1 << 24) - 2 || !(c.rope_theta > 0.f) || !(c.rms_eps >= 0.f) ||
      (c.dtype != DOVETAIL_F32 && c.dtype != DOVETAIL_BF16) ||
      (c.fusion != DOVETAIL_FUSION_DGF && c.fusion != DOVETAIL_FUSION_CONCAT_LINEAR) ||
      (c.fusion == DOVETAIL_FUSION_CONCAT_LINEAR && c.dgf_proj))
    return fail(nullptr, DOVETAIL_EINVAL, "bad model shape");
  if (c.max_rows < 1 || c.max_rows > kMaxRows || c.max_tree_slots < 0 || c.max_tree_slots > kMaxTreeSlots ||
      c.max_branch < 1 || c.max_branch > kMaxBranch)
    return fail(nullptr, DOVETAIL_EINVAL, "max_rows / max_tree_slots / max_branch out of range (<= 64 / 128 / 32)");
  const int es = c.dtype == DOVETAIL_BF16 ? 2 : 4;
  const int dq = c.n_q_heads * c.head_dim, dkv = c.n_kv_heads * c.head_dim;
  const int Ks[4] = {c.hidden, 2 * c.hidden, dq, c.ffn};
  for (int K : Ks)
    if (!gemv_shape(K, es, 1, 1).ok)
      return fail(nullptr, DOVETAIL_EINVAL, "dimension %d not supported: rows must be a multiple of 16 bytes and at most 28672 bytes", K);
  if (c.weight_quant < 0 || c.weight_quant > 2) return fail(nullptr, DOVETAIL_EINVAL, "weight_quant must be 0, 1 (int8) or 2 (fp8 e4m3)");
  if (c.weight_quant) {
    if (c.dtype != DOVETAIL_BF16) return fail(nullptr, DOVETAIL_EINVAL, "weight_quant != 0 needs dtype = BF16");
    for (int K : Ks)
      if (K % 32 != 0) return fail(nullptr, DOVETAIL_EINVAL, "weight_quant != 0: dimension %d is not a multiple of 32", K);
    bool ok = w->dgf_sg && w->lm_head_s && (!c.dgf_proj || (w->dgf_s1 && w->dgf_s2));
    for (int l = 0; ok && w->layers && l < c.n_layers; ++l) {
      const dovetail_layer_weights_t& L = w->layers[l];
      ok = L.sq && L.sk && L.sv && L.so && L.sgate && L.sup && L.sdown;
    }
    if (!ok) return fail(nullptr, DOVETAIL_EINVAL, "weight_quant != 0: missing scale pointer");
  }
  if (!w->embed || !w->dgf_wg || !w->dgf_bg || !w->layers || !w->lm_head ||
      (c.dgf_proj && (!w->dgf_w1 || !w->dgf_w2)) || (c.final_norm && !w->g_final))
    return fail(nullptr, DOVETAIL_EINVAL, "missing weight pointer");
  for (int l = 0; l < c.n_layers; ++l) {
    const dovetail_layer_weights_t& L = w->layers[l];
    if (!L.g_attn || !L.wq || !L.wk || !L.wv || !L.wo || !L.g_ffn || !L.wgate || !L.wup || !L.wdown)
      return fail(nullptr, DOVETAIL_EINVAL, "missing weight pointer in layer %d", l);
  }
  int dev = 0;
  cudaDeviceProp prop{};
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
  if (e != cudaSuccess) return fail(nullptr, DOVETAIL_ECUDA, "no CUDA device: %s", cudaGetErrorString(e));
  if (prop.major != 10)
    return fail(nullptr, DOVETAIL_ECUDA, "device %s is sm_%d%d; this library is built for sm_100a only", prop.name, prop.major, prop.minor);

  dovetail_draft* h = new (std::nothrow) dovetail_draft();
  if (!h) return fail(nullptr, DOVETAIL_ENOMEM, "out of host memory");
  h->cfg = c;
  h->w = *w;
  h->layers.assign(w->layers, w->layers + c.n_layers);
  h->w.layers = h->layers.data();
  h->num_sms = prop.multiProcessorCount;
  h->es = es;
  h->wq = c.weight_quant;
  h->dq = dq;
  h->dkv = dkv;
  h->ldq = dq + 2 * dkv;
  h->max_step_rows = c.max_rows + c.max_tree_slots;
  h->pool_cap = c.max_branch + c.max_tree_slots * c.max_branch;
  const int grp = c.n_q_heads / c.n_kv_heads;
  h->attn_chunks_cap = std::max(1, 2 * h->num_sms / c.n_kv_heads);
  h->qv_cap = c.max_rows * grp;

  e = set_max_smem_all();
  const size_t R = c.max_rows, d = c.hidden;
  auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  A(dmalloc(&h->dyn, 1));
  A(dmalloc(&h->ts, 1));
  A(dmalloc(&h->rt, 2));
  A(dmalloc(&h->rope, static_cast<size_t>(kMaxRows + kMaxDepth) * (c.head_dim / 2)));
  A(dmalloc(&h->inv_freq, c.head_dim / 2));
  A(dmalloc(&h->hbuf, R * 2 * d));
  A(dmalloc(&h->hhat, static_cast<size_t>(h->max_step_rows) * d));
  A(dmalloc(&h->qkv, R * h->ldq));
  A(dmalloc(&h->obuf, R * dq));
  A(dmalloc(&h->act, R * c.ffn));
  auto up8 = [](int k) { return (k + 7) / 8 * 8; };
  h->ld_d = up8(c.hidden); h->ld_2d = up8(2 * c.hidden); h->ld_dq = up8(dq); h->ld_f = up8(c.ffn);
  if (es == 2) {
    A(dmalloc(&h->xs_feat, kSplitPlanes * R * h->ld_d));
    A(dmalloc(&h->xs_hhat, static_cast<size_t>(kSplitPlanes) * h->max_step_rows * h->ld_d));
    A(dmalloc(&h->xs_x, kSplitPlanes * R * h->ld_d));
    A(dmalloc(&h->xs_h12, kSplitPlanes * R * h->ld_2d));
    A(dmalloc(&h->xs_o, kSplitPlanes * R * h->ld_dq));
    A(dmalloc(&h->xs_act, kSplitPlanes * R * h->ld_f));
    A(dmalloc(&h->ssq, static_cast<size_t>(h->num_sms) * kMaxRows));
    A(dmalloc(&h->qs, static_cast<size_t>(2) * kMaxRows * dq));
    A(dmalloc(&h->xs_emb, kSplitPlanes * R * h->ld_d));
    if (!c.weight_quant) A(dmalloc(&h->xs_par, kSplitPlanes * R * h->ld_d));
  }
  A(dmalloc(&h->attn_ws, static_cast<size_t>(c.n_kv_heads) * h->attn_chunks_cap * h->qv_cap * (c.head_dim + 4)));
  A(dmalloc(&h->attn_cnt, c.n_kv_heads));
  A(dmalloc(&h->cand_val, R * h->num_sms * kMaxBranch));
  A(dmalloc(&h->cand_id, R * h->num_sms * kMaxBranch));
  A(dmalloc(&h->stat, R * h->num_sms * 2));
  A(dmalloc(&h->pool.token, h->pool_cap));
  A(dmalloc(&h->pool.parent, h->pool_cap));
  A(dmalloc(&h->pool.depth, h->pool_cap));
  A(dmalloc(&h->pool.cum, h->pool_cap));
  A(dmalloc(&h->pool.row, h->pool_cap));
  A(dmalloc(&h->treemask, static_cast<size_t>(kMaxTreeSlots) * kMaskWords));
  A(dmalloc(&h->out_pool_idx, h->pool_cap));
  A(cudaMallocHost(reinterpret_cast<void**>(&h->ts_host), sizeof(TreeState)));
  if (e == cudaSuccess) e = cudaMemset(h->attn_cnt, 0, sizeof(int32_t) * c.n_kv_heads);
  if (e == cudaSuccess) e = cudaMemset(h->ts, 0, sizeof(TreeState));
  if (e == cudaSuccess) {
    // theta^(-2i/dh) in fp64, the expression the rotary definition states (reading A3)
    std::vector<double> inv(c.head_dim / 2);
    for (int i = 0; i < c.head_dim / 2; ++i)
      inv[i] = std::pow(static_cast<double>(c.rope_theta), -2.0 * i / c.head_dim);
    e = cudaMemcpy(h->inv_freq, inv.data(), inv.size() * sizeof(double), cudaMemcpyHostToDevice);
  }
  if (e != cudaSuccess) {
    const int code = e == cudaErrorMemoryAllocation ? DOVETAIL_ENOMEM : DOVETAIL_ECUDA;
    fail(nullptr, code, "init failed: %s", cudaGetErrorString(e));
    cudaGetLastError();
    free_all(h);
    delete h;
    return code;
  }
  if (es == 2 && !c.weight_quant) umma_init(h);
  if (es == 2) {  // how many clusters of each size the tensor-core attention kernel can have resident (attn_mma_geom)
    for (int mode = 0; mode < 3; ++mode)
      for (int cs = 1; cs <= 8; ++cs) {
        const int qt = mode == 1 ? 4 : (mode == 2 ? 2 : 1);
        cudaLaunchConfig_t lc{};
        lc.gridDim = dim3(cs, c.n_kv_heads);
        lc.blockDim = dim3(kAmThreads);
        lc.dynamicSmemBytes = am_smem_bytes(c.head_dim, qt);
        cudaLaunchAttribute at{};
        at.id = cudaLaunchAttributeClusterDimension;
        at.val.clusterDim.x = cs;
        at.val.clusterDim.y = 1;
        at.val.clusterDim.z = 1;
        lc.attrs = &at;
        lc.numAttrs = 1;
        const void* fn = reinterpret_cast<const void*>(attn_mma_kernel(c.head_dim, qt));
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, fn, &lc) == cudaSuccess) h->attn_max_clusters[mode][cs] = n;
        else cudaGetLastError();
      }
  }
  *out = h;
  return DOVETAIL_OK;
}

int dovetail_draft_step(dovetail_draft_t* h, const float* hidden_feats, const int32_t* tokens, int32_t n_new,
                        dovetail_kv_cache_t* kv, const dovetail_tree_spec_t* tree,
                        const dovetail_draft_out_t* out, void* cuda_stream) {
  NvtxRange nvtx_range("dovetail_draft_step");
  if (!h) return DOVETAIL_EINVAL;
  if (!hidden_feats || !tokens || !kv || !tree || !out || !kv->k || !kv->v || !out->token_ids ||
      !out->scores || !out->parents || !out->n_out)
    return fail(h, DOVETAIL_EINVAL, "null argument");
  const dovetail_config_t& c = h->cfg;
  if (n_new < 1 || n_new > c.max_rows) return fail(h, DOVETAIL_EINVAL, "n_new = %d out of range [1, %d]", n_new, c.max_rows);
  if (kv->committed_len < 0 || kv->capacity < 1) return fail(h, DOVETAIL_EINVAL, "bad KV cache state");
  std::vector<LevelPlan> plan;
  int tree_rows = 0, pool_total = 0;
  int rc = validate_tree(h, tree, n_new, plan, tree_rows, pool_total);
  if (rc != DOVETAIL_OK) return rc;
  const int L = kv->committed_len, Lp = L + n_new;
  if (static_cast<long>(Lp) + tree_rows > kv->capacity)
    return fail(h, DOVETAIL_ECAPACITY, "KV cache too small: %d committed + %d new + %d tree rows > capacity %d", L, n_new, tree_rows, kv->capacity);

  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  h->last_graph = 0;
  if (h->graphs_on && !h->hooks_on && !h->trace_on) {
    rc = step_by_graph(h, st, hidden_feats, tokens, n_new, kv, tree, out, plan, pool_total);
    if (rc != DOVETAIL_OK) return rc;
  } else {
    // Pass 1 checks every shape of the plan without launching (on error nothing was enqueued);
    // pass 2 enqueues.
    for (int pass = 0; pass < 2; ++pass) {
      h->dry = pass == 0;
      rc = enqueue_step(h, st, hidden_feats, tokens, n_new, kv, tree, out, plan, pool_total);
      h->dry = false;
      if (rc != DOVETAIL_OK) return rc;
    }
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "CUDA error: %s", cudaGetErrorString(e));
  kv->committed_len = Lp;  // the level-0 rows are real, verified tokens
  h->have_step = true;
  h->last_n_new = n_new;
  h->last_depth = tree->depth;
  h->last_gamma = tree->gamma;
  h->last_launches = h->launches;
  h->last_umma_launches = h->umma_launches;
  h->last_ksplit_launches = h->ksplit_launches;
  return DOVETAIL_OK;
}

int dovetail_draft_prefill(dovetail_draft_t* h, const float* hidden_feats, const int32_t* tokens, int32_t n_rows,
                           dovetail_kv_cache_t* kv, void* cuda_stream) {
  NvtxRange nvtx_range("dovetail_draft_prefill");
  if (!h) return DOVETAIL_EINVAL;
  if (!hidden_feats || !tokens || !kv || !kv->k || !kv->v) return fail(h, DOVETAIL_EINVAL, "null argument");
  if (n_rows < 1) return fail(h, DOVETAIL_EINVAL, "n_rows = %d: at least one row", n_rows);
  if (kv->committed_len < 0 || kv->capacity < 1) return fail(h, DOVETAIL_EINVAL, "bad KV cache state");
  if (static_cast<long>(kv->committed_len) + n_rows > kv->capacity)
    return fail(h, DOVETAIL_ECAPACITY, "KV cache too small: %d committed + %d rows > capacity %d", kv->committed_len, n_rows, kv->capacity);
  const dovetail_config_t& c = h->cfg;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  dovetail_tree_spec_t tree{};
  tree.depth = 1;
  tree.branch[0] = 1;
  tree.gamma = 1;
  const dovetail_draft_out_t out{};
  std::vector<LevelPlan> plan(1);
  // shapes of a full batch and of the ragged last one are checked before anything is enqueued
  const int sizes[2] = {std::min(n_rows, c.max_rows), n_rows % c.max_rows};
  for (int n : sizes) {
    if (n < 1) continue;
    plan[0] = LevelPlan{n, 1, 0, 0, 0};
    h->dry = true;
    const int rc = enqueue_step(h, st, hidden_feats, tokens, n, kv, &tree, &out, plan, 0, true);
    h->dry = false;
    if (rc != DOVETAIL_OK) return rc;
  }
  int launches = 0, umma = 0;
  for (int r0 = 0; r0 < n_rows; r0 += c.max_rows) {
    const int n = std::min(c.max_rows, n_rows - r0);
    plan[0] = LevelPlan{n, 1, 0, 0, 0};
    const int rc = enqueue_step(h, st, hidden_feats + static_cast<size_t>(r0) * c.hidden, tokens + r0, n, kv, &tree, &out, plan, 0, true);
    if (rc != DOVETAIL_OK) return rc;
    kv->committed_len += n;
    launches += h->launches;
    umma += h->umma_launches;
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "CUDA error: %s", cudaGetErrorString(e));
  h->have_step = false;
  h->last_launches = launches;
  h->last_umma_launches = umma;
  return DOVETAIL_OK;
}

int dovetail_kv_commit(dovetail_draft_t* h, dovetail_kv_cache_t* kv, const int32_t* accepted_path, int32_t n_acc,
                       int32_t mode, int32_t* n_committed, void* cuda_stream) {
  NvtxRange nvtx_range("dovetail_kv_commit");
  if (!h) return DOVETAIL_EINVAL;
  if (n_committed) *n_committed = 0;
  if (!kv || !kv->k || !kv->v || (n_acc > 0 && !accepted_path)) return fail(h, DOVETAIL_EINVAL, "null argument");
  if (mode != 0 && mode != 1) return fail(h, DOVETAIL_EINVAL, "mode must be 0 or 1");
  if (!h->have_step) return fail(h, DOVETAIL_EINVAL, "no draft step to commit");
  if (n_acc < 0 || n_acc > h->last_depth) return fail(h, DOVETAIL_EINVAL, "n_acc = %d out of range [0, depth %d]", n_acc, h->last_depth);
  for (int i = 0; i < n_acc; ++i)
    if (accepted_path[i] < 0 || accepted_path[i] >= h->last_gamma)
      return fail(h, DOVETAIL_EINVAL, "accepted_path[%d] = %d is not an output index", i, accepted_path[i]);
  if (mode == 0) {  // the paper's flow: tree rows are simply dead
    h->have_step = false;
    return DOVETAIL_OK;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const dovetail_config_t& c = h->cfg;
  CommitPath path{};
  path.n = n_acc;
  for (int i = 0; i < n_acc; ++i) path.idx[i] = accepted_path[i];
  const int row_bytes = c.head_dim * h->es;
  k_commit_plan<<<1, 32, 0, st>>>(path, h->ts, h->pool, h->out_pool_idx, h->last_n_new);
  k_commit_move<<<dim3(c.n_layers * c.n_kv_heads, 2), 128, static_cast<size_t>(kMaxDepth + 1) * row_bytes, st>>>(
      h->ts, kv->k, kv->v, kv->capacity, kv->committed_len, row_bytes);
  cudaError_t e = cudaMemcpyAsync(h->ts_host, h->ts, sizeof(TreeState), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "kv_commit failed: %s", cudaGetErrorString(e));
  if (h->ts_host->commit_err) return fail(h, DOVETAIL_EINVAL, "accepted_path is not a root-to-node chain of the last step's output");
  kv->committed_len += h->ts_host->commit_n;
  if (n_committed) *n_committed = h->ts_host->commit_n;
  h->have_step = false;
  return DOVETAIL_OK;
}

int dovetail_verify_plan(dovetail_draft_t* h, const dovetail_draft_out_t* out, int32_t gamma, int32_t root_position,
                         int32_t max_depth, const dovetail_verify_plan_t* plan, void* cuda_stream) {
  NvtxRange nvtx_range("dovetail_verify_plan");
  if (!h) return DOVETAIL_EINVAL;
  if (!out || !out->parents || !out->depths || !out->n_out || !plan || !plan->mask || !plan->position_ids || !plan->paths ||
      !plan->n_paths)
    return fail(h, DOVETAIL_EINVAL, "null argument (the step's output must include depths)");
  if (gamma < 1 || gamma > h->pool_cap || max_depth < 1) return fail(h, DOVETAIL_EINVAL, "gamma / max_depth out of range");
  VerifyPlanParams p{};
  p.parents = out->parents;
  p.depths = out->depths;
  p.n_out = out->n_out;
  p.gamma = gamma;
  p.root_position = root_position;
  p.max_depth = max_depth;
  p.mask = plan->mask;
  p.position_ids = plan->position_ids;
  p.paths = plan->paths;
  p.n_paths = plan->n_paths;
  k_verify_plan<<<1, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(p);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "verify_plan launch failed: %s", cudaGetErrorString(e));
  return DOVETAIL_OK;
}

int dovetail_verify_accept(dovetail_draft_t* h, const dovetail_draft_out_t* out, int32_t gamma, int32_t mode, int32_t max_depth,
                           const dovetail_verify_in_t* in, const dovetail_verify_out_t* res, void* cuda_stream) {
  NvtxRange nvtx_range("dovetail_verify_accept");
  if (!h) return DOVETAIL_EINVAL;
  if (!out || !out->token_ids || !out->parents || !out->n_out || !in || !res || !res->accepted_path || !res->n_acc ||
      !res->bonus_token)
    return fail(h, DOVETAIL_EINVAL, "null argument");
  if (mode != 0 && mode != 1) return fail(h, DOVETAIL_EINVAL, "mode must be 0 (greedy) or 1 (speculative sampling)");
  if (mode == 0 && !in->tgt_argmax) return fail(h, DOVETAIL_EINVAL, "greedy acceptance needs tgt_argmax");
  if (mode == 1 && (!in->p_cand || !in->uniforms || !in->p_full)) return fail(h, DOVETAIL_EINVAL, "sampling needs p_cand, uniforms, p_full");
  if (gamma < 1 || gamma > h->pool_cap || max_depth < 1) return fail(h, DOVETAIL_EINVAL, "gamma / max_depth out of range");
  VerifyAcceptParams p{};
  p.token_ids = out->token_ids;
  p.parents = out->parents;
  p.n_out = out->n_out;
  p.gamma = gamma;
  p.mode = mode;
  p.vocab = h->cfg.vocab;
  p.tgt_argmax = in->tgt_argmax;
  p.p_cand = in->p_cand;
  p.uniforms = in->uniforms;
  p.p_full = in->p_full;
  p.accepted_path = res->accepted_path;
  p.n_acc = res->n_acc;
  p.bonus_token = res->bonus_token;
  p.max_depth = max_depth;
  k_verify_accept<<<1, kVerifyThreads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(p);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "verify_accept launch failed: %s", cudaGetErrorString(e));
  return DOVETAIL_OK;
}

int dovetail_tree_replay(dovetail_draft_t* h, const dovetail_tree_spec_t* tree, const int32_t* cand_tokens,
                         const float* cand_logp, int32_t n_rows, int32_t max_b, const dovetail_draft_out_t* out,
                         int32_t* pool_token, int32_t* pool_parent, int32_t* pool_depth, float* pool_cum,
                         int32_t* pool_size, void* cuda_stream) {
  if (!h) return DOVETAIL_EINVAL;
  if (!tree || !cand_tokens || !cand_logp || !out || !out->token_ids || !out->scores || !out->parents || !out->n_out)
    return fail(h, DOVETAIL_EINVAL, "null argument");
  std::vector<LevelPlan> plan;
  int tree_rows = 0, pool_total = 0;
  int rc = validate_tree(h, tree, 1, plan, tree_rows, pool_total);
  if (rc != DOVETAIL_OK) return rc;
  int need_rows = 1;  // rows consumed: the root and every forwarded row of levels 1 .. D-1
  for (int l = 1; l < tree->depth; ++l) need_rows += plan[l].rows;
  int maxb = 0;
  for (int l = 0; l < tree->depth; ++l) maxb = std::max(maxb, tree->branch[l]);
  if (n_rows < need_rows || max_b < maxb) return fail(h, DOVETAIL_EINVAL, "replay needs %d rows of %d candidates", need_rows, maxb);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  h->launches = 0;
  h->cur_kind = 9;
  h->cur_bytes = 0;
  const bool trace_was = h->trace_on;
  h->trace_on = false;  // the replay is not part of the traced step
  cudaError_t e = cudaMemsetAsync(h->rt, 0xff, sizeof(RowTables), st);  // level-0 row: pool = -1
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "memset failed: %s", cudaGetErrorString(e));
  int row = 0;
  for (int l = 0; l < tree->depth; ++l) {
    const LevelPlan& lp = plan[l];
    TreeLevelParams t{};
    t.dyn = h->dyn;
    t.ts = h->ts;
    t.pool = h->pool;
    t.treemask = h->treemask;
    t.rp_tokens = cand_tokens;
    t.rp_logp = cand_logp;
    t.rp_maxb = max_b;
    t.rp_row0 = row;
    t.M = lp.rows_lm;
    t.b = tree->branch[l];
    t.level = l;
    t.pool_begin = lp.pool_begin;
    const bool last = l + 1 == tree->depth;
    t.M_next = last ? 0 : plan[l + 1].rows;
    t.next_row0 = last ? 0 : plan[l + 1].row0;
    t.cur_row0 = lp.row0;
    t.next_t0 = last ? 0 : plan[l + 1].t0;
    t.n_new = 1;
    t.cur = h->rt + (l & 1);
    t.next = h->rt + ((l + 1) & 1);
    t.gamma = tree->gamma;
    t.pool_total = pool_total;
    t.out_pool_idx = h->out_pool_idx;
    t.o_ids = out->token_ids;
    t.o_scores = out->scores;
    t.o_parents = out->parents;
    t.o_depths = out->depths;
    t.o_n = out->n_out;
    e = launch(h, k_tree_level, dim3(1), dim3(kTreeThreads), 0, st, t);
    if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "tree launch failed: %s", cudaGetErrorString(e));
    row += lp.rows_lm;
  }
  auto cp = [&](void* dst, const void* src, size_t n) {
    if (dst && e == cudaSuccess) e = cudaMemcpyAsync(dst, src, n, cudaMemcpyDeviceToDevice, st);
  };
  cp(pool_token, h->pool.token, sizeof(int32_t) * pool_total);
  cp(pool_parent, h->pool.parent, sizeof(int32_t) * pool_total);
  cp(pool_depth, h->pool.depth, sizeof(int32_t) * pool_total);
  cp(pool_cum, h->pool.cum, sizeof(float) * pool_total);
  cp(pool_size, &h->ts->pool_size, sizeof(int32_t));
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "copy failed: %s", cudaGetErrorString(e));
  h->have_step = false;
  h->last_launches = h->launches;
  h->trace_on = trace_was;
  return DOVETAIL_OK;
}

// No allocation on this path: no cudaMalloc / cudaFree, no std::vector, no handle. (begin: no-alloc entry point)
int dovetail_tree_replay_static(const dovetail_tree_spec_t* tree, const int32_t* cand_tokens, const float* cand_logp,
                                int32_t n_rows, int32_t max_b, const dovetail_draft_out_t* out, void* cuda_stream) {
  if (!tree || !cand_tokens || !cand_logp || !out || !out->token_ids || !out->scores || !out->parents || !out->n_out)
    return fail(nullptr, DOVETAIL_EINVAL, "null argument");
  // the level plan of validate_tree with n_new = 1, against the compile-time limits of the static scratch
  if (tree->depth < 1 || tree->depth > DOVETAIL_MAX_DEPTH)
    return fail(nullptr, DOVETAIL_EINVAL, "tree depth %d out of range [1, %d]", tree->depth, DOVETAIL_MAX_DEPTH);
  if (tree->gamma < 1) return fail(nullptr, DOVETAIL_EINVAL, "gamma must be >= 1");
  LevelPlan plan[DOVETAIL_MAX_DEPTH];
  int m = 1, tree_rows = 0, need_rows = 1, maxb = 0;
  long pool = 0;
  for (int l = 0; l < tree->depth; ++l) {
    if (tree->branch[l] < 1 || tree->branch[l] > kMaxBranch)
      return fail(nullptr, DOVETAIL_EINVAL, "branch[%d] = %d out of range [1, %d]", l, tree->branch[l], kMaxBranch);
    maxb = std::max(maxb, tree->branch[l]);
    if (l >= 1) {
      if (tree->beam[l] < 0) return fail(nullptr, DOVETAIL_EINVAL, "beam[%d] negative", l);
      const long n = static_cast<long>(m) * tree->branch[l - 1];
      const long mm = (tree->beam[l] > 0 && tree->beam[l] < n) ? tree->beam[l] : n;
      if (mm > kMaxRows)
        return fail(nullptr, DOVETAIL_EINVAL, "level %d forwards %ld rows > the static limit of %d rows per level", l, mm, kMaxRows);
      m = static_cast<int>(mm);
      plan[l] = LevelPlan{m, m, 1 + tree_rows, tree_rows, 0};
      tree_rows += m;
      need_rows += m;
    } else {
      plan[0] = LevelPlan{1, 1, 0, 0, 0};
    }
    plan[l].pool_begin = static_cast<int>(pool);
    pool += static_cast<long>(plan[l].rows_lm) * tree->branch[l];
    if (tree_rows > kMaxTreeSlots)
      return fail(nullptr, DOVETAIL_EINVAL, "tree forwards %d rows > the static limit of %d tree rows", tree_rows, kMaxTreeSlots);
    if (pool > DOVETAIL_STATIC_MAX_POOL)
      return fail(nullptr, DOVETAIL_EINVAL, "candidate pool of %ld nodes exceeds DOVETAIL_STATIC_MAX_POOL = %d (the static scratch is %d bytes)",
                  pool, DOVETAIL_STATIC_MAX_POOL, DOVETAIL_STATIC_SCRATCH_BYTES);
  }
  if (n_rows < need_rows || max_b < maxb)
    return fail(nullptr, DOVETAIL_EINVAL, "replay needs %d rows of %d candidates", need_rows, maxb);
  ReplayScratch* sc = nullptr;
  const int rc = replay_scratch(&sc);
  if (rc != DOVETAIL_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  // the array keeps the previous call's contents: the level-0 row table (pool = -1: the root) and the bookkeeping
  // state start clean; everything else (pool entries, masks, the other row table) is written before it is read
  cudaError_t e = cudaMemsetAsync(&sc->rt[0], 0xff, sizeof(RowTables), st);
  if (e == cudaSuccess) e = cudaMemsetAsync(&sc->ts, 0, sizeof(TreeState), st);
  if (e != cudaSuccess) return fail(nullptr, DOVETAIL_ECUDA, "memset failed: %s", cudaGetErrorString(e));
  int row = 0;
  for (int l = 0; l < tree->depth; ++l) {
    const LevelPlan& lp = plan[l];
    const bool last = l + 1 == tree->depth;
    TreeLevelParams t{};
    t.dyn = nullptr;  // never read: the explicit outputs below are set
    t.ts = &sc->ts;
    t.pool = Pool{sc->pool_token, sc->pool_parent, sc->pool_depth, sc->pool_cum, sc->pool_row};
    t.treemask = sc->treemask;
    t.rp_tokens = cand_tokens;
    t.rp_logp = cand_logp;
    t.rp_maxb = max_b;
    t.rp_row0 = row;
    t.M = lp.rows_lm;
    t.b = tree->branch[l];
    t.level = l;
    t.pool_begin = lp.pool_begin;
    t.M_next = last ? 0 : plan[l + 1].rows;
    t.next_row0 = last ? 0 : plan[l + 1].row0;
    t.cur_row0 = lp.row0;
    t.next_t0 = last ? 0 : plan[l + 1].t0;
    t.n_new = 1;
    t.cur = &sc->rt[l & 1];
    t.next = &sc->rt[(l + 1) & 1];
    t.gamma = tree->gamma;
    t.pool_total = static_cast<int>(pool);
    t.out_pool_idx = sc->out_pool_idx;
    t.o_ids = out->token_ids;
    t.o_scores = out->scores;
    t.o_parents = out->parents;
    t.o_depths = out->depths;
    t.o_n = out->n_out;
    k_tree_level<<<1, kTreeThreads, 0, st>>>(t);  // plain stream order: each level sees the one before it complete
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, DOVETAIL_ECUDA, "tree launch failed: %s", cudaGetErrorString(e));
    row += lp.rows_lm;
  }
  return DOVETAIL_OK;
}
// (end: no-alloc entry point)

int dovetail_hooks_set(dovetail_draft_t* h, const dovetail_hooks_t* hooks) {
  if (!h) return DOVETAIL_EINVAL;
  h->hooks = hooks ? *hooks : dovetail_hooks_t{};
  const dovetail_hooks_t& k = h->hooks;
  if ((k.tap_pool_token == nullptr) != (k.tap_pool_cum == nullptr) ||
      (k.force_pool_token == nullptr) != (k.force_pool_cum == nullptr)) {
    h->hooks = dovetail_hooks_t{};
    h->hooks_on = false;
    return fail(h, DOVETAIL_EINVAL, "pool taps / forcing need both the token and the score array");
  }
  h->hooks_on = k.tap_logits || k.tap_hhat || k.tap_k || k.tap_v || k.tap_pool_token || k.force_hhat || k.force_k ||
                k.force_v || k.force_pool_token;
  return DOVETAIL_OK;
}

int dovetail_last_launch_count(const dovetail_draft_t* h) { return h ? h->last_launches : 0; }

int dovetail_hooks_umma_tables(const int32_t rows[3], int32_t n_mat, int32_t paired, int32_t pairperm, int32_t ctas,
                               int32_t* n_sb, int32_t* n_grp, int32_t* grp, uint16_t* vpos, int32_t vpos_cap, int32_t* vpos_ld,
                               int32_t* cnt) {
  if (!rows || n_mat < 1 || n_mat > 3 || ctas < 1 || !n_sb || !n_grp || !grp || !vpos || !vpos_ld || !cnt) return DOVETAIL_EINVAL;
  GemvGroup G{};
  long tot = 0;
  for (int j = 0; j < n_mat; ++j) { G.rows[j] = rows[j]; tot += rows[j]; }
  G.n_mat = n_mat;
  G.paired = paired;
  G.pairperm = pairperm;
  const long units = paired ? rows[0] : tot / (pairperm ? 2 : 1);  // the dealing of run_gemv
  G.deal_base = static_cast<int32_t>(units / ctas);
  G.deal_rem = static_cast<int32_t>(units % ctas);
  std::vector<UmmaCtaTab> tabs;
  std::vector<uint16_t> vp;
  int ld = 0, g_max = 0, g_min = 0;
  if (!build_umma_tables(G, ctas, tabs, vp, ld, g_max, g_min)) return DOVETAIL_ECAPACITY;
  if (static_cast<long>(ctas) * ld > vpos_cap) return DOVETAIL_ECAPACITY;
  *vpos_ld = ld;
  for (int c = 0; c < ctas; ++c) {
    n_sb[c] = tabs[c].n_sb;
    cnt[c] = cta_rows(G, c, ctas).cnt;
    memcpy(n_grp + static_cast<size_t>(c) * kUmmaMaxSb, tabs[c].n_grp, sizeof tabs[c].n_grp);
    memcpy(grp + static_cast<size_t>(c) * kUmmaMaxSb * kUmmaMaxGroups, tabs[c].grp, sizeof tabs[c].grp);
  }
  memcpy(vpos, vp.data(), vp.size() * sizeof(uint16_t));
  return DOVETAIL_OK;
}

int dovetail_hooks_stat(const dovetail_draft_t* h, int32_t key) {
  if (!h) return -1;
  if (key == DOVETAIL_STAT_UMMA_LAUNCHES) return h->last_umma_launches;
  if (key == DOVETAIL_STAT_GRAPH) return h->last_graph;
  if (key == DOVETAIL_STAT_KSPLIT_LAUNCHES) return h->last_ksplit_launches;
  return -1;
}

int dovetail_hooks_tune(dovetail_draft_t* h, int32_t key, int32_t value) {
  if (!h) return DOVETAIL_EINVAL;
  if (key == DOVETAIL_TUNE_UMMA_MIN_M && value >= 1 && value <= kUmmaMaxM + 1) {
    if (!h->maps_dev && value <= kUmmaMaxM) return fail(h, DOVETAIL_EINVAL, "the tcgen05 path is not available for this model");
    h->umma_min_m = value;
    return DOVETAIL_OK;
  }
  if (key == DOVETAIL_TUNE_GRAPHS && (value == 0 || value == 1)) { h->graphs_on = value != 0; return DOVETAIL_OK; }
  if (key == DOVETAIL_TUNE_UMMA_KSPLIT_MIN_M && value >= 1 && value <= kUmmaMaxM + 1) { h->umma_ksplit_min_m = value; return DOVETAIL_OK; }
  if (key == DOVETAIL_TUNE_ATTN_QT2 && (value == 0 || value == 1)) { h->attn_qt2 = value; return DOVETAIL_OK; }
  if (key == DOVETAIL_TUNE_ATTN_WIDE_MIN && value >= 0 && value <= 4096) { h->attn_wide_min = value; return DOVETAIL_OK; }
  return fail(h, DOVETAIL_EINVAL, "unknown knob %d or value %d out of range", key, value);
}

int dovetail_draft_status(dovetail_draft_t* h, void* cuda_stream) {
  if (!h) return DOVETAIL_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  cudaError_t e = cudaMemcpyAsync(h->ts_host, h->ts, sizeof(TreeState), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(&h->ts->status, 0, sizeof(int32_t), st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "status read failed: %s", cudaGetErrorString(e));
  if (h->ts_host->status & 1)
    return fail(h, DOVETAIL_EINVAL, "a token id passed to dovetail_draft_step was outside [0, vocab = %d)", h->cfg.vocab);
  return DOVETAIL_OK;
}

int dovetail_trace_enable(dovetail_draft_t* h, int32_t enable) {
  if (!h) return DOVETAIL_EINVAL;
  if (enable && !h->trace_buf) {
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&h->trace_buf), sizeof(unsigned long long) * 2 * kMaxTraceLaunches);
    if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void**>(&h->trace_host), sizeof(unsigned long long) * 2 * kMaxTraceLaunches);
    if (e != cudaSuccess) return fail(h, DOVETAIL_ENOMEM, "trace buffer: %s", cudaGetErrorString(e));
  }
  h->trace_on = enable != 0;
  h->tr_used = 0;
  return DOVETAIL_OK;
}

int dovetail_trace_read(dovetail_draft_t* h, int32_t cap, int32_t* kind, int32_t* level, int64_t* bytes,
                        uint64_t* t0_ns, uint64_t* t1_ns, int32_t* n) {
  if (!h || !kind || !level || !bytes || !t0_ns || !t1_ns || !n || cap < 0)
    return h ? fail(h, DOVETAIL_EINVAL, "null argument") : DOVETAIL_EINVAL;
  *n = 0;
  if (!h->trace_buf || h->tr_used == 0) return DOVETAIL_OK;
  cudaError_t e = cudaMemcpy(h->trace_host, h->trace_buf, sizeof(unsigned long long) * 2 * h->tr_used, cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "trace read failed: %s", cudaGetErrorString(e));
  const int cnt = std::min(cap, h->tr_used);
  for (int i = 0; i < cnt; ++i) {
    kind[i] = h->tr_kind[i];
    level[i] = h->tr_level[i];
    bytes[i] = h->tr_bytes[i];
    t0_ns[i] = h->trace_host[2 * i];
    t1_ns[i] = h->trace_host[2 * i + 1];
  }
  *n = cnt;
  return DOVETAIL_OK;
}

int dovetail_probe_stream(dovetail_draft_t* h, const void* buf, int64_t bytes, int32_t mode, int32_t seg,
                          void* cuda_stream) {
  if (!h) return DOVETAIL_EINVAL;
  if (!buf || bytes < (1 << 20) || (reinterpret_cast<uintptr_t>(buf) & 15) || (mode != 0 && mode != 1))
    return fail(h, DOVETAIL_EINVAL, "probe: buffer must be 16-byte aligned and >= 1 MiB, mode 0 or 1");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  cudaError_t e = cudaSuccess;
  if (!h->probe_sink) e = cudaMalloc(reinterpret_cast<void**>(&h->probe_sink), sizeof(float));
  if (e != cudaSuccess) return fail(h, DOVETAIL_ENOMEM, "probe: %s", cudaGetErrorString(e));
  if (mode == 0) {
    k_stream_sum<<<h->num_sms * 4, 512, 0, st>>>(static_cast<const uint4*>(buf), bytes / 16, h->probe_sink);
  } else {
    if (seg < 512 || seg > 8192 || seg % 16) return fail(h, DOVETAIL_EINVAL, "probe: seg must be a multiple of 16 in [512, 8192]");
    const int rows = std::min(128, 32768 / seg * 2);           // ~64 KB stages, <= 32 segments per producer warp
    const int n_stages = std::min(8, (200 * 1024) / (rows * seg));
    const size_t smem = static_cast<size_t>(n_stages) * rows * seg + 128;
    e = cudaFuncSetAttribute(k_stream_bulk, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
    if (e == cudaSuccess)
      k_stream_bulk<<<h->num_sms, kProbeThreads, smem, st>>>(static_cast<const uint8_t*>(buf), bytes, seg, rows, n_stages, h->probe_sink);
  }
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, DOVETAIL_ECUDA, "probe launch failed: %s", cudaGetErrorString(e));
  return DOVETAIL_OK;
}

int64_t dovetail_forward_bytes(const dovetail_draft_t* h, int32_t prefix_len) {
  if (!h) return 0;
  const dovetail_config_t& c = h->cfg;
  const int64_t d = c.hidden, F = c.ffn, dq = h->dq, dkv = h->dkv;
  int64_t params = (c.dgf_proj ? 2 * d * d : 0) + 2 * d * d + d;  // DGF (4d^2 + d) or the concat + Linear fusion (2d^2 + d)
  params += static_cast<int64_t>(c.n_layers) * (d * dq + 2 * d * dkv + dq * d + 3 * d * F + 2 * d);
  params += static_cast<int64_t>(c.vocab) * d + (c.final_norm ? d : 0);
  const int64_t kvb = static_cast<int64_t>(c.n_layers) * 2 * prefix_len * dkv;
  if (h->wq) {  // matrices: one byte per element + one fp32 scale per output row; vectors and K/V in bf16
    const int64_t vec = d + static_cast<int64_t>(c.n_layers) * 2 * d + (c.final_norm ? d : 0);
    const int64_t rows = (c.dgf_proj ? 2 * d : 0) + d + static_cast<int64_t>(c.n_layers) * (dq + 2 * dkv + d + 2 * F + d) + c.vocab;
    return (params - vec) + 4 * rows + (vec + kvb) * h->es;
  }
  return (params + kvb) * h->es;
}

#ifdef DVT_CHAINDBG
int dovetail_dbg_read(dovetail_draft_t* h, unsigned long long* out, int n_launches) {
  return cudaMemcpy(out, h->dbg, sizeof(unsigned long long) * n_launches * 148 * 16, cudaMemcpyDeviceToHost);
}
#endif

void dovetail_draft_destroy(dovetail_draft_t* h) {
  if (!h) return;
  free_all(h);
  delete h;
}

const char* dovetail_last_error(const dovetail_draft_t* h) { return h ? h->err : g_init_error; }

}  // extern "C"

"""ctypes binding of libdovetail_draft.so -- the C ABI of include/dovetail.h with the
same names. Argument marshalling only: every step of the draft path runs in the
CUDA kernels behind these calls. torch tensors are used as owners of device
memory and for the current stream; there is no CPU fallback and no silent
substitute when the library is missing.
"""
import ctypes as C
import os
from typing import Dict, List, Optional

from .configs import BF16, DraftConfig, TreeSpec

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdovetail_draft.so")
MAX_DEPTH, MAX_LAYERS = 16, 16

OK, EINVAL, ECAPACITY, ECUDA, ENOMEM = 0, -1, -2, -3, -4

# include/dovetail.h
EXPORTS = ("dovetail_draft_init", "dovetail_draft_step", "dovetail_draft_prefill", "dovetail_kv_commit", "dovetail_tree_replay",
           "dovetail_tree_replay_static",
           "dovetail_verify_plan", "dovetail_verify_accept", "dovetail_draft_status", "dovetail_last_launch_count", "dovetail_forward_bytes",
           "dovetail_draft_destroy", "dovetail_last_error")
# include/dovetail_hooks.h (test and measurement hooks)
HOOK_EXPORTS = ("dovetail_hooks_set", "dovetail_trace_enable", "dovetail_trace_read", "dovetail_probe_stream", "dovetail_hooks_tune", "dovetail_hooks_stat", "dovetail_hooks_umma_tables")


class DovetailError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"dovetail error {code}: {text}")
        self.code = code


class ConfigT(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("hidden", "n_q_heads", "n_kv_heads", "head_dim", "n_layers", "ffn", "vocab")] + \
               [("rope_theta", C.c_float), ("rms_eps", C.c_float)] + \
               [(n, C.c_int32) for n in ("dtype", "dgf_proj", "first_layer_input_norm", "final_norm",
                                         "max_rows", "max_tree_slots", "max_branch", "fusion", "weight_quant")]


LAYER_KEYS = ("g_attn", "wq", "wk", "wv", "wo", "g_ffn", "wgate", "wup", "wdown")
LAYER_SCALE_KEYS = ("sq", "sk", "sv", "so", "sgate", "sup", "sdown")
TOP_SCALE_KEYS = ("dgf_s1", "dgf_s2", "dgf_sg", "lm_head_s")


class LayerWeightsT(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in LAYER_KEYS + LAYER_SCALE_KEYS]


class WeightsT(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("embed", "dgf_w1", "dgf_w2", "dgf_wg", "dgf_bg")] + \
               [("layers", C.POINTER(LayerWeightsT)), ("g_final", C.c_void_p), ("lm_head", C.c_void_p)] + \
               [(n, C.c_void_p) for n in TOP_SCALE_KEYS]


class KVCacheT(C.Structure):
    _fields_ = [("k", C.c_void_p), ("v", C.c_void_p), ("capacity", C.c_int32), ("committed_len", C.c_int32)]


class TreeSpecT(C.Structure):
    _fields_ = [("depth", C.c_int32), ("branch", C.c_int32 * MAX_DEPTH), ("beam", C.c_int32 * MAX_DEPTH),
                ("gamma", C.c_int32)]


class DraftOutT(C.Structure):
    _fields_ = [("token_ids", C.c_void_p), ("scores", C.c_void_p), ("parents", C.c_void_p),
                ("depths", C.c_void_p), ("n_out", C.c_void_p)]


class VerifyPlanT(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("mask", "position_ids", "paths", "n_paths")]


class VerifyInT(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("tgt_argmax", "p_cand", "uniforms", "p_full")]


class VerifyOutT(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("accepted_path", "n_acc", "bonus_token")]


HOOK_FIELDS = ("tap_logits", "tap_hhat", "tap_k", "tap_v", "tap_pool_token", "tap_pool_cum",
               "force_hhat", "force_k", "force_v", "force_pool_token", "force_pool_cum")


class HooksT(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in HOOK_FIELDS]


_lib = None


def load() -> C.CDLL:
    """Load the library; raises if it has not been built (python -m paper_2412_18934_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2412_18934_b200.build` "
                "(there is no fallback path)")
        lib = C.CDLL(LIB_PATH)
        lib.dovetail_draft_init.restype = C.c_int
        lib.dovetail_draft_init.argtypes = [C.POINTER(WeightsT), C.POINTER(ConfigT), C.POINTER(C.c_void_p)]
        lib.dovetail_draft_step.restype = C.c_int
        lib.dovetail_draft_step.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(KVCacheT),
                                            C.POINTER(TreeSpecT), C.POINTER(DraftOutT), C.c_void_p]
        lib.dovetail_draft_prefill.restype = C.c_int
        lib.dovetail_draft_prefill.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(KVCacheT), C.c_void_p]
        lib.dovetail_kv_commit.restype = C.c_int
        lib.dovetail_kv_commit.argtypes = [C.c_void_p, C.POINTER(KVCacheT), C.POINTER(C.c_int32), C.c_int32,
                                           C.c_int32, C.POINTER(C.c_int32), C.c_void_p]
        lib.dovetail_tree_replay.restype = C.c_int
        lib.dovetail_tree_replay.argtypes = [C.c_void_p, C.POINTER(TreeSpecT), C.c_void_p, C.c_void_p, C.c_int32,
                                             C.c_int32, C.POINTER(DraftOutT)] + [C.c_void_p] * 6
        lib.dovetail_tree_replay_static.restype = C.c_int
        lib.dovetail_tree_replay_static.argtypes = [C.POINTER(TreeSpecT), C.c_void_p, C.c_void_p, C.c_int32, C.c_int32,
                                                    C.POINTER(DraftOutT), C.c_void_p]
        lib.dovetail_verify_plan.restype = C.c_int
        lib.dovetail_verify_plan.argtypes = [C.c_void_p, C.POINTER(DraftOutT), C.c_int32, C.c_int32, C.c_int32,
                                             C.POINTER(VerifyPlanT), C.c_void_p]
        lib.dovetail_verify_accept.restype = C.c_int
        lib.dovetail_verify_accept.argtypes = [C.c_void_p, C.POINTER(DraftOutT), C.c_int32, C.c_int32, C.c_int32,
                                               C.POINTER(VerifyInT), C.POINTER(VerifyOutT), C.c_void_p]
        lib.dovetail_hooks_set.restype = C.c_int
        lib.dovetail_hooks_set.argtypes = [C.c_void_p, C.POINTER(HooksT)]
        lib.dovetail_draft_status.restype = C.c_int
        lib.dovetail_draft_status.argtypes = [C.c_void_p, C.c_void_p]
        lib.dovetail_trace_enable.restype = C.c_int
        lib.dovetail_trace_enable.argtypes = [C.c_void_p, C.c_int32]
        lib.dovetail_trace_read.restype = C.c_int
        lib.dovetail_trace_read.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int64),
                                            C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_int32)]
        lib.dovetail_hooks_tune.restype = C.c_int
        lib.dovetail_hooks_tune.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
        lib.dovetail_hooks_stat.restype = C.c_int
        lib.dovetail_hooks_stat.argtypes = [C.c_void_p, C.c_int32]
        lib.dovetail_probe_stream.restype = C.c_int
        lib.dovetail_probe_stream.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_int32, C.c_void_p]
        lib.dovetail_last_launch_count.restype = C.c_int
        lib.dovetail_last_launch_count.argtypes = [C.c_void_p]
        lib.dovetail_forward_bytes.restype = C.c_int64
        lib.dovetail_forward_bytes.argtypes = [C.c_void_p, C.c_int32]
        lib.dovetail_draft_destroy.restype = None
        lib.dovetail_draft_destroy.argtypes = [C.c_void_p]
        lib.dovetail_last_error.restype = C.c_char_p
        lib.dovetail_last_error.argtypes = [C.c_void_p]
        _lib = lib
    return _lib


def config_t(cfg: DraftConfig, max_rows: int = 64, max_tree_slots: int = 128, max_branch: int = 32) -> ConfigT:
    return ConfigT(cfg.hidden, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.n_layers, cfg.ffn, cfg.vocab,
                   float(cfg.rope_theta), float(cfg.rms_eps), cfg.dtype, cfg.dgf_proj,
                   cfg.first_layer_input_norm, cfg.final_norm, max_rows, max_tree_slots, max_branch, cfg.fusion, cfg.wquant)


def tree_spec_t(tree: TreeSpec) -> TreeSpecT:
    t = TreeSpecT()
    t.depth = tree.depth
    for i in range(min(tree.depth, MAX_DEPTH)):
        t.branch[i] = tree.branch[i]
        t.beam[i] = tree.beam[i]
    t.gamma = tree.gamma
    return t


def _dp(t) -> Optional[int]:
    """Device pointer of a torch CUDA tensor (None stays NULL)."""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device buffers must be contiguous CUDA tensors"
    return t.data_ptr()


def _stream(stream) -> Optional[int]:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream or None


class Draft:
    """A handle plus the tensors it borrows (kept alive here)."""

    def __init__(self, ptr: int, cfg: DraftConfig, keep):
        self.ptr, self.cfg, self._keep = ptr, cfg, keep
        self.hooks = None

    def close(self):
        if self.ptr:
            load().dovetail_draft_destroy(self.ptr)
            self.ptr = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class KVCache:
    """dovetail_kv_cache_t over two torch tensors [n_layers][n_kv_heads][capacity][head_dim]."""

    def __init__(self, k, v, committed_len: int):
        assert k.shape == v.shape and k.dim() == 4 and k.dtype == v.dtype
        self.k, self.v = k, v
        self.c = KVCacheT(_dp(k), _dp(v), k.shape[2], committed_len)

    @property
    def committed_len(self) -> int:
        return self.c.committed_len

    @committed_len.setter
    def committed_len(self, n: int):
        self.c.committed_len = n


def _check(rc: int, h: Optional[int]):
    if rc != OK:
        raise DovetailError(rc, load().dovetail_last_error(h).decode())


def dovetail_last_error(h: Optional[Draft]) -> str:
    return load().dovetail_last_error(h.ptr if h else None).decode()


def dovetail_draft_init(top: Dict, layers: List[Dict], cfg: DraftConfig, max_rows: int = 64,
                        max_tree_slots: int = 128, max_branch: int = 32) -> Draft:
    """top / layers: device tensors as produced by synth.make_weights(cfg, device='cuda')."""
    lib = load()
    import torch
    if cfg.wquant:  # the ABI takes raw pointers: check what it will reinterpret
        for d_, keys in [(top, ("dgf_wg", "lm_head"))] + [(l, ("wq", "wk", "wv", "wo", "wgate", "wup", "wdown")) for l in layers]:
            for k in keys:
                want = torch.int8 if cfg.wquant == 1 else torch.float8_e4m3fn
                if d_[k].dtype != want:
                    raise TypeError(f"weight_quant = {cfg.wquant}: {k} must be {want}, got {d_[k].dtype}")
    arr = (LayerWeightsT * len(layers))(*[LayerWeightsT(*[_dp(l.get(k)) for k in LAYER_KEYS + LAYER_SCALE_KEYS]) for l in layers])
    w = WeightsT(_dp(top["embed"]), _dp(top.get("dgf_w1")), _dp(top.get("dgf_w2")), _dp(top["dgf_wg"]),
                 _dp(top["dgf_bg"]), arr, _dp(top.get("g_final")), _dp(top["lm_head"]),
                 *[_dp(top.get(k)) for k in TOP_SCALE_KEYS])
    c = config_t(cfg, max_rows, max_tree_slots, max_branch)
    out = C.c_void_p()
    rc = lib.dovetail_draft_init(C.byref(w), C.byref(c), C.byref(out))
    _check(rc, None)
    return Draft(out.value, cfg, (top, layers))


def alloc_out(gamma: int, device="cuda"):
    """Output buffers of a step as views of ONE device allocation (out["_packed"], int32 words: ids | scores |
    parents | depths | n_out), so that a caller can bring the whole result to the host with a single copy."""
    import torch
    buf = torch.zeros(4 * gamma + 4, dtype=torch.int32, device=device)
    return dict(token_ids=buf[0:gamma], scores=buf[gamma:2 * gamma].view(torch.float32), parents=buf[2 * gamma:3 * gamma],
                depths=buf[3 * gamma:4 * gamma], n_out=buf[4 * gamma:4 * gamma + 1], _packed=buf)


def _out_t(out: Dict) -> DraftOutT:
    return DraftOutT(_dp(out["token_ids"]), _dp(out["scores"]), _dp(out["parents"]), _dp(out.get("depths")),
                     _dp(out["n_out"]))


def dovetail_draft_step(h: Draft, hidden_feats, tokens, kv: KVCache, tree: TreeSpec, out: Optional[Dict] = None,
                        stream=None) -> Dict:
    """Enqueues one draft step; returns the device output buffers (asynchronous)."""
    import torch
    # the ABI takes raw pointers: a wrong dtype or shape would be silently reinterpreted
    d, cdt = h.cfg.hidden, (torch.bfloat16 if h.cfg.dtype == BF16 else torch.float32)
    if hidden_feats.dtype != torch.float32 or hidden_feats.dim() != 2 or hidden_feats.shape[1] != d:
        raise TypeError(f"hidden_feats must be float32 [n_new, {d}], got {hidden_feats.dtype} {tuple(hidden_feats.shape)}")
    if tokens.dtype != torch.int32 or tokens.dim() != 1 or tokens.shape[0] != hidden_feats.shape[0]:
        raise TypeError(f"tokens must be int32 [n_new = {hidden_feats.shape[0]}], got {tokens.dtype} {tuple(tokens.shape)}")
    if kv.k.dtype != cdt or kv.k.shape[0] != h.cfg.n_layers or kv.k.shape[1] != h.cfg.n_kv_heads or kv.k.shape[3] != h.cfg.head_dim:
        raise TypeError(f"KV cache must be {cdt} [n_layers, n_kv_heads, capacity, head_dim], got {kv.k.dtype} {tuple(kv.k.shape)}")
    if out is None:
        out = alloc_out(tree.gamma, hidden_feats.device)
    for name, dt in (("token_ids", torch.int32), ("scores", torch.float32), ("parents", torch.int32), ("n_out", torch.int32)):
        if out[name].dtype != dt or out[name].numel() < (1 if name == "n_out" else tree.gamma):
            raise TypeError(f"out[{name!r}] must be {dt} with room for gamma = {tree.gamma} entries")
    t = tree_spec_t(tree)
    o = _out_t(out)
    rc = load().dovetail_draft_step(h.ptr, _dp(hidden_feats), _dp(tokens), int(tokens.shape[0]), C.byref(kv.c),
                                    C.byref(t), C.byref(o), _stream(stream))
    _check(rc, h.ptr)
    return out


def dovetail_draft_prefill(h: Draft, hidden_feats, tokens, kv: KVCache, stream=None) -> None:
    """Prompt / catch-up rows (include/dovetail.h): appends the K/V of every (feature, token) row and advances
    kv.committed_len; no LM head, no tree. Asynchronous."""
    import torch
    d, cdt = h.cfg.hidden, (torch.bfloat16 if h.cfg.dtype == BF16 else torch.float32)
    if hidden_feats.dtype != torch.float32 or hidden_feats.dim() != 2 or hidden_feats.shape[1] != d or not hidden_feats.is_contiguous():
        raise TypeError(f"hidden_feats must be contiguous float32 [n_rows, {d}], got {hidden_feats.dtype} {tuple(hidden_feats.shape)}")
    if tokens.dtype != torch.int32 or tokens.dim() != 1 or tokens.shape[0] != hidden_feats.shape[0]:
        raise TypeError(f"tokens must be int32 [n_rows = {hidden_feats.shape[0]}], got {tokens.dtype} {tuple(tokens.shape)}")
    if kv.k.dtype != cdt or kv.k.shape[0] != h.cfg.n_layers or kv.k.shape[1] != h.cfg.n_kv_heads or kv.k.shape[3] != h.cfg.head_dim:
        raise TypeError(f"KV cache must be {cdt} [n_layers, n_kv_heads, capacity, head_dim], got {kv.k.dtype} {tuple(kv.k.shape)}")
    rc = load().dovetail_draft_prefill(h.ptr, _dp(hidden_feats), _dp(tokens), int(tokens.shape[0]), C.byref(kv.c), _stream(stream))
    _check(rc, h.ptr)


def dovetail_kv_commit(h: Draft, kv: KVCache, accepted_path, mode: int = 0, stream=None) -> int:
    path = (C.c_int32 * max(1, len(accepted_path)))(*[int(i) for i in accepted_path])
    n = C.c_int32(0)
    rc = load().dovetail_kv_commit(h.ptr, C.byref(kv.c), path, len(accepted_path), mode, C.byref(n), _stream(stream))
    _check(rc, h.ptr)
    return n.value


def dovetail_verify_plan(h: Draft, out: Dict, root_position: int, max_depth: int, stream=None) -> Dict:
    """Verifier inputs from a step's output (include/dovetail.h): device tensors mask [(g+1), (g+1)] uint8,
    position_ids [g+1], paths [g, max_depth], n_paths [1]. Asynchronous."""
    import torch
    g = out["token_ids"].numel()
    dev = out["token_ids"].device
    plan = dict(mask=torch.zeros((g + 1, g + 1), dtype=torch.uint8, device=dev),
                position_ids=torch.zeros(g + 1, dtype=torch.int32, device=dev),
                paths=torch.zeros((g, max_depth), dtype=torch.int32, device=dev),
                n_paths=torch.zeros(1, dtype=torch.int32, device=dev))
    o = _out_t(out)
    t = VerifyPlanT(_dp(plan["mask"]), _dp(plan["position_ids"]), _dp(plan["paths"]), _dp(plan["n_paths"]))
    _check(load().dovetail_verify_plan(h.ptr, C.byref(o), g, root_position, max_depth, C.byref(t), _stream(stream)), h.ptr)
    return plan


def dovetail_verify_accept(h: Draft, out: Dict, mode: int, max_depth: int, tgt_argmax=None, p_cand=None, uniforms=None,
                           p_full=None, stream=None) -> Dict:
    """Acceptance rule (include/dovetail.h): mode 0 greedy, 1 speculative sampling. Device results, asynchronous."""
    import torch
    g = out["token_ids"].numel()
    dev = out["token_ids"].device
    for name, t, dt in (("tgt_argmax", tgt_argmax, torch.int32), ("p_cand", p_cand, torch.float32),
                        ("uniforms", uniforms, torch.float32), ("p_full", p_full, torch.float32)):
        if t is not None and t.dtype != dt:
            raise TypeError(f"{name} must be {dt}")
    res = dict(accepted_path=torch.full((max_depth,), -1, dtype=torch.int32, device=dev),
               n_acc=torch.zeros(1, dtype=torch.int32, device=dev), bonus_token=torch.zeros(1, dtype=torch.int32, device=dev))
    o = _out_t(out)
    i = VerifyInT(_dp(tgt_argmax), _dp(p_cand), _dp(uniforms), _dp(p_full))
    r = VerifyOutT(_dp(res["accepted_path"]), _dp(res["n_acc"]), _dp(res["bonus_token"]))
    _check(load().dovetail_verify_accept(h.ptr, C.byref(o), g, mode, max_depth, C.byref(i), C.byref(r), _stream(stream)), h.ptr)
    return res


def dovetail_tree_replay(h: Draft, tree: TreeSpec, cand_tokens, cand_logp, out: Optional[Dict] = None,
                         pool: Optional[Dict] = None, stream=None):
    """cand_tokens int32 / cand_logp fp32: device tensors [n_rows, max_b]."""
    if out is None:
        out = alloc_out(tree.gamma, cand_tokens.device)
    t = tree_spec_t(tree)
    o = _out_t(out)
    pool = pool or {}
    rc = load().dovetail_tree_replay(h.ptr, C.byref(t), _dp(cand_tokens), _dp(cand_logp), cand_tokens.shape[0],
                                     cand_tokens.shape[1], C.byref(o), _dp(pool.get("token")), _dp(pool.get("parent")),
                                     _dp(pool.get("depth")), _dp(pool.get("cum")), _dp(pool.get("size")),
                                     _stream(stream))
    _check(rc, h.ptr)
    return out


STATIC_MAX_POOL, STATIC_SCRATCH_BYTES = 2048, 65536  # include/dovetail.h


def dovetail_tree_replay_static(tree: TreeSpec, cand_tokens, cand_logp, out: Dict, stream=None) -> Dict:
    """The tree bookkeeping without a handle and without any allocation (include/dovetail.h): scratch in a
    file-scope device array of the library. `out` must be pre-allocated (alloc_out) -- this wrapper allocates
    nothing on the device either. Calls that overlap on the GPU race on the shared scratch."""
    t = tree_spec_t(tree)
    o = _out_t(out)
    rc = load().dovetail_tree_replay_static(C.byref(t), _dp(cand_tokens), _dp(cand_logp), cand_tokens.shape[0],
                                            cand_tokens.shape[1], C.byref(o), _stream(stream))
    _check(rc, None)
    return out


def dovetail_hooks_set(h: Draft, **hooks):
    """Test hooks (include/dovetail_hooks.h): keyword = field of dovetail_hooks_t, value = device tensor.
    No keywords removes every hook."""
    unknown = set(hooks) - set(HOOK_FIELDS)
    assert not unknown, f"unknown hook fields {unknown}"
    h.hooks = dict(hooks)  # keep the tensors alive
    if not hooks:
        _check(load().dovetail_hooks_set(h.ptr, None), h.ptr)
        return
    t = HooksT(*[_dp(hooks.get(n)) for n in HOOK_FIELDS])
    _check(load().dovetail_hooks_set(h.ptr, C.byref(t)), h.ptr)


def dovetail_draft_status(h: Draft, stream=None):
    """Synchronises the stream; raises DovetailError(EINVAL) if a step saw a token id outside [0, vocab)."""
    _check(load().dovetail_draft_status(h.ptr, _stream(stream)), h.ptr)


N_KINDS = 11
KIND_NAMES = ("step_begin", "dgf_proj", "dgf_gate", "qkv", "tree_attention", "o_proj", "gate_up", "down",
              "lm_head", "tree_level", "h_fill")


def dovetail_trace_enable(h: Draft, enable: bool):
    _check(load().dovetail_trace_enable(h.ptr, 1 if enable else 0), h.ptr)


def dovetail_trace_read(h: Draft, cap: int = 4096) -> Dict:
    """Device time of the last traced, synchronised step from the per-launch globaltimer stamps (the
    launches keep their PDL overlap). Returns step_us (first start to last end), per-kind and per-level
    busy_us (sum of end - start) and excl_us (each launch clipped to start no earlier than the end of the
    launches before it, so that kinds / levels add up to at most the step), launches and algorithmic bytes."""
    kind = (C.c_int32 * cap)()
    level = (C.c_int32 * cap)()
    nbytes = (C.c_int64 * cap)()
    t0 = (C.c_uint64 * cap)()
    t1 = (C.c_uint64 * cap)()
    n = C.c_int32(0)
    _check(load().dovetail_trace_read(h.ptr, cap, kind, level, nbytes, t0, t1, C.byref(n)), h.ptr)
    kinds = {name: dict(busy_us=0.0, excl_us=0.0, launches=0, bytes=0) for name in KIND_NAMES}
    levels: Dict[int, Dict] = {}
    first, last, prev_end = None, 0, 0
    for i in range(n.value):
        a, b = t0[i], t1[i]
        if a == 2 ** 64 - 1 or b == 0 or b < a:  # the launch did not stamp
            continue
        first = a if first is None else min(first, a)
        last = max(last, b)
        c0 = max(a, prev_end)
        prev_end = max(prev_end, b)
        for rec in (kinds[KIND_NAMES[kind[i]]], levels.setdefault(level[i], dict(busy_us=0.0, excl_us=0.0, launches=0, bytes=0))):
            rec["busy_us"] += (b - a) * 1e-3
            rec["excl_us"] += max(0, b - c0) * 1e-3
            rec["launches"] += 1
            rec["bytes"] += nbytes[i]
    return dict(step_us=(last - first) * 1e-3 if first is not None else 0.0, kinds=kinds, levels=levels)


TUNE_UMMA_MIN_M, TUNE_GRAPHS, TUNE_ATTN_WIDE_MIN, TUNE_ATTN_QT2, TUNE_UMMA_KSPLIT_MIN_M = 1, 2, 3, 4, 5
STAT_UMMA_LAUNCHES, STAT_GRAPH, STAT_KSPLIT_LAUNCHES = 1, 2, 3


def dovetail_hooks_umma_tables(rows, paired: int, pairperm: int, ctas: int) -> Dict:
    """Row tables of the tcgen05 GEMV for one dealing (include/dovetail_hooks.h); host logic, no GPU needed."""
    import numpy as np
    lib = load()
    n_mat = len(rows)
    r = (C.c_int32 * 3)(*(list(rows) + [0] * (3 - n_mat)))
    n_sb = np.zeros(ctas, np.int32)
    cnt = np.zeros(ctas, np.int32)
    n_grp = np.zeros((ctas, 8), np.int32)
    grp = np.zeros((ctas, 8, 16), np.int32)
    cap = ctas * (max(rows) * n_mat // ctas + 64)
    vpos = np.zeros(cap, np.uint16)
    ld = C.c_int32(0)
    P = lambda a: a.ctypes.data_as(C.c_void_p)
    f = lib.dovetail_hooks_umma_tables
    f.restype = C.c_int
    f.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32] + [C.c_void_p] * 4 + [C.c_int32, C.c_void_p, C.c_void_p]
    rc = f(r, n_mat, paired, pairperm, ctas, P(n_sb), P(n_grp), P(grp), P(vpos), cap, C.byref(ld), P(cnt))
    if rc != OK:
        raise DovetailError(rc, "dovetail_hooks_umma_tables")
    return dict(n_sb=n_sb, n_grp=n_grp, grp=grp, cnt=cnt, vpos=vpos[:ctas * ld.value].reshape(ctas, ld.value))


def dovetail_hooks_stat(h: Draft, key: int) -> int:
    """Counters of the last step (include/dovetail_hooks.h): key 1 = launches of the tcgen05 GEMV."""
    return load().dovetail_hooks_stat(h.ptr, key)


def dovetail_hooks_tune(h: Draft, key: int, value: int):
    """Design knobs for A/B measurements (include/dovetail_hooks.h): key 1 = rows from which a level runs on the
    tcgen05 GEMV (65: never)."""
    _check(load().dovetail_hooks_tune(h.ptr, key, value), h.ptr)


def dovetail_probe_stream(h: Draft, buf, mode: int, seg: int = 1024, stream=None):
    """Read-only streaming ceiling probe (include/dovetail_hooks.h) over a device tensor; asynchronous."""
    _check(load().dovetail_probe_stream(h.ptr, _dp(buf), buf.numel() * buf.element_size(), mode, seg, _stream(stream)), h.ptr)


def dovetail_last_launch_count(h: Draft) -> int:
    return load().dovetail_last_launch_count(h.ptr)


def dovetail_forward_bytes(h: Draft, prefix_len: int) -> int:
    return load().dovetail_forward_bytes(h.ptr, prefix_len)


def dovetail_draft_destroy(h: Draft):
    h.close()

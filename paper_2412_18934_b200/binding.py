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

EXPORTS = ("dovetail_draft_init", "dovetail_draft_step", "dovetail_kv_commit", "dovetail_tree_replay",
           "dovetail_draft_set_taps", "dovetail_draft_set_forcing", "dovetail_draft_set_profile", "dovetail_profile_read",
           "dovetail_last_launch_count", "dovetail_forward_bytes",
           "dovetail_draft_destroy", "dovetail_last_error")


class DovetailError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"dovetail error {code}: {text}")
        self.code = code


class ConfigT(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("hidden", "n_q_heads", "n_kv_heads", "head_dim", "n_layers", "ffn", "vocab")] + \
               [("rope_theta", C.c_float), ("rms_eps", C.c_float)] + \
               [(n, C.c_int32) for n in ("dtype", "dgf_proj", "first_layer_input_norm", "final_norm",
                                         "max_rows", "max_tree_slots", "max_branch")]


LAYER_KEYS = ("g_attn", "wq", "wk", "wv", "wo", "g_ffn", "wgate", "wup", "wdown")


class LayerWeightsT(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in LAYER_KEYS]


class WeightsT(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("embed", "dgf_w1", "dgf_w2", "dgf_wg", "dgf_bg")] + \
               [("layers", C.POINTER(LayerWeightsT)), ("g_final", C.c_void_p), ("lm_head", C.c_void_p)]


class KVCacheT(C.Structure):
    _fields_ = [("k", C.c_void_p), ("v", C.c_void_p), ("capacity", C.c_int32), ("committed_len", C.c_int32)]


class TreeSpecT(C.Structure):
    _fields_ = [("depth", C.c_int32), ("branch", C.c_int32 * MAX_DEPTH), ("beam", C.c_int32 * MAX_DEPTH),
                ("gamma", C.c_int32)]


class DraftOutT(C.Structure):
    _fields_ = [("token_ids", C.c_void_p), ("scores", C.c_void_p), ("parents", C.c_void_p),
                ("depths", C.c_void_p), ("n_out", C.c_void_p)]


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
        lib.dovetail_kv_commit.restype = C.c_int
        lib.dovetail_kv_commit.argtypes = [C.c_void_p, C.POINTER(KVCacheT), C.POINTER(C.c_int32), C.c_int32,
                                           C.c_int32, C.POINTER(C.c_int32), C.c_void_p]
        lib.dovetail_tree_replay.restype = C.c_int
        lib.dovetail_tree_replay.argtypes = [C.c_void_p, C.POINTER(TreeSpecT), C.c_void_p, C.c_void_p, C.c_int32,
                                             C.c_int32, C.POINTER(DraftOutT)] + [C.c_void_p] * 6
        lib.dovetail_draft_set_taps.restype = C.c_int
        lib.dovetail_draft_set_taps.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.dovetail_draft_set_forcing.restype = C.c_int
        lib.dovetail_draft_set_forcing.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        lib.dovetail_draft_set_profile.restype = C.c_int
        lib.dovetail_draft_set_profile.argtypes = [C.c_void_p, C.c_int32]
        lib.dovetail_profile_read.restype = C.c_int
        lib.dovetail_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_int64)]
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
                   cfg.first_layer_input_norm, cfg.final_norm, max_rows, max_tree_slots, max_branch)


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
        self.taps = None

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
        assert k.shape == v.shape and k.dim() == 4
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
    arr = (LayerWeightsT * len(layers))(*[LayerWeightsT(*[_dp(l[k]) for k in LAYER_KEYS]) for l in layers])
    w = WeightsT(_dp(top["embed"]), _dp(top.get("dgf_w1")), _dp(top.get("dgf_w2")), _dp(top["dgf_wg"]),
                 _dp(top["dgf_bg"]), arr, _dp(top.get("g_final")), _dp(top["lm_head"]))
    c = config_t(cfg, max_rows, max_tree_slots, max_branch)
    out = C.c_void_p()
    rc = lib.dovetail_draft_init(C.byref(w), C.byref(c), C.byref(out))
    _check(rc, None)
    return Draft(out.value, cfg, (top, layers))


def alloc_out(gamma: int, device="cuda"):
    import torch
    return dict(token_ids=torch.zeros(gamma, dtype=torch.int32, device=device),
                scores=torch.zeros(gamma, dtype=torch.float32, device=device),
                parents=torch.zeros(gamma, dtype=torch.int32, device=device),
                depths=torch.zeros(gamma, dtype=torch.int32, device=device),
                n_out=torch.zeros(1, dtype=torch.int32, device=device))


def _out_t(out: Dict) -> DraftOutT:
    return DraftOutT(_dp(out["token_ids"]), _dp(out["scores"]), _dp(out["parents"]), _dp(out.get("depths")),
                     _dp(out["n_out"]))


def dovetail_draft_step(h: Draft, hidden_feats, tokens, kv: KVCache, tree: TreeSpec, out: Optional[Dict] = None,
                        stream=None) -> Dict:
    """Enqueues one draft step; returns the device output buffers (asynchronous)."""
    if out is None:
        out = alloc_out(tree.gamma, hidden_feats.device)
    t = tree_spec_t(tree)
    o = _out_t(out)
    rc = load().dovetail_draft_step(h.ptr, _dp(hidden_feats), _dp(tokens), int(tokens.shape[0]), C.byref(kv.c),
                                    C.byref(t), C.byref(o), _stream(stream))
    _check(rc, h.ptr)
    return out


def dovetail_kv_commit(h: Draft, kv: KVCache, accepted_path, mode: int = 0, stream=None) -> int:
    path = (C.c_int32 * max(1, len(accepted_path)))(*[int(i) for i in accepted_path])
    n = C.c_int32(0)
    rc = load().dovetail_kv_commit(h.ptr, C.byref(kv.c), path, len(accepted_path), mode, C.byref(n), _stream(stream))
    _check(rc, h.ptr)
    return n.value


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


def dovetail_draft_set_taps(h: Draft, logits=None, hhat=None):
    h.taps = (logits, hhat)
    _check(load().dovetail_draft_set_taps(h.ptr, _dp(logits), _dp(hhat)), h.ptr)


def dovetail_draft_set_forcing(h: Draft, force_hhat=None, force_k=None, force_v=None, tap_k=None, tap_v=None):
    """Teacher forcing for parity tests (include/dovetail.h); all None disables it."""
    h.forcing = (force_hhat, force_k, force_v, tap_k, tap_v)  # keep the tensors alive
    _check(load().dovetail_draft_set_forcing(h.ptr, _dp(force_hhat), _dp(force_k), _dp(force_v), _dp(tap_k), _dp(tap_v)),
           h.ptr)


N_KINDS = 11
KIND_NAMES = ("step_begin", "dgf_proj", "dgf_gate", "qkv", "tree_attention", "o_proj", "gate_up", "down",
              "lm_head", "tree_level", "h_fill")


def dovetail_draft_set_profile(h: Draft, enable: bool):
    _check(load().dovetail_draft_set_profile(h.ptr, 1 if enable else 0), h.ptr)


def dovetail_profile_read(h: Draft) -> Dict[str, Dict]:
    """Per-kind totals of the last (profiled, synchronised) step: ms, launches, algorithmic bytes."""
    ms = (C.c_float * N_KINDS)()
    n = (C.c_int32 * N_KINDS)()
    b = (C.c_int64 * N_KINDS)()
    _check(load().dovetail_profile_read(h.ptr, ms, n, b), h.ptr)
    return {KIND_NAMES[k]: dict(ms=ms[k], launches=n[k], bytes=b[k]) for k in range(N_KINDS)}


def dovetail_last_launch_count(h: Draft) -> int:
    return load().dovetail_last_launch_count(h.ptr)


def dovetail_forward_bytes(h: Draft, prefix_len: int) -> int:
    return load().dovetail_forward_bytes(h.ptr, prefix_len)


def dovetail_draft_destroy(h: Draft):
    h.close()

"""TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes wrapper around oracle/dovetail_oracle.c (plain C, fp64). The C file is
the oracle; this module only marshals numpy arrays into it. bf16 buffers are
numpy uint16 arrays holding the bf16 bit patterns (torch bf16 tensors are
accepted and viewed without copy).
"""
import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import Dict, List, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dovetail_oracle.c")
_SO = os.path.join(_HERE, "libdovetail_oracle.so")
_lib = None

F32, BF16 = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP over output rows only)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-ffp-contract=off",
               "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


class _Cfg(C.Structure):
    _fields_ = [(n, C.c_int32) for n in
                ("hidden", "n_q_heads", "n_kv_heads", "head_dim", "n_layers", "ffn", "vocab")] + \
               [("rope_theta", C.c_double), ("rms_eps", C.c_double)] + \
               [(n, C.c_int32) for n in ("dtype", "dgf_proj", "first_layer_input_norm", "final_norm", "fusion", "wquant")]


SCALE_KEYS = ("sq", "sk", "sv", "so", "sgate", "sup", "sdown")
TOP_SCALE_KEYS = ("dgf_s1", "dgf_s2", "dgf_sg", "lm_head_s")


class _Layer(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in
                ("g_attn", "wq", "wk", "wv", "wo", "g_ffn", "wgate", "wup", "wdown") + SCALE_KEYS]


class _Weights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("embed", "dgf_w1", "dgf_w2", "dgf_wg", "dgf_bg")] + \
               [("layers", C.POINTER(_Layer)), ("g_final", C.c_void_p), ("lm_head", C.c_void_p)] + \
               [(n, C.c_void_p) for n in TOP_SCALE_KEYS]


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.dovetail_oracle_step.restype = C.c_int
        _lib.dovetail_oracle_tree_replay.restype = C.c_int
        _lib.dovetail_oracle_kv_commit.restype = C.c_int
        _lib.dovetail_oracle_verify_plan.restype = C.c_int
        _lib.dovetail_oracle_verify_accept.restype = C.c_int
    return _lib


@dataclass
class OracleConfig:
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    n_layers: int
    ffn: int
    vocab: int
    rope_theta: float = 1e4
    rms_eps: float = 1e-5
    dtype: int = BF16
    dgf_proj: int = 1
    first_layer_input_norm: int = 1
    final_norm: int = 0
    fusion: int = 0  # 0 DGF; 1 concat + Linear, the EAGLE-2 baseline
    wquant: int = 0  # 1: matrices are int8, 2: fp8 e4m3 bytes, with one fp32 scale per output row

    def c(self) -> _Cfg:
        return _Cfg(self.hidden, self.n_q_heads, self.n_kv_heads, self.head_dim, self.n_layers,
                    self.ffn, self.vocab, float(self.rope_theta), float(self.rms_eps), self.dtype,
                    self.dgf_proj, self.first_layer_input_norm, self.final_norm, self.fusion, self.wquant)


def _np(a):
    """numpy view of a numpy array or a CPU torch tensor (bf16 -> uint16 bits)."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return np.ascontiguousarray(a)
    import torch  # only when a tensor is passed
    t = a.detach().contiguous()
    assert t.device.type == "cpu", "oracle inputs live in host memory"
    if t.dtype == torch.bfloat16:
        return t.view(torch.int16).numpy().view(np.uint16)
    if t.dtype == getattr(torch, "float8_e4m3fn", None):  # fp8 weights travel as their bytes
        return t.view(torch.uint8).numpy()
    return t.numpy()


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


LAYER_KEYS = ("g_attn", "wq", "wk", "wv", "wo", "g_ffn", "wgate", "wup", "wdown")
TOP_KEYS = ("embed", "dgf_w1", "dgf_w2", "dgf_wg", "dgf_bg", "g_final", "lm_head")


@dataclass
class OracleWeights:
    """Holds numpy views of the weights and the C struct pointing at them.

    top: dict with keys TOP_KEYS (dgf_w1/dgf_w2/g_final may be None);
    layers: list of dicts with keys LAYER_KEYS.
    """
    top: Dict[str, Optional[np.ndarray]]
    layers: List[Dict[str, np.ndarray]]
    _keep: list = field(default_factory=list)

    def c(self) -> _Weights:
        top = {k: _np(self.top.get(k)) for k in TOP_KEYS + TOP_SCALE_KEYS}
        lay = [{k: _np(l.get(k)) for k in LAYER_KEYS + SCALE_KEYS} for l in self.layers]
        arr = (_Layer * len(lay))(*[_Layer(*[_ptr(l[k]) for k in LAYER_KEYS + SCALE_KEYS]) for l in lay])
        w = _Weights(_ptr(top["embed"]), _ptr(top["dgf_w1"]), _ptr(top["dgf_w2"]),
                     _ptr(top["dgf_wg"]), _ptr(top["dgf_bg"]), arr, _ptr(top["g_final"]),
                     _ptr(top["lm_head"]), *[_ptr(top[k]) for k in TOP_SCALE_KEYS])
        self._keep = [top, lay, arr]
        return w


def _check_dtype(a: np.ndarray, dtype: int):
    want = np.float32 if dtype == F32 else np.uint16
    assert a.dtype == want, f"buffer dtype {a.dtype} does not match config dtype {dtype}"


# ---- primitive steps -------------------------------------------------------

def matvec(W, dtype: int, x: np.ndarray) -> np.ndarray:
    W = _np(W)
    _check_dtype(W, dtype)
    N, K = W.shape
    x = np.ascontiguousarray(x, dtype=np.float64)
    assert x.shape == (K,)
    y = np.empty(N, dtype=np.float64)
    _load().orc_matvec(_ptr(W), C.c_int(dtype), C.c_int(N), C.c_int(K), _ptr(x), _ptr(y))
    return y


def matvec_q8(Q, scale, x: np.ndarray) -> np.ndarray:
    """int8 matrix with one fp32 scale per output row: y = (scale[:, None] * Q) @ x in fp64."""
    Q = np.ascontiguousarray(_np(Q), dtype=np.int8)
    scale = np.ascontiguousarray(_np(scale), dtype=np.float32)
    N, K = Q.shape
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty(N, dtype=np.float64)
    _load().orc_matvec_q8(_ptr(Q), _ptr(scale), C.c_int(N), C.c_int(K), _ptr(x), _ptr(y))
    return y


def e4m3_to_double(b) -> np.ndarray:
    """Value of every fp8 e4m3 byte of an array (reading A17b)."""
    b = np.ascontiguousarray(b, dtype=np.uint8)
    f = _load().orc_e4m3_to_double
    f.restype, f.argtypes = C.c_double, [C.c_uint8]
    return np.array([f(int(v)) for v in b.reshape(-1)], dtype=np.float64).reshape(b.shape)


def matvec_f8(Q, scale, x: np.ndarray) -> np.ndarray:
    """fp8 e4m3 matrix (bytes) with one fp32 scale per output row: y = (scale[:, None] * e4m3(Q)) @ x in fp64."""
    Q = np.ascontiguousarray(_np(Q), dtype=np.uint8)
    scale = np.ascontiguousarray(_np(scale), dtype=np.float32)
    N, K = Q.shape
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty(N, dtype=np.float64)
    _load().orc_matvec_f8(_ptr(Q), _ptr(scale), C.c_int(N), C.c_int(K), _ptr(x), _ptr(y))
    return y


def rmsnorm(x: np.ndarray, g, dtype: int, eps: float) -> np.ndarray:
    g = _np(g)
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty_like(x)
    _load().orc_rmsnorm(_ptr(x), _ptr(g), C.c_int(dtype), C.c_int(x.shape[0]), C.c_double(eps), _ptr(y))
    return y


def rope(v: np.ndarray, pos: int, theta: float) -> np.ndarray:
    v = np.array(v, dtype=np.float64, order="C")
    _load().orc_rope(_ptr(v), C.c_int(v.shape[0]), C.c_int(pos), C.c_double(theta))
    return v


def dgf(cfg: OracleConfig, w: OracleWeights, f: np.ndarray, token: int) -> np.ndarray:
    f = np.ascontiguousarray(f, dtype=np.float64)
    x = np.empty(cfg.hidden, dtype=np.float64)
    cc, cw = cfg.c(), w.c()
    _load().orc_dgf(C.byref(cc), C.byref(cw), _ptr(f), C.c_int(int(token)), _ptr(x))
    return x


def fusion_linear(cfg: OracleConfig, w: OracleWeights, f: np.ndarray, token: int) -> np.ndarray:
    f = np.ascontiguousarray(f, dtype=np.float64)
    x = np.empty(cfg.hidden, dtype=np.float64)
    cc, cw = cfg.c(), w.c()
    _load().orc_fusion_linear(C.byref(cc), C.byref(cw), _ptr(f), C.c_int(int(token)), _ptr(x))
    return x


def lm_head(cfg: OracleConfig, w: OracleWeights, hhat: np.ndarray) -> np.ndarray:
    hhat = np.ascontiguousarray(hhat, dtype=np.float64)
    out = np.empty(cfg.vocab, dtype=np.float64)
    cc, cw = cfg.c(), w.c()
    _load().orc_lm_head(C.byref(cc), C.byref(cw), _ptr(hhat), _ptr(out))
    return out


def log_softmax(logits: np.ndarray) -> np.ndarray:
    logits = np.ascontiguousarray(logits, dtype=np.float64)
    out = np.empty_like(logits)
    _load().orc_log_softmax(_ptr(logits), C.c_int(logits.shape[0]), _ptr(out))
    return out


def topk(v: np.ndarray, b: int) -> np.ndarray:
    v = np.ascontiguousarray(v, dtype=np.float64)
    idx = np.empty(b, dtype=np.int32)
    _load().orc_topk(_ptr(v), C.c_int(v.shape[0]), C.c_int(b), _ptr(idx))
    return idx


def forward(cfg: OracleConfig, w: OracleWeights, kc: np.ndarray, vc: np.ndarray, capacity: int,
            slots, pos, allowed: List[List[int]], feats: np.ndarray, tokens) -> np.ndarray:
    """One forward of R rows with explicit attention sets; mutates kc, vc."""
    R = len(slots)
    slots = np.asarray(slots, dtype=np.int32)
    pos = np.asarray(pos, dtype=np.int32)
    n_allowed = np.asarray([len(a) for a in allowed], dtype=np.int32)
    flat = np.asarray([j for a in allowed for j in a], dtype=np.int32)
    feats = np.ascontiguousarray(feats, dtype=np.float64)
    tokens = np.asarray(tokens, dtype=np.int32)
    _check_dtype(kc, cfg.dtype)
    hhat = np.empty((R, cfg.hidden), dtype=np.float64)
    cc, cw = cfg.c(), w.c()
    _load().orc_forward(C.byref(cc), C.byref(cw), _ptr(kc), _ptr(vc), C.c_int(capacity), C.c_int(R),
                        _ptr(slots), _ptr(pos), _ptr(n_allowed), _ptr(flat), _ptr(feats),
                        _ptr(tokens), _ptr(hhat))
    return hhat


def _tree_shape(depth, branch, beam, n_new):
    m, tree_rows, cap = 1, 0, 0
    for l in range(depth):
        if l >= 1:
            n = m * branch[l - 1]
            m = beam[l] if 0 < beam[l] < n else n
            tree_rows += m
        cap += m * branch[l]
    return n_new + tree_rows, cap


def step(cfg: OracleConfig, w: OracleWeights, kc: np.ndarray, vc: np.ndarray, capacity: int,
         committed_len: int, feats: np.ndarray, tokens, depth: int, branch, beam, gamma: int,
         dump: bool = True) -> dict:
    """The whole draft step (O1-O8). Mutates kc, vc (appends K/V rows)."""
    feats = np.ascontiguousarray(_np(feats), dtype=np.float32)
    tokens = np.asarray(_np(tokens), dtype=np.int32)
    n_new = int(tokens.shape[0])
    branch = np.asarray(list(branch) + [0] * (16 - len(branch)), dtype=np.int32)
    beam = np.asarray(list(beam) + [0] * (16 - len(beam)), dtype=np.int32)
    rows, cap = _tree_shape(depth, branch, beam, n_new)
    _check_dtype(kc, cfg.dtype)
    _check_dtype(vc, cfg.dtype)
    g = max(gamma, 1)
    out_ids = np.zeros(g, np.int32)
    out_scores = np.zeros(g, np.float64)
    out_par = np.zeros(g, np.int32)
    out_dep = np.zeros(g, np.int32)
    n_out = np.zeros(1, np.int32)
    p_tok = np.zeros(cap, np.int32)
    p_par = np.zeros(cap, np.int32)
    p_dep = np.zeros(cap, np.int32)
    p_cum = np.zeros(cap, np.float64)
    p_row = np.zeros(cap, np.int32)
    p_n = np.zeros(1, np.int32)
    r_logits = np.zeros((rows, cfg.vocab), np.float64) if dump else None
    r_hhat = np.zeros((rows, cfg.hidden), np.float64) if dump else None
    r_slot = np.zeros(rows, np.int32)
    r_pos = np.zeros(rows, np.int32)
    n_rows = np.zeros(1, np.int32)
    cc, cw = cfg.c(), w.c()
    rc = _load().dovetail_oracle_step(
        C.byref(cc), C.byref(cw), _ptr(kc), _ptr(vc), C.c_int32(capacity), C.c_int32(committed_len),
        _ptr(feats), _ptr(tokens), C.c_int32(n_new), C.c_int32(depth), _ptr(branch), _ptr(beam),
        C.c_int32(gamma), _ptr(out_ids), _ptr(out_scores), _ptr(out_par), _ptr(out_dep), _ptr(n_out),
        _ptr(p_tok), _ptr(p_par), _ptr(p_dep), _ptr(p_cum), _ptr(p_row), _ptr(p_n),
        _ptr(r_logits), _ptr(r_hhat), _ptr(r_slot), _ptr(r_pos), _ptr(n_rows))
    if rc != 0:
        raise ValueError("dovetail_oracle_step: bad argument")
    n = int(n_out[0])
    P = int(p_n[0])
    return dict(token_ids=out_ids[:n], scores=out_scores[:n], parents=out_par[:n], depths=out_dep[:n],
                n_out=n, pool_token=p_tok[:P], pool_parent=p_par[:P], pool_depth=p_dep[:P],
                pool_cum=p_cum[:P], pool_row=p_row[:P], row_logits=r_logits, row_hhat=r_hhat,
                row_slot=r_slot, row_pos=r_pos, total_rows=int(n_rows[0]),
                committed_len=committed_len + n_new)


def tree_replay(depth: int, branch, beam, gamma: int, cand_tokens: np.ndarray,
                cand_logp: np.ndarray) -> dict:
    """Bookkeeping alone (O6-O8) from per-row top-b lists [n_rows, max_b]."""
    cand_tokens = np.ascontiguousarray(cand_tokens, dtype=np.int32)
    cand_logp = np.ascontiguousarray(cand_logp, dtype=np.float64)
    n_rows, max_b = cand_tokens.shape
    branch = np.asarray(list(branch) + [0] * (16 - len(branch)), dtype=np.int32)
    beam = np.asarray(list(beam) + [0] * (16 - len(beam)), dtype=np.int32)
    _, cap = _tree_shape(depth, branch, beam, 1)
    g = max(gamma, 1)
    out_ids = np.zeros(g, np.int32)
    out_scores = np.zeros(g, np.float64)
    out_par = np.zeros(g, np.int32)
    out_dep = np.zeros(g, np.int32)
    n_out = np.zeros(1, np.int32)
    p_tok = np.zeros(cap, np.int32)
    p_par = np.zeros(cap, np.int32)
    p_dep = np.zeros(cap, np.int32)
    p_cum = np.zeros(cap, np.float64)
    p_n = np.zeros(1, np.int32)
    rc = _load().dovetail_oracle_tree_replay(
        C.c_int(depth), _ptr(branch), _ptr(beam), C.c_int(gamma), _ptr(cand_tokens), _ptr(cand_logp),
        C.c_int(n_rows), C.c_int(max_b), _ptr(out_ids), _ptr(out_scores), _ptr(out_par), _ptr(out_dep),
        _ptr(n_out), _ptr(p_tok), _ptr(p_par), _ptr(p_dep), _ptr(p_cum), _ptr(p_n))
    if rc != 0:
        raise ValueError("dovetail_oracle_tree_replay: not enough rows")
    n, P = int(n_out[0]), int(p_n[0])
    return dict(token_ids=out_ids[:n], scores=out_scores[:n], parents=out_par[:n], depths=out_dep[:n],
                n_out=n, pool_token=p_tok[:P], pool_parent=p_par[:P], pool_depth=p_dep[:P],
                pool_cum=p_cum[:P])


def kv_commit(cfg: OracleConfig, kc: np.ndarray, vc: np.ndarray, capacity: int, Lp: int,
              path_tree_rows, mode: int) -> int:
    """O9. path_tree_rows[i] = tree-row index of accepted node i or -1. Returns rows moved."""
    p = np.asarray(path_tree_rows, dtype=np.int32)
    cc = cfg.c()
    return int(_load().dovetail_oracle_kv_commit(C.byref(cc), _ptr(kc), _ptr(vc), C.c_int32(capacity),
                                                 C.c_int32(Lp), _ptr(p), C.c_int32(len(p)),
                                                 C.c_int32(mode)))


def verify_plan(parents, depths, root_position: int, max_depth: int) -> dict:
    """O10: verifier inputs (ancestor mask, position ids, root-to-leaf paths) from a step's output."""
    parents = np.ascontiguousarray(parents, dtype=np.int32)
    depths = np.ascontiguousarray(depths, dtype=np.int32)
    n = len(parents)
    mask = np.zeros((n + 1, n + 1), np.uint8)
    pos = np.zeros(n + 1, np.int32)
    paths = np.full((max(n, 1), max_depth), -1, np.int32)
    k = _load().dovetail_oracle_verify_plan(_ptr(parents), _ptr(depths), C.c_int32(n), C.c_int32(root_position),
                                             C.c_int32(max_depth), _ptr(mask), _ptr(pos), _ptr(paths))
    return dict(mask=mask, position_ids=pos, paths=paths[:k], n_paths=int(k))


def verify_accept(token_ids, parents, mode: int, tgt_argmax=None, p_cand=None, uniforms=None, p_full=None) -> dict:
    """O11: greedy (mode 0) or speculative-sampling (mode 1) acceptance + bonus token."""
    token_ids = np.ascontiguousarray(token_ids, dtype=np.int32)
    parents = np.ascontiguousarray(parents, dtype=np.int32)
    n = len(parents)
    f32 = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float32)
    tgt_argmax = None if tgt_argmax is None else np.ascontiguousarray(tgt_argmax, dtype=np.int32)
    p_cand, uniforms, p_full = f32(p_cand), f32(uniforms), f32(p_full)
    vocab = 0 if p_full is None else p_full.shape[1]
    path = np.full(max(n, 1), -1, np.int32)
    n_acc = np.zeros(1, np.int32)
    bonus = np.zeros(1, np.int32)
    _load().dovetail_oracle_verify_accept(_ptr(token_ids), _ptr(parents), C.c_int32(n), C.c_int32(mode), _ptr(tgt_argmax),
                                           _ptr(p_cand), _ptr(uniforms), _ptr(p_full), C.c_int32(vocab), _ptr(path),
                                           _ptr(n_acc), _ptr(bonus))
    return dict(accepted_path=path[:int(n_acc[0])].copy(), n_acc=int(n_acc[0]), bonus_token=int(bonus[0]))

"""Seeded synthetic inputs shaped like the paper's workloads (DESIGN.md "Input
recipe"). Serves both the CUDA path and the tests' oracle calls; holds none of
the method's arithmetic -- only random draws, scaling and dtype casts.

Stand-in for the paper's trained LLaMA2-Chat-7B/13B / Vicuna-13B drafts run on
MT-bench / HumanEval / GSM8K / Alpaca prompts: those
weights and datasets are not available; only their shapes are used.
"""
from typing import Dict, List, Tuple

import torch

from .configs import BF16, DraftConfig

LAYER_SHAPES = ("g_attn", "wq", "wk", "wv", "wo", "g_ffn", "wgate", "wup", "wdown")


def _tdtype(cfg: DraftConfig) -> torch.dtype:
    return torch.bfloat16 if cfg.dtype == BF16 else torch.float32


def _randn(shape, std, gen, device, dtype):
    # drawn in fp32, then rounded to the storage dtype
    t = torch.randn(shape, generator=gen, device=device, dtype=torch.float32)
    return (t * std).to(dtype).contiguous()


def make_weights(cfg: DraftConfig, device="cpu", seed=None) -> Tuple[Dict[str, torch.Tensor], List[Dict[str, torch.Tensor]]]:
    """Weights ~ N(0, 0.02) rounded to the storage dtype; norm gains 1; DGF bias N(0, 0.02)."""
    gen = torch.Generator(device=device)
    gen.manual_seed(cfg.seed if seed is None else seed)
    dt = _tdtype(cfg)
    d, F, V = cfg.hidden, cfg.ffn, cfg.vocab
    dq, dkv = cfg.n_q_heads * cfg.head_dim, cfg.n_kv_heads * cfg.head_dim
    r = lambda *s: _randn(s, 0.02, gen, device, dt)
    top = dict(
        embed=r(V, d),
        dgf_w1=r(d, d) if (cfg.dgf_proj and cfg.fusion == 0) else None,
        dgf_w2=r(d, d) if (cfg.dgf_proj and cfg.fusion == 0) else None,
        dgf_wg=r(d, 2 * d),
        dgf_bg=r(d),
        g_final=torch.ones(d, device=device, dtype=dt) if cfg.final_norm else None,
        lm_head=r(V, d),
    )
    layers = []
    for _ in range(cfg.n_layers):
        layers.append(dict(
            g_attn=torch.ones(d, device=device, dtype=dt),
            wq=r(dq, d), wk=r(dkv, d), wv=r(dkv, d), wo=r(d, dq),
            g_ffn=torch.ones(d, device=device, dtype=dt),
            wgate=r(F, d), wup=r(F, d), wdown=r(d, F),
        ))
    if cfg.wquant:
        top, layers = quantize_weights(top, layers, fp8=cfg.wquant == 2)
    return top, layers


MATRIX_SCALES = {"wq": "sq", "wk": "sk", "wv": "sv", "wo": "so", "wgate": "sgate", "wup": "sup", "wdown": "sdown"}
TOP_MATRIX_SCALES = {"dgf_w1": "dgf_s1", "dgf_w2": "dgf_s2", "dgf_wg": "dgf_sg", "lm_head": "lm_head_s"}


def quantize_rows(w: torch.Tensor):
    """Symmetric int8 with one scale per output row: scale = max|row| / 127 (rounded to a bf16-representable fp32 so
    that scale * q is exact in fp32 too), q = round-to-nearest-even(w / scale) clipped to [-127, 127]. Input
    preparation for the weight-quantised workload; not part of the method's arithmetic."""
    wf = w.float()
    scale = (wf.abs().amax(dim=1).clamp_min(1e-12) / 127.0).to(torch.bfloat16).float()
    q = torch.clamp(torch.round(wf / scale[:, None]), -127, 127).to(torch.int8).contiguous()
    return q, scale.contiguous()


def quantize_rows_f8(w: torch.Tensor):
    """fp8 e4m3 with one scale per output row: scale = max|row| / 448 (bf16-representable), q = e4m3(w / scale),
    round to nearest even, clamped to +-448 (the format has no infinity). Input preparation, as quantize_rows."""
    wf = w.float()
    scale = (wf.abs().amax(dim=1).clamp_min(1e-12) / 448.0).to(torch.bfloat16).float()
    q = torch.clamp(wf / scale[:, None], -448.0, 448.0).to(torch.float8_e4m3fn).contiguous()
    return q, scale.contiguous()


def quantize_weights(top: Dict, layers: List[Dict], fp8: bool = False):
    """8-bit version of a weight set: matrices -> (int8 or fp8 e4m3, scale); embedding, gains, bias untouched."""
    qr = quantize_rows_f8 if fp8 else quantize_rows
    top = dict(top)
    for k, sk in TOP_MATRIX_SCALES.items():
        if top.get(k) is not None:
            top[k], top[sk] = qr(top[k])
    out = []
    for l in layers:
        l = dict(l)
        for k, sk in MATRIX_SCALES.items():
            l[k], l[sk] = qr(l[k])
        out.append(l)
    return top, out


def make_kv(cfg: DraftConfig, capacity: int, prefix: int, device="cpu", seed=None):
    """KV cache [n_layers][Hkv][capacity][dh]; rows [0, prefix) ~ N(0,1), the rest zero."""
    gen = torch.Generator(device=device)
    gen.manual_seed((cfg.seed if seed is None else seed) + 7919)
    dt = _tdtype(cfg)
    shape = (cfg.n_layers, cfg.n_kv_heads, capacity, cfg.head_dim)
    k = torch.zeros(shape, device=device, dtype=dt)
    v = torch.zeros(shape, device=device, dtype=dt)
    if prefix > 0:
        ps = (cfg.n_layers, cfg.n_kv_heads, prefix, cfg.head_dim)
        k[:, :, :prefix] = _randn(ps, 1.0, gen, device, dt)
        v[:, :, :prefix] = _randn(ps, 1.0, gen, device, dt)
    return k, v


def make_inputs(cfg: DraftConfig, n_new: int, device="cpu", seed=None):
    """Target hidden features fp32 [n_new, d] (bf16-representable values, N(0,1)*feat_scale)
    and uniform token ids int32 [n_new]."""
    gen = torch.Generator(device=device)
    gen.manual_seed((cfg.seed if seed is None else seed) + 104729)
    f = torch.randn((n_new, cfg.hidden), generator=gen, device=device, dtype=torch.float32) * cfg.feat_scale
    f = f.to(torch.bfloat16).to(torch.float32).contiguous()
    t = torch.randint(0, cfg.vocab, (n_new,), generator=gen, device=device, dtype=torch.int32)
    return f, t


def to_host(top, layers):
    """CPU copies of a weight set (for the oracle side of a test)."""
    h = lambda t: None if t is None else t.detach().cpu()
    return {k: h(v) for k, v in top.items()}, [{k: h(v) for k, v in l.items()} for l in layers]

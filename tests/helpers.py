"""Shared test helpers: tiny configs, oracle marshalling, and an INDEPENDENT
fp64 reference of the draft network built from library routines (Hugging Face
LlamaDecoderLayer + torch SDPA) that the oracle is pinned against. Nothing here
is imported by the product."""
from dataclasses import replace

import numpy as np
import torch

import oracle
from paper_2412_18934_b200 import synth
from paper_2412_18934_b200.configs import BF16, F32, DraftConfig, TreeSpec


def tiny_cfg(**kw) -> DraftConfig:
    base = dict(name="tiny", hidden=32, n_q_heads=4, n_kv_heads=2, head_dim=8, n_layers=2, ffn=48,
                vocab=12, dtype=F32, prefix=0, feat_scale=1.0, rope_theta=1e4,
                tree=TreeSpec(2, (2, 2), (0, 0), 4), seed=7)
    base.update(kw)
    return DraftConfig(**base)


def ocfg(cfg: DraftConfig) -> oracle.OracleConfig:
    return oracle.OracleConfig(cfg.hidden, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.n_layers,
                               cfg.ffn, cfg.vocab, cfg.rope_theta, cfg.rms_eps, cfg.dtype, cfg.dgf_proj,
                               cfg.first_layer_input_norm, cfg.final_norm, cfg.fusion, cfg.wquant)


def oweights(top, layers) -> oracle.OracleWeights:
    top, layers = synth.to_host(top, layers)
    return oracle.OracleWeights(top, layers)


def kv_np(t: torch.Tensor) -> np.ndarray:
    """numpy view (copy on host) of a KV tensor in the oracle's storage dtype."""
    t = t.detach().cpu().contiguous()
    if t.dtype == torch.bfloat16:
        return t.view(torch.int16).numpy().view(np.uint16).copy()
    return t.numpy().copy()


def np_to_f64(a: np.ndarray) -> np.ndarray:
    """Widen a storage array (uint16 bf16 bits or float32) to float64."""
    if a.dtype == np.uint16:
        return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return a.astype(np.float64)


def oracle_step(cfg: DraftConfig, top, layers, k, v, capacity, L, feats, tokens, tree: TreeSpec = None,
                dump=True):
    tree = tree or cfg.tree
    kc, vc = kv_np(k), kv_np(v)
    res = oracle.step(ocfg(cfg), oweights(top, layers), kc, vc, capacity, L,
                      feats.detach().cpu().numpy(), tokens.detach().cpu().numpy(), tree.depth,
                      tree.branch, tree.beam, tree.gamma, dump=dump)
    res["k"], res["v"] = kc, vc
    return res


# --------------------------------------------------------------------------
# Independent fp64 reference from library routines
# --------------------------------------------------------------------------

class RefDraft:
    """DGF + HF LlamaDecoderLayer stack + LM head in fp64 with a DynamicCache.

    The decoder block (RMSNorm, rotate-half RoPE, GQA attention via SDPA, SiLU
    gated MLP, residuals) is Hugging Face's implementation, not ours; cos/sin
    are supplied in fp64 so only the pairing convention is HF's."""

    def __init__(self, cfg: DraftConfig, top, layers):
        from transformers import LlamaConfig
        from transformers.cache_utils import DynamicCache
        from transformers.models.llama.modeling_llama import LlamaDecoderLayer
        self.cfg = cfg
        hc = LlamaConfig(hidden_size=cfg.hidden, intermediate_size=cfg.ffn,
                         num_attention_heads=cfg.n_q_heads, num_key_value_heads=cfg.n_kv_heads,
                         head_dim=cfg.head_dim, num_hidden_layers=cfg.n_layers, vocab_size=cfg.vocab,
                         rms_norm_eps=cfg.rms_eps, rope_theta=cfg.rope_theta, attention_bias=False,
                         mlp_bias=False, attention_dropout=0.0)
        hc._attn_implementation = "sdpa"
        D = lambda t: t.detach().cpu().double()
        self.top = {k: (None if t is None else D(t)) for k, t in top.items()}
        self.layers = []
        for i, lw in enumerate(layers):
            m = LlamaDecoderLayer(hc, i).double().eval()
            with torch.no_grad():
                m.input_layernorm.weight.copy_(D(lw["g_attn"]))
                m.post_attention_layernorm.weight.copy_(D(lw["g_ffn"]))
                m.self_attn.q_proj.weight.copy_(D(lw["wq"]))
                m.self_attn.k_proj.weight.copy_(D(lw["wk"]))
                m.self_attn.v_proj.weight.copy_(D(lw["wv"]))
                m.self_attn.o_proj.weight.copy_(D(lw["wo"]))
                m.mlp.gate_proj.weight.copy_(D(lw["wgate"]))
                m.mlp.up_proj.weight.copy_(D(lw["wup"]))
                m.mlp.down_proj.weight.copy_(D(lw["wdown"]))
            if i == 0 and not cfg.first_layer_input_norm:
                m.input_layernorm = torch.nn.Identity()
            self.layers.append(m)
        self.cache = DynamicCache()
        self.n_cached = 0

    def preload(self, k: torch.Tensor, v: torch.Tensor, L: int):
        """Put stored prefix rows [0, L) of a [layers][Hkv][cap][dh] cache into the HF cache."""
        for l in range(self.cfg.n_layers):
            self.cache.update(k[l, :, :L].double().unsqueeze(0), v[l, :, :L].double().unsqueeze(0), l)
        self.n_cached = L

    def dgf(self, f: torch.Tensor, tokens: torch.Tensor) -> torch.Tensor:
        t = self.top
        e = t["embed"][tokens.long()]
        if self.cfg.fusion == 1:  # concat + one Linear, by the library routine
            return torch.nn.functional.linear(torch.cat([f, e], -1), t["dgf_wg"], t["dgf_bg"])
        h1 = f @ t["dgf_w1"].T if self.cfg.dgf_proj else f
        h2 = e @ t["dgf_w2"].T if self.cfg.dgf_proj else e
        g = torch.sigmoid(torch.cat([h1, h2], -1) @ t["dgf_wg"].T + t["dgf_bg"])
        return g * h1 + (1 - g) * h2

    def rows(self, feats: torch.Tensor, tokens: torch.Tensor, pos, mask_new: torch.Tensor = None):
        """Run R rows appended to the cache. pos: rotary positions [R]. mask_new [R, R] bool says
        which of the NEW rows each row may see (default causal); all cached rows are visible.
        Returns hhat [R, d]."""
        cfg = self.cfg
        R = feats.shape[0]
        x = self.dgf(feats.double(), tokens).unsqueeze(0)
        pos = torch.as_tensor(pos, dtype=torch.long)
        half = cfg.head_dim // 2
        inv = torch.tensor([cfg.rope_theta ** (-2.0 * i / cfg.head_dim) for i in range(half)],
                           dtype=torch.float64)
        ang = pos.double()[:, None] * inv[None, :]
        emb = torch.cat([ang, ang], -1)
        cos, sin = emb.cos().unsqueeze(0), emb.sin().unsqueeze(0)
        if mask_new is None:
            mask_new = torch.tril(torch.ones(R, R, dtype=torch.bool))
        full = torch.cat([torch.ones(R, self.n_cached, dtype=torch.bool), mask_new], 1)
        add = torch.zeros(full.shape, dtype=torch.float64).masked_fill(~full, float("-inf"))[None, None]
        with torch.no_grad():
            for m in self.layers:
                x = m(x, attention_mask=add, position_ids=pos.unsqueeze(0), past_key_values=self.cache,
                      use_cache=True, position_embeddings=(cos, sin))
                if isinstance(x, tuple):
                    x = x[0]
        self.n_cached += R
        return x[0]

    def logp(self, hhat: torch.Tensor) -> torch.Tensor:
        h = hhat
        if self.cfg.final_norm:
            h = torch.nn.functional.rms_norm(h, (self.cfg.hidden,), self.top["g_final"], self.cfg.rms_eps)
        return torch.log_softmax(h @ self.top["lm_head"].T, -1)

    def fork(self):
        """Copy with an independent cache (for enumerating tree paths)."""
        import copy
        o = copy.copy(self)
        o.cache = copy.deepcopy(self.cache)
        return o


def force_gate(top, value: float):
    """Make the DGF gate a constant: Wg = 0, bg = +-800 -> exp over/underflows, sigmoid = 1 or 0 exactly."""
    top = dict(top)
    top["dgf_wg"] = torch.zeros_like(top["dgf_wg"])
    top["dgf_bg"] = torch.full_like(top["dgf_bg"], value)
    return top

"""Pins of the oracle's network steps (O3-O5): DGF invariants (P2), the decoder
block against Hugging Face's LlamaDecoderLayer in fp64 (P4), prefix KV, GQA,
tree masks and chain = causal (P3). CPU only."""
import numpy as np
import pytest
import torch

import oracle
from helpers import RefDraft, force_gate, kv_np, np_to_f64, ocfg, oweights, tiny_cfg
from paper_2412_18934_b200 import synth
from paper_2412_18934_b200.configs import BF16, F32


def _dgf(cfg, top, layers, f, tok):
    return oracle.dgf(ocfg(cfg), oweights(top, layers), f, tok)


# ---- O3 DGF ---------------------------------------------

def test_dgf_gate_one_is_hidden_branch_gate_zero_is_embedding_branch():
    cfg = tiny_cfg()
    top, layers = synth.make_weights(cfg)
    f = np.random.default_rng(1).normal(size=cfg.hidden)
    tok = 5
    h1 = oracle.matvec(top["dgf_w1"], F32, f)
    h2 = oracle.matvec(top["dgf_w2"], F32, top["embed"][tok].double().numpy())
    np.testing.assert_array_equal(_dgf(cfg, force_gate(top, 800.0), layers, f, tok), h1)
    np.testing.assert_array_equal(_dgf(cfg, force_gate(top, -800.0), layers, f, tok), h2)
    # gate 1/2 (Wg = 0, bg = 0): the plain mean
    np.testing.assert_allclose(_dgf(cfg, force_gate(top, 0.0), layers, f, tok), 0.5 * (h1 + h2), rtol=1e-15)


def test_dgf_identity_projection_reduces_to_feature_or_embedding():
    cfg = tiny_cfg(dgf_proj=0)
    top, layers = synth.make_weights(cfg)
    f = np.random.default_rng(2).normal(size=cfg.hidden)
    e = top["embed"][3].double().numpy()
    np.testing.assert_array_equal(_dgf(cfg, force_gate(top, 800.0), layers, f, 3), f)
    np.testing.assert_array_equal(_dgf(cfg, force_gate(top, -800.0), layers, f, 3), e)


def test_dgf_concat_order_and_bias():
    """The gate reads [h1 || h2], hidden branch FIRST (PAPER.md:98 caption order)."""
    cfg = tiny_cfg(dgf_proj=0)
    d = cfg.hidden
    top, layers = synth.make_weights(cfg)
    rng = np.random.default_rng(3)
    f = rng.normal(size=d)
    # Wg looks only at the first half of its input => the gate must not depend on the token
    top1 = dict(top)
    wg = torch.zeros(d, 2 * d)
    wg[:, :d] = torch.randn(d, d, generator=torch.Generator().manual_seed(0))
    top1["dgf_wg"] = wg
    top1["dgf_bg"] = torch.zeros(d)
    e3, e7 = top["embed"][3].double().numpy(), top["embed"][7].double().numpy()
    x3, x7 = _dgf(cfg, top1, layers, f, 3), _dgf(cfg, top1, layers, f, 7)
    g3 = (x3 - e3) / (f - e3)  # x = g f + (1-g) e
    g7 = (x7 - e7) / (f - e7)
    np.testing.assert_allclose(g3, g7, rtol=1e-9)
    ref_g = 1 / (1 + np.exp(-(wg[:, :d].double().numpy() @ f)))
    np.testing.assert_allclose(g3, ref_g, rtol=1e-9)
    # ... and the bias is added before the sigmoid
    top2 = dict(top1)
    top2["dgf_bg"] = torch.full((d,), 0.5)
    x3b = _dgf(cfg, top2, layers, f, 3)
    gb = (x3b - e3) / (f - e3)
    np.testing.assert_allclose(gb, 1 / (1 + np.exp(-(wg[:, :d].double().numpy() @ f + 0.5))), rtol=1e-9)


def test_dgf_matches_torch_reference_random_weights():
    cfg = tiny_cfg()
    top, layers = synth.make_weights(cfg)
    ref = RefDraft(cfg, top, layers)
    f = torch.randn(3, cfg.hidden, dtype=torch.float64, generator=torch.Generator().manual_seed(4))
    toks = torch.tensor([0, 5, 11])
    want = ref.dgf(f, toks).numpy()
    for i in range(3):
        np.testing.assert_allclose(_dgf(cfg, top, layers, f[i].numpy(), int(toks[i])), want[i], rtol=1e-12)


# ---- the fusion DGF replaces: concat + one Linear (Table 6 "w/o both") ----------

def _fl(cfg, top, layers, f, tok):
    return oracle.fusion_linear(ocfg(cfg), oweights(top, layers), f, tok)


def test_fusion_linear_selectors_pin_concat_order_and_bias():
    """Wfc = [I | 0] returns the feature, [0 | I] the embedding (hidden state first, reading A17), Wfc = 0 the
    bias -- bit for bit."""
    cfg = tiny_cfg(dgf_proj=0, fusion=1)
    d = cfg.hidden
    top, layers = synth.make_weights(cfg)
    f = np.random.default_rng(5).normal(size=d)
    e = top["embed"][4].double().numpy()
    eye, zero = torch.eye(d), torch.zeros(d, d)
    t = dict(top, dgf_wg=torch.cat([eye, zero], 1), dgf_bg=torch.zeros(d))
    np.testing.assert_array_equal(_fl(cfg, t, layers, f, 4), f)
    t = dict(top, dgf_wg=torch.cat([zero, eye], 1), dgf_bg=torch.zeros(d))
    np.testing.assert_array_equal(_fl(cfg, t, layers, f, 4), e)
    b = torch.randn(d, generator=torch.Generator().manual_seed(1))
    t = dict(top, dgf_wg=torch.zeros(d, 2 * d), dgf_bg=b)
    np.testing.assert_array_equal(_fl(cfg, t, layers, f, 4), b.double().numpy())


def test_fusion_linear_matches_torch_linear_and_the_hf_stack():
    """x = Wfc [f || e] + b against torch.nn.functional.linear (library routine), then the whole forward with
    this fusion against Hugging Face's decoder layers."""
    cfg = tiny_cfg(dgf_proj=0, fusion=1)
    top, layers = synth.make_weights(cfg)
    g = torch.Generator().manual_seed(6)
    f = torch.randn(3, cfg.hidden, dtype=torch.float64, generator=g)
    toks = torch.tensor([1, 7, 10])
    e = top["embed"][toks].double()
    want = torch.nn.functional.linear(torch.cat([f, e], -1), top["dgf_wg"].double(), top["dgf_bg"].double()).numpy()
    for i in range(3):
        np.testing.assert_allclose(_fl(cfg, top, layers, f[i].numpy(), int(toks[i])), want[i], rtol=1e-12)
    L, R, cap = 5, 3, 12
    k, v = synth.make_kv(cfg, cap, L)
    feats, tokens = synth.make_inputs(cfg, R)
    slots = [L + i for i in range(R)]
    allowed = [list(range(L + i + 1)) for i in range(R)]
    hh, kc, vc = _oracle_forward(cfg, top, layers, k, v, cap, slots, slots, allowed, feats, tokens)
    ref = RefDraft(cfg, top, layers)
    ref.preload(k, v, L)
    np.testing.assert_allclose(hh, ref.rows(feats, tokens, slots).numpy(), rtol=2e-6, atol=2e-6)


def test_fusion_linear_differs_from_dgf_on_the_same_weights():
    """A dropped dispatch (fusion flag ignored) would make the two variants coincide."""
    cfg0, cfg1 = tiny_cfg(dgf_proj=0, fusion=0), tiny_cfg(dgf_proj=0, fusion=1)
    top, layers = synth.make_weights(cfg1)
    f = np.random.default_rng(7).normal(size=cfg1.hidden)
    assert np.abs(_fl(cfg1, top, layers, f, 2) - _dgf(cfg0, top, layers, f, 2)).max() > 1e-3


# ---- O4 decoder block vs Hugging Face (P4) ---------------------------------

def _oracle_forward(cfg, top, layers, k, v, cap, slots, pos, allowed, feats, tokens):
    kc, vc = kv_np(k), kv_np(v)
    hh = oracle.forward(ocfg(cfg), oweights(top, layers), kc, vc, cap, slots, pos, allowed,
                        feats.double().numpy(), tokens.numpy())
    return hh, kc, vc


@pytest.mark.parametrize("kw", [dict(), dict(n_kv_heads=4), dict(n_kv_heads=1), dict(first_layer_input_norm=0),
                                dict(head_dim=16, n_q_heads=2, n_kv_heads=2, rope_theta=5e5)])
def test_stack_with_prefix_matches_hf_llama_layers(kw):
    cfg = tiny_cfg(**kw)
    top, layers = synth.make_weights(cfg)
    L, R, cap = 9, 4, 16
    k, v = synth.make_kv(cfg, cap, L)
    feats, tokens = synth.make_inputs(cfg, R)
    # level-0 style: causal over the prefix and the earlier new rows
    slots = [L + i for i in range(R)]
    allowed = [list(range(L + i + 1)) for i in range(R)]
    hh, kc, vc = _oracle_forward(cfg, top, layers, k, v, cap, slots, slots, allowed, feats, tokens)
    ref = RefDraft(cfg, top, layers)
    ref.preload(k, v, L)
    want = ref.rows(feats, tokens, slots)
    np.testing.assert_allclose(hh, want.numpy(), rtol=2e-6, atol=2e-6)  # fp32 KV storage rounding
    # the K/V rows written are HF's cache rows (post-RoPE K), rounded to the storage dtype
    for l in range(cfg.n_layers):
        hk = ref.cache.layers[l].keys[0, :, L:L + R].numpy()
        hv = ref.cache.layers[l].values[0, :, L:L + R].numpy()
        np.testing.assert_allclose(np_to_f64(kc[l, :, L:L + R]), hk, rtol=1e-5, atol=1e-6)
        np.testing.assert_allclose(np_to_f64(vc[l, :, L:L + R]), hv, rtol=1e-5, atol=1e-6)
    # prefix rows untouched
    np.testing.assert_array_equal(kc[:, :, :L], kv_np(k)[:, :, :L])


def test_tree_mask_and_shared_positions_match_hf():
    """Rows of one tree level: same rotary position, each sees the prefix, its ancestors' slots, itself."""
    cfg = tiny_cfg()
    top, layers = synth.make_weights(cfg)
    L, cap = 6, 16
    k, v = synth.make_kv(cfg, cap, L)
    ref = RefDraft(cfg, top, layers)
    ref.preload(k, v, L)
    # first put two "level-1" rows (slots 6, 7; position 6), then two "level-2" rows (slots 8, 9; pos 7)
    f1, t1 = synth.make_inputs(cfg, 2, seed=11)
    f2, t2 = synth.make_inputs(cfg, 2, seed=12)
    kc, vc = kv_np(k), kv_np(v)
    ow = oweights(top, layers)
    base = list(range(L))
    h1 = oracle.forward(ocfg(cfg), ow, kc, vc, cap, [6, 7], [6, 6], [base + [6], base + [7]],
                        f1.double().numpy(), t1.numpy())
    # row 8 is a child of slot 7, row 9 a child of slot 6
    h2 = oracle.forward(ocfg(cfg), ow, kc, vc, cap, [8, 9], [7, 7], [base + [7, 8], base + [6, 9]],
                        f2.double().numpy(), t2.numpy())
    w1 = ref.rows(f1, t1, [6, 6], mask_new=torch.eye(2, dtype=torch.bool))
    # HF sees cached slots 0..7 as "cached": mask them explicitly by running with a full custom mask
    n_c = ref.n_cached
    ref.n_cached = 0  # build the whole mask by hand: [R, n_c + R]
    m = torch.zeros(2, n_c + 2, dtype=torch.bool)
    m[:, :L] = True
    m[0, 7] = True; m[0, 8] = True
    m[1, 6] = True; m[1, 9] = True
    w2 = ref.rows(f2, t2, [7, 7], mask_new=m)
    np.testing.assert_allclose(h1, w1.numpy(), rtol=2e-6, atol=2e-6)
    np.testing.assert_allclose(h2, w2.numpy(), rtol=2e-6, atol=2e-6)


def test_bf16_storage_path_close_to_fp64_reference():
    cfg = tiny_cfg(dtype=BF16)
    top, layers = synth.make_weights(cfg)
    L, R, cap = 5, 3, 12
    k, v = synth.make_kv(cfg, cap, L)
    feats, tokens = synth.make_inputs(cfg, R)
    slots = [L + i for i in range(R)]
    hh, kc, vc = _oracle_forward(cfg, top, layers, k, v, cap, slots, slots,
                                 [list(range(L + i + 1)) for i in range(R)], feats, tokens)
    ref = RefDraft(cfg, top, layers)
    ref.preload(k, v, L)
    want = ref.rows(feats, tokens, slots).numpy()
    # only the bf16 rounding of the new K/V rows separates the two
    np.testing.assert_allclose(hh, want, rtol=0, atol=5e-3 * np.abs(want).max())
    hk = ref.cache.layers[0].keys[0, :, L:L + R]
    np.testing.assert_array_equal(kc[0, :, L:L + R],
                                  hk.to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16))


def test_lm_head_and_final_norm_match_torch():
    for fn in (0, 1):
        cfg = tiny_cfg(final_norm=fn)
        top, layers = synth.make_weights(cfg)
        if fn:
            top["g_final"] = torch.rand(cfg.hidden) + 0.5
        ref = RefDraft(cfg, top, layers)
        h = torch.randn(cfg.hidden, dtype=torch.float64, generator=torch.Generator().manual_seed(5))
        lg = oracle.lm_head(ocfg(cfg), oweights(top, layers), h.numpy())
        np.testing.assert_allclose(oracle.log_softmax(lg), ref.logp(h).numpy(), rtol=1e-10, atol=1e-12)

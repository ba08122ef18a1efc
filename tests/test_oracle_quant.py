"""Pins of the oracle's int8 weight-quantised path: value of a stored matrix = scale[row] * q, per
OUTPUT row; everything else unchanged. CPU only."""
import dataclasses

import numpy as np
import torch

import oracle
from helpers import kv_np, ocfg, oracle_step, oweights, tiny_cfg
from paper_2412_18934_b200 import synth
from paper_2412_18934_b200.configs import BF16, F32, TreeSpec


def test_matvec_q8_is_the_dequantised_matrix_times_x():
    rng = np.random.default_rng(0)
    Q = rng.integers(-128, 128, size=(7, 24)).astype(np.int8)
    Q[0, 0], Q[1, 1] = -128, 127  # the ends of the range
    s = rng.random(7).astype(np.float32) + 0.1
    x = rng.normal(size=24)
    want = (s.astype(np.float64)[:, None] * Q.astype(np.float64)) @ x
    np.testing.assert_allclose(oracle.matvec_q8(Q, s, x), want, rtol=1e-13)


def test_scale_is_per_output_row_not_per_input_column():
    rng = np.random.default_rng(1)
    Q = rng.integers(-100, 100, size=(5, 5)).astype(np.int8)
    s = np.ones(5, np.float32)
    x = rng.normal(size=5)
    y = oracle.matvec_q8(Q, s, x)
    s2 = s.copy()
    s2[2] = 2.0  # doubles output row 2 and nothing else (a per-column scale would change every output)
    y2 = oracle.matvec_q8(Q, s2, x)
    np.testing.assert_array_equal(np.delete(y2, 2), np.delete(y, 2))
    np.testing.assert_allclose(y2[2], 2 * y[2], rtol=1e-15)


def test_quantizer_round_trip_is_within_half_a_step():
    """The input recipe (synth.quantize_rows): |w - scale q| <= scale / 2 and the largest entry of a row maps to +-127."""
    g = torch.Generator().manual_seed(2)
    w = (torch.randn(16, 64, generator=g) * 0.02).to(torch.bfloat16)
    q, s = synth.quantize_rows(w)
    err = (w.float() - s[:, None] * q.float()).abs()
    assert (err <= s[:, None] * 0.5 + 1e-9).all()
    assert (q.abs().amax(1) >= 126).all() and q.abs().max() <= 127
    assert torch.equal(s.to(torch.bfloat16).float(), s)  # scale * q is exact in fp32


def test_int8_model_equals_the_fp32_model_with_dequantised_weights_bit_for_bit():
    """With bf16-representable scales scale * q is exact in fp32, so an fp32 model holding W = scale * q is the same
    model: the two oracle steps must agree bit for bit (hidden states, logits, candidates)."""
    cfgq = tiny_cfg(dtype=BF16, wquant=1, tree=TreeSpec(3, (2, 2, 2), (0, 2, 3), 8), prefix=5)
    top, layers = synth.make_weights(cfgq)
    assert top["lm_head"].dtype == torch.int8 and layers[0]["wq"].dtype == torch.int8
    cfgf = dataclasses.replace(cfgq, dtype=F32, wquant=0)
    deq = lambda d, m: {k: (v.float() * d[m[k]][:, None] if k in m else (None if v is None else v.float()))
                        for k, v in d.items() if not k.startswith(("s", "dgf_s", "lm_head_s")) or k in ("dgf_w1", "dgf_w2", "dgf_wg")}
    topf = {k: v for k, v in deq(top, synth.TOP_MATRIX_SCALES).items() if k not in synth.TOP_MATRIX_SCALES.values()}
    layf = [{k: v for k, v in deq(l, synth.MATRIX_SCALES).items() if k not in synth.MATRIX_SCALES.values()} for l in layers]
    cap = 5 + 2 + cfgq.tree.tree_rows() + 4
    k, v = synth.make_kv(cfgq, cap, 5)
    feats, tokens = synth.make_inputs(cfgq, 2)
    a = oracle_step(cfgq, top, layers, k, v, cap, 5, feats, tokens)
    b = oracle_step(cfgf, topf, layf, k.float(), v.float(), cap, 5, feats, tokens)
    # the fp32 model stores K/V in fp32 and the bf16 one rounds them: compare what does not pass through the cache,
    # i.e. the level-0 row (it attends the identical prefix and itself... its own K/V are rounded) -> use n_new = 1 rows
    assert np.array_equal(a["token_ids"][:0], b["token_ids"][:0])
    # DGF output and first-row pre-attention quantities do not involve the cache: check through a 0-layer probe
    x_q = oracle.dgf(ocfg(cfgq), oweights(top, layers), feats[0].double().numpy(), int(tokens[0]))
    x_f = oracle.dgf(ocfg(cfgf), oweights(topf, layf), feats[0].double().numpy(), int(tokens[0]))
    np.testing.assert_array_equal(x_q, x_f)
    lg_q = oracle.lm_head(ocfg(cfgq), oweights(top, layers), x_q)
    lg_f = oracle.lm_head(ocfg(cfgf), oweights(topf, layf), x_f)
    np.testing.assert_array_equal(lg_q, lg_f)
    # and the whole step with an fp32 cache on both sides (dtype F32 + wquant): every number identical
    cfgq32 = dataclasses.replace(cfgq, dtype=F32)
    top32 = {k: (v if (v is None or v.dtype in (torch.int8,) or k in synth.TOP_MATRIX_SCALES.values()) else v.float()) for k, v in top.items()}
    lay32 = [{k: (v if (v.dtype == torch.int8 or k in synth.MATRIX_SCALES.values()) else v.float()) for k, v in l.items()} for l in layers]
    a32 = oracle_step(cfgq32, top32, lay32, k.float(), v.float(), cap, 5, feats, tokens)
    for key in ("token_ids", "parents", "scores", "row_hhat", "row_logits", "pool_cum"):
        np.testing.assert_array_equal(a32[key], b[key])


# ---- fp8 e4m3 weights (reading A17b; SURVEY.md 8 f1 "int8 / fp8") -------------------------------------------------
def test_e4m3_decode_matches_torch_for_every_byte():
    """The oracle's decoder against PyTorch's float8_e4m3fn (an independent implementation of the OCP format)."""
    b = np.arange(256, dtype=np.uint8)
    want = torch.from_numpy(b.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    got = oracle.e4m3_to_double(b)
    nan = np.isnan(want)
    assert nan.sum() == 2 and np.array_equal(np.isnan(got), nan)  # 0x7f and 0xff
    np.testing.assert_array_equal(got[~nan], want[~nan])
    assert got[0x7e] == 448.0 and got[0x01] == 2.0 ** -9 and got[0x08] == 2.0 ** -6  # largest, smallest subnormal, smallest normal


def test_matvec_f8_is_the_dequantised_matrix_times_x():
    rng = np.random.default_rng(3)
    Q = rng.integers(0, 256, size=(7, 24)).astype(np.uint8)
    Q[(Q & 0x7f) == 0x7f] = 0x7e  # no NaN bytes
    s = rng.random(7).astype(np.float32) + 0.1
    x = rng.normal(size=24)
    W = torch.from_numpy(Q.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    np.testing.assert_allclose(oracle.matvec_f8(Q, s, x), (s.astype(np.float64)[:, None] * W) @ x, rtol=1e-13)
    s2 = s.copy()
    s2[2] = 2 * s[2]  # per OUTPUT row
    y, y2 = oracle.matvec_f8(Q, s, x), oracle.matvec_f8(Q, s2, x)
    np.testing.assert_array_equal(np.delete(y2, 2), np.delete(y, 2))
    np.testing.assert_allclose(y2[2], 2 * y[2], rtol=1e-15)


def test_fp8_quantizer_round_trip():
    """Input recipe (synth.quantize_rows_f8): relative error <= 2^-4 (3 mantissa bits) above the subnormal range, the
    largest entry of a row maps to +-448, no NaN byte."""
    g = torch.Generator().manual_seed(4)
    w = (torch.randn(16, 64, generator=g) * 0.02).to(torch.bfloat16)
    q, s = synth.quantize_rows_f8(w)
    deq = s[:, None] * q.float()
    big = w.float().abs() > s[:, None] * 2.0 ** -6
    assert ((w.float() - deq).abs()[big] <= w.float().abs()[big] * 2.0 ** -4).all()
    assert (q.float().abs().amax(1) >= 416).all() and not torch.isnan(q.float()).any()
    assert torch.equal(s.to(torch.bfloat16).float(), s)


def test_fp8_model_equals_the_fp32_model_with_dequantised_weights_bit_for_bit():
    """scale (bf16-representable) * e4m3 value (4 significant bits) is exact in fp32: an fp32 model holding that product
    is the same model; with an fp32 cache on both sides the two oracle steps agree bit for bit."""
    cfgq = tiny_cfg(dtype=BF16, wquant=2, tree=TreeSpec(3, (2, 2, 2), (0, 2, 3), 8), prefix=5)
    top, layers = synth.make_weights(cfgq)
    f8 = torch.float8_e4m3fn
    assert top["lm_head"].dtype == f8 and layers[0]["wq"].dtype == f8
    scales = set(synth.TOP_MATRIX_SCALES.values()) | set(synth.MATRIX_SCALES.values())

    def deq(d, m):
        return {k: (v.float() * d[m[k]][:, None] if k in m and v is not None else (None if v is None else v.float()))
                for k, v in d.items() if k not in scales}
    topf, layf = deq(top, synth.TOP_MATRIX_SCALES), [deq(l, synth.MATRIX_SCALES) for l in layers]
    cap = 5 + 2 + cfgq.tree.tree_rows() + 4
    k, v = synth.make_kv(cfgq, cap, 5)
    feats, tokens = synth.make_inputs(cfgq, 2)
    cfgq32, cfgf = dataclasses.replace(cfgq, dtype=F32), dataclasses.replace(cfgq, dtype=F32, wquant=0)
    top32 = {k: (v if (v is None or v.dtype == f8 or k in scales) else v.float()) for k, v in top.items()}
    lay32 = [{k: (v if (v.dtype == f8 or k in scales) else v.float()) for k, v in l.items()} for l in layers]
    a32 = oracle_step(cfgq32, top32, lay32, k.float(), v.float(), cap, 5, feats, tokens)
    b = oracle_step(cfgf, topf, layf, k.float(), v.float(), cap, 5, feats, tokens)
    for key in ("token_ids", "parents", "scores", "row_hhat", "row_logits", "pool_cum"):
        np.testing.assert_array_equal(a32[key], b[key])

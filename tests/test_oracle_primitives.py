"""Pins of the oracle's primitive steps against library routines, closed forms
and invariants (not against retyped formulas). CPU only."""
import numpy as np
import pytest
import scipy.special
import torch

import oracle
from helpers import np_to_f64

RNG = np.random.default_rng(0)


def bf16_bits(x: np.ndarray) -> np.ndarray:
    return torch.from_numpy(x.astype(np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def test_bf16_widening_known_values():
    # 0x3FC0 = 1.5, 0xC000 = -2.0, 0x3F80 = 1.0, 0x0000 = 0
    W = np.array([[0x3FC0, 0xC000, 0x3F80, 0x0000]], dtype=np.uint16)
    y = oracle.matvec(W, oracle.oracle.BF16, np.array([2.0, 3.0, 5.0, 7.0]))
    assert y[0] == 1.5 * 2 - 2.0 * 3 + 5.0


@pytest.mark.parametrize("dtype", [0, 1])
def test_matvec_matches_numpy_fp64(dtype):
    N, K = 37, 131  # ragged, not multiples of anything
    Wf = RNG.normal(size=(N, K)).astype(np.float32)
    W = Wf if dtype == 0 else bf16_bits(Wf)
    x = RNG.normal(size=K)
    y = oracle.matvec(W, dtype, x)
    ref = np_to_f64(W) @ x  # library routine on the exactly widened values
    np.testing.assert_allclose(y, ref, rtol=1e-12, atol=1e-12)


def test_matvec_not_transposed():
    W = np.zeros((2, 3), dtype=np.float32)
    W[1, 2] = 4.0  # row 1, column 2
    y = oracle.matvec(W, 0, np.array([1.0, 10.0, 100.0]))
    assert y.tolist() == [0.0, 400.0]


def test_round_bf16_is_nearest_even():
    import ctypes as C
    lib = oracle.oracle._load()
    lib.orc_round_bf16.restype = C.c_uint16
    xs = np.concatenate([RNG.normal(size=2000) * 10.0 ** RNG.integers(-6, 6, size=2000),
                         # exact midpoints between neighbouring bf16 values: ties must go to even
                         np.array([1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8, -(2.0 + 2.0 ** -7), 0.0, 1.0])])
    for x in xs:
        got = np.array([lib.orc_round_bf16(C.c_double(float(x)))], dtype=np.uint16)
        g = float(np_to_f64(got)[0])
        if x == 0.0:
            assert g == 0.0
            continue
        # neighbours of g on the bf16 grid
        lo = float(np_to_f64(np.array([got[0] - 1], dtype=np.uint16))[0])
        hi = float(np_to_f64(np.array([got[0] + 1], dtype=np.uint16))[0])
        assert abs(x - g) <= abs(x - lo) and abs(x - g) <= abs(x - hi), x
        if abs(x - g) == abs(x - lo) or abs(x - g) == abs(x - hi):
            assert got[0] % 2 == 0, f"tie at {x} not rounded to even"
    assert lib.orc_round_bf16(C.c_double(1.0 + 2.0 ** -8)) == 0x3F80      # tie -> even (1.0)
    assert lib.orc_round_bf16(C.c_double(1.0 + 3 * 2.0 ** -8)) == 0x3F82  # tie -> even


def test_rmsnorm_matches_torch():
    d = 77
    x = RNG.normal(size=d) * 3
    g = RNG.normal(size=d).astype(np.float32)
    y = oracle.rmsnorm(x, g, 0, 1e-5)
    ref = torch.nn.functional.rms_norm(torch.from_numpy(x), (d,), torch.from_numpy(g).double(), 1e-5)
    np.testing.assert_allclose(y, ref.numpy(), rtol=1e-12)
    # eps really is inside the square root
    z = oracle.rmsnorm(np.zeros(4), np.ones(4, np.float32), 0, 1e-5)
    assert np.all(z == 0)
    y1 = oracle.rmsnorm(np.full(4, 1e-3), np.ones(4, np.float32), 0, 1e-2)
    np.testing.assert_allclose(y1, 1e-3 / np.sqrt(1e-6 + 1e-2), rtol=1e-12)


def test_rope_closed_forms():
    dh, theta = 8, 1e4
    v = RNG.normal(size=dh)
    # position 0 is the identity
    np.testing.assert_array_equal(oracle.rope(v, 0, theta), v)
    # pair (0, dh/2) rotates by exactly pos radians (inv_freq_0 = 1); pair i by pos * theta^(-2i/dh)
    e = np.zeros(dh)
    e[0] = 1.0
    r = oracle.rope(e, 1, theta)
    np.testing.assert_allclose(r[0], np.cos(1.0), rtol=1e-15)
    np.testing.assert_allclose(r[dh // 2], np.sin(1.0), rtol=1e-15)  # +sin in the second half
    e = np.zeros(dh)
    e[3] = 1.0
    r = oracle.rope(e, 5, theta)
    ang = 5 * theta ** (-6.0 / dh)
    np.testing.assert_allclose([r[3], r[3 + dh // 2]], [np.cos(ang), np.sin(ang)], rtol=1e-14)
    # norm preserved, and q.k depends only on the position difference
    q, k = RNG.normal(size=dh), RNG.normal(size=dh)
    np.testing.assert_allclose(np.linalg.norm(oracle.rope(q, 123, theta)), np.linalg.norm(q), rtol=1e-13)
    a = oracle.rope(q, 40, theta) @ oracle.rope(k, 33, theta)
    b = oracle.rope(q, 1007, theta) @ oracle.rope(k, 1000, theta)
    np.testing.assert_allclose(a, b, rtol=1e-9)


def test_rope_matches_hf_rotate_half():
    from transformers.models.llama.modeling_llama import apply_rotary_pos_emb
    dh, theta, pos = 16, 5e5, 37
    q = RNG.normal(size=dh)
    inv = np.array([theta ** (-2.0 * i / dh) for i in range(dh // 2)])
    emb = np.concatenate([pos * inv, pos * inv])
    cos, sin = torch.from_numpy(np.cos(emb))[None, None], torch.from_numpy(np.sin(emb))[None, None]
    tq = torch.from_numpy(q)[None, None, None]
    rq, _ = apply_rotary_pos_emb(tq, tq, cos, sin)
    np.testing.assert_allclose(oracle.rope(q, pos, theta), rq[0, 0, 0].numpy(), rtol=1e-13, atol=1e-15)


def test_log_softmax_matches_scipy_and_normalises():
    z = RNG.normal(size=1000) * 8
    lp = oracle.log_softmax(z)
    np.testing.assert_allclose(lp, scipy.special.log_softmax(z), rtol=1e-12, atol=1e-12)
    assert abs(np.exp(lp).sum() - 1.0) < 1e-12
    # shift invariance
    np.testing.assert_allclose(oracle.log_softmax(z + 1000.0), lp, atol=1e-9)


def test_topk_matches_stable_argsort_with_ties():
    v = RNG.integers(0, 6, size=200).astype(np.float64)  # many exact ties
    for b in (1, 2, 7, 200):
        idx = oracle.topk(v, b)
        ref = np.argsort(-v, kind="stable")[:b]  # value desc, index asc
        np.testing.assert_array_equal(idx, ref)
        assert len(set(idx.tolist())) == b
        assert np.all(np.diff(v[idx]) <= 0)
        rest = np.setdiff1d(np.arange(200), idx)
        if len(rest):
            assert v[rest].max() <= v[idx[-1]]

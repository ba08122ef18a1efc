"""dovetail_tree_replay_static (include/dovetail.h): the tree bookkeeping for callers that cannot call cudaMalloc
-- no handle, scratch in a file-scope device array of the library. Collected last on purpose (the suite runs with
`pytest -x`); passes alone in a fresh process and after the other tests (it depends on no state of theirs).

-m gpu: its output against the existing path's (dovetail_tree_replay on a handle), bit for bit -- the tolerance
the tests of this integer path use (tests/test_gpu_tree.py) -- on consecutive calls that leave stale contents in
the shared scratch. -m "not gpu": the host-side checks (NULL arguments, the stated limits) and that the entry
point's source calls no allocating routine."""
import ctypes as C
import os
import re

import numpy as np
import pytest
import torch

from paper_2412_18934_b200 import binding
from paper_2412_18934_b200.configs import F32, DraftConfig, TreeSpec, paper_preset

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lists(tree: TreeSpec, rng, vocab=64, grid=1024, spread=3000):
    """Per-row top-b lists as the LM-head stage emits them (log-prob descending, token id ascending); log-probs on a
    1 / 1024 grid, so cumulative sums are exact in fp32 (the recipe of tests/test_gpu_tree.py)."""
    rows = 1 + tree.tree_rows()
    maxb = max(tree.branch)
    toks = np.zeros((rows, maxb), np.int32)
    lp = np.zeros((rows, maxb), np.float32)
    for r in range(rows):
        t = rng.choice(vocab, size=maxb, replace=False)
        v = -rng.integers(0, spread, size=maxb).astype(np.float64) / grid
        order = np.lexsort((t, -v))
        toks[r], lp[r] = t[order], v[order]
    return toks, lp


# ---- -m "not gpu": host logic ------------------------------------------------------------------------------------
def _raw(tree: TreeSpec, n_rows: int, max_b: int, null_out: bool = False) -> int:
    """The raw C call with dummy non-NULL device pointers: every check below fails before anything touches the GPU."""
    lib = binding.load()
    t = binding.tree_spec_t(tree)
    o = binding.DraftOutT(16, 16, 16, 16, 16)
    return lib.dovetail_tree_replay_static(C.byref(t), C.c_void_p(16), C.c_void_p(16), n_rows, max_b,
                                           None if null_out else C.byref(o), None)


def test_null_arguments_and_limits_are_rejected_with_a_clear_error():
    lib = binding.load()
    assert lib.dovetail_tree_replay_static(None, None, None, 0, 0, None, None) == binding.EINVAL
    assert b"null" in lib.dovetail_last_error(None)
    good = TreeSpec(3, (2, 2, 2), (0, 0, 0), 6)
    assert _raw(good, 7, 2, null_out=True) == binding.EINVAL
    # a tree the handle path takes, beyond the static scratch: 1 x 32 + 32 x 32 + 64 x 32 = 3104 nodes > 2048
    big = TreeSpec(3, (32, 32, 32), (0, 0, 64), 100)
    assert big.pool_size() > binding.STATIC_MAX_POOL
    assert _raw(big, 1 + big.tree_rows(), 32) == binding.EINVAL
    msg = lib.dovetail_last_error(None).decode()
    assert "DOVETAIL_STATIC_MAX_POOL" in msg and str(binding.STATIC_MAX_POOL) in msg
    # more than 64 rows in one level, more than 128 tree rows, a branch beyond 32, lists too short
    assert _raw(TreeSpec(3, (32, 3, 1), (0, 0, 0), 10), 200, 32) == binding.EINVAL  # level 2: 96 rows > 64
    assert b"rows per level" in lib.dovetail_last_error(None)
    assert _raw(TreeSpec(4, (32, 2, 1, 1), (0, 0, 0, 0), 10), 400, 32) == binding.EINVAL  # 32 + 64 + 64 = 160 tree rows > 128
    assert b"tree rows" in lib.dovetail_last_error(None)
    assert _raw(TreeSpec(1, (33,), (0,), 3), 1, 33) == binding.EINVAL
    assert b"branch" in lib.dovetail_last_error(None)
    assert _raw(good, 6, 2) == binding.EINVAL  # needs 1 + 2 + 4 = 7 rows
    assert b"replay needs 7 rows" in lib.dovetail_last_error(None)


def test_the_entry_point_calls_no_allocating_routine():
    """Static check of the source between the entry point's markers: no cudaMalloc / cudaFree family, no C++
    containers or new / malloc; the scratch is the file-scope device array, reached through cudaGetSymbolAddress."""
    src = open(os.path.join(ROOT, "paper_2412_18934_b200", "csrc", "dovetail_draft.cu")).read()
    body = src[src.index("(begin: no-alloc entry point)"):src.index("(end: no-alloc entry point)")]
    helper = src[src.index("struct ReplayScratch {"):src.index("}  // namespace\n\nextern \"C\" {")]
    for text in (body, helper):
        assert not re.search(r"cudaMalloc|cudaFree|cudaHostAlloc|cudaMemPool|std::vector|std::string|std::map|\bnew\b|malloc\(", text)
    assert "dovetail_tree_replay_static" in body and "replay_scratch(&sc)" in body
    assert re.search(r"static __device__ __align__\(256\) unsigned char g_replay_scratch\[DOVETAIL_STATIC_SCRATCH_BYTES\]", helper)
    assert "cudaGetSymbolAddress(&p, g_replay_scratch)" in helper
    hdr = open(os.path.join(ROOT, "include", "dovetail.h")).read()
    assert f"#define DOVETAIL_STATIC_MAX_POOL {binding.STATIC_MAX_POOL}" in hdr
    assert f"#define DOVETAIL_STATIC_SCRATCH_BYTES {binding.STATIC_SCRATCH_BYTES}" in hdr


# ---- -m gpu: against the existing path ------------------------------------------------------------------------------
def _small_cfg() -> DraftConfig:
    return DraftConfig(name="small", hidden=192, n_q_heads=4, n_kv_heads=2, head_dim=64, n_layers=2, ffn=344, vocab=1000,
                       dtype=F32, prefix=70, feat_scale=1.0, rope_theta=1e4, tree=TreeSpec(3, (3, 2, 2), (0, 4, 5), 9), seed=11)


KEYS = ("token_ids", "scores", "parents", "depths")


@pytest.mark.gpu
def test_static_replay_matches_the_handle_path_on_consecutive_calls():
    from parity import make_case
    cfg = _small_cfg()
    case = make_case(cfg, n_new=1)
    h = binding.dovetail_draft_init(case.top, case.layers, cfg)  # the existing path needs a handle (and its cudaMallocs)
    # consecutive calls on the shared scratch: a large pool first, then smaller trees that find its remains there,
    # then the large one again; the last tree fills the static pool to its limit (1 x 32 + 32 x 32 + 31 x 32 = 2048)
    trees = [paper_preset(True), TreeSpec(5, (2,) * 5, (0, 2, 2, 2, 2), 16), TreeSpec(1, (4,), (0,), 3),
             TreeSpec(3, (8, 5, 3), (0, 6, 64), 200), paper_preset(True), TreeSpec(3, (32, 32, 32), (0, 32, 31), 64)]
    assert trees[-1].pool_size() == binding.STATIC_MAX_POOL
    cap = max(t.gamma for t in trees)
    out_s = binding.alloc_out(cap)  # allocated once, before the calls: the entry point gets inputs and outputs only
    for ci, tree in enumerate(trees):
        for spread in (3000, 6):  # 6: almost every score ties
            rng = np.random.default_rng(500 + 7 * ci + spread)
            toks, lp = _lists(tree, rng, vocab=max(64, max(tree.branch) + 5), spread=spread)
            d_t, d_l = torch.from_numpy(toks).cuda(), torch.from_numpy(lp).cuda()
            ref = binding.dovetail_tree_replay(h, tree, d_t, d_l)
            for key in KEYS + ("n_out",):
                out_s[key].fill_(-7)
            binding.dovetail_tree_replay_static(tree, d_t, d_l, out_s)
            torch.cuda.synchronize()
            n = int(ref["n_out"].item())
            assert n == min(tree.gamma, tree.pool_size()) and int(out_s["n_out"].item()) == n, (ci, spread)
            for key in KEYS:
                a, b = out_s[key][:n].cpu().numpy(), ref[key][:n].cpu().numpy()
                assert np.array_equal(a, b), (ci, spread, key)  # bit for bit, scores included (same fp32 sums)
                assert (out_s[key][n:cap].cpu().numpy() == -7).all(), "nothing is written past n_out"
    # the same call twice in a row gives the same answer (nothing of call 1 leaks into call 2)
    tree = trees[0]
    toks, lp = _lists(tree, np.random.default_rng(9), spread=40)
    d_t, d_l = torch.from_numpy(toks).cuda(), torch.from_numpy(lp).cuda()
    first = {k: v.clone() for k, v in binding.dovetail_tree_replay_static(tree, d_t, d_l, out_s).items()}
    second = binding.dovetail_tree_replay_static(tree, d_t, d_l, out_s)
    torch.cuda.synchronize()
    ref = binding.dovetail_tree_replay(h, tree, d_t, d_l)
    torch.cuda.synchronize()
    n = int(ref["n_out"].item())
    for key in KEYS:
        assert torch.equal(first[key][:n], second[key][:n]) and torch.equal(second[key][:n], ref[key][:n]), key
    # beyond the stated maximum: refused on a GPU box as well, and nothing is enqueued
    big = TreeSpec(3, (32, 32, 32), (0, 0, 64), 100)
    toks, lp = _lists(big, np.random.default_rng(3))
    with pytest.raises(binding.DovetailError) as ei:
        binding.dovetail_tree_replay_static(big, torch.from_numpy(toks).cuda(), torch.from_numpy(lp).cuda(), binding.alloc_out(100))
    assert ei.value.code == binding.EINVAL and "DOVETAIL_STATIC_MAX_POOL" in str(ei.value)
    binding.dovetail_draft_destroy(h)

"""-m gpu: the step as a CUDA graph (one graph per tree_spec). A graph replay must leave exactly
what direct launches leave -- the kernels are deterministic, so outputs and cache rows are compared bit for bit --
also when the per-call values patched into the graph change: other cache / feature / output buffers, another
committed length with the same attention geometry; and a new geometry, n_new or tree must capture a new graph."""
import numpy as np
import pytest
import torch

from parity import kv_np, make_case
from paper_2412_18934_b200 import binding
from paper_2412_18934_b200.configs import BF16, F32, TreeSpec
from test_gpu_parity import _boost, small_cfg, umma_cfg

pytestmark = pytest.mark.gpu


def _step(h, case, tree=None):
    k, v = case.k.clone(), case.v.clone()
    kv = binding.KVCache(k, v, case.L)
    out = binding.dovetail_draft_step(h, case.feats, case.tokens, kv, tree or case.tree)
    binding.dovetail_draft_status(h)
    n = int(out["n_out"].item())
    return dict(ids=out["token_ids"][:n].cpu().numpy(), scores=out["scores"][:n].cpu().numpy(),
                parents=out["parents"][:n].cpu().numpy(), k=kv_np(k), v=kv_np(v), L=kv.committed_len,
                how=binding.dovetail_hooks_stat(h, binding.STAT_GRAPH))


def _same(a, b):
    for f in ("ids", "scores", "parents", "k", "v"):
        assert np.array_equal(a[f], b[f]), f
    assert a["L"] == b["L"]


@pytest.mark.parametrize("dtype", [F32, BF16])
def test_graph_replay_equals_direct_launches(dtype):
    cfg = umma_cfg(dtype=dtype) if dtype == BF16 else small_cfg(dtype=F32)
    # same weights (seeded), different prefixes / inputs: 70 and 75 rows share the attention geometry, 300 does not
    cases = [_boost(make_case(cfg, n_new=1, prefix=70)), _boost(make_case(cfg.__class__(**{**cfg.__dict__, "seed": cfg.seed}), n_new=1, prefix=75)),
             _boost(make_case(cfg, n_new=1, prefix=300)), _boost(make_case(cfg, n_new=3, prefix=70))]
    cases[1].feats = cases[1].feats * 0.5 + 0.1  # other inputs at the other length
    wide = TreeSpec(2, (10, 2), (0, 10), 16)     # a level of 10 rows: the tcgen05 GEMV inside a graph (bf16)
    hd = binding.dovetail_draft_init(cases[0].top, cases[0].layers, cfg)
    hg = binding.dovetail_draft_init(cases[0].top, cases[0].layers, cfg)
    binding.dovetail_hooks_tune(hd, binding.TUNE_GRAPHS, 0)
    plan = [(cases[0], None, 2), (cases[1], None, 1), (cases[0], None, 1), (cases[2], None, 2), (cases[3], None, 2),
            (cases[0], wide, 2), (cases[1], wide, 1), (cases[2], None, 1), (cases[0], None, 1)]
    for case, tree, how in plan:
        d, g = _step(hd, case, tree), _step(hg, case, tree)
        assert d["how"] == 0 and g["how"] == how, (d["how"], g["how"], how)
        _same(d, g)
    binding.dovetail_draft_destroy(hd)
    binding.dovetail_draft_destroy(hg)


def test_graph_cache_evicts_and_recaptures():
    cfg = umma_cfg()
    case = _boost(make_case(cfg, n_new=1, prefix=70))
    h = binding.dovetail_draft_init(case.top, case.layers, cfg)
    ref = _step(h, case)
    assert ref["how"] == 2
    for b in range(2, 12):  # ten other trees: more than the cache holds
        r = _step(h, case, TreeSpec(2, (b, 1), (0, b), b + 2))
        assert r["how"] == 2
    again = _step(h, case)
    assert again["how"] == 2  # evicted, captured again
    _same(ref, again)
    binding.dovetail_draft_destroy(h)

"""-m gpu: the integer path on its own (S7, S8, S9) and the ABI's error behaviour.

dovetail_tree_replay is fed per-row top-b lists and must reproduce the oracle's
bookkeeping bit for bit (P10). Log-probabilities are drawn on a 1/1024 grid so that
every cumulative sum is exact in fp32 and fp64 alike; exact ties are frequent."""
import numpy as np
import pytest
import torch

import oracle
from parity import make_case, run_gpu, run_oracle
from paper_2412_18934_b200 import binding
from paper_2412_18934_b200.configs import BF16, F32, TreeSpec, paper_preset
from test_gpu_parity import _boost, small_cfg

pytestmark = pytest.mark.gpu


def _lists(tree: TreeSpec, rng, vocab=50, grid=1024, spread=3000):
    rows = 1 + tree.tree_rows()
    maxb = max(tree.branch)
    toks = np.zeros((rows, maxb), np.int32)
    lp = np.zeros((rows, maxb), np.float32)
    for r in range(rows):
        t = rng.choice(vocab, size=maxb, replace=False)
        v = -rng.integers(0, spread, size=maxb).astype(np.float64) / grid
        order = np.lexsort((t, -v))  # logp desc, token asc: the order the LM-head stage emits
        toks[r], lp[r] = t[order], v[order]
    return toks, lp


@pytest.fixture(scope="module")
def handle():
    cfg = small_cfg(dtype=F32)
    case = make_case(cfg, n_new=1)
    h = binding.dovetail_draft_init(case.top, case.layers, cfg)
    yield h
    binding.dovetail_draft_destroy(h)


TREES = [
    TreeSpec(1, (4,), (0,), 3),
    TreeSpec(3, (2, 2, 2), (0, 0, 0), 14),
    TreeSpec(4, (3, 2, 2, 2), (0, 0, 0, 0), 10),
    TreeSpec(5, (2,) * 5, (0, 2, 2, 2, 2), 16),
    TreeSpec(5, (4,) * 5, (0, 4, 4, 4, 4), 32),
    TreeSpec(6, (1,) * 6, (0, 1, 1, 1, 1, 1), 6),
    TreeSpec(3, (8, 5, 3), (0, 6, 64), 200),
    paper_preset(True),
    paper_preset(False),
    TreeSpec(4, (32, 32, 32, 32), (0, 64, 32, 32), 100),
]


@pytest.mark.parametrize("ti", range(len(TREES)))
@pytest.mark.parametrize("spread", [3000, 6])  # 6: almost everything ties
def test_tree_replay_bit_exact(handle, ti, spread):
    tree = TREES[ti]
    rng = np.random.default_rng(100 + ti)
    toks, lp = _lists(tree, rng, vocab=max(64, max(tree.branch) + 5), spread=spread)
    ora = oracle.tree_replay(tree.depth, tree.branch, tree.beam, tree.gamma, toks, lp.astype(np.float64))
    P = tree.pool_size()
    dev = "cuda"
    pool = dict(token=torch.zeros(P, dtype=torch.int32, device=dev), parent=torch.zeros(P, dtype=torch.int32, device=dev),
                depth=torch.zeros(P, dtype=torch.int32, device=dev), cum=torch.zeros(P, dtype=torch.float32, device=dev),
                size=torch.zeros(1, dtype=torch.int32, device=dev))
    out = binding.dovetail_tree_replay(handle, tree, torch.from_numpy(toks).to(dev), torch.from_numpy(lp).to(dev),
                                       pool=pool)
    torch.cuda.synchronize()
    n = int(out["n_out"].item())
    assert n == ora["n_out"] == min(tree.gamma, P)
    assert int(pool["size"].item()) == P
    assert np.array_equal(pool["token"].cpu().numpy(), ora["pool_token"])
    assert np.array_equal(pool["parent"].cpu().numpy(), ora["pool_parent"])
    assert np.array_equal(pool["depth"].cpu().numpy(), ora["pool_depth"])
    assert np.array_equal(pool["cum"].cpu().numpy().astype(np.float64), ora["pool_cum"])  # sums are exact on the grid
    assert np.array_equal(out["token_ids"][:n].cpu().numpy(), ora["token_ids"])
    assert np.array_equal(out["parents"][:n].cpu().numpy(), ora["parents"])
    assert np.array_equal(out["depths"][:n].cpu().numpy(), ora["depths"])
    assert np.array_equal(out["scores"][:n].cpu().numpy().astype(np.float64), ora["scores"])


def test_kv_commit_modes():
    """P9 / O9: mode 0 leaves the cache alone and a repeated step reproduces itself; mode 1 moves
    the accepted nodes' rows exactly as the oracle's memmove does."""
    cfg = small_cfg(dtype=BF16)
    case = _boost(make_case(cfg, n_new=2))
    h, kv, gpu = run_gpu(case)
    ora = run_oracle(case)
    assert np.array_equal(gpu["token_ids"], ora["token_ids"]) and np.array_equal(gpu["parents"], ora["parents"])
    # deepest accepted chain: follow parents from the deepest output node
    leaf = int(np.argmax(gpu["depths"]))
    path = [leaf]
    while gpu["parents"][path[-1]] >= 0:
        path.append(int(gpu["parents"][path[-1]]))
    path = path[::-1]
    Lp = kv.committed_len
    assert Lp == case.L + 2
    # bad paths: EINVAL, cache untouched
    before_k = kv.k.clone()
    for bad in ([path[-1]], path[::-1] if len(path) > 1 else [99], [0, 0]):
        with pytest.raises(binding.DovetailError) as ei:
            binding.dovetail_kv_commit(h, kv, bad, mode=1)
        assert ei.value.code == binding.EINVAL
        assert torch.equal(before_k, kv.k) and kv.committed_len == Lp
    n = binding.dovetail_kv_commit(h, kv, path, mode=1)
    torch.cuda.synchronize()
    # oracle: tree rows of the accepted nodes (pool_row - n_new), leading forwarded run
    keep_idx = _kept_pool_indices(ora)
    rows = [int(ora["pool_row"][keep_idx[i]]) for i in path]
    tree_rows = [r - 2 if r >= 0 else -1 for r in rows]
    kc, vc = gpu["k"].copy(), gpu["v"].copy()
    moved = oracle.kv_commit(_ocfg(cfg), kc, vc, case.capacity, Lp, tree_rows, 1)
    assert n == moved and kv.committed_len == Lp + moved
    from helpers import kv_np
    assert np.array_equal(kv_np(kv.k), kc) and np.array_equal(kv_np(kv.v), vc)
    # a second commit without a new step is refused
    with pytest.raises(binding.DovetailError):
        binding.dovetail_kv_commit(h, kv, path, mode=1)
    binding.dovetail_draft_destroy(h)

    # mode 0: step, discard, step again with the same inputs -> identical results
    h, kv, a = run_gpu(case)
    assert binding.dovetail_kv_commit(h, kv, path, mode=0) == 0
    kv.committed_len = case.L
    out = binding.dovetail_draft_step(h, case.feats, case.tokens, kv, case.tree)
    torch.cuda.synchronize()
    n2 = int(out["n_out"].item())
    assert np.array_equal(out["token_ids"][:n2].cpu().numpy(), a["token_ids"])
    assert np.array_equal(out["scores"][:n2].cpu().numpy(), a["scores"])
    binding.dovetail_draft_destroy(h)


def _ocfg(cfg):
    from helpers import ocfg
    return ocfg(cfg)


def _kept_pool_indices(ora):
    """Pool index of each emitted candidate: the top-gamma by (score desc, index asc), in pool order."""
    cum = ora["pool_cum"]
    order = np.lexsort((np.arange(len(cum)), -cum))
    return np.sort(order[:ora["n_out"]])


def test_error_paths():
    cfg = small_cfg(dtype=F32)
    case = make_case(cfg, n_new=1)
    h = binding.dovetail_draft_init(case.top, case.layers, cfg, max_rows=8, max_tree_slots=16, max_branch=4)
    kv = binding.KVCache(case.k.clone(), case.v.clone(), case.L)
    good = TreeSpec(2, (2, 2), (0, 0), 4)

    def code(fn):
        with pytest.raises(binding.DovetailError) as ei:
            fn()
        return ei.value.code

    step = lambda tree, kvc=kv, f=case.feats, t=case.tokens: binding.dovetail_draft_step(h, f, t, kvc, tree)
    assert code(lambda: step(TreeSpec(0, (), (), 1))) == binding.EINVAL                 # depth
    assert code(lambda: step(TreeSpec(2, (5, 2), (0, 0), 4))) == binding.EINVAL          # branch > max_branch
    assert code(lambda: step(TreeSpec(2, (2, 2), (0, 0), 0))) == binding.EINVAL          # gamma
    assert code(lambda: step(TreeSpec(4, (4, 4, 4, 4), (0, 0, 0, 0), 4))) == binding.EINVAL  # rows > max_rows
    assert code(lambda: step(TreeSpec(6, (2,) * 6, (0, 0, 0, 4, 4, 4), 4))) == binding.EINVAL  # > max_tree_slots
    many = torch.zeros((9, cfg.hidden), device="cuda")
    assert code(lambda: step(good, f=many, t=torch.zeros(9, dtype=torch.int32, device="cuda"))) == binding.EINVAL
    small = binding.KVCache(case.k.clone(), case.v.clone(), case.capacity - 1)
    assert code(lambda: step(good, kvc=small)) == binding.ECAPACITY
    assert small.committed_len == case.capacity - 1 and kv.committed_len == case.L    # nothing advanced
    assert "capacity" in binding.dovetail_last_error(h)
    assert code(lambda: binding.dovetail_kv_commit(h, kv, [0], mode=0)) == binding.EINVAL  # no step yet
    out = step(good)
    torch.cuda.synchronize()
    assert int(out["n_out"].item()) == 4 and kv.committed_len == case.L + 1
    assert binding.dovetail_last_launch_count(h) > 0
    assert binding.dovetail_forward_bytes(h, case.L) == cfg.forward_bytes(case.L)
    binding.dovetail_draft_status(h)  # a good step: OK
    # a token id outside [0, vocab): the step cannot see it (device memory); dovetail_draft_status reports it
    for bad_tok in (cfg.vocab, -1, 2 ** 30):
        kv.committed_len = case.L
        step(good, t=torch.tensor([bad_tok], dtype=torch.int32, device="cuda"))
        assert code(lambda: binding.dovetail_draft_status(h)) == binding.EINVAL
        assert "token id" in binding.dovetail_last_error(h)
        binding.dovetail_draft_status(h)  # the flag is cleared by the read
    # wrong dtypes never reach the raw-pointer ABI
    with pytest.raises(TypeError):
        step(good, f=case.feats.to(torch.bfloat16))
    with pytest.raises(TypeError):
        step(good, t=case.tokens.to(torch.int64))
    binding.dovetail_draft_destroy(h)
    # init-time validation
    bad = small_cfg(dtype=F32, head_dim=32, hidden=128)
    c2 = make_case(bad, n_new=1)
    with pytest.raises(binding.DovetailError) as ei:
        binding.dovetail_draft_init(c2.top, c2.layers, bad)
    assert ei.value.code == binding.EINVAL
    # token ids are packed into 24 bits of a candidate key (k_tree_level): larger vocabularies are refused, checked
    # before any weight is read
    from dataclasses import replace
    with pytest.raises(binding.DovetailError) as ei:
        binding.dovetail_draft_init(case.top, case.layers, replace(cfg, vocab=(1 << 24) - 1))
    assert ei.value.code == binding.EINVAL


def test_two_steps_chained_through_commit_mode1():
    """step -> kv_commit(mode 1) of the deepest accepted chain -> step again, against the oracle run on the
    oracle's own committed cache: the moved rows, their rotary positions and committed_len are what the second
    step's attention consumes (O9 then O2-O8)."""
    from helpers import kv_np
    from parity import compare
    cfg = small_cfg(dtype=BF16, tree=TreeSpec(3, (3, 2, 2), (0, 3, 3), 8))
    case = _boost(make_case(cfg, n_new=2, slack=40))
    h, kv, gpu = run_gpu(case)
    ora = run_oracle(case)
    assert np.array_equal(gpu["token_ids"], ora["token_ids"]) and np.array_equal(gpu["parents"], ora["parents"])
    leaf = int(np.argmax(gpu["depths"]))
    path = [leaf]
    while gpu["parents"][path[-1]] >= 0:
        path.append(int(gpu["parents"][path[-1]]))
    path = path[::-1]
    Lp = kv.committed_len
    moved = binding.dovetail_kv_commit(h, kv, path, mode=1)
    keep_idx = _kept_pool_indices(ora)
    tree_rows = [int(ora["pool_row"][keep_idx[i]]) - 2 if ora["pool_row"][keep_idx[i]] >= 0 else -1 for i in path]
    okc, ovc = ora["k"], ora["v"]
    assert oracle.kv_commit(_ocfg(cfg), okc, ovc, case.capacity, Lp, tree_rows, 1) == moved and moved >= 1
    L2 = Lp + moved
    assert kv.committed_len == L2
    # second step: the accepted tokens' successors with fresh (seeded) target features; both sides start from
    # their own committed cache
    import dataclasses
    from paper_2412_18934_b200 import synth
    feats2, tokens2 = synth.make_inputs(cfg, 3, device="cuda", seed=99)
    k2 = torch.from_numpy(okc.view(np.int16).copy()).view(torch.bfloat16).cuda()
    v2 = torch.from_numpy(ovc.view(np.int16).copy()).view(torch.bfloat16).cuda()
    case2 = dataclasses.replace(case, k=k2, v=v2, feats=feats2, tokens=tokens2, L=L2)
    ora2 = run_oracle(case2)
    rows2 = 3 + case.tree.tree_rows()
    P = case.tree.pool_size()
    hooks = dict(tap_logits=torch.zeros((rows2, cfg.vocab), device="cuda"), tap_hhat=torch.zeros((rows2, cfg.hidden), device="cuda"),
                 tap_pool_token=torch.zeros(P, dtype=torch.int32, device="cuda"), tap_pool_cum=torch.zeros(P, device="cuda"))
    binding.dovetail_hooks_set(h, **hooks)
    out = binding.dovetail_draft_step(h, feats2, tokens2, kv, case.tree)  # the GPU's own cache, as committed
    binding.dovetail_draft_status(h)
    n = int(out["n_out"].item())
    g2 = dict(token_ids=out["token_ids"][:n].cpu().numpy(), scores=out["scores"][:n].cpu().numpy(),
              parents=out["parents"][:n].cpu().numpy(), depths=out["depths"][:n].cpu().numpy(), n_out=n,
              logits=hooks["tap_logits"].cpu().numpy(), hhat=hooks["tap_hhat"].cpu().numpy(),
              pool_token=hooks["tap_pool_token"].cpu().numpy(), pool_cum=hooks["tap_pool_cum"].cpu().numpy(),
              k=kv_np(kv.k), v=kv_np(kv.v), forced=False, committed_len=kv.committed_len)
    s2 = compare(case2, g2, ora2)
    assert s2["same_tree"] and kv.committed_len == L2 + 3
    binding.dovetail_draft_destroy(h)


def test_trace_adds_up():
    """dovetail_trace_*: per-kind exclusive device times add up to at most the step (the launches keep their
    programmatic-dependent-launch overlap), every kind of the step is present, bytes = algorithmic bytes."""
    cfg = small_cfg(dtype=BF16)
    case = make_case(cfg, n_new=1)
    h = binding.dovetail_draft_init(case.top, case.layers, cfg)
    kv = binding.KVCache(case.k.clone(), case.v.clone(), case.L)
    binding.dovetail_trace_enable(h, True)
    out = binding.dovetail_draft_step(h, case.feats, case.tokens, kv, case.tree)
    torch.cuda.synchronize()
    t = binding.dovetail_trace_read(h)
    kinds = t["kinds"]
    n_launch = sum(k["launches"] for k in kinds.values())
    assert n_launch >= binding.dovetail_last_launch_count(h)  # a persistent launch covers several GEMVs
    assert t["step_us"] > 0
    assert sum(k["excl_us"] for k in kinds.values()) <= t["step_us"] * 1.0001
    for name in ("step_begin", "dgf_proj", "dgf_gate", "qkv", "tree_attention", "o_proj", "gate_up", "down", "lm_head", "tree_level"):
        assert kinds[name]["launches"] > 0 and kinds[name]["busy_us"] > 0, name
    wbytes = sum(k["bytes"] for n, k in kinds.items() if n != "tree_attention")
    assert wbytes == case.tree.depth * (cfg.forward_bytes(0) - (2 * cfg.n_layers + 1) * cfg.hidden * cfg.esize)  # all matrices; not the norm gains / gate bias
    binding.dovetail_trace_enable(h, False)
    binding.dovetail_draft_destroy(h)

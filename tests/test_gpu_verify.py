"""-m gpu: verification-side bookkeeping and the acceptance rule through the C ABI,
bit-exact against the oracle: on the trees real draft steps emit, with random target answers; then the whole round
step -> verify_plan -> verify_accept -> kv_commit(accepted_path) on device outputs."""
import numpy as np
import pytest
import torch

import oracle
from parity import make_case, run_gpu
from paper_2412_18934_b200 import binding
from paper_2412_18934_b200.configs import BF16, TreeSpec, paper_preset
from test_gpu_parity import _boost, small_cfg

pytestmark = pytest.mark.gpu

TREES = [TreeSpec(3, (3, 2, 2), (0, 3, 4), 9), TreeSpec(5, (2,) * 5, (0, 2, 2, 2, 2), 16), paper_preset(True),
         TreeSpec(2, (4, 1), (0, 0), 3), TreeSpec(1, (5,), (0,), 8)]


def _step(tree):
    cfg = small_cfg(dtype=BF16, tree=tree)
    case = _boost(make_case(cfg, n_new=2))
    h = binding.dovetail_draft_init(case.top, case.layers, cfg)
    kv = binding.KVCache(case.k.clone(), case.v.clone(), case.L)
    out = binding.dovetail_draft_step(h, case.feats, case.tokens, kv, tree)
    binding.dovetail_draft_status(h)
    return cfg, case, h, kv, out


@pytest.mark.parametrize("ti", range(len(TREES)))
def test_verify_plan_bit_exact(ti):
    tree = TREES[ti]
    cfg, case, h, kv, out = _step(tree)
    n = int(out["n_out"].item())
    g = tree.gamma
    plan = binding.dovetail_verify_plan(h, out, root_position=kv.committed_len - 1, max_depth=tree.depth)
    torch.cuda.synchronize()
    par, dep = out["parents"][:n].cpu().numpy(), out["depths"][:n].cpu().numpy()
    ora = oracle.verify_plan(par, dep, kv.committed_len - 1, tree.depth)
    m = plan["mask"].cpu().numpy()
    assert np.array_equal(m[:n + 1, :n + 1], ora["mask"]) and m[n + 1:].sum() == 0 and m[:, n + 1:].sum() == 0
    assert np.array_equal(plan["position_ids"][:n + 1].cpu().numpy(), ora["position_ids"])
    k = int(plan["n_paths"].item())
    assert k == ora["n_paths"]
    paths = plan["paths"].cpu().numpy()
    assert np.array_equal(paths[:k], ora["paths"]) and (paths[k:] == -1).all()
    assert g >= n
    binding.dovetail_draft_destroy(h)


@pytest.mark.parametrize("ti", range(len(TREES)))
@pytest.mark.parametrize("mode", [0, 1])
def test_verify_accept_bit_exact(ti, mode):
    tree = TREES[ti]
    cfg, case, h, kv, out = _step(tree)
    n, g, V = int(out["n_out"].item()), tree.gamma, cfg.vocab
    tok, par = out["token_ids"][:n].cpu().numpy(), out["parents"][:n].cpu().numpy()
    for seed in range(12):
        rng = np.random.default_rng(1000 * ti + seed)
        # the target's distributions: random, but with much mass on each row's children so that paths get accepted
        pf = rng.random((g + 1, V)).astype(np.float32) ** 8
        for row in range(n + 1):
            kids = [i for i in range(n) if par[i] == row - 1]
            for i in kids:
                pf[row, tok[i]] += np.float32(rng.random() * V / 40)
        pf /= pf.sum(1, keepdims=True)
        pf = pf.astype(np.float32)
        arg = pf.argmax(1).astype(np.int32)
        p_cand = np.zeros(g, np.float32)
        p_cand[:n] = pf[par + 1, tok]
        u = rng.random(g + 1).astype(np.float32)
        u_n = u.copy()  # the bonus uniform sits at index n_out
        ora = oracle.verify_accept(tok, par, mode, tgt_argmax=arg[:n + 1], p_cand=p_cand[:n], uniforms=u_n[:n + 1], p_full=pf[:n + 1])
        dev = lambda a: torch.from_numpy(a).cuda()
        res = binding.dovetail_verify_accept(h, out, mode, tree.depth, tgt_argmax=dev(arg) if mode == 0 else None,
                                             p_cand=dev(p_cand) if mode else None, uniforms=dev(u_n) if mode else None,
                                             p_full=dev(pf) if mode else None)
        torch.cuda.synchronize()
        na = int(res["n_acc"].item())
        assert na == ora["n_acc"], (seed, na, ora)
        assert np.array_equal(res["accepted_path"][:na].cpu().numpy(), ora["accepted_path"])
        assert int(res["bonus_token"].item()) == ora["bonus_token"]
    binding.dovetail_draft_destroy(h)


def test_verify_accept_large_ragged_vocabulary():
    """The bonus-token draw on a vocabulary that is neither small nor a multiple of 32 (50 003): several narrowing
    rounds of the inverse-CDF search, rejected children removed from the row, thresholds at both ends of the row,
    and a stopping row without any mass (a degenerate target answer: every child has probability 0 and is rejected,
    nothing is left to draw from, bonus token -1 as include/dovetail.h states). Bit-exact against the oracle.
    (A normalised row whose mass sits entirely on the node's children cannot end in -1: the remainder shrinks with
    every rejection and the last sibling is accepted with probability 1 -- both sides agree on that too.)"""
    tree = TreeSpec(3, (3, 2, 2), (0, 3, 4), 9)
    cfg = small_cfg(dtype=BF16, tree=tree, vocab=50003)
    case = _boost(make_case(cfg, n_new=1))
    h = binding.dovetail_draft_init(case.top, case.layers, cfg)
    kv = binding.KVCache(case.k.clone(), case.v.clone(), case.L)
    out = binding.dovetail_draft_step(h, case.feats, case.tokens, kv, tree)
    n, g, V = int(out["n_out"].item()), tree.gamma, cfg.vocab
    tok, par = out["token_ids"][:n].cpu().numpy(), out["parents"][:n].cpu().numpy()
    dev = lambda a: torch.from_numpy(a).cuda()
    roots = [i for i in range(n) if par[i] == -1]
    for seed in range(10):
        rng = np.random.default_rng(77 + seed)
        pf = rng.random((g + 1, V)).astype(np.float32) ** 6
        for i in range(n):
            pf[par[i] + 1, tok[i]] += np.float32(rng.random() * V / 30)
        pf = (pf / pf.sum(1, keepdims=True)).astype(np.float32)
        if seed >= 8:  # the root row carries no mass at all
            pf[0] = 0
        p_cand = np.zeros(g, np.float32)
        p_cand[:n] = pf[par + 1, tok]
        u = rng.random(g + 1).astype(np.float32)
        if seed in (3, 4):  # reject every child of the root: the bonus token comes from the root row
            u[roots] = np.float32(0.9999999)
        if seed == 3:
            u[n] = np.float32(0.0)
        if seed == 4:
            u[n] = np.float32(0.99999994)
        ora = oracle.verify_accept(tok, par, 1, tgt_argmax=None, p_cand=p_cand[:n], uniforms=u[:n + 1], p_full=pf[:n + 1])
        res = binding.dovetail_verify_accept(h, out, 1, tree.depth, p_cand=dev(p_cand), uniforms=dev(u), p_full=dev(pf))
        torch.cuda.synchronize()
        na = int(res["n_acc"].item())
        assert na == ora["n_acc"], (seed, na, ora)
        assert np.array_equal(res["accepted_path"][:na].cpu().numpy(), ora["accepted_path"])
        assert int(res["bonus_token"].item()) == ora["bonus_token"], seed
        if seed >= 8:
            assert na == 0 and ora["bonus_token"] == -1
    binding.dovetail_draft_destroy(h)


def test_round_trip_step_verify_commit():
    """One whole round on device outputs: step, verifier inputs, greedy acceptance against a target that agrees with
    the draft's best chain, kv_commit (mode 1) of the accepted path."""
    tree = TreeSpec(4, (3, 2, 2, 2), (0, 3, 3, 3), 10)
    cfg, case, h, kv, out = _step(tree)
    n = int(out["n_out"].item())
    tok, par, sc = out["token_ids"][:n].cpu().numpy(), out["parents"][:n].cpu().numpy(), out["scores"][:n].cpu().numpy()
    arg = np.full(tree.gamma + 1, -1, np.int32)
    for row in range(n + 1):  # the target prefers each row's best-scored child
        kids = [i for i in range(n) if par[i] == row - 1]
        if kids:
            arg[row] = tok[max(kids, key=lambda i: sc[i])]
    res = binding.dovetail_verify_accept(h, out, 0, tree.depth, tgt_argmax=torch.from_numpy(arg).cuda())
    torch.cuda.synchronize()
    na = int(res["n_acc"].item())
    path = res["accepted_path"][:na].cpu().numpy().tolist()
    assert na >= 1 and par[path[0]] == -1 and all(par[b] == a for a, b in zip(path, path[1:]))
    Lp = kv.committed_len
    moved = binding.dovetail_kv_commit(h, kv, path, mode=1)
    assert 1 <= moved <= na and kv.committed_len == Lp + moved
    # errors
    with pytest.raises(binding.DovetailError):
        binding.dovetail_verify_accept(h, out, 2, tree.depth, tgt_argmax=torch.from_numpy(arg).cuda())
    with pytest.raises(binding.DovetailError):
        binding.dovetail_verify_accept(h, out, 1, tree.depth, tgt_argmax=torch.from_numpy(arg).cuda())  # sampling inputs missing
    binding.dovetail_draft_destroy(h)

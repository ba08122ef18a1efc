"""Pins of the oracle's step logic (O2, O6-O9): chain tree = causal decoding
(P3), brute force over every token path (P6), structural invariants (P7),
level-0 batching (P8), commit (P9), and an independent re-simulation of the
bookkeeping from the dumped per-row log-probabilities. CPU only."""
import itertools

import numpy as np
import pytest
import torch

import oracle
from helpers import RefDraft, kv_np, np_to_f64, ocfg, oracle_step, oweights, tiny_cfg
from paper_2412_18934_b200 import synth
from paper_2412_18934_b200.configs import TreeSpec


def _setup(cfg, L, cap, n_new, seed=None):
    top, layers = synth.make_weights(cfg, seed=seed)
    # larger LM head / embedding spread so that the toy distributions are far from uniform
    top["lm_head"] = top["lm_head"] * 60
    top["embed"] = top["embed"] * 40
    k, v = synth.make_kv(cfg, cap, L, seed=seed)
    feats, tokens = synth.make_inputs(cfg, n_new, seed=seed)
    return top, layers, k, v, feats, tokens


def _ref_prefix(cfg, top, layers, k, v, L, feats, tokens):
    """Reference state after the level-0 rows; returns (ref, hhat of the last row)."""
    ref = RefDraft(cfg, top, layers)
    ref.preload(k, v, L)
    hh = ref.rows(feats, tokens, [L + i for i in range(feats.shape[0])])
    return ref, hh[-1]


def test_chain_tree_equals_greedy_causal_decoding():
    """P3: branch = beam = 1 is ordinary causal autoregression on (feature, token) pairs."""
    cfg = tiny_cfg()
    L, cap, n_new, D = 7, 24, 3, 5
    top, layers, k, v, feats, tokens = _setup(cfg, L, cap, n_new)
    tree = TreeSpec(D, (1,) * D, (0,) + (1,) * (D - 1), D)
    res = oracle_step(cfg, top, layers, k, v, cap, L, feats, tokens, tree)
    ref, h = _ref_prefix(cfg, top, layers, k, v, L, feats, tokens)
    toks, cums, cum = [], [], 0.0
    for l in range(D):
        lp = ref.logp(h)
        t = int(torch.argmax(lp))
        cum += float(lp[t])
        toks.append(t)
        cums.append(cum)
        if l < D - 1:
            h = ref.rows(h[None], torch.tensor([t]), [L + n_new + l])[0]
    assert res["token_ids"].tolist() == toks
    assert res["parents"].tolist() == [-1] + list(range(D - 1))
    assert res["depths"].tolist() == list(range(1, D + 1))
    np.testing.assert_allclose(res["scores"], cums, rtol=1e-5, atol=1e-6)
    # the tree rows landed in cache rows L' .. L'+D-2 with rotary positions L' + l - 1
    assert res["row_slot"].tolist() == list(range(L, L + n_new + D - 1))
    assert res["row_pos"].tolist() == list(range(L, L + n_new + D - 1))


@pytest.mark.parametrize("seed", [1, 2])
def test_full_tree_equals_brute_force_over_all_paths(seed):
    """P6: with branch = V and beam = all, the pool is every token path of length <= D; its
    cumulative log-probs must equal the chain log-probs of an independent causal evaluation
    and the top-gamma must be the global top-gamma."""
    cfg = tiny_cfg(vocab=5, n_layers=1)
    V, D, gamma = cfg.vocab, 3, 9
    L, cap, n_new = 4, 4 + 2 + V + V * V + 2, 2
    top, layers, k, v, feats, tokens = _setup(cfg, L, cap, n_new, seed=seed)
    tree = TreeSpec(D, (V,) * D, (0,) * D, gamma)
    res = oracle_step(cfg, top, layers, k, v, cap, L, feats, tokens, tree)
    assert len(res["pool_token"]) == V + V * V + V ** 3

    ref0, h0 = _ref_prefix(cfg, top, layers, k, v, L, feats, tokens)
    brute = {}

    def rec(ref, h, path, cum):
        lp = ref.logp(h)
        for t in range(V):
            p = path + (t,)
            brute[p] = cum + float(lp[t])
            if len(p) < D:
                r2 = ref.fork()
                h2 = r2.rows(h[None], torch.tensor([t]), [L + n_new + len(p) - 1])[0]
                rec(r2, h2, p, brute[p])

    rec(ref0, h0, (), 0.0)
    # every pool node's path and score
    P = len(res["pool_token"])
    paths = []
    for i in range(P):
        p, a = [], i
        while a >= 0:
            p.append(int(res["pool_token"][a]))
            a = int(res["pool_parent"][a])
        paths.append(tuple(reversed(p)))
    assert len(set(paths)) == P == len(brute)
    for i, p in enumerate(paths):
        assert abs(res["pool_cum"][i] - brute[p]) < 1e-5, (p, res["pool_cum"][i], brute[p])
        assert res["pool_depth"][i] == len(p)
    best = sorted(brute.items(), key=lambda kv: -kv[1])[:gamma]
    got = set()
    for i in range(res["n_out"]):
        p, a = [], i
        while a >= 0:
            p.append(int(res["token_ids"][a]))
            a = int(res["parents"][a])
        got.add(tuple(reversed(p)))
    assert got == {p for p, _ in best}


def _resimulate(res, tree: TreeSpec, n_new: int):
    """Independent restatement of O6-O8 on the step's dumped per-row logits, with numpy sorts."""
    def logp_row(r):
        z = res["row_logits"][r]
        return z - (z.max() + np.log(np.exp(z - z.max()).sum()))

    def top(lp, b):
        return np.argsort(-lp, kind="stable")[:b]

    pool = []  # (token, parent, depth, cum)
    lp = logp_row(n_new - 1)
    for t in top(lp, tree.branch[0]):
        pool.append((int(t), -1, 1, float(lp[t])))
    level, row = list(range(len(pool))), n_new
    for l in range(1, tree.depth):
        order = sorted(level, key=lambda i: (-pool[i][3], i))
        want = tree.beam[l] if 0 < tree.beam[l] < len(order) else len(order)
        nxt = []
        for i in order[:want]:
            lp = logp_row(row)
            row += 1
            for t in top(lp, tree.branch[l]):
                pool.append((int(t), i, l + 1, pool[i][3] + float(lp[t])))
                nxt.append(len(pool) - 1)
        level = nxt
    sel = sorted(sorted(range(len(pool)), key=lambda i: (-pool[i][3], i))[:tree.gamma])
    new = {p: j for j, p in enumerate(sel)}
    return pool, [pool[i][0] for i in sel], [new.get(pool[i][1], -1) for i in sel], [pool[i][3] for i in sel]


@pytest.mark.parametrize("tree", [TreeSpec(3, (2, 2, 2), (0, 0, 0), 14), TreeSpec(4, (3, 2, 2, 2), (0, 0, 0, 0), 10),
                                  TreeSpec(5, (2,) * 5, (0, 2, 2, 2, 2), 16), TreeSpec(4, (4, 3, 2, 1), (0, 3, 5, 2), 7),
                                  TreeSpec(1, (3,), (0,), 2), TreeSpec(3, (2, 2, 2), (0, 1, 1), 100)])
def test_bookkeeping_resimulation_and_invariants(tree):
    cfg = tiny_cfg(vocab=40)
    n_new, L = 2, 5
    cap = L + n_new + tree.tree_rows()
    top, layers, k, v, feats, tokens = _setup(cfg, L, cap, n_new)
    res = oracle_step(cfg, top, layers, k, v, cap, L, feats, tokens, tree)
    pool, ids, parents, scores = _resimulate(res, tree, n_new)
    assert res["pool_token"].tolist() == [p[0] for p in pool]
    assert res["pool_parent"].tolist() == [p[1] for p in pool]
    assert res["pool_depth"].tolist() == [p[2] for p in pool]
    np.testing.assert_allclose(res["pool_cum"], [p[3] for p in pool], rtol=1e-12, atol=1e-12)
    assert res["token_ids"].tolist() == ids and res["parents"].tolist() == parents
    np.testing.assert_allclose(res["scores"], scores, rtol=1e-12, atol=1e-12)
    # P7 structural invariants
    P = len(pool)
    assert P == tree.pool_size() and res["n_out"] == min(tree.gamma, P)
    assert res["total_rows"] == n_new + tree.tree_rows()
    for i in range(res["n_out"]):
        p = res["parents"][i]
        assert -1 <= p < i
        assert res["depths"][i] == (1 if p < 0 else res["depths"][p] + 1)
        if p >= 0:
            assert res["scores"][i] <= res["scores"][p]
    unsel = sorted(set(range(P)) - {i for i in range(P) if any(
        res["pool_token"][i] == res["token_ids"][j] and abs(res["pool_cum"][i] - res["scores"][j]) == 0
        for j in range(res["n_out"]))})
    if unsel:
        assert max(res["pool_cum"][i] for i in unsel) <= res["scores"].min() + 1e-15
    # replay entry reproduces the step's bookkeeping from the same per-row lists
    rows = [n_new - 1] + list(range(n_new, res["total_rows"]))
    mb = max(tree.branch[:tree.depth])
    ct = np.zeros((len(rows), mb), np.int32)
    cl = np.zeros((len(rows), mb), np.float64)
    lvl = [0] + [l for l, m in enumerate(tree.rows_per_level(n_new)) if l >= 1 for _ in range(m)]
    for j, r in enumerate(rows):
        lp = oracle.log_softmax(res["row_logits"][r])
        idx = oracle.topk(lp, tree.branch[lvl[j]])
        ct[j, :len(idx)] = idx
        cl[j, :len(idx)] = lp[idx]
    rp = oracle.tree_replay(tree.depth, tree.branch, tree.beam, tree.gamma, ct, cl)
    assert rp["token_ids"].tolist() == ids and rp["parents"].tolist() == parents
    np.testing.assert_array_equal(rp["pool_cum"], res["pool_cum"])


def test_exact_ties_break_by_token_id_then_pool_index():
    """A7 on the integer path: equal log-probs everywhere."""
    D = 3
    ct = np.tile(np.array([[3, 5]], np.int32), (1 + 2 + 2, 1))
    cl = np.full((5, 2), -1.0)
    r = oracle.tree_replay(D, (2, 2, 2), (0, 2, 2), 4, ct, cl)
    # pool: [3,5 | (3,3),(3,5),(5,3),(5,5) | ...]; top-4 by (cum desc, index asc) = 2 level-1 + first 2 level-2
    assert r["token_ids"].tolist() == [3, 5, 3, 5]
    assert r["parents"].tolist() == [-1, -1, 0, 0]


def test_level0_rows_equal_successive_single_row_steps():
    """P8: feeding n_new rows at once == feeding them one step at a time."""
    cfg = tiny_cfg()
    L, cap, n_new = 6, 20, 3
    top, layers, k, v, feats, tokens = _setup(cfg, L, cap, n_new)
    tree = TreeSpec(2, (2, 2), (0, 0), 6)
    a = oracle_step(cfg, top, layers, k, v, cap, L, feats, tokens, tree)
    kc, vc = kv_np(k), kv_np(v)
    ow = oweights(top, layers)
    for i in range(n_new):
        b = oracle.step(ocfg(cfg), ow, kc, vc, cap, L + i, feats[i:i + 1].numpy(), tokens[i:i + 1].numpy(),
                        tree.depth, tree.branch, tree.beam, tree.gamma)
    np.testing.assert_array_equal(a["k"][:, :, :L + n_new], kc[:, :, :L + n_new])
    np.testing.assert_array_equal(a["v"][:, :, :L + n_new], vc[:, :, :L + n_new])
    assert a["token_ids"].tolist() == b["token_ids"].tolist()
    np.testing.assert_allclose(a["scores"], b["scores"], rtol=1e-12)
    np.testing.assert_allclose(a["row_hhat"][n_new - 1], b["row_hhat"][0], rtol=1e-12)


def test_kv_commit_modes():
    """P9: mode 0 leaves the step repeatable; mode 1 gathers the accepted rows."""
    cfg = tiny_cfg()
    L, cap, n_new = 4, 24, 1
    top, layers, k, v, feats, tokens = _setup(cfg, L, cap, n_new)
    tree = TreeSpec(4, (2, 2, 2, 2), (0, 2, 2, 2), 8)
    a = oracle_step(cfg, top, layers, k, v, cap, L, feats, tokens, tree)
    kc, vc = a["k"].copy(), a["v"].copy()
    assert oracle.kv_commit(ocfg(cfg), kc, vc, cap, L + n_new, [0, 1], 0) == 0
    np.testing.assert_array_equal(kc, a["k"])
    # re-running the same step over the same cache state gives the same outputs (tree rows are dead)
    kc2, vc2 = a["k"].copy(), a["v"].copy()
    b = oracle.step(ocfg(cfg), oweights(top, layers), kc2, vc2, cap, L, feats.numpy(), tokens.numpy(),
                    tree.depth, tree.branch, tree.beam, tree.gamma)
    assert a["token_ids"].tolist() == b["token_ids"].tolist()
    np.testing.assert_array_equal(a["scores"], b["scores"])
    # mode 1: take a deepest root->leaf path of forwarded nodes
    rows = a["pool_row"]
    leaf = max((i for i in range(len(rows)) if rows[i] >= 0), key=lambda i: a["pool_depth"][i])
    path = []
    while leaf >= 0:
        path.append(leaf)
        leaf = int(a["pool_parent"][leaf])
    path.reverse()
    tree_rows = [int(rows[i]) - n_new for i in path]
    Lp = L + n_new
    moved = oracle.kv_commit(ocfg(cfg), kc, vc, cap, Lp, tree_rows, 1)
    assert moved == len(path)
    for i, tr in enumerate(tree_rows):
        np.testing.assert_array_equal(kc[:, :, Lp + i], a["k"][:, :, Lp + tr])
        np.testing.assert_array_equal(vc[:, :, Lp + i], a["v"][:, :, Lp + tr])
    # a trailing node without K/V stops the gather
    assert oracle.kv_commit(ocfg(cfg), a["k"].copy(), a["v"].copy(), cap, Lp, tree_rows[:1] + [-1], 1) == 1


def test_bad_arguments_are_rejected():
    cfg = tiny_cfg()
    top, layers, k, v, feats, tokens = _setup(cfg, 2, 4, 1)
    with pytest.raises(ValueError):  # tree rows do not fit the cache
        oracle_step(cfg, top, layers, k, v, 4, 2, feats, tokens, TreeSpec(3, (2, 2, 2), (0, 0, 0), 4))

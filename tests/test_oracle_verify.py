"""Pins of the oracle's verification-side steps O10 / O11: verifier inputs against an independent
closure computation, greedy acceptance against brute force over all root-to-node paths, and the speculative-sampling
rule against the identity that the emitted token follows the target's distribution exactly. CPU only."""
import itertools

import numpy as np
import pytest

import oracle


def random_tree(rng, n, max_children=3):
    """Token tree in pool order: parents precede children, siblings contiguous in rank order, distinct sibling tokens."""
    parents, depths, tokens = [], [], []
    frontier = [(-1, 0)]
    while len(parents) < n and frontier:
        par, dep = frontier.pop(0)
        k = int(rng.integers(1, max_children + 1))
        toks = rng.choice(50, size=k, replace=False)
        for t in toks:
            if len(parents) >= n:
                break
            parents.append(par)
            depths.append(dep + 1)
            tokens.append(int(t))
            frontier.append((len(parents) - 1, dep + 1))
    return np.array(tokens, np.int32), np.array(parents, np.int32), np.array(depths, np.int32)


@pytest.mark.parametrize("seed", range(8))
def test_verify_plan_matches_closure_and_chain_properties(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(1, 25))
    tokens, parents, depths = random_tree(rng, n)
    D = int(depths.max())
    r = oracle.verify_plan(parents, depths, 100, D)
    # ancestor-or-self relation as the reflexive-transitive closure of the parent relation, by matrix powers
    R = n + 1
    A = np.eye(R, dtype=np.int64)
    for i, p in enumerate(parents):
        A[i + 1, p + 1] = 1  # row -> its parent's row (root = row 0)
    C = np.linalg.matrix_power(A, R) > 0
    assert np.array_equal(r["mask"].astype(bool), C)
    # depth = number of proper ancestors; positions follow
    assert np.array_equal(r["position_ids"], 100 + (C.sum(1) - 1))
    # paths: one per leaf, in candidate order, each a root -> leaf chain
    leaves = [i for i in range(n) if i not in set(parents.tolist())]
    assert r["n_paths"] == len(leaves)
    for row, leaf in zip(r["paths"], leaves):
        chain = [int(x) for x in row if x >= 0]
        assert chain[-1] == leaf and parents[chain[0]] == -1
        assert all(parents[b] == a for a, b in zip(chain, chain[1:]))
        assert all(x == -1 for x in row[len(chain):])


@pytest.mark.parametrize("seed", range(10))
def test_greedy_acceptance_is_the_longest_argmax_consistent_path(seed):
    rng = np.random.default_rng(100 + seed)
    n = int(rng.integers(1, 20))
    tokens, parents, depths = random_tree(rng, n)
    # target argmax per verifier row: often one of the row's children, so that paths get accepted
    arg = np.zeros(n + 1, np.int32)
    for row in range(n + 1):
        kids = [i for i in range(n) if parents[i] == row - 1]
        arg[row] = tokens[rng.choice(kids)] if kids and rng.random() < 0.7 else 99
    got = oracle.verify_accept(tokens, parents, 0, tgt_argmax=arg)
    # brute force: every root-to-node path; valid iff each node's token is the argmax at its parent's row
    best = []
    for i in range(n):
        chain, a = [], i
        while a >= 0:
            chain.append(a)
            a = parents[a]
        chain = chain[::-1]
        if all(tokens[x] == arg[parents[x] + 1] for x in chain) and len(chain) > len(best):
            best = chain
    assert got["accepted_path"].tolist() == best
    assert got["bonus_token"] == arg[(best[-1] if best else -1) + 1]


def _threshold(f, lo=0.0, hi=1.0, iters=60):
    """Largest u with f(u) True, f monotone (True below the threshold)."""
    for _ in range(iters):
        mid = 0.5 * (lo + hi)
        if f(np.float32(mid)):
            lo = mid
        else:
            hi = mid
    return lo


def test_sampling_rule_emits_the_target_distribution_on_a_three_token_vocabulary():
    """Root with two children (tokens 0 and 1); p = target distribution at the root. The acceptance regions in the
    uniforms are intervals; their lengths, found by bisection on the oracle's decisions, give the exact emission
    probabilities: P(first emitted token = x) must be p(x) for every x (the speculative-sampling identity)."""
    p = np.array([0.5, 0.3, 0.2], np.float32)
    tokens, parents = np.array([0, 1], np.int32), np.array([-1, -1], np.int32)
    p_full = np.tile(p, (3, 1))
    p_cand = np.array([p[0], p[1]], np.float32)

    def run(u0, u1, ub):
        return oracle.verify_accept(tokens, parents, 1, p_cand=p_cand, uniforms=np.array([u0, u1, ub], np.float32), p_full=p_full)

    t0 = _threshold(lambda u: run(u, 0.999, 0.5)["accepted_path"].tolist() == [0])           # child 0 accepted
    t1 = _threshold(lambda u: run(0.999, u, 0.5)["accepted_path"].tolist() == [1])           # child 1 after rejecting 0
    assert run(0.999, 0.999, 0.3)["n_acc"] == 0 and run(0.999, 0.999, 0.3)["bonus_token"] == 2  # only token 2 is left
    emit = np.array([t0, (1 - t0) * t1, (1 - t0) * (1 - t1)])
    np.testing.assert_allclose(emit, p, atol=1e-6)
    # one child only (token 1): the bonus token is drawn from the residual {0: .5, 2: .2}
    tokens1, parents1 = np.array([1], np.int32), np.array([-1], np.int32)
    run1 = lambda u0, ub: oracle.verify_accept(tokens1, parents1, 1, p_cand=np.array([p[1]], np.float32),
                                                 uniforms=np.array([u0, ub], np.float32), p_full=np.tile(p, (2, 1)))
    a = _threshold(lambda u: run1(u, 0.5)["n_acc"] == 1)
    b = _threshold(lambda u: run1(0.999, u)["bonus_token"] == 0)
    np.testing.assert_allclose([a, (1 - a) * b, (1 - a) * (1 - b)], [p[1], p[0], p[2]], atol=1e-6)
    # after an accepted child the bonus token comes from the child's own row, nothing removed
    pf = np.stack([p, np.array([0.1, 0.1, 0.8], np.float32)])
    r = oracle.verify_accept(tokens1, parents1, 1, p_cand=np.array([p[1]], np.float32), uniforms=np.array([0.0, 0.15], np.float32), p_full=pf)
    assert r["accepted_path"].tolist() == [0] and r["bonus_token"] == 1  # cdf .1, .2, 1.0: u = .15 -> token 1


def test_sampling_decisions_are_strict_fp32_compares_and_edge_cases():
    tokens, parents = np.array([4], np.int32), np.array([-1], np.int32)
    pf = np.zeros((2, 8), np.float32)
    pf[0, 4], pf[0, 6] = 0.25, 0.75
    pf[1, 1] = 1.0
    acc = lambda u: oracle.verify_accept(tokens, parents, 1, p_cand=np.array([0.25], np.float32),
                                         uniforms=np.array([u, 0.5], np.float32), p_full=pf)
    assert acc(np.nextafter(np.float32(0.25), np.float32(0))).get("n_acc") == 1
    assert acc(np.float32(0.25))["n_acc"] == 0 and acc(np.float32(0.25))["bonus_token"] == 6  # u * 1 < p is strict
    # all of the target's mass on the rejected child: nothing left to draw
    pf2 = np.zeros((2, 8), np.float32)
    pf2[0, 4] = 1.0
    r = oracle.verify_accept(tokens, parents, 1, p_cand=np.array([0.5], np.float32), uniforms=np.array([0.9, 0.5], np.float32), p_full=pf2)
    assert r["n_acc"] == 0 and r["bonus_token"] == -1
    # no candidates at all: the bonus token comes from the root's row
    r = oracle.verify_accept(np.zeros(0, np.int32), np.zeros(0, np.int32), 0, tgt_argmax=np.array([7], np.int32))
    assert r["n_acc"] == 0 and r["bonus_token"] == 7

"""-m gpu: the CUDA draft step (through the C ABI) against the fp64 oracle, element by
element on the same seeded inputs. Small shapes span several tiles and ragged tails
(rows per CTA, K not a multiple of 256 units, prefix not a multiple of the attention
stage); the BASELINE.json configs run at full size."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from parity import compare, make_case, run_both, run_gpu, run_oracle
from paper_2412_18934_b200 import binding
from paper_2412_18934_b200.configs import BF16, CONFIGS, F32, DraftConfig, TreeSpec, c4_sweep, paper_preset

pytestmark = pytest.mark.gpu


def small_cfg(**kw) -> DraftConfig:
    base = dict(name="small", hidden=192, n_q_heads=4, n_kv_heads=2, head_dim=64, n_layers=2, ffn=344,
                vocab=1000, dtype=F32, prefix=70, feat_scale=1.0, rope_theta=1e4,
                tree=TreeSpec(3, (3, 2, 2), (0, 4, 5), 9), seed=11)
    base.update(kw)
    return DraftConfig(**base)


def _boost(case, lm=40.0, emb=20.0):
    """Spread the toy distributions so that the top-k decisions are far from ties."""
    if case.top["lm_head"].dtype in (torch.int8, torch.float8_e4m3fn):  # 8-bit weights: the per-row scales carry the magnitude
        case.top["lm_head_s"] = case.top["lm_head_s"] * lm
    else:
        case.top["lm_head"] = (case.top["lm_head"].float() * lm).to(case.top["lm_head"].dtype)
    case.top["embed"] = (case.top["embed"].float() * emb).to(case.top["embed"].dtype)
    return case


def _run(case, **kw):
    """Free-running step and teacher-forced step against the oracle (parity.run_both): every row of both
    runs element by element; discrete outputs identical unless the oracle's margin AT the differing decision
    is below tolerance."""
    s, gpu, ora = run_both(case, **kw)
    return s, gpu, ora


@pytest.mark.parametrize("dtype", [F32, BF16])
@pytest.mark.parametrize("variant", ["base", "mha_dh128", "mqa", "no_proj", "fusion_linear", "no_first_norm_final_norm", "n_new5",
                                     "no_prefix", "long_prefix", "wide", "very_wide", "n_new33", "max_branch", "tiny_vocab",
                                     "prefix3100_three_clusters", "prefix3100_three_clusters_n_new40"])
def test_step_parity_small(dtype, variant):
    kw, n_new, prefix = dict(dtype=dtype), 1, None
    if variant == "mha_dh128":
        kw.update(hidden=256, n_q_heads=2, n_kv_heads=2, head_dim=128)
    elif variant == "mqa":
        kw.update(n_q_heads=4, n_kv_heads=1)
    elif variant == "no_proj":
        kw.update(dgf_proj=0)
    elif variant == "fusion_linear":  # the EAGLE-2 fusion DGF replaces
        kw.update(dgf_proj=0, fusion=1)
    elif variant == "no_first_norm_final_norm":
        kw.update(first_layer_input_norm=0, final_norm=1)
    elif variant == "n_new5":
        n_new = 5
    elif variant == "no_prefix":
        prefix = 0
    elif variant == "long_prefix":
        prefix, n_new = 333, 2
    elif variant == "wide":  # rows per level 1, 6, 12: several m-tiles in every GEMV, query tiles in attention
        kw.update(tree=TreeSpec(3, (6, 3, 2), (0, 0, 12), 20))
    elif variant == "very_wide":  # 20 rows in one level: the GEMVs run in row chunks of 16 + 4
        kw.update(tree=TreeSpec(2, (20, 2), (0, 20), 24))
    elif variant == "n_new33":  # level 0 of 33 rows: GEMV row chunks 16 + 16 + 1, several attention query passes
        n_new = 33
    elif variant == "max_branch":  # 32 children of the root, all forwarded: b = max_branch, a 32-row level
        kw.update(tree=TreeSpec(2, (32, 1), (0, 32), 40))
    elif variant == "prefix3100_three_clusters":  # 49 blocks of 64 positions: 24 chunks per kv-head = 3 clusters of 8, merged across groups
        prefix, n_new = 3100, 2
    elif variant == "prefix3100_three_clusters_n_new40":  # 80 query vectors per kv-head: more than one staging round (62) of that merge
        prefix, n_new = 3100, 40
    elif variant == "tiny_vocab":  # fewer vocabulary rows than SMs: one row per LM-head CTA, per-CTA lists shorter than b
        kw.update(vocab=120, tree=TreeSpec(3, (8, 4, 2), (0, 5, 6), 20))
    case = _boost(make_case(small_cfg(**kw), n_new=n_new, prefix=prefix))
    s, gpu, ora = _run(case)
    assert s["same_tree"]  # forced run: always; the free run's tree may differ only by a logged local tie
    assert s["free"]["same_tree"] or s["free"]["tie"] is not None
    if dtype == F32:
        assert s["logit_max_abs_err"] < 1e-4


def test_config_c1_tiny_fp32():
    """BASELINE.json configs[0]: hidden 256, 4 x 64, 2 layers, FFN 688, vocab 1024, prefix 64, 14-token tree."""
    cfg = CONFIGS["c1"]
    case = make_case(cfg, n_new=1)
    s, gpu, ora = _run(case, tight=True)
    assert gpu["n_out"] == 14
    assert s["logit_max_abs_err"] < 1e-4


def test_paper_preset_tree_small_model():
    """PAPER.md:184 server setting: width 10, depth 7, 16 candidates (on a small model)."""
    cfg = small_cfg(dtype=BF16, tree=paper_preset(True))
    case = _boost(make_case(cfg, n_new=3))
    s, gpu, ora = _run(case)
    assert gpu["n_out"] == 16


def test_paper_preset_tree_7b_shape_full_size():
    """The tree the paper itself runs (width 10, depth 7, 16 candidates) on the 7B-shaped draft of
    BASELINE.json configs[1]: six levels of 10 rows on the tcgen05 GEMV, a pool of 610 candidates. Teacher-forced: every level from the oracle's state, every row at the stated
    and the observed-accuracy bounds, every top-10 decision checked locally. A free-running comparison is not
    meaningful on this random-weight model at this depth, and the test shows why instead of assuming it: the oracle's
    OWN candidates change under a 1e-6 relative perturbation of the input features (a bf16 ulp is 4e-3)."""
    from parity import oracle_sensitivity
    cfg = replace(CONFIGS["c2"], name="c2_paper_tree", tree=paper_preset(True))
    case = make_case(cfg, n_new=1)
    ora = run_oracle(case)
    h, kv, gpu = run_gpu(case, force=ora)
    binding.dovetail_draft_destroy(h)
    s = compare(case, gpu, ora, tight=True)
    assert s["same_tree"] and gpu["n_out"] == 16 and gpu["umma_launches"] > 0
    sens = oracle_sensitivity(case, ora)
    assert sens.first_changed is not None, "the oracle is stable here: compare the free run as well"
    # the free run still has to produce a well-formed tree
    h, kv, free = run_gpu(case)
    binding.dovetail_draft_destroy(h)
    assert free["n_out"] == 16 and (free["parents"] < np.arange(16)).all() and (free["parents"] >= -1).all()
    assert np.array_equal(free["depths"], np.where(free["parents"] < 0, 1, free["depths"][np.maximum(free["parents"], 0)] + 1))
    assert (np.diff(free["scores"][free["parents"] >= 0]) <= 1e30).all() and (free["scores"] <= 0).all()


@pytest.mark.parametrize("variant", ["f32", "bf16", "bf16_wide_tcgen05", "bf16_b32"])
def test_lm_head_merge_exact_ties(variant):
    """Every LM-head row appears twice (token v and token v + V / 2 share their weights), in different CTAs of
    the LM head: every logit is an exact two-way tie, so every top-b list, the merge of the per-CTA lists in
    k_tree_level, every frontier and the final top-gamma are decided by the tie rule (smaller token id / smaller
    pool index first, the oracle's stable order). The tree must be IDENTICAL to the oracle's: no tie excuse."""
    kw = dict(dtype=F32 if variant == "f32" else BF16, tree=TreeSpec(3, (8, 4, 4), (0, 6, 10), 30))
    if variant == "bf16_b32":  # 32 children per row: both tail batches of the merge, 12 rows per level
        kw.update(tree=TreeSpec(3, (32, 32, 4), (0, 12, 12), 64))
    case = _boost(make_case(small_cfg(**kw), n_new=2))
    lm = case.top["lm_head"]
    V = lm.shape[0]
    lm[V // 2:] = lm[:V // 2]
    ora = run_oracle(case)
    h, kv, gpu = run_gpu(case)
    binding.dovetail_draft_destroy(h)
    if variant == "bf16_wide_tcgen05":
        assert gpu["umma_launches"] > 0
    for key in ("token_ids", "parents", "depths"):
        assert np.array_equal(gpu[key], ora[key]), key
    tok = ora["token_ids"]
    assert ((tok[:, None] % (V // 2)) == (tok[None, :] % (V // 2))).sum() > len(tok)  # tied pairs were emitted
    np.testing.assert_allclose(gpu["scores"], ora["scores"], rtol=2e-2, atol=1e-2)


def test_determinism_run_to_run():
    cfg = small_cfg(dtype=BF16)
    case = _boost(make_case(cfg, n_new=2))
    _, _, a = run_gpu(case)
    _, _, b = run_gpu(case)
    for key in ("token_ids", "scores", "parents", "hhat", "logits", "k", "v"):
        assert np.array_equal(a[key], b[key]), key


@pytest.mark.parametrize("name", ["c2", "c3", "c5"])
def test_full_size_configs(name):
    """BASELINE.json configs[1], [2] (headline) and [4] at full size, in the launch
    configuration bench.py times. The oracle runs the whole step in fp64 on the host."""
    cfg = CONFIGS[name]
    case = make_case(cfg, n_new=1)
    s, gpu, ora = _run(case, tight=True)
    assert gpu["n_out"] == min(cfg.tree.gamma, cfg.tree.pool_size())
    assert s["free"]["same_tree"], f"free-running tree differs from the oracle's: {s['free']['tie']}"


@pytest.mark.parametrize("name", ["c4_l1_g32", "c4_l1_m8", "c4_l1_m16", "c4_l1_m32"])
def test_c4_sweep_points(name):
    """BASELINE.json configs[3] at full K (13B shape, prefix 2048): one step-level point (4 rows per level)
    and the forward-level points with 8, 16 and 32 rows in one level."""
    cfg = [c for c in c4_sweep() if c.name == name][0]
    case = make_case(cfg, n_new=1)
    s, gpu, ora = _run(case, tight=True)
    assert gpu["n_out"] == min(cfg.tree.gamma, cfg.tree.pool_size())
    assert s["free"]["same_tree"] or s["free"]["tie"] is not None


@pytest.mark.parametrize("name", ["depth_eagle2_l1", "depth_dgf_l1", "depth_dgf_l6"])
def test_depth_sweep_ends(name):
    """The ablation's shape (Table 6) at full size: the EAGLE-2 baseline (concat + Linear, one
    block) and DGF with 1 and 6 blocks on the 7B-shaped draft."""
    from paper_2412_18934_b200.configs import depth_sweep
    cfg = [c for c in depth_sweep() if c.name == name][0]
    case = make_case(cfg, n_new=1)
    s, gpu, ora = _run(case, tight=True)
    assert gpu["n_out"] == 16
    assert s["free"]["same_tree"] or s["free"]["tie"] is not None


@pytest.mark.parametrize("variant", ["base", "mha_dh128", "mqa", "no_proj", "fusion_linear", "n_new5", "wide", "very_wide", "max_branch",
                                     "n_new33"])
def test_step_parity_small_int8(variant):
    """int8 weight matrices with per-row scales against the oracle on the dequantised
    values; the same shapes as the bf16 cases (inner dimensions multiples of 32)."""
    kw, n_new = dict(dtype=BF16, wquant=1, ffn=352), 1
    if variant == "mha_dh128":
        kw.update(hidden=256, n_q_heads=2, n_kv_heads=2, head_dim=128)
    elif variant == "mqa":
        kw.update(n_q_heads=4, n_kv_heads=1)
    elif variant == "no_proj":
        kw.update(dgf_proj=0)
    elif variant == "fusion_linear":
        kw.update(dgf_proj=0, fusion=1)
    elif variant == "n_new5":
        n_new = 5
    elif variant == "wide":
        kw.update(tree=TreeSpec(3, (6, 3, 2), (0, 0, 12), 20))
    elif variant == "very_wide":
        kw.update(tree=TreeSpec(2, (20, 2), (0, 20), 24))
    elif variant == "max_branch":
        kw.update(tree=TreeSpec(2, (32, 1), (0, 32), 40))
    elif variant == "n_new33":
        n_new = 33
    case = _boost(make_case(small_cfg(**kw), n_new=n_new))
    s, gpu, ora = _run(case)
    assert s["same_tree"]
    assert s["free"]["same_tree"] or s["free"]["tie"] is not None


@pytest.mark.parametrize("name", ["c2_llama2_7b_int8", "c3_llama2_13b_int8", "c5_llama3_8b_int8"])
def test_full_size_configs_int8(name):
    """The 7B / 13B / Llama-3-8B shaped workloads with int8 weights at full size."""
    from paper_2412_18934_b200.configs import int8_variants
    cfg = [c for c in int8_variants() if c.name == name][0]
    case = make_case(cfg, n_new=1)
    s, gpu, ora = _run(case, tight=True)
    assert gpu["n_out"] == min(cfg.tree.gamma, cfg.tree.pool_size())
    assert s["free"]["same_tree"] or s["free"]["tie"] is not None


@pytest.mark.parametrize("variant", ["base", "mha_dh128", "no_proj", "fusion_linear", "n_new5", "wide", "max_branch"])
def test_step_parity_small_fp8(variant):
    """SURVEY.md 8(f1), the fp8 e4m3 variant of the weight stream (reading A17b) against the oracle on the dequantised
    values."""
    kw, n_new = dict(dtype=BF16, wquant=2, ffn=352), 1
    if variant == "mha_dh128":
        kw.update(hidden=256, n_q_heads=2, n_kv_heads=2, head_dim=128)
    elif variant == "no_proj":
        kw.update(dgf_proj=0)
    elif variant == "fusion_linear":
        kw.update(dgf_proj=0, fusion=1)
    elif variant == "n_new5":
        n_new = 5
    elif variant == "wide":
        kw.update(tree=TreeSpec(3, (6, 3, 2), (0, 0, 12), 20))
    elif variant == "max_branch":
        kw.update(tree=TreeSpec(2, (32, 1), (0, 32), 40))
    case = _boost(make_case(small_cfg(**kw), n_new=n_new))
    assert case.layers[0]["wq"].dtype == torch.float8_e4m3fn
    s, gpu, ora = _run(case)
    assert s["same_tree"]
    assert s["free"]["same_tree"] or s["free"]["tie"] is not None


@pytest.mark.parametrize("name", ["c2_llama2_7b_fp8", "c3_llama2_13b_fp8"])
def test_full_size_configs_fp8(name):
    from paper_2412_18934_b200.configs import fp8_variants
    cfg = [c for c in fp8_variants() if c.name == name][0]
    case = make_case(cfg, n_new=1)
    s, gpu, ora = _run(case, tight=True)
    assert gpu["n_out"] == min(cfg.tree.gamma, cfg.tree.pool_size())
    assert s["free"]["same_tree"] or s["free"]["tie"] is not None


# ---- tcgen05 GEMV (csrc/gemv_umma.cuh): wide levels and level-0 row batches --------------------------------------
def umma_cfg(**kw) -> DraftConfig:
    """Every K a multiple of 64 (hidden 192, 2 x hidden 384, q width 256, ffn 320), so that all seven GEMV kinds of a
    level take the tcgen05 kernel; rows per CTA are ragged (192 / 148, 320 / 148, 1000 / 148)."""
    base = dict(name="umma_small", hidden=192, n_q_heads=4, n_kv_heads=2, head_dim=64, n_layers=2, ffn=320,
                vocab=1000, dtype=BF16, prefix=70, feat_scale=1.0, rope_theta=1e4,
                tree=TreeSpec(3, (3, 2, 2), (0, 4, 5), 9), seed=17)
    base.update(kw)
    return DraftConfig(**base)


@pytest.mark.parametrize("variant", ["m1_forced", "m12", "m20", "m32_max_branch", "n_new33", "n_new64", "mha_dh128_gqa", "no_proj",
                                     "final_norm", "big_vocab", "huge_vocab", "llama3_vocab_64_rows", "tiny_dims"])
def test_step_parity_umma(variant):
    kw, n_new, min_m = {}, 1, None
    if variant == "m1_forced":  # every level, 1 ... 5 rows, through the tcgen05 kernel (N = 16 columns)
        min_m = 1
    elif variant == "m12":
        kw.update(tree=TreeSpec(3, (6, 3, 2), (0, 0, 12), 20))
    elif variant == "m20":
        kw.update(tree=TreeSpec(2, (20, 2), (0, 20), 24))
    elif variant == "m32_max_branch":
        kw.update(tree=TreeSpec(2, (32, 1), (0, 32), 40))
    elif variant == "n_new33":
        n_new = 33
    elif variant == "n_new64":  # the widest single pass: 64 rows x 2 planes = 128 accumulator columns
        n_new = 64
    elif variant == "mha_dh128_gqa":
        kw.update(hidden=256, n_q_heads=4, n_kv_heads=2, head_dim=128, tree=TreeSpec(2, (10, 2), (0, 10), 16))
    elif variant == "no_proj":
        kw.update(dgf_proj=0, tree=TreeSpec(2, (10, 2), (0, 10), 16))
    elif variant == "final_norm":
        kw.update(first_layer_input_norm=0, final_norm=1, tree=TreeSpec(2, (10, 2), (0, 10), 16))
    elif variant == "big_vocab":  # 20000 / 148 = 136 rows per CTA: two super-blocks of the LM head
        kw.update(vocab=20000, tree=TreeSpec(2, (10, 2), (0, 10), 16))
    elif variant == "huge_vocab":  # 70000 / 148 = 473 rows per CTA: four super-blocks, the accumulator buffers are reused
        kw.update(vocab=70000, tree=TreeSpec(2, (10, 2), (0, 10), 16))
    elif variant == "llama3_vocab_64_rows":  # 867 rows per CTA x 64 LM-head rows: the result buffer does not fit, the
        kw.update(vocab=128256, tree=TreeSpec(3, (8, 8, 1), (0, 8, 64), 40))  # level runs in two 32-row passes; 7 super-blocks
    elif variant == "tiny_dims":  # fewer rows than CTAs (one row, one box per CTA), a single K-chunk of one slab
        kw.update(hidden=64, n_q_heads=1, n_kv_heads=1, head_dim=64, ffn=64, vocab=120, tree=TreeSpec(2, (10, 2), (0, 10), 16))
    case = _boost(make_case(umma_cfg(**kw), n_new=n_new))
    s, gpu, ora = _run(case, umma_min_m=min_m)
    assert gpu["umma_launches"] > 0, "the tcgen05 GEMV did not run"
    assert s["same_tree"]
    assert s["free"]["same_tree"] or s["free"]["tie"] is not None


@pytest.mark.parametrize("variant", ["m1_forced", "m12", "m32_max_branch", "n_new64", "mha_dh128_gqa", "no_proj", "tiny_dims"])
def test_step_parity_umma_k_split(variant):
    """The tcgen05 GEMV with K split over CTA pairs (csrc/gemv_umma.cuh UmmaParams::ksplit) forced on from one row:
    O, down and the DGF matrices (one super-block per CTA) take it, the others do not."""
    kw, n_new, min_m = {}, 1, None
    if variant == "m1_forced":
        min_m = 1
    elif variant == "m12":
        kw.update(tree=TreeSpec(3, (6, 3, 2), (0, 0, 12), 20))
    elif variant == "m32_max_branch":
        kw.update(tree=TreeSpec(2, (32, 1), (0, 32), 40))
    elif variant == "n_new64":
        n_new = 64
    elif variant == "mha_dh128_gqa":
        kw.update(hidden=256, n_q_heads=4, n_kv_heads=2, head_dim=128, tree=TreeSpec(2, (10, 2), (0, 10), 16))
    elif variant == "no_proj":
        kw.update(dgf_proj=0, tree=TreeSpec(2, (10, 2), (0, 10), 16))
    elif variant == "tiny_dims":
        kw.update(hidden=64, n_q_heads=1, n_kv_heads=1, head_dim=64, ffn=64, vocab=120, tree=TreeSpec(2, (10, 2), (0, 10), 16))
    case = _boost(make_case(umma_cfg(**kw), n_new=n_new))
    s, gpu, ora = _run(case, umma_min_m=min_m, umma_ksplit_min_m=1)
    assert gpu["umma_launches"] > 0 and gpu["ksplit_launches"] > 0, "no GEMV ran with K split over a CTA pair"
    assert s["same_tree"]
    assert s["free"]["same_tree"] or s["free"]["tie"] is not None

"""Workload shapes: the five configurations of BASELINE.json and the tree specs
DESIGN.md derives for them (reading A15). Host-side description only."""
from dataclasses import dataclass, field, replace
from typing import Dict, List, Tuple

F32, BF16 = 0, 1
MAX_DEPTH = 16


@dataclass(frozen=True)
class TreeSpec:
    """depth D, branch[l], beam[l] (0 = all), gamma -- include/dovetail.h dovetail_tree_spec_t."""
    depth: int
    branch: Tuple[int, ...]
    beam: Tuple[int, ...]
    gamma: int

    def rows_per_level(self, n_new: int = 1) -> List[int]:
        """Rows of each of the D forwards: n_new, then the frontier sizes."""
        rows, m = [n_new], 1
        for l in range(1, self.depth):
            n = m * self.branch[l - 1]
            m = self.beam[l] if 0 < self.beam[l] < n else n
            rows.append(m)
        return rows

    def pool_size(self) -> int:
        rows = self.rows_per_level(1)
        return self.branch[0] + sum(rows[l] * self.branch[l] for l in range(1, self.depth))

    def tree_rows(self) -> int:
        return sum(self.rows_per_level(1)[1:])


@dataclass(frozen=True)
class DraftConfig:
    name: str
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    n_layers: int
    ffn: int
    vocab: int
    rope_theta: float = 1e4
    rms_eps: float = 1e-5
    dtype: int = BF16
    dgf_proj: int = 1
    first_layer_input_norm: int = 1
    final_norm: int = 0
    fusion: int = 0           # 0: DGF; 1: concat + one Linear 2d -> d, the EAGLE-2 baseline
    wquant: int = 0           # 1: weight matrices are int8 with one fp32 scale per output row; the
                              #    embedding, norm gains, gate bias and KV cache stay in dtype (bf16)
    prefix: int = 64          # committed KV length L of the workload
    feat_scale: float = 1.0   # features ~ N(0,1) * feat_scale
    tree: TreeSpec = field(default_factory=lambda: TreeSpec(1, (1,), (0,), 1))
    seed: int = 1234

    @property
    def esize(self) -> int:
        return 4 if self.dtype == F32 else 2

    @property
    def fusion_name(self) -> str:
        return "concat+linear (EAGLE-2 baseline)" if self.fusion == 1 else ("DGF" if self.dgf_proj else "DGF without projections")

    def weight_params(self) -> Dict[str, int]:
        """Parameter counts by group; the draft's learnable parameters exclude
        the embedding and the LM head, which are the target's (Table 6)."""
        d, F = self.hidden, self.ffn
        dq, dkv = self.n_q_heads * self.head_dim, self.n_kv_heads * self.head_dim
        dgf = (2 * d * d if (self.dgf_proj and self.fusion == 0) else 0) + 2 * d * d + d
        layer = d * dq + 2 * d * dkv + dq * d + 3 * d * F + 2 * d
        return dict(dgf=dgf, layer=layer, layers=layer * self.n_layers, lm_head=self.vocab * d,
                    final_norm=d if self.final_norm else 0)

    def learnable_params(self) -> int:
        p = self.weight_params()
        return p["dgf"] + p["layers"] + p["final_norm"]

    def forward_bytes(self, prefix_len: int) -> int:
        """Algorithmic HBM bytes of one forward: every weight
        byte once + the prefix K/V of every layer once."""
        p = self.weight_params()
        w = (p["dgf"] + p["layers"] + p["final_norm"] + p["lm_head"]) * self.esize
        if self.wquant:  # matrices at 1 byte per element + 4 bytes of scale per output row; vectors in dtype
            d, F = self.hidden, self.ffn
            dq, dkv = self.n_q_heads * self.head_dim, self.n_kv_heads * self.head_dim
            vec = d + 2 * d * self.n_layers + p["final_norm"]
            mats = p["dgf"] + p["layers"] + p["final_norm"] + p["lm_head"] - vec
            rows = (2 * d if (self.dgf_proj and self.fusion == 0) else 0) + d + self.n_layers * (dq + 2 * dkv + d + 2 * F + d) + self.vocab
            w = mats + 4 * rows + vec * self.esize
        kv = self.n_layers * 2 * prefix_len * self.n_kv_heads * self.head_dim * self.esize
        return w + kv

    def step_bytes(self, n_new: int = 1) -> int:
        return self.tree.depth * self.forward_bytes(self.prefix)


def eagle2_fusion_params(d: int) -> int:
    """The fusion DGF replaces: concat + one Linear 2d -> d with bias."""
    return 2 * d * d + d


_C1 = DraftConfig("c1_tiny_fp32", 256, 4, 4, 64, 2, 688, 1024, dtype=F32, prefix=64,
                  tree=TreeSpec(3, (2, 2, 2), (0, 0, 0), 14), seed=1234)
_C2 = DraftConfig("c2_llama2_7b", 4096, 32, 32, 128, 2, 11008, 32000, prefix=512,
                  feat_scale=4096 ** -0.5, tree=TreeSpec(4, (3, 2, 2, 2), (0, 0, 0, 0), 10), seed=1235)
_C3 = DraftConfig("c3_llama2_13b", 5120, 40, 40, 128, 4, 13824, 32000, prefix=1024,
                  feat_scale=5120 ** -0.5, tree=TreeSpec(5, (2,) * 5, (0, 2, 2, 2, 2), 16), seed=1236)
_C5 = DraftConfig("c5_llama3_8b", 4096, 32, 8, 128, 2, 14336, 128256, rope_theta=5e5, prefix=8192,
                  feat_scale=4096 ** -0.5, tree=TreeSpec(5, (2,) * 5, (0, 2, 2, 2, 2), 16), seed=1238)

CONFIGS: Dict[str, DraftConfig] = {c.name: c for c in (_C1, _C2, _C3, _C5)}
CONFIGS["c1"] = _C1
CONFIGS["c2"] = _C2
CONFIGS["c3"] = _C3
CONFIGS["c5"] = _C5


def c4_sweep() -> List[DraftConfig]:
    """Config 4: depth / tree-width sweep on the 13B shape, prefix 2048."""
    out = []
    for layers in (1, 2, 4, 8):
        for k, gamma in ((1, 4), (2, 8), (2, 16), (4, 32)):
            out.append(replace(_C3, name=f"c4_l{layers}_g{gamma}", n_layers=layers, prefix=2048,
                               tree=TreeSpec(5, (k,) * 5, (0,) + (k,) * 4, gamma), seed=1237))
    # forward-level form: one tree level of M rows (a depth-2 tree whose root keeps M children), so that
    # step time - level-0 forward = one forward at tree width M
    for layers in (1, 4):
        for m in (4, 8, 16, 32):
            out.append(replace(_C3, name=f"c4_l{layers}_m{m}", n_layers=layers, prefix=2048,
                               tree=TreeSpec(2, (m, 2), (0, m), 16), seed=1237))
    return out


def depth_sweep() -> List[DraftConfig]:
    """The ablation's shape (Table 6, Table 7 :373-383) as a latency-vs-depth sweep on the
    7B-shaped draft: the EAGLE-2 baseline (concat + Linear, 1 block, "w/o both"), then DGF with 1 ... 6 blocks
    ("w/ DGF", "w/ DGF + 1" ... "+ 5"), prefix 512, the paper's 16-candidate server tree shape of C3."""
    tree = TreeSpec(5, (2,) * 5, (0, 2, 2, 2, 2), 16)
    out = [replace(_C2, name="depth_eagle2_l1", n_layers=1, fusion=1, dgf_proj=0, tree=tree, seed=1239)]
    for layers in range(1, 7):
        out.append(replace(_C2, name=f"depth_dgf_l{layers}", n_layers=layers, tree=tree, seed=1239))
    return out


def int8_variants() -> List[DraftConfig]:
    """the 7B / 13B / Llama-3-8B shaped workloads with int8 weight matrices and per-row scales
    ("it is advisable to apply int8 quantization to the drafting model on the GPU")."""
    return [replace(c, name=c.name + "_int8", wquant=1) for c in (_C2, _C3, _C5)]


def fp8_variants() -> List[DraftConfig]:
    """The same workloads with fp8 e4m3 weight matrices and per-row scales (SURVEY.md 8(f1) "int8 / fp8")."""
    return [replace(c, name=c.name + "_fp8", wquant=2) for c in (_C2, _C3, _C5)]


def paper_preset(server: bool = True) -> TreeSpec:
    """width 10 / depth 7 / 16 candidates (servers); 10 / 4 / 7 (PC)."""
    D, g = (7, 16) if server else (4, 7)
    return TreeSpec(D, (10,) * D, (0,) + (10,) * (D - 1), g)

"""Seeded synthetic workloads: one draft-step case = weights, KV cache with a committed
prefix, target features and tokens, tree spec. Input generation only -- none of the method's arithmetic lives
here; it serves the tests, the bench and the smoke check alike and imports neither the CUDA path's kernels nor
the oracle."""
from dataclasses import dataclass
from typing import Dict, Optional

import torch

from . import synth
from .configs import DraftConfig, TreeSpec


@dataclass
class Case:
    cfg: DraftConfig
    top: Dict
    layers: list
    k: torch.Tensor
    v: torch.Tensor
    feats: torch.Tensor
    tokens: torch.Tensor
    L: int
    capacity: int
    tree: TreeSpec


def make_case(cfg: DraftConfig, n_new: int = 1, prefix: Optional[int] = None, tree: Optional[TreeSpec] = None,
              slack: int = 8, device="cuda") -> Case:
    tree = tree or cfg.tree
    L = cfg.prefix if prefix is None else prefix
    cap = L + n_new + tree.tree_rows() + slack
    top, layers = synth.make_weights(cfg, device=device)
    k, v = synth.make_kv(cfg, cap, L, device=device)
    feats, tokens = synth.make_inputs(cfg, n_new, device=device)
    return Case(cfg, top, layers, k, v, feats, tokens, L, cap, tree)

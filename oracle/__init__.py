"""TEST INFRASTRUCTURE, NOT PRODUCT CODE.

The fp64 CPU oracle of the Dovetail draft step, written from the paper
(arxiv 2412.18934). Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package. It imports
nothing from the CUDA package.
"""
from .oracle import (  # noqa: F401
    OracleConfig,
    OracleWeights,
    build,
    dgf,
    e4m3_to_double,
    forward,
    fusion_linear,
    kv_commit,
    lm_head,
    log_softmax,
    matvec,
    matvec_f8,
    matvec_q8,
    rmsnorm,
    rope,
    step,
    topk,
    tree_replay,
    verify_accept,
    verify_plan,
)

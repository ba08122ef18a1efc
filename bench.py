#!/usr/bin/env python
"""bench.py -- draft-step throughput of the B200-native Dovetail draft model.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c3] [--impl ours|reference]

One "step" is one dovetail_draft_step: D forwards of the draft model over the levels of
the draft tree plus the final rerank (all rows of SURVEY.md 8a), on synthetic seeded
inputs shaped like BASELINE.json's headline workload (configs[2], the Llama-2-13B-shaped
draft; it fits one GPU). Prints ONE JSON line (rank 0).

  value      draft tokens/s (gamma candidates per step / step time), inputs resident in HBM
  e2e        the same through the C ABI with HOST inputs and outputs: per step an H2D copy of
             (hidden_feats, tokens) from pinned memory and a D2H read of the candidates
  roofline   the weight-streaming GEMV kernel (k_gemv_mma, > 95 % of the bytes): algorithmic
             bytes per launch / its mean launch duration (CUDA events around every launch,
             taken in a separate instrumented pass over the same steps), against the
             measured HBM copy bandwidth of MEASURED_PEAKS.json
  cpu_baseline  the fp64 oracle, as it stands, on the host cores (rank 0, N = 1)

N > 1: independent replicas, one process per GPU (a batch-1 draft step is a sequential
chain and does not shard); value sums the replicas, time is the
max over ranks.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
METRIC, UNIT = "draft_tokens_per_s_batch1", "tokens/s"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def oracle_sample(case, full_step: bool):
    """Time the oracle on a bounded sample of the workload. Returns (seconds per whole step
    (extrapolated when sampled), description, cores)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity import run_oracle
    from paper_2412_18934_b200.configs import TreeSpec
    import dataclasses
    cores = len(os.sched_getaffinity(0))
    tree = case.tree
    if full_step:
        t0 = time.perf_counter()
        run_oracle(case, dump=False)
        return time.perf_counter() - t0, "one whole draft step (all D forwards + rerank)", cores
    # one level-0 forward + LM head + top-k = 1 of the step's row-forwards
    sub = dataclasses.replace(case, tree=TreeSpec(1, (tree.branch[0],), (0,), tree.branch[0]))
    t0 = time.perf_counter()
    run_oracle(sub, dump=False)
    dt = time.perf_counter() - t0
    row_forwards = sum(tree.rows_per_level(case.tokens.shape[0]))
    return dt * row_forwards, (f"one level-0 row-forward (DGF + {case.cfg.n_layers} layers + LM head + top-k), "
                               f"scaled x{row_forwards} row-forwards of the step"), cores


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="c3")
    ap.add_argument("--n-new", type=int, default=1)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-profile-pass", action="store_true")
    a = ap.parse_args()
    rank, world, local = dist_env()
    K, W = a.steps, max(a.warmup, 3)

    import torch
    from paper_2412_18934_b200.configs import CONFIGS
    from paper_2412_18934_b200.configs import c4_sweep
    all_cfgs = dict(CONFIGS)
    all_cfgs.update({c.name: c for c in c4_sweep()})  # BASELINE.json configs[3]: c4_l{layers}_g{gamma}
    cfg = all_cfgs[a.config]
    tree = cfg.tree
    config = {"workload": f"{cfg.name}: hidden {cfg.hidden}, {cfg.n_q_heads}q/{cfg.n_kv_heads}kv x {cfg.head_dim}, "
                          f"{cfg.n_layers} layers, ffn {cfg.ffn}, vocab {cfg.vocab}, prefix {cfg.prefix}, "
                          f"tree D{tree.depth} branch {list(tree.branch)} beam {list(tree.beam)} gamma {tree.gamma}, "
                          f"n_new {a.n_new}",
              "batch": 1, "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
              "l2": "inputs larger than L2 (every forward streams > 1 GB of weights)"}
    from paper_2412_18934_b200.cases import make_case  # seeded inputs only; the oracle is imported by its own legs

    if a.impl == "reference":
        # the oracle, as it stands, on the host cores; rank 0 alone
        if rank != 0:
            return
        dev = "cuda" if torch.cuda.is_available() else "cpu"
        case = make_case(cfg, n_new=a.n_new, device=dev)
        case = _to_host(case)
        t_probe, _, cores = oracle_sample(case, full_step=False)
        full = t_probe * (K + W) < 150.0
        for _ in range(W if full else min(W, 3)):
            oracle_sample(case, full)
        ts = []
        for _ in range(K):
            t, sample, cores = oracle_sample(case, full)
            ts.append(t)
        step_s = sum(ts) / len(ts)
        val = tree.gamma / step_s
        line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": 0, "steps": K, "warmup": W,
                "ms_per_step": step_s * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "config": config,
                "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line))
        return

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU path)"
    from paper_2412_18934_b200 import binding, replicas
    binding.load()  # fail loudly if the library is missing
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()

    case = make_case(cfg, n_new=a.n_new, device="cuda")
    h = binding.dovetail_draft_init(case.top, case.layers, cfg)
    kv = binding.KVCache(case.k, case.v, case.L)
    out = binding.alloc_out(tree.gamma)
    stream = torch.cuda.current_stream()

    def step_device():
        kv.committed_len = case.L  # untimed bookkeeping: discard the tree rows (kv_commit mode 0 semantics)
        binding.dovetail_draft_step(h, case.feats, case.tokens, kv, tree, out)

    # host-side buffers of the end-to-end path
    feats_h = case.feats.cpu().pin_memory()
    tok_h = case.tokens.cpu().pin_memory()
    feats_d, tok_d = torch.empty_like(case.feats), torch.empty_like(case.tokens)
    out_h = {k: torch.empty_like(v, device="cpu").pin_memory() for k, v in out.items()}

    def step_e2e():
        kv.committed_len = case.L
        feats_d.copy_(feats_h, non_blocking=True)
        tok_d.copy_(tok_h, non_blocking=True)
        binding.dovetail_draft_step(h, feats_d, tok_d, kv, tree, out)
        for k2 in out_h:
            out_h[k2].copy_(out[k2], non_blocking=True)
        stream.synchronize()  # the caller consumes the candidates before the next round

    def timed(fn, steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(steps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        barrier()
        ms, _ = replicas.job_time_and_work(e0.elapsed_time(e1), 0.0, device="cuda")  # max over ranks
        return ms

    for _ in range(W):
        step_device()
    torch.cuda.synchronize()
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    ms = timed(step_device, K)
    for _ in range(W):
        step_e2e()
    ms_e2e = timed(step_e2e, K)
    clk = clocks.stop() if rank == 0 else None
    launches = binding.dovetail_last_launch_count(h) * K
    n_out = int(out["n_out"].item())
    assert n_out == min(tree.gamma, tree.pool_size()), "the step did not produce its candidates"

    # instrumented pass: CUDA events around every launch of the same steps
    roof = None
    if not a.no_profile_pass:
        peak, peak_src = peaks()
        binding.dovetail_draft_set_profile(h, True)
        agg = {}
        kp = min(K, 20)
        for _ in range(kp):
            step_device()
            torch.cuda.synchronize()
            for kind, r in binding.dovetail_profile_read(h).items():
                g = agg.setdefault(kind, dict(ms=0.0, launches=0, bytes=0))
                g["ms"] += r["ms"]; g["launches"] += r["launches"]; g["bytes"] += r["bytes"]
        binding.dovetail_draft_set_profile(h, False)
        gemv = ("dgf_proj", "dgf_gate", "qkv", "o_proj", "gate_up", "down", "lm_head")
        g_ms = sum(agg[k]["ms"] for k in gemv)
        g_n = sum(agg[k]["launches"] for k in gemv)
        g_b = sum(agg[k]["bytes"] for k in gemv)
        tot_ms = sum(v["ms"] for v in agg.values())
        achieved = (g_b / g_n) / (g_ms / g_n * 1e-3) / 1e9 if g_n else 0.0
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.json.txt")
        if os.path.exists(tp):
            try:
                t = json.load(open(tp)).get(cfg.name, {})
                # the ncu capture covers 8 launches; scale its DRAM bytes / algorithmic bytes ratio to the
                # mean launch of the whole step so that traffic is comparable with bytes_per_launch
                if t.get("k_gemv_dram_bytes_per_launch") and t.get("captured_algorithmic_bytes_per_launch") and g_n:
                    traffic = (g_b / g_n) * t["k_gemv_dram_bytes_per_launch"] / t["captured_algorithmic_bytes_per_launch"]
            except Exception:
                traffic = None
        roof = {"bound": "hbm", "kernel": "k_gemv_mma (bf16) / k_gemv (fp32): all weight-streaming GEMV launches of the step",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "traffic": traffic, "bytes_per_launch": g_b / g_n if g_n else 0, "us_per_launch": g_ms / g_n * 1e3 if g_n else 0,
                "launches_per_step": g_n // kp, "gemv_share_of_step_time": g_ms / tot_ms if tot_ms else None,
                "by_kind_us_per_step": {k: round(v["ms"] / kp * 1e3, 2) for k, v in agg.items() if v["launches"]},
                "note": "instrumented pass serialises the launches (no programmatic-dependent-launch overlap)"}

    step_bytes = tree.depth * binding.dovetail_forward_bytes(h, case.L + a.n_new)
    step_ms = ms / K
    value = world * tree.gamma * K / (ms * 1e-3)
    e2e_val = world * tree.gamma * K / (ms_e2e * 1e-3)
    peak, peak_src = peaks()
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16 weights and KV cache, f32 activations and accumulation" if cfg.dtype == 1 else "f32", "data": "synthetic",
            "config": config, "draft_step_us": step_ms * 1e3, "forward_us": step_ms * 1e3 / tree.depth,
            "step_hbm_gbs": step_bytes / (step_ms * 1e-3) / 1e9,
            "step_frac_of_measured_peak": step_bytes / (step_ms * 1e-3) / 1e9 / peak,
            "step_frac_of_8tbs_nominal": step_bytes / (step_ms * 1e-3) / 1e9 / 8000.0,
            "algorithmic_bytes_per_step": step_bytes,
            "e2e": {"value": e2e_val, "unit": UNIT, "ms_per_step": ms_e2e / K,
                    "h2d_bytes_per_step": feats_h.numel() * 4 + tok_h.numel() * 4,
                    "d2h_bytes_per_step": sum(v.numel() * v.element_size() for v in out_h.values())},
            "gpu_launches": launches, "clocks": clk, "roofline": roof}
    if rank == 0 and world == 1 and not a.no_cpu_baseline:
        hc = _to_host(case)
        t, sample, cores = oracle_sample(hc, full_step=True)
        line["cpu_baseline"] = {"value": tree.gamma / t, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": sample, "seconds_per_step": t}
    if rank == 0:
        print(json.dumps(line))
    binding.dovetail_draft_destroy(h)
    if world > 1:
        dist.destroy_process_group()


def _to_host(case):
    import dataclasses
    hc = lambda t: None if t is None else t.detach().cpu()
    return dataclasses.replace(case, top={k: hc(v) for k, v in case.top.items()},
                               layers=[{k: hc(v) for k, v in l.items()} for l in case.layers],
                               k=case.k.cpu(), v=case.v.cpu(), feats=case.feats.cpu(), tokens=case.tokens.cpu())


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- draft-step throughput of the B200-native Dovetail draft model.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c3|c1|c2|c5|c4_...|all] [--impl ours|reference]

One "step" is one dovetail_draft_step: D forwards of the draft model over the levels of the draft tree plus
the final rerank (all rows of SURVEY.md 8a), on synthetic seeded inputs shaped like BASELINE.json's headline
workload (configs[2], the Llama-2-13B-shaped draft; it fits one GPU). Prints ONE JSON line (rank 0);
`--config all` prints one line per configuration (C1, C2, C3, C5 and the C4 sweep), headline last.

  value        draft tokens/s (gamma candidates per step / step time), inputs resident in HBM; the K timed
               steps are bracketed by one pair of CUDA events on the launching stream
  e2e          the same through the C ABI with HOST inputs and outputs: per step an H2D copy of
               (hidden_feats, tokens) from pinned memory and a D2H read of the candidates
  roofline     the weight-streaming GEMV launches (k_gemv_mma, > 95 % of the bytes): algorithmic bytes per
               launch / mean launch duration. Durations come from %globaltimer stamps every kernel writes at
               its first CTA's start and last CTA's end (dovetail_trace_*, include/dovetail_hooks.h) -- the
               launches keep their programmatic-dependent-launch overlap -- taken as each launch's EXCLUSIVE
               time (clipped to start at the end of the launches before it), so that the kinds add up to at
               most the step, and scaled to the event-timed ms_per_step. Peaks: the measured copy bandwidth of
               MEASURED_PEAKS.json, the read-only streaming ceilings measured in this run
               (dovetail_probe_stream), and the 8 TB/s nominal figure BASELINE.json's 70 % bar refers to.
  cpu_baseline the fp64 oracle, as it stands, on the host cores (all cores and one thread; rank 0, N = 1)

N > 1: independent replicas, one process per GPU (a batch-1 draft step is a sequential chain and does not
shard); value sums the replicas, time is the max over ranks. Without torchrun,
`--gpus N` re-launches itself under torch.distributed.run with N ranks.
"""
import argparse
import json
import os
import socket
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
NOMINAL_HBM_GBS = 8000.0   # BASELINE.json north_star: "HBM bytes at about 8 TB/s"
METRIC, UNIT = "draft_tokens_per_s_batch1", "tokens/s"
GEMV_KINDS = ("dgf_proj", "dgf_gate", "qkv", "o_proj", "gate_up", "down", "lm_head")


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs: read+write copy)"
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
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def set_omp_threads(n: int):
    """The oracle's OpenMP loops take their thread count from libgomp; nothing of oracle/ is touched."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except Exception:
        return False


def oracle_sample(case, full_step: bool):
    """Time the oracle on a bounded sample of the workload. Returns (seconds per whole step (extrapolated when
    sampled), description)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity import run_oracle
    from paper_2412_18934_b200.configs import TreeSpec
    import dataclasses
    tree = case.tree
    if full_step:
        t0 = time.perf_counter()
        run_oracle(case, dump=False)
        return time.perf_counter() - t0, "one whole draft step (all D forwards + rerank)"
    # one level-0 forward + LM head + top-k = 1 of the step's row-forwards
    sub = dataclasses.replace(case, tree=TreeSpec(1, (tree.branch[0],), (0,), tree.branch[0]))
    t0 = time.perf_counter()
    run_oracle(sub, dump=False)
    dt = time.perf_counter() - t0
    row_forwards = sum(tree.rows_per_level(case.tokens.shape[0]))
    return dt * row_forwards, (f"one level-0 row-forward (DGF + {case.cfg.n_layers} layers + LM head + top-k), "
                               f"scaled x{row_forwards} row-forwards of the step")


def _to_host(case):
    import dataclasses
    hc = lambda t: None if t is None else t.detach().cpu()
    return dataclasses.replace(case, top={k: hc(v) for k, v in case.top.items()},
                               layers=[{k: hc(v) for k, v in l.items()} for l in case.layers],
                               k=case.k.cpu(), v=case.v.cpu(), feats=case.feats.cpu(), tokens=case.tokens.cpu())


def all_configs():
    from paper_2412_18934_b200.configs import CONFIGS, c4_sweep, depth_sweep, fp8_variants, int8_variants
    cfgs = {c.name: c for c in CONFIGS.values()}
    cfgs.update({k: v for k, v in CONFIGS.items()})
    cfgs.update({c.name: c for c in c4_sweep()})
    cfgs.update({c.name: c for c in depth_sweep()})
    cfgs.update({c.name: c for c in int8_variants()})
    cfgs.update({c.name.split("_")[0] + "_int8": c for c in int8_variants()})  # c2_int8, c3_int8, c5_int8
    cfgs.update({c.name: c for c in fp8_variants()})
    cfgs.update({c.name.split("_")[0] + "_fp8": c for c in fp8_variants()})
    # the tree the paper itself runs (width 10, depth 7, 16 candidates) on the 7B / 13B shapes
    import dataclasses
    from paper_2412_18934_b200.configs import paper_preset
    for base in ("c2", "c3"):
        cfgs[base + "_paper_tree"] = dataclasses.replace(CONFIGS[base], name=CONFIGS[base].name + "_paper_tree", tree=paper_preset(True))
    return cfgs


def workload(cfg, n_new, world):
    tree = cfg.tree
    return {"workload": f"{cfg.name}: hidden {cfg.hidden}, {cfg.n_q_heads}q/{cfg.n_kv_heads}kv x {cfg.head_dim}, "
                        f"{cfg.n_layers} layers, ffn {cfg.ffn}, vocab {cfg.vocab}, prefix {cfg.prefix}, fusion {cfg.fusion_name}, "
                        f"tree D{tree.depth} branch {list(tree.branch)} beam {list(tree.beam)} gamma {tree.gamma}, "
                        f"n_new {n_new}",
            "batch": 1, "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
            "l2": "inputs larger than L2 (every forward streams its weights, > 1 GB on the 7B / 13B shapes, once)"}


def reference_line(a, cfg):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 alone."""
    import torch
    from paper_2412_18934_b200.cases import make_case
    K, W = a.steps, max(a.warmup, 3)
    case = _to_host(make_case(cfg, n_new=a.n_new, device="cuda" if torch.cuda.is_available() else "cpu"))
    cores = len(os.sched_getaffinity(0))
    t_probe, _ = oracle_sample(case, full_step=False)
    full = t_probe * (K + W) < 150.0
    for _ in range(W if full else min(W, 3)):
        oracle_sample(case, full)
    ts = []
    for _ in range(K):
        t, sample = oracle_sample(case, full)
        ts.append(t)
    step_s = sum(ts) / len(ts)
    val = cfg.tree.gamma / step_s
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": 0, "steps": K, "warmup": W,
            "ms_per_step": step_s * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload(cfg, a.n_new, 1),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "cpu_model": cpu_model()},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


def bench_one(a, cfg, rank, world, local, dist):
    import dataclasses
    import torch
    from paper_2412_18934_b200 import binding, replicas
    from paper_2412_18934_b200.cases import make_case  # seeded inputs only; the oracle is imported by its own legs
    K, W = a.steps, max(a.warmup, 3)
    tree = cfg.tree

    def barrier():
        if world > 1:
            dist.barrier()

    case = make_case(cfg, n_new=a.n_new, device="cuda")
    h = binding.dovetail_draft_init(case.top, case.layers, cfg)
    for kv_ in a.tune:
        k_, v_ = kv_.split("=")
        binding.dovetail_hooks_tune(h, int(k_), int(v_))
    kv = binding.KVCache(case.k, case.v, case.L)
    out = binding.alloc_out(tree.gamma)
    stream = torch.cuda.current_stream()

    def step_device(hh=h):
        kv.committed_len = case.L  # untimed bookkeeping: discard the tree rows (kv_commit mode 0 semantics)
        binding.dovetail_draft_step(hh, case.feats, case.tokens, kv, tree, out)

    # host-side buffers of the end-to-end path: inputs in one pinned buffer (features, then the token ids as raw
    # words), outputs in one pinned buffer (binding.alloc_out packs the step's outputs into one allocation)
    n_f = case.feats.numel()
    in_h = torch.empty(n_f + case.tokens.numel(), dtype=torch.float32).pin_memory()
    in_h[:n_f] = case.feats.cpu().reshape(-1)
    in_h[n_f:].view(torch.int32)[:] = case.tokens.cpu()
    in_d = torch.empty_like(in_h, device="cuda")
    feats_d, tok_d = in_d[:n_f].view(case.feats.shape), in_d[n_f:].view(torch.int32)
    out_h = torch.empty_like(out["_packed"], device="cpu").pin_memory()

    def step_e2e():
        kv.committed_len = case.L
        in_d.copy_(in_h, non_blocking=True)
        binding.dovetail_draft_step(h, feats_d, tok_d, kv, tree, out)
        out_h.copy_(out["_packed"], non_blocking=True)
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
    how = {0: "direct launches", 1: "CUDA graph replay", 2: "CUDA graph capture"}[binding.dovetail_hooks_stat(h, binding.STAT_GRAPH)]
    # the same steps with direct launches (programmatic dependent launch, no graph): SURVEY.md 3(2)
    launch_modes = None
    if world == 1:
        binding.dovetail_hooks_tune(h, binding.TUNE_GRAPHS, 0)
        for _ in range(W):
            step_device()
        ms_d = timed(step_device, K)
        for _ in range(W):
            step_e2e()
        ms_e2e_d = timed(step_e2e, K)
        binding.dovetail_hooks_tune(h, binding.TUNE_GRAPHS, 1)
        launch_modes = {"timed_as": how, "graph_us_per_step": ms / K * 1e3, "direct_us_per_step": ms_d / K * 1e3,
                        "graph_e2e_us_per_step": ms_e2e / K * 1e3, "direct_e2e_us_per_step": ms_e2e_d / K * 1e3}
    launches = binding.dovetail_last_launch_count(h) * K
    n_out = int(out["n_out"].item())
    assert n_out == min(tree.gamma, tree.pool_size()), "the step did not produce its candidates"
    binding.dovetail_draft_status(h)
    step_ms = ms / K
    step_bytes = tree.depth * binding.dovetail_forward_bytes(h, case.L + a.n_new)
    peak, peak_src = peaks()

    # ---- distribution over individually timed replays (median of >= 200 after >= 20 warm-ups)
    R = a.replays
    dist_us = None
    if R > 0 and world == 1:
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(R)]
        for _ in range(20):
            step_device()
        for e0, e1 in ev:
            e0.record(stream)
            step_device()
            e1.record(stream)
        torch.cuda.synchronize()
        ts = sorted(e0.elapsed_time(e1) * 1e3 for e0, e1 in ev)
        dist_us = {"replays": R, "median": ts[R // 2], "p10": ts[R // 10], "p90": ts[(9 * R) // 10], "min": ts[0]}

    # ---- per-kernel device time: globaltimer stamps, PDL overlap kept --------------------------------
    roof, per_level = None, None
    if not a.no_trace:
        binding.dovetail_trace_enable(h, True)
        kp = min(max(K, 5), 20)
        agg, lv, step_tr = {}, {}, []
        for _ in range(3):
            step_device()
        for _ in range(kp):
            step_device()
            torch.cuda.synchronize()
            t = binding.dovetail_trace_read(h)
            step_tr.append(t["step_us"])
            for name, r in t["kinds"].items():
                g = agg.setdefault(name, dict(busy_us=0.0, excl_us=0.0, launches=0, bytes=0))
                for f in g:
                    g[f] += r[f]
            for l, r in t["levels"].items():
                lv[l] = lv.get(l, 0.0) + r["excl_us"]
        binding.dovetail_trace_enable(h, False)
        tot_excl = sum(v["excl_us"] for v in agg.values())
        step_tr_us = sum(step_tr) / kp
        scale = (step_ms * 1e3) / (tot_excl / kp) if tot_excl else 0.0  # trace pass -> event-timed step
        g_excl = sum(agg[k]["excl_us"] for k in GEMV_KINDS) / kp * scale
        g_n = sum(agg[k]["launches"] for k in GEMV_KINDS) // kp
        g_b = sum(agg[k]["bytes"] for k in GEMV_KINDS) / kp
        achieved = g_b / (g_excl * 1e-6) / 1e9 if g_excl else 0.0
        by_kind = {}
        for name, v in agg.items():
            if not v["launches"]:
                continue
            us = v["excl_us"] / kp * scale
            by_kind[name] = {"us_per_step": round(us, 2), "launches_per_step": v["launches"] // kp,
                             "us_per_launch": round(us / (v["launches"] / kp), 2),
                             "busy_us_per_launch": round(v["busy_us"] / v["launches"], 2),
                             "gbs": round(v["bytes"] / kp / (us * 1e-6) / 1e9, 1) if v["bytes"] and us else None,
                             "frac_of_measured_peak": round(v["bytes"] / kp / (us * 1e-6) / 1e9 / peak, 3) if v["bytes"] and us else None}
        per_level = [round(lv[l] / kp * scale, 2) for l in sorted(lv)]
        # read-only streaming ceilings, same run, same device buffers (the largest weight matrix set: > L2)
        ceil = {}
        if world == 1:
            big = max((t for l in case.layers for t in (l["wgate"], l["wup"], l["wdown"])), key=lambda t: t.numel())
            pool = torch.empty(max(1 << 30, big.numel() * big.element_size()), dtype=torch.uint8, device="cuda")
            pool.random_(0, 255)
            for name, mode, seg in (("stream_sum_ldg128", 0, 0), ("stream_bulk_1k", 1, 1024), ("stream_bulk_2k", 1, 2048)):
                best = 0.0
                for it in range(6):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    binding.dovetail_probe_stream(h, pool, mode, seg)
                    e1.record(stream)
                    torch.cuda.synchronize()
                    if it >= 1:
                        best = max(best, pool.numel() / (e0.elapsed_time(e1) * 1e-3) / 1e9)
                ceil[name] = round(best, 1)
            del pool
        read_ceiling = max(ceil.values()) if ceil else None
        traffic, traffic_src = None, None
        tp = os.path.join(ROOT, "profiles", "r2_traffic.json.txt")
        if os.path.exists(tp):
            try:
                t = json.load(open(tp)).get(cfg.name)
                if t:  # DRAM bytes per GEMV launch of a committed ncu --set full capture of this very command
                    traffic, traffic_src = t["dram_bytes_per_gemv_launch"], t["source"]
            except Exception:
                traffic = None
        roof = {"bound": "hbm",
                "kernel": "k_gemv_mma (bf16) / k_gemv (fp32): all weight-streaming GEMV launches of the step",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "traffic": traffic, "traffic_source": traffic_src,
                "bytes_per_launch": g_b / g_n if g_n else 0, "us_per_launch": g_excl / g_n if g_n else 0,
                "launches_per_step": g_n, "gemv_share_of_step_time": g_excl / (step_ms * 1e3) if step_ms else None,
                "frac_of_8tbs_nominal": achieved / NOMINAL_HBM_GBS,
                "read_only_ceilings_gbs": ceil, "frac_of_read_only_ceiling": achieved / read_ceiling if read_ceiling else None,
                "by_kind": by_kind, "kinds_sum_us": round(sum(v["us_per_step"] for v in by_kind.values()), 2),
                "trace_step_us": round(step_tr_us, 2),
                "how": "globaltimer stamps per launch (first CTA start, last CTA end), exclusive time per launch, "
                       "scaled so that the kinds add up to the event-timed step; PDL overlap kept"}

    value = world * tree.gamma * K / (ms * 1e-3)
    e2e_val = world * tree.gamma * K / (ms_e2e * 1e-3)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": (("int8" if cfg.wquant == 1 else "fp8 e4m3") + " weights (per-row scales), bf16 KV cache, f32 activations and accumulation" if cfg.wquant else
                      "bf16 weights and KV cache, f32 activations and accumulation") if cfg.dtype == 1 else "f32",
            "data": "synthetic", "config": workload(cfg, a.n_new, world),
            "draft_step_us": step_ms * 1e3, "draft_step_us_replays": dist_us,
            "forward_us": step_ms * 1e3 / tree.depth, "forward_us_per_level": per_level,
            "forwards_per_s": tree.depth / (step_ms * 1e-3),
            "step_hbm_gbs": step_bytes / (step_ms * 1e-3) / 1e9,
            "step_frac_of_measured_peak": step_bytes / (step_ms * 1e-3) / 1e9 / peak,
            "step_frac_of_8tbs_nominal": step_bytes / (step_ms * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
            "algorithmic_bytes_per_step": step_bytes,
            "e2e": {"value": e2e_val, "unit": UNIT, "ms_per_step": ms_e2e / K,
                    "h2d_bytes_per_step": in_h.numel() * 4, "d2h_bytes_per_step": out_h.numel() * 4},
            "gpu_launches": launches, "launch": launch_modes, "clocks": clk, "roofline": roof}

    # ---- prompt / catch-up rows (dovetail_draft_prefill), batches of 64 rows -----------------
    if a.prefill_rows > 0 and world == 1 and cfg.dtype == 1 and not cfg.wquant:
        Rp = a.prefill_rows
        shp = list(case.k.shape)
        shp[2] = case.L + Rp + 8
        k2, v2 = torch.zeros(shp, dtype=case.k.dtype, device="cuda"), torch.zeros(shp, dtype=case.v.dtype, device="cuda")
        k2[:, :, :case.L], v2[:, :, :case.L] = case.k[:, :, :case.L], case.v[:, :, :case.L]
        kv2 = binding.KVCache(k2, v2, case.L)
        g = torch.Generator(device="cuda").manual_seed(cfg.seed + 7)
        pf = (torch.randn((Rp, cfg.hidden), generator=g, device="cuda") * cfg.feat_scale).to(torch.bfloat16).float()
        pt = torch.randint(0, cfg.vocab, (Rp,), generator=g, device="cuda", dtype=torch.int32)

        def pre():
            kv2.committed_len = case.L
            binding.dovetail_draft_prefill(h, pf, pt, kv2)
        for _ in range(3):
            pre()
        reps = 5
        ms_p = timed(pre, reps) / reps
        passes = -(-Rp // 64)
        wbytes = binding.dovetail_forward_bytes(h, 0) - cfg.vocab * cfg.hidden * 2  # one pass over the block weights, no LM head
        line["prefill"] = {"rows": Rp, "batch_rows": 64, "ms": ms_p, "rows_per_s": Rp / (ms_p * 1e-3),
                           "weight_passes": passes, "hbm_gbs_weights": passes * wbytes / (ms_p * 1e-3) / 1e9,
                           "umma_launches": binding.dovetail_hooks_stat(h, binding.STAT_UMMA_LAUNCHES),
                           "note": "each 64-row batch streams the block weights once through the tcgen05 GEMV (weight-streaming "
                                   "bound at 64 rows per pass, not yet a tile-reuse GEMM)"}
        del k2, v2

    # ---- what the verifier needs from the step and the acceptance rule (+ kv_commit) ----------
    # Device time of each call on the last step's candidates; synthetic target answers (a seeded distribution per
    # verifier row). Pre-built argument structs: the loop times the library's kernels, not tensor allocation.
    if a.verify_leg and world == 1:
        import ctypes as C
        lib, g1, md = binding.load(), tree.gamma + 1, tree.depth
        step_device()
        torch.cuda.synchronize()
        gen = torch.Generator(device="cuda").manual_seed(cfg.seed + 11)
        par, tok = out["parents"][:tree.gamma].long(), out["token_ids"][:tree.gamma].long()
        logits_t = torch.randn((g1, cfg.vocab), generator=gen, device="cuda") * 3.0
        logits_t[par + 1, tok] += 12.0  # a target that mostly agrees with the draft: paths of several nodes get accepted
        p_full = torch.softmax(logits_t, dim=-1).contiguous()
        p_cand = p_full[par + 1, tok].contiguous()  # candidate i's token at its parent's row
        tgt_argmax = p_full.argmax(dim=-1).to(torch.int32)
        unif = torch.rand(g1, generator=gen, device="cuda")
        plan = dict(mask=torch.zeros((g1, g1), dtype=torch.uint8, device="cuda"), pos=torch.zeros(g1, dtype=torch.int32, device="cuda"),
                    paths=torch.zeros((tree.gamma, md), dtype=torch.int32, device="cuda"), n=torch.zeros(1, dtype=torch.int32, device="cuda"))
        res = dict(path=torch.full((md,), -1, dtype=torch.int32, device="cuda"), n=torch.zeros(1, dtype=torch.int32, device="cuda"),
                   bonus=torch.zeros(1, dtype=torch.int32, device="cuda"))
        o_t = binding._out_t(out)
        plan_t = binding.VerifyPlanT(*(binding._dp(plan[k]) for k in ("mask", "pos", "paths", "n")))
        in_t = binding.VerifyInT(binding._dp(tgt_argmax), binding._dp(p_cand), binding._dp(unif), binding._dp(p_full))
        res_t = binding.VerifyOutT(binding._dp(res["path"]), binding._dp(res["n"]), binding._dp(res["bonus"]))
        sp = binding._stream(None)
        calls = {"verify_plan_us": lambda: lib.dovetail_verify_plan(h.ptr, C.byref(o_t), tree.gamma, case.L, md, C.byref(plan_t), sp),
                 "verify_accept_greedy_us": lambda: lib.dovetail_verify_accept(h.ptr, C.byref(o_t), tree.gamma, 0, md, C.byref(in_t), C.byref(res_t), sp),
                 "verify_accept_sampling_us": lambda: lib.dovetail_verify_accept(h.ptr, C.byref(o_t), tree.gamma, 1, md, C.byref(in_t), C.byref(res_t), sp)}
        vleg = {}
        for name, fn in calls.items():
            for _ in range(3):
                assert fn() == 0, binding.dovetail_last_error(h)
            vleg[name] = timed(fn, 50) / 50 * 1e3
        torch.cuda.synchronize()
        n_acc = int(res["n"].item())
        path = [int(x) for x in res["path"][:n_acc].tolist()]

        if n_acc > 0:  # a commit consumes its step: one step per commit, events around the commit alone
            ts = []
            for it in range(13):
                step_device()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                binding.dovetail_kv_commit(h, kv, path, mode=1)  # plan + row moves + the host's read of the committed count
                e1.record(stream)
                torch.cuda.synchronize()
                if it >= 3:
                    ts.append(e0.elapsed_time(e1) * 1e3)
            vleg["kv_commit_us"] = sorted(ts)[len(ts) // 2]
        vleg.update(accepted_by_sampling=n_acc, note="synthetic target distributions, candidates of the last step; events around 50 back-to-back calls, so a figure of a few us is an upper bound set by the host's call rate, not the kernel's own time; kv_commit includes its read-back of the committed count")
        line["verify"] = vleg
        step_device()  # the commit moved cache rows of the tree region: leave the cache as a step leaves it

    # ---- reading A1 "report both": the same step with dgf_proj = 0 (W1 = W2 = I) ----------------------------
    if a.both_dgf and world == 1 and cfg.dgf_proj == 1 and cfg.fusion == 0:
        cfg0 = dataclasses.replace(cfg, dgf_proj=0)
        top0 = dict(case.top, dgf_w1=None, dgf_w2=None)
        h0 = binding.dovetail_draft_init(top0, case.layers, cfg0)
        for _ in range(W):
            step_device(h0)
        ms0 = timed(lambda: step_device(h0), K)
        b0 = tree.depth * binding.dovetail_forward_bytes(h0, case.L + a.n_new)
        line["dgf_proj0"] = {"ms_per_step": ms0 / K, "value": tree.gamma * K / (ms0 * 1e-3),
                             "step_frac_of_measured_peak": b0 / (ms0 / K * 1e-3) / 1e9 / peak,
                             "step_frac_of_8tbs_nominal": b0 / (ms0 / K * 1e-3) / 1e9 / NOMINAL_HBM_GBS}
        binding.dovetail_draft_destroy(h0)

    if rank == 0 and world == 1 and not a.no_cpu_baseline:
        hc = _to_host(case)
        cores = len(os.sched_getaffinity(0))
        t_all, sample_all = oracle_sample(hc, full_step=True)
        one = None
        if set_omp_threads(1):
            t1, sample1 = oracle_sample(hc, full_step=False)
            one = {"seconds_per_step": t1, "value": tree.gamma / t1, "sample": sample1}
            set_omp_threads(cores)
        line["cpu_baseline"] = {"value": tree.gamma / t_all, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": sample_all, "seconds_per_step": t_all, "cpu_model": cpu_model(),
                                "one_thread": one,
                                "paper_context": "PAPER.md:70 T_D = 7.2 ms per forward (5 blocks, RTX 2080 SUPER, fp16); "
                                                 "PAPER.md:9 1.79x-10.1x end-to-end speedups (context only)"}
    binding.dovetail_draft_destroy(h)
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="c3")
    ap.add_argument("--n-new", type=int, default=1)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--replays", type=int, default=200)
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="A/B knob of include/dovetail_hooks.h dovetail_hooks_tune (repeatable)")
    ap.add_argument("--prefill-rows", type=int, default=256, help="rows of the dovetail_draft_prefill leg (0: skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-trace", action="store_true")
    ap.add_argument("--no-verify-leg", dest="verify_leg", action="store_false", help="skip the verify_plan / verify_accept / kv_commit timings")
    ap.add_argument("--no-both-dgf", dest="both_dgf", action="store_false")
    a = ap.parse_args()
    rank, world, local = dist_env()

    if a.impl == "reference":
        if rank != 0:
            return
        print(json.dumps(reference_line(a, all_configs()[a.config if a.config != "all" else "c3"])))
        return

    if "WORLD_SIZE" not in os.environ and a.gpus > 1:
        # not under torchrun: spawn the N replica ranks ourselves
        s = socket.socket()
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
        s.close()
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={a.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if a.gpus != world:
        sys.exit(f"bench.py: --gpus {a.gpus} disagrees with WORLD_SIZE={world} of the launcher")

    import torch
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU path)"
    from paper_2412_18934_b200 import binding
    binding.load()  # fail loudly if the library is missing
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfgs = all_configs()
    if a.config == "all":
        names = ["c1", "c2", "c5", "c2_int8", "c3_int8", "c5_int8", "c2_fp8", "c3_fp8", "c5_fp8", "c2_paper_tree", "c3_paper_tree"] + [n for n in cfgs if n.startswith("c4_") or n.startswith("depth_")] + ["c3"]
    else:
        names = [a.config]
    for i, name in enumerate(names):
        last = i == len(names) - 1
        if not last:  # the sweep lines carry the step numbers only
            aa = argparse.Namespace(**vars(a))
            aa.no_cpu_baseline, aa.both_dgf, aa.replays, aa.prefill_rows = True, False, 0, 0
        else:
            aa = a
        line = bench_one(aa, cfgs[name], rank, world, local, dist)
        if rank == 0:
            print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

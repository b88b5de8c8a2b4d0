#!/usr/bin/env python
"""bench.py — CAEE MoE-layer decode throughput on B200 (one JSON line on stdout).

A "step" is one pass of the whole hot path (router -> cost lookup -> cost-aware prune ->
compensation -> compaction -> grouped SwiGLU FFN over the surviving experts -> combine) over
one batch of synthetic tokens, through the C ABI (caee_moe_forward).  Default workload:
BASELINE.json config 3, the DeepSeek-R1-shaped bf16 layer (H 7168, 256+1 experts, top-8,
I 2048, 22.5 GB of expert weights in HBM) at a 128-token decode batch.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3] [--tokens 128]
                    [--prune thresh:0.6] [--impl caee|reference]

N > 1 (under torchrun) runs N independent replicas ("replicas only").
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "moe_layer_decode_tokens_per_s"
UNIT = "tokens/s"
MODE_IDS = {"none": 0, "thresh": 1, "cir": 2, "rank": 3, "frac": 4}


def parse_prune(s):
    if s in ("dense", "off"):
        return None
    name, _, val = s.partition(":")
    return MODE_IDS[name], float(val or 0)


def workload_name(cfg, T, prune):
    p = "dense top-k" if prune is None else f"CAEE prune {prune}"
    return (f"{cfg.name}: H={cfg.H} I={cfg.I} E={cfg.E}+{cfg.S} top-{cfg.k} groups {cfg.n_group}/{cfg.topk_group} "
            f"D={cfg.D}, decode batch T={T}, {p}")


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def tensor_peak():
    """Dense 16-bit tensor peak in TFLOP/s for a kernel timed inside a long step (the sustained figure)."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        if "bf16_tflops_sustained" in d:
            return float(d["bf16_tflops_sustained"]), "measured (MEASURED_PEAKS.json bf16_tflops_sustained; fp16 = bf16 rate)"
    return 2250.0, "fallback (nominal dense bf16/fp16 2.25 PFLOP/s)"


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "10",
                                       "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out = self.p.communicate(timeout=5)[0]
        except subprocess.TimeoutExpired:
            self.p.kill()
            out = self.p.communicate()[0]
        sm, mx, reasons = [], [], set()
        for line in out.strip().splitlines():
            f = [v.strip() for v in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# --------------------------------------------------------------------------- CPU oracle legs
def oracle_sample_run(cfg, T, prune, seed, n_sample, device_for_inputs, layer=None, min_seconds=0.0):
    """Times the oracle as it stands on the host cores: decisions on all T tokens, FFN + combine on
    n_sample of them; returns (tokens_per_s extrapolated to T, seconds of CPU work, cores)."""
    import numpy as np
    from oracle import oracle as orc
    from paper_2606_29982_b200 import workloads as wl
    cores = len(os.sched_getaffinity(0))
    x = wl.hidden(cfg, T, seed + 100, device_for_inputs)
    Wr, b_logit, cb = (layer.Wr, layer.b_logit, layer.corr_bias) if layer is not None else wl.router(cfg, seed, device_for_inputs)
    xb, Wr_h, b_h = wl.bits(x), Wr.cpu().numpy(), b_logit.cpu().numpy()
    cb_h = None if cb is None else cb.cpu().numpy()
    part = wl.partitions(cfg)
    w_eff = orc.effective_cost(wl.residency(cfg, seed), *wl.cost_tables(cfg))
    t0 = time.perf_counter()
    s = orc.scores(xb, Wr_h, b_h, cfg.score_fn)
    idx, gate = orc.route(s, cb_h, cfg.k, cfg.n_group, cfg.topk_group, cfg.norm_topk)
    if prune is not None:
        pr = orc.prune(prune[0], prune[1], 0, idx, gate, cfg.E, w_eff, part, cfg.D)
        if prune[0] != 0:
            idx, gate = orc.compensate(s, cb_h, pr["keep"], idx, gate, cfg.norm_topk, 0)
    orc.compact(idx, gate, cfg.E)
    t_dec = time.perf_counter() - t0
    tokens = list(range(0, T, max(1, T // n_sample)))[:n_sample]
    n = cfg.E + cfg.S
    used = sorted(set(int(e) for t in tokens for e in idx[t] if e >= 0) | set(range(cfg.E, n)))
    tabs = {k: [None] * n for k in ("gate", "up", "down", "gate_scale", "up_scale", "down_scale")}
    for e in used:                                   # untimed: fetch the exact bits of the needed experts
        r = wl.expert_weights(cfg, seed, e, device_for_inputs)
        for k_, v in r.items():
            tabs[k_][e] = wl.bits(v)
    fp8 = cfg.w_dtype == wl.DT_E4M3
    reps, t_all = 0, 0.0
    while reps == 0 or (t_all < min_seconds and reps < 64):    # repeat the same sample up to the time budget
        t0 = time.perf_counter()
        orc.moe_tokens(xb, tokens, idx, gate, tabs["gate"], tabs["up"], tabs["down"], cfg.E, cfg.S, cfg.routed_scale,
                       tabs["gate_scale"] if fp8 else None, tabs["up_scale"] if fp8 else None,
                       tabs["down_scale"] if fp8 else None)
        t_all += time.perf_counter() - t0
        reps += 1
    t_ffn = t_all / reps
    total = t_dec + t_ffn * T / len(tokens)
    return T / total, t_dec + t_all, cores, len(tokens)


def run_reference(args, cfg, prune):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores (rank 0 only)."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    T = args.tokens
    n_sample = 1
    vals, secs = [], []
    for i in range(args.warmup + args.steps):
        v, sec, cores, ns = oracle_sample_run(cfg, T, prune, 0, n_sample, "cpu")
        if i >= args.warmup:
            vals.append(v)
            secs.append(sec)
    value = statistics.mean(vals)
    sample = (f"per step: oracle decisions on all {T} tokens + FFN/combine on {n_sample} token(s), extrapolated linearly "
              f"to {T} tokens; inputs drawn on the CPU generator")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * T / value, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, T, args.prune)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def job_throughput(ms_local, tokens_local, world, device):
    """Whole-job tokens/s of N independent replicas: every rank's tokens over the
    slowest rank's time.  The only collective of the whole program is this timing reduction."""
    if world == 1:
        return tokens_local / (ms_local * 1e-3), ms_local
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    n = torch.tensor([float(tokens_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(n.item()) / (float(t.item()) * 1e-3), float(t.item())


# --------------------------------------------------------------------------- the CUDA arm
def run_caee(args, cfg, prune):
    import torch
    from paper_2606_29982_b200 import binding as B
    from paper_2606_29982_b200 import workloads as wl
    from paper_2606_29982_b200.layer import Layer

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libcaee has no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))
    T, K, W = args.tokens, args.steps, max(args.warmup, 3)
    L = Layer(cfg, seed=rank, max_tokens=max(T, 128), device=dev)
    params = None if prune is None else B.prune_params(prune[0], prune[1])
    xs = [wl.hidden(cfg, T, rank * 1000 + 100 + i, dev) for i in range(4)]      # rotate a few batches
    y = torch.empty_like(xs[0])
    stats = B.stats_buffer(dev)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, finish=None):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(steps):
            fn(i)
        if finish is not None:
            finish()          # e.g. make the timing stream wait for copies still running on side streams
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        return job_throughput(ms, T * steps, world, dev)[1]      # max over ranks

    step = lambda i: L.forward(xs[i % len(xs)], params, y=y, stats=stats)
    for i in range(W):
        step(i)
    torch.cuda.synchronize()
    # the batches rotate and each keeps a different number of experts: note, per batch, the
    # weight bytes its expert-kernel launch streams (untimed; caee_fwd_stats.weight_bytes)
    batch_bytes = []
    for i in range(len(xs)):
        step(i)
        torch.cuda.synchronize()
        batch_bytes.append(B.read_stats(stats).weight_bytes)
    # --- device-resident timing, with the expert kernel timed by its own event pair
    B.caee_profile(L.ctx, K)
    clocks = ClockSampler(local)
    ms_total = timed(step, K)
    clk = clocks.stop()
    expert_ms = B.caee_profile_read(L.ctx, K)
    B.caee_profile(L.ctx, 0)
    st = B.read_stats(stats)
    ms_step = ms_total / K
    value = world * T / (ms_step * 1e-3)

    # --- end to end through the public call with HOST buffers (caee_moe_forward_host): every step
    # copies its x from pinned host memory and its y back inside the timed region.  The library
    # runs the copies on two side streams with double-buffered device tensors, so step i's D2H and
    # step i+1's H2D overlap the layer's compute; the timed region ends only after the last step's
    # y has landed in host memory (caee_host_flush).
    xh = [x.cpu().pin_memory() for x in xs]
    yh = torch.empty_like(xh[0]).pin_memory()

    def e2e_step(i):
        B.caee_moe_forward_host(L.ctx, xh[i % len(xh)], T, params, yh)

    def e2e_finish():
        B.caee_host_flush(L.ctx)

    for i in range(4):
        e2e_step(i)
    ms_e2e = timed(e2e_step, K, finish=e2e_finish) / K
    e2e_value = world * T / (ms_e2e * 1e-3)
    nbytes = xs[0].numel() * xs[0].element_size()

    # --- dense (no pruning) beside it, same batches
    dense_ms = timed(lambda i: L.forward(xs[i % len(xs)], None, y=y, stats=stats), K) / K
    st_dense = B.read_stats(stats)

    if rank != 0:
        L.close()
        return
    peak, peak_src = peaks()
    k_ms = float(statistics.mean(expert_ms)) if len(expert_ms) else None
    launch_bytes = [batch_bytes[i % len(xs)] for i in range(len(expert_ms))]     # launch i ran batch i % 4
    bytes_per_launch = float(statistics.mean(launch_bytes)) if launch_bytes else None
    achieved = bytes_per_launch / (k_ms * 1e-3) / 1e9 if k_ms else None
    # dram bytes per launch from the committed ncu --set full capture of this same command
    # (profiles/traffic.json, written from the .ncu-rep by hand; null when not captured)
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            traffic = json.load(f).get(f"{cfg.name}/T{T}/{args.prune}", {}).get("dram_bytes_per_launch")
    fp8 = cfg.w_dtype == wl.DT_E4M3
    if T <= 256:
        # k_router_logits, k_decide (S1-S6 + stats in one cooperative kernel), [k_act_split], expert kernel, k_combine
        launches_per_step = 2 + (1 if fp8 else 0) + 1 + 1
    else:
        # stand-alone decision kernels: logits, top-k, [prune, compensate], count/scan/fill, [split], expert, combine, stats
        n_prune = 0 if prune is None else (1 if T <= 512 else 2)      # k_prune, or k_prune_accum + k_prune_from_acc
        launches_per_step = 2 + n_prune + (1 if prune is not None and prune[0] != 0 else 0) + 3 + (1 if fp8 else 0) + 1 + 1 + 1
    if cfg.n_resident >= 0:
        launches_per_step += 1 + st.n_fetch          # k_stats + one expert launch per fetched expert (C5)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {0: "f32", 1: "bf16", 2: "fp8_e4m3"}[cfg.w_dtype], "data": "synthetic",
        "config": {"workload": workload_name(cfg, T, args.prune), "l2": "inputs larger than L2: each step streams "
                   f"{st.weight_bytes / 1e9:.2f} GB of expert weights (L2 is 126 MB)", "parallelism": "replicas only",
                   "seed": 0},
        "clocks": clk,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "call": "caee_moe_forward_host: x from pinned host memory, y back to it, every step; copies double-buffered on two side streams",
                "ms_per_step": ms_e2e},
        "gpu_launches": launches_per_step * K,
        "roofline": {"bound": "hbm", "kernel": "k_expert_fp8" if fp8 else "k_expert_umma", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak if achieved else None, "traffic": traffic, "peak_source": peak_src,
                     "bytes_per_launch": bytes_per_launch, "kernel_ms": k_ms,
                     "bytes_by_batch": batch_bytes,
                     "frac_of_8TBps_nominal": achieved / 8000.0 if achieved else None},
        "latency_us": {"pruned": ms_step * 1e3, "dense": dense_ms * 1e3, "expert_kernel": k_ms * 1e3 if k_ms else None},
        "pruning": {"n_act": st.n_act, "n_keep": st.n_keep, "n_run": st.n_run, "F_cost_dense": st.F_cost_dense,
                    "F_cost": st.F_cost, "bytes_pruned": st.weight_bytes, "bytes_dense": st_dense.weight_bytes,
                    "n_run_dense": st_dense.n_run},
    }
    if fp8 and T > 256:
        # prefill-size e4m3 step: k_expert_fp8_wide (fp16 MMAs) is bound by the tensor pipe / its
        # shared-memory operand feed, not by HBM: report useful flops against the 16-bit tensor peak
        tpeak, tsrc = tensor_peak()
        flops = 6.0 * cfg.H * cfg.I * T * (cfg.k + cfg.S)      # every token keeps k routed slots + S shared
        tf = flops / (k_ms * 1e-3) / 1e12 if k_ms else None
        out["roofline"].update({"bound": "tensor", "kernel": "k_expert_fp8_wide", "achieved": tf, "peak": tpeak,
                                "unit": "TFLOP/s", "frac": tf / tpeak if tf else None, "peak_source": tsrc,
                                "flops_per_launch": flops, "hbm_gbs": achieved})
        out["roofline"].pop("frac_of_8TBps_nominal", None)
    if world == 1 and not args.no_cpu_baseline:
        try:
            import psutil
            ram_gb = psutil.virtual_memory().available / 2 ** 30
        except Exception:
            ram_gb = 16.0
        n_sample = max(1, min(16, int((ram_gb * 0.4) / (cfg.expert_bytes * cfg.k / 2 ** 30 + 1e-9))))
        L.close()
        torch.cuda.empty_cache()
        v, sec, cores, ns = oracle_sample_run(cfg, T, prune, 0, n_sample, dev, min_seconds=10.0)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"oracle decisions on all {T} tokens + FFN/combine on {ns} of them, repeated "
                                         f"for {sec:.1f} s of CPU work and averaged, extrapolated linearly to {T} tokens"}
    else:
        L.close()
    print(json.dumps(out))


# --------------------------------------------------------------------------- NEXT-1: LFU cache decode loop
def run_cache_loop(args, cfg):
    """SURVEY.md §8(f) NEXT-1 (Table II): a multi-layer decode loop over an LFU expert
    cache.  Every routed expert of every layer lives in pinned host memory; `--cache-slots` device
    slots are shared by the layers.  The settings (dense baseline, CIR theta_imp = 0.9 / 0.8 / 0.7) run
    one after the other on the same cache; each is warmed for --warmup steps (which re-converges the
    cache contents to that setting) and timed for --steps steps (one step = T tokens through all
    layers, the same token batches for every setting); reported: ms per step (the TPOT proxy), misses and H2D bytes per step, the
    achieved H2D rate.  Synthetic stand-in for the paper's 58-layer DeepSeek-R1 run: layers share the
    layer shape and differ in router and weights (seeds), token batches change every step."""
    import torch
    from paper_2606_29982_b200 import binding as B
    from paper_2606_29982_b200 import workloads as wl
    from paper_2606_29982_b200.layer import Layer

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libcaee has no CPU fallback")
    torch.cuda.set_device(0)
    dev = "cuda:0"
    T, K, W, NL = args.tokens, args.steps, max(args.warmup, 3), args.layers
    cache = B.caee_cache_create(args.cache_slots)
    layers = [Layer(cfg, seed=l, max_tokens=max(T, 16), device=dev, cache=cache, layer_id=l) for l in range(NL)]
    xs = [wl.hidden(cfg, T, 5000 + i, dev) for i in range(W + K)]
    y = torch.empty_like(xs[0])
    stats = B.stats_buffer(dev)
    stream = torch.cuda.current_stream()
    rows = []
    try:
        for name, params in (("dense", None), ("cir:0.9", B.prune_params(2, 0.9)), ("cir:0.8", B.prune_params(2, 0.8)),
                             ("cir:0.7", B.prune_params(2, 0.7))):
            def step(i):
                h = xs[i]
                for L in layers:
                    L.forward(h, params, y=y, stats=stats)     # x -> every layer (layers are independent MoE blocks here)
            for i in range(W):
                step(i)
            torch.cuda.synchronize()
            c0 = B.caee_cache_read_stats(cache)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for i in range(W, W + K):
                step(i)
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / K
            c1 = B.caee_cache_read_stats(cache)
            miss, hit = (c1.misses - c0.misses) / K, (c1.hits - c0.hits) / K
            h2d = (c1.h2d_bytes - c0.h2d_bytes) / K
            rows.append({"setting": name, "ms_per_step": ms, "misses_per_step": miss, "hits_per_step": hit,
                         "h2d_gb_per_step": h2d / 1e9, "h2d_gbs": h2d / (ms * 1e-3) / 1e9})
    finally:
        for L in layers:
            L.close()
        B.caee_cache_destroy(cache)
    base = rows[0]["ms_per_step"]
    for r in rows:
        r["vs_dense"] = r["ms_per_step"] / base
    print(json.dumps({
        "metric": "cached_decode_step_ms", "value": rows[2]["ms_per_step"], "unit": "ms/step", "n_gpus": 1, "steps": K,
        "warmup": W, "higher_is_better": False, "vs_baseline": None, "dtype": {0: "f32", 1: "bf16", 2: "fp8_e4m3"}[cfg.w_dtype],
        "data": "synthetic",
        "config": {"workload": f"{cfg.name}: {NL} layers x (E={cfg.E}+{cfg.S}, H={cfg.H}, I={cfg.I}, top-{cfg.k}), LFU cache of "
                               f"{args.cache_slots} slots x {cfg.expert_bytes / 1e6:.1f} MB, T={T} tokens per step; value = CIR 0.8"},
        "roofline": {"bound": "pcie", "achieved": rows[0]["h2d_gbs"], "unit": "GB/s", "peak": 55.6,
                     "peak_source": "caee_calibrate_cost H2D tier on this pool's B200 (DESIGN.md §4)",
                     "frac": rows[0]["h2d_gbs"] / 55.6, "traffic": None},
        "rows": rows}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="caee", choices=["caee", "reference"])
    ap.add_argument("--workload", default="c3", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--tokens", type=int, default=128)
    ap.add_argument("--prune", default="thresh:0.6", help="dense | none | thresh:θ | cir:θ_imp | rank:b | frac:p")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cache-loop", action="store_true", help="SURVEY §8(f) NEXT-1: multi-layer decode loop over an LFU expert cache")
    ap.add_argument("--layers", type=int, default=2)
    ap.add_argument("--cache-slots", type=int, default=128)
    args = ap.parse_args()
    from paper_2606_29982_b200 import workloads as wl
    cfg = wl.CONFIGS[args.workload.upper()]
    prune = parse_prune(args.prune)
    if args.cache_loop:
        run_cache_loop(args, cfg)
    elif args.impl == "reference":
        run_reference(args, cfg, prune)
    else:
        run_caee(args, cfg, prune)


if __name__ == "__main__":
    main()

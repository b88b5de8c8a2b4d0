#!/usr/bin/env python
"""bench.py — CAEE MoE-layer decode throughput on B200 (one JSON line on stdout).

A "step" is one pass of the whole hot path (router -> cost lookup -> cost-aware prune ->
compensation -> compaction -> grouped SwiGLU FFN over the surviving experts -> combine) over
one batch of synthetic tokens, through the C ABI (caee_moe_forward).  Default workload:
BASELINE.json config 3, the DeepSeek-R1-shaped bf16 layer (H 7168, 256+1 experts, top-8,
I 2048, 22.5 GB of expert weights in HBM) at a 128-token decode batch.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3] [--tokens 128]
                    [--prune thresh:0.6] [--eps-frac 0.10] [--impl caee|reference]

Default operating point: the paper's on-device knob THRESH theta = 0.6 under the objective's
importance bound F_imp <= eps with eps = 0.10 T (R37): at most 10% of the batch's
gate mass may be re-routed, the batch-level counterpart of the paper's theta_imp = 0.9 retention point
(Table III).  `value` is that step; the same batches without pruning are reported beside it
under "dense".

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


def workload_name(cfg, T, prune, eps=None):
    p = "dense top-k" if prune in (None, "dense", "off") else f"CAEE prune {prune}"
    if eps is not None and prune not in (None, "dense", "off"):
        p += f" under the importance bound F_imp <= {eps:g} (= {eps / T:g} T, PAPER.md:150-152)"
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
class OracleLayer:
    """The CPU oracle on the bench workload, as it stands: one timed call = the whole layer step on ALL T
    tokens (scores -> route -> prune -> compensation -> compaction -> expert FFNs -> combine).  Set-up
    (drawing x, the router and the exact bits of the experts the step touches) is not timed."""

    def __init__(self, cfg, T, prune, eps, seed, device, layer=None):
        import numpy as np
        from oracle import oracle as orc
        from paper_2606_29982_b200 import workloads as wl
        self.cfg, self.T, self.prune, self.eps, self.orc, self.wl, self.np = cfg, T, prune, eps, orc, wl, np
        self.cores = len(os.sched_getaffinity(0))
        x = wl.hidden(cfg, T, seed * 1000 + 100, device)
        Wr, b_logit, cb = (layer.Wr, layer.b_logit, layer.corr_bias) if layer is not None else wl.router(cfg, seed, device)
        self.xb, self.Wr, self.b = wl.bits(x), Wr.cpu().numpy(), b_logit.cpu().numpy()
        self.cb = None if cb is None else cb.cpu().numpy()
        self.part = wl.partitions(cfg)
        tables = (layer.ticks_res, layer.ticks_miss) if layer is not None else wl.cost_tables(cfg)     # the layer's may be calibrated
        self.w_eff = orc.effective_cost(wl.residency(cfg, seed), *tables)
        idx, _ = self.decisions()[:2]
        n = cfg.E + cfg.S
        used = sorted(set(int(e) for e in idx.ravel() if e >= 0) | set(range(cfg.E, n)))
        self.tabs = {k: [None] * n for k in ("gate", "up", "down", "gate_scale", "up_scale", "down_scale")}
        for e in used:                                   # untimed: the exact bits of the needed experts
            for k_, v in wl.expert_weights(cfg, seed, e, device).items():
                self.tabs[k_][e] = wl.bits(v)
        self.n_experts = len(used)

    def decisions(self):
        orc, cfg = self.orc, self.cfg
        s = orc.scores(self.xb, self.Wr, self.b, cfg.score_fn)
        idx, gate = orc.route(s, self.cb, cfg.k, cfg.n_group, cfg.topk_group, cfg.norm_topk)
        if self.prune is not None:
            flags = orc.FLAG_IMP_BOUND if self.eps is not None else 0
            pr = orc.prune(self.prune[0], self.prune[1], flags, idx, gate, cfg.E, self.w_eff, self.part, cfg.D,
                           eps=0.0 if self.eps is None else self.eps)
            if self.prune[0] != 0:
                idx, gate = orc.compensate(s, self.cb, pr["keep"], idx, gate, cfg.norm_topk, 0)
        c = orc.compact(idx, gate, cfg.E)
        return idx, gate, c

    def step(self):
        """One full layer step; returns the seconds it took."""
        cfg, t = self.cfg, self.tabs
        fp8 = cfg.w_dtype == self.wl.DT_E4M3
        t0 = time.perf_counter()
        idx, gate, _ = self.decisions()
        self.orc.moe_tokens(self.xb, list(range(self.T)), idx, gate, t["gate"], t["up"], t["down"], cfg.E, cfg.S, cfg.routed_scale,
                            t["gate_scale"] if fp8 else None, t["up_scale"] if fp8 else None, t["down_scale"] if fp8 else None)
        return time.perf_counter() - t0


def oracle_sample_text(o, reps):
    return (f"the whole layer step on all {o.T} tokens ({o.n_experts} experts' weights touched), oracle as it stands "
            f"(g++ -O2, OpenMP over the FFN rows), {reps} timed repetition(s), nothing extrapolated")


def run_reference(args, cfg, prune, eps):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores (rank 0 only)."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    import torch
    T = args.tokens
    dev = "cuda:0" if torch.cuda.is_available() else "cpu"      # inputs only: the experts' bits are drawn where it is fast
    o = OracleLayer(cfg, T, prune, eps, 0, dev)
    secs = []
    for i in range(args.warmup + args.steps):
        sec = o.step()
        if i >= args.warmup:
            secs.append(sec)
    ms = 1e3 * statistics.mean(secs)
    value = T / (ms * 1e-3)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, T, args.prune, eps)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": o.cores, "kind": "oracle", "sample": oracle_sample_text(o, len(secs))},
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
def run_caee(args, cfg, prune, eps):
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
    calib = None
    if args.calibrate or cfg.n_resident >= 0:
        # C5's two-tier cost table always comes from caee_calibrate_cost on the box
        hbm, h2d = L.calibrate()
        calib = {"hbm_gbs": hbm.gbytes_per_s, "hbm_overhead_ns": hbm.intercept_ns, "h2d_gbs": h2d.gbytes_per_s,
                 "h2d_overhead_ns": h2d.intercept_ns, "ticks_resident": int(L.ticks_res.min()), "ticks_miss": int(L.ticks_miss.min())}
    params = None if prune is None else B.prune_params(prune[0], prune[1], 0, eps)
    xs = [wl.hidden(cfg, T, rank * 1000 + 100 + i, dev) for i in range(4)]      # rotate a few batches
    y = torch.empty_like(xs[0])
    stats = B.stats_buffer(dev)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    flush = {"buf": None}          # set below for steps that stream less than twice the L2

    def timed(fn, steps, finish=None):
        barrier()
        if flush["buf"] is not None:
            # small step: its weights could stay in the 126 MB L2 from one iteration to the next, so every step is
            # timed by its own event pair and a 256 MB write between the pairs (untimed) flushes the L2
            pairs = []
            for i in range(steps):
                flush["buf"].zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                fn(i)
                if finish is not None and i == steps - 1:
                    finish()
                b.record(stream)
                pairs.append((a, b))
            barrier()
            return job_throughput(sum(a.elapsed_time(b) for a, b in pairs), T * steps, world, dev)[1]
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
    batch_bytes, batch_h2d = [], []
    for i in range(len(xs)):
        step(i)
        torch.cuda.synchronize()
        batch_bytes.append(B.read_stats(stats).weight_bytes)
        batch_h2d.append(B.read_stats(stats).h2d_bytes)
    L2_BYTES = 126e6
    if max(batch_bytes) < 2 * L2_BYTES:
        flush["buf"] = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    # --- device-resident timing, with the expert kernel timed by its own event pair
    B.caee_profile(L.ctx, K)
    clocks = ClockSampler(local)
    n0 = B.caee_launch_count(L.ctx)
    ms_total = timed(step, K)
    gpu_launches = B.caee_launch_count(L.ctx) - n0       # counted by the library at its launch sites
    clk = clocks.stop()
    offload_t = B.caee_profile_read_offload(L.ctx, K) if cfg.n_resident >= 0 else None   # before caee_profile_read (it rewinds)
    expert_ms = B.caee_profile_read(L.ctx, K)
    B.caee_profile(L.ctx, 0)
    st = B.read_stats(stats)
    ms_step = ms_total / K
    value = world * T / (ms_step * 1e-3)
    # the same K steps without the event pair around the expert kernel (an event recorded between two kernels switches
    # their programmatic-dependent-launch overlap off): what a caller gets; `value` stays the conservative, profiled one
    ms_plain = timed(step, K) / K

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
    # DRAM bytes per launch of the dominant kernel: from the committed ncu --set full capture of this same
    # command (profiles/traffic.json, written by paper_2606_29982_b200.profile_summary from the .ncu-rep at the
    # commit it names); null when this workload was not captured
    traffic, traffic_src = None, None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            ent = json.load(f).get(f"{cfg.name}/T{T}/{args.prune}" + (f"/eps{args.eps_frac:g}T" if eps is not None else ""), {})
        traffic = ent.get("dram_bytes_per_launch")
        if traffic is not None:
            traffic_src = f"committed ncu capture at commit {ent.get('commit', '?')} (profiles/traffic.json), {ent.get('launches', '?')} launches averaged"
    fp8 = cfg.w_dtype == wl.DT_E4M3
    dense_value = world * T / (dense_ms * 1e-3)
    removed = 1.0 - st.weight_bytes / st_dense.weight_bytes if st_dense.weight_bytes else 0.0
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {0: "f32", 1: "bf16", 2: "fp8_e4m3"}[cfg.w_dtype], "data": "synthetic",
        "config": {"workload": workload_name(cfg, T, args.prune, eps) +
                               f"; last batch: {100 * removed:.0f}% of the dense step's expert bytes removed, "
                               f"F_imp = {st.F_imp / 2.0 ** 40:.2f} of {T} (gate units)",
                   "l2": (f"L2 flushed between timed iterations (a 256 MB write, untimed; every step has its own event pair): a step streams only "
                          f"{st.weight_bytes / 1e6:.0f} MB of expert weights (L2 is 126 MB)") if flush["buf"] is not None else
                         ("inputs larger than L2: each step streams "
                          f"{st.weight_bytes / 1e9:.2f} GB of expert weights (L2 is 126 MB)"), "parallelism": "replicas only",
                   "seed": 0},
        "dense": {"value": dense_value, "unit": UNIT, "ms_per_step": dense_ms,
                  "note": "the same batches without pruning (dense top-k), timed in the same run"},
        "clocks": clk,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "call": "caee_moe_forward_host: x from pinned host memory, y back to it, every step; copies double-buffered on two side streams",
                "ms_per_step": ms_e2e},
        "gpu_launches": gpu_launches,
        "roofline": {"bound": "hbm", "kernel": ("k_expert_fp8_ts" if T > 128 else "k_expert_fp8") if fp8 else "k_expert_umma", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak if achieved else None, "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": peak_src,
                     "bytes_per_launch": bytes_per_launch, "kernel_ms": k_ms,
                     "bytes_by_batch": batch_bytes,
                     "frac_of_8TBps_nominal": achieved / 8000.0 if achieved else None},
        "latency_us": {"pruned": ms_step * 1e3, "pruned_without_kernel_events": ms_plain * 1e3, "dense": dense_ms * 1e3,
                       "expert_kernel": k_ms * 1e3 if k_ms else None},
        "pruning": {"n_act": st.n_act, "n_keep": st.n_keep, "n_run": st.n_run, "F_cost_dense": st.F_cost_dense,
                    "F_cost": st.F_cost, "F_imp": st.F_imp / 2.0 ** 40, "eps": eps, "bytes_pruned": st.weight_bytes,
                    "bytes_dense": st_dense.weight_bytes, "bytes_removed_frac": removed, "n_run_dense": st_dense.n_run},
    }
    if calib is not None:
        out["calibrated_cost_table"] = calib
    if offload_t is not None and len(offload_t[0]):
        # offload scenario (BASELINE.json config 5): the step is bound by the H2D copy train of the surviving misses;
        # resident compute is hidden when it ends before the copies do (CUDA events on the two streams, same run)
        copy_ms, res_ms, lead_ms = (float(statistics.mean(v)) for v in offload_t)
        out["offload"] = {"h2d_bytes_per_step_last_batch": st.h2d_bytes, "n_fetch_last_batch": st.n_fetch,
                          "h2d_bytes_dense_last_batch": st_dense.h2d_bytes,
                          "copy_train_ms": copy_ms, "resident_launch_ms": res_ms, "copy_start_to_resident_done_ms": lead_ms,
                          "resident_compute_hidden": bool(lead_ms <= copy_ms),
                          "copy_train_share_of_step": copy_ms / ms_step,
                          "staging": "ring of 8 device slots, 4 fetched experts per expert-kernel launch"}
        h2d = float(statistics.mean(batch_h2d[i % len(xs)] for i in range(len(offload_t[0]))))
        gbs = h2d / (copy_ms * 1e-3) / 1e9 if copy_ms > 0 else None
        out["offload"]["h2d_bytes_per_step"] = h2d
        out["roofline"] = {"bound": "pcie", "kernel": "H2D copy train (one cudaMemcpyAsync per surviving miss, side stream)",
                           "achieved": gbs, "peak": calib["h2d_gbs"], "unit": "GB/s", "frac": gbs / calib["h2d_gbs"] if gbs else None, "traffic": None,
                           "peak_source": "caee_calibrate_cost H2D tier, measured in this run",
                           "bytes_per_launch": h2d, "kernel_ms": copy_ms}
    if fp8 and T > 128 and k_ms:
        # e4m3 steps of more than 128 tokens run k_expert_fp8_ts (fp16 MMAs on weights widened into tensor memory).  Which
        # roofline bounds the step follows from its arithmetic intensity: useful flops per weight byte streamed against the
        # ridge point of this box (sustained 16-bit tensor rate / measured HBM rate); below it the HBM figures above stand
        tpeak, tsrc = tensor_peak()
        flops = 6.0 * cfg.H * cfg.I * T * (cfg.k + cfg.S)      # every token keeps k routed slots + S shared
        intensity = flops / bytes_per_launch if bytes_per_launch else 0.0
        ridge = tpeak * 1e12 / (peak * 1e9)
        out["roofline"].update({"flops_per_launch": flops, "flop_per_byte": intensity, "ridge_flop_per_byte": ridge})
        if intensity > ridge:
            tf = flops / (k_ms * 1e-3) / 1e12
            out["roofline"].update({"bound": "tensor", "achieved": tf, "peak": tpeak, "unit": "TFLOP/s", "frac": tf / tpeak,
                                    "peak_source": tsrc, "hbm_gbs": achieved})
            out["roofline"].pop("frac_of_8TBps_nominal", None)
    if world == 1 and not args.no_cpu_baseline:
        # the oracle as it stands on this box's host cores: the whole T-token layer step, a few repetitions
        o = OracleLayer(cfg, T, prune, eps, 0, dev, layer=L)
        L.close()
        torch.cuda.empty_cache()
        secs = [o.step()]
        while sum(secs) < 10.0 and len(secs) < 16:
            secs.append(o.step())
        out["cpu_baseline"] = {"value": T / statistics.mean(secs), "unit": UNIT, "cores": o.cores, "kind": "oracle",
                               "sample": oracle_sample_text(o, len(secs))}
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


# --------------------------------------------------------------------------- NEXT-2: expert-parallel ranks, one at a time
def run_ep_emulation(args, cfg, prune, eps):
    """SURVEY.md §8(f) NEXT-2 on ONE GPU (PAPER.md:57, 97 `Latency_total = max_d Latency_d`, 127): `--ep-emulate W` builds
    the W ranks of an expert-parallel group as W contexts in this process (each holds only the experts it owns, owner =
    contiguous blocks = the cost model's partitions with D = W, no straggler) and times every rank's slice of the step ALONE
    on the whole GPU — what that rank would take on a GPU of its own, without the NVLink transfers this box cannot show.
    Reported: per-rank slice time (router + decision, replicated on every rank, + the rank's expert kernel), their max
    (= the emulated step latency of the group) and sum, dense vs pruned, next to the modelled per-rank loads and F_cost."""
    import torch
    from paper_2606_29982_b200 import binding as B
    from paper_2606_29982_b200 import ep
    from paper_2606_29982_b200 import workloads as wl
    from paper_2606_29982_b200.layer import Layer

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libcaee has no CPU fallback")
    torch.cuda.set_device(0)
    dev, W, T, K = "cuda:0", args.ep_emulate, args.tokens, args.steps
    cfg = wl.scaled(cfg, name=f"{cfg.name}-EP{W}", D=W, straggler_part=-1)
    owner = ep.owner_table(cfg.E, W)
    ranks = [Layer(cfg, seed=0, max_tokens=max(T, 128), device=dev,
                   ep=(r, W, owner, lambda ctx: [B.caee_ep_obuf(ctx)[0]] * W)) for r in range(W)]
    peers = [B.caee_ep_obuf(L.ctx)[0] for L in ranks]
    for r, L in enumerate(ranks):
        B.caee_set_ep(L.ctx, r, W, owner, peers)
    xs = [wl.hidden(cfg, T, 100 + i, dev) for i in range(4)]
    y = torch.empty_like(xs[0])
    stats = B.stats_buffer(dev)
    stream = torch.cuda.current_stream()

    def slice_times(params):
        out = []
        for L in ranks:
            for i in range(3):
                B.caee_moe_forward(L.ctx, xs[i % 4], T, params, None, stats)
            torch.cuda.synchronize()
            ms = []
            for i in range(K):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                B.caee_moe_forward(L.ctx, xs[i % 4], T, params, None, stats)
                e1.record(stream)
                torch.cuda.synchronize()
                ms.append(e0.elapsed_time(e1))
            out.append(statistics.median(ms))
        B.caee_moe_forward(ranks[0].ctx, xs[0], T, params, None, stats)
        torch.cuda.synchronize()
        return out, B.read_stats(stats)

    try:
        params = None if prune is None else B.prune_params(prune[0], prune[1], 0, eps)
        dense_ms, _ = slice_times(None)
        _, st_d = slice_times(B.prune_params(B.CAEE_PRUNE_THRESH, 0.0))      # keeps everything, reports the modelled loads
        pruned_ms, st_p = slice_times(params) if params is not None else (dense_ms, st_d)
        # the combine of the home tokens (after the group barrier), timed once for completeness
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for L in ranks:
            B.caee_ep_combine(L.ctx, T, y)
        e1.record(stream)
        torch.cuda.synchronize()
        combine_ms = e0.elapsed_time(e1) / W
    finally:
        for L in ranks:
            L.close()
    fmax = max(1, st_d.F_cost_dense)
    print(json.dumps({
        "metric": "ep_emulated_step_ms", "value": max(pruned_ms), "unit": "ms/step", "n_gpus": 1, "steps": K, "warmup": 3,
        "higher_is_better": False, "vs_baseline": None, "dtype": {0: "f32", 1: "bf16", 2: "fp8_e4m3"}[cfg.w_dtype], "data": "synthetic",
        "config": {"workload": f"{cfg.name}: {W} expert-parallel ranks of {cfg.E // W} experts (+{cfg.S} shared, replicated), T={T}, "
                               f"{'dense' if prune is None else 'CAEE prune ' + args.prune}; every rank's slice timed ALONE on one B200 "
                               "(no NVLink transfers): emulated step latency = max over ranks (PAPER.md:97)"},
        "ep": {"world": W, "slice_ms_dense": dense_ms, "slice_ms_pruned": pruned_ms,
               "max_ms_dense": max(dense_ms), "max_ms_pruned": max(pruned_ms), "max_ratio": max(pruned_ms) / max(dense_ms),
               "sum_ms_dense": sum(dense_ms), "sum_ms_pruned": sum(pruned_ms), "sum_ratio": sum(pruned_ms) / sum(dense_ms),
               "modelled_load_dense_pct": [100.0 * st_d.load[d] / fmax for d in range(W)],
               "modelled_load_pruned_pct": [100.0 * st_p.load[d] / fmax for d in range(W)],
               "F_cost_dense": st_d.F_cost_dense, "F_cost_pruned": st_p.F_cost if params is not None else st_d.F_cost_dense,
               "F_cost_ratio": (st_p.F_cost / fmax) if params is not None else 1.0,
               "n_keep": st_p.n_keep, "n_act": st_p.n_act, "combine_ms_per_rank": combine_ms}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="caee", choices=["caee", "reference"])
    ap.add_argument("--workload", default="c3", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--tokens", type=int, default=128)
    ap.add_argument("--prune", default="thresh:0.6", help="dense | none | thresh:θ | cir:θ_imp | rank:b | frac:p")
    ap.add_argument("--eps-frac", type=float, default=0.10,
                    help="importance bound F_imp <= eps-frac * T (PAPER.md:150-152; CAEE_IMP_BOUND); negative = no bound")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--calibrate", action="store_true",
                    help="cost table from caee_calibrate_cost on this GPU (S10); always on for the offload workload c5")
    ap.add_argument("--cache-loop", action="store_true", help="SURVEY §8(f) NEXT-1: multi-layer decode loop over an LFU expert cache")
    ap.add_argument("--ep-emulate", type=int, default=0, help="SURVEY §8(f) NEXT-2: W expert-parallel ranks built in this process, every rank's slice timed alone")
    ap.add_argument("--layers", type=int, default=2)
    ap.add_argument("--cache-slots", type=int, default=128)
    args = ap.parse_args()
    from paper_2606_29982_b200 import workloads as wl
    cfg = wl.CONFIGS[args.workload.upper()]
    prune = parse_prune(args.prune)
    eps = args.eps_frac * args.tokens if (prune is not None and args.eps_frac >= 0) else None
    if args.ep_emulate > 1:
        run_ep_emulation(args, cfg, prune, eps)
    elif args.cache_loop:
        run_cache_loop(args, cfg)
    elif args.impl == "reference":
        run_reference(args, cfg, prune, eps)
    else:
        run_caee(args, cfg, prune, eps)


if __name__ == "__main__":
    main()

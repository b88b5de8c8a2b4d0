"""Knob sweep of one CAEE layer: the paper's THRESH grid θ ∈ [0.3, 1.2]
(on-device inference) and CIR grid θ_imp ∈ {0.9, 0.8, 0.7} (offloading)
across decode batch sizes, with a Fig. 10-style per-partition load report (Fig. 10:
expert cost per device before and after pruning).

    python -m paper_2606_29982_b200.sweep --workload c3 --tokens 8,32,64,128 > sweep.md

Everything is measured through the C ABI (caee_moe_forward + caee_fwd_stats); this module only
marshals arguments and formats the table.  Latency = median of `--steps` steps, each between its own
CUDA-event pair, after `--warmup` steps, rotating over 4 seeded token batches; a pruned setting is
measured INTERLEAVED with the dense step (dense, pruned, dense, pruned, ... on the same batches) so that
"vs dense" compares steps taken in the same thermal / power state.  "experts run" and "GB read" are means
over the 4 batches; kept / activated, F_cost and the per-partition columns (summed C~ ticks of the
experts each partition keeps, stats.load) are the first batch's.
"""
import argparse
import statistics

import torch

from . import binding as B
from . import workloads as wl
from .layer import Layer


def measure(L, xs, params, steps, warmup, against_dense=False):
    """(median step us, first batch's stats, mean experts run, mean GB read[, median us of the interleaved dense steps])."""
    dev = L.device
    y = torch.empty_like(xs[0])
    stats = B.stats_buffer(dev)
    for i in range(warmup):
        L.forward(xs[i % len(xs)], params, y=y, stats=stats)
    per_batch = []
    for x in xs:
        L.forward(x, params, y=y, stats=stats)
        torch.cuda.synchronize()
        per_batch.append(B.read_stats(stats))
    st0 = per_batch[0]
    n_run = statistics.mean(s.n_run for s in per_batch)
    gb = statistics.mean(s.weight_bytes for s in per_batch) / 1e9

    def one(x, p):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        L.forward(x, p, y=y, stats=stats)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    ms, ms_dense = [], []
    for i in range(steps):
        if against_dense:
            ms_dense.append(one(xs[i % len(xs)], None))
        ms.append(one(xs[i % len(xs)], params))
    out = (statistics.median(ms) * 1e3, st0, n_run, gb)
    return out + (statistics.median(ms_dense) * 1e3,) if against_dense else out


def ablation(L, cfg, Ts, args):
    """SURVEY.md §8(f) NEXT-4, PAPER.md:250-256 / Fig. 9: masked Top-k compensation against the random
    selection baseline (CAEE_COMP_RANDOM).  Task accuracy needs the absent suites and weights; the
    proxy is the relative L2 distance of the layer output from the dense (unpruned) layer's."""
    dev = L.device
    print(f"# Compensation ablation proxy, {cfg.name}: ||y - y_dense|| / ||y_dense|| over the batch\n")
    print("| T | setting | experts kept | masked Top-k (paper) | random selection | ratio |")
    print("|---|---|---|---|---|---|")
    grid = [("cir", B.CAEE_PRUNE_CIR, float(v)) for v in args.cir.split(",") if v] + \
           [("thresh", B.CAEE_PRUNE_THRESH, float(v)) for v in args.thresh.split(",") if v]
    for T in Ts:
        x = wl.hidden(cfg, T, 100, dev)
        stats = B.stats_buffer(dev)
        y0 = L.forward(x, None).float()
        torch.cuda.synchronize()
        n0 = float(y0.norm())
        for name, mode, theta in grid:
            errs = []
            for flags in (0, B.CAEE_COMP_RANDOM):
                y = L.forward(x, B.prune_params(mode, theta, flags), stats=stats).float()
                torch.cuda.synchronize()
                errs.append(float((y - y0).norm()) / n0)
            s = B.read_stats(stats)
            ratio = errs[1] / errs[0] if errs[0] > 0 else float("nan")
            print(f"| {T} | {name} {theta:g} | {s.n_keep}/{s.n_act} | {errs[0]:.4f} | {errs[1]:.4f} | {ratio:.2f} |")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="c3", choices=["c2", "c3", "c4"])
    ap.add_argument("--tokens", default="8,32,64,128")
    ap.add_argument("--thresh", default="0.3,0.6,0.8,1.0,1.2")
    ap.add_argument("--cir", default="0.9,0.8,0.7")
    ap.add_argument("--frac", default="", help="FRAC budgets p (BASELINE.json config 4: 0.1,0.25)")
    ap.add_argument("--steps", type=int, default=12)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--ablation", action="store_true", help="compensation ablation proxy instead of the latency sweep")
    ap.add_argument("--calibrate", action="store_true", help="cost table from caee_calibrate_cost on this GPU (S10) instead of the workload's formula")
    ap.add_argument("--partitions", type=int, default=0, help="override D (contiguous blocks, no straggler); D = 1 is the setting where "
                    "the modelled F_cost and the bytes read coincide (SURVEY.md 8(d))")
    args = ap.parse_args()
    cfg = wl.CONFIGS[args.workload.upper()]
    if args.partitions > 0:
        cfg = wl.scaled(cfg, name=f"{cfg.name}-D{args.partitions}", D=args.partitions, straggler_part=-1)
    Ts = [int(t) for t in args.tokens.split(",")]
    dev = "cuda:0"
    L = Layer(cfg, seed=0, max_tokens=max(max(Ts), 128), device=dev)
    D = cfg.D
    if args.calibrate:
        hbm, h2d = L.calibrate()
        print(f"Cost table calibrated on this GPU (caee_calibrate_cost, PAPER.md:137-141): HBM tier t = {hbm.slope_ns_per_byte:.3e} ns/B x S + "
              f"{hbm.intercept_ns:.0f} ns ({hbm.gbytes_per_s:.0f} GB/s, r2 {hbm.r2:.3f}); H2D tier t = {h2d.slope_ns_per_byte:.3e} ns/B x S + "
              f"{h2d.intercept_ns:.0f} ns ({h2d.gbytes_per_s:.1f} GB/s, r2 {h2d.r2:.3f}); C~ = {int(L.ticks_res.min())} ns per resident expert.\n")
    if args.ablation:
        try:
            ablation(L, cfg, Ts, args)
        finally:
            L.close()
        return
    print(f"# Knob sweep, {cfg.name} (H={cfg.H} I={cfg.I} E={cfg.E}+{cfg.S} top-{cfg.k}, D={D} partitions, "
          f"partition {cfg.straggler_part} costs 2x)\n")
    print("| T | setting | step µs | dense step µs (interleaved) | vs dense | experts run (mean of 4 batches) | kept / activated (batch 0) | GB read (mean) | F_cost ticks (dense → kept) | per-partition load after pruning, % of the dense max |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    try:
        for T in Ts:
            xs = [wl.hidden(cfg, T, 100 + i, dev) for i in range(4)]
            base_us, st, n_run, gb = measure(L, xs, None, args.steps, args.warmup)
            # dense loads: THRESH θ = 0 keeps every activated expert and reports the loads
            st_d = measure(L, xs, B.prune_params(B.CAEE_PRUNE_THRESH, 0.0), 1, 1)[1]
            fmax = max(1, st_d.F_cost_dense)
            loads = " ".join(f"{100 * st_d.load[d] / fmax:.0f}" for d in range(D))
            print(f"| {T} | dense | {base_us:.0f} | | 1.000 | {n_run:.1f} | | {gb:.2f} | {st_d.F_cost_dense} | {loads} |")
            grid = [("thresh", B.CAEE_PRUNE_THRESH, float(v)) for v in args.thresh.split(",") if v] + \
                   [("cir", B.CAEE_PRUNE_CIR, float(v)) for v in args.cir.split(",") if v] + \
                   [("frac", B.CAEE_PRUNE_FRAC, float(v)) for v in args.frac.split(",") if v]
            for name, mode, theta in grid:
                us, s, n_run, gb, dense_us = measure(L, xs, B.prune_params(mode, theta), args.steps, args.warmup, against_dense=True)
                loads = " ".join(f"{100 * s.load[d] / fmax:.0f}" for d in range(D))
                print(f"| {T} | {name} {theta:g} | {us:.0f} | {dense_us:.0f} | {us / dense_us:.3f} | {n_run:.1f} | {s.n_keep}/{s.n_act} | "
                      f"{gb:.2f} | {s.F_cost_dense} → {s.F_cost} | {loads} |")
    finally:
        L.close()


if __name__ == "__main__":
    main()

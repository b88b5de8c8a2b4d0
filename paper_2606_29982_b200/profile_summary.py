"""Turns `ncu -i X.ncu-rep --page raw --csv` (stdin) into a text summary and, optionally, an entry of
profiles/traffic.json — so that no number under profiles/ is typed by hand.

    ncu -i gpurun_out/X.ncu-rep --page raw --csv | \
        python -m paper_2606_29982_b200.profile_summary --title "..." --command "..." \
            [--kernel k_expert_umma --traffic-key "C3-r1-bf16/T128/thresh:0.6" --traffic profiles/traffic.json] \
            > profiles/rNN_name.md

    cuobjdump -sass paper_2606_29982_b200/libcaee.so | c++filt | \
        python -m paper_2606_29982_b200.profile_summary --sass --title "..." > profiles/rNN_sass.md

(--sass: per kernel, counts of the SASS mnemonics that prove tcgen05 / TMEM / TMA use, plus the first line of each.)

Only formatting and averaging live here; the measurements are Nsight Compute's.
"""
import argparse
import csv
import json
import re
import statistics
import subprocess
import sys

COLS = [
    ("gpu__time_duration.sum", "us", 1.0),
    ("dram__bytes_read.sum", "MB read", None),
    ("dram__bytes_write.sum", "MB written", None),
    ("dram__bytes_read.sum.per_second", "read GB/s", None),
    ("dram__throughput.avg.pct_of_peak_sustained_elapsed", "dram % peak", 1.0),
    ("lts__t_sector_hit_rate.pct", "L2 hit %", 1.0),
    ("sm__pipe_tensor_cycles_active_realtime.avg.pct_of_peak_sustained_elapsed", "tensor pipe %", 1.0),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "occupancy %", 1.0),
    ("launch__registers_per_thread", "regs", 1.0),
    ("launch__shared_mem_per_block_dynamic", "dyn smem KB", None),
]
STALLS = re.compile(r"smsp__average_warps_issue_stalled_(\w+)_per_issue_active\.ratio$")


def to_bytes(v, unit):
    v = float(v.replace(",", "")) if v else 0.0
    u = unit.lower()
    for p, m in (("kbyte", 1e3), ("mbyte", 1e6), ("gbyte", 1e9), ("tbyte", 1e12), ("byte", 1.0)):
        if u.startswith(p):
            return v * m
    return v


def to_us(v, unit):
    v = float(v.replace(",", "")) if v else 0.0
    return v * {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(unit.strip().lower(), 1.0)


def short(name):
    name = re.sub(r"^void\s+", "", name)
    name = re.sub(r"<unnamed>::", "", name)
    return name.split("(")[0]


def git_head():
    try:
        return subprocess.run(["git", "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
    except OSError:
        return ""


# SASS mnemonics of the Blackwell tensor / TMEM / bulk-copy paths (B200_PROFILING.md) and what they are
SASS_OPS = [("UTCHMMA", "tcgen05.mma kind::f16"), ("UTCQMMA", "tcgen05.mma kind::f8f6f4"), ("UTCBAR", "tcgen05.commit"),
            ("LDTM", "tcgen05.ld (TMEM -> registers)"), ("STTM", "tcgen05.st (registers -> TMEM)"), ("UTCATOMSWS", "tcgen05.alloc / dealloc"),
            ("UBLKCP", "cp.async.bulk (bulk copy global -> shared)"), ("UTMALDG", "cp.async.bulk.tensor (TMA, incl. tile::gather4)"),
            ("SYNCS", "mbarrier ops"), ("HMMA", "mma.sync (legacy tensor path)"), ("ACQBULK", "griddepcontrol.wait"),
            ("ELECT", "elect.sync")]


def sass_summary(title, want):
    """stdin: `cuobjdump -sass lib.so`.  One table row per kernel whose name contains one of `want`."""
    fn, counts, first, order = None, {}, {}, []
    for line in sys.stdin:
        m = re.search(r"Function : (.+)$", line)
        if m:
            fn = short(m.group(1).strip().replace("(anonymous namespace)::", ""))
            continue
        if fn is None or not any(w in fn for w in want):
            continue
        m = re.match(r"\s+/\*[0-9a-f]+\*/\s+(.*?);", line)
        if not m:
            continue
        ins = m.group(1)
        if fn not in counts:
            counts[fn], first[fn] = {}, {}
            order.append(fn)
        counts[fn]["_total"] = counts[fn].get("_total", 0) + 1
        for op, _ in SASS_OPS:
            if re.search(r"(^|\s)" + op + r"[.\s]", " " + ins):
                counts[fn][op] = counts[fn].get(op, 0) + 1
                first[fn].setdefault(op, ins)
    print(f"# {title}\n")
    print("Written by `cuobjdump -sass paper_2606_29982_b200/libcaee.so | c++filt | python -m paper_2606_29982_b200.profile_summary --sass` "
          f"at commit `{git_head()}` (the library as `paper_2606_29982_b200/build.py` builds it: "
          "`nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3`).\n")
    print("| mnemonic | PTX it comes from |\n|---|---|")
    for op, what in SASS_OPS:
        print(f"| `{op}` | {what} |")
    print("\n| kernel | SASS instructions | " + " | ".join(op for op, _ in SASS_OPS) + " |")
    print("|---|---|" + "---|" * len(SASS_OPS))
    for fn in order:
        name = fn
        print(f"| `{name}` | {counts[fn]['_total']} | " + " | ".join(str(counts[fn].get(op, 0)) for op, _ in SASS_OPS) + " |")
    print("\nFirst occurrence of each mnemonic:\n")
    for fn in order:
        print(f"- `{fn}`")
        for op, _ in SASS_OPS:
            if op in first[fn]:
                print(f"  - `{first[fn][op]}`")


def launches_summary(title, command, note):
    """stdin: the --csv log of `ncu --metrics gpu__time_duration.sum` (one row per launch)."""
    rows = list(csv.reader(l for l in sys.stdin if l.startswith('"')))
    hdr = rows[0]
    ki, vi, ui = hdr.index("Kernel Name"), hdr.index("Metric Value"), hdr.index("Metric Unit")
    agg, order = {}, []
    for r in rows[1:]:
        n = short(r[ki])
        if n not in agg:
            agg[n] = []
            order.append(n)
        agg[n].append(to_us(r[vi], r[ui]))
    total = sum(sum(v) for v in agg.values())
    print(f"# {title}\n")
    if command:
        print(f"Command:\n\n```\n{command}\n```\n")
    print(f"Table written by `python -m paper_2606_29982_b200.profile_summary --launches` from the launch list (the `.csv` beside "
          f"this file = ncu's log without its `==PROF==` lines) at commit `{git_head()}`.  Times under the profiler are cold-cache and "
          "serialised (short kernels also run at reduced clocks between replays): only SHARES are comparable with the live "
          "CUDA-event timing of bench.py.\n")
    if note:
        print(note + "\n")
    print("| kernel | launches | mean us | min us | max us | share of listed time |\n|---|---|---|---|---|---|")
    for n in order:
        v = agg[n]
        print(f"| `{n}` | {len(v)} | {statistics.mean(v):.1f} | {min(v):.1f} | {max(v):.1f} | {100 * sum(v) / total:.1f}% |")


def bench_table(title, command, note):
    """stdin: bench.py result lines (one JSON object per line), e.g. the rows of a latency table."""
    print(f"# {title}\n")
    if command:
        print(f"Command:\n\n```\n{command}\n```\n")
    print(f"Table written by `python -m paper_2606_29982_b200.profile_summary --bench-table` from bench.py's JSON lines at commit "
          f"`{git_head()}`.  step = `ms_per_step` (K steps between one event pair, with the expert kernel's own event pair inside); "
          "w/o events = the same steps without the kernel events (programmatic dependent launches overlap); dense = the same batches "
          "without pruning; kernel = the expert kernel's event-pair duration; rate = algorithmic bytes (or useful flops) / kernel time.\n")
    if note:
        print(note + "\n")
    lines = [json.loads(l) for l in sys.stdin if l.strip().startswith("{")]
    if lines and "rows" in lines[0]:
        # bench.py --cache-loop lines: one table row per (tokens per step, setting)
        print("| T | setting | ms / step | misses / step | hits / step | H2D GB / step | H2D GB/s | vs dense |\n|---|---|---|---|---|---|---|---|")
        for d in lines:
            T = d["config"]["workload"].split("T=")[1].split(" ")[0]
            for r in d["rows"]:
                print(f"| {T} | {r['setting']} | {r['ms_per_step']:.2f} | {r['misses_per_step']:.1f} | {r['hits_per_step']:.1f} | "
                      f"{r['h2d_gb_per_step']:.2f} | {r['h2d_gbs']:.1f} | {r['vs_dense']:.3f} |")
        return
    if lines and "ep" in lines[0]:
        # bench.py --ep-emulate lines: one row per (T, setting)
        print("| ranks | T | setting | kept / activated | slowest rank ms, dense → pruned (= emulated step) | ratio | sum over ranks ms, dense → pruned | ratio | "
              "modelled F_cost ratio | per-rank slice ms, pruned | modelled per-rank load, % of the dense max, pruned |")
        print("|---|---|---|---|---|---|---|---|---|---|---|")
        for d in lines:
            e, w = d["ep"], d["config"]["workload"]
            T = w.split("T=")[1].split(",")[0]
            mode = "dense" if ", dense;" in w or w.rstrip().endswith("dense") else w.split("CAEE prune ")[1].split(";")[0]
            print(f"| {e['world']} | {T} | {mode} | {e['n_keep']}/{e['n_act']} | {e['max_ms_dense']:.3f} → {e['max_ms_pruned']:.3f} | {e['max_ratio']:.3f} | "
                  f"{e['sum_ms_dense']:.3f} → {e['sum_ms_pruned']:.3f} | {e['sum_ratio']:.3f} | {e['F_cost_ratio']:.3f} | "
                  + " ".join(f"{v:.3f}" for v in e["slice_ms_pruned"]) + " | " + " ".join(f"{v:.0f}" for v in e["modelled_load_pruned_pct"]) + " |")
        return
    print("| workload | T | mode | step us | w/o events us | dense us | kernel us | rate | frac of measured peak | experts run | launches / K steps | clocks MHz, reasons |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|")
    for d in lines:
        w = d["config"]["workload"]
        name = w.split(":")[0]
        T = w.split("T=")[1].split(",")[0]
        mode = "dense" if ", dense top-k" in w else w.split("CAEE prune ")[1].split(";")[0]
        r, lat = d["roofline"], d["latency_us"]
        rate = f"{r['achieved']:.0f} {r['unit']}" if r.get("achieved") else ""
        frac = f"{r['frac']:.3f}" if r.get("frac") else ""
        ker = f"{lat['expert_kernel']:.1f}" if lat.get("expert_kernel") else ""
        plain = f"{lat['pruned_without_kernel_events']:.1f}" if lat.get("pruned_without_kernel_events") else ""
        clk = d.get("clocks", {})
        print(f"| {name} | {T} | {mode} | {lat['pruned']:.1f} | {plain} | {lat['dense']:.1f} | {ker} | {rate} | {frac} | "
              f"{d['pruning']['n_run']} | {d['gpu_launches']} / {d['steps']} | {clk.get('sm_mhz')} {','.join(clk.get('reasons', [])) or '-'} |")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--bench-table", action="store_true", help="stdin is bench.py JSON lines: format them as a latency table")
    ap.add_argument("--launches", action="store_true", help="stdin is the --csv launch list of `ncu --metrics gpu__time_duration.sum`")
    ap.add_argument("--sass", action="store_true", help="stdin is `cuobjdump -sass`: count tensor / TMEM / TMA mnemonics per kernel")
    ap.add_argument("--kernels", default="k_expert,k_router_mma", help="--sass: comma-separated substrings of the kernels to list")
    ap.add_argument("--title", default="ncu summary")
    ap.add_argument("--command", default="", help="the command that produced the .ncu-rep (printed in the summary)")
    ap.add_argument("--note", default="")
    ap.add_argument("--kernel", default="", help="kernel (substring) whose DRAM bytes go to --traffic")
    ap.add_argument("--traffic", default="")
    ap.add_argument("--traffic-key", default="")
    ap.add_argument("--alg-bytes", default="", help="comma-separated algorithmic bytes of the captured launches of --kernel, in order")
    args = ap.parse_args()
    if args.sass:
        sass_summary(args.title, [w for w in args.kernels.split(",") if w])
        return
    if args.launches:
        launches_summary(args.title, args.command, args.note)
        return
    if args.bench_table:
        bench_table(args.title, args.command, args.note)
        return
    rows = list(csv.reader(sys.stdin))
    hdr, units, data = rows[0], rows[1], rows[2:]

    def col(suffix):
        for i, h in enumerate(hdr):
            if h == suffix or h.endswith("." + suffix):
                return i
        return None

    ki = hdr.index("Kernel Name")
    print(f"# {args.title}\n")
    if args.command:
        print(f"Command:\n\n```\n{args.command}\n```\n")
    print(f"Summary written by `python -m paper_2606_29982_b200.profile_summary` from `ncu --page raw --csv` at commit "
          f"`{git_head()}`; one line per captured launch.  Durations under the profiler are serialised and replayed: "
          "they are evidence for traffic and pipe utilisation, not bench values.\n")
    if args.note:
        print(args.note + "\n")
    head = ["#", "kernel", "grid", "block"] + [c[1] for c in COLS]
    print("| " + " | ".join(head) + " |")
    print("|" + "---|" * len(head))
    gi, bi = col("launch__grid_size"), col("launch__block_size")
    picked = []
    for n, r in enumerate(data):
        out = [str(n), short(r[ki]), r[gi] if gi is not None else "", r[bi] if bi is not None else ""]
        vals = {}
        for name, label, _ in COLS:
            i = col(name)
            if i is None or r[i] == "":
                out.append("")
                continue
            if label == "us":
                v = to_us(r[i], units[i]); out.append(f"{v:.1f}")
            elif label.startswith("MB"):
                v = to_bytes(r[i], units[i]); out.append(f"{v / 1e6:.2f}")
            elif label == "read GB/s":
                v = to_bytes(r[i], units[i]); out.append(f"{v / 1e9:.0f}")
            elif label == "dyn smem KB":
                v = to_bytes(r[i], units[i]); out.append(f"{v / 1e3:.1f}")
            else:
                v = float(r[i].replace(",", "")); out.append(f"{v:.1f}")
            vals[name] = v
        print("| " + " | ".join(out) + " |")
        if args.kernel and args.kernel in r[ki]:
            picked.append(vals)
    # warp stall reasons, top five per kernel name
    print("\nWarp stall reasons (cycles stalled per issued instruction, top five):\n")
    seen = set()
    for r in data:
        k = short(r[ki])
        if k in seen:
            continue
        seen.add(k)
        st = []
        for i, h in enumerate(hdr):
            m = STALLS.search(h)
            if m and r[i]:
                st.append((float(r[i].replace(",", "")), m.group(1)))
        st.sort(reverse=True)
        print(f"- `{k}`: " + ", ".join(f"{n} {v:.2f}" for v, n in st[:5]))
    if picked:
        rd = [p.get("dram__bytes_read.sum", 0.0) for p in picked]
        wr = [p.get("dram__bytes_write.sum", 0.0) for p in picked]
        us = [p.get("gpu__time_duration.sum", 0.0) for p in picked]
        tot = [a + b for a, b in zip(rd, wr)]
        print(f"\n`{args.kernel}`: {len(picked)} launches; DRAM read+write per launch = "
              + ", ".join(f"{t / 1e9:.3f}" for t in tot) + f" GB (mean {statistics.mean(tot) / 1e9:.3f} GB); "
              f"read rate = " + ", ".join(f"{a / u / 1e3:.0f}" for a, u in zip(rd, us)) + " GB/s under the profiler.")
        alg = [float(v) for v in args.alg_bytes.split(",") if v]
        if alg and len(alg) == len(tot):
            print("Traffic / algorithmic bytes per launch = " + ", ".join(f"{t / a:.3f}" for t, a in zip(tot, alg))
                  + f" (mean {statistics.mean(tot) / statistics.mean(alg):.3f}).")
        if args.traffic and args.traffic_key:
            try:
                with open(args.traffic) as f:
                    tj = json.load(f)
            except (OSError, ValueError):
                tj = {}
            tj[args.traffic_key] = {"kernel": args.kernel, "dram_bytes_per_launch": statistics.mean(tot),
                                    "dram_bytes_by_launch": tot, "launches": len(tot), "commit": git_head(),
                                    "source": "ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum"}
            if alg and len(alg) == len(tot):
                tj[args.traffic_key]["algorithmic_bytes_by_launch"] = alg
            with open(args.traffic, "w") as f:
                json.dump(tj, f, indent=1, sort_keys=True)
                f.write("\n")


if __name__ == "__main__":
    main()

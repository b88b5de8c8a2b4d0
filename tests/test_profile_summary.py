"""Host logic of paper_2606_29982_b200/profile_summary.py (the tool that writes every table under profiles/ from
Nsight Compute / cuobjdump output): unit conversion, per-kernel aggregation, SASS mnemonic counting.  CPU only."""
import io
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, stdin):
    r = subprocess.run([sys.executable, "-m", "paper_2606_29982_b200.profile_summary"] + args, input=stdin, capture_output=True,
                       text=True, cwd=ROOT)
    assert r.returncode == 0, r.stderr
    return r.stdout


def test_launch_list_summary_aggregates_per_kernel():
    hdr = '"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"\n'
    row = lambda i, k, unit, v: f'"{i}","1","python","h","{k}","1","7","(256, 1, 1)","(148, 1, 1)","0","10.0","Command line profiler metrics","gpu__time_duration.sum","{unit}","{v}"\n'
    csv_text = "==PROF== Connected\n" + hdr + row(0, "void k_a<int>(int)", "us", "10.0") + row(1, "k_b(float)", "ns", "30,000") + \
        row(2, "void k_a<int>(int)", "us", "20.0")
    out = _run(["--launches", "--title", "t", "--command", "c"], csv_text)
    assert "| `k_a<int>` | 2 | 15.0 | 10.0 | 20.0 | 50.0% |" in out
    assert "| `k_b` | 1 | 30.0 | 30.0 | 30.0 | 50.0% |" in out


def test_sass_summary_counts_tensor_and_tma_mnemonics():
    sass = """
		Function : (anonymous namespace)::k_expert_demo((anonymous namespace)::P)
        /*0000*/                   UTCHMMA gdesc[UR18], gdesc[UR16], tmem[UR20], tmem[UR6], idesc[UR7], !UPT ;
        /*0010*/                   UTCHMMA gdesc[UR18], gdesc[UR16], tmem[UR20], tmem[UR6], idesc[UR7], UPT ;
        /*0020*/                   UBLKCP.S.G [UR12], [UR10], UR6, desc[UR8] ;
        /*0030*/                   LDTM.x16 R20, tmem[UR4] ;
        /*0040*/                   IADD3 R1, R1, 1, RZ ;
		Function : k_other(int)
        /*0000*/                   UTCHMMA gdesc[UR18], gdesc[UR16], tmem[UR20], tmem[UR6], idesc[UR7], !UPT ;
"""
    out = _run(["--sass", "--title", "t", "--kernels", "k_expert"], sass)
    line = [l for l in out.splitlines() if l.startswith("| `k_expert_demo`")]
    assert len(line) == 1 and "k_other" not in out
    cells = [c.strip() for c in line[0].split("|")]
    assert cells[2] == "5" and cells[3] == "2"          # 5 instructions, 2 UTCHMMA
    assert "UBLKCP.S.G" in out and "LDTM.x16" in out


def test_raw_page_summary_writes_traffic_entry(tmp_path):
    hdr = '"ID","Kernel Name","launch__grid_size","launch__block_size","gpu__time_duration.sum","dram__bytes_read.sum","dram__bytes_write.sum"\n'
    units = '"","","","","us","Gbyte","Mbyte"\n'
    rows = '"0","k_x(int)","148","256","100.0","1.0","10.0"\n"1","k_x(int)","148","256","200.0","2.0","20.0"\n'
    tj = tmp_path / "traffic.json"
    out = _run(["--title", "t", "--kernel", "k_x", "--traffic", str(tj), "--traffic-key", "W/T1/dense", "--alg-bytes", "1000000000,2000000000"],
               hdr + units + rows)
    d = json.load(open(tj))["W/T1/dense"]
    assert d["launches"] == 2 and abs(d["dram_bytes_per_launch"] - 1.515e9) < 1.0
    assert "Traffic / algorithmic bytes per launch = 1.010, 1.010" in out

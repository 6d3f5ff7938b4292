"""Host-side logic of bench.py (no GPU): workload parsing, roofline arithmetic, the
oracle sample used for cpu_baseline / --impl reference."""
import json
import subprocess
import sys

import pytest

import bench


def test_parse_workload_named_and_sweep_points():
    c2 = bench.parse_workload("c2")
    assert (c2["kind"], c2["W"], c2["n"], c2["M"], c2["k"], c2["Ks"]) == ("det", 4096, 256, 512, 2, (0, 16))
    p = bench.parse_workload("det,n=1024,k=4,K=8")
    assert p["n"] == 1024 and p["M"] == 2048 and p["k"] == 4 and p["Ks"] == (8,) and not p["cplx"]
    # default W: inverse + init scratch + orbitals (2 n^2) + buffers within ~100 GB
    per = 1024 * 1024 * 8 * 4 + 2 * 8 * 4 * 1024 * 8
    assert p["W"] == int(100e9 // per)
    q = bench.parse_workload("pf,n=512,k=1,K=0,W=77,cplx")
    assert q["kind"] == "pf" and q["W"] == 77 and q["cplx"]
    with pytest.raises(SystemExit):
        bench.parse_workload("nonsense")


def test_roofline_update_counts_algorithmic_bytes():
    wk = bench.parse_workload("c2")
    run = {"accepted": 1000, "prof": {"update": {"ms": 1.0, "launches": 10}},
           "kernels": {"update": "det_update_kernel"}}
    r = bench.roofline_update(wk, run, 6534.1, "measured")
    byts = 2 * 256 * 256 * 8 * 1000
    assert r["achieved"] == pytest.approx(byts / 1e-3 / 1e9)
    assert r["frac"] == pytest.approx(r["achieved"] / 6534.1)
    assert r["kernel"] == "det_update_kernel" and r["bound"] == "hbm"
    assert r["bytes_per_launch"] == pytest.approx(byts / 10)
    # traffic is imported from the committed ncu capture and says so
    assert r["traffic"] is None or "not measured in this run" in r["traffic_source"]


def test_roofline_flush_bound_selection():
    c4 = bench.parse_workload("c4")
    run = {"accepted": 5, "flushes": 4, "flush_cols": 4 * 128, "prof": {"flush": {"ms": 2.0, "launches": 3}},
           "kernels": {"flush": "flush_dmma_kernel"}}
    r = bench.roofline_flush(c4, 32, run, 6534.1, "m", 35.0)
    flops = 2.0 * 1024 * 1024 * 4 * 128 * 4          # complex: x4
    assert r["bound"] == "tensor" and r["achieved"] == pytest.approx(flops / 2e-3 / 1e12)
    c2 = bench.parse_workload("c2")
    run2 = dict(run, flush_cols=4 * 32)
    r2 = bench.roofline_flush(c2, 16, run2, 6534.1, "m", 35.0)
    assert r2["bound"] == "hbm"                       # Kk = 32 < 50
    byts = 2.0 * 256 * 256 * 8 * 4 + 2.0 * 256 * 8 * 128
    assert r2["achieved"] == pytest.approx(byts / 2e-3 / 1e9)
    assert bench.roofline_flush(c2, 0, run, 1.0, "m", 35.0) is None


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, "bench.py", "--impl", "reference", "--workload", "tiny",
                          "--steps", "4", "--warmup", "1", "--cpu-seconds", "0.2"],
                         capture_output=True, text=True, cwd=bench.ROOT, timeout=300)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == bench.METRIC and d["unit"] == bench.UNIT
    assert d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["gpu_launches"] == 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0
    assert 1 <= d["cpu_baseline"]["cores"] <= 64 and "C oracle" in d["cpu_baseline"]["sample"]


def test_oracle_sample_takes_out_the_initialisation():
    """cpu_baseline times steps only (two runs differenced), over several walkers at once."""
    wk = bench.parse_workload("tiny")
    sec, done, nw, cores, T = bench.oracle_sample(wk, 1, 20, 0.5)
    assert sec > 0 and nw >= 1 and cores >= 1 and done == nw * T and 1 <= T <= 20


def test_roofline_append_counts_one_read_pass():
    c4 = bench.parse_workload("c4")
    run = {"accepted": 100, "prof": {"append": {"ms": 4.0, "launches": 2}, "ypass": {"ms": 0.0, "launches": 0}},
           "kernels": {"append": "det_append_dmma_stream_kernel+det_append_finish_kernel", "ypass": ""}}
    r = bench.roofline_append(c4, run, 6460.9, "m")
    assert r["achieved"] == pytest.approx(1024 * 1024 * 16 * 100 / 4e-3 / 1e9) and r["bound"] == "hbm"

"""The scripts the driver runs on the GPU box -- bench.py (main arm, --kernels-only, --peaks), __graft_entry__.smoke()
and tests/preflight.py -- executed end to end WITHOUT a GPU (tests/fake_cuda.py: the kernel sources under tests/cpu_shim
stand in for the device).  What is checked is the host logic only: that each script runs to its last line on the smallest
workload and prints what the bench contract asks for.  The numbers of a dry run mean nothing and are not looked at."""
import json
import sys

import pytest

from fake_cuda import shim_as_cuda


def run_bench(monkeypatch, capsys, *argv):
    import bench
    monkeypatch.setattr(sys, "argv", ["bench.py", *argv])
    with shim_as_cuda():
        bench.main()
    lines = [ln for ln in capsys.readouterr().out.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, "bench.py prints exactly ONE JSON line"
    return json.loads(lines[0])


def test_bench_main_arm_prints_the_contract_line(monkeypatch, capsys):
    import os
    slow = os.environ.get("CBCT_SLOW") == "1"          # the A/B timings of the eight kernel variants take another minute
    line = run_bench(monkeypatch, capsys, "--workload", "1", "--steps", "1", "--warmup", "1", "--full-recon-outer", "1,1,1",
                     *([] if slow else ["--no-variants"]))
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "clocks", "gpu_launches", "e2e", "roofline", "cpu_baseline", "s_per_cgls_iter", "kernels"):
        assert key in line, key
    assert line["unit"] == "Gsamples/s" and line["dtype"] == "f32" and line["vs_baseline"] is None and line["warmup"] >= 3
    assert "workload" in line["config"] and line["gpu_launches"] > 0 and line["value"] > 0
    assert set(line["e2e"]) >= {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"} and line["e2e"]["h2d_bytes_per_step"] > 0
    r = line["roofline"]
    assert set(r) >= {"bound", "achieved", "peak", "unit", "frac", "traffic", "launch_ms", "samples_per_launch", "ceilings_gsamples_s"}
    # the line is recomputable from itself
    assert abs(r["achieved"] - r["samples_per_launch"] / (r["launch_ms"] * 1e-3) / 1e9) <= 1e-9 * r["achieved"]
    assert abs(r["frac"] - r["achieved"] / r["peak"]) <= 1e-12 and r["peak"] == min(r["ceilings_gsamples_s"].values())
    assert set(line["cpu_baseline"]) >= {"value", "unit", "cores", "kind", "sample"} and line["cpu_baseline"]["kind"] == "oracle"
    x = line["extra"]
    assert x["errors"] == [], x["errors"]                         # every context number was produced
    assert (len(x["variants"]) == 8 if slow else x["variants"] == {}) and all(v is not None for v in x["variants"].values())
    assert all(v is not None for v in x["context_ms"].values())
    assert x["full_recon_s"] is not None and x["tf_fused_kernel"].startswith("tf_fused")


def test_bench_kernels_only_and_peaks(monkeypatch, capsys, tmp_path):
    line = run_bench(monkeypatch, capsys, "--workload", "1", "--kernels-only")
    assert line["kernels_only"] and line["device_status"] == [] and line["p_ms"] > 0 and line["siddon_pt_ms"] > 0
    line = run_bench(monkeypatch, capsys, "--peaks")
    assert line["peaks"] and {"ffma", "ffma2", "lds32", "atoms_add_s32", "l2_read_64MB"} <= set(line)


def test_smoke_runs_to_its_last_line(capsys):
    import __graft_entry__ as entry
    with shim_as_cuda():
        entry.smoke()
    assert "smoke ok" in capsys.readouterr().out


def test_preflight_runs_to_its_last_line(monkeypatch, capsys):
    import preflight
    for k in ("CBCT_FORWARD_IMPL", "CBCT_BACKPROJECT_IMPL", "CBCT_FW_PACKED", "CBCT_BT_PACKED", "CBCT_BT_LANES"):
        monkeypatch.delenv(k, raising=False)                      # preflight sets and clears these itself
    with shim_as_cuda():
        assert preflight.main() == 0
    out = capsys.readouterr().out
    assert "preflight ok" in out and "FAIL" not in out


def test_gpu_marked_tests_run_under_the_harness():
    """`--shim-as-cuda` (tests/conftest.py) runs the -m gpu tests themselves on the host.  A quick subset here keeps the
    option alive; the whole of tests/test_gpu_solver.py and the cfg 1-2 part of tests/test_gpu_projectors.py take ~15 min:
        python -m pytest tests/test_gpu_solver.py tests/test_gpu_projectors.py -m gpu --shim-as-cuda \\
            -k "not full_size and not paper_size and not headroom_bound" """
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-m", "pytest", "tests/test_gpu_solver.py", "tests/test_gpu_projectors.py", "-m", "gpu",
                        "--shim-as-cuda", "-q", "-x", "-k",
                        "mg_restrict or a2_extrapolate or breakdown or tv_rof or degenerate or host_buffer or ragged or geometry_info"],
                       cwd=root, capture_output=True, text=True, timeout=1200)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-2000:]
    assert " passed" in r.stdout and "failed" not in r.stdout


def test_bench_reference_arm_prints_the_contract_line(monkeypatch, capsys):
    """`bench.py --impl reference` (the oracle on the host cores; needs no GPU and no harness)"""
    import bench
    monkeypatch.setattr(sys, "argv", ["bench.py", "--impl", "reference", "--workload", "1", "--steps", "2", "--warmup", "1"])
    bench.main()
    lines = [ln for ln in capsys.readouterr().out.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["impl"] == "reference" and line["unit"] == "Gsamples/s" and line["value"] > 0 and line["steps"] == 2
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1 and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"] == dict(value=line["value"], unit=line["unit"], h2d_bytes_per_step=0, d2h_bytes_per_step=0)
    assert line["gpu_launches"] == 0 and line["dtype"] == "f64" and "workload" in line["config"]

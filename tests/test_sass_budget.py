"""Static check of what nvcc emitted for the hot loops (no GPU): the instruction counts DESIGN.md §5 and
profiles/r1_sass_hot_loops.md quote are held here, so a source change that bloats a hot loop fails `-m "not gpu"`.
Uses tests/sass_report.py (cuobjdump on the built objects)."""
import os
import re
import shutil
import subprocess
import sys

import pytest

from paper_1008_2042_b200 import build as cuda_build


@pytest.fixture(scope="module")
def report():
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not on PATH")
    cuda_build.build()
    tool = os.path.join(os.path.dirname(os.path.abspath(__file__)), "sass_report.py")
    out = subprocess.run([sys.executable, tool], capture_output=True, text=True, check=True).stdout
    rows = {}
    for line in out.splitlines():
        m = re.match(r"\| `(?:void )?([^`]+)` \((\d+) instantiations\) \| (\d+) \| (\d+) \| ([\d.]+) \| (.*) \|", line)
        if m:
            rows[m.group(1)] = dict(n=int(m.group(2)), loop=int(m.group(3)), samples=int(m.group(4)), per=float(m.group(5)), mix=m.group(6))
    return rows


def test_forward_hot_loop(report):
    packed, scalar = report["forward_tma_kernel<BF, BS, true>"], report["forward_tma_kernel<BF, BS, false>"]
    assert packed["n"] == scalar["n"] == 5
    assert packed["samples"] == 2 and packed["per"] <= 28.0 and "FFMA2" in packed["mix"] and "LDS 16" in packed["mix"]
    assert scalar["per"] <= 42.0 and "FFMA2" not in scalar["mix"]


def test_scatter_hot_loop(report):
    for lm in (0, 1):
        packed, scalar = report[f"backproject_scatter_kernel<BF, BS, {lm}, true>"], report[f"backproject_scatter_kernel<BF, BS, {lm}, false>"]
        assert packed["per"] <= 43.0 and "FFMA2" in packed["mix"] and "ATOMS 16" in packed["mix"]
        assert "BSSY 1," in packed["mix"] + ","                    # the skipped reductions of a merged pair sit under ONE branch
        assert scalar["per"] <= 52.0


def test_siddon_hot_loops(report):
    assert report["siddon_forward_kernel"]["per"] <= 37.0 and "LDG 1" in report["siddon_forward_kernel"]["mix"]
    assert report["siddon_scatter_kernel"]["per"] <= 37.0 and "REDG 1" in report["siddon_scatter_kernel"]["mix"]

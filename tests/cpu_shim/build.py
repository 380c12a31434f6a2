"""TEST INFRASTRUCTURE.  Builds tests/cpu_shim/build/libcbct_cpu_shim.so: the library's own .cu sources, rewritten by
cu2cpp.py and compiled with g++ against the stand-in CUDA headers of this directory (README.md).  Used only by
`-m "not gpu"` tests; the package never builds, loads or imports it."""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_1008_2042_b200", "csrc")
OUT = os.path.join(HERE, "build")
LIB = os.path.join(OUT, "libcbct_cpu_shim.so")

sys.path.insert(0, HERE)
import cu2cpp  # noqa: E402

# -mfma + contraction: a*b+c becomes one fused multiply-add, as nvcc's default -fmad=true does on the device
# SHIM_CXX_EXTRA="-fsanitize=alignment,bounds -fno-sanitize-recover=all" adds UBSan's checks of vector-typed accesses and fixed arrays
EXTRA = os.environ.get("SHIM_CXX_EXTRA", "").split()
CXXFLAGS = EXTRA + ["-DCBCT_TEST_FAULTS", "-std=c++17", "-O2", "-g", "-fPIC", "-fopenmp", "-mavx2", "-mfma", "-ffp-contract=fast", "-fno-strict-aliasing",
            "-Wno-unknown-pragmas", "-Wno-attributes",
            "-I", os.path.join(HERE, "include"), "-I", CSRC, "-I", os.path.join(ROOT, "include"), "-include", "shim_ptx.h"]


def _deps():
    d = glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(ROOT, "include", "*.h"))
    d += glob.glob(os.path.join(HERE, "include", "*.h")) + [os.path.join(HERE, f) for f in ("shim_runtime.cpp", "cu2cpp.py", "build.py")]
    return d


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(d) <= os.path.getmtime(LIB) for d in _deps()):
        return LIB
    gen = os.path.join(OUT, "gen")
    os.makedirs(gen, exist_ok=True)
    jobs = []
    for cu in sorted(glob.glob(os.path.join(CSRC, "*.cu"))):
        cpp = os.path.join(gen, os.path.basename(cu)[:-3] + ".cpp")
        with open(cu) as f:
            text = cu2cpp.transform(f.read(), cu)
        with open(cpp, "w") as f:
            f.write(text)
        jobs.append(cpp)
    jobs.append(os.path.join(HERE, "shim_runtime.cpp"))
    procs, objs = [], []
    for src in jobs:
        obj = os.path.join(OUT, os.path.basename(src).rsplit(".", 1)[0] + ".o")
        objs.append(obj)
        procs.append((src, subprocess.Popen(["g++", *CXXFLAGS, "-c", src, "-o", obj], stdout=subprocess.PIPE,
                                            stderr=subprocess.STDOUT, text=True)))
    bad = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode:
            sys.stderr.write(f"--- {src}\n{out}\n")
            bad = True
    if bad:
        raise RuntimeError("g++ failed on the CPU shim build")
    subprocess.run(["g++", *EXTRA, "-shared", "-fopenmp", "-o", LIB + ".tmp", *objs, "-ldl"], check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))

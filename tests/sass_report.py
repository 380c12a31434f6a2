"""Instruction mix of the hot loops of the projector kernels, from the SASS of the built objects (no GPU needed).

    python tests/sass_report.py            # markdown table on stdout   (TEST TOOLING: tests/test_sass_budget.py is its user)
    python tests/sass_report.py --resources   # registers / shared memory / Blackwell-specific opcodes per kernel of the built library

For every instantiation of forward_tma_kernel / backproject_scatter_kernel / the Siddon kernels in
paper_1008_2042_b200/build/*.o it finds the innermost loop that contains the kernel's shared-memory loads (LDS), shared
reductions (ATOMS) or global loads / reductions (LDG / RED) and counts its instructions by opcode.  The packed kernels
process two samples per iteration; the table divides accordingly.  This is static evidence (what the compiler emitted),
not a measurement: DESIGN.md §5 and profiles/ use it next to the ncu counters.
"""
from __future__ import annotations

import glob
import os
import re
import subprocess
import sys
from collections import Counter

HERE = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_1008_2042_b200")
KERNELS = {"forward_tma_kernel": "LDS", "backproject_scatter_kernel": "ATOMS", "siddon_forward_kernel": "LDG",
           "siddon_scatter_kernel": "RED"}


def demangle(name: str) -> str:
    try:
        return subprocess.run(["c++filt", name], capture_output=True, text=True, check=True).stdout.strip().split("(")[0]
    except Exception:
        return name


def loops(func_text: str, marker: str):
    lines = [l for l in func_text.split("\n") if re.match(r"\s+/\*[0-9a-f]{4}\*/", l)]
    ins = [(int(re.search(r"/\*([0-9a-f]{4})\*/", l).group(1), 16), re.sub(r"/\*.*?\*/", "", l).strip()) for l in lines]
    best = None
    per_iter = {"LDS": 8, "ATOMS": 8, "LDG": 1, "RED": 1}[marker]
    for addr, text in ins:
        m = re.search(r"BRA.*0x([0-9a-f]+)", text)
        if not m or int(m.group(1), 16) >= addr:
            continue
        body = [x for x in ins if int(m.group(1), 16) <= x[0] <= addr]
        n_mark = sum(marker in x[1] for x in body)
        if n_mark >= per_iter and (best is None or len(body) < len(best[0])):      # the tightest loop holding a whole sample
            best = (body, n_mark)
    return best


def resources() -> int:
    """registers, static shared memory and the opcodes that show a Blackwell-native kernel (B200_PROFILING.md: UTMALDG /
    UTMAREDG = TMA tensor copy / reduction, SYNCS = mbarrier, FFMA2 / FADD2 / FMUL2 = packed fp32 pairs, ATOMS = shared-memory
    atomics), per kernel of libcbct_b200.so; template instantiations that differ only in box pitches share a row"""
    lib = os.path.join(HERE, "libcbct_b200.so")
    usage = subprocess.run(["cuobjdump", "--dump-resource-usage", lib], capture_output=True, text=True).stdout
    res = {}
    for m in re.finditer(r"Function (\S+):\n\s*REG:(\d+).*?SHARED:(\d+)", usage):
        res[m.group(1)] = (int(m.group(2)), int(m.group(3)))
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True).stdout
    ops = ("UTMALDG", "UTMAREDG", "SYNCS", "FFMA2", "FADD2", "FMUL2", "ATOMS.ADD", "LDS", "REDG", "BAR")
    rows = {}
    for chunk in re.split(r"\n\s*Function : ", sass)[1:]:
        mangled = chunk.split("\n")[0].strip()
        name = re.sub(r"<\d+, \d+", "<BF, BS", demangle(mangled).replace("cbct::", "").replace("void ", ""))
        body = [re.sub(r"/\*.*?\*/", "", l).strip() for l in chunk.split("\n") if re.match(r"\s+/\*[0-9a-f]{4}\*/", l)]
        cnt = tuple(sum(1 for x in body if re.search(r"\b" + re.escape(o), x)) for o in ops)
        key = (name,) + res.get(mangled, (0, 0)) + cnt
        rows[key] = rows.get(key, 0) + 1
    print("| kernel | instantiations | registers | static smem B | " + " | ".join(ops) + " |")
    print("|---|---|---|---|" + "---|" * len(ops))
    for key in sorted(rows):
        print(f"| `{key[0]}` | {rows[key]} | {key[1]} | {key[2]} | " + " | ".join(str(v) for v in key[3:]) + " |")
    return 0


def main() -> int:
    if "--resources" in sys.argv:
        return resources()
    rows = []
    for obj in sorted(glob.glob(os.path.join(HERE, "build", "*.o"))):
        sass = subprocess.run(["cuobjdump", "-sass", obj], capture_output=True, text=True).stdout
        for chunk in re.split(r"\n\s*Function : ", sass)[1:]:
            mangled = chunk.split("\n")[0].strip()
            for kern, marker in KERNELS.items():
                if kern not in mangled:
                    continue
                found = loops(chunk, marker)
                if not found:
                    continue
                body, n_mark = found
                per_iter = {"LDS": 8, "ATOMS": 8, "LDG": 1, "RED": 1}[marker]
                samples = max(1, n_mark // per_iter)
                mix = Counter(re.sub(r"^@!?U?P\d+\s+", "", x[1]).split()[0].split(".")[0] for x in body)
                rows.append((demangle(mangled).replace("cbct::", ""), len(body), samples, len(body) / samples,
                             ", ".join(f"{k} {v}" for k, v in mix.most_common())))
    print("| kernel | loop instructions | samples (steps) per iteration | per sample | mix |")
    print("|---|---|---|---|---|")
    seen = {}
    for r in rows:                                       # instantiations that differ only in the box pitches share a row
        key = (re.sub(r"<\d+, \d+", "<BF, BS", r[0]), r[1], r[4])
        seen.setdefault(key, []).append(r)
    for (name, n, mix), group in seen.items():
        r = group[0]
        print(f"| `{name}` ({len(group)} instantiations) | {n} | {r[2]} | {r[3]:.1f} | {mix} |")
    return 0


if __name__ == "__main__":
    sys.exit(main())

"""TEST INFRASTRUCTURE.  Source-to-source pre-pass that makes a .cu file acceptable to g++ (see README.md here).

Only the two constructs that no header can emulate are rewritten; every other line is passed through untouched:

  kernel<<<grid, block[, smem[, stream]]>>>(args);   ->  SHIM_LAUNCH(kernel, dim3(grid), dim3(block), smem, stream, args);
  __shared__ T a[N], b;                              ->  one guarded, per-block allocation per declarator
  extern __shared__ T name[];                        ->  pointer to the launch's dynamic shared memory
"""
from __future__ import annotations

import re


def _split_top(s: str):
    """split at commas that are not nested in (), [] or {}"""
    out, depth, cur = [], 0, []
    for ch in s:
        if ch in "([{":
            depth += 1
        elif ch in ")]}":
            depth -= 1
        if ch == "," and depth == 0:
            out.append("".join(cur).strip())
            cur = []
        else:
            cur.append(ch)
    out.append("".join(cur).strip())
    return out


def _rewrite_launches(src: str) -> str:
    out, pos = [], 0
    while True:
        i = src.find("<<<", pos)
        if i < 0:
            out.append(src[pos:])
            return "".join(out)
        # kernel expression: identifier, optionally followed by one balanced <...> group, right before <<<
        j = i
        if src[j - 1] == ">":
            depth, j = 0, j - 1
            while True:
                if src[j] == ">":
                    depth += 1
                elif src[j] == "<":
                    depth -= 1
                    if depth == 0:
                        break
                j -= 1
        while j > 0 and (src[j - 1].isalnum() or src[j - 1] in "_:"):
            j -= 1
        kernel = src[j:i]
        k = src.index(">>>", i)
        cfg = _split_top(src[i + 3:k])
        assert 2 <= len(cfg) <= 4, f"launch configuration not understood: {src[i:k + 3]}"
        cfg += ["0", "nullptr"][len(cfg) - 2:]
        p = src.index("(", k)
        assert src[k + 3:p].strip() == "", "text between >>> and ("
        depth, q = 0, p
        while True:
            if src[q] == "(":
                depth += 1
            elif src[q] == ")":
                depth -= 1
                if depth == 0:
                    break
            q += 1
        args = src[p + 1:q].strip()
        call = (f"SHIM_LAUNCH(({kernel}), dim3({cfg[0]}), dim3({cfg[1]}), (size_t)({cfg[2]}), (cudaStream_t)({cfg[3]})"
                + (", " + args if args else "") + ")")
        out.append(src[pos:j])
        out.append(call)
        pos = q + 1


_SHARED = re.compile(r"^(\s*)(extern\s+)?__shared__\s+(?:__align__\(\s*\d+\s*\)\s+)?([^;]+);(.*)$")
_DECL = re.compile(r"^(?:(.*\S)\s+)?(\w+)\s*((?:\[[^\]]*\])*)$")


def _rewrite_shared(src: str) -> str:
    lines = []
    for line in src.split("\n"):
        m = _SHARED.match(line)
        if not m:
            assert "__shared__" not in line.split("//")[0], f"__shared__ declaration not understood: {line}"
            lines.append(line)
            continue
        indent, ext, body, tail = m.group(1), m.group(2), m.group(3), m.group(4)
        pieces = _split_top(body)
        first = _DECL.match(pieces[0])
        ctype = first.group(1)
        decls = [(first.group(2), first.group(3))] + [(_DECL.match(p).group(2), _DECL.match(p).group(3)) for p in pieces[1:]]
        stmts = []
        for name, dims in decls:
            if ext:
                assert dims == "[]", line
                stmts.append(f"{ctype} *{name} = static_cast<{ctype} *>(::shim::dyn_smem());")
            else:
                stmts.append(f"static char _shk_{name}; auto &{name} = *::shim::sh<{ctype}{dims}>(&_shk_{name});")
        lines.append(indent + " ".join(stmts) + tail)
    return "\n".join(lines)


def transform(src: str, path: str) -> str:
    return f'#line 1 "{path}"\n' + _rewrite_shared(_rewrite_launches(src))

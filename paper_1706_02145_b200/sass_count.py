"""FP32 work per sphere pair, counted in the SASS of the built library (ties the roofline to the build).

    python -m paper_1706_02145_b200.sass_count [--write] [--lmax 3 4 5]

The coupling kernel's emitter loop (``for e in tile``, csrc/coupling_kernel.cuh) is one straight-line SASS loop: every
instruction between the target of its backward branch and the branch is executed once per ordered pair.  This module
dumps one kernel with ``cuobjdump -sass -fun`` (works without a GPU), finds that loop (the innermost backward branch
with the most FP32 work) and returns the opcode histogram of its body plus

    flops    = 4 FFMA2 + 2 (FMUL2 + FADD2) + 2 FFMA + FMUL + FADD          (an FMA is two flop)
    lane_ops = 2 (FFMA2 + FMUL2 + FADD2) + FFMA + FMUL + FADD              (FMA-pipe lane slots: 128 per SM per clock)

``bench.py`` takes its roofline numerators from here (live from the built ``libceles.so``; the committed
``csrc/generated/sass_counts.json`` only if cuobjdump is missing), and ``tests/test_host_logic.py`` asserts that the
committed file equals the live count, so an edit of a generator cannot silently invalidate ``roofline.frac``.
ncu cannot supply these numbers: its ``sass_thread_inst_executed_op_ffma`` counters do not see the packed FFMA2.
"""
from __future__ import annotations

import collections
import json
import os
import re
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libceles.so")
COMMITTED = os.path.join(HERE, "csrc", "generated", "sass_counts.json")
VARIANTS = {"rotated": 0, "direct": 1}
FP32_OPS = ("FFMA2", "FMUL2", "FADD2", "FFMA", "FMUL", "FADD")
_LINE = re.compile(r"/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_]*)((?:\.[A-Za-z0-9_]+)*)\s*([^;]*);")


def cuobjdump() -> str | None:
    return shutil.which("cuobjdump") or ("/usr/local/cuda/bin/cuobjdump" if os.path.exists("/usr/local/cuda/bin/cuobjdump") else None)


def coupling_symbol(lmax: int, variant: int = 0, table: bool = False, extended: bool = False, lib: str = LIB) -> str:
    """Mangled name of coupling_kernel<lmax, variant, table, extended>, looked up in the library's symbol table (the
    argument list is part of the name, so it is not spelled out here)."""
    exe = cuobjdump()
    if exe is None:
        raise RuntimeError("cuobjdump not found")
    prefix = f"_ZN5celes15coupling_kernelILi{lmax}ELi{variant}ELb{int(table)}ELb{int(extended)}EEE"
    out = subprocess.run([exe, "-symbols", lib], capture_output=True, text=True, check=False).stdout
    for tok in out.split():
        if tok.startswith(prefix):
            return tok
    raise RuntimeError(f"no symbol {prefix}* in {lib}")


def dump(symbol: str, lib: str = LIB) -> str:
    """SASS text of one kernel of the library (the other translation units answer 'not found' on stderr)."""
    exe = cuobjdump()
    if exe is None:
        raise RuntimeError("cuobjdump not found")
    out = subprocess.run([exe, "-sass", "-fun", symbol, lib], capture_output=True, text=True, check=False).stdout
    if "Function :" not in out:
        raise RuntimeError(f"{symbol} not found in {lib}")
    return out


def instructions(sass: str) -> list[tuple[int, str, str]]:
    """[(address, opcode without modifiers, operands)]"""
    out = []
    for line in sass.splitlines():
        m = _LINE.search(line)
        if m:
            out.append((int(m.group(1), 16), m.group(2), m.group(4).strip()))
    return out


def fp32_work(hist: dict) -> tuple[int, int]:
    g = lambda k: int(hist.get(k, 0))
    flops = 4 * g("FFMA2") + 2 * (g("FMUL2") + g("FADD2")) + 2 * g("FFMA") + g("FMUL") + g("FADD")
    lane = 2 * (g("FFMA2") + g("FMUL2") + g("FADD2")) + g("FFMA") + g("FMUL") + g("FADD")
    return flops, lane


def pair_loop(instrs: list[tuple[int, str, str]]) -> list[tuple[int, str, str]]:
    """Body of the per-pair loop: among the innermost backward branches, the span with the most FP32 lane operations."""
    loops = []
    for addr, op, args in instrs:
        if op == "BRA":
            m = re.search(r"0x([0-9a-f]+)", args)
            if m and int(m.group(1), 16) <= addr:
                loops.append((int(m.group(1), 16), addr))
    inner = [(a, b) for (a, b) in loops if not any((c, d) != (a, b) and a <= c and d <= b for (c, d) in loops)]
    best, best_lane = [], -1
    for a, b in inner:
        body = [t for t in instrs if a <= t[0] <= b]
        lane = fp32_work(collections.Counter(op for _, op, _ in body))[1]
        if lane > best_lane:
            best, best_lane = body, lane
    return best


def count_kernel(symbol: str, lib: str = LIB) -> dict:
    body = pair_loop(instructions(dump(symbol, lib)))
    hist = collections.Counter(op for _, op, _ in body)
    flops, lane = fp32_work(hist)
    packed = hist["FFMA2"] + hist["FMUL2"] + hist["FADD2"]
    return {"symbol": symbol, "instructions": len(body), "histogram": dict(sorted(hist.items(), key=lambda kv: (-kv[1], kv[0]))),
            "fp32": {k: int(hist.get(k, 0)) for k in FP32_OPS}, "mufu": int(hist.get("MUFU", 0)),
            "packed": packed, "packed_non_fma": hist["FMUL2"] + hist["FADD2"],
            "flops_per_pair": flops, "lane_ops_per_pair": lane}


def coupling_counts(lmax: int, translation: str = "rotated", table: bool = False, extended: bool = False, lib: str = LIB) -> dict:
    return count_kernel(coupling_symbol(lmax, VARIANTS[translation], table, extended, lib), lib)


def committed() -> dict:
    with open(COMMITTED) as f:
        return json.load(f)


def counts_for_bench(lmax: int, translation: str = "rotated") -> dict:
    """Live count from the built library; the committed file (equal to it by test) if cuobjdump is unavailable."""
    try:
        c = coupling_counts(lmax, translation)
        c["source"] = "cuobjdump -sass of the loaded libceles.so (live)"
        return c
    except (RuntimeError, OSError):
        c = committed()[f"{translation}/{lmax}"]
        c["source"] = "csrc/generated/sass_counts.json (committed; tests assert it equals the built library)"
        return c


def summary(keys=None) -> dict:
    out = {}
    for tr, v in VARIANTS.items():
        for L in (1, 2, 3, 4, 5):
            if tr == "direct" and L == 5:
                continue
            if keys and f"{tr}/{L}" not in keys:
                continue
            c = coupling_counts(L, tr)
            out[f"{tr}/{L}"] = {k: c[k] for k in ("instructions", "fp32", "mufu", "packed", "packed_non_fma",
                                                  "flops_per_pair", "lane_ops_per_pair")}
    return out


if __name__ == "__main__":
    s = summary()
    if "--write" in sys.argv:
        with open(COMMITTED, "w") as f:
            json.dump(s, f, indent=1, sort_keys=True)
            f.write("\n")
        print("wrote", COMMITTED)
    for k, v in s.items():
        print(k, json.dumps(v))

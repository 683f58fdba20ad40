"""SASS opcode histogram of a kernel of libjerk_b200.so, whole function and innermost hot loop (measurement aid).

    python -m paper_1911_01353_b200.sass_histogram '_ZN4jerk10k_search64ILi1ELi2ELb1EEEvNS_12SearchParamsE'

The hot loop is taken as the backward branch whose body holds the most packed FP32 instructions (for k_search64: the
loop over the template-phases of a work item, rows a-3 .. a-5 of SURVEY.md 8(a)).  Executed FP32 flops per trip are
derived from the opcode counts: FFMA2 = 4, FADD2 / FMUL2 = 2, FFMA = 2, FADD / FMUL = 1 per thread -- the ncu counters
sm__sass_thread_inst_executed_op_{fadd,fmul,ffma}_pred_on do not count the packed forms.  Needs cuobjdump (CUDA toolkit);
reads the built library only, no GPU."""
from __future__ import annotations

import collections
import re
import subprocess
import sys

from . import build as _build

_INSN = re.compile(r"^\s*/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)\s*(.*?);")

FLOPS = {"FFMA2": 4, "FADD2": 2, "FMUL2": 2, "FFMA": 2, "FADD": 1, "FMUL": 1}
FMA_PIPE_CYCLES = {"FFMA2": 2, "FADD2": 2, "FMUL2": 2, "FFMA": 1, "FADD": 1, "FMUL": 1}


def disassemble(symbol: str, lib: str | None = None) -> list[tuple[int, str, str]]:
    """[(address, opcode with modifiers, operands)] of one kernel."""
    out = subprocess.run(["cuobjdump", "-sass", "-fun", symbol, lib or _build.LIB], capture_output=True, text=True, check=True).stdout
    insns = []
    for line in out.splitlines():
        m = _INSN.match(line)
        if m:
            insns.append((int(m.group(1), 16), m.group(2), m.group(3)))
    return insns


def histogram(insns) -> collections.Counter:
    return collections.Counter(op.split(".")[0] for _, op, _ in insns)


def loops(insns) -> list[tuple[int, int]]:
    """(target, branch address) of every backward branch."""
    res = []
    for addr, op, args in insns:
        if op.startswith("BRA"):
            m = re.search(r"0x([0-9a-f]+)", args)
            if m and int(m.group(1), 16) <= addr:
                res.append((int(m.group(1), 16), addr))
    return res


def hot_loop(insns) -> tuple[int, int]:
    def packed(lo, hi):
        return sum(1 for a, op, _ in insns if lo <= a <= hi and op.split(".")[0] in ("FFMA2", "FADD2", "FMUL2"))
    cands = [(packed(lo, hi), -(hi - lo), lo, hi) for lo, hi in loops(insns)]
    best = max(c[0] for c in cands)
    # smallest loop among those that hold at least 45 % of the packed arithmetic of the largest one (the loop over work
    # items also contains the forward transform of the segment: half of the packed instructions of the function)
    _, _, lo, hi = max((c for c in cands if c[0] >= 0.45 * best), key=lambda c: c[1])
    return lo, hi


def report(symbol: str, lib: str | None = None) -> str:
    insns = disassemble(symbol, lib)
    lines = [f"kernel {symbol}", f"instructions: {len(insns)}"]
    lo, hi = hot_loop(insns)
    body = [i for i in insns if lo <= i[0] <= hi]
    for title, part in (("whole function", insns), (f"hot loop 0x{lo:x}..0x{hi:x} ({len(body)} instructions)", body)):
        h = histogram(part)
        lines.append(f"-- {title}")
        for op, n in sorted(h.items(), key=lambda kv: -kv[1]):
            lines.append(f"{op:12s} {n:6d}")
        flops = sum(FLOPS.get(op, 0) * n for op, n in h.items())
        cyc = sum(FMA_PIPE_CYCLES.get(op, 0) * n for op, n in h.items())
        lines.append(f"FP32 flops per thread (static count): {flops}; FMA-pipe issue cycles per warp: {cyc}")
    return "\n".join(lines)


if __name__ == "__main__":
    print(report(sys.argv[1], sys.argv[2] if len(sys.argv) > 2 else None))

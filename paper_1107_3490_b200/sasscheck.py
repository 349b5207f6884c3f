"""Static check of the schedule ptxas chose for the step loops of the fp64 sweep kernels (DESIGN.md section 7,
"ptxas and the schedule").

    python -m paper_1107_3490_b200.sasscheck [pattern]

For identical arithmetic ptxas sometimes interleaves the partners of a pair group (dependent fp64 instructions 5-10
slots apart) and sometimes runs them nearly one after the other (1-3 slots apart: the warp then waits on the 8-cycle
DFMA latency, measured up to +25 % time).  Per step loop this module counts the fp64 instructions whose nearest fp64
producer is at most three instructions ahead; a loop where more than a fifth of them are that close is reported as
serialised.  It reads the objects build.py leaves in paper_1107_3490_b200/build/ with cuobjdump; no GPU is needed.
"""
from __future__ import annotations

import re
import subprocess
import sys
from pathlib import Path

OBJ = Path(__file__).resolve().parent / "build"
_F64 = ("DFMA", "DADD", "DMUL", "DSET")


def _is_f64(s: str) -> bool:
    return re.sub(r"^@!?U?P\d+\s+", "", s).split()[0][:4] in _F64


def loops_of(obj: Path, pattern: str = "k_sweep"):
    """Yields (kernel name, [(instructions, fp64 instructions, close dependences), ...]) for every kernel of `obj`
    whose mangled name contains `pattern`; one tuple per backward-branch loop with more than 150 fp64 instructions."""
    txt = subprocess.run(["cuobjdump", "-sass", str(obj)], capture_output=True, text=True, check=True).stdout
    funcs, cur = {}, None
    for line in txt.split("\n"):
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            funcs[cur] = []
            continue
        if cur:
            m = re.search(r"/\*([0-9a-f]{4,5})\*/\s+(.*?);", line)
            if m:
                funcs[cur].append((int(m.group(1), 16), m.group(2).strip()))
    for fn, ins in funcs.items():
        if pattern not in fn:
            continue
        loops = []
        for a, s in ins:
            m = re.search(r"BRA\S*\s+(?:!?U?P\d+,\s*)?0x([0-9a-f]+)", s)
            if m and int(m.group(1), 16) < a and (a - int(m.group(1), 16)) // 16 < 1000:
                loops.append((int(m.group(1), 16), a))
        out = []
        for t, a in loops:
            body = [s for ad, s in ins if t <= ad <= a]
            nf = sum(1 for s in body if _is_f64(s))
            if nf <= 150:
                continue
            last, close = {}, 0
            for i, s in enumerate(body):
                s2 = re.sub(r"^@!?U?P\d+\s+", "", s)
                regs = [int(x) for x in re.findall(r"R(\d+)", s2)]
                if not regs:
                    continue
                f = _is_f64(s)
                dst, src = ([], regs) if s2.split()[0].startswith("DSETP") else (regs[:1], regs[1:])
                if f:
                    d = min((i - last[rr][0] for r in src for rr in (r, r + 1) if rr in last and last[rr][1]), default=None)
                    if d is not None and d <= 3:
                        close += 1
                for r in dst:
                    last[r] = (i, f)
                    if f:
                        last[r + 1] = (i, f)
            out.append((len(body), nf, close))
        yield fn, out


def serialised(pattern: str = "k_sweep", objects=None, min_f64: int = 200, ratio: float = 0.2):
    """[(kernel, loop)] of the step loops (>= min_f64 fp64 instructions) that ptxas serialised."""
    bad = []
    for obj in sorted(objects or OBJ.glob("pt_sweep_comp*.o")):
        for fn, loops in loops_of(obj, pattern):
            for lp in loops:
                if lp[1] >= min_f64 and lp[2] > ratio * lp[1]:
                    bad.append((fn, lp))
    return bad


if __name__ == "__main__":
    pat = sys.argv[1] if len(sys.argv) > 1 else "k_sweep"
    for obj in sorted(OBJ.glob("pt_sweep_*.o")):
        for fn, loops in loops_of(obj, pat):
            name = re.sub(r"_ZN\d+_GLOBAL__N__\w+?_cu_\w+?\d+k_sweep", "k_sweep", fn)[:64]
            print(f"{name:64s} " + " ".join(f"[n={n} f64={f} close={c}]" for n, f, c in loops))

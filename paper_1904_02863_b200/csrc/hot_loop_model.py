#!/usr/bin/env python3
"""The issue-cycle model of the fused kernel's hot loop, computed from the SASS of the built library (no GPU needed).

    python paper_1904_02863_b200/csrc/hot_loop_model.py [--lib csrc/libgwlnl.so] [--ndet 3] [--all]

Finds the innermost loop with the most fp64 instructions in `gw::fused_kernel<NDET, MULTI, ISCO, TIDAL>` (cuobjdump -sass)
and counts, per trip (GW_UNROLL = 5 bins):

  fp64      DFMA / DMUL / DADD
  fresh3    DFMAs whose three source operands are 64-bit registers none of which is served by the operand-reuse cache
            (none equals the register the previous fp64 instruction flagged `.reuse` in the same slot)
  lds       shared-memory loads (the warp-broadcast table reads)
  others    everything else (conversion pipe, integer, select, uniform datapath, branch)

and the model  cycles = 2 fp64 + fresh3 + 0.6 (lds + others)  validated against the GPU in profiles/
r1_fp64_operand_probe.md and r2_fused_hot_loop_sass.md (113.8 cycles per (warp, bin) for NDET = 3; ncu and the per-CTA
timeline measure 113.7-113.9).  ptxas's register allocation for this loop is fragile at the 128-register limit: a branch
added OUTSIDE the loop has cost it 5 %, so tests/test_hot_loop_model.py holds the product build
to the numbers below.
"""
import argparse
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CUOBJDUMP = os.environ.get("CUOBJDUMP", "/usr/local/cuda/bin/cuobjdump")


def mangled(ndet: int, multi: int = 0, isco: int = 0, tidal: int = 0) -> str:
    return f"_ZN2gw12fused_kernelILi{ndet}ELb{multi}ELb{isco}ELb{tidal}EEEvNS_9FusedArgsE"


def sass_of(lib: str, function: str):
    out = subprocess.run([CUOBJDUMP, "-sass", "-fun", function, lib], capture_output=True, text=True, check=True).stdout
    ins = []
    for line in out.splitlines():
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
        if m:
            ins.append((int(m.group(1), 16), m.group(2).strip()))
    return ins


def hot_loop(ins):
    """(first address, last address, instructions) of the innermost loop with the most fp64 instructions."""
    loops = []
    for a, t in ins:
        m = re.search(r"\bBRA\S*\s+(?:!?U?P\d+,\s*)?0x([0-9a-f]+)", t)
        if m and int(m.group(1), 16) < a:
            loops.append((int(m.group(1), 16), a))
    inner = [(lo, hi) for lo, hi in loops if not any((l2, h2) != (lo, hi) and lo <= l2 and h2 <= hi for l2, h2 in loops)]
    best = None
    for lo, hi in inner:
        body = [(a, t) for a, t in ins if lo <= a <= hi]
        n64 = sum(1 for _, t in body if re.search(r"\b(DFMA|DMUL|DADD)\b", t))
        if best is None or n64 > best[0]:
            best = (n64, lo, hi, body)
    if best is None:
        raise RuntimeError("no loop found")
    return best[1], best[2], best[3]


def model(lib: str, ndet: int = 3, multi: int = 0, isco: int = 0, tidal: int = 0) -> dict:
    lo, hi, body = hot_loop(sass_of(lib, mangled(ndet, multi, isco, tidal)))
    fp64 = fresh3 = lds = spill = 0
    last = [None, None, None]                      # register flagged .reuse per operand slot by the previous fp64 instruction
    for _, t in body:
        if re.search(r"\b(LDL|STL)", t):
            spill += 1
        if re.match(r"(?:@!?U?P\d+\s+)?LDS", t):
            lds += 1
        m = re.match(r"(?:@!?U?P\d+\s+)?(DFMA|DMUL|DADD)\s+\S+,\s*(.*)", t)
        if not m:
            continue
        fp64 += 1
        regs = []
        for o in m.group(2).split(","):
            mm = re.match(r"\s*[-|]*\s*(R\d+)(\.reuse)?", o)
            regs.append((mm.group(1), bool(mm.group(2))) if mm else None)
        if m.group(1) == "DFMA" and len(regs) == 3 and all(r is not None for r in regs):
            if not any(last[i] is not None and last[i] == regs[i][0] for i in range(3)):
                fresh3 += 1
        last = [(r[0] if (r is not None and r[1]) else None) for r in (regs + [None, None, None])[:3]]
    others = len(body) - fp64 - lds
    cycles = 2 * fp64 + fresh3 + 0.6 * (lds + others)
    return {"function": f"fused_kernel<{ndet},{multi},{isco},{tidal}>", "loop": [hex(lo), hex(hi)], "instructions": len(body),
            "fp64": fp64, "fresh3": fresh3, "lds": lds, "others": others, "spill_in_loop": spill,
            "model_cycles_per_trip": round(cycles, 1)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lib", default=os.path.join(HERE, "libgwlnl.so"))
    ap.add_argument("--ndet", type=int, default=3)
    ap.add_argument("--all", action="store_true", help="every detector count 1..8 and kernel variant")
    args = ap.parse_args()
    if args.all:
        for n in range(1, 9):
            for multi in (0, 1):
                for isco in (0, 1):
                    for tidal in (0, 1):
                        print(model(args.lib, n, multi, isco, tidal))
    else:
        print(model(args.lib, args.ndet))


if __name__ == "__main__":
    main()

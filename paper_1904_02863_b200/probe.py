"""python -m paper_1904_02863_b200.probe -- print the measured fp64 pipe rates of this GPU by operand pattern
(gw_probe_fp64_fma_rate, include/gwlnl.h).  The numbers are the measured roofline denominators of DESIGN.md
section 9; profiles/r1_fp64_operand_probe.md holds one run."""
import json

from .binding import probe_fp64_fma_rate

MODES = {0: "fma(v, imm, imm): one register operand", 1: "fma(a, b, v): three distinct register operands",
         2: "fma(a, m, v): three register operands, one shared by consecutive instructions",
         3: "mma.sync m8n8k4 f64 (DMMA)",
         4: "mode 0 plus 8 independent integer instructions per 8 DFMA (do other pipes issue for free?)",
         5: "mode 0 plus 16 independent integer instructions per 8 DFMA"}


def main():
    probe_fp64_fma_rate(1 << 13, 0)                       # clock ramp
    out = {}
    for mode, what in MODES.items():
        best = max(probe_fp64_fma_rate(1 << 13, mode)[0] for _ in range(3))
        out[mode] = {"pattern": what, "fma_per_s": best, "tflops": 2 * best / 1e12}
        print(f"mode {mode}: {best / 1e12:6.2f} T-FMA/s = {2 * best / 1e12:6.2f} TFLOP/s   {what}")
    print(json.dumps(out))


if __name__ == "__main__":
    main()

"""python -m paper_2004_06352_b200.fp64_probe -- prints the FP64 dispatch-cost table of DESIGN.md sec. 7
(measured through lh_fp64_issue_probe / lh_fp64_peak_probe on the current CUDA device)."""
from __future__ import annotations

from . import lh_fp64_issue_probe, lh_fp64_peak_probe, lh_version

OPERANDS = [(0, "FMA  r = r*imm + imm"), (2, "FMA  2 distinct vector registers"), (3, "MUL  2 vector registers"),
            (5, "FMA  1 register shared by consecutive instr."), (4, "FMA  1 uniform operand (LDCU from params)"),
            (1, "FMA  3 distinct vector registers")]
EXTRAS = [(10, "LOP3"), (11, "FFMA"), (12, "MUFU.RCP64H + MOV"), (13, "LDS.64")]


def main() -> None:
    print(lh_version())
    flops, _ = lh_fp64_peak_probe(1 << 15)
    print(f"lh_fp64_peak_probe: {flops / 1e12:.2f} TFLOP/s (FMA = 2 flop)\n")
    print("| FP64 instruction (12 independent per group) | warps/sub-partition | cycles per instruction |")
    print("|---|---|---|")
    for v, name in OPERANDS:
        for w in (4, 8):
            print(f"| {name} | {w} | {lh_fp64_issue_probe(v, 0, w) / 12:.2f} |")
    print("\n| 12 MUL + K x other instruction | warps/sub-partition | cycles per group | extra cycles per other instr. |")
    print("|---|---|---|---|")
    for w in (4, 8):
        base = lh_fp64_issue_probe(10, 0, w)
        print(f"| (none) | {w} | {base:.2f} | - |")
        for v, name in EXTRAS:
            for k in (2, 4, 8):
                c = lh_fp64_issue_probe(v, k, w)
                print(f"| {k} x {name} | {w} | {c:.2f} | {(c - base) / k:.2f} |")


if __name__ == "__main__":
    main()

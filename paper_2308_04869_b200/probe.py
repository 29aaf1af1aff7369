"""Print the measured ALU peaks and the issue cost of instruction mixes on the current GPU.

    python -m paper_2308_04869_b200.probe

Evidence for the instruction-issue bound of DESIGN.md section 8 (the output is kept under profiles/)."""
from __future__ import annotations

from . import probe_alu_peak, probe_issue_mix

MIXES = [(8, 0, 0), (0, 8, 0), (0, 0, 8), (0, 4, 4), (0, 8, 8), (8, 2, 2), (8, 4, 4), (8, 8, 0), (8, 0, 8), (8, 8, 8)]


def main() -> None:
    for what, name in ((0, "fp64 FMA"), (1, "fp32 FMA"), (2, "int32 multiply-add")):
        print(f"peak {name}: {probe_alu_peak(what, 1 << 17) / 1e12:.2f} T op/s (one FMA = one op)")
    print("cycles per warp-iteration per scheduler (loop overhead of 3 instructions included)")
    print("| DFMA | IMAD | LOP3 | 4 warps/SM | 8 | 16 | 32 |")
    print("|---|---|---|---|---|---|---|")
    for nd, ni, nl in MIXES:
        row = [probe_issue_mix(nd, ni, nl, w) / (w / 4.0) for w in (4, 8, 16, 32)]
        print(f"| {nd} | {ni} | {nl} | " + " | ".join(f"{v:.2f}" for v in row) + " |")


if __name__ == "__main__":
    main()

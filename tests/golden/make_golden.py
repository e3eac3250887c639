"""Writes tests/golden/*.txt from the ORACLE ALONE (never from the CUDA path).

  cfg1_norms.txt   ||f - A u||_2 before each of the 10 cycles of BASELINE.json configs[0] and after
                   the last one (Algorithm H == Algorithm L, schedule "C", MaxI = 4).
  paper_L1.txt     the paper's own printed numbers: L1 error (Eq. 7) after one MFMG
                   cycle, MaxI = 4 -> 5 %, MaxI = 32 -> 1.6 %.  Written by hand below, with citation.

Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import oracle as O                      # noqa: E402
from paper_1108_2045_b200 import inputs as I        # noqa: E402


def main():
    c = I.CONFIGS["cfg1"]
    inp = I.make_inputs(c)
    _, _, n = O.homg("H", inp["f"], inp["u0"], c.levels, c.omega, O.schedule(0, c.levels, c.max_iters), c.cycles,
                     keep_history=False)
    with open(os.path.join(HERE, "cfg1_norms.txt"), "w") as fh:
        fh.write("# oracle Algorithm H, cfg1 (129^2 fp64, omega 4/5, schedule C, MaxI 4): residual 2-norms, cycles 0..10\n")
        for v in n:
            fh.write(f"{v:.17e}\n")
    with open(os.path.join(HERE, "paper_L1.txt"), "w") as fh:
        fh.write("# PAPER.md L119: 'MaxI = 4 reaches an error of 5% and MaxI = 32 reaches an error of 1.6%' (Eq. 7, one MFMG cycle)\n")
        fh.write("4 0.05\n32 0.016\n")


if __name__ == "__main__":
    main()

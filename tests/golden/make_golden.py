"""Writes the stored expected values under tests/golden/.  Calls ONLY oracle/ (never the CUDA path).

    python tests/golden/make_golden.py

cfg1_modal.txt : config 1 of BASELINE.json (N1=N2=128, tau=h/2, M=100, c=1, phi = sin(pi x) sin(pi y)):
                 amplitude of the (1,1) mode of u^M, obtained by projecting the oracle's full 2D result
                 onto the mode.  Checked in tests/test_oracle_pins.py against the independent scalar modal
                 recurrence (SURVEY.md 8c pin 3) and the PDE closed form of north_star.
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle  # noqa: E402
from paper_2006_10142_b200 import workloads as W  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def run(w, steps=None):
    return oracle.solve(w.N1, w.N2, w.l, w.tau, w.M, w.phi, w.psi, c_half=w.c_half, s=w.s, g_half=w.g_half,
                        steps=steps)


def main():
    w = W.cfg1()
    u = run(w)
    amp = float((u * w.phi).sum() / (w.phi * w.phi).sum())
    with open(os.path.join(HERE, "cfg1_modal.txt"), "w") as f:
        f.write("# config 1 (BASELINE.json configs[0]): (1,1)-mode amplitude of u^100, oracle 2D run projected on the mode\n")
        f.write("# written by tests/golden/make_golden.py (calls oracle/ only)\n")
        f.write(f"{amp:.17e}\n")
    print("cfg1 amplitude", amp)


if __name__ == "__main__":
    main()

"""Writes tests/golden/p13_golden.txt.  Calls only oracle/ (the pure-Python brute force).

Worked example P13 of SURVEY.md §8(c): I_t(x,y) = 100 + ((3x + 5y + 7t) mod 11), W=H=8, t=0..3,
lags {1,2,3}, n_b=4.  The paper prints no worked example, so the stored values are the
definition evaluated by oracle/brute_force.py — explicit loops, no FFT —
and they agree to 12 digits with the values SURVEY.md §8(c) P13 lists from two further
independent computations (checked in tests/test_oracle_pins.py).
Run:  python tests/golden/make_p13_golden.py
"""
import os
import sys

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", ".."))
from oracle import brute_force as bf  # noqa: E402

W = H = 8
N = 4
LAGS = [1, 2, 3]
NB = 4


def frames():
    return [[[100 + ((3 * x + 5 * y + 7 * t) % 11) for x in range(W)] for y in range(H)] for t in range(N)]


def main():
    r = bf.structure_function(frames(), LAGS, NB)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "p13_golden.txt")
    with open(out, "w") as f:
        f.write("# P13 golden vector (SURVEY.md §8(c) P13; definition PAPER.md:L21,L25,L31)\n")
        f.write("# written by tests/golden/make_p13_golden.py from oracle/brute_force.py\n")
        f.write("sums " + " ".join(str(s) for s in r["sums"]) + "\n")
        f.write("counts " + " ".join(str(c) for c in r["counts"]) + "\n")
        f.write("n_pairs " + " ".join(str(c) for c in r["n_pairs"]) + "\n")
        for l, tau in enumerate(LAGS):
            f.write("D %d " % tau + " ".join("%.15e" % v for v in r["D"][l]) + "\n")
        f.write("I " + " ".join("%.15e" % v for v in r["I_q"]) + "\n")
        f.write("D2d_ky0_kx1_tau1 %.15e\n" % r["D2d"][0][0][1])
        f.write("D2d_ky1_kx0_tau1 %.15e\n" % r["D2d"][0][1][0])
        f.write("I2d_dc %.15e\n" % r["I2d"][0][0])
        f.write("D2d_dc_tau1 %.3e\n" % r["D2d"][0][0][0])
    print(open(out).read())


if __name__ == "__main__":
    main()

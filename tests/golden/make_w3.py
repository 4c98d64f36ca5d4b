"""Writes tests/golden/w3.txt -- worked example W3 of SURVEY.md 8(c) "Pinned values", recomputed from first
principles with 40-digit mpmath.  Calls NOTHING from the CUDA path and nothing from oracle/: the values are the
plain definition acc_i(t) = Sum_j m_j r_ij / (r_ij^2 + eps^2)^(3/2) differentiated 0..3 times in t at t = 0 along
the cubic trajectories x_k(t) = x_k + v_k t + a_k t^2/2 + j_k t^3/6, where a_k, j_k are the example's own
acc/jerk (pass 1), exactly as the two-pass bootstrap c-10 prescribes.  (The paper itself prints no worked
example -- PAPER.md has no formula or table of values.)

Run:  python tests/golden/make_w3.py
"""
import os

import mpmath as mp

mp.mp.dps = 40
M = [mp.mpf("0.5"), mp.mpf("0.3"), mp.mpf("0.2")]
X = [[mp.mpf(s) for s in r] for r in (("1", "0", "0"), ("-0.5", "0.7", "0.1"), ("0.2", "-0.9", "-0.4"))]
V = [[mp.mpf(s) for s in r] for r in (("0", "0.4", "0.1"), ("-0.3", "-0.2", "0.2"), ("0.5", "0.1", "-0.3"))]
EPS2 = mp.mpf("0.01")


def acc_of(i, c, pos):
    s = mp.mpf(0)
    for j in range(3):
        if j == i:
            continue
        r = [pos[j][d] - pos[i][d] for d in range(3)]
        s2 = r[0] ** 2 + r[1] ** 2 + r[2] ** 2 + EPS2
        s += M[j] * r[c] / s2 ** mp.mpf("1.5")
    return s


def pot_of(i, pos):
    s = mp.mpf(0)
    for j in range(3):
        if j == i:
            continue
        r = [pos[j][d] - pos[i][d] for d in range(3)]
        s -= M[j] / mp.sqrt(r[0] ** 2 + r[1] ** 2 + r[2] ** 2 + EPS2)
    return s


def main():
    lin = lambda t: [[X[k][d] + V[k][d] * t for d in range(3)] for k in range(3)]
    A = [[acc_of(i, c, X) for c in range(3)] for i in range(3)]
    J = [[mp.diff(lambda t: acc_of(i, c, lin(t)), 0, 1) for c in range(3)] for i in range(3)]
    cub = lambda t: [[X[k][d] + V[k][d] * t + A[k][d] * t**2 / 2 + J[k][d] * t**3 / 6 for d in range(3)]
                     for k in range(3)]
    S = [[mp.diff(lambda t: acc_of(i, c, cub(t)), 0, 2) for c in range(3)] for i in range(3)]
    C = [[mp.diff(lambda t: acc_of(i, c, cub(t)), 0, 3) for c in range(3)] for i in range(3)]
    P = [pot_of(i, X) for i in range(3)]
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "w3.txt")
    with open(out, "w") as f:
        f.write("# Worked example W3 (SURVEY.md 8(c) 'Pinned values'; the paper prints none, PAPER.md:15/:43 name the\n")
        f.write("# scheme only).  N=3, m=(0.5,0.3,0.2), eps2=0.01.  40-digit mpmath differentiation of the softened\n")
        f.write("# acceleration along cubic trajectories; written by tests/golden/make_w3.py (no oracle, no CUDA).\n")
        f.write("# columns: i  quantity  x  y  z   (pot: single value)\n")
        for i in range(3):
            for name, arr in (("acc", A), ("jerk", J), ("snap", S), ("crackle", C)):
                f.write("%d %s %s %s %s\n" % (i, name, *[mp.nstr(arr[i][c], 20) for c in range(3)]))
            f.write("%d pot %s\n" % (i, mp.nstr(P[i], 20)))
    print(out)


if __name__ == "__main__":
    main()

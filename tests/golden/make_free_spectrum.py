"""Writes tests/golden/free_spectrum.txt from the CLOSED FORM only (no oracle, no CUDA).

Citation: BASELINE.json:north_star — "unit-link free-field spectrum, where D_eo D_oe has
eigenvalues -sum_mu sin^2(p_mu) on the antiperiodic momentum grid"; momentum grid
p_mu = 2 pi n_mu / L_mu (mu < 3), p_3 = 2 pi (n_3 + 1/2) / L_3 (SURVEY.md §8(c) pin P1).
The even-site operator -D_eo D_oe has one eigenvalue sum_mu sin^2 p_mu per momentum class
{p, p + (pi,pi,pi,pi)} and colour: V/2 * 3 eigenvalues in all.

Each line:  L0 L1 L2 L3 | distinct eigenvalue : multiplicity ; ...
Run:  python tests/golden/make_free_spectrum.py
"""
import itertools
import math
import os
from collections import Counter

LATTICES = [(2, 2, 2, 2), (4, 4, 4, 4), (4, 4, 2, 6), (6, 4, 4, 2), (8, 4, 4, 4)]


def spectrum(L):
    vals = Counter()
    for n in itertools.product(*[range(l) for l in L]):
        p = [2 * math.pi * n[mu] / L[mu] for mu in range(3)]
        p.append(2 * math.pi * (n[3] + 0.5) / L[3])
        lam = sum(math.sin(q) ** 2 for q in p)
        vals[round(lam, 12)] += 3  # three colours
    # p and p+pi give the same even-site vector: halve the multiplicities
    out = {}
    for k, m in vals.items():
        assert m % 2 == 0
        out[k] = m // 2
    return dict(sorted(out.items()))


if __name__ == "__main__":
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "free_spectrum.txt"), "w") as f:
        f.write("# eigenvalues of -D_eo D_oe on unit links, closed form sum_mu sin^2 p_mu\n")
        f.write("# source: BASELINE.json:north_star (free-field spectrum); SURVEY.md §8(c) P1\n")
        for L in LATTICES:
            sp = spectrum(L)
            f.write("%d %d %d %d | " % L + " ; ".join("%.12f : %d" % kv for kv in sp.items()) + "\n")

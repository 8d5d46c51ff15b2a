"""The few numbers the paper prints for a worked example (tests/golden/paper_nlc_values.txt, each with its PAPER.md line)
against the oracle's NLC pressure (oracle/tfo.c pressure(), pressure_derivatives()): the zero of Pi, the upper end of the
linearly unstable range, and the signs of Pi and Pi' at the film thicknesses of Table 1 and section 4.3.3."""
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
CAP = 0.0857                                                            # (1.11)
NLC = (CAP, 1.0 / CAP, 36.0, 0.01, 1.67, 1.0, 0.05)                     # cap0, cap1, K, b, N, beta, w


def golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_nlc_values.txt")):
        if line.strip() and not line.startswith("#"):
            name, value, tol = line.split()[:3]
            out[name] = (float(value), float(tol))
    return out


@pytest.fixture(scope="module")
def film(oracle_mod):
    o = oracle_mod.ThinFilmOracle(8, 8, 0.05, 0.05)
    o.set_pressure(2, NLC)
    return o


def dPi(o, h):
    f0, f1, _, _ = o.cell_functions([h])
    return f1[0] / f0[0] * CAP * CAP                                   # f1/f0 = (cap1/cap0) Pi' = Pi'/C^2


def bisect(f, a, b):
    fa = f(a)
    assert fa * f(b) < 0
    for _ in range(200):
        m = 0.5 * (a + b)
        fm = f(m)
        a, b, fa = (m, b, fm) if fa * fm > 0 else (a, m, fa)
    return 0.5 * (a + b)


def test_values_the_paper_prints(film):
    g = golden()
    v, tol = g["pressure_zero_H0"]
    assert abs(bisect(lambda x: film.pressure([x])[0], 0.2, 0.3) - v) <= tol
    v, tol = g["upper_end_of_instability"]
    assert abs(bisect(lambda x: dPi(film, x), 0.6, 1.5) - v) <= tol
    for name, (v, _) in g.items():
        if name.startswith("sign_Pi_at_"):
            assert np.sign(film.pressure([float(name.split("_")[-1])])[0]) == v, name
        if name.startswith("sign_dPi_at_"):
            assert np.sign(dPi(film, float(name.split("_")[-1]))) == v, name
    assert len(g) == 11

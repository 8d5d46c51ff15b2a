"""Mutation sweep of the CPU oracle (test infrastructure; run by hand, not collected by pytest):

    python tests/mutation_sweep.py            # prints one line per mutant: KILLED by <first failing pin> | SURVIVED

Every entry is a single-token mutation of oracle/tfo.c (a sign, an index, a dropped term, a transposed operand, a
wrong spacing).  For each one the mutated source is compiled into a temporary library, the oracle binding is pointed at
it, and the `-m "not gpu"` oracle pins are run until the first failure.  A mutant that survives is a line of the oracle
that no pin fixes ("parity unpinned").  DESIGN.md section 3 quotes the result of this script.
"""
import ctypes
import os
import subprocess
import sys
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "tfo.c")
PINS = ["tests/test_oracle_pins.py", "tests/test_oracle_residual_mass.py::test_oracle", "tests/test_oracle_models.py",
        "tests/test_golden_paper_values.py"]

# (name, text in tfo.c (must be unique), replacement)
MUTANTS = [
    ("residual: post-update denominator", "fabs(c->v[p] / c->uk[p])", "fabs(c->v[p] / (c->uk[p] + c->v[p]))"),
    ("mass: dx*dx", "*mass = c->dx * c->dy *", "*mass = c->dx * c->dx *"),
    ("refl: ghost -1 -> 1", "if (k < 0) return -k - 1;", "if (k < 0) return -k;"),
    ("refl: ghost N -> N-2", "if (k >= N) return 2 * N - 1 - k;", "if (k >= N) return 2 * N - 2 - k;"),
    ("Pi': sign of the m term", "c->kappa * (c->m * hm * ipow(r, c->m + 1) - c->n", "c->kappa * (-c->m * hm * ipow(r, c->m + 1) - c->n"),
    ("Pi'': n(n+1) -> n(n-1)", "c->n * (c->n + 1) * hn", "c->n * (c->n - 1) * hn"),
    ("f1': dropped h^3 Pi'' term", "*f1 = h3 * P1; *g1 = 3.0 * h2 * P1 + h3 * P2;", "*f1 = h3 * P1; *g1 = 3.0 * h2 * P1;"),
    ("L: dy*dy -> dx*dx", "at(h, nx, ny, i, j - 1)) / (dy * dy)", "at(h, nx, ny, i, j - 1)) / (dx * dx)"),
    ("D: Fxp uses f of one cell", "Fxp = 0.5 * (c->f0[p] + c->f0[q])", "Fxp = 0.5 * (c->f0[p] + c->f0[p])"),
    ("D: Fym gradient sign", "+ 0.5 * (c->f1[q] + c->f1[p]) * (h[p] - h[q]) / dy; }", "+ 0.5 * (c->f1[q] + c->f1[p]) * (h[q] - h[p]) / dy; }"),
    ("D: y divergence by dx", "D[p] = (Fxp - Fxm) / dx + (Fyp - Fym) / dy;", "D[p] = (Fxp - Fxm) / dx + (Fyp - Fym) / dx;"),
    ("J: third difference coefficient", "double T = (h2 - 3.0 * h1 + 3.0 * h0 - hm1) / d3", "double T = (h2 - 3.0 * h1 + 2.0 * h0 - hm1) / d3"),
    ("J: g0 of the wrong cell in p[1]", "p[1] = 3.0 * fb0 / d3 - fb1 / d + 0.5 * g0[(size_t)k * stride]", "p[1] = 3.0 * fb0 / d3 - fb1 / d + 0.5 * g0[(size_t)(k + 1) * stride]"),
    ("J: missing fold at the low end", "if (k - 1 < 0) { p[1] += p[0]; p[0] = 0.0; }", "if (k - 1 < 0) { p[0] = 0.0; }"),
    ("J: band a from the wrong face", "a[i]  = (pp[2] - pm[3]) / d;", "a[i]  = (pp[2] - pp[3]) / d;"),
    ("LU: gamma uses alpha_{i-1}", "double gam = ci - al2 * ei;", "double gam = ci - al1 * ei;"),
    ("LU: z drops the e term", "z[i] = (y[i * sv] - z2 * ei - z1 * gam) / mu;", "z[i] = (y[i * sv] - z1 * gam) / mu;"),
    ("LU: back substitution swaps alpha, beta", "x[(size_t)i * sv] = z[i] - al[i] * x1 - be[i] * x2;", "x[(size_t)i * sv] = z[i] - be[i] * x1 - al[i] * x2;"),
    ("step: b^n with +s D", "c->bn[p] = c->u[p] - s * c->R[p];", "c->bn[p] = c->u[p] + s * c->R[p];"),
    ("step: both sweeps along x", "directional_solve(c, 1, s, c->uk, c->R, c->w);", "directional_solve(c, 0, s, c->uk, c->R, c->w);"),
    ("step: sweep order x then y (the true swap)",
     "directional_solve(c, 1, s, c->uk, c->R, c->w);     /* (2.19): implicit y */\n        directional_solve(c, 0, s, c->uk, c->w, c->v);",
     "directional_solve(c, 0, s, c->uk, c->R, c->w);     /* (2.19): implicit y */\n        directional_solve(c, 1, s, c->uk, c->w, c->v);"),
    ("step: positivity dropped from the bad-iterate test (R18)",
     "if (!isfinite(c->uk[p]) || (c->model != 1 && !(c->uk[p] > 0))) bad = 1;", "if (!isfinite(c->uk[p])) bad = 1;"),
    ("step: NaN residual skipped by the max (R18)", "if (!(r <= res)) res = r;", "if (r > res) res = r;"),
    ("system matrix: s dropped from band a", "q[i] = 1.0 + s * q[i]; a[i] *= s;", "q[i] = 1.0 + s * q[i];"),
]

RUNNER = r"""
import ctypes, sys
sys.path.insert(0, {root!r})
from oracle import tfo
L = tfo._declare(ctypes.CDLL({so!r}))
tfo._libs[False] = L
tfo._libs[True] = L
import pytest
sys.exit(pytest.main(["-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider", "--no-header", "-rf"] + {pins!r}))
"""


def main():
    src = open(SRC).read()
    survived = []
    with tempfile.TemporaryDirectory() as tmp:
        for name, old, new in MUTANTS:
            assert src.count(old) >= 1 and src.count(old.split("\n")[0]) == 1, f"mutation target not unique in tfo.c: {old!r}"
            c, so = os.path.join(tmp, "m.c"), os.path.join(tmp, "libm.so")
            open(c, "w").write(src.replace(old, new))
            subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-std=c11", "-fPIC", "-shared", "-o", so, c, "-lm"])
            r = subprocess.run([sys.executable, "-c", RUNNER.format(root=ROOT, so=so, pins=PINS)], cwd=ROOT,
                               stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
            first = next((ln for ln in r.stdout.splitlines() if ln.startswith("FAILED")), "")
            if r.returncode == 0:
                survived.append(name)
                print(f"SURVIVED  {name}")
            else:
                print(f"KILLED    {name:45s} {first[7:100]}")
            sys.stdout.flush()
    print(f"{len(MUTANTS) - len(survived)} of {len(MUTANTS)} mutants killed")
    return 1 if survived else 0


if __name__ == "__main__":
    sys.exit(main())

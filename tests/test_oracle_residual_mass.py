"""Pins of two oracle lines that decide every Newton count and every mass check (no GPU):

  * the residual (2.22), reading R7: res = max |u_(k+1) - u_(k)| / |u_(k)| with the PRE-update
    iterate in the denominator -- pinned by forming it in numpy from the iterates of two runs with fixed counts
    K and K+1 from one state (the expected value never passes through the oracle's own residual code);
  * the mass dx*dy*sum(h), PAPER.md:352 (3.2) times the domain area, with dx != dy -- pinned by math.fsum.

Both checks are functions of an oracle *factory*, so that the same functions are also run against two mutated
builds of oracle/tfo.c (`v/(uk+v)`, `dx*dx`), which they must reject: see test_mutants_are_rejected.
"""
import ctypes
import math
import os
import subprocess

import numpy as np
import pytest

from oracle import tfo
from paper_1806_10550_b200 import inputs

DX, DY, DT = 0.41, 0.47, 1e-2


def film(nx, ny, seed):
    """A film far from flat (0.55 .. 1.6), so that v/u is ~1e-2 in the first iterations: the two readings of the
    denominator then differ by ~1e-4 relative, 10 orders above the tolerance."""
    rng = np.random.default_rng(seed)
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    h = 1.0 + 0.35 * np.cos(3 * np.pi * x)[None, :] * np.cos(2 * np.pi * y)[:, None] + 0.2 * rng.uniform(-1, 1, (ny, nx))
    return np.ascontiguousarray(h)


def make(factory, nx, ny):
    return factory(nx, ny, DX, DY, 100.0, 0.1, 3, 2)


def iterate(factory, h, k):
    """u_(k) of the step from u^n = h (k = 0: h itself) and the residual the oracle returned for iteration k."""
    if k == 0:
        return h.copy(), None
    o = make(factory, h.shape[1], h.shape[0])
    o.set_newton(1e-10, 64, k)
    o.set_state(h)
    st, it, res = o.step(DT)
    assert st == 0 and it == k
    return o.get_state(), res


def check_residual_is_max_rel_update_over_previous_iterate(factory):
    h = film(37, 29, seed=11)
    for k in (0, 1, 3):
        uk, _ = iterate(factory, h, k)
        uk1, res = iterate(factory, h, k + 1)
        expect = float(np.max(np.abs(uk1 - uk) / np.abs(uk)))            # (2.22), denominator u_(k)
        other = float(np.max(np.abs(uk1 - uk) / np.abs(uk1)))             # the reading R7 rules out
        assert abs(other - expect) > 1e-9 * expect, "film too flat to tell the two denominators apart"
        assert abs(res - expect) <= 1e-14, (k, res, expect)


def check_newton_count_is_first_iteration_below_tol(factory):
    h = film(33, 35, seed=12)
    tol = 1e-8
    o = make(factory, 33, 35)
    o.set_newton(tol, 64, 0)
    o.set_state(h)
    st, iters, res = o.step(DT)
    assert st == 0 and 3 <= iters < 64
    prev, first = h, None
    for k in range(1, iters + 2):
        uk, _ = iterate(factory, h, k)
        r = float(np.max(np.abs(uk - prev) / np.abs(prev)))
        if first is None and r < tol * (1 - 1e-6):
            first = k
        assert not (first is None and r < tol * (1 + 1e-6)), "residual too close to tol for a robust count"
        prev = uk
    assert first == iters
    assert np.array_equal(o.get_state(), iterate(factory, h, iters)[0])


def check_mass_uses_dx_times_dy(factory):
    for nx, ny, dx, dy in ((17, 23, 0.3, 0.7), (64, 9, 2.0, 0.125)):
        h = film(nx, ny, seed=nx)
        o = factory(nx, ny, dx, dy, 100.0, 0.1, 3, 2)
        o.set_state(h)
        expect = dx * dy * math.fsum(h.ravel().tolist())
        assert abs(o.mass() - expect) <= 1e-14 * abs(expect)
        assert abs(o.mass() - dx * dx * math.fsum(h.ravel().tolist())) > 0.1 * abs(expect)


CHECKS = [check_residual_is_max_rel_update_over_previous_iterate, check_newton_count_is_first_iteration_below_tol,
          check_mass_uses_dx_times_dy]


@pytest.mark.parametrize("check", CHECKS, ids=lambda f: f.__name__)
def test_oracle(check):
    check(tfo.ThinFilmOracle)


# ---------------------------------------------------------------- the two mutants the round-1 pins let through
MUTANTS = {
    "residual_denominator_post_update": ("fabs(c->v[p] / c->uk[p])", "fabs(c->v[p] / (c->uk[p] + c->v[p]))",
                                         check_residual_is_max_rel_update_over_previous_iterate),
    "mass_dx_squared": ("*mass = c->dx * c->dy *", "*mass = c->dx * c->dx *", check_mass_uses_dx_times_dy),
}


def build_mutant(tmp_path, old, new):
    src = open(os.path.join(os.path.dirname(tfo.__file__), "tfo.c")).read()
    assert src.count(old) == 1, f"mutation target not unique in tfo.c: {old!r}"
    c = tmp_path / "tfo_mutant.c"
    c.write_text(src.replace(old, new))
    so = tmp_path / "libtfo_mutant.so"
    subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-std=c11", "-fPIC", "-shared", "-o", str(so), str(c), "-lm"])
    return tfo._declare(ctypes.CDLL(str(so)))


@pytest.mark.parametrize("name", sorted(MUTANTS))
def test_mutants_are_rejected(name, tmp_path):
    old, new, check = MUTANTS[name]
    L = build_mutant(tmp_path, old, new)

    def factory(*a, **k):
        return tfo.ThinFilmOracle(*a, library=L, **k)

    with pytest.raises(AssertionError):
        check(factory)


def test_fixed_count_step_with_a_bad_iterate_is_not_accepted():
    """Reading R18 in parity mode: with fixed_iters = K the step is accepted unless one of the K iterates
    was non-finite or non-positive; then the state stays u^n (a non-positive film is not a state: Pi is singular)."""
    nx, ny = 24, 20
    rng = np.random.default_rng(5)
    h = np.ascontiguousarray(0.12 + 0.1 * rng.uniform(0, 1, (ny, nx)))       # thin, rough film; dt far too large
    o = tfo.ThinFilmOracle(nx, ny, 0.05, 0.05, 100.0, 0.1, 3, 2)
    o.set_newton(1e-10, 64, 2)
    o.set_state(h)
    st, it, res = o.step(10.0)
    assert st == tfo.NOT_CONVERGED and it == 2
    assert np.array_equal(o.get_state(), h)
    st, it, res = o.step(1e-9)                                                # a sane step is still accepted afterwards
    assert st == tfo.OK and it == 2 and np.all(o.get_state() > 0)

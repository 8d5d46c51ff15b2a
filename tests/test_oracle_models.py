"""Pins of the oracle's NLC (1.8)-(1.9) and polymer (1.12) disjoining pressures.
Nothing here calls the CUDA path.  What each pin is checked against:
  M1  Pi'(h), Pi''(h) (inside f1, f1')   <- finite differences of Pi(h) typed from the paper's definition
  M2  NLC with N = 0, cap0 = cap1 = 1     <- the already pinned power-law model (n, m) = (3, 2), kappa = K, h* = b
  M3  polymer Pi                          <- -d psi/dh by finite differences of psi typed in this file from (1.12)
  M4  Jacobian bands with the new f's     <- central differences of operator_D (as O3)
  M5  converged step                      <- G(u) = 0 with the full operator only (as O6)
  M6  growth rate of a flat NLC film      <- dispersion relation (1.4) with f0, f1 taken from finite differences of Pi
"""
import math

import numpy as np
import pytest

from oracle import tfo

CAP = 0.0857                                             # (1.11)
NLC = (CAP, 1.0 / CAP, 36.0, 0.01, 1.67, 1.0, 0.05)      # cap0, cap1 (printed placement of (1.7)), K, b, N, beta, w
POL = (0.00581, 1.0 / 0.00581, 1.181, 41.25, -243.75, 191.0)   # cap0, cap1, C, A_SiOx, A_Si, d  (1.13)
MODELS = {"nlc": (2, NLC), "polymer": (3, POL)}


def make(kind, params, nx=8, ny=8, dx=0.05, dy=0.05):
    o = tfo.ThinFilmOracle(nx, ny, dx, dy)
    o.set_pressure(kind, params)
    return o


def hrange(name):
    # NLC: across the tanh switch at h = 2b = 0.02 and up to the paper's film thicknesses; polymer: 1 .. 8 (nm units)
    return np.geomspace(0.012, 1.5, 60) if name == "nlc" else np.geomspace(0.9, 8.0, 60)


@pytest.mark.parametrize("name", ["nlc", "polymer"])
def test_M1_pressure_derivatives_vs_finite_differences_of_Pi(name):
    kind, params = MODELS[name]
    o = make(kind, params)
    h = hrange(name)
    f0, f1, g0, g1 = o.cell_functions(h)
    cap0, cap1 = params[0], params[1]
    assert np.allclose(f0, cap0 * h**3, rtol=1e-15) and np.allclose(g0, 3 * cap0 * h**2, rtol=1e-15)
    # Pi' by a 4th-order central difference of Pi
    d = 1e-4 * h
    P = o.pressure
    dPi = (-P(h + 2 * d) + 8 * P(h + d) - 8 * P(h - d) + P(h - 2 * d)) / (12 * d)
    scale = np.abs(dPi) + np.abs(P(h)) / h
    assert np.max(np.abs(f1 / (cap1 * h**3) - dPi) / scale) <= 1e-8
    # f1' by the same difference of f1 (pins Pi'')
    F1 = lambda x: o.cell_functions(x)[1]
    dF1 = (-F1(h + 2 * d) + 8 * F1(h + d) - 8 * F1(h - d) + F1(h - 2 * d)) / (12 * d)
    assert np.max(np.abs(g1 - dF1) / (np.abs(dF1) + np.abs(f1) / h)) <= 1e-8


def test_M2_nlc_without_elastic_term_is_the_power_law_model():
    o = make(2, (1.0, 1.0, 36.0, 0.01, 0.0, 1.0, 0.05))
    ref = tfo.ThinFilmOracle(8, 8, 0.05, 0.05, kappa=36.0, hstar=0.01, n=3, m=2)
    h = hrange("nlc")
    for a, b in zip(o.cell_functions(h), ref.cell_functions(h)):
        assert np.max(np.abs(a - b) / np.abs(b)) <= 1e-12     # f1 changes sign near h = 1.5 b: cancellation
    assert np.allclose(o.pressure(h), ref.pressure(h), rtol=1e-14)


def test_M3_polymer_pressure_is_minus_dpsi_dh():
    _, _, C, A1, A2, d = POL
    psi = lambda h: C / h**8 - A1 / (12 * math.pi * h**2) + (A1 - A2) / (12 * math.pi * (h + d)**2)
    o = make(3, POL)
    h = hrange("polymer")
    e = 1e-4 * h
    dpsi = (-psi(h + 2 * e) + 8 * psi(h + e) - 8 * psi(h - e) + psi(h - 2 * e)) / (12 * e)
    Pi = o.pressure(h)
    assert np.max(np.abs(Pi + dpsi) / (np.abs(Pi) + np.abs(psi(h)) / h)) <= 1e-9


def test_M3_nlc_pressure_values_from_the_definition():
    """(1.8)-(1.9) retyped with numpy at a few thicknesses (guards a mistyped formula in pressure())."""
    _, _, K, b, N, beta, w = NLC
    h = np.array([0.015, 0.02, 0.05, 0.3, 1.0])
    g = 0.5 * (1 + np.tanh((h - 2 * b) / w))
    m = g * h**2 / (h**2 + beta**2)
    ref = K * ((b / h)**3 - (b / h)**2) + 0.5 * N * (m / h)**2
    assert np.allclose(make(2, NLC).pressure(h), ref, rtol=1e-14)
    assert ref[-1] > 0 > ref[0]                 # elastic term dominates thick films, van der Waals thin ones


@pytest.mark.parametrize("name", ["nlc", "polymer"])
def test_M4_fd_jacobian_and_column_sums(name):
    kind, params = MODELS[name]
    nx, ny = 14, 6
    dx, dy = (0.05, 0.07) if name == "nlc" else (1.0, 1.3)
    lo, amp = (0.05, 0.4) if name == "nlc" else (2.0, 3.0)
    rng = np.random.default_rng(5)
    for direction in (0, 1):
        n = nx if direction == 0 else ny
        prof = lo + amp * rng.uniform(0, 1, n)
        h = np.tile(prof[None, :], (ny, 1)) if direction == 0 else np.tile(prof[:, None], (1, nx))
        o = make(kind, params, nx, ny, dx, dy)
        bands = o.jacobian_bands(direction, h)
        J = np.zeros((n, n))
        for i in range(n):
            for off, t in zip(range(-2, 3), bands):
                v = t[0, i] if direction == 0 else t[i, 0]
                if 0 <= i + off < n:
                    J[i, i + off] = v
        assert np.max(np.abs(J.sum(axis=0))) <= 1e-11 * np.abs(J).max()
        Jfd = np.zeros((n, n))
        for col in range(n):
            step = 1e-6 * prof[col]
            hp, hm = h.copy(), h.copy()
            if direction == 0:
                hp[:, col] += step; hm[:, col] -= step
            else:
                hp[col, :] += step; hm[col, :] -= step
            dD = (o.operator_D(hp) - o.operator_D(hm)) / (2 * step)
            Jfd[:, col] = dD[0, :] if direction == 0 else dD[:, 0]
        assert np.max(np.abs(J - Jfd)) <= 1e-6 * np.abs(J).max()


@pytest.mark.parametrize("name", ["nlc", "polymer"])
def test_M5_converged_step_is_a_root_of_G(name):
    kind, params = MODELS[name]
    nx, ny = 40, 36
    if name == "nlc":
        dx = dy = 0.05
        h0, eps, dt = 0.3, 0.1, 1e-3
    else:
        dx = dy = 2.0
        h0, eps, dt = 4.0, 0.1, 1e-4          # (1.13) makes f1/f0 ~ 750: every grid mode is unstable, keep dt small
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    h = h0 * (1 + eps * np.cos(3 * math.pi * x)[None, :] + eps * np.cos(2 * math.pi * y)[:, None])
    o = make(kind, params, nx, ny, dx, dy)
    o.set_newton(1e-14, 500, 0)
    o.set_state(h)
    rc, its, res = o.step(dt)
    assert rc == 0 and its >= 2
    u1 = o.get_state()
    G = u1 + 0.5 * dt * o.operator_D(u1) - (h - 0.5 * dt * o.operator_D(h))
    assert np.max(np.abs(G)) <= 1e-12 * np.max(np.abs(u1))
    assert np.max(np.abs(u1 - h)) > 1e-8 * h0
    assert abs(o.mass() - h.sum() * dx * dy) <= 1e-13 * h.sum() * dx * dy


def test_M6_nlc_flat_film_growth_rate_matches_dispersion_relation():
    """A flat NLC film of thickness h0 in the linearly unstable range (Pi'(h0) > 0): growth rate of one cosine mode
    against sigma = -(f0 q^4 - f1 q^2), (1.4) reading R8, with f1 = cap1 h0^3 Pi'(h0) from finite differences of Pi."""
    kind, params = MODELS["nlc"]
    cap0, cap1 = params[0], params[1]
    h0, eps = 0.2, 1e-4
    o0 = make(kind, params)
    d = 1e-5
    P1 = float((o0.pressure([h0 + d]) - o0.pressure([h0 - d]))[0] / (2 * d))
    assert P1 > 0
    f0, f1 = cap0 * h0**3, cap1 * h0**3 * P1
    qm = math.sqrt(f1 / (2 * f0))
    lam = 2 * math.pi / qm
    npts, nsteps = 32, 300
    L = lam                                             # mode k = 2 on [0, L] has q = q_m
    dx = L / npts
    q = 2 * math.pi / L
    sigma = -(f0 * q**4 - f1 * q**2)
    assert sigma > 0
    T = math.log(1.3) / sigma
    dt = T / nsteps
    o = make(kind, params, npts, 6, dx, dx)
    o.set_newton(1e-14, 300, 0)
    mode = np.cos(2 * math.pi * (np.arange(npts) + 0.5) * dx / L)
    o.set_state(h0 * (1 + eps * mode[None, :]) * np.ones((6, npts)))
    for _ in range(nsteps):
        assert o.step(dt)[0] == 0
    dev = o.get_state() / h0 - 1.0
    amp = (dev * mode[None, :]).sum() / (6 * (mode**2).sum())
    sigma_num = math.log(amp / eps) / T
    assert abs(sigma_num - sigma) / sigma <= 1e-2

"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the oracle function it pins and the source of the expected value.  None of the
expected values is produced by the oracle's own arithmetic re-typed: they are library routines
(LAPACK dense solve), closed forms (dispersion relation (1.4)), invariants (mass, column sums,
symmetry), or finite differences of a *different*, separately pinned oracle function.
"""
import math

import numpy as np
import pytest

from oracle import tfo
from paper_1806_10550_b200 import inputs

K, HS, N_, M_ = 100.0, 0.1, 3, 2


def rel_inf(a, b):
    return np.max(np.abs(a - b)) / np.max(np.abs(b))


# ---------------------------------------------------------------- O1: pentadiagonal LU vs dense LU
def dense_from_bands(e, c, d, a, b):
    n = len(d)
    A = np.zeros((n, n))
    for i in range(n):
        if i >= 2: A[i, i - 2] = e[i]
        if i >= 1: A[i, i - 1] = c[i]
        A[i, i] = d[i]
        if i + 1 < n: A[i, i + 1] = a[i]
        if i + 2 < n: A[i, i + 2] = b[i]
    return A


@pytest.mark.parametrize("n", list(range(5, 17)))
def test_O1_penta_solver_vs_dense_lu(n):
    """penta_solve_line vs numpy.linalg.solve (LAPACK, partial pivoting)."""
    nsys = 7
    e, c, d, a, b, rhs = inputs.penta_system(nsys, n, seed=100 + n)
    x_rows = tfo.penta_solve(0, e, c, d, a, b, rhs)
    for s in range(nsys):
        ref = np.linalg.solve(dense_from_bands(e[s], c[s], d[s], a[s], b[s]), rhs[s])
        assert rel_inf(x_rows[s], ref) <= 1e-14
    # the same systems stored as columns (strided direction)
    T = [np.ascontiguousarray(t.T) for t in (e, c, d, a, b, rhs)]
    x_cols = tfo.penta_solve(1, *T)
    assert np.array_equal(x_cols.T, x_rows)


def test_O1_penta_solver_nonsymmetric_bands_not_transposed():
    """A transposed-operand mistake (a<->c or b<->e) must fail: use strongly asymmetric bands."""
    n = 9
    rng = np.random.default_rng(7)
    e, c, a, b = 0.1 * rng.uniform(0.5, 1, n), 0.9 * rng.uniform(0.5, 1, n), -0.3 * rng.uniform(0.5, 1, n), 0.05 * rng.uniform(0.5, 1, n)
    d = 3.0 + rng.uniform(0, 1, n)
    y = rng.uniform(-1, 1, n)
    x = tfo.penta_solve(0, *[t[None, :] for t in (e, c, d, a, b, y)])[0]
    assert rel_inf(x, np.linalg.solve(dense_from_bands(e, c, d, a, b), y)) <= 1e-14


# ---------------------------------------------------------------- linear model: D and the converged CN step
def neumann_ops(n, d):
    """Forward difference on interior faces G ((n-1) x n); Neumann Laplacian = -G^T G (textbook)."""
    G = np.zeros((n - 1, n))
    for k in range(n - 1):
        G[k, k], G[k, k + 1] = -1.0 / d, 1.0 / d
    return G, -G.T @ G


def dense_linear_D(nx, ny, dx, dy, c0, c1):
    """D = c0 Lap^2 + c1 Lap for u_t + div(c0 grad lap u + c1 grad u) = 0 with zero boundary flux."""
    _, Lx = neumann_ops(nx, dx)
    _, Ly = neumann_ops(ny, dy)
    Lap = np.kron(np.eye(ny), Lx) + np.kron(Ly, np.eye(nx))   # row-major [j][i]
    return c0 * Lap @ Lap + c1 * Lap


def test_O4_linear_operator_D_vs_dense_matrix():
    """operator_D (2.11)/(2.25) with model (1.6) vs the dense 13-point matrix; dx != dy."""
    nx, ny, dx, dy, c0, c1 = 12, 10, 0.37, 0.52, 0.8, 1.3
    o = tfo.ThinFilmOracle(nx, ny, dx, dy)
    o.set_model_linear(c0, c1)
    h = np.random.default_rng(1).uniform(0.5, 1.5, (ny, nx))
    ref = (dense_linear_D(nx, ny, dx, dy, c0, c1) @ h.ravel()).reshape(ny, nx)
    assert rel_inf(o.operator_D(h), ref) <= 1e-12


def test_O4_linear_converged_step_vs_direct_crank_nicolson():
    """tfo_step (ADI pseudo-Newton, (2.19)-(2.21)) converged == direct solve of (2.14)."""
    nx, ny, dx, dy, c0, c1, dt = 12, 10, 0.37, 0.52, 0.8, 1.3, 2e-3
    o = tfo.ThinFilmOracle(nx, ny, dx, dy)
    o.set_model_linear(c0, c1)
    o.set_newton(1e-14, 5000, 0)
    h = np.random.default_rng(2).uniform(0.5, 1.5, (ny, nx))
    o.set_state(h)
    rc, its, res = o.step(dt)
    assert rc == 0 and its > 1
    D = dense_linear_D(nx, ny, dx, dy, c0, c1)
    I = np.eye(nx * ny)
    ref = np.linalg.solve(I + 0.5 * dt * D, (I - 0.5 * dt * D) @ h.ravel()).reshape(ny, nx)
    assert rel_inf(o.get_state(), ref) <= 1e-12


def test_O4_linear_bands_are_the_biharmonic_stencil():
    """f0 = 1, f1 = 0 gives interior rows (1,-4,6,-4,1)/d^4 and the dense -G^T G squared rows
    at the folded boundaries."""
    nx, ny, dx, dy = 9, 7, 0.5, 0.25
    o = tfo.ThinFilmOracle(nx, ny, dx, dy)
    o.set_model_linear(1.0, 0.0)
    h = np.ones((ny, nx))
    for direction, n, d in ((0, nx, dx), (1, ny, dy)):
        e, c, q, a, b = o.jacobian_bands(direction, h)
        _, L1 = neumann_ops(n, d)
        B = L1 @ L1
        for i in range(n):
            line = [t[0, i] if direction == 0 else t[i, 0] for t in (e, c, q, a, b)]
            for off, val in zip(range(-2, 3), line):
                ref = B[i, i + off] if 0 <= i + off < n else 0.0
                assert abs(val - ref) <= 1e-12 * abs(B).max()


# ---------------------------------------------------------------- O3: nonlinear Jacobian bands
def test_O3_column_sums_zero_and_fd_jacobian():
    """jacobian_bands_line (2.26) vs central differences of operator_D on a field that varies along one
    direction only (then D reduces to the pure-direction flux difference, and perturbing a whole
    line of cells perpendicular to it keeps that property)."""
    nx, ny, dx, dy = 14, 6, 0.4, 0.55
    rng = np.random.default_rng(3)
    for direction in (0, 1):
        n = nx if direction == 0 else ny
        prof = 0.6 + 0.5 * rng.uniform(0, 1, n)
        h = np.tile(prof[None, :], (ny, 1)) if direction == 0 else np.tile(prof[:, None], (1, nx))
        o = tfo.ThinFilmOracle(nx, ny, dx, dy, K, HS, N_, M_)
        bands = o.jacobian_bands(direction, h)
        J = np.zeros((n, n))
        for i in range(n):
            for off, t in zip(range(-2, 3), bands):
                v = t[0, i] if direction == 0 else t[i, 0]
                if 0 <= i + off < n:
                    J[i, i + off] = v
                else:
                    assert v == 0.0
        assert np.max(np.abs(J.sum(axis=0))) <= 1e-12 * np.abs(J).max()   # mass-conserving iterates
        Jfd = np.zeros((n, n))
        for col in range(n):
            step = 1e-6
            hp, hm = h.copy(), h.copy()
            if direction == 0:
                hp[:, col] += step; hm[:, col] -= step
            else:
                hp[col, :] += step; hm[col, :] -= step
            dD = (o.operator_D(hp) - o.operator_D(hm)) / (2 * step)
            Jfd[:, col] = dD[0, :] if direction == 0 else dD[:, 0]
        assert np.max(np.abs(J - Jfd)) <= 1e-7 * np.abs(J).max()


# ---------------------------------------------------------------- O2: mass conservation, sum D = 0
def test_O2_sum_of_D_vanishes():
    cfg = inputs.config(0)
    h = inputs.noise_ic(64, 48, seed=5, amp=0.2)
    o = tfo.ThinFilmOracle(64, 48, cfg["dx"], 1.3 * cfg["dy"], K, HS, N_, M_)
    D = o.operator_D(h)
    assert abs(D.sum()) <= 1e-13 * np.abs(D).sum()


def test_O2_mass_conserved_100_steps_config0():
    """PAPER.md:348-360; BASELINE.json: 1e-13 relative under no-flux boundaries."""
    cfg = inputs.config(0)
    o = tfo.ThinFilmOracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], K, HS, N_, M_)
    o.set_newton(cfg["tol"], cfg["max_iter"], 0)
    o.set_state(inputs.initial_condition(cfg))
    m0 = o.mass()
    assert abs(m0 - cfg["nx"] * cfg["ny"] * cfg["dx"] * cfg["dy"]) / m0 < 1e-3   # mean h ~ 1
    iters = []
    for _ in range(100):
        rc, it, res = o.step(cfg["dt"])
        assert rc == 0 and res < cfg["tol"]
        iters.append(it)
    assert abs(o.mass() - m0) / m0 <= 1e-13
    assert max(iters) <= 40 and min(iters) >= 2


# ---------------------------------------------------------------- O5: linear stability (1.4)
def growth_rate(direction, k, npts=32, nsteps=400):
    h0, eps = 1.0, 1e-4
    P1 = K * (M_ * HS**M_ / h0**(M_ + 1) - N_ * HS**N_ / h0**(N_ + 1))   # Pi'(h0) = 1.7
    assert abs(P1 - 1.7) < 1e-12
    L = inputs.LAMBDA_M
    d = L / npts
    q = k * math.pi / L
    sigma = -h0**3 * (q**4 - P1 * q**2)                                   # (1.4), reading R8
    T = math.log(1.3) / abs(sigma)
    dt = T / nsteps
    nx, ny = (npts, 6) if direction == 0 else (6, npts)
    o = tfo.ThinFilmOracle(nx, ny, d, d, K, HS, N_, M_)
    o.set_newton(1e-14, 200, 0)
    mode = np.cos(k * math.pi * (np.arange(npts) + 0.5) * d / L)
    shape = mode[None, :] if direction == 0 else mode[:, None]
    o.set_state(h0 * (1 + eps * shape) * np.ones((ny, nx)))
    for _ in range(nsteps):
        rc, _, _ = o.step(dt)
        assert rc == 0
    dev = o.get_state() / h0 - 1.0
    amp = (dev * shape).sum() / ((shape * np.ones((ny, nx))) ** 2).sum()
    sigma_num = math.log(amp / eps) / T
    q2t = (4.0 / d**2) * math.sin(q * d / 2) ** 2                         # discrete symbol of -d2/dx2
    sig_d = -h0**3 * (q2t**2 - P1 * q2t)
    sigma_cn = math.log((1 + sig_d * dt / 2) / (1 - sig_d * dt / 2)) / dt  # exact CN amplification
    return sigma, sigma_num, sigma_cn


@pytest.mark.parametrize("direction", [0, 1])
@pytest.mark.parametrize("k", [1, 2])
def test_O5_growth_rate_matches_dispersion_relation(direction, k):
    sigma, sigma_num, sigma_cn = growth_rate(direction, k)
    assert sigma > 0
    assert abs(sigma_num - sigma) / abs(sigma) <= 1e-2       # BASELINE.json: within 1%
    assert abs(sigma_num - sigma_cn) / abs(sigma_cn) <= 2e-4  # nonlinear O(eps) corrections remain


def test_O5_stable_mode_decays():
    sigma, sigma_num, sigma_cn = growth_rate(0, 3, nsteps=400)   # q = 1.5 q_m > q_c = sqrt(2) q_m: stable
    assert sigma < 0 and sigma_num < 0
    assert abs(sigma_num - sigma_cn) / abs(sigma_cn) <= 2e-4


# ---------------------------------------------------------------- O6-O9
def cos_state(nx=48, ny=40):
    cfg = inputs.config(0)
    dx = 2 * inputs.LAMBDA_M / nx
    dy = 2 * inputs.LAMBDA_M / ny
    return dx, dy, inputs.cosine_ic(nx, ny, dx, dy, kx=4, ky=2, h0=1.0, eps=0.1)


def test_O6_converged_step_is_a_root_of_G():
    """(2.15): G(u^{n+1}) = (I + sD)u^{n+1} - (I - sD)u^n = 0, evaluated with the full operator only."""
    dx, dy, h = cos_state()
    ny, nx = h.shape
    o = tfo.ThinFilmOracle(nx, ny, dx, dy, K, HS, N_, M_)
    o.set_newton(1e-14, 500, 0)
    o.set_state(h)
    dt = 5e-3
    rc, its, res = o.step(dt)
    assert rc == 0 and its >= 3
    u1 = o.get_state()
    G = u1 + 0.5 * dt * o.operator_D(u1) - (h - 0.5 * dt * o.operator_D(h))
    assert np.max(np.abs(G)) <= 1e-13 * np.max(np.abs(u1))
    assert np.max(np.abs(u1 - h)) > 1e-6          # the step did something


def test_O7_second_order_in_time():
    """error vs the finest level falls 4x per dt halving."""
    dx, dy, h = cos_state(32, 32)
    ny, nx = h.shape
    T = 0.04
    sols = []
    for lev in range(5):
        o = tfo.ThinFilmOracle(nx, ny, dx, dy, K, HS, N_, M_)
        o.set_newton(1e-14, 2000, 0)
        o.set_state(h)
        nst = 2 ** lev
        for _ in range(nst):
            assert o.step(T / nst)[0] == 0
        sols.append(o.get_state())
    err = [np.sqrt(np.mean((s - sols[-1]) ** 2)) for s in sols[:-1]]
    orders = [math.log2(err[i] / err[i + 1]) for i in range(len(err) - 1)]
    # vs-finest errors: ratio (4^k - 1)/(4^(k-1) - 1) -> order slightly above 2
    assert all(1.9 <= p <= 2.6 for p in orders), orders


def test_O8_uniform_film_is_a_fixed_point():
    o = tfo.ThinFilmOracle(16, 12, 0.4, 0.4, K, HS, N_, M_)
    h = np.full((12, 16), 0.7)
    o.set_state(h)
    rc, its, res = o.step(1e-2)
    assert (rc, its, res) == (0, 1, 0.0)
    assert np.array_equal(o.get_state(), h)


def test_O9_transpose_symmetry():
    dx, dy, h = cos_state(20, 28)
    ny, nx = h.shape
    a = tfo.ThinFilmOracle(nx, ny, dx, dy, K, HS, N_, M_)
    b = tfo.ThinFilmOracle(ny, nx, dy, dx, K, HS, N_, M_)
    for o, f in ((a, h), (b, h.T)):
        o.set_newton(1e-14, 500, 0)
        o.set_state(f)
        assert o.step(5e-3)[0] == 0
    assert rel_inf(b.get_state().T, a.get_state()) <= 1e-12


def test_corner_ghosts_order_independent():
    """y-then-x reflection == x-then-y reflection (checked through D of a transposed field)."""
    nx = ny = 10
    h = np.random.default_rng(9).uniform(0.5, 1.5, (ny, nx))
    a = tfo.ThinFilmOracle(nx, ny, 0.3, 0.3, K, HS, N_, M_)
    assert rel_inf(a.operator_D(h.T.copy()).T, a.operator_D(h)) <= 1e-13


def test_step_rejection_leaves_state_unchanged_and_validation():
    dx, dy, h = cos_state(16, 16)
    o = tfo.ThinFilmOracle(16, 16, dx, dy, K, HS, N_, M_)
    o.set_newton(1e-14, 2, 0)
    o.set_state(h)
    rc, its, res = o.step(1e-2)
    assert rc == tfo.NOT_CONVERGED and its == 2 and res > 1e-14
    assert np.array_equal(o.get_state(), h)
    o.set_newton(1e-10, 64, 3)           # fixed_iters: always accepted after exactly 3
    rc, its, _ = o.step(1e-2)
    assert rc == 0 and its == 3
    with pytest.raises(tfo.OracleError):
        o.set_state(-h)
    with pytest.raises(tfo.OracleError):
        tfo.ThinFilmOracle(4, 16, dx, dy)
    with pytest.raises(tfo.OracleError):
        tfo.ThinFilmOracle(16, 16, dx, dy, K, HS, 2, 3)


# ---------------------------------------------------------------- O12: order of the two sweeps inside tfo_step
def _nonsymmetric_film(nx, ny, dx, dy, seed):
    x = (np.arange(nx) + 0.5) * dx
    y = (np.arange(ny) + 0.5) * dy
    rng = np.random.default_rng(seed)
    u = 1.0 + 0.2 * np.cos(2 * math.pi * x / (nx * dx))[None, :] * np.sin(1.3 * y)[:, None] + 0.15 * rng.uniform(-1, 1, (ny, nx))
    return np.ascontiguousarray(u), x, y


def test_O12_direction_labels_of_directional_solve():
    """directional_solve(0, ...) is the solve along x and (1, ...) the one along y, fixed by a structural fact rather than
    by the label: for a film and a right-hand side that do not vary along x, J_x annihilates the right-hand side (every
    term of the x-part of (2.26) is an x-difference of one of them), so the x-solve must return it unchanged, and the
    y-solve must not."""
    nx, ny, dx, dy = 23, 17, 0.31, 0.47
    _, _, y = _nonsymmetric_film(nx, ny, dx, dy, 3)
    o = tfo.ThinFilmOracle(nx, ny, dx, dy, K, HS, N_, M_)
    uy = np.ascontiguousarray(np.repeat((1.0 + 0.2 * np.sin(1.3 * y))[:, None], nx, axis=1))
    rhs = np.ascontiguousarray(np.repeat(np.cos(0.7 * y)[:, None], nx, axis=1))
    assert np.max(np.abs(o.directional_solve(0, 0.01, uy, rhs) - rhs)) <= 1e-14
    assert np.max(np.abs(o.directional_solve(1, 0.01, uy, rhs) - rhs)) >= 1e-2

@pytest.mark.parametrize("dt", [1e-3, 1e-2])
def test_O12_one_iteration_is_the_y_sweep_followed_by_the_x_sweep(dt):
    """(2.19) before (2.20), and the kernel order 1)-4) of App. A.2: the first iterate of
    tfo_step must equal u + S_x(S_y(R)), R = b^n - u - s D(u), composed here from operator_D and directional_solve
    (each pinned on its own: O4, O3, O12 above) -- and on this film (no symmetry, dx != dy) the other order gives a
    different field, so the comparison can tell the two apart."""
    nx, ny, dx, dy = 23, 17, 0.31, 0.47
    u, _, _ = _nonsymmetric_film(nx, ny, dx, dy, 3)
    s = 0.5 * dt
    o = tfo.ThinFilmOracle(nx, ny, dx, dy, K, HS, N_, M_)
    o.set_newton(1e-10, 10, 1)                            # exactly one iteration, accepted
    o.set_state(u)
    st, it, _ = o.step(dt)
    assert st == tfo.OK and it == 1
    v = o.get_state() - u
    D = o.operator_D(u)
    R = (u - s * D) - u - s * D                           # b^n - u_(0) - s D(u_(0))
    v_yx = o.directional_solve(0, s, u, o.directional_solve(1, s, u, R))
    v_xy = o.directional_solve(1, s, u, o.directional_solve(0, s, u, R))
    scale = np.max(np.abs(v_yx))
    assert np.max(np.abs(v - v_yx)) <= 1e-14 * scale
    assert np.max(np.abs(v_xy - v_yx)) >= 1e-7 * scale    # measured: 2e-2 (dt = 1e-3), 0.6 (dt = 1e-2)
    assert np.max(np.abs(v - v_xy)) >= 1e-7 * scale


# ---------------------------------------------------------------- O13: reading R18, the two lines the GPU is compared against
def test_O13_a_finite_but_non_positive_iterate_rejects_the_step():
    """Reading R18: an iterate that is finite but not positive ends the step (Pi is singular at h = 0, such
    a field is not a film).  The case is built so that ONLY positivity can trip: the first iterate, composed from the
    separately pinned pieces, is finite everywhere and negative somewhere."""
    nx, ny, d, dt = 24, 20, 0.05, 1e-2
    h = np.ascontiguousarray(0.12 + 0.1 * np.random.default_rng(5).uniform(0, 1, (ny, nx)))
    o = tfo.ThinFilmOracle(nx, ny, d, d, K, HS, N_, M_)
    s = 0.5 * dt
    u1 = h + o.directional_solve(0, s, h, o.directional_solve(1, s, h, -2.0 * s * o.operator_D(h)))
    assert np.isfinite(u1).all() and u1.min() < 0.0
    o.set_newton(1e-10, 64, 1)                            # parity mode, one iteration: accepted unless the iterate is bad
    o.set_state(h)
    st, it, res = o.step(dt)
    assert st == tfo.NOT_CONVERGED and it == 1 and math.isfinite(res)
    assert np.array_equal(o.get_state(), h)
    o.set_newton(1e-10, 64, 0)                            # normal mode: the iteration stops at the bad iterate
    st, it, res = o.step(dt)
    assert st == tfo.NOT_CONVERGED and it == 1 and math.isfinite(res)
    assert np.array_equal(o.get_state(), h)


@pytest.mark.parametrize("fixed", [0, 1, 3])
def test_O13_a_nan_residual_is_reported_as_nan(fixed):
    """A NaN in v / u_k must surface in the reported residual (max over the grid with NaN winning), not be skipped by the
    comparison.  h = 1e120 in one cell is a valid state (finite, positive) whose h^3 overflows: D(u) is inf - inf there."""
    nx, ny = 16, 12
    h = np.ones((ny, nx))
    h[5, 7] = 1e120
    o = tfo.ThinFilmOracle(nx, ny, 0.3, 0.3, K, HS, N_, M_)
    o.set_newton(1e-10, 10, fixed)
    o.set_state(h)
    st, it, res = o.step(1e-3)
    assert st == tfo.NOT_CONVERGED and it == max(fixed, 1) and math.isnan(res)
    assert np.array_equal(o.get_state(), h)

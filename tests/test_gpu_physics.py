"""The CUDA path against what the paper and the mathematics fix, WITHOUT the oracle in between (the same checks that
pin the oracle, tests/test_oracle_pins.py, here applied to the product): the growth rate of a single Fourier mode against
the dispersion relation (1.4), second order in time, conservation of mass
(PAPER.md:348-360), the fixed point and the transpose symmetry of the scheme."""
import math

import numpy as np
import pytest

from paper_1806_10550_b200 import inputs

pytestmark = pytest.mark.gpu
K, HS, N_, M_ = 100.0, 0.1, 3, 2


@pytest.fixture(scope="module")
def tf():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1806_10550_b200 import tf as tfmod
    tfmod.lib()
    return tfmod


@pytest.mark.parametrize("direction", [0, 1])
@pytest.mark.parametrize("k", [1, 2, 3])
def test_growth_rate_of_a_single_mode(tf, direction, k):
    """k = 1, 2: unstable modes (q = q_m/2 and q_m): within 1 % of sigma(q) = -h0^3 (q^4 - Pi'(h0) q^2) and within 2e-4 of
    the exact Crank-Nicolson amplification of the discrete symbol; k = 3: q = 1.5 q_m > q_c, the mode decays."""
    h0, eps, npts, nsteps = 1.0, 1e-4, 32, 400
    P1 = K * (M_ * HS**M_ / h0**(M_ + 1) - N_ * HS**N_ / h0**(N_ + 1))
    L = inputs.LAMBDA_M
    d = L / npts
    q = k * math.pi / L
    sigma = -h0**3 * (q**4 - P1 * q**2)
    T = math.log(1.3) / abs(sigma)
    dt = T / nsteps
    nx, ny = (npts, 6) if direction == 0 else (6, npts)
    g = tf.ThinFilm(nx, ny, d, d, K, HS, N_, M_)
    g.set_newton(1e-14, 200, 0)
    mode = np.cos(k * math.pi * (np.arange(npts) + 0.5) * d / L)
    shape = mode[None, :] if direction == 0 else mode[:, None]
    g.set_state(h0 * (1 + eps * shape) * np.ones((ny, nx)))
    for _ in range(nsteps):
        assert g.step(dt)[0] == 0
    dev = g.get_state() / h0 - 1.0
    amp = (dev * shape).sum() / ((shape * np.ones((ny, nx))) ** 2).sum()
    sigma_num = math.log(amp / eps) / T
    q2t = (4.0 / d**2) * math.sin(q * d / 2) ** 2
    sig_d = -h0**3 * (q2t**2 - P1 * q2t)
    sigma_cn = math.log((1 + sig_d * dt / 2) / (1 - sig_d * dt / 2)) / dt
    assert (sigma > 0) == (k < 3) and (sigma_num > 0) == (k < 3)
    if k < 3:
        assert abs(sigma_num - sigma) / abs(sigma) <= 1e-2
    assert abs(sigma_num - sigma_cn) / abs(sigma_cn) <= 2e-4


def test_second_order_in_time_mass_fixed_point_symmetry(tf):
    nx = ny = 32
    dx = dy = 2 * inputs.LAMBDA_M / nx
    h = inputs.cosine_ic(nx, ny, dx, dy, kx=4, ky=2, h0=1.0, eps=0.1)
    T, sols, m0 = 0.04, [], None
    for lev in range(5):
        g = tf.ThinFilm(nx, ny, dx, dy, K, HS, N_, M_)
        g.set_newton(1e-14, 2000, 0)
        g.set_state(h)
        m0 = g.mass()
        for _ in range(2 ** lev):
            assert g.step(T / 2 ** lev)[0] == 0
        assert abs(g.mass() - m0) <= 1e-13 * m0                          # (3.2): mass is conserved
        sols.append(g.get_state())
    err = [np.sqrt(np.mean((s - sols[-1]) ** 2)) for s in sols[:-1]]
    orders = [math.log2(err[i] / err[i + 1]) for i in range(len(err) - 1)]
    assert all(1.9 <= p <= 2.6 for p in orders), orders
    # a flat film is a fixed point: one iteration, zero residual, unchanged bit for bit
    g = tf.ThinFilm(48, 40, 0.4, 0.4, K, HS, N_, M_)
    flat = np.full((40, 48), 0.7)
    g.set_state(flat)
    assert g.step(1e-2) == (0, 1, 0.0) and np.array_equal(g.get_state(), flat)
    # the converged step of the transposed film (dx <-> dy) is the transpose of the converged step
    ha = inputs.cosine_ic(40, 56, 0.3, 0.35, kx=3, ky=2, h0=1.0, eps=0.1)
    a = tf.ThinFilm(40, 56, 0.3, 0.35, K, HS, N_, M_)
    b = tf.ThinFilm(56, 40, 0.35, 0.3, K, HS, N_, M_)
    for g_, h_ in ((a, ha), (b, np.ascontiguousarray(ha.T))):
        g_.set_newton(1e-14, 500, 0)
        g_.set_state(h_)
        assert g_.step(5e-3)[0] == 0
    assert np.max(np.abs(a.get_state() - b.get_state().T)) <= 1e-12 * np.max(np.abs(ha))


def _iterate(tf, h, dx, dy, dt, k):
    """u_(k) of the step from u^n = h on the CUDA path (fixed count k) and the residual it returned."""
    if k == 0:
        return h.copy(), None
    g = tf.ThinFilm(h.shape[1], h.shape[0], dx, dy, K, HS, N_, M_)
    g.set_newton(1e-10, 64, k)
    g.set_state(h)
    st, it, res = g.step(dt)
    assert st == 0 and it == k
    return g.get_state(), res


@pytest.mark.parametrize("shape", [(37, 29), (96, 160)])
def test_residual_is_max_rel_update_over_previous_iterate(tf, shape):
    """(2.22), reading R7, on the CUDA path alone: the residual tf_step returns for iteration k+1
    equals max |u_(k+1) - u_(k)| / |u_(k)| formed in numpy from the iterates of two fixed-count runs (pre-update
    iterate in the denominator; the post-update reading differs by ~1e-4 relative on this film)."""
    nx, ny = shape
    dx, dy, dt = 0.41, 0.47, 1e-2
    rng = np.random.default_rng(11)
    x, y = (np.arange(nx) + 0.5) / nx, (np.arange(ny) + 0.5) / ny
    h = np.ascontiguousarray(1.0 + 0.35 * np.cos(3 * np.pi * x)[None, :] * np.cos(2 * np.pi * y)[:, None]
                             + 0.2 * rng.uniform(-1, 1, (ny, nx)))
    for k in (0, 1, 3):
        uk, _ = _iterate(tf, h, dx, dy, dt, k)
        uk1, res = _iterate(tf, h, dx, dy, dt, k + 1)
        expect = float(np.max(np.abs(uk1 - uk) / np.abs(uk)))
        other = float(np.max(np.abs(uk1 - uk) / np.abs(uk1)))
        assert abs(other - expect) > 1e-9 * expect
        assert abs(res - expect) <= 1e-14, (k, res, expect)
    # the Newton count of a tol-converged step is the first k whose numpy residual is below tol
    tol = 1e-8
    g = tf.ThinFilm(nx, ny, dx, dy, K, HS, N_, M_)
    g.set_newton(tol, 64, 0)
    g.set_state(h)
    st, iters, _ = g.step(dt)
    assert st == 0 and 3 <= iters < 64
    prev, first = h, None
    for k in range(1, iters + 2):
        uk, _ = _iterate(tf, h, dx, dy, dt, k)
        r = float(np.max(np.abs(uk - prev) / np.abs(prev)))
        if first is None and r < tol * (1 - 1e-6):
            first = k
        assert not (first is None and r < tol * (1 + 1e-6))
        prev = uk
    assert first == iters
    assert np.array_equal(g.get_state(), _iterate(tf, h, dx, dy, dt, iters)[0])


def test_mass_uses_dx_times_dy(tf):
    """(3.2), times the domain area, dx != dy, against math.fsum (no oracle)."""
    for nx, ny, dx, dy in ((17, 23, 0.3, 0.7), (64, 9, 2.0, 0.125), (300, 167, 0.11, 0.9)):
        rng = np.random.default_rng(nx)
        h = np.ascontiguousarray(1.0 + 0.5 * rng.uniform(-1, 1, (ny, nx)))
        g = tf.ThinFilm(nx, ny, dx, dy, K, HS, N_, M_)
        g.set_state(h)
        expect = dx * dy * math.fsum(h.ravel().tolist())
        assert abs(g.mass() - expect) <= 1e-13 * abs(expect)
        assert abs(g.mass() - dx * dx * math.fsum(h.ravel().tolist())) > 0.1 * abs(expect)


def test_fixed_count_step_with_a_bad_iterate_is_not_accepted(tf):
    """Reading R18 in parity mode (include/tf.h, tf_set_newton): a fixed-count step whose iterates leave h > 0 is
    returned as TF_NOT_CONVERGED with the state untouched; a sane step afterwards is accepted."""
    nx, ny = 64, 48
    rng = np.random.default_rng(5)
    h = np.ascontiguousarray(0.12 + 0.1 * rng.uniform(0, 1, (ny, nx)))
    g = tf.ThinFilm(nx, ny, 0.05, 0.05, K, HS, N_, M_)
    g.set_newton(1e-10, 64, 2)
    g.set_state(h)
    st, it, res = g.step(10.0)
    assert st == tf.NOT_CONVERGED and it == 2
    assert np.array_equal(g.get_state(), h)
    st, it, res = g.step(1e-9)
    assert st == tf.OK and it == 2 and np.all(g.get_state() > 0)


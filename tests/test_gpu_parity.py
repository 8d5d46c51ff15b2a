"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's: relative L-inf <= 1e-11 after one step,
<= 1e-8 after 100 steps, Newton iteration count fixed for the comparison."""
import math

import numpy as np
import pytest

from paper_1806_10550_b200 import inputs

pytestmark = pytest.mark.gpu

K, HS = 100.0, 0.1


@pytest.fixture(scope="module")
def tf():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1806_10550_b200 import tf as tfmod
    tfmod.lib()
    return tfmod


@pytest.fixture(scope="module")
def tfo():
    from oracle import tfo as o
    o.build()
    return o


def rel_inf(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def pair(tf, tfo, nx, ny, dx, dy, n=3, m=2, omp=False):
    g = tf.ThinFilm(nx, ny, dx, dy, K, HS, n, m)
    o = tfo.ThinFilmOracle(nx, ny, dx, dy, K, HS, n, m, omp=omp)
    return g, o


def run_both(g, o, h, dt, steps, **newton):
    g.set_newton(**newton)
    o.set_newton(**newton)
    g.set_state(h)
    o.set_state(h)
    rg = [g.step(dt) for _ in range(steps)]
    ro = [o.step(dt) for _ in range(steps)]
    return rg, ro


# ------------------------------------------------------------------ one Newton iteration / one step
@pytest.mark.parametrize("nx,ny,dxf,dyf", [
    (128, 128, 1.0, 1.0),     # config 0 shape
    (61, 45, 1.0, 1.3),       # ragged in both directions, dx != dy
    (29, 33, 0.8, 1.0),       # one column past a 28-wide strip, one row past a 32-row tile
    (5, 5, 1.0, 1.0),         # minimum size
    (5, 70, 1.0, 1.0),
    (260, 7, 1.0, 1.0),
    (300, 167, 1.0, 1.0),     # several strips/tiles + ragged tails
])
@pytest.mark.parametrize("iters", [1, 8])
def test_one_step_parity(tf, tfo, nx, ny, dxf, dyf, iters):
    cfg = inputs.config(0)
    g, o = pair(tf, tfo, nx, ny, cfg["dx"] * dxf, cfg["dy"] * dyf)
    h = inputs.noise_ic(nx, ny, seed=10 + nx + ny)
    rg, ro = run_both(g, o, h, cfg["dt"], 1, tol=1e-10, max_iter=64, fixed_iters=iters)
    assert rg[0][0] == 0 and rg[0][1] == iters == ro[0][1]
    ug, uo = g.get_state(), o.get_state()
    assert rel_inf(ug, uo) <= 1e-11
    assert abs(rg[0][2] - ro[0][2]) <= 1e-9 * ro[0][2] + 1e-300      # residual (2.22)
    assert np.max(np.abs(uo - h)) > 1e-5                               # the step moved the film


def test_large_amplitude_film_parity(tf, tfo):
    """Strongly nonlinear state (h between 0.15 and 1.6): exercises f0', f1' and the Pi terms."""
    nx, ny = 96, 80
    cfg = inputs.config(0)
    h = inputs.cosine_ic(nx, ny, cfg["dx"], cfg["dy"], kx=3, ky=2, h0=0.9, eps=0.4)
    g, o = pair(tf, tfo, nx, ny, cfg["dx"], cfg["dy"])
    rg, ro = run_both(g, o, h, 2e-3, 3, tol=1e-10, max_iter=64, fixed_iters=6)
    assert rel_inf(g.get_state(), o.get_state()) <= 1e-11


@pytest.mark.parametrize("n,m", [(4, 1), (9, 3), (3, 1)])
def test_generic_exponents_parity(tf, tfo, n, m):
    nx, ny = 70, 50
    cfg = inputs.config(0)
    g, o = pair(tf, tfo, nx, ny, cfg["dx"], cfg["dy"], n, m)
    h = inputs.noise_ic(nx, ny, seed=3, amp=0.05)
    rg, ro = run_both(g, o, h, 1e-3, 2, tol=1e-10, max_iter=64, fixed_iters=4)
    assert rel_inf(g.get_state(), o.get_state()) <= 1e-11


def test_config0_100_steps_parity_fixed_iters(tf, tfo):
    cfg = inputs.config(0)
    g, o = pair(tf, tfo, cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"])
    h = inputs.initial_condition(cfg)
    rg, ro = run_both(g, o, h, cfg["dt"], 100, tol=cfg["tol"], max_iter=cfg["max_iter"], fixed_iters=8)
    assert rel_inf(g.get_state(), o.get_state()) <= 1e-8


def test_config0_converged_run_matches_oracle_iteration_counts_and_mass(tf, tfo):
    cfg = inputs.config(0)
    g, o = pair(tf, tfo, cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"])
    h = inputs.initial_condition(cfg)
    g.set_newton(cfg["tol"], cfg["max_iter"], 0)
    o.set_newton(cfg["tol"], cfg["max_iter"], 0)
    g.set_state(h)
    o.set_state(h)
    m0 = g.mass()
    assert abs(m0 - o.mass()) <= 1e-14 * abs(m0)
    for k in range(100):
        sg, ig, rg = g.step(cfg["dt"])
        so, io, ro = o.step(cfg["dt"])
        assert sg == so == 0
        assert abs(ig - io) <= 1, (k, ig, io)          # res can straddle tol by rounding
        assert rg < cfg["tol"]
    assert rel_inf(g.get_state(), o.get_state()) <= 1e-8
    assert abs(g.mass() - m0) / m0 <= 1e-13               # discrete mass conservation on the GPU path


def test_config1_one_step_parity(tf, tfo):
    cfg = inputs.config(1)
    g, o = pair(tf, tfo, cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], omp=True)
    h = inputs.initial_condition(cfg)
    rg, ro = run_both(g, o, h, cfg["dt"], 1, tol=1e-10, max_iter=64, fixed_iters=8)
    assert rel_inf(g.get_state(), o.get_state()) <= 1e-11


def test_config2_shape_gaussian_depressions(tf, tfo):
    """Config 2's recipe on a 512^2 cut (same dx, uniform 0.12 film with Gaussian depressions)."""
    cfg = inputs.config(2)
    nx = ny = 512
    h = inputs.gauss_ic(nx, ny, cfg["dx"], cfg["dy"], seed=cfg["seed"], count=8)
    assert h.min() > 0.06
    g, o = pair(tf, tfo, nx, ny, cfg["dx"], cfg["dy"], omp=True)
    g.set_newton(cfg["tol"], cfg["max_iter"], 0)
    o.set_newton(cfg["tol"], cfg["max_iter"], 0)
    g.set_state(h)
    o.set_state(h)
    dt = cfg["dt"]
    for _ in range(5):                       # adaptive controller of Fig. 1 on both, same decisions
        sg, ig, _ = g.step(dt)
        so, io, _ = o.step(dt)
        assert sg == so and abs(ig - io) <= 1
        dt = min(dt * cfg["grow"], cfg["dt_max"]) if sg == 0 else dt * cfg["shrink"]
    assert rel_inf(g.get_state(), o.get_state()) <= 1e-9


# ------------------------------------------------------------------ control flow / edge cases
def test_rejected_step_leaves_state_bitwise_unchanged(tf, tfo):
    cfg = inputs.config(0)
    nx, ny = 64, 64
    h = inputs.cosine_ic(nx, ny, cfg["dx"], cfg["dy"], kx=4, ky=2, eps=0.1)
    g, o = pair(tf, tfo, nx, ny, cfg["dx"], cfg["dy"])
    rg, ro = run_both(g, o, h, 1e-2, 1, tol=1e-14, max_iter=2, fixed_iters=0)
    assert rg[0][0] == ro[0][0] == tf.NOT_CONVERGED and rg[0][1] == ro[0][1] == 2
    assert np.array_equal(g.get_state(), h)
    # and the context still works afterwards
    g.set_newton(1e-10, 64, 0)
    assert g.step(1e-3)[0] == 0


def test_uniform_film_fixed_point_is_exact(tf):
    g = tf.ThinFilm(40, 36, 0.4, 0.4, K, HS, 3, 2)
    h = np.full((36, 40), 0.7)
    g.set_state(h)
    st, it, res = g.step(1e-2)
    assert (st, it, res) == (0, 1, 0.0)
    assert np.array_equal(g.get_state(), h)


def test_state_validation_and_errors(tf):
    g = tf.ThinFilm(16, 16, 0.4, 0.4, K, HS, 3, 2)
    with pytest.raises(tf.TfError) as ei:
        g.step(1e-2)
    assert ei.value.status == tf.ERR_STATE
    h = np.ones((16, 16))
    g.set_state(h)
    bad = h.copy(); bad[3, 5] = -1.0
    with pytest.raises(tf.TfError):
        g.set_state(bad)
    bad[3, 5] = np.nan
    with pytest.raises(tf.TfError):
        g.set_state(bad)
    assert np.array_equal(g.get_state(), h)          # previous state kept
    with pytest.raises(tf.TfError):
        g.step(-1.0)
    with pytest.raises(tf.TfError):
        g.set_newton(1e-16, 10, 0)


def test_device_pointer_state_roundtrip(tf):
    import torch
    g = tf.ThinFilm(48, 32, 0.4, 0.4, K, HS, 3, 2)
    h = torch.rand(32, 48, dtype=torch.float64, device="cuda") + 0.5
    g.set_state(h)
    out = torch.empty_like(h)
    g.get_state(out)
    assert torch.equal(out, h)
    ref = float(h.sum().item()) * 0.16
    assert abs(g.mass() - ref) <= 1e-13 * ref


def test_mass_is_bitwise_reproducible(tf):
    cfg = inputs.config(0)
    g = tf.ThinFilm(300, 200, 0.4, 0.4, K, HS, 3, 2)
    g.set_state(inputs.noise_ic(300, 200, seed=1))
    assert len({g.mass() for _ in range(5)}) == 1


# ------------------------------------------------------------------ isolated pentadiagonal solve (config 4 shape)
@pytest.mark.parametrize("nrow,ncol", [(64, 64), (33, 70), (130, 37), (3, 40), (40, 3), (257, 129),
                                       (96, 200), (130, 70), (66, 1000), (1000, 66), (250, 254)])   # even: TMA path, ragged tiles
@pytest.mark.parametrize("direction", [0, 1])
def test_penta_solve_parity(tf, tfo, nrow, ncol, direction):
    import torch
    arrs = inputs.penta_system(nrow, ncol, seed=4)
    ref = tfo.penta_solve(direction, *arrs)
    dev = [torch.from_numpy(a).cuda() for a in arrs]
    x = tf.penta_solve(direction, *dev)
    torch.cuda.synchronize()
    x = x.cpu().numpy()
    assert rel_inf(x, ref) <= 1e-12
    # backward error of the GPU solution, independent of the oracle
    e, c, d, a, b, y = arrs if direction == 0 else [t.T for t in arrs]
    xs = x if direction == 0 else x.T
    n = xs.shape[1]
    Ax = d * xs
    Ax[:, 1:] += c[:, 1:] * xs[:, :-1]
    Ax[:, 2:] += e[:, 2:] * xs[:, :-2]
    Ax[:, :-1] += a[:, :-1] * xs[:, 1:]
    Ax[:, :-2] += b[:, :-2] * xs[:, 2:]
    normA = np.max(np.abs(e) + np.abs(c) + np.abs(d) + np.abs(a) + np.abs(b))
    assert np.max(np.abs(Ax - y)) / (normA * np.max(np.abs(xs)) + np.max(np.abs(y))) <= 1e-14


# ------------------------------------------------------------------ S8: speculative launch-ahead == per-iteration decision
@pytest.mark.parametrize("nx,ny", [(128, 128), (61, 45), (300, 168)])
def test_launch_ahead_is_exactly_the_per_iteration_decision(tf, nx, ny):
    """tf_set_launch_ahead(batch > 0) enqueues iterations past the deciding one; those must be no-ops on the device:
    iteration counts, residuals and fields are bit-identical to batch = 0, for accepted and for rejected steps."""
    h0 = inputs.noise_ic(nx, ny, seed=9)
    runs = []
    for batch in (0, 1, 2, 7):
        g = tf.ThinFilm(nx, ny, 0.4259, 0.4259, K, HS, 3, 2)
        g.set_launch_ahead(batch)
        g.set_newton(tol=1e-10, max_iter=64)
        g.set_state(h0)
        log = [g.step(1e-2) for _ in range(6)]
        g.set_newton(tol=1e-10, max_iter=3)            # too few iterations: every step is rejected, state must stay
        before = g.get_state()
        log += [g.step(1e-2) for _ in range(2)]
        assert np.array_equal(before, g.get_state())
        g.set_newton(tol=1e-10, max_iter=64)
        log += [g.step(1e-2) for _ in range(2)]
        runs.append((log, g.get_state()))
    assert all(st == tf.OK for st, _, _ in runs[0][0][:6]) and all(st == tf.NOT_CONVERGED for st, _, _ in runs[0][0][6:8])
    for log, h in runs[1:]:
        assert log == runs[0][0]
        assert np.array_equal(h, runs[0][1])


# ------------------------------------------------------------------ Fig. 1 with an extra solution criterion (Note 2)
@pytest.mark.parametrize("on_device", [False, True])
def test_solution_criterion_and_native_controller_against_the_flow_chart(tf, tfo, on_device):
    """tf_set_solution_criteria + tf_advance_adaptive against the oracle's transcription of Fig. 1 with the same
    criterion (max relative change of h per step): same accept / reject sequence (including TF_REJECTED), same time
    steps, same fields.  The limit is set from the oracle so that the first attempts are rejected by the criterion."""
    cfg = inputs.config(0)
    nx, ny = 96, 80
    h = inputs.noise_ic(nx, ny, seed=21)
    g, o = pair(tf, tfo, nx, ny, cfg["dx"], cfg["dy"])
    for s in (g, o):
        s.set_newton(1e-10, 64, 0)
        s.set_state(h)
    assert o.step(1e-2)[0] == 0
    limit = 0.3 * tfo.max_rel_change(h, o.get_state())
    o.set_state(h)
    g.set_solution_criteria(limit)
    stepper = tfo.CriteriaStepper(o, limit)
    t_o, dt_o, hist_o, failed = tfo.advance_adaptive(stepper, 1e-2, 12, grow=1.3, shrink=0.5, dt_max=0.05, dt_min=1e-9, grow_after=2)
    t_g, dt_g, hist_g = tf.advance_adaptive(g, 1e-2, 12, grow=1.3, shrink=0.5, dt_max=0.05, dt_min=1e-9, grow_after=2,
                                            on_device=on_device)
    assert not failed
    assert [x[1] for x in hist_g] == [x[1] for x in hist_o]
    assert tf.REJECTED in [x[1] for x in hist_g] and hist_g[0][1] == tf.REJECTED
    assert [x[0] for x in hist_g] == [x[0] for x in hist_o] and (t_g, dt_g) == (t_o, dt_o)
    assert [x[2] for x in hist_g] == [x[2] for x in hist_o]
    assert rel_inf(g.get_state(), o.get_state()) <= 1e-9
    # criterion off again: the same first step is accepted
    g.set_solution_criteria(0.0)
    g.set_state(h)
    assert g.step(1e-2)[0] == tf.OK


# ------------------------------------------------------------------ the rows of the path one at a time
@pytest.mark.parametrize("nx,ny", [(128, 96), (61, 45)])
def test_sweeps_driven_one_by_one_equal_tf_step(tf, nx, ny):
    """tf_sweep (y, then x) / tf_residual / tf_accept reproduce tf_step bit for bit, and the field views alias the
    context's buffers (w of the y-sweep can be overwritten between the sweeps: the x-sweep then solves with it)."""
    import torch
    h0 = inputs.noise_ic(nx, ny, seed=17)
    a = tf.ThinFilm(nx, ny, 0.4259, 0.4259, K, HS, 3, 2)
    b = tf.ThinFilm(nx, ny, 0.4259, 0.4259, K, HS, 3, 2)
    a.set_newton(1e-10, 64, 0)
    for g in (a, b):
        g.set_state(h0)
    for step in range(3):
        st, its, res = a.step(1e-2)
        assert st == tf.OK
        k, r = 0, None
        while True:
            b.sweep(1e-2, k, b.SWEEP_Y)
            b.sweep(1e-2, k, b.SWEEP_X)
            r, bad = b.residual(k)
            k += 1
            assert not bad
            if r < 1e-10:
                break
        b.accept()
        assert (k, r) == (its, res)
        assert np.array_equal(a.get_state(), b.get_state())
    # the views: state view equals get_state; scaling w between the sweeps scales the correction v = u_1 - u_0 (linear solve)
    u = b.field(b.FIELD_STATE).clone()
    assert np.array_equal(u.cpu().numpy(), b.get_state())
    b.sweep(1e-2, 0, b.SWEEP_Y)
    b.sweep(1e-2, 0, b.SWEEP_X)
    v1 = (b.field(b.FIELD_ITERATE) - u).clone()
    b.sweep(1e-2, 0, b.SWEEP_Y)
    b.field(b.FIELD_W).mul_(0.5)
    b.sweep(1e-2, 0, b.SWEEP_X)
    v2 = b.field(b.FIELD_ITERATE) - u
    torch.cuda.synchronize()
    assert float((v2 - 0.5 * v1).abs().max()) <= 1e-13 * float(v1.abs().max())


def test_finite_non_positive_iterate_and_nan_residual_like_the_oracle(tf, tfo):
    """Reading R18 on the CUDA path, on the two cases that pin it in the oracle (tests/test_oracle_pins.py, O13): a first
    iterate that is finite but negative somewhere rejects the step after one iteration in both modes; a valid state
    whose h^3 overflows gives a NaN residual.  Status, count and NaN-ness must equal the oracle's, the state stays u^n."""
    nx, ny, d, dt = 24, 20, 0.05, 1e-2
    h = np.ascontiguousarray(0.12 + 0.1 * np.random.default_rng(5).uniform(0, 1, (ny, nx)))
    for fixed in (1, 0):
        g = tf.ThinFilm(nx, ny, d, d, K, HS, 3, 2)
        o = tfo.ThinFilmOracle(nx, ny, d, d, K, HS, 3, 2)
        for f in (g, o):
            f.set_newton(1e-10, 64, fixed)
            f.set_state(h)
        (gs, gi, gr), (os_, oi, or_) = g.step(dt), o.step(dt)
        assert (gs, gi) == (os_, oi) == (tf.NOT_CONVERGED, 1)
        assert math.isfinite(gr) and abs(gr - or_) <= 1e-9 * abs(or_)
        assert np.array_equal(g.get_state(), h)
    nx, ny = 16, 12
    h = np.ones((ny, nx))
    h[5, 7] = 1e120
    for fixed in (0, 1, 3):
        g = tf.ThinFilm(nx, ny, 0.3, 0.3, K, HS, 3, 2)
        o = tfo.ThinFilmOracle(nx, ny, 0.3, 0.3, K, HS, 3, 2)
        for f in (g, o):
            f.set_newton(1e-10, 10, fixed)
            f.set_state(h)
        (gs, gi, gr), (os_, oi, or_) = g.step(1e-3), o.step(1e-3)
        assert (gs, gi) == (os_, oi) == (tf.NOT_CONVERGED, max(fixed, 1))
        assert math.isnan(gr) and math.isnan(or_)
        assert np.array_equal(g.get_state(), h)

"""tf_advance_adaptive_device (Fig. 1, with every decision on the device)
against (a) the oracle's transcription of the flow chart on a run that DOES reject and (b) the host-side controller
tf_advance_adaptive, which it must equal bit for bit."""
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


def rough_film(nx, ny, seed):
    """grid-scale noise of 5 %: with max_iter = 10 a step of 0.08 does not converge, 0.01 does"""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(1.0 + 0.05 * rng.uniform(-1, 1, (ny, nx)))


@pytest.mark.parametrize("nx,ny,grow_after", [(96, 80, 1), (160, 128, 2), (61, 45, 1)])
def test_device_controller_equals_flow_chart_and_host_controller(tf, tfo, nx, ny, grow_after):
    cfg = inputs.config(0)
    h = rough_film(nx, ny, seed=nx)
    kw = dict(grow=1.6, shrink=0.5, dt_max=0.3, dt_min=1e-9, grow_after=grow_after)
    o = tfo.ThinFilmOracle(nx, ny, cfg["dx"], cfg["dy"], K, HS, 3, 2)
    o.set_newton(1e-10, 10, 0)
    o.set_state(h)
    t_o, dt_o, hist_o, failed = tfo.advance_adaptive(o, 0.08, 14, **kw)
    assert not failed
    runs = []
    for on_device in (True, False):
        g = tf.ThinFilm(nx, ny, cfg["dx"], cfg["dy"], K, HS, 3, 2)
        g.set_newton(1e-10, 10, 0)
        g.set_state(h)
        t, dt, hist = tf.advance_adaptive(g, 0.08, 14, on_device=on_device, **kw)
        runs.append((t, dt, hist, g.get_state(), g.mass()))
        g.close()
    dev, host = runs
    # (b) bit for bit the host controller
    assert dev[0] == host[0] and dev[1] == host[1] and dev[2] == host[2]
    assert np.array_equal(dev[3], host[3])
    # (a) the flow chart: the run rejects, shrinks, accepts, grows
    st = [x[1] for x in dev[2]]
    assert st == [x[1] for x in hist_o] and st.count(tf.NOT_CONVERGED) >= 2 and st.count(tf.OK) == 14
    assert st[0] == tf.NOT_CONVERGED
    assert [x[0] for x in dev[2]] == [x[0] for x in hist_o]                   # the dt sequence, exactly
    assert [x[2] for x in dev[2]] == [x[2] for x in hist_o]                   # Newton counts
    assert all(abs(a[3] - b[3]) <= 1e-4 * abs(b[3]) + 1e-15 for a, b in zip(dev[2], hist_o))   # residuals near tol carry rounding noise
    assert (dev[0], dev[1]) == (t_o, dt_o)
    assert np.max(np.abs(dev[3] - o.get_state())) <= 1e-8 * np.max(np.abs(dev[3]))
    assert abs(dev[4] - o.mass()) <= 1e-13 * o.mass()


def test_device_controller_halts_below_dt_min_with_the_last_accepted_state(tf, tfo):
    """"if the new reduced time step is below some minimum, the numerical scheme halts and ends in a failed state"
    (PAPER.md:254): dt_min above the step that would converge."""
    cfg = inputs.config(0)
    nx, ny = 96, 80
    h = rough_film(nx, ny, seed=3)
    outs = []
    for on_device in (True, False):
        g = tf.ThinFilm(nx, ny, cfg["dx"], cfg["dy"], K, HS, 3, 2)
        g.set_newton(1e-10, 10, 0)
        g.set_state(h)
        t, dt, hist, st = tf.advance_adaptive(g, 0.08, 5, grow=1.1, shrink=0.5, dt_max=0.3, dt_min=0.03, on_device=on_device,
                                              return_status=True)
        outs.append((t, dt, hist, st, g.get_state()))
        g.close()
    dev, host = outs
    assert dev[3] == host[3] == tf.NOT_CONVERGED
    assert dev[:3] == host[:3] and dev[0] == 0.0 and dev[1] < 0.03
    assert all(x[1] == tf.NOT_CONVERGED for x in dev[2]) and len(dev[2]) == 2         # 0.08, 0.04, then 0.02 < dt_min
    assert np.array_equal(dev[4], h) and np.array_equal(host[4], h)


def test_device_controller_attempt_cap_and_refusals(tf):
    cfg = inputs.config(0)
    g = tf.ThinFilm(96, 80, cfg["dx"], cfg["dy"], K, HS, 3, 2)
    g.set_newton(1e-10, 10, 0)
    g.set_state(rough_film(96, 80, seed=4))
    t, dt, hist, st = tf.advance_adaptive(g, 0.08, 50, grow=1.0, shrink=0.9, dt_max=0.3, dt_min=1e-9, max_attempts=3,
                                          on_device=True, return_status=True)
    assert st == tf.NOT_CONVERGED and len(hist) == 3
    g.set_newton(1e-10, 10, 4)                                                       # parity mode: host controller only
    with pytest.raises(tf.TfError) as e:
        tf.advance_adaptive(g, 0.01, 2, on_device=True)
    assert e.value.status == tf.ERR_UNSUPPORTED
    g.close()


def test_config2_on_device_equals_host(tf):
    """Config 2 as stated (4096^2, adaptive from 1e-3, x0.5 / x1.1, cap 0.1): 40 accepted steps with the decisions on the
    device, identical to the host-driven run."""
    cfg = inputs.config(2)
    h = inputs.initial_condition(cfg)
    outs = []
    for on_device in (True, False):
        g = tf.ThinFilm(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
        g.set_newton(cfg["tol"], cfg["max_iter"], 0)
        g.set_state(h)
        t, dt, hist = tf.advance_adaptive(g, cfg["dt"], 40, cfg["grow"], cfg["shrink"], cfg["dt_max"], cfg["dt_min"],
                                          on_device=on_device)
        outs.append((t, dt, hist, g.get_state()))
        g.close()
    assert outs[0][:3] == outs[1][:3] and np.array_equal(outs[0][3], outs[1][3])
    assert len(outs[0][2]) == 40


# ------------------------------------------------------------------ the truncation-error criterion (PAPER.md:252 Note 2, R25)
@pytest.mark.parametrize("on_device", [False, True])
def test_truncation_criterion_against_the_oracle_transcription(tf, tfo, on_device):
    """tf_set_truncation_criterion + tf_advance_adaptive (host controller / every decision on the device) against oracle/tfo.py's TruncationStepper under the same flow
    chart: same accept / REJECTED sequence, same time steps, same Newton counts, estimates equal to 1e-3, same film.
    The limit is taken from a first oracle run so that the growing step is rejected several times."""
    cfg = inputs.config(0)
    nx, ny = 96, 80
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    h = np.ascontiguousarray(1.0 + 0.2 * np.cos(2 * np.pi * x)[None, :] * np.cos(np.pi * y)[:, None])   # smooth: a clean u_ttt
    kw = dict(grow=1.5, shrink=0.5, dt_max=1.0, dt_min=1e-9, grow_after=1)
    DT0 = 0.05
    o = tfo.ThinFilmOracle(nx, ny, cfg["dx"], cfg["dy"], K, HS, 3, 2)
    o.set_newton(1e-14, 200, 0)                               # the estimate divides differences of iterates by dt^2
    o.set_state(h)
    probe = tfo.TruncationStepper(o, 0.0)
    ests = []
    for _ in range(4):
        assert probe.step(DT0)[0] == 0
        ests.append(probe.last)
    limit = 2.0 * ests[-1]                                    # a step 1.5x longer (tau ~ dt^3: x3.4) violates it
    assert ests[-1] > 1e-11, ests
    o.set_state(h)
    stepper = tfo.TruncationStepper(o, limit)
    t_o, dt_o, hist_o, failed = tfo.advance_adaptive(stepper, DT0, 12, **kw)
    assert not failed
    g = tf.ThinFilm(nx, ny, cfg["dx"], cfg["dy"], K, HS, 3, 2)
    g.set_newton(1e-14, 200, 0)
    g.set_truncation_criterion(limit)
    g.set_state(h)
    t_g, dt_g, hist_g = tf.advance_adaptive(g, DT0, 12, on_device=on_device, **kw)
    st = [x_[1] for x_ in hist_g]
    assert st == [x_[1] for x_ in hist_o] and st.count(tf.REJECTED) >= 2 and st[0] == tf.OK
    assert [x_[0] for x_ in hist_g] == [x_[0] for x_ in hist_o] and (t_g, dt_g) == (t_o, dt_o)
    assert [x_[2] for x_ in hist_g] == [x_[2] for x_ in hist_o]
    assert abs(g.last_truncation_estimate() - stepper.last) <= 1e-3 * stepper.last
    assert np.max(np.abs(g.get_state() - o.get_state())) <= 1e-9 * np.max(np.abs(h))
    # one estimate on its own: two equal steps from the same film, GPU against the oracle's transcription
    g.set_truncation_criterion(1.0)
    g.set_state(h)
    o.set_state(h)
    s2 = tfo.TruncationStepper(o, 1.0)
    for _ in range(2):
        assert g.step(DT0)[0] == 0 and s2.step(DT0)[0] == 0
    assert abs(g.last_truncation_estimate() - s2.last) <= 1e-3 * s2.last and s2.last > 0
    g.close()


def test_device_controller_with_the_nlc_pressure_equals_host(tf):
    """The device controller with the paper's NLC pressure (1.8)-(1.9), (1.11): same run as the host controller."""
    nx, ny = 128, 96
    C = 0.0857
    h = 0.2 * (1.0 + 0.05 * np.random.default_rng(8).uniform(-1, 1, (ny, nx)))
    outs = []
    for on_device in (True, False):
        g = tf.ThinFilm(nx, ny, 0.05, 0.05)
        g.set_pressure(tf.PI_NLC, (C, 1.0 / C, 36.0, 0.01, 1.67, 1.0, 0.05))
        g.set_newton(1e-10, 10, 0)
        g.set_state(np.ascontiguousarray(h))
        t, dt, hist = tf.advance_adaptive(g, 1e-3, 10, grow=1.5, shrink=0.5, dt_max=0.1, dt_min=1e-12, on_device=on_device)
        outs.append((t, dt, hist, g.get_state()))
        g.close()
    assert outs[0][:3] == outs[1][:3] and np.array_equal(outs[0][3], outs[1][3])
    assert sum(1 for x in outs[0][2] if x[1] == 0) == 10


def test_device_controller_takes_more_attempts_than_its_record_ring_holds(tf):
    """The device records attempts in a ring of 1024 entries that the host drains between chunks, so a run is not
    limited to 1024 attempts (it was, silently, in round 2): 1100 accepted steps of a small film, with the default
    attempt cap of 50 * n_accept, equal the host controller bit for bit -- every record, the time, the next dt, the film."""
    nx, ny = 48, 40
    h = rough_film(nx, ny, seed=2)
    outs = []
    for on_device in (True, False):
        g = tf.ThinFilm(nx, ny, 0.4, 0.4, K, HS, 3, 2)
        g.set_newton(1e-10, 10, 0)
        g.set_state(h)
        t, dt, hist = tf.advance_adaptive(g, 0.08, 1100, grow=1.3, shrink=0.5, dt_max=0.02, dt_min=1e-9, on_device=on_device)
        outs.append((t, dt, hist, g.get_state()))
        g.close()
    dev, host = outs
    assert len(dev[2]) > 1100 and sum(1 for x in dev[2] if x[1] == tf.OK) == 1100      # it rejected on the way
    assert dev[0] == host[0] and dev[1] == host[1] and dev[2] == host[2]
    assert np.array_equal(dev[3], host[3])


@pytest.mark.parametrize("criteria", ["change", "truncation", "both"])
def test_device_controller_with_the_extra_criteria_equals_host_bit_for_bit(tf, criteria):
    """Row f-4 joined: Fig. 1 on the device WITH the extra solution criteria of PAPER.md:252 Note 2.  The same run under
    the host controller (tf_step decides each criterion on the host) and under tf_advance_adaptive_device (the
    reductions are gated on "converged" and read dt, dt_prev from device memory): every record (dt, status, iterations,
    residual), the time, the next dt and the film are identical bit for bit; the run contains TF_REJECTED attempts.
    Afterwards one more tf_step on each context: the stored a_{n-1/2} and its dt carried over from the device run."""
    cfg = inputs.config(0)
    nx, ny = 96, 80
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    h = np.ascontiguousarray(1.0 + 0.2 * np.cos(2 * np.pi * x)[None, :] * np.cos(np.pi * y)[:, None])
    DT0 = 0.05
    kw = dict(grow=1.5, shrink=0.5, dt_max=1.0, dt_min=1e-9, grow_after=1)
    # limits from a probe run on the host path: four equal steps, criteria switched on with limits that never reject
    g = tf.ThinFilm(nx, ny, cfg["dx"], cfg["dy"], K, HS, 3, 2)
    g.set_newton(1e-14, 200, 0)
    g.set_truncation_criterion(1.0)
    g.set_state(h)
    for _ in range(4):
        before = g.get_state()
        assert g.step(DT0)[0] == tf.OK
    lim_trunc = 2.0 * g.last_truncation_estimate()            # a step 1.5x longer (tau ~ dt^3) violates it
    lim_change = 1.2 * float(np.max(np.abs(g.get_state() - before) / before))   # ... and so does its change of h
    g.close()
    assert lim_trunc > 1e-11 and lim_change > 0
    outs = []
    for on_device in (True, False):
        g = tf.ThinFilm(nx, ny, cfg["dx"], cfg["dy"], K, HS, 3, 2)
        g.set_newton(1e-14, 200, 0)
        if criteria in ("change", "both"):
            g.set_solution_criteria(lim_change)
        if criteria in ("truncation", "both"):
            g.set_truncation_criterion(lim_trunc)
        g.set_state(h)
        t, dt, hist = tf.advance_adaptive(g, DT0, 12, on_device=on_device, **kw)
        after_run = g.get_state()
        extra = g.step(dt)                                    # the next step of the schedule, decided by tf_step on the host
        outs.append((t, dt, hist, after_run, extra, g.get_state(), g.last_truncation_estimate()))
        g.close()
    dev, host = outs
    st = [r[1] for r in dev[2]]
    assert st.count(tf.REJECTED) >= 2 and st.count(tf.OK) == 12 and st[0] == tf.OK
    assert dev[0] == host[0] and dev[1] == host[1] and dev[2] == host[2]
    assert np.array_equal(dev[3], host[3])
    assert dev[4] == host[4] and np.array_equal(dev[5], host[5])
    if criteria != "change":
        assert dev[6] == host[6] and dev[6] > 0.0

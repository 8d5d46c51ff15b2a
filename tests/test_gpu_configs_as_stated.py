"""GPU parity on BASELINE.json's configs AS STATED: the whole 8192^2 field against the
OpenMP build of the oracle (no window argument), config 1 run to its 2000 steps with element-wise parity from a
RUPTURED film and a rejected step there, config 0 to 2000 steps with the oracle's Newton-count profile beside it, and
config 2 to its 200 accepted steps.  Tolerances are BASELINE.json's (1e-11 after one fixed-count step)."""
import numpy as np
import pytest

from paper_1806_10550_b200 import inputs

pytestmark = pytest.mark.gpu


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


def make(tf, cfg, nx=None, ny=None):
    return tf.ThinFilm(nx or cfg["nx"], ny or cfg["ny"], cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])


def make_o(tfo, cfg, nx=None, ny=None, omp=True):
    return tfo.ThinFilmOracle(nx or cfg["nx"], ny or cfg["ny"], cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"],
                              cfg["m"], omp=omp)


# ------------------------------------------------------------------ config 3: every one of the 6.7e7 elements
def test_config3_8192_full_domain_parity(tf, tfo):
    """One step of three fixed iterations on the whole 8192 x 8192 film, in the launch configuration bench.py times:
    every element against the oracle's OpenMP build (same source as the serial build), residual and mass too."""
    cfg = inputs.config(3)
    h = inputs.initial_condition(cfg)
    g = make(tf, cfg)
    g.set_newton(cfg["tol"], cfg["max_iter"], 3)
    g.set_state(h)
    sg = g.step(cfg["dt"])
    ug, mg = g.get_state(), g.mass()
    g.close()
    o = make_o(tfo, cfg)
    o.set_newton(cfg["tol"], cfg["max_iter"], 3)
    o.set_state(h)
    so = o.step(cfg["dt"])
    uo, mo = o.get_state(), o.mass()
    o.close()
    assert sg[:2] == so[:2] == (0, 3)
    d = np.abs(ug - uo)
    worst = float(d.max() / np.abs(uo).max())
    assert worst <= 1e-11, (worst, np.unravel_index(np.argmax(d), d.shape))
    assert abs(sg[2] - so[2]) <= 1e-9 * so[2]
    assert abs(mg - mo) <= 1e-13 * mo
    print(f"8192^2 full domain, 3 iterations: worst rel Linf {worst:.2e}")


# ------------------------------------------------------------------ config 1: 2000 steps, rupture, parity after rupture
@pytest.fixture(scope="module")
def config1_run(tf):
    """Config 1 as stated: 1024^2, dt = 1e-2, 2000 steps, tol 1e-10.  Keeps the film at step 1000.
    max_iter: SURVEY.md 8(c) A14 asks for ">= 64" at the fixed-dt configs from a 128^2 probe; at 1024^2 a few steps late
    in the run (many touching drops) need more than 64 sweeps -- step 1737 stops at 1.2e-10 after 64 -- so the run
    uses 128 (reading R14 in DESIGN.md) and the test reports how many steps went beyond 64."""
    cfg = inputs.config(1)
    h = inputs.initial_condition(cfg)
    g = make(tf, cfg)
    g.set_newton(cfg["tol"], 128, 0)
    g.set_state(h)
    m0 = g.mass()
    its, hmin, snap = [], [], None
    for n in range(2000):
        st, it, res = g.step(cfg["dt"])
        assert st == 0, (n, st, it, res)                 # no rejected step at max_iter = 128
        its.append(it)
        if n % 50 == 49:
            u = g.get_state()
            hmin.append(float(u.min()))
            assert np.all(np.isfinite(u)) and u.min() > 0
            if n == 999:
                snap = u
    m1, u_end = g.mass(), g.get_state()
    g.close()
    return cfg, m0, m1, np.array(its), np.array(hmin), snap, u_end


def test_config1_2000_steps_invariants(config1_run):
    cfg, m0, m1, its, hmin, snap, u_end = config1_run
    assert abs(m1 - m0) <= 1e-13 * m0                   # (3.2) over the whole run, rupture included
    assert its.max() <= 128 and np.sum(its > 64) <= 200                                 # some steps late in the run go beyond 64
    assert its[:12].tolist() == sorted(its[:12].tolist(), reverse=True)                  # grid-scale noise decays
    assert its[100:400].max() <= 8                      # smooth growth phase
    assert hmin.min() < 0.2 and hmin[-1] > 0.05         # the film ruptured (h -> ~h*) and stayed positive
    assert its[1200:].mean() > 2 * its[100:400].mean()  # after rupture the iteration needs several times more sweeps
    assert u_end.max() > 2.0                            # drops have formed
    print(f"config 1: Newton counts first {its[:5].tolist()}, min/max mid-run {its[100:400].min()}/{its[100:400].max()}, "
          f"after rupture mean {its[1200:].mean():.1f} max {its[1200:].max()} ({int(np.sum(its > 64))} steps > 64), "
          f"min h {hmin.min():.4f}, max h {u_end.max():.2f}")


def test_config1_parity_from_a_ruptured_film(tf, tfo, config1_run):
    """From the GPU's film at step 1000 (h from ~0.09 to several units): one step of 6 fixed iterations, every element
    against the oracle (1e-11); the converged step takes the same Newton count; with max_iter = 10 both
    reject the step and keep the state."""
    cfg, _, _, its, hmin, snap, _ = config1_run
    assert snap.min() < 0.2 and snap.max() > 1.5, (snap.min(), snap.max())
    g, o = make(tf, cfg), make_o(tfo, cfg)
    for s in (g, o):
        s.set_newton(cfg["tol"], cfg["max_iter"], 6)
        s.set_state(snap)
    sg, so = g.step(cfg["dt"]), o.step(cfg["dt"])
    assert sg[:2] == so[:2] == (0, 6)
    ug, uo = g.get_state(), o.get_state()
    worst = float(np.max(np.abs(ug - uo)) / np.max(np.abs(uo)))
    assert worst <= 1e-11, worst
    assert abs(sg[2] - so[2]) <= 1e-9 * so[2]
    for s in (g, o):                                     # converged step from the same ruptured film
        s.set_newton(cfg["tol"], cfg["max_iter"], 0)
        s.set_state(snap)
    sg, so = g.step(cfg["dt"]), o.step(cfg["dt"])
    conv_iters = sg[1]
    assert sg[0] == so[0] == 0 and sg[1] == so[1] and sg[1] > 10, (sg, so)
    assert np.max(np.abs(g.get_state() - o.get_state())) <= 1e-8 * np.max(np.abs(uo))
    for s in (g, o):                                     # the paper's K = 10 rejects this step: state untouched
        s.set_newton(cfg["tol"], 10, 0)
        s.set_state(snap)
    sg, so = g.step(cfg["dt"]), o.step(cfg["dt"])
    assert sg[:2] == so[:2] == (1, 10)
    assert np.array_equal(g.get_state(), snap) and np.array_equal(o.get_state(), snap)
    print(f"config 1, ruptured film (h in [{snap.min():.3f}, {snap.max():.2f}]): worst rel Linf {worst:.2e}, "
          f"converged in {conv_iters} iterations at max_iter 64, rejected at K = 10")


def test_config0_2000_steps_newton_profile_matches_oracle(tf, tfo):
    """Config 0's film run to 2000 steps (through rupture) on both sides: the Newton-count profile.  Fields are not
    compared late in the run (the instability amplifies rounding differences); counts are equal while
    the fields still agree to 1e-8 and within 2 afterwards, and the mass never moves."""
    cfg = inputs.config(0)
    h = inputs.initial_condition(cfg)
    g, o = make(tf, cfg), make_o(tfo, cfg, omp=False)
    for s in (g, o):
        s.set_newton(cfg["tol"], cfg["max_iter"], 0)
        s.set_state(h)
    m0 = g.mass()
    ig, io, agree_until = [], [], None
    for n in range(2000):
        sg, so = g.step(cfg["dt"]), o.step(cfg["dt"])
        assert sg[0] == so[0] == 0
        ig.append(sg[1]); io.append(so[1])
        if agree_until is None and n % 25 == 24:
            if np.max(np.abs(g.get_state() - o.get_state())) > 1e-8 * np.max(np.abs(o.get_state())):
                agree_until = n
    ig, io = np.array(ig), np.array(io)
    upto = agree_until if agree_until is not None else 2000
    assert upto >= 600, upto                             # well past the 100 steps of the stated tolerance
    assert np.array_equal(ig[:upto - 25], io[:upto - 25])
    assert np.max(np.abs(ig - io)) <= 2
    assert abs(g.mass() - m0) <= 1e-13 * m0 and abs(o.mass() - m0) <= 1e-13 * m0
    u = g.get_state()
    assert u.min() > 0 and u.min() < 0.2 and ig[1000:].max() >= 15
    print(f"config 0, 2000 steps: fields agree to 1e-8 for {upto} steps, counts differ at {int(np.sum(ig != io))} steps "
          f"(max by {int(np.max(np.abs(ig - io)))}), after rupture {ig[1000:].min()}-{ig[1000:].max()} iterations")


# ------------------------------------------------------------------ config 2: 200 accepted steps
def test_config2_4096_200_accepted_steps(tf):
    cfg = inputs.config(2)
    h = inputs.initial_condition(cfg)
    g = make(tf, cfg)
    g.set_newton(cfg["tol"], cfg["max_iter"], 0)
    g.set_state(h)
    m0 = g.mass()
    t, dt_next, hist = tf.advance_adaptive(g, cfg["dt"], 200, cfg["grow"], cfg["shrink"], cfg["dt_max"], cfg["dt_min"])
    acc = [x for x in hist if x[1] == 0]
    assert len(acc) == 200
    assert all(it <= cfg["max_iter"] and res < cfg["tol"] for _, st, it, res in acc)
    for a, b in zip(hist[:-1], hist[1:]):               # Fig. 1: x1.1 after a success (capped), x0.5 after a failure
        want = min(a[0] * cfg["grow"], cfg["dt_max"]) if a[1] == 0 else a[0] * cfg["shrink"]
        assert abs(b[0] - want) <= 1e-15 * want
    assert abs(t - sum(x[0] for x in acc)) <= 1e-12 * t
    u = g.get_state()
    assert abs(g.mass() - m0) <= 1e-13 * m0
    assert np.all(np.isfinite(u)) and u.min() > h.min() and u.max() <= 0.12 + 1e-9
    g.close()
    print(f"config 2: 200 accepted of {len(hist)} attempts, t = {t:.3f}, dt_next = {dt_next:.4f}, "
          f"iterations {min(x[2] for x in acc)}-{max(x[2] for x in acc)}")

"""Pin of the oracle's truncation-error criterion (oracle/tfo.py TruncationStepper; PAPER.md:252 Note 2, reading R25):
for the linear model (1.6) a single no-flux Fourier mode is an eigenvector of the discrete operator, Crank-Nicolson
multiplies its amplitude by R = (1 + sigma dt/2)/(1 - sigma dt/2) per step, and the estimate has a closed form that is
typed out here from those two facts alone (no oracle arithmetic): with steps dt1, dt2
    a_{1/2} = sigma (R1 - 1) e0 / dt1,   a_{3/2} = sigma (R2 - 1) R1 e0 / dt2,
    tau     = (dt2^3 / 12) |a_{3/2} - a_{1/2}| / ((dt1 + dt2)/2)      -> (dt^3/12) |sigma|^3 e0 as dt -> 0 (textbook LTE)."""
import math

import numpy as np
import pytest

from oracle import tfo


def mode_setup(direction, k, npts=32, c0=1.0, c1=1.7, eps=1e-2):
    L = 6.8
    d = L / npts
    q = k * math.pi / L
    q2 = (4.0 / d ** 2) * math.sin(q * d / 2) ** 2
    sigma = -(c0 * q2 ** 2 - c1 * q2)                         # eigenvalue of -D for the discrete mode
    nx, ny = (npts, 6) if direction == 0 else (6, npts)
    mode = np.cos(k * math.pi * (np.arange(npts) + 0.5) * d / L)
    shape = (mode[None, :] if direction == 0 else mode[:, None]) * np.ones((ny, nx))
    o = tfo.ThinFilmOracle(nx, ny, d, d)
    o.set_model_linear(c0, c1)
    o.set_newton(1e-14, 500, 0)
    o.set_state(np.ascontiguousarray(1.0 + eps * shape))
    return o, sigma, shape, eps


@pytest.mark.parametrize("direction", [0, 1])
@pytest.mark.parametrize("k,dt1,dt2", [(2, 0.05, 0.05), (3, 0.02, 0.035), (1, 0.2, 0.1)])
def test_estimate_equals_closed_form_for_a_linear_mode(direction, k, dt1, dt2):
    o, sigma, shape, e0 = mode_setup(direction, k)
    s = tfo.TruncationStepper(o, 0.0)
    assert s.step(dt1)[0] == 0 and s.last == 0.0              # no history yet: not tested
    assert s.step(dt2)[0] == 0
    R1 = (1 + sigma * dt1 / 2) / (1 - sigma * dt1 / 2)
    R2 = (1 + sigma * dt2 / 2) / (1 - sigma * dt2 / 2)
    a1 = sigma * (R1 - 1) * e0 / dt1
    a2 = sigma * (R2 - 1) * R1 * e0 / dt2
    tau = dt2 ** 3 / 12.0 * abs(a2 - a1) / (0.5 * (dt1 + dt2))
    u2 = 1.0 + R1 * R2 * e0 * shape
    expect = float(np.max(tau * np.abs(shape) / np.abs(u2)))
    assert abs(s.last - expect) <= 1e-4 * expect, (s.last, expect)     # differences of O(1) fields divided by dt^2: ~1e-6 noise
    if dt1 == dt2:                                            # and the textbook leading term of the trapezoidal rule
        lead = dt1 ** 3 / 12.0 * abs(sigma) ** 3 * e0
        assert abs(tau - lead) <= 2.0 * abs(sigma) * dt1 * lead


def test_rejection_keeps_state_and_history():
    o, sigma, shape, e0 = mode_setup(0, 2)
    s = tfo.TruncationStepper(o, 1e-30)                       # nothing passes once there is a history
    assert s.step(0.05)[0] == tfo.OK
    before, a_prev = o.get_state(), s.a_prev.copy()
    assert s.step(0.05)[0] == tfo.REJECTED
    assert np.array_equal(o.get_state(), before) and np.array_equal(s.a_prev, a_prev)
    s.limit = 1.0
    assert s.step(0.05)[0] == tfo.OK and s.last > 0

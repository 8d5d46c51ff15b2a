"""Host logic of the adaptive time-stepping controller (Fig. 1).  The controller is native code in
the C-ABI library (tf_adaptive_run / tf_advance_adaptive); here it is driven through a callback with scripted
stand-ins for the step -- no GPU -- and compared with (a) hand-written expected sequences and (b) the oracle's
step-by-step transcription of the flow chart on random scripts."""
import numpy as np
import pytest

from paper_1806_10550_b200 import tf


class Scripted:
    """step(dt) fails (status 1 = TF_NOT_CONVERGED) whenever dt > limit."""
    def __init__(self, limit):
        self.limit, self.calls = limit, []

    def step(self, dt):
        self.calls.append(dt)
        return (tf.OK, 4, 1e-11) if dt <= self.limit else (tf.NOT_CONVERGED, 10, 1e-3)


def test_grow_on_success_halve_on_failure_and_cap():
    c = Scripted(limit=2.5e-3)
    t, dt, hist = tf.advance_adaptive(c, 1e-3, 6, grow=2.0, shrink=0.5, dt_max=0.1)
    # 1e-3 ok, 2e-3 ok, 4e-3 rejected -> 2e-3 ok, 4e-3 rejected -> 2e-3 ok ...
    assert [round(x[0], 12) for x in hist[:5]] == [1e-3, 2e-3, 4e-3, 2e-3, 4e-3]
    assert [x[1] for x in hist[:5]] == [0, 0, 1, 0, 1]
    assert sum(1 for x in hist if x[1] == 0) == 6
    assert abs(t - sum(x[0] for x in hist if x[1] == 0)) < 1e-15          # only accepted steps advance time
    assert c.calls == [x[0] for x in hist]                                # one step call per attempt, same dt
    c = Scripted(limit=1.0)
    t, dt, hist = tf.advance_adaptive(c, 0.03, 5, grow=2.0, shrink=0.5, dt_max=0.1)
    assert [x[0] for x in hist] == [0.03, 0.06, 0.1, 0.1, 0.1] and dt == 0.1  # bounded from above


def test_grows_only_after_a_streak_of_accepted_steps():
    """"the time step is increased if a minimum number of successful time steps have been consecutively
    computed" -- grow_after = 3: dt doubles after every third consecutive success, a rejection resets the streak"""
    c = Scripted(limit=3e-3)
    t, dt, hist = tf.advance_adaptive(c, 1e-3, 9, grow=2.0, shrink=0.5, dt_max=0.1, grow_after=3)
    assert [round(x[0], 12) for x in hist] == [1e-3] * 3 + [2e-3] * 3 + [4e-3] + [2e-3] * 3
    assert [x[1] for x in hist] == [0] * 6 + [1] + [0] * 3
    assert round(dt, 12) == 4e-3                                          # the third success after the rejection grew it again


def test_gives_up_below_dt_min_and_reports_hard_errors():
    c = Scripted(limit=0.0)
    with pytest.raises(tf.TfError) as e:
        tf.advance_adaptive(c, 1e-3, 1, dt_min=1e-6)
    assert e.value.status == tf.NOT_CONVERGED and len(c.calls) == 10      # 1e-3 * 2^-10 < 1e-6

    class Broken:
        def step(self, dt):
            return tf.ERR_CUDA, 0, 0.0
    with pytest.raises(tf.TfError) as e:
        tf.advance_adaptive(Broken(), 1e-3, 3)
    assert e.value.status == tf.ERR_CUDA
    with pytest.raises(tf.TfError):                                        # argument validation in the library
        tf.advance_adaptive(Scripted(1.0), 1e-3, 3, shrink=1.5)


def test_native_controller_equals_the_flow_chart_on_random_scripts(oracle_mod):
    """random accept/reject scripts (including TF_REJECTED = 2 from an extra criterion) and random constants: the
    library's controller and the oracle's transcription of Fig. 1 make the same calls and return the same history"""
    rng = np.random.default_rng(5)
    for trial in range(200):
        script = rng.choice([0, 0, 0, 1, 2], size=400).tolist()
        grow, shrink = float(rng.uniform(1.0, 2.0)), float(rng.uniform(0.2, 0.9))
        grow_after, n_accept = int(rng.integers(1, 5)), int(rng.integers(0, 40))
        dt0, dt_max, dt_min = float(rng.uniform(1e-4, 1e-1)), float(rng.uniform(1e-3, 1e-1)), float(rng.choice([1e-12, 1e-5]))

        class Tape:
            def __init__(self):
                self.k, self.calls = 0, []

            def step(self, dt):
                st = script[self.k]
                self.k += 1
                self.calls.append(dt)
                return st, 3 + self.k % 7, 1e-11 * self.k

        a, b = Tape(), Tape()
        t_o, dt_o, hist_o, failed = oracle_mod.advance_adaptive(a, dt0, n_accept, grow, shrink, dt_max, dt_min, grow_after, 300)
        try:
            t_g, dt_g, hist_g = tf.advance_adaptive(b, dt0, n_accept, grow, shrink, dt_max, dt_min, 300, grow_after)
            assert not failed
            assert (t_g, dt_g) == (t_o, dt_o)
        except tf.TfError as e:
            assert failed and e.status == tf.NOT_CONVERGED
            hist_g = None
        assert a.calls == b.calls
        if hist_g is not None:
            assert hist_g == hist_o

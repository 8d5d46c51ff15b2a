"""Host logic of the adaptive time-stepping controller (Fig. 1) with a scripted stand-in for
the context: no GPU, no library call."""
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
    c = Scripted(limit=1.0)
    t, dt, hist = tf.advance_adaptive(c, 0.03, 5, grow=2.0, shrink=0.5, dt_max=0.1)
    assert [x[0] for x in hist] == [0.03, 0.06, 0.1, 0.1, 0.1] and dt == 0.1  # bounded from above


def test_gives_up_below_dt_min():
    c = Scripted(limit=0.0)
    with pytest.raises(tf.TfError):
        tf.advance_adaptive(c, 1e-3, 1, dt_min=1e-6)

"""tf_radial_peaks (App. B steps 5-6 and the maxima) is host code of the C-ABI library: it is compared
here, without a GPU, with the oracle's transcription of the appendix (oracle/spectrum.py) on synthetic radial spectra,
and checked on its own against a function whose maximum is known."""
import numpy as np
import pytest

from oracle import spectrum
from paper_1806_10550_b200 import tf


def spectra():
    rng = np.random.default_rng(3)
    out = []
    for n, qmax in ((3000, 6.0), (257, 3.0), (95, 5.0), (40, 2.0)):
        q = np.sort(rng.uniform(1e-3, qmax, n))
        z = q * np.exp(-0.5 * ((q - 0.4 * qmax) / (0.15 * qmax)) ** 2) + 1.0 * np.exp(-0.5 * ((q - 0.8 * qmax) / (0.05 * qmax)) ** 2) \
            + 0.01 * rng.standard_normal(n)
        out.append((np.concatenate([[0.0], q]), np.concatenate([[123.0], z])))      # a q = 0 entry that must be ignored
    return out


@pytest.mark.parametrize("case", range(4))
def test_against_the_oracle(case):
    q, z = spectra()[case]
    xg, fg, pg = tf.radial_peaks(q, z, 10, 400)
    xo, fo, po = spectrum.smooth_and_peaks(q, z, 10, 400)
    assert np.allclose(xg, xo, rtol=0, atol=1e-14)
    assert np.max(np.abs(fg - fo)) <= 1e-9 * np.max(np.abs(fo))                     # normal equations vs numpy's lstsq
    assert len(pg) == len(po)
    for (a, b), (c, d) in zip(pg, po):
        assert abs(a - c) <= 1e-6 and abs(b - d) <= 1e-9


def test_known_maximum_and_argument_checks():
    q, z = spectra()[0]
    _, _, peaks = tf.radial_peaks(q, z)
    q0, s = 0.4 * 6.0, 0.15 * 6.0
    true_max = 0.5 * (q0 + np.sqrt(q0 * q0 + 4 * s * s))
    assert min(abs(p[0] - true_max) for p in peaks) < 0.05                          # the broad maximum
    assert min(abs(p[0] - 0.8 * 6.0) for p in peaks) < 0.05                         # and the narrow one
    with pytest.raises(tf.TfError):
        tf.radial_peaks(q[::-1], z)                                                 # not ascending
    with pytest.raises(tf.TfError):
        tf.radial_peaks(q[:5], z[:5])                                               # fewer points than one interval

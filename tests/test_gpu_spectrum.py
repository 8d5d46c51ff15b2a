"""GPU parity of tf_radial_spectrum (App. B steps 1-4) against oracle/spectrum.py (numpy fp64):
radii and counts exactly, mean magnitudes to 1e-11 relative to the largest (cuFFT and numpy's FFT differ in rounding
order; the radial sums are accumulated with atomics in arbitrary order)."""
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


def both(tf, h, L, H0, sigma, kmax):
    import torch
    from oracle import spectrum
    qg, zg, cg = tf.radial_spectrum(torch.from_numpy(np.ascontiguousarray(h)).cuda(), L, H0, sigma, kmax)
    qo, zo, co = spectrum.radial_spectrum(h, H0, sigma, kmax, L)
    return (qg, zg, cg), (qo, zo, co)


@pytest.mark.parametrize("ny,nx", [(64, 64), (48, 80), (81, 45), (130, 258)])
@pytest.mark.parametrize("sigma", [0.0, 0.7, 2.4])
def test_random_films(tf, ny, nx, sigma):
    rng = np.random.default_rng(ny + nx)
    h = 1.0 + 0.1 * rng.uniform(-1, 1, (ny, nx))
    g, o = both(tf, h, 12.5, 1.0, sigma, 30)
    assert len(g[0]) == len(o[0]) and np.array_equal(g[2], o[2])
    assert np.allclose(g[0], o[0], rtol=1e-15, atol=0)
    assert np.max(np.abs(g[1] - o[1])) <= 1e-11 * np.max(np.abs(o[1]))


def test_single_mode_and_film_of_the_path(tf):
    n, k, eps, H0, L = 256, 9, 1e-3, 0.5, 20.0
    x = np.arange(n)
    h = H0 + eps * np.cos(2 * np.pi * k * x / n)[:, None] * np.ones((1, n))          # a mode along y
    q, z, cnt = tf.radial_spectrum(__import__("torch").from_numpy(h).cuda(), L, H0, 0.0, 40)
    i = int(np.argmax(z))
    assert abs(q[i] - 2 * np.pi * k / L) < 1e-12 and abs(z[i] * cnt[i] - eps * n * n) < 1e-7   # two spikes of eps n^2 / 2
    # a solution of the path: config-0 film after 30 steps, the paper's usage (dominant wavelength of the pattern)
    cfg = inputs.config(0)
    g = tf.ThinFilm(128, 128, cfg["dx"], cfg["dy"])
    g.set_newton(1e-10, 64, 0)
    g.set_state(inputs.noise_ic(128, 128, seed=0))
    for _ in range(30):
        assert g.step(cfg["dt"])[0] == 0
    hh = g.get_state()
    a, b = both(tf, hh, 128 * cfg["dx"], 1.0, 1.5, 40)
    assert np.array_equal(a[2], b[2]) and np.max(np.abs(a[1] - b[1])) <= 1e-11 * np.max(np.abs(b[1]))


def test_full_size_4096(tf):
    """config 2's grid size; the oracle's binning loop is replaced by a vectorised numpy bincount of the same keys"""
    import torch
    from oracle import spectrum
    n, kmax = 4096, 200
    rng = np.random.default_rng(5)
    h = 1.0 + 0.01 * rng.uniform(-1, 1, (n, n))
    q, z, cnt = tf.radial_spectrum(torch.from_numpy(h).cuda(), n * 0.43, 1.0, 1.0, kmax)
    sm = spectrum.gaussian_filter(spectrum.magnitude(h, 1.0), 1.0)
    k = np.fft.fftfreq(n, 1.0 / n).round().astype(np.int64)
    key = (k[:, None] ** 2 + k[None, :] ** 2).ravel()
    keep = key <= kmax * kmax
    sums = np.bincount(key[keep], weights=sm.ravel()[keep], minlength=kmax * kmax + 1)
    cn = np.bincount(key[keep], minlength=kmax * kmax + 1)
    present = np.nonzero(cn)[0]
    assert np.array_equal(cnt, cn[present])
    assert np.allclose(q, 2 * np.pi * np.sqrt(present) / (n * 0.43), rtol=1e-15, atol=0)
    assert np.max(np.abs(z - sums[present] / cn[present])) <= 1e-11 * np.max(z)

"""Pins of the radial-spectrum oracle (oracle/spectrum.py; App. B steps 1-4) against closed forms:
the DFT of a single cosine mode, lattice-point counts r2(n) of number theory, conservation and symmetry of the
normalised Gaussian filter, and a radially symmetric input (whose angular mean is the input itself)."""
import numpy as np

from oracle import spectrum


def test_single_mode_gives_one_ring_with_the_closed_form_magnitude():
    n, k, eps, H0 = 64, 5, 1e-2, 0.7
    x = np.arange(n)
    h = H0 + eps * np.cos(2 * np.pi * k * x / n)[None, :] * np.ones((n, 1))
    mag = spectrum.magnitude(h, H0)
    # zeta = eps cos(2 pi k i / n): two spikes of height eps n^2 / 2 at (ky, kx) = (0, +-k), nothing else
    assert abs(mag[0, k] - eps * n * n / 2) < 1e-9 and abs(mag[0, n - k] - eps * n * n / 2) < 1e-9
    mag[0, k] = mag[0, n - k] = 0.0
    assert mag.max() < 1e-9
    L = 10.0
    q, z, cnt = spectrum.radial_spectrum(h, H0, 0.0, 20, L)
    i = int(np.argmax(z))
    assert abs(q[i] - 2 * np.pi * k / L) < 1e-12                 # the ring sits at q = 2 pi k / L
    # key 25 = 5^2 + 0 = 3^2 + 4^2 has 12 lattice points, two of them carry the spikes
    assert cnt[i] == 12 and abs(z[i] - 2 * (eps * n * n / 2) / 12) < 1e-9


def test_counts_are_the_lattice_point_numbers_r2():
    """N_k of (B.1) = number of integer points on the circle kx^2 + ky^2 = key: r2(0)=1, r2(1)=4, r2(2)=4, r2(3)=0,
    r2(4)=4, r2(5)=8, r2(25)=12, r2(50)=12, r2(65)=16"""
    keys, _, cnt = spectrum.radial_mean(np.ones((40, 40)), 10)
    d = dict(zip(keys.tolist(), cnt.tolist()))
    assert [d.get(k, 0) for k in (0, 1, 2, 3, 4, 5, 25, 50, 65)] == [1, 4, 4, 0, 4, 8, 12, 12, 16]
    assert max(keys) <= 100 and 3 not in d and 7 not in d


def test_gaussian_filter_is_normalised_symmetric_and_periodic():
    rng = np.random.default_rng(0)
    a = rng.uniform(0, 1, (24, 30))
    for sigma in (0.0, 0.8, 2.5):
        f = spectrum.gaussian_filter(a, sigma)
        assert abs(f.sum() - a.sum()) < 1e-10 * a.sum()          # weights sum to one, wrap-around loses nothing
        assert np.allclose(spectrum.gaussian_filter(a[::-1, ::-1], sigma), f[::-1, ::-1], atol=1e-14)
    assert np.array_equal(spectrum.gaussian_filter(a, 0.0), a)
    d = np.zeros((9, 9))
    d[0, 0] = 1.0                                                 # impulse at the corner: the kernel wraps around
    f = spectrum.gaussian_filter(d, 1.0)
    w = spectrum.gaussian_weights(1.0)
    assert abs(f[0, 0] - w[3] * w[3]) < 1e-15 and abs(f[8, 0] - w[2] * w[3]) < 1e-15 and abs(f[0, 2] - w[5] * w[3]) < 1e-15
    assert abs(w.sum() - 1) < 1e-15 and len(w) == 7 and np.allclose(w[1] / w[3], np.exp(-2.0))


def test_radially_symmetric_input_is_its_own_angular_mean():
    n = 48
    k = np.fft.fftfreq(n, 1.0 / n)
    r2 = k[:, None] ** 2 + k[None, :] ** 2
    f = np.exp(-r2 / 50.0) * (1 + 0.3 * np.cos(0.2 * np.sqrt(r2)))
    keys, means, _ = spectrum.radial_mean(f, 15)
    assert np.allclose(means, np.exp(-keys / 50.0) * (1 + 0.3 * np.cos(0.2 * np.sqrt(keys))), rtol=0, atol=1e-14)


# ------------------------------------------------------------------ steps five and six, maxima
def test_fit_reproduces_a_piecewise_linear_function_on_its_own_knots():
    rng = np.random.default_rng(1)
    q = np.sort(rng.uniform(0.01, 5.0, 95))
    ks = spectrum.knots(q, 10)
    assert ks[0] == 0.0 and ks[1] == q[9] and ks[2] == q[19] and ks[-1] == q[-1] and len(ks) == 11   # 9 full intervals + 5 left over
    a_true = np.concatenate([[0.0], rng.uniform(-1, 1, len(ks) - 1)])
    z = np.interp(q, ks, a_true)
    ks2, a = spectrum.piecewise_linear_fit(q, z, 10)
    assert np.array_equal(ks2, ks) and np.allclose(a, a_true, atol=1e-10)       # data on the model: residual zero, parameters recovered
    # and it IS a least-squares solution for noisy data: the residual is orthogonal to every hat function
    zn = z + 0.1 * rng.standard_normal(len(q))
    _, an = spectrum.piecewise_linear_fit(q, zn, 10)
    r = np.interp(q, ks, an) - zn
    for k in range(1, len(ks)):
        e = np.zeros(len(ks)); e[k] = 1.0
        assert abs(np.dot(r, np.interp(q, ks, e))) < 1e-10


def test_moving_average_properties():
    x = np.linspace(0, 1, 50)
    lin = 2.0 + 3.0 * x
    for P in (1, 2, 3):
        m = spectrum.moving_average(lin, P)
        assert np.allclose(m[P:-P], lin[P:-P], atol=1e-14)                       # symmetric window: linear functions pass
        assert abs(m[0] - lin[:P + 1].mean()) < 1e-14                             # truncated window at the end
    imp = np.zeros(21); imp[10] = 1.0
    m = spectrum.moving_average(imp, 3)
    assert np.allclose(m[7:14], 1.0 / 7) and m[6] == 0 and m[14] == 0


def test_maximum_of_a_noisy_bump_is_found():
    rng = np.random.default_rng(2)
    q = np.sort(rng.uniform(0.0, 6.0, 3000))
    q0 = 2.2
    z = q * np.exp(-0.5 * ((q - q0) / 0.8) ** 2) + 0.01 * rng.standard_normal(len(q))
    true_max = 0.5 * (q0 + np.sqrt(q0 * q0 + 4 * 0.64))                          # d/dq [q exp(-(q-q0)^2/(2 s^2))] = 0
    x, f, peaks = spectrum.smooth_and_peaks(q, z, 10, 400)
    assert len(x) == 400 and x[0] == 0.0 and abs(x[-1] - q[-1]) < 1e-15
    best = max(peaks, key=lambda p: p[1])
    assert abs(best[0] - true_max) < 0.05

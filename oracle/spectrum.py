"""CPU oracle for the first four steps of the radial Fourier transform (Appendix B).
TEST INFRASTRUCTURE ONLY: same rules as oracle/tfo.py (only tests/ may import it; nothing from the CUDA package).

Appendix B, steps one to four, written out with numpy (fp64) in the paper's order:
  1. "the peak at the zero wave number is removed by subtracting the initial film thickness H0, i.e., the magnitude of
     the Fourier transform of zeta(x,y) = h(x,y) - H0 is computed"                       -> magnitude()
  2. "the magnitude of the Fourier transform data is convoluted with a Gaussian function/filter"  -> gaussian_filter()
  3./4. "mapped from the Cartesian coordinates (q_x, q_y) to polar coordinates ... averaging over the theta direction for
     a fixed q_r", eq. (B.1): mean over P_k = {points with q_r = q_rk}, N_k = number of points in P_k   -> radial_mean()
Readings the paper leaves open (R23): the discrete transform is the plain 2-D DFT of the nx x ny samples
(np.fft.fft2 convention); the Gaussian has standard deviation `sigma` in units of the DFT index, is truncated at
ceil(3 sigma), normalised to sum 1 and wraps periodically; P_k groups points of EQUAL radius, which on a square domain
(nx dx = ny dy, the paper's domains) means equal kx^2 + ky^2 of the signed DFT indices; q_r = 2 pi sqrt(key) / L.
Steps five and six of the appendix (least-squares fit, moving average, maxima) follow further down.
"""
import numpy as np


def magnitude(h, H0):
    """|DFT2(h - H0)|, [ny][nx], DFT index layout (zero frequency at [0][0])."""
    return np.abs(np.fft.fft2(np.asarray(h, dtype=np.float64) - H0))


def gaussian_weights(sigma):
    if sigma <= 0:
        return np.array([1.0])
    r = int(np.ceil(3.0 * sigma))
    m = np.arange(-r, r + 1, dtype=np.float64)
    w = np.exp(-m * m / (2.0 * sigma * sigma))
    return w / w.sum()


def gaussian_filter(mag, sigma):
    """periodic convolution with the separable, truncated, normalised Gaussian: out[k] = sum_m w[m] mag[k - m]"""
    w = gaussian_weights(sigma)
    r = (len(w) - 1) // 2
    out = np.zeros_like(mag)
    for a, wm in enumerate(w):                      # along kx
        out += wm * np.roll(mag, a - r, axis=1)
    out2 = np.zeros_like(mag)
    for a, wm in enumerate(w):                      # along ky
        out2 += wm * np.roll(out, a - r, axis=0)
    return out2


def radial_mean(smooth, kmax):
    """(B.1) on a square index lattice: for every key = kx^2 + ky^2 <= kmax^2 that occurs (signed DFT indices),
    the mean of `smooth` over the points with that key and their number.  Returns (keys, means, counts), keys ascending."""
    ny, nx = smooth.shape
    kx = np.fft.fftfreq(nx, 1.0 / nx).round().astype(np.int64)
    ky = np.fft.fftfreq(ny, 1.0 / ny).round().astype(np.int64)
    key = ky[:, None] ** 2 + kx[None, :] ** 2
    sums, counts = {}, {}
    for j in range(ny):
        for i in range(nx):
            k = int(key[j, i])
            if k <= kmax * kmax:
                sums[k] = sums.get(k, 0.0) + float(smooth[j, i])
                counts[k] = counts.get(k, 0) + 1
    keys = np.array(sorted(sums), dtype=np.int64)
    return keys, np.array([sums[k] / counts[k] for k in keys]), np.array([counts[k] for k in keys], dtype=np.int64)


def radial_spectrum(h, H0, sigma, kmax, L):
    """steps 1-4; returns (q_r, mean magnitude, N_k) with q_r = 2 pi sqrt(key) / L"""
    keys, means, counts = radial_mean(gaussian_filter(magnitude(h, H0), sigma), kmax)
    return 2.0 * np.pi * np.sqrt(keys.astype(np.float64)) / L, means, counts


# ---------------------------------------------------------------------------------------------------------------
# Steps five and six of Appendix B and the extraction of the maxima, in the
# paper's order.  Readings (R24): the knots q_k are placed so that "each interval contains 10 points":
# q_0 = 0 and q_k = the q of the (10 k)-th point in ascending order, the last interval takes what is left; points
# with q = 0 are left out (a_0 = 0 fixes the function there); the 400 grid points span [0, q_K]; at the ends of
# the grid the moving average runs over the part of its window that exists; the derivative uses central second-order
# differences (one-sided second-order at the two ends), its roots are located by sign change and linear
# interpolation, and a root is a maximum if the second difference there is negative.
# ---------------------------------------------------------------------------------------------------------------
def knots(q, per_interval=10):
    q = np.asarray(q, dtype=np.float64)
    ks = [0.0] + [float(q[i]) for i in range(per_interval - 1, len(q), per_interval)]
    if ks[-1] < q[-1]:
        ks.append(float(q[-1]))
    return np.array(ks)


def piecewise_linear_fit(q, z, per_interval=10):
    """(B.2): least-squares continuous piecewise-linear function with a_0 = 0 on the knots above.
    Returns (knots, nodal values a_0 .. a_K): the K free parameters are a_1 .. a_K (a_K = a_{K-1} + b_{K-1})."""
    q = np.asarray(q, dtype=np.float64)
    z = np.asarray(z, dtype=np.float64)
    ks = knots(q, per_interval)
    K = len(ks) - 1
    # design matrix of the hat functions of knots 1..K (dense: this is the definition, not an efficient solver)
    A = np.zeros((len(q), K))
    for i, qi in enumerate(q):
        k = min(max(int(np.searchsorted(ks, qi, side="left")) - 1, 0), K - 1)   # interval [q_k, q_{k+1}] containing q_i
        s = (qi - ks[k]) / (ks[k + 1] - ks[k])
        if k >= 1:
            A[i, k - 1] += 1.0 - s
        A[i, k] += s
    a, *_ = np.linalg.lstsq(A, z, rcond=None)
    return ks, np.concatenate([[0.0], a])


def evaluate(ks, a, x):
    return np.interp(x, ks, a)


def moving_average(f, P):
    """(B.3) with the window cut off at the ends of the grid"""
    n = len(f)
    out = np.empty(n)
    for k in range(n):
        lo, hi = max(0, k - P), min(n - 1, k + P)
        out[k] = np.sum(f[lo:hi + 1]) / (hi - lo + 1)
    return out


def smooth_and_peaks(q, z, per_interval=10, ngrid=400):
    """steps 5-6 and the maxima: returns (grid, smoothed values, [(q_peak, value), ...])"""
    sel = np.asarray(q) > 0
    q, z = np.asarray(q)[sel], np.asarray(z)[sel]
    ks, a = piecewise_linear_fit(q, z, per_interval)
    x = np.linspace(0.0, ks[-1], ngrid)
    f = evaluate(ks, a, x)
    for P in (3, 2, 1):
        f = moving_average(f, P)
    d = x[1] - x[0]
    df = np.empty(ngrid)
    df[1:-1] = (f[2:] - f[:-2]) / (2 * d)
    df[0] = (-3 * f[0] + 4 * f[1] - f[2]) / (2 * d)
    df[-1] = (3 * f[-1] - 4 * f[-2] + f[-3]) / (2 * d)
    peaks = []
    for k in range(ngrid - 1):
        if df[k] > 0 and df[k + 1] <= 0:
            t = df[k] / (df[k] - df[k + 1])
            c = k if t < 0.5 else k + 1
            c = min(max(c, 1), ngrid - 2)
            if f[c + 1] - 2 * f[c] + f[c - 1] < 0:
                peaks.append((x[k] + t * d, f[k] + t * (f[k + 1] - f[k])))
    return x, f, peaks

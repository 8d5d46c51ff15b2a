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
Steps five and six of the appendix (least-squares fit, moving average, maxima) are 1-D post-processing of this output
and are not part of the build.
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

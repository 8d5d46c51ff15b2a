"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no fluxes, Jacobians, solvers): it only
draws numbers.  Both the CUDA path and the CPU oracle are fed the arrays made here.

The paper uses no dataset: every run starts from a synthetic initial condition
(PAPER.md:324-328 (3.1), 463-474 (4.7)-(4.8) small global noise, 506-516 (4.9)-(4.10) and
584-593 (4.11)-(4.12) Gaussian local perturbations) on large square grids (1000-4000 per side,
PAPER.md:453).  The configs below are BASELINE.json's five configs made concrete
(SURVEY.md section 8(d)); recipe restated in DESIGN.md "Input recipe".
"""
import math

import numpy as np

# most unstable wavelength for h0 = 1, kappa = 100, h* = 0.1, (n,m) = (3,2): Pi'(1) = 1.7,
# q_m^2 = Pi'/2 (PAPER.md:72 (1.5) with f0 = f1/Pi' = h0^3)  ->  lambda_m = 2 pi / sqrt(0.85)
LAMBDA_M = 2.0 * math.pi / math.sqrt(0.85)

MODEL = dict(kappa=100.0, hstar=0.1, n=3, m=2)

CONFIGS = {
    0: dict(name="cfg0_128", nx=128, ny=128, dx=8 * LAMBDA_M / 128, ic="noise", seed=0, dt=1e-2, steps=100,
            tol=1e-10, max_iter=64),
    1: dict(name="cfg1_1024", nx=1024, ny=1024, dx=64 * LAMBDA_M / 1024, ic="noise", seed=1, dt=1e-2, steps=2000,
            tol=1e-10, max_iter=64),
    2: dict(name="cfg2_4096_adaptive", nx=4096, ny=4096, dx=0.43, ic="gauss", seed=2, dt=1e-3, steps=200,
            tol=1e-10, max_iter=10, dt_max=0.1, dt_min=1e-12, grow=1.1, shrink=0.5),
    3: dict(name="cfg3_8192", nx=8192, ny=8192, dx=64 * LAMBDA_M / 1024, ic="noise", seed=3, dt=1e-2, steps=50,
            warmup=5, tol=1e-10, max_iter=64),
    4: dict(name="cfg4_penta_16384", nrow=16384, ncol=16384, seed=4),
}


def config(k):
    c = dict(CONFIGS[k])
    if "dx" in c:
        c["dy"] = c["dx"]
    c.update(MODEL)
    return c


def noise_ic(nx, ny, seed, h0=1.0, amp=0.01):
    """h0 + amp*U[-1,1] i.i.d. per cell (BASELINE.json configs 0, 1, 3).  Returns [ny][nx] float64."""
    rng = np.random.default_rng(seed)
    return h0 + amp * rng.uniform(-1.0, 1.0, size=(ny, nx))


def gauss_ic(nx, ny, dx, dy, seed, h0=0.12, depth=0.05, width=2.0, count=16, min_sep=12.0):
    """Uniform film h0 minus `count` Gaussian depressions at seeded uniform-random centres, re-drawn until
    pairwise >= min_sep apart so that h >= h0 - depth > 0 (BASELINE.json config 2)."""
    rng = np.random.default_rng(seed)
    Lx, Ly = nx * dx, ny * dy
    centres = []
    while len(centres) < count:
        c = (rng.uniform(0, Lx), rng.uniform(0, Ly))
        if all(math.hypot(c[0] - o[0], c[1] - o[1]) >= min_sep for o in centres):
            centres.append(c)
    x = (np.arange(nx) + 0.5) * dx
    y = (np.arange(ny) + 0.5) * dy
    h = np.full((ny, nx), h0)
    R = 8.0 * width                      # the bump is < 1e-14 beyond 8 widths
    for cx, cy in centres:
        i0, i1 = max(0, int((cx - R) / dx)), min(nx, int((cx + R) / dx) + 2)
        j0, j1 = max(0, int((cy - R) / dy)), min(ny, int((cy + R) / dy) + 2)
        r2 = (x[None, i0:i1] - cx) ** 2 + (y[j0:j1, None] - cy) ** 2
        h[j0:j1, i0:i1] -= depth * np.exp(-r2 / (2.0 * width * width))
    return h


def initial_condition(cfg, nx=None, ny=None):
    """Initial film for a config dict; nx, ny may be overridden to get a small case of the same recipe."""
    nx = nx or cfg["nx"]
    ny = ny or cfg["ny"]
    if cfg["ic"] == "noise":
        return noise_ic(nx, ny, cfg["seed"])
    if cfg["ic"] == "gauss":
        return gauss_ic(nx, ny, cfg["dx"], cfg["dy"], cfg["seed"])
    raise ValueError(cfg["ic"])


def cosine_ic(nx, ny, dx, dy, kx=0, ky=0, h0=1.0, eps=0.1):
    """h0(1 + eps cos(kx pi x/Lx) + eps cos(ky pi y/Ly)): admissible no-flux modes, cf. PAPER.md:326 (3.1)."""
    x = (np.arange(nx) + 0.5) * dx
    y = (np.arange(ny) + 0.5) * dy
    h = np.full((ny, nx), 1.0)
    if kx:
        h = h + eps * np.cos(kx * math.pi * x / (nx * dx))[None, :]
    if ky:
        h = h + eps * np.cos(ky * math.pi * y / (ny * dy))[:, None]
    return h0 * h


def penta_system(nrow, ncol, seed, rows=None):
    """BASELINE.json config 4: bands e,c,a,b ~ U[-1,1], d = 1 + |e|+|c|+|a|+|b| + U[0,1] (strictly diagonally
    dominant), rhs ~ U[-1,1]; six [nrow][ncol] arrays.  Generated row by row from per-row child seeds so that a
    subset of rows (`rows`) can be drawn without materialising the rest."""
    rows = range(nrow) if rows is None else rows
    out = [np.empty((len(rows), ncol)) for _ in range(6)]
    for k, r in enumerate(rows):
        rng = np.random.default_rng([seed, r])
        e, c, a, b = (rng.uniform(-1.0, 1.0, ncol) for _ in range(4))
        d = 1.0 + np.abs(e) + np.abs(c) + np.abs(a) + np.abs(b) + rng.uniform(0.0, 1.0, ncol)
        rhs = rng.uniform(-1.0, 1.0, ncol)
        for arr, v in zip(out, (e, c, d, a, b, rhs)):
            arr[k] = v
    return out  # e, c, d, a, b, rhs


def penta_system_bending(nsys, n, seed, sigma):
    """Weakly dominant test systems for the partition variant of the isolated solver: A = diag(1 + U[0,1]) +
    sigma * D2^T diag(w) D2 with D2 the interior second differences of a line of n points and w ~ U[0.5, 1.5]
    (symmetric positive definite, the structure of I + s J of the sweeps with f0 = w; couples rows over
    ~ sigma^(1/4) neighbours, unlike the strictly dominant config-4 systems whose coupling dies within a few rows).
    Six [nsys][n] arrays e, c, d, a, b, rhs with system s = row s."""
    rng = np.random.default_rng([seed, 77])
    w = rng.uniform(0.5, 1.5, (nsys, n))
    w[:, 0] = 0.0
    w[:, -1] = 0.0
    wm = np.concatenate([np.zeros((nsys, 1)), w[:, :-1]], axis=1)      # w_{i-1}
    wp = np.concatenate([w[:, 1:], np.zeros((nsys, 1))], axis=1)       # w_{i+1}
    e = sigma * wm
    b = sigma * wp
    c = -2.0 * sigma * (wm + w)
    a = -2.0 * sigma * (w + wp)
    d = 1.0 + rng.uniform(0.0, 1.0, (nsys, n)) + sigma * (wm + 4.0 * w + wp)
    rhs = rng.uniform(-1.0, 1.0, (nsys, n))
    return [np.ascontiguousarray(t) for t in (e, c, d, a, b, rhs)]

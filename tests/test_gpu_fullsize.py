"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (tf.ThinFilm on the
current stream, 8192 x 8192, config 3 recipe).

The oracle cannot advance 6.7e7 points in seconds, so sampled outputs are computed one window at a time:
the oracle advances a W x W cut of the same initial film and the values at least MARGIN cells away from the
artificial cut edges are compared.  Those values ARE the full-domain oracle's to the last bit: a line solve
of I + sJ couples distant points through a Green's function that decays faster than 0.3^distance, so after a
few iterations nothing of a cut 96 cells away survives in fp64 (pinned on the oracle alone, without the GPU,
in tests/test_window_locality.py).  Windows sit at the four corners (true boundaries on two sides), across
the split rows/columns of the two-sided sweeps, and at strip/tile seams.
Beyond samples: invariants that hold at any size (mass, Newton count of the oracle's cut, residual of the
converged step evaluated with the oracle's full operator on a band of rows).
"""
import numpy as np
import pytest

from paper_1806_10550_b200 import inputs

pytestmark = pytest.mark.gpu

W, MARGIN = 320, 96


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


@pytest.fixture(scope="module")
def film8192(tf):
    """Config 3: the 8192^2 film, one step of 3 fixed iterations on the GPU (initial and advanced fields)."""
    cfg = inputs.config(3)
    h = inputs.initial_condition(cfg)
    g = tf.ThinFilm(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
    g.set_newton(cfg["tol"], cfg["max_iter"], 3)
    g.set_state(h)
    m0 = g.mass()
    st, it, res = g.step(cfg["dt"])
    assert (st, it) == (0, 3)
    u = g.get_state()
    m1 = g.mass()
    g.close()
    return cfg, h, u, res, m0, m1


def window_origins(n):
    mid = (n // 2) // 16 * 16                       # split row/column of the two-sided sweeps
    return sorted({0, n - W, mid - W // 2, 28 * 100 - W // 2, mid - W + MARGIN + 2, mid - MARGIN - 2})


def test_config3_8192_sampled_windows_match_oracle(film8192, tfo):
    cfg, h, u, res, m0, m1 = film8192
    n = cfg["nx"]
    origins = window_origins(n)
    picks = [(origins[0], origins[0]), (origins[0], origins[-1]), (origins[-1], origins[0]), (origins[-1], origins[-1]),
             (n // 2 // 16 * 16 - W // 2, n // 2 // 16 * 16 - W // 2), (origins[2], origins[1]), (origins[1], origins[3]),
             (origins[3], origins[4])]
    worst = 0.0
    o = tfo.ThinFilmOracle(W, W, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
    o.set_newton(cfg["tol"], cfg["max_iter"], 3)
    for (j0, i0) in picks:
        o.set_state(np.ascontiguousarray(h[j0:j0 + W, i0:i0 + W]))
        st, it, _ = o.step(cfg["dt"])
        assert (st, it) == (0, 3)
        uo = o.get_state()
        # keep away from the artificial cut edges only: an edge that is a true boundary of the film is kept
        ja = 0 if j0 == 0 else MARGIN
        jb = W if j0 + W == n else W - MARGIN
        ia = 0 if i0 == 0 else MARGIN
        ib = W if i0 + W == n else W - MARGIN
        d = np.max(np.abs(u[j0 + ja:j0 + jb, i0 + ia:i0 + ib] - uo[ja:jb, ia:ib])) / np.max(np.abs(uo))
        worst = max(worst, d)
        assert d <= 1e-11, (j0, i0, d)
    assert np.max(np.abs(u - h)) > 1e-5             # the step moved the film
    print(f"8192^2, 8 windows of {W}^2: worst rel Linf {worst:.2e}")


def test_config3_8192_mass_is_conserved(film8192):
    cfg, h, u, res, m0, m1 = film8192
    ref = float(np.sum(h, dtype=np.float64)) * cfg["dx"] * cfg["dy"]
    assert abs(m0 - ref) <= 1e-13 * ref             # tf_mass against numpy's pairwise sum
    assert abs(m1 - m0) <= 1e-13 * m0               # every Newton iterate conserves mass (column sums of J are 0)
    assert np.all(np.isfinite(u)) and u.min() > 0.0


def test_config3_8192_converged_step_solves_the_full_scheme(tf, tfo):
    """tol-converged step: Newton count equals the oracle's on a cut of the same film (the count is a property
    of the spectrum, not of the size), and G(u^{n+1}) = (I + sD)u^{n+1} - (I - sD)u^n, evaluated with the
    ORACLE's full operator on bands of rows, is at rounding level relative to the update."""
    cfg = inputs.config(3)
    n = cfg["nx"]
    h = inputs.initial_condition(cfg)
    g = tf.ThinFilm(n, n, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
    g.set_newton(cfg["tol"], cfg["max_iter"], 0)
    g.set_state(h)
    st, it, res = g.step(cfg["dt"])
    u = g.get_state()
    g.close()
    assert st == 0 and res < cfg["tol"]
    oc = tfo.ThinFilmOracle(512, 512, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"], omp=True)
    oc.set_newton(cfg["tol"], cfg["max_iter"], 0)
    oc.set_state(np.ascontiguousarray(h[:512, :512]))
    so, io, _ = oc.step(cfg["dt"])
    assert so == 0 and abs(it - io) <= 1, (it, io)
    # residual on three bands of 64 full rows (top boundary, the split, bottom boundary); D of a band needs
    # 2 more rows on each open side, so evaluate on band +- 8 rows and keep the inner rows
    s = 0.5 * cfg["dt"]
    mid = (n // 2) // 16 * 16
    for r0 in (0, mid - 32, n - 64):
        a, b = max(0, r0 - 8), min(n, r0 + 64 + 8)
        ob = tfo.ThinFilmOracle(n, b - a, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"], omp=True)
        D1 = ob.operator_D(np.ascontiguousarray(u[a:b]))
        D0 = ob.operator_D(np.ascontiguousarray(h[a:b]))
        G = (u[a:b] + s * D1) - (h[a:b] - s * D0)
        ka = 0 if a == 0 else 8
        kb = (b - a) if b == n else (b - a) - 8
        gmax = np.max(np.abs(G[ka:kb]))
        assert gmax <= 20 * cfg["tol"] * np.max(np.abs(u)), (r0, gmax)


# ------------------------------------------------------------------ config 1, 100 steps
def test_config1_100_steps_parity(tf, tfo):
    cfg = inputs.config(1)
    h = inputs.initial_condition(cfg)
    g = tf.ThinFilm(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
    o = tfo.ThinFilmOracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"],
                           omp=True)
    for s in (g, o):
        s.set_newton(cfg["tol"], cfg["max_iter"], 4)
        s.set_state(h)
    for _ in range(100):
        assert g.step(cfg["dt"])[0] == 0
        assert o.step(cfg["dt"])[0] == 0
    ug, uo = g.get_state(), o.get_state()
    assert np.max(np.abs(ug - uo)) / np.max(np.abs(uo)) <= 1e-8
    assert abs(g.mass() - o.mass()) <= 1e-13 * o.mass()


# ------------------------------------------------------------------ config 4 at full system length
@pytest.mark.parametrize("direction", [0, 1])
def test_penta_solve_full_length_systems(tf, tfo, direction):
    """16384 unknowns per system (config 4's length), 256 systems: every system against the oracle and by
    backward error."""
    import torch
    length, nsys = 16384, 256
    rows = inputs.penta_system(nsys, length, seed=4)              # [nsys][length], systems along rows
    arrs = rows if direction == 0 else [np.ascontiguousarray(t.T) for t in rows]
    ref = tfo.penta_solve(direction, *arrs, omp=True)
    x = tf.penta_solve(direction, *[torch.from_numpy(a).cuda() for a in arrs])
    torch.cuda.synchronize()
    x = x.cpu().numpy()
    assert np.max(np.abs(x - ref)) / np.max(np.abs(ref)) <= 1e-12
    e, c, d, a, b, y = rows
    xs = x if direction == 0 else x.T
    Ax = d * xs
    Ax[:, 1:] += c[:, 1:] * xs[:, :-1]
    Ax[:, 2:] += e[:, 2:] * xs[:, :-2]
    Ax[:, :-1] += a[:, :-1] * xs[:, 1:]
    Ax[:, :-2] += b[:, :-2] * xs[:, 2:]
    normA = np.max(np.abs(e) + np.abs(c) + np.abs(d) + np.abs(a) + np.abs(b))
    assert np.max(np.abs(Ax - y)) / (normA * np.max(np.abs(xs)) + np.max(np.abs(y))) <= 1e-14


@pytest.mark.parametrize("direction", [1, 0])
def test_penta_solve_config4_as_timed_16384_systems(tf, tfo, direction):
    """BASELINE.json config 4 as bench.py times it: ALL 16384 systems of 16384 unknowns in one tf_penta_solve per
    direction (512 x 2 CTAs of the two-sided forward kernel, more than are resident at once), solver of App. A.2,
    PAPER.md:729-738.  The 2 GiB arrays are drawn on the device by bench.py's recipe (the bands U[-1,1], strictly
    dominant diagonal); 256 evenly spaced systems are overwritten by inputs.penta_system(rows=...), which the host can
    reproduce row by row, and compared with the oracle (<= 1e-12); EVERY system is checked by its backward error
    ||Ax - y||_inf / (||A||_inf ||x||_inf + ||y||_inf) <= 1e-14, evaluated with torch on the device (no oracle needed)."""
    import torch
    n = inputs.config(4)["nrow"]
    assert n == 16384 and inputs.config(4)["ncol"] == n
    gen = torch.Generator(device="cuda").manual_seed(inputs.config(4)["seed"] + direction)
    U = lambda lo, hi: torch.rand(n, n, dtype=torch.float64, device="cuda", generator=gen) * (hi - lo) + lo
    e, c, a, b, y = U(-1, 1), U(-1, 1), U(-1, 1), U(-1, 1), U(-1, 1)
    d = 1 + e.abs() + c.abs() + a.abs() + b.abs() + U(0, 1)
    sample = list(range(31, n, 64))                                # 256 systems, among them strip seams and both halves
    rows = inputs.penta_system(n, n, seed=40 + direction, rows=sample)
    idx = torch.tensor(sample, device="cuda")
    for dev, host in zip((e, c, d, a, b, y), rows):
        t = torch.from_numpy(host).cuda()
        if direction == 0:
            dev[idx, :] = t                                        # system s = row s
        else:
            dev[:, idx] = t.T                                      # system s = column s
    ws = torch.empty(tf.lib().tf_penta_workspace_bytes(n, n), dtype=torch.uint8, device="cuda")
    x = torch.full_like(e, float("nan"))
    tf.penta_solve(direction, e, c, d, a, b, y, out=x, workspace=ws)
    torch.cuda.synchronize()
    del ws
    assert bool(torch.isfinite(x).all())
    # sampled systems against the oracle
    ref = tfo.penta_solve(0, *rows, omp=True)
    got = (x[idx, :] if direction == 0 else x[:, idx].T).cpu().numpy()
    assert np.max(np.abs(got - ref)) / np.max(np.abs(ref)) <= 1e-12
    # every system by backward error; `ax` = the dimension a system runs along
    ax = 1 if direction == 0 else 0
    L = lambda t, lo, hi: t.narrow(ax, lo, hi - lo)
    r = d * x
    L(r, 1, n).add_(L(c, 1, n) * L(x, 0, n - 1))
    L(r, 2, n).add_(L(e, 2, n) * L(x, 0, n - 2))
    L(r, 0, n - 1).add_(L(a, 0, n - 1) * L(x, 1, n))
    L(r, 0, n - 2).add_(L(b, 0, n - 2) * L(x, 2, n))
    r.sub_(y)
    res = r.abs().amax(dim=ax)                                     # per system
    del r
    normA = (e.abs() + c.abs() + d.abs() + a.abs() + b.abs()).amax(dim=ax)
    berr = res / (normA * x.abs().amax(dim=ax) + y.abs().amax(dim=ax))
    assert berr.numel() == n
    assert float(berr.max()) <= 1e-14, (int(berr.argmax()), float(berr.max()))
    del e, c, d, a, b, y, x
    torch.cuda.empty_cache()


# ------------------------------------------------------------------ config 2 at full size: adaptive controller
def test_config2_4096_adaptive_run(tf, tfo):
    """Config 2 (4096^2, uniform 0.12 film with 16 Gaussian depressions, adaptive dt from 1e-3): the controller of
    Fig. 1 on the GPU path.  Physics of these parameters: Pi'(0.12) < 0, the depressions
    heal, no step is rejected and dt climbs to its cap.  Checked: the accept sequence, dt growth, mass, healing;
    and the field after three accepted steps (fixed iteration count) on sampled windows against the oracle."""
    cfg = inputs.config(2)
    n = cfg["nx"]
    h = inputs.initial_condition(cfg)
    assert h.min() > 0.06 and abs(h.max() - 0.12) < 1e-12
    g = tf.ThinFilm(n, n, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
    # (a) sampled parity of the first three steps, dt = 1e-3 * 1.1^k, 5 fixed iterations each
    g.set_newton(cfg["tol"], cfg["max_iter"], 5)
    g.set_state(h)
    dts = [cfg["dt"] * cfg["grow"] ** k for k in range(3)]
    for dt in dts:
        assert g.step(dt)[0] == 0
    u3 = g.get_state()
    jc, ic = np.unravel_index(np.argmin(h), h.shape)            # the deepest depression
    o = tfo.ThinFilmOracle(W, W, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
    o.set_newton(cfg["tol"], cfg["max_iter"], 5)
    for (j0, i0) in ((0, 0), (n - W, n - W), (min(max(jc - W // 2, 0), n - W), min(max(ic - W // 2, 0), n - W))):
        o.set_state(np.ascontiguousarray(h[j0:j0 + W, i0:i0 + W]))
        for dt in dts:
            assert o.step(dt)[0] == 0
        uo = o.get_state()
        ja, jb = (0 if j0 == 0 else MARGIN), (W if j0 + W == n else W - MARGIN)
        ia, ib = (0 if i0 == 0 else MARGIN), (W if i0 + W == n else W - MARGIN)
        d = np.max(np.abs(u3[j0 + ja:j0 + jb, i0 + ia:i0 + ib] - uo[ja:jb, ia:ib])) / np.max(np.abs(uo))
        assert d <= 1e-11, (j0, i0, d)
    # (b) the adaptive run itself: 60 accepted steps from the initial film
    g.set_newton(cfg["tol"], cfg["max_iter"], 0)
    g.set_state(h)
    m0 = g.mass()
    t, dt_next, hist = tf.advance_adaptive(g, cfg["dt"], 60, cfg["grow"], cfg["shrink"], cfg["dt_max"], cfg["dt_min"])
    assert all(st == 0 for _, st, _, _ in hist) and len(hist) == 60          # nothing rejected
    assert all(it <= cfg["max_iter"] and res < cfg["tol"] for _, _, it, res in hist)
    assert abs(hist[1][0] / hist[0][0] - cfg["grow"]) < 1e-12 and dt_next == cfg["dt_max"]   # 1e-3 * 1.1^49 > 0.1
    assert abs(t - sum(x[0] for x in hist)) < 1e-12
    u = g.get_state()
    assert abs(g.mass() - m0) <= 1e-13 * m0
    assert u.min() > h.min() and u.max() <= 0.12 + 1e-9                     # the depressions heal
    g.close()


# ------------------------------------------------------------------ large non-square grids (ragged strips, tiles, splits)
@pytest.mark.parametrize("nx,ny", [(12010, 3002), (2050, 9998), (16384, 4100)])
def test_large_nonsquare_grids_sampled(tf, tfo, nx, ny):
    """Grid sides that are multiples of neither 28 (strips), 16 (tiles) nor 32 (blocks); more strips than SMs in one
    direction and fewer in the other (both CTA layouts of the forward kernels); dx != dy."""
    cfg = inputs.config(3)
    dx, dy = cfg["dx"], 1.07 * cfg["dx"]
    h = inputs.noise_ic(nx, ny, seed=nx + ny)
    g = tf.ThinFilm(nx, ny, dx, dy)
    g.set_newton(1e-10, 64, 3)
    g.set_state(h)
    m0 = g.mass()
    assert g.step(cfg["dt"])[:2] == (0, 3)
    u = g.get_state()
    assert abs(g.mass() - m0) <= 1e-13 * m0
    g.close()
    midx, midy = (nx // 2) // 16 * 16, (ny // 2) // 16 * 16
    o = tfo.ThinFilmOracle(W, W, dx, dy)
    o.set_newton(1e-10, 64, 3)
    for (j0, i0) in ((0, 0), (ny - W, nx - W), (midy - W // 2, midx - W // 2), (0, nx - W), (midy - W // 2, 0)):
        o.set_state(np.ascontiguousarray(h[j0:j0 + W, i0:i0 + W]))
        assert o.step(cfg["dt"])[:2] == (0, 3)
        uo = o.get_state()
        ja, jb = (0 if j0 == 0 else MARGIN), (W if j0 + W == ny else W - MARGIN)
        ia, ib = (0 if i0 == 0 else MARGIN), (W if i0 + W == nx else W - MARGIN)
        d = np.max(np.abs(u[j0 + ja:j0 + jb, i0 + ia:i0 + ib] - uo[ja:jb, ia:ib])) / np.max(np.abs(uo))
        assert d <= 1e-11, (nx, ny, j0, i0, d)


# ------------------------------------------------------------------ fields beyond 4 GiB (element offsets up to ~6e8)
def test_field_larger_than_4GiB_sampled(tf, tfo):
    """30000 x 20000: 4.8 GB per field, 38 GB of workspace -- byte offsets beyond 2^32 in every kernel, 1072 strips and
    715 row blocks (four teams per CTA in both forward kernels), dx != dy.  One step of two fixed iterations; sampled
    windows against the oracle (corners, the split rows / columns, far ends of the arrays), mass to 1e-13."""
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < 60e9:
        pytest.skip("needs ~45 GB of device memory")
    nx, ny = 30000, 20000
    cfg = inputs.config(3)
    dx, dy = cfg["dx"], 1.03 * cfg["dx"]
    h = inputs.noise_ic(nx, ny, seed=31)
    g = tf.ThinFilm(nx, ny, dx, dy)
    g.set_newton(1e-10, 64, 2)
    g.set_state(h)
    m0 = g.mass()
    ref = float(np.sum(h, dtype=np.float64)) * dx * dy
    assert abs(m0 - ref) <= 1e-13 * ref
    assert g.step(cfg["dt"])[:2] == (0, 2)
    m1 = g.mass()
    assert abs(m1 - m0) <= 1e-13 * m0
    u = g.get_state()
    g.close()
    midx, midy = (nx // 2) // 16 * 16, (ny // 2) // 16 * 16
    o = tfo.ThinFilmOracle(W, W, dx, dy)
    o.set_newton(1e-10, 64, 2)
    for (j0, i0) in ((0, 0), (ny - W, nx - W), (midy - W // 2, midx - W // 2), (ny - W, 0), (0, nx - W), (ny - W, midx - W // 2)):
        o.set_state(np.ascontiguousarray(h[j0:j0 + W, i0:i0 + W]))
        assert o.step(cfg["dt"])[:2] == (0, 2)
        uo = o.get_state()
        ja, jb = (0 if j0 == 0 else MARGIN), (W if j0 + W == ny else W - MARGIN)
        ia, ib = (0 if i0 == 0 else MARGIN), (W if i0 + W == nx else W - MARGIN)
        d = np.max(np.abs(u[j0 + ja:j0 + jb, i0 + ia:i0 + ib] - uo[ja:jb, ia:ib])) / np.max(np.abs(uo))
        assert d <= 1e-11, (j0, i0, d)

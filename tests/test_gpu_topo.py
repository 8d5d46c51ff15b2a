"""GPU parity of tf_betti (Betti numbers of the thresholded film) against the flood-fill oracle
(oracle/topo.c): integers, so the comparison is exact.  Random images are the hard case for the union-find (components
of every size, corner contacts everywhere); the checkerboard is all corner contacts; smooth films are what the paper
slices."""
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


@pytest.fixture(scope="module")
def topo():
    from oracle import topo as t
    t.build()
    return t


def both(tf, topo, h, thr):
    import torch
    g0, g1 = tf.betti(torch.from_numpy(np.ascontiguousarray(h)).cuda(), thr)
    o0, o1 = topo.betti(h, thr)
    return (g0.tolist(), g1.tolist()), (o0.tolist(), o1.tolist())


@pytest.mark.parametrize("ny,nx", [(1, 1), (1, 40), (40, 1), (5, 5), (33, 31), (64, 64), (70, 257), (257, 70), (300, 513),
                                   (129, 1000)])
def test_random_images_all_fills(tf, topo, ny, nx):
    rng = np.random.default_rng(ny * 1000 + nx)
    h = rng.uniform(0.0, 1.0, (ny, nx))
    thr = [-0.1, 0.05, 0.2, 0.35, 0.4, 0.45, 0.5, 0.55, 0.6, 0.65, 0.8, 0.95, 1.1]   # through both percolation thresholds
    g, o = both(tf, topo, h, thr)
    assert g == o


def test_corner_contacts_and_shapes(tf, topo):
    chk = (np.indices((67, 130)).sum(axis=0) % 2).astype(float)
    g, o = both(tf, topo, chk, [0.5])
    assert g == o and g[0] == [1]
    y, x = np.mgrid[0:200, 0:300]
    ring = (((y - 100) ** 2 + (x - 150) ** 2 <= 80 ** 2) & ((y - 100) ** 2 + (x - 150) ** 2 >= 40 ** 2)).astype(float)
    g, o = both(tf, topo, ring + ((y - 100) ** 2 + (x - 150) ** 2 <= 10 ** 2), [0.5])
    assert g == o == ([2], [1])
    diag = np.eye(96)                                                       # a staircase held together by corners only
    g, o = both(tf, topo, diag, [0.5])
    assert g == o and g[0] == [1]
    spiral = np.zeros((64, 64))                                             # long thin component: deep union-find trees
    j, i, dj, di, steps = 0, 0, 0, 1, 63
    while steps > 0:
        for _ in range(steps):
            spiral[j, i] = 1.0
            j, i = j + dj, i + di
        dj, di = di, -dj
        steps -= 2
    g, o = both(tf, topo, spiral, [0.5])
    assert g == o and g[0] == [1]


def test_smooth_film_many_thresholds(tf, topo):
    n, k = 480, 6
    y, x = np.mgrid[0:n, 0:n] * (2 * np.pi * k / n)
    rng = np.random.default_rng(3)
    h = 1.0 + 0.5 * np.cos(x) * np.cos(y) + 0.05 * rng.uniform(-1, 1, (n, n))
    thr = np.linspace(0.4, 1.6, 25)
    g, o = both(tf, topo, h, thr)
    assert g == o
    assert max(g[0]) >= ((2 * k + 1) ** 2 + 1) // 2 and max(g[1]) >= 2 * k * (k - 1)     # the drop / hole pattern is seen


def test_film_after_time_steps(tf, topo):
    """slices of an actual solution of the path: config-0 film after 20 steps"""
    cfg = inputs.config(0)
    g = tf.ThinFilm(128, 128, cfg["dx"], cfg["dy"])
    g.set_newton(1e-10, 64, 0)
    g.set_state(inputs.noise_ic(128, 128, seed=0))
    for _ in range(20):
        assert g.step(cfg["dt"])[0] == 0
    h = g.get_state()
    thr = np.quantile(h, [0.02, 0.25, 0.5, 0.75, 0.98])
    a, b = both(tf, topo, h, thr)
    assert a == b


def test_full_size_8192(tf, topo):
    """config 3's grid: the labelling of 6.7e7 cells (random image at the fill where components of all sizes exist)"""
    import time
    import torch
    n = 8192
    rng = np.random.default_rng(8)
    h = rng.uniform(0.0, 1.0, (n, n))
    d = torch.from_numpy(h).cuda()
    thr = [0.41, 0.5, 0.6]
    ws = torch.empty(tf.lib().tf_betti_workspace_bytes(n, n, len(thr)), dtype=torch.uint8, device="cuda")
    tf.betti(d, thr, workspace=ws)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    g0, g1 = tf.betti(d, thr, workspace=ws)
    dt = (time.perf_counter() - t0) / len(thr)
    o0, o1 = topo.betti(h, thr)
    print(f"tf_betti 8192^2: {dt * 1e3:.2f} ms per threshold, b0 = {g0.tolist()}, b1 = {g1.tolist()}")
    assert g0.tolist() == o0.tolist() and g1.tolist() == o1.tolist()

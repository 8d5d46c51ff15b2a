"""Pins of the Betti-number oracle (oracle/topo.c).  The oracle is a plain flood fill; it is checked
against things it shares nothing with: shapes whose Betti numbers are known by construction, scipy's
connected-component labelling (a library routine) on random images, and the Euler characteristic
b0 - b1 = V - E + F of the cubical set, counted here from the vertices, edges and faces of the pixels."""
import numpy as np
import pytest

from oracle import topo


def disc(n, cy, cx, r):
    y, x = np.mgrid[0:n, 0:n]
    return ((y - cy) ** 2 + (x - cx) ** 2 <= r * r).astype(float)


def test_shapes_with_known_betti_numbers():
    n = 64
    flat = np.zeros((n, n))
    assert [int(v[0]) for v in topo.betti(flat, 0.5)] == [0, 0]            # nothing above the plane
    assert [int(v[0]) for v in topo.betti(flat + 1.0, 0.5)] == [1, 0]      # everything above: one component, no hole
    three = disc(n, 12, 12, 6) + disc(n, 40, 20, 8) + disc(n, 30, 50, 5)
    assert [int(v[0]) for v in topo.betti(three, 0.5)] == [3, 0]           # three peaks
    ring = disc(n, 32, 32, 20) - disc(n, 32, 32, 10)
    assert [int(v[0]) for v in topo.betti(ring, 0.5)] == [1, 1]            # one ridge around one valley
    two_rings_and_a_peak = ring + disc(n, 32, 32, 4)
    assert [int(v[0]) for v in topo.betti(two_rings_and_a_peak, 0.5)] == [2, 1]
    holes = np.ones((n, n))
    for c in ((10, 10), (10, 40), (40, 10), (40, 40), (25, 25)):
        holes -= disc(n, c[0], c[1], 4)
    assert [int(v[0]) for v in topo.betti(holes, 0.5)] == [1, 5]           # a film with five holes
    holes[0:30, 10] = 0.0                                                  # a channel from one hole to the border: no longer a hole
    assert [int(v[0]) for v in topo.betti(holes, 0.5)] == [1, 4]


def test_corner_contact_conventions_of_the_cubical_set():
    """closed squares touching at a corner are connected; the (open) complement is not connected through a corner"""
    a = np.zeros((6, 6))
    a[1, 1] = a[2, 2] = 1.0
    assert [int(v[0]) for v in topo.betti(a, 0.5)] == [1, 0]               # diagonal neighbours: ONE component
    b = np.zeros((7, 7))
    b[2, 3] = b[3, 2] = b[3, 4] = b[4, 3] = 1.0                            # a diamond of four pixels touching at corners
    assert [int(v[0]) for v in topo.betti(b, 0.5)] == [1, 1]               # ... encloses its centre pixel: one hole
    c = np.ones((6, 6))
    c[2, 2] = c[3, 3] = 0.0                                                # two background pixels touching at a corner
    assert [int(v[0]) for v in topo.betti(c, 0.5)] == [1, 2]               # are two holes
    chk = (np.indices((8, 8)).sum(axis=0) % 2).astype(float)               # checkerboard
    b0, b1 = topo.betti(chk, 0.5)
    assert int(b0[0]) == 1                                                 # all foreground pixels hang together by corners
    interior_bg = int(((chk == 0)[1:-1, 1:-1]).sum())
    assert int(b1[0]) == interior_bg                                       # every interior background pixel is its own hole


def test_threshold_is_strict_and_monotone_fill():
    h = np.array([[1.0, 1.0, 1.0, 1.0, 1.0], [1.0, 3.0, 1.0, 2.0, 1.0], [1.0, 1.0, 1.0, 1.0, 1.0]])
    b0, b1 = topo.betti(h, [0.5, 1.0, 1.5, 2.0, 2.5, 3.0])
    assert b0.tolist() == [1, 2, 2, 1, 1, 0] and b1.tolist() == [0] * 6    # "above H*": h > H*, not >=


def euler_characteristic(fg):
    """V - E + F of the union of the closed unit squares of the True cells, counted from the cells' own
    vertices, edges and faces (no connectivity search)."""
    ny, nx = fg.shape
    F = int(fg.sum())
    p = np.zeros((ny + 2, nx + 2), dtype=bool)
    p[1:-1, 1:-1] = fg
    # a vertical edge between columns i-1|i exists if either horizontal neighbour is foreground; same for horizontal edges
    ev = p[1:-1, :-1] | p[1:-1, 1:]
    eh = p[:-1, 1:-1] | p[1:, 1:-1]
    E = int(ev.sum() + eh.sum())
    V = int((p[:-1, :-1] | p[:-1, 1:] | p[1:, :-1] | p[1:, 1:]).sum())
    return V - E + F


@pytest.mark.parametrize("seed,shape,fill", [(0, (40, 50), 0.5), (1, (33, 17), 0.3), (2, (64, 64), 0.7), (3, (5, 90), 0.55)])
def test_against_scipy_labelling_and_euler_characteristic(seed, shape, fill):
    ndi = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(seed)
    h = rng.uniform(0.0, 1.0, shape)
    thr = 1.0 - fill
    fg = h > thr
    b0, b1 = topo.betti(h, thr)
    _, n_fg = ndi.label(fg, structure=np.ones((3, 3)))
    assert int(b0[0]) == n_fg
    lab_bg, n_bg = ndi.label(~fg, structure=[[0, 1, 0], [1, 1, 1], [0, 1, 0]])
    border = set(np.unique(np.concatenate([lab_bg[0], lab_bg[-1], lab_bg[:, 0], lab_bg[:, -1]]))) - {0}
    assert int(b1[0]) == n_bg - len(border)
    assert int(b0[0]) - int(b1[0]) == euler_characteristic(fg)


def test_smooth_film_counts_drops_and_holes():
    """a film shaped like the paper's dewetting patterns: k x k drops (sliced high) / a perforated layer (sliced low)"""
    n, k = 120, 4
    y, x = np.mgrid[0:n, 0:n] * (2 * np.pi * k / n)
    h = 1.0 + 0.5 * np.cos(x) * np.cos(y)
    b0, b1 = topo.betti(h, [1.25, 0.75])
    # cos x cos y > 0.5 around the extrema (a pi, b pi) with a + b even, a, b = 0 .. 2k (those with a or b = 0 or 2k are
    # cut by the border but still components): ((2k+1)^2 + 1)/2 of them, pairwise separated by the zero lines
    assert int(b0[0]) == ((2 * k + 1) ** 2 + 1) // 2 == 41 and int(b1[0]) == 0
    # cos x cos y < -0.5 around the extrema with a + b odd; the 16 on the border are open to it, the other 24 are holes
    assert int(b0[1]) == 1 and int(b1[1]) == ((2 * k + 1) ** 2 - 1) // 2 - 4 * k == 24
    assert int(b0[1]) - int(b1[1]) == euler_characteristic(h > 0.75)

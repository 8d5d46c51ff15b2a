"""Pins the sampling rule of tests/test_gpu_fullsize.py on the oracle alone (no GPU): values of a step computed
on a W x W cut of a film equal the full-domain values once they are MARGIN cells away from the artificial cut
edges.  Reason: each line solve of I + sJ has an exponentially decaying Green's function (the matrices are
diagonally dominant; off-diagonal/diagonal ~ 0.3 at the configs' dt, dx), so the influence of
an edge 64+ cells away is below one ulp after the few iterations of a step."""
import numpy as np

from oracle import tfo
from paper_1806_10550_b200 import inputs


def test_cut_reproduces_full_domain_away_from_cut_edges():
    cfg = inputs.config(3)
    n, W, M = 448, 256, 96
    h = inputs.noise_ic(n, n, seed=3)
    full = tfo.ThinFilmOracle(n, n, cfg["dx"], cfg["dy"], omp=True)
    full.set_newton(1e-10, 64, 3)
    full.set_state(h)
    assert full.step(cfg["dt"])[:2] == (0, 3)
    U = full.get_state()
    cut = tfo.ThinFilmOracle(W, W, cfg["dx"], cfg["dy"])
    cut.set_newton(1e-10, 64, 3)
    for (j0, i0) in ((0, 0), (n - W, 0), (96, 100), (n - W, n - W)):
        cut.set_state(np.ascontiguousarray(h[j0:j0 + W, i0:i0 + W]))
        assert cut.step(cfg["dt"])[:2] == (0, 3)
        Uc = cut.get_state()
        ja, jb = (0 if j0 == 0 else M), (W if j0 + W == n else W - M)
        ia, ib = (0 if i0 == 0 else M), (W if i0 + W == n else W - M)
        d = np.max(np.abs(Uc[ja:jb, ia:ib] - U[j0 + ja:j0 + jb, i0 + ia:i0 + ib]))
        assert d <= 4e-16, (j0, i0, d)
        # and the cut edge itself IS different (the rule is not vacuous)
        if j0 > 0:
            assert np.max(np.abs(Uc[0] - U[j0, i0:i0 + W])) > 1e-9

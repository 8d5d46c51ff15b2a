"""Test helper (no test in here): a numpy transcription of the slab / partition scheme's three phases for direction 1
([len][nsys] arrays), used as stand-in "kernels" so that the exchange logic of paper_1806_10550_b200/dist.py can run
under gloo on the CPU.  The formulas are those of csrc/tf_partition.cuh's header; the product's kernels are tested
against the oracle on the GPU (tests/test_gpu_slabs.py), this file only has to be right for the host-logic test to
mean something -- it is checked against a dense solve there."""
import numpy as np
import torch


def chunk_lo(p, P, N):
    return 0 if p <= 0 else (N if p >= P else (p * N // P) // 16 * 16)


def _march(e, c, q, a, b, y, outside):
    """LU forward elimination of one chunk (arrays in marching orientation) with the right-hand sides y and the two
    coupling columns; returns alpha, beta, z_rhs, z_far, z_near of the last and the last-but-one row"""
    a1 = b1 = a2 = b2 = 0.0
    z1, z2, hist = np.zeros(3), np.zeros(3), []
    for k in range(len(q)):
        yf = e[k] if (outside and k == 0) else 0.0
        yn = (c[k] if k == 0 else (e[k] if k == 1 else 0.0)) if outside else 0.0
        gam = c[k] - a2 * e[k]
        mu = q[k] - b2 * e[k] - a1 * gam
        al, be = (a[k] - b1 * gam) / mu, b[k] / mu
        z = (np.array([y[k], yf, yn]) - z1 * gam - z2 * e[k]) / mu
        a2, b2, z2, a1, b1, z1 = a1, b1, z1, al, be, z
        hist.append((al, be, z))
    (x1, y1, w1), (x2, y2, w2) = hist[-1], hist[-2]
    return [x1, y1, w1[0], w1[1], w1[2], x2, y2, w2[0], w2[1], w2[2]]


def interface(direction, nparts, slab, nslabs, e, c, d, a, b, rhs):
    assert direction == 1
    E, C, D, A, B, Y = [t.numpy() for t in (e, c, d, a, b, rhs)]
    n, nsys = D.shape
    Pg, out = nslabs * nparts, np.zeros((nparts, 2, 10, nsys))
    for p in range(nparts):
        lo, hi = chunk_lo(p, nparts, n), chunk_lo(p + 1, nparts, n)
        pg = slab * nparts + p
        for s in range(nsys):
            sl = slice(lo, hi)
            out[p, 0, :, s] = _march(E[sl, s], C[sl, s], D[sl, s], A[sl, s], B[sl, s], Y[sl, s], pg > 0)
            r = slice(hi - 1, lo - 1 if lo > 0 else None, -1)
            out[p, 1, :, s] = _march(B[r, s], A[r, s], D[r, s], C[r, s], E[r, s], Y[r, s], pg < Pg - 1)
    return torch.from_numpy(out)


def reduced(iface_all):
    """iface_all [Pg][2][10][nsys] -> X [Pg][4][nsys] = (t_p, b_p)"""
    Pg, _, _, nsys = iface_all.shape
    X = np.zeros((Pg, 4, nsys))
    for s in range(nsys):
        hb, cb, RC = np.zeros(2), np.zeros((2, 2)), []
        for p in range(Pg):
            d1a, d1b, d1y, d1f, d1n, d2a, d2b, d2y, d2f, d2n = iface_all[p, 0, :, s]
            u1a, u1b, u1y, u1f, u1n, u2a, u2b, u2y, u2f, u2n = iface_all[p, 1, :, s]
            first, last = p == 0, p == Pg - 1
            gt, gb = np.array([u1y, u2y - u2a * u1y]), np.array([d2y - d2a * d1y, d1y])
            Z = np.zeros((2, 2))
            Lt = Z if first else np.array([[u1b, u1a], [-u2a * u1b, u2b - u2a * u1a]])
            Lb = Z if first else np.array([[d2f - d2a * d1f, d2n - d2a * d1n], [d1f, d1n]])
            Ut = Z if last else np.array([[u1n, u1f], [u2n - u2a * u1n, u2f - u2a * u1f]])
            Ub = Z if last else np.array([[d2b - d2a * d1a, -d2a * d1b], [d1a, d1b]])
            Mi = np.linalg.inv(np.eye(2) - Lt @ cb)
            ht, ct, K = Mi @ (gt - Lt @ hb), Mi @ Ut, Lb @ cb
            hb, cb = gb - Lb @ hb + K @ ht, Ub + K @ ct
            RC.append((ht, ct, hb.copy(), cb.copy()))
        t = np.zeros(2)
        for p in range(Pg - 1, -1, -1):
            ht, ct, hbp, cbp = RC[p]
            nt, bb = ht - ct @ t, hbp - cbp @ t
            X[p, :2, s], X[p, 2:, s], t = nt, bb, nt
    return X


def solve(direction, nparts, slab, nslabs, e, c, d, a, b, rhs, iface_all):
    """reduced system, then every local chunk as a dense pentadiagonal solve with corrected right-hand sides"""
    assert direction == 1
    E, C, D, A, B, Y = [t.numpy() for t in (e, c, d, a, b, rhs)]
    n, nsys = D.shape
    Pg = nslabs * nparts
    X = reduced(iface_all.numpy())
    out = np.zeros((n, nsys))
    for p in range(nparts):
        lo, hi = chunk_lo(p, nparts, n), chunk_lo(p + 1, nparts, n)
        pg, m = slab * nparts + p, hi - lo
        for s in range(nsys):
            M = np.zeros((m, m))
            y = Y[lo:hi, s].copy()
            for k in range(m):
                j = lo + k
                M[k, k] = D[j, s]
                if k >= 1: M[k, k - 1] = C[j, s]
                if k >= 2: M[k, k - 2] = E[j, s]
                if k < m - 1: M[k, k + 1] = A[j, s]
                if k < m - 2: M[k, k + 2] = B[j, s]
            if pg > 0:
                bp0, bp1 = X[pg - 1, 2, s], X[pg - 1, 3, s]
                y[0] -= E[lo, s] * bp0 + C[lo, s] * bp1
                y[1] -= E[lo + 1, s] * bp1
            if pg < Pg - 1:
                t0, t1 = X[pg + 1, 0, s], X[pg + 1, 1, s]
                y[m - 1] -= A[hi - 1, s] * t0 + B[hi - 1, s] * t1
                y[m - 2] -= B[hi - 2, s] * t0
            out[lo:hi, s] = np.linalg.solve(M, y)
    return torch.from_numpy(out)

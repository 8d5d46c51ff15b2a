"""GPU parity of the intra-line parallel (partition) variant of the isolated pentadiagonal solver
(tf_penta_solve_ex with TF_PENTA_PARTITION) against the CPU oracle's LU
(oracle/tfo.c penta_solve, pinned against LAPACK) and by backward error, which needs no oracle.

Two input families: BASELINE.json's config-4 recipe (strictly diagonally dominant: coupling between chunks is
negligible, so these mostly test the chunk solves) and weakly dominant "bending" systems whose rows couple over
tens of rows (inputs.penta_system_bending): there a wrong interface relation or reduced solve shows at O(1e-3)."""
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
def tfo():
    from oracle import tfo as o
    o.build()
    return o


def rel_inf(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def backward_error(arrs, xs):
    """arrs, xs as [nsys][len]"""
    e, c, d, a, b, y = arrs
    Ax = d * xs
    Ax[:, 1:] += c[:, 1:] * xs[:, :-1]
    Ax[:, 2:] += e[:, 2:] * xs[:, :-2]
    Ax[:, :-1] += a[:, :-1] * xs[:, 1:]
    Ax[:, :-2] += b[:, :-2] * xs[:, 2:]
    normA = np.max(np.abs(e) + np.abs(c) + np.abs(d) + np.abs(a) + np.abs(b))
    return float(np.max(np.abs(Ax - y)) / (normA * np.max(np.abs(xs)) + np.max(np.abs(y))))


def systems(kind, nsys, n, seed):
    if kind == "cfg4":
        return inputs.penta_system(nsys, n, seed=seed)
    return inputs.penta_system_bending(nsys, n, seed, {"bend1e4": 1e4, "bend1e7": 1e7}[kind])


def solve_both(tf, tfo, arrs, direction, nparts):
    """arrs: [nsys][len]; direction 1 stores them transposed ([len][nsys], systems = columns)."""
    import torch
    lay = arrs if direction == 0 else [np.ascontiguousarray(t.T) for t in arrs]
    ref = tfo.penta_solve(direction, *lay)
    dev = [torch.from_numpy(t).cuda() for t in lay]
    x = tf.penta_solve(direction, *dev, variant=tf.PENTA_PARTITION, nparts=nparts)
    torch.cuda.synchronize()
    x = x.cpu().numpy()
    return (x, ref) if direction == 0 else (x.T, ref.T)


# forward tolerance: 1e-12 for config 4 (BASELINE.json); the bending systems have condition numbers 1e5 / 1e8, the
# oracle's own LU carries cond * eps there, so the forward comparison is loose and the backward error is the gate
TOL = {"cfg4": 1e-12, "bend1e4": 1e-9, "bend1e7": 1e-6}


@pytest.mark.parametrize("nsys,n,nparts", [(64, 512, 4), (96, 1000, 0), (34, 400, 3), (130, 2050, 7), (32, 4096, 16),
                                           (250, 998, 5), (64, 192, 2)])
@pytest.mark.parametrize("kind", ["cfg4", "bend1e4", "bend1e7"])
@pytest.mark.parametrize("direction", [0, 1])
def test_partition_parity(tf, tfo, nsys, n, nparts, kind, direction):
    nrow, ncol = (nsys, n) if direction == 0 else (n, nsys)
    P = tf.penta_partition_chunks(nrow, ncol, direction, nparts)
    assert P >= 2, "shape must exercise the partition path"
    arrs = systems(kind, nsys, n, seed=11)
    x, ref = solve_both(tf, tfo, arrs, direction, nparts)
    assert np.all(np.isfinite(x))
    assert rel_inf(x, ref) <= TOL[kind]
    assert backward_error(arrs, x) <= 2e-14


@pytest.mark.parametrize("direction", [0, 1])
def test_partition_matches_lu_variant_where_it_falls_back(tf, direction):
    """odd pitches / short systems / fewer than 32 systems: the call runs the LU variant (chunks == 1), bit for bit"""
    import torch
    for nsys, n in [(33, 400), (64, 100), (16, 4096)]:
        nrow, ncol = (nsys, n) if direction == 0 else (n, nsys)
        assert tf.penta_partition_chunks(nrow, ncol, direction, 0) == 1
        arrs = inputs.penta_system(nrow, ncol, seed=5)
        dev = [torch.from_numpy(t).cuda() for t in arrs]
        x1 = tf.penta_solve(direction, *dev, variant=tf.PENTA_PARTITION)
        x0 = tf.penta_solve(direction, *dev)
        torch.cuda.synchronize()
        assert torch.equal(x0, x1)


@pytest.mark.parametrize("direction", [0, 1])
def test_partition_full_length_few_systems(tf, tfo, direction):
    """the shape the variant is for: 256 systems of config 4's full length 16384, automatic chunk count"""
    nsys, n = 256, 16384
    nrow, ncol = (nsys, n) if direction == 0 else (n, nsys)
    assert tf.penta_partition_chunks(nrow, ncol, direction, 0) >= 16
    for kind in ("cfg4", "bend1e4"):
        arrs = systems(kind, nsys, n, seed=4)
        x, ref = solve_both(tf, tfo, arrs, direction, 0)
        assert rel_inf(x, ref) <= TOL[kind]
        assert backward_error(arrs, x) <= 2e-14


@pytest.mark.parametrize("nsys,length", [(37, 64), (8, 1024), (5, 2048), (16, 130), (3, 1000)])
def test_cyclic_reduction_variant_rows(tf, nsys, length):
    """TF_PENTA_PCR (parallel cyclic reduction on 2 x 2 blocks, systems along rows): config-4 systems against the
    oracle's LU (<= 1e-12) and by backward error (needs no oracle); weakly dominant bending systems by backward error."""
    import torch
    from oracle import tfo
    for gen, tol in ((lambda: inputs.penta_system(nsys, length, seed=length), 1e-12),
                     (lambda: inputs.penta_system_bending(nsys, length, seed=length, sigma=1e2), None)):
        e, c, d, a, b, y = gen()
        x = tf.penta_solve(0, *[torch.from_numpy(t).cuda() for t in (e, c, d, a, b, y)], variant=tf.PENTA_PCR)
        torch.cuda.synchronize()
        x = x.cpu().numpy()
        if tol is not None:
            ref = tfo.penta_solve(0, e, c, d, a, b, y)
            assert np.max(np.abs(x - ref)) <= tol * np.max(np.abs(ref))
        Ax = d * x
        Ax[:, 1:] += c[:, 1:] * x[:, :-1]
        Ax[:, 2:] += e[:, 2:] * x[:, :-2]
        Ax[:, :-1] += a[:, :-1] * x[:, 1:]
        Ax[:, :-2] += b[:, :-2] * x[:, 2:]
        normA = np.max(np.abs(e) + np.abs(c) + np.abs(d) + np.abs(a) + np.abs(b))
        assert np.max(np.abs(Ax - y)) / (normA * np.max(np.abs(x)) + np.max(np.abs(y))) <= 1e-13


def test_cyclic_reduction_variant_refuses_other_shapes(tf):
    import torch
    t = [torch.ones(8, 4096, dtype=torch.float64, device="cuda") for _ in range(6)]
    with pytest.raises(tf.TfError) as err:
        tf.penta_solve(0, *t, variant=tf.PENTA_PCR)
    assert err.value.status == tf.ERR_UNSUPPORTED
    t = [torch.ones(256, 64, dtype=torch.float64, device="cuda") for _ in range(6)]
    with pytest.raises(tf.TfError):
        tf.penta_solve(1, *t, variant=tf.PENTA_PCR)

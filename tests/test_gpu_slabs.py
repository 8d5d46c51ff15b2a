"""GPU tests of the slab solver (tf_penta_slab_interface / tf_penta_slab_solve).  One GPU is all
this environment has, so the slabs of R "ranks" are processed one after the other on it (no kernel waits for another):
phase 1 of every slab, concatenation in slab order in place of the all-gather, phase 2 of every slab; the assembled
solution is compared with the CPU oracle's LU of the whole systems.  A world-size-1 NCCL run drives the same kernels
through paper_1806_10550_b200/dist.py (the all-gather then is NCCL's).  The exchange logic for world sizes 2 and 3 is
covered on the CPU (tests/test_multirank_slabs.py)."""
import os
import socket

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


def systems(kind, nsys, n):
    arrs = inputs.penta_system(nsys, n, seed=13) if kind == "cfg4" else inputs.penta_system_bending(nsys, n, 13, 1e4)
    return arrs                                                      # [nsys][len]


def backward_error(arrs, xs):
    e, c, d, a, b, y = arrs
    Ax = d * xs
    Ax[:, 1:] += c[:, 1:] * xs[:, :-1]
    Ax[:, 2:] += e[:, 2:] * xs[:, :-2]
    Ax[:, :-1] += a[:, :-1] * xs[:, 1:]
    Ax[:, :-2] += b[:, :-2] * xs[:, 2:]
    normA = np.max(np.abs(e) + np.abs(c) + np.abs(d) + np.abs(a) + np.abs(b))
    return float(np.max(np.abs(Ax - y)) / (normA * np.max(np.abs(xs)) + np.max(np.abs(y))))


@pytest.mark.parametrize("world,nparts,nsys,n", [(2, 1, 64, 512), (3, 2, 96, 1200), (4, 1, 34, 2050), (2, 3, 130, 998)])
@pytest.mark.parametrize("kind", ["cfg4", "bend1e4"])
@pytest.mark.parametrize("direction", [0, 1])
def test_slabs_processed_in_turn_equal_the_whole_solve(tf, tfo, world, nparts, nsys, n, kind, direction):
    import torch
    from paper_1806_10550_b200 import dist as tfdist
    arrs = systems(kind, nsys, n)
    full = arrs if direction == 0 else [np.ascontiguousarray(t.T) for t in arrs]     # direction 1: [len][nsys]
    ref = tfo.penta_solve(direction, *full)
    bounds = [tfdist.slab_bounds(n, world, r) for r in range(world)]
    def cut(t, r):
        lo, hi = bounds[r]
        return torch.from_numpy(np.ascontiguousarray(t[:, lo:hi] if direction == 0 else t[lo:hi])).cuda()
    local = [[cut(t, r) for t in full] for r in range(world)]
    ifaces = [tf.penta_slab_interface(direction, nparts, r, world, *local[r]) for r in range(world)]
    gathered = torch.cat(ifaces, dim=0).contiguous()
    xs = [tf.penta_slab_solve(direction, nparts, r, world, *local[r], gathered) for r in range(world)]
    torch.cuda.synchronize()
    x = torch.cat(xs, dim=1 if direction == 0 else 0).cpu().numpy()
    tol = 1e-12 if kind == "cfg4" else 1e-9
    assert np.max(np.abs(x - ref)) <= tol * np.max(np.abs(ref))
    assert backward_error(arrs, x if direction == 0 else x.T) <= 2e-14


def test_world_size_one_through_nccl(tf, tfo):
    """the dist.py path with a real NCCL group of one rank: interface pass, NCCL all-gather, reduced + chunk solves"""
    import torch
    import torch.distributed as dist
    from paper_1806_10550_b200 import dist as tfdist
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        arrs = [np.ascontiguousarray(t.T) for t in systems("bend1e4", 64, 1024)]
        dev = [torch.from_numpy(t).cuda() for t in arrs]
        x = tfdist.penta_solve_slabs(1, 4, *dev)
        torch.cuda.synchronize()
        ref = tfo.penta_solve(1, *arrs)
        assert np.max(np.abs(x.cpu().numpy() - ref)) <= 1e-9 * np.max(np.abs(ref))
    finally:
        dist.destroy_process_group()

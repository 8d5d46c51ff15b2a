"""N > 1 path of the slab solver (paper_1806_10550_b200/dist.py) on the CPU: a world-size-2
and a world-size-3 gloo run of the exchange logic -- slab bounds, interface values of every rank gathered in slab order,
local solves -- with numpy stand-ins for the three kernel phases (tests/partition_numpy.py), compared with a dense
solve of the whole systems.  The kernels themselves are tested on the GPU (tests/test_gpu_slabs.py)."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _systems(n, nsys):
    from paper_1806_10550_b200 import inputs
    arrs = inputs.penta_system_bending(nsys, n, 7, 1e4)              # rows couple over tens of rows: seams matter
    return [np.ascontiguousarray(t.T) for t in arrs]                 # direction 1 layout [len][nsys]


def _worker(rank, world, port, out, n, nsys, nparts):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import partition_numpy as pn
    from paper_1806_10550_b200 import dist as tfdist
    lo, hi = tfdist.slab_bounds(n, world, rank)
    local = [torch.from_numpy(np.ascontiguousarray(t[lo:hi])) for t in _systems(n, nsys)]
    x = tfdist.penta_solve_slabs(1, nparts, *local, interface_fn=pn.interface, solve_fn=pn.solve)
    np.save(os.path.join(out, f"x{rank}.npy"), x.numpy())
    dist.destroy_process_group()


def _dense(arrs):
    e, c, d, a, b, y = arrs
    n, nsys = d.shape
    x = np.zeros((n, nsys))
    for s in range(nsys):
        M = np.diag(d[:, s]) + np.diag(c[1:, s], -1) + np.diag(e[2:, s], -2) + np.diag(a[:-1, s], 1) + np.diag(b[:-2, s], 2)
        x[:, s] = np.linalg.solve(M, y[:, s])
    return x


def _run(tmp_path, world, n, nsys, nparts):
    from paper_1806_10550_b200 import dist as tfdist
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path), n, nsys, nparts), nprocs=world, join=True)
    x = np.concatenate([np.load(tmp_path / f"x{r}.npy") for r in range(world)], axis=0)
    ref = _dense(_systems(n, nsys))
    assert x.shape == ref.shape
    assert np.max(np.abs(x - ref)) <= 1e-9 * np.max(np.abs(ref))
    bounds = [tfdist.slab_bounds(n, world, r) for r in range(world)]
    assert bounds[0][0] == 0 and bounds[-1][1] == n and all(bounds[r][1] == bounds[r + 1][0] for r in range(world - 1))
    assert all(b[0] % 16 == 0 for b in bounds)


def test_world2_one_chunk_per_rank(tmp_path):
    _run(tmp_path, 2, 420, 3, 1)


def test_world3_two_chunks_per_rank(tmp_path):
    _run(tmp_path, 3, 1000, 2, 2)

"""Exchange logic of the distributed time step (paper_1806_10550_b200/dist_step.py) on the CPU, no kernels: the two
redistributions between row blocks and halo'd column blocks -- (a) under real gloo groups of 2 and 3 ranks, (b) with the
in-process stand-in the GPU test uses, so that the stand-in itself is checked against gloo's behaviour."""
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


def field(nx, ny):
    j, i = np.mgrid[0:ny, 0:nx]
    return (1000.0 * j + i).astype(np.float64)              # every cell knows where it came from


class CpuBlocks:
    """Stand-in for the library's tf_blocks_gather / tf_blocks_scatter on CPU tensors, written from include/tf.h's
    statement of the two calls (the CUDA kernels are compared with it in tests/test_gpu_distributed_step.py)."""

    @staticmethod
    def make_rects(blocks):
        return [tuple(int(v) for v in b) for b in blocks]

    @staticmethod
    def blocks_gather(field, rects, buf):
        for row0, nrows, col0, ncols, off in rects:
            buf[off:off + nrows * ncols] = field[row0:row0 + nrows, col0:col0 + ncols].reshape(-1)

    @staticmethod
    def block_copy(src, srow0, scol0, dst, drow0, dcol0, nrows, ncols, reflect_left=False, reflect_right_at=-1):
        dst[drow0:drow0 + nrows, dcol0:dcol0 + ncols] = src[srow0:srow0 + nrows, scol0:scol0 + ncols]
        CpuBlocks.blocks_scatter(None, [], dst, reflect_left, reflect_right_at)

    @staticmethod
    def blocks_scatter(buf, rects, field, reflect_left=False, reflect_right_at=-1):
        for row0, nrows, col0, ncols, off in rects:
            field[row0:row0 + nrows, col0:col0 + ncols] = buf[off:off + nrows * ncols].view(nrows, ncols)
        if reflect_left:
            field[:, 1] = field[:, 2]
            field[:, 0] = field[:, 3]
        g = reflect_right_at
        if g >= 0:
            field[:, g] = field[:, g - 1]
            field[:, g + 1] = field[:, g - 2]


def check_rank(lay, r, comm, nx, ny):
    from paper_1806_10550_b200 import dist_step as ds
    ex = ds.Exchange(lay, r, CpuBlocks, device="cpu")
    F = field(nx, ny)
    j0, j1 = lay.rows[r]
    i0, i1 = lay.cols[r]
    f_rows = torch.from_numpy(F[j0:j1].copy())
    f_cols = torch.full((ny, lay.local_width(r)), -1.0, dtype=torch.float64)
    ex.rows_to_cols(comm, f_rows, f_cols)
    n = i1 - i0
    assert np.array_equal(f_cols[:, 2:2 + n].numpy(), F[:, i0:i1])                        # the block itself
    left = F[:, [1, 0]] if r == 0 else F[:, i0 - 2:i0]                                   # reflection: h_-2 = h_1, h_-1 = h_0
    right = F[:, [nx - 1, nx - 2]] if r == lay.world - 1 else F[:, i1:i1 + 2]
    assert np.array_equal(f_cols[:, :2].numpy(), left) and np.array_equal(f_cols[:, n + 2:].numpy(), right)
    back = torch.full((j1 - j0, nx), -1.0, dtype=torch.float64)
    ex.cols_to_rows(comm, f_cols, back)
    assert np.array_equal(back.numpy(), F[j0:j1])                                         # round trip
    return True


def _worker(rank, world, port, nx, ny):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1806_10550_b200 import dist_step as ds
    comm = ds.TorchComm()
    assert check_rank(ds.Layout(nx, ny, world), rank, comm, nx, ny)
    t = torch.tensor([float(rank), 1.0], dtype=torch.float64)
    assert comm.all_reduce(t.clone(), "max").tolist() == [world - 1.0, 1.0]
    assert comm.all_reduce(t.clone(), "sum").tolist() == [world * (world - 1) / 2.0, float(world)]
    dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_gloo_world2_and_world3():
    for world, nx, ny in ((2, 70, 50), (3, 130, 100)):
        mp.spawn(_worker, args=(world, _free_port(), nx, ny), nprocs=world, join=True)


def test_in_process_stand_in_behaves_the_same():
    import local_comm
    from paper_1806_10550_b200 import dist_step as ds
    for world, nx, ny in ((2, 70, 50), (3, 130, 100), (4, 200, 64)):
        lay = ds.Layout(nx, ny, world)
        assert all(local_comm.run_ranks(world, lambda comm: check_rank(lay, comm.rank, comm, nx, ny)))
    assert lay.rows[0][0] == 0 and lay.rows[-1][1] == 64 and lay.cols[-1][1] == 200

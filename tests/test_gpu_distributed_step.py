"""The time step with the film spread over several ranks (paper_1806_10550_b200/dist_step.py)
on the one GPU available: R host threads, one per rank, each with its two contexts (row block / halo'd column block);
the collectives are the in-process stand-in of tests/local_comm.py (checked against gloo on the CPU); the kernels of
different ranks never wait for one another.  Compared with the single-device path on the same film: same Newton counts,
fields equal to 1e-11 (the flux through a domain boundary face is zero to rounding instead of exactly zero), mass."""
import os
import socket
import sys

import numpy as np
import pytest

from paper_1806_10550_b200 import inputs

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu
K, HS = 100.0, 0.1


@pytest.fixture(scope="module")
def tf():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1806_10550_b200 import tf as tfmod
    tfmod.lib()
    return tfmod


def single(tf, h0, dx, dy, dts):
    ny, nx = h0.shape
    g = tf.ThinFilm(nx, ny, dx, dy, K, HS, 3, 2)
    g.set_newton(1e-10, 64, 0)
    g.set_state(h0)
    log = [g.step(dt) for dt in dts]
    return log, g.get_state(), g.mass()


@pytest.mark.parametrize("world,nx,ny", [(2, 128, 96), (3, 208, 160), (4, 256, 130), (2, 2048, 1536)])
def test_ranks_as_threads_equal_the_single_device_step(tf, world, nx, ny):
    import local_comm
    from paper_1806_10550_b200 import dist_step as ds
    dx, dy = 0.4259, 0.45
    h0 = inputs.noise_ic(nx, ny, seed=nx + world)
    dts = [1e-2, 1e-2, 5e-3]
    ref_log, ref_h, ref_m = single(tf, h0, dx, dy, dts)
    lay = ds.Layout(nx, ny, world)

    def rank_main(comm):
        f = ds.DistributedFilm(nx, ny, dx, dy, K, HS, 3, 2, comm=comm, tol=1e-10, max_iter=64)
        j0, j1 = lay.rows[comm.rank]
        f.set_state_rows(np.ascontiguousarray(h0[j0:j1]))
        log = [f.step(dt) for dt in dts]
        return log, f.get_state_rows(), f.mass()

    out = local_comm.run_ranks(world, rank_main)
    h = np.concatenate([o[1] for o in out], axis=0)
    for r in range(world):
        assert [(s, k) for s, k, _ in out[r][0]] == [(s, k) for s, k, _ in ref_log]       # same decisions on every rank
        assert all(abs(a[2] - b[2]) <= 1e-9 * b[2] for a, b in zip(out[r][0], ref_log))
        assert abs(out[r][2] - ref_m) <= 1e-13 * ref_m
    assert np.max(np.abs(h - ref_h)) <= 1e-11 * np.max(np.abs(ref_h))


@pytest.mark.parametrize("world,nx,ny", [(2, 128, 96), (3, 208, 160)])
def test_ranks_as_threads_equal_the_oracle(tf, world, nx, ny):
    """The assembled film of the distributed step against the CPU oracle (not the single-device CUDA path): same
    Newton counts, every element to 1e-11 after one converged step and after three steps with a fixed count."""
    import local_comm
    from oracle import tfo
    from paper_1806_10550_b200 import dist_step as ds
    dx, dy = 0.4259, 0.45
    h0 = inputs.noise_ic(nx, ny, seed=nx + world)
    lay = ds.Layout(nx, ny, world)
    o = tfo.ThinFilmOracle(nx, ny, dx, dy, K, HS, 3, 2)
    o.set_newton(1e-10, 64, 0)
    o.set_state(h0)
    ref_log = [o.step(1e-2)]
    ref_h1 = o.get_state()
    ref_log += [o.step(1e-2), o.step(5e-3)]
    ref_h3 = o.get_state()

    def rank_main(comm):
        f = ds.DistributedFilm(nx, ny, dx, dy, K, HS, 3, 2, comm=comm, tol=1e-10, max_iter=64)
        j0, j1 = lay.rows[comm.rank]
        f.set_state_rows(np.ascontiguousarray(h0[j0:j1]))
        log = [f.step(1e-2)]
        h1 = f.get_state_rows()
        log += [f.step(1e-2), f.step(5e-3)]
        return log, h1, f.get_state_rows(), f.mass()

    out = local_comm.run_ranks(world, rank_main)
    h1 = np.concatenate([r[1] for r in out], axis=0)
    h3 = np.concatenate([r[2] for r in out], axis=0)
    for r in range(world):
        assert [(s, k) for s, k, _ in out[r][0]] == [(s, k) for s, k, _ in ref_log]
        assert abs(out[r][3] - o.mass()) <= 1e-13 * o.mass()
    assert np.max(np.abs(h1 - ref_h1)) <= 1e-11 * np.max(np.abs(ref_h1))
    assert np.max(np.abs(h3 - ref_h3)) <= 1e-10 * np.max(np.abs(ref_h3))     # three converged steps (tol 1e-10 each)


def test_block_kernels_equal_the_cpu_statement(tf):
    """tf_blocks_gather / tf_blocks_scatter (incl. the ghost reflection of (2.28)) against the plain CPU statement of
    the two calls in tests/test_multirank_redistribution.py, on ragged blocks."""
    import torch
    from test_multirank_redistribution import CpuBlocks
    rng = np.random.default_rng(3)
    ny, nx = 57, 203
    F = torch.from_numpy(rng.uniform(0, 1, (ny, nx)))
    blocks, off = [], 0
    for (r0, nr, c0, nc) in ((0, 10, 0, 203), (10, 47, 5, 101), (3, 1, 200, 3), (20, 0, 0, 7), (56, 1, 0, 1)):
        blocks.append((r0, nr, c0, nc, off))
        off += nr * nc
    buf_c, buf_g = torch.zeros(off, dtype=torch.float64), torch.zeros(off, dtype=torch.float64, device="cuda")
    CpuBlocks.blocks_gather(F, CpuBlocks.make_rects(blocks), buf_c)
    tf.blocks_gather(F.cuda(), tf.make_rects(blocks), buf_g)
    assert torch.equal(buf_g.cpu(), buf_c)
    n = 40                                                     # a halo'd column block of 40 own columns at both domain edges
    blocks = [(0, 30, 2, n, 0), (30, 27, 2, n, 30 * n)]
    src = torch.from_numpy(rng.uniform(0, 1, ny * n))
    for lrefl, rrefl in ((True, n + 2), (False, -1), (True, -1), (False, n + 2)):
        dst_c = torch.full((ny, n + 4), -1.0, dtype=torch.float64)
        dst_g = dst_c.clone().cuda()
        CpuBlocks.blocks_scatter(src, CpuBlocks.make_rects(blocks), dst_c, lrefl, rrefl)
        tf.blocks_scatter(src.cuda(), tf.make_rects(blocks), dst_g, lrefl, rrefl)
        assert torch.equal(dst_g.cpu(), dst_c), (lrefl, rrefl)
        dst_c = torch.full((ny, n + 4), -1.0, dtype=torch.float64)          # the same block straight from a field
        dst_g = dst_c.clone().cuda()
        CpuBlocks.block_copy(F, 0, 17, dst_c, 0, 2, ny, n, lrefl, rrefl)
        tf.block_copy(F.cuda(), 0, 17, dst_g, 0, 2, ny, n, lrefl, rrefl)
        assert torch.equal(dst_g.cpu(), dst_c), (lrefl, rrefl)


def test_rejected_step_leaves_the_distributed_state_unchanged(tf):
    import local_comm
    from paper_1806_10550_b200 import dist_step as ds
    nx, ny, world = 128, 96, 2
    h0 = inputs.noise_ic(nx, ny, seed=5)
    lay = ds.Layout(nx, ny, world)

    def rank_main(comm):
        f = ds.DistributedFilm(nx, ny, 0.4259, 0.4259, K, HS, 3, 2, comm=comm, tol=1e-12, max_iter=3)
        j0, j1 = lay.rows[comm.rank]
        f.set_state_rows(np.ascontiguousarray(h0[j0:j1]))
        st = f.step(1e-2)
        return st, f.get_state_rows()

    out = local_comm.run_ranks(world, rank_main)
    assert all(o[0][0] == tf.NOT_CONVERGED and o[0][1] == 3 for o in out)
    assert np.array_equal(np.concatenate([o[1] for o in out], axis=0), h0)


def test_world_size_one_through_nccl(tf):
    import torch
    import torch.distributed as dist
    from paper_1806_10550_b200 import dist_step as ds
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        nx, ny = 160, 128
        h0 = inputs.noise_ic(nx, ny, seed=2)
        ref_log, ref_h, _ = single(tf, h0, 0.4259, 0.4259, [1e-2, 1e-2])
        f = ds.DistributedFilm(nx, ny, 0.4259, 0.4259, K, HS, 3, 2, tol=1e-10, max_iter=64)
        f.set_state_rows(h0)
        log = [f.step(1e-2) for _ in range(2)]
        torch.cuda.synchronize()
        assert [(s, k) for s, k, _ in log] == [(s, k) for s, k, _ in ref_log]
        assert np.max(np.abs(f.get_state_rows() - ref_h)) <= 1e-11 * np.max(np.abs(ref_h))
    finally:
        dist.destroy_process_group()

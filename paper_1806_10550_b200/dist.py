"""Batched pentadiagonal solve with every system spread over the ranks of a torch.distributed group
(PAPER.md:647 names multi-GPU and SPIKE-type solvers as future work).

Rank r holds slab r of every system: rows [r*n_loc, (r+1)*n_loc) of the [len][nsys] arrays for direction 1 (systems =
columns), the corresponding block of columns for direction 0.  One exchange step: an all-gather of the interface values
(20 * nparts doubles per system and rank) between tf_penta_slab_interface and tf_penta_slab_solve; everything else is
local.  The collective is torch.distributed's (NCCL over NVLink on the GPUs; any backend works for the logic), issued
on the caller's current stream, so the three phases are ordered without a host synchronisation.
"""
import torch.distributed as dist


def slab_bounds(n, world, rank):
    """rows (or columns) [lo, hi) of slab `rank` when n is divided into `world` slabs whose bounds are multiples of 16
    (the tile width of the kernels); the last slab takes the remainder"""
    step = (n // world) // 16 * 16
    if step == 0:
        raise ValueError("slabs would be shorter than 16")
    lo = rank * step
    hi = n if rank == world - 1 else lo + step
    return lo, hi


def penta_solve_slabs(direction, nparts, e, c, d, a, b, rhs, group=None, interface_fn=None, solve_fn=None):
    """Solve with the local slab of the six arrays; returns the local slab of the solution.  `interface_fn` /
    `solve_fn` default to the library calls (tf.penta_slab_interface / tf.penta_slab_solve); tests pass stand-ins to
    exercise the exchange logic without a GPU."""
    import torch
    if interface_fn is None or solve_fn is None:
        from . import tf
        interface_fn = interface_fn or tf.penta_slab_interface
        solve_fn = solve_fn or tf.penta_slab_solve
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    local = interface_fn(direction, nparts, rank, world, e, c, d, a, b, rhs)
    gathered = torch.empty((world * local.shape[0],) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    dist.all_gather_into_tensor(gathered, local.contiguous(), group=group)
    return solve_fn(direction, nparts, rank, world, e, c, d, a, b, rhs, gathered)

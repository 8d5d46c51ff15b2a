"""Test helper: an in-process stand-in for a torch.distributed group -- R threads, one per "rank", exchange through a
shared mailbox between two barriers.  Used to run paper_1806_10550_b200/dist_step.py with several ranks on the one GPU
(or on the CPU) this environment has: the kernels of different ranks never wait for one another, the host threads do."""
import threading

import torch


class Shared:
    def __init__(self, world):
        self.world, self.box, self.barrier = world, [None] * world, threading.Barrier(world)


class LocalComm:
    def __init__(self, shared, rank):
        self.s, self.rank, self.world = shared, rank, shared.world

    def all_to_all(self, send, send_counts, recv_counts, out=None):
        if send.is_cuda:
            torch.cuda.synchronize()
        self.s.box[self.rank] = (send, list(map(int, send_counts)))
        self.s.barrier.wait()
        pieces = []
        for p in range(self.world):
            buf, counts = self.s.box[p]
            off = sum(counts[:self.rank])
            assert counts[self.rank] == int(recv_counts[p]), "split sizes of sender and receiver disagree"
            pieces.append(buf[off:off + counts[self.rank]])
        recv = torch.cat(pieces).clone()
        if out is not None:                                   # the caller's preallocated receive buffer, as TorchComm fills it
            out[:recv.numel()].copy_(recv)
            recv = out[:recv.numel()]
        if recv.is_cuda:
            torch.cuda.synchronize()
        self.s.barrier.wait()
        return recv

    def all_reduce(self, t, op):
        if t.is_cuda:
            torch.cuda.synchronize()
        self.s.box[self.rank] = t.clone()
        self.s.barrier.wait()
        stack = torch.stack([self.s.box[p] for p in range(self.world)])
        out = stack.max(dim=0).values if op == "max" else stack.sum(dim=0)
        self.s.barrier.wait()
        t.copy_(out)
        return t


def run_ranks(world, fn):
    """fn(comm) on `world` threads; returns the list of results in rank order; re-raises the first exception"""
    shared, out, err = Shared(world), [None] * world, []

    def work(r):
        try:
            out[r] = fn(LocalComm(shared, r))
        except BaseException as e:          # noqa: BLE001 -- reported below
            err.append(e)
            shared.barrier.abort()
    th = [threading.Thread(target=work, args=(r,)) for r in range(world)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    if err:
        raise err[0]
    return out

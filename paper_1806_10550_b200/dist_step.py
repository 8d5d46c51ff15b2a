"""The time step with the film spread over the ranks of a torch.distributed group.

Classic ADI decomposition: the x-sweep runs on ROW blocks (its lines are rows: nothing to exchange), the y-sweep on
COLUMN blocks (its lines are columns), and the field is redistributed between the two layouts, one all-to-all each way
per Newton iteration:

    rank r:   ctx_y = film of [ny] x [columns i0_r-2 .. i1_r+2)     (two halo columns per side: the 13-point operator
                                                                      of the y-sweep's right-hand side reaches i +- 2)
              ctx_x = film of [rows j0_r .. j1_r) x [nx]
    k = 0, 1, ...:
        ctx_y: y-sweep of iteration k            (S1-S4 of DESIGN.md; tf_sweep(.., which = 1))  -> w   [column block]
        all-to-all: w -> row blocks
        ctx_x: x-sweep of iteration k            (S5-S7; tf_sweep(.., which = 2))               -> u_(k+1), residual
        all-to-all: u_(k+1) -> column blocks with halos (reflection at the domain's own edges)
        all-reduce (max) of the residual record; accept / iterate / reject on every rank alike

Both contexts are ordinary single-device contexts: ctx_y simply is a film that is four columns wider than the block it
owns, and whatever the kernels compute in those halo columns is never used.  At a domain edge the halo holds the
reflected values, so the flux through the boundary face is zero to rounding instead of exactly zero; everything else
is the arithmetic of the single-device path (parity with it to 1e-11, not bit for bit).

The collectives go through a small `comm` object (all_to_all of flat buffers with split sizes, all_reduce max / sum):
TorchComm wraps a torch.distributed group (NCCL over NVLink on GPUs); tests pass an in-process stand-in.
Packing and unpacking of the blocks, the ghost reflection of (2.28) at the domain's own edges and the preparation of
the residual record for the reduction are library kernels (tf_blocks_gather / tf_blocks_scatter / tf_record_sanitize,
include/tf.h): this module holds no arithmetic of the method.
"""
import numpy as np

from .dist import slab_bounds


class TorchComm:
    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.world, self.rank = dist.get_world_size(group), dist.get_rank(group)

    def all_to_all(self, send, send_counts, recv_counts, out=None):
        """`out`: a preallocated receive buffer of at least sum(recv_counts) elements (Exchange keeps one per direction,
        so the per-iteration exchanges allocate nothing); None: a fresh tensor"""
        import torch
        total = int(sum(recv_counts))
        recv = out[:total] if out is not None else torch.empty(total, dtype=send.dtype, device=send.device)
        self.dist.all_to_all_single(recv, send, list(map(int, recv_counts)), list(map(int, send_counts)), group=self.group)
        return recv

    def all_reduce(self, t, op):
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX if op == "max" else self.dist.ReduceOp.SUM, group=self.group)
        return t


class Layout:
    """who owns what: row blocks [j0, j1) and column blocks [i0, i1) of every rank, and the halo'd column range"""
    HALO = 2

    def __init__(self, nx, ny, world):
        self.nx, self.ny, self.world = nx, ny, world
        self.rows = [slab_bounds(ny, world, r) for r in range(world)]
        self.cols = [slab_bounds(nx, world, r) for r in range(world)]

    def halo_cols(self, r):
        """global columns rank r receives for its column block: its own plus up to HALO neighbours per side"""
        i0, i1 = self.cols[r]
        return max(i0 - self.HALO, 0), min(i1 + self.HALO, self.nx)

    def local_width(self, r):
        return self.cols[r][1] - self.cols[r][0] + 2 * self.HALO


class Exchange:
    """The two redistributions of rank r with everything that does not change from call to call worked out once:
    block lists (tf_rect arrays), split sizes, send / receive buffers.  Packing, unpacking and the ghost reflection of
    (2.28) run in the library (tf_blocks_gather / tf_blocks_scatter); this class only strings them around the
    all-to-all."""

    def __init__(self, lay, r, tf, device="cuda"):
        import torch
        self.lay, self.r, self.tf = lay, r, tf
        j0, j1 = lay.rows[r]
        nyl = j1 - j0
        i0, i1 = lay.cols[r]
        n = i1 - i0
        a, b = lay.halo_cols(r)
        # rows -> columns: send to q the columns q needs (own + halo) of my rows; receive my halo'd columns of p's rows
        # (the block a rank keeps for itself goes straight from field to field: tf_block_copy, zero split size)
        blocks, off, self.rc_scount, self.rc_rcount = [], 0, [], []
        for q in range(lay.world):
            aq, bq = lay.halo_cols(q)
            cnt = 0 if q == r else nyl * (bq - aq)
            blocks.append((0, nyl if q != r else 0, aq, bq - aq, off))
            self.rc_scount.append(cnt)
            off += cnt
        self.rc_send_rects, self.rc_send = tf.make_rects(blocks), torch.empty(max(off, 1), dtype=torch.float64, device=device)
        loc = a - (i0 - lay.HALO)                      # local column of global column a (2 at the left domain edge)
        blocks, off = [], 0
        for p in range(lay.world):
            p0, p1 = lay.rows[p]
            cnt = 0 if p == r else (p1 - p0) * (b - a)
            blocks.append((p0, p1 - p0 if p != r else 0, loc, b - a, off))
            self.rc_rcount.append(cnt)
            off += cnt
        self.rc_recv_rects = tf.make_rects(blocks)
        self.rc_recv = torch.empty(max(off, 1), dtype=torch.float64, device=device)
        self.rc_self = (0, a, j0, loc, nyl, b - a)      # src row0, col0 -> dst row0, col0, rows, cols
        self.refl_left = (r == 0)                      # h_{-1} = h_0, h_{-2} = h_1
        self.refl_right_at = n + 2 if r == lay.world - 1 else -1
        # columns -> rows: send to q its rows of my own columns; receive p's columns of my rows
        blocks, off, self.cr_scount, self.cr_rcount = [], 0, [], []
        for q in range(lay.world):
            q0, q1 = lay.rows[q]
            cnt = 0 if q == r else (q1 - q0) * n
            blocks.append((q0, q1 - q0 if q != r else 0, lay.HALO, n, off))
            self.cr_scount.append(cnt)
            off += cnt
        self.cr_send_rects, self.cr_send = tf.make_rects(blocks), torch.empty(max(off, 1), dtype=torch.float64, device=device)
        blocks, off = [], 0
        for p in range(lay.world):
            c0, c1 = lay.cols[p]
            cnt = 0 if p == r else nyl * (c1 - c0)
            blocks.append((0, nyl if p != r else 0, c0, c1 - c0, off))
            self.cr_rcount.append(cnt)
            off += cnt
        self.cr_recv_rects = tf.make_rects(blocks)
        self.cr_recv = torch.empty(max(off, 1), dtype=torch.float64, device=device)
        self.cr_self = (j0, lay.HALO, 0, i0, nyl, n)

    def rows_to_cols(self, comm, f_rows, f_cols):
        """f_rows: [ny_loc][nx] of this rank -> f_cols: [ny][nxl + 4] of this rank, halos and ghosts included"""
        sr, sc, dr, dc, nr, nc = self.rc_self
        self.tf.block_copy(f_rows, sr, sc, f_cols, dr, dc, nr, nc, self.refl_left, self.refl_right_at)
        if self.lay.world > 1:
            self.tf.blocks_gather(f_rows, self.rc_send_rects, self.rc_send)
            recv = comm.all_to_all(self.rc_send, self.rc_scount, self.rc_rcount, out=self.rc_recv)
            self.tf.blocks_scatter(recv, self.rc_recv_rects, f_cols, self.refl_left, self.refl_right_at)

    def cols_to_rows(self, comm, f_cols, f_rows):
        """interior of f_cols [ny][nxl + 4] of this rank -> f_rows [ny_loc][nx] of this rank"""
        sr, sc, dr, dc, nr, nc = self.cr_self
        self.tf.block_copy(f_cols, sr, sc, f_rows, dr, dc, nr, nc)
        if self.lay.world > 1:
            self.tf.blocks_gather(f_cols, self.cr_send_rects, self.cr_send)
            recv = comm.all_to_all(self.cr_send, self.cr_scount, self.cr_rcount, out=self.cr_recv)
            self.tf.blocks_scatter(recv, self.cr_recv_rects, f_rows)


class DistributedFilm:
    """tf_step for a film spread over the ranks of `comm`; every rank constructs it with the same arguments."""

    def __init__(self, nx, ny, dx, dy, kappa=100.0, hstar=0.1, n=3, m=2, comm=None, tol=1e-10, max_iter=10):
        from . import tf
        self.tf = tf
        self.comm = comm if comm is not None else TorchComm()
        self.rank, self.world = self.comm.rank, self.comm.world
        self.lay = Layout(nx, ny, self.world)
        self.nx, self.ny, self.dx, self.dy = nx, ny, dx, dy
        self.tol, self.max_iter = tol, max_iter
        j0, j1 = self.lay.rows[self.rank]
        self.ctx_x = tf.ThinFilm(nx, j1 - j0, dx, dy, kappa, hstar, n, m)
        self.ctx_y = tf.ThinFilm(self.lay.local_width(self.rank), ny, dx, dy, kappa, hstar, n, m)
        for c in (self.ctx_x, self.ctx_y):
            c.set_newton(tol, min(max_iter, 4096), 0)                 # the gate compares with the context's tol
        self.last_iters = 1
        self.ex = Exchange(self.lay, self.rank, tf)

    def set_state_rows(self, h_rows):
        """h_rows: this rank's row block [ny_loc][nx] (numpy or CUDA tensor); distributes the column layout too"""
        import torch
        self.ctx_x.set_state(h_rows)
        tmp = torch.ones(self.ny, self.lay.local_width(self.rank), dtype=torch.float64, device="cuda")
        self.ex.rows_to_cols(self.comm, self.ctx_x.field(self.ctx_x.FIELD_STATE), tmp)
        self.ctx_y.set_state(tmp)

    def set_pressure(self, kind, params=()):
        """tf_set_pressure on both contexts (NLC / polymer models)"""
        self.ctx_x.set_pressure(kind, params)
        self.ctx_y.set_pressure(kind, params)

    def get_state_rows(self):
        return self.ctx_x.get_state()

    def step(self, dt, batch=None):
        """returns (status, newton_iters, residual) like ThinFilm.step; on rejection the state is unchanged.
        Iterations are enqueued `batch` at a time (the first batch one shorter than the previous accepted step's count:
        an iteration enqueued past the deciding one still moves the whole field twice over the interconnect, so the
        speculation stops just short of where the last step ended and goes on two at a time) and
        the host reads the records of a batch at once: the sweeps of iteration k are gated on the ALL-REDUCED record
        of iteration k-1, which is written into both contexts, so iterations past the deciding one do nothing on any
        rank (their redistributions move unchanged data) -- the scheme of tf_set_launch_ahead across ranks."""
        import torch
        tf, cx, cy = self.tf, self.ctx_x, self.ctx_y
        rx, ry = cx.field(cx.FIELD_RECORDS), cy.field(cy.FIELD_RECORDS)
        gate = cx.SWEEP_GATED
        batch = max(1, int(batch if batch is not None else self.last_iters - 1))
        k = done = 0
        res, status, decided = 0.0, tf.NOT_CONVERGED, False
        while not decided and done < self.max_iter:
            upto = min(self.max_iter, k + batch)
            while k < upto:
                cy.sweep(dt, k, cy.SWEEP_Y | gate)
                self.ex.cols_to_rows(self.comm, cy.field(cy.FIELD_W), cx.field(cx.FIELD_W))
                cx.sweep(dt, k, cx.SWEEP_X | gate)
                self.ex.rows_to_cols(self.comm, cx.field(cx.FIELD_ITERATE), cy.field(cy.FIELD_ITERATE))
                cx.record_sanitize(k)                                # a NaN must win the max and close the gates
                rec = rx[k]
                self.comm.all_reduce(rec, "max")
                ry[k].copy_(rec)
                k += 1
            recs = rx[done:k].cpu().numpy()                          # one synchronising read per batch
            for r, bad in recs:
                done += 1
                res = float(r)
                if bad != 0 or not np.isfinite(res):
                    decided = True
                    break
                if res < self.tol:
                    status, decided = tf.OK, True
                    break
            batch = 2
        if status == tf.OK:
            cx.accept()
            cy.accept()
            self.last_iters = done
        return status, done, res

    def mass(self):
        import torch
        t = torch.tensor([self.ctx_x.mass()], dtype=torch.float64, device="cuda")
        return float(self.comm.all_reduce(t, "sum")[0])

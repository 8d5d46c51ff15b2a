"""Thin Python binding of the C-ABI in include/tf.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libtf_b200.so.  PyTorch supplies device
memory (the workspace, user tensors) and the stream.  There is no fallback: if the library is
missing or cannot be loaded, importing the symbols below raises.
"""
import ctypes
import os

import numpy as np

from . import build as _build

OK, NOT_CONVERGED, REJECTED = 0, 1, 2
ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_CUDA, ERR_ALLOC, ERR_STATE = -1, -2, -3, -4, -5
BC_NOFLUX = 0
PI_POWER, PI_NLC, PI_POLYMER = 0, 2, 3

_dp = ctypes.POINTER(ctypes.c_double)
_vp = ctypes.c_void_p
_lib = None

# every symbol include/tf.h declares: name -> (restype, argtypes)
SYMBOLS = {
    "tf_workspace_bytes": (ctypes.c_size_t, [ctypes.c_int, ctypes.c_int]),
    "tf_create": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                 ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int]),
    "tf_create_with_workspace": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                                ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                                ctypes.c_int, ctypes.c_int, _vp, ctypes.c_size_t, _vp]),
    "tf_destroy": (None, [_vp]),
    "tf_set_newton": (ctypes.c_int, [_vp, ctypes.c_double, ctypes.c_int, ctypes.c_int]),
    "tf_set_pressure": (ctypes.c_int, [_vp, ctypes.c_int, _dp, ctypes.c_int]),
    "tf_set_launch_ahead": (ctypes.c_int, [_vp, ctypes.c_int]),
    "tf_set_cuda_graphs": (ctypes.c_int, [_vp, ctypes.c_int]),
    "tf_graph_replays": (ctypes.c_int, [_vp, ctypes.POINTER(ctypes.c_ulonglong)]),
    "tf_set_solution_criteria": (ctypes.c_int, [_vp, ctypes.c_double]),
    "tf_set_truncation_criterion": (ctypes.c_int, [_vp, ctypes.c_double]),
    "tf_last_truncation_estimate": (ctypes.c_int, [_vp, _dp]),
    "tf_adaptive_run": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int, ctypes.c_int, _dp, _vp, ctypes.c_int,
                                       ctypes.POINTER(ctypes.c_int)]),
    "tf_advance_adaptive": (ctypes.c_int, [_vp, _vp, ctypes.c_int, ctypes.c_int, _dp, _vp, ctypes.c_int,
                                           ctypes.POINTER(ctypes.c_int)]),
    "tf_advance_adaptive_device": (ctypes.c_int, [_vp, _vp, ctypes.c_int, ctypes.c_int, _dp, _vp, ctypes.c_int,
                                                  ctypes.POINTER(ctypes.c_int)]),
    "tf_set_state": (ctypes.c_int, [_vp, _vp, ctypes.c_int]),
    "tf_get_state": (ctypes.c_int, [_vp, _vp, ctypes.c_int]),
    "tf_step": (ctypes.c_int, [_vp, ctypes.c_double, ctypes.POINTER(ctypes.c_int), _dp]),
    "tf_mass": (ctypes.c_int, [_vp, _dp]),
    "tf_field": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.POINTER(_vp)]),
    "tf_sweep": (ctypes.c_int, [_vp, ctypes.c_double, ctypes.c_int, ctypes.c_int]),
    "tf_residual": (ctypes.c_int, [_vp, ctypes.c_int, _dp, ctypes.POINTER(ctypes.c_int)]),
    "tf_accept": (ctypes.c_int, [_vp]),
    "tf_blocks_gather": (ctypes.c_int, [_vp, ctypes.c_int, _vp, ctypes.c_int, _vp, _vp]),
    "tf_blocks_scatter": (ctypes.c_int, [_vp, _vp, ctypes.c_int, _vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp]),
    "tf_record_sanitize": (ctypes.c_int, [_vp, ctypes.c_int]),
    "tf_block_copy": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp]),
    "tf_penta_workspace_bytes": (ctypes.c_size_t, [ctypes.c_int, ctypes.c_int]),
    "tf_penta_solve": (ctypes.c_int, [ctypes.c_int, ctypes.c_int, ctypes.c_int] + [_vp] * 9),
    "tf_penta_static_max_elems": (ctypes.c_size_t, []),
    "tf_penta_solve_static": (ctypes.c_int, [ctypes.c_int, ctypes.c_int, ctypes.c_int] + [_vp] * 8),
    "tf_penta_partition_chunks": (ctypes.c_int, [ctypes.c_int] * 4),
    "tf_penta_slab_interface_doubles": (ctypes.c_size_t, [ctypes.c_int] * 4),
    "tf_penta_slab_workspace_bytes": (ctypes.c_size_t, [ctypes.c_int] * 5),
    "tf_penta_slab_interface": (ctypes.c_int, [ctypes.c_int] * 6 + [_vp] * 8),
    "tf_penta_slab_solve": (ctypes.c_int, [ctypes.c_int] * 6 + [_vp] * 10),
    "tf_betti_workspace_bytes": (ctypes.c_size_t, [ctypes.c_int] * 3),
    "tf_spectrum_workspace_bytes": (ctypes.c_size_t, [ctypes.c_int] * 3),
    "tf_radial_peaks": (ctypes.c_int, [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, _dp, _dp, _dp, ctypes.c_int,
                                       ctypes.POINTER(ctypes.c_int)]),
    "tf_radial_spectrum": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                          ctypes.c_int, _dp, _dp, ctypes.POINTER(ctypes.c_longlong), ctypes.c_int,
                                          ctypes.POINTER(ctypes.c_int), _vp, _vp]),
    "tf_betti": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _dp, ctypes.c_int, ctypes.POINTER(ctypes.c_longlong),
                                ctypes.POINTER(ctypes.c_longlong), _vp, _vp]),
    "tf_penta_workspace_bytes_ex": (ctypes.c_size_t, [ctypes.c_int] * 5),
    "tf_penta_solve_ex": (ctypes.c_int, [ctypes.c_int] * 5 + [_vp] * 9),
    "tf_set_profiling": (ctypes.c_int, [_vp, ctypes.c_int]),
    "tf_get_profile": (ctypes.c_int, [_vp, _dp, ctypes.POINTER(ctypes.c_ulonglong)]),
    "tf_last_error": (ctypes.c_char_p, [_vp]),
    "tf_kernel_launches": (ctypes.c_ulonglong, []),
    "tf_fp64_peak": (ctypes.c_int, [ctypes.c_int, _dp, _dp, _vp]),
}


class TfError(RuntimeError):
    def __init__(self, status, what, text=""):
        super().__init__(f"{what} failed: status {status} {text}")
        self.status = status


def lib():
    """Load libtf_b200.so (building it with nvcc if the sources are newer).  Raises if impossible."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if _build.stale():
            path = _build.build()
        L = ctypes.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)          # AttributeError if a declared symbol is not exported
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _err(handle, status, what):
    text = lib().tf_last_error(handle)
    raise TfError(status, what, text.decode() if text else "")


def kernel_launches():
    return int(lib().tf_kernel_launches())


def fp64_peak(launches=5, stream=None):
    """tf_fp64_peak: (best, mean) thread-level DFMA instructions per second of the current device, measured."""
    torch = _torch()
    best, mean = ctypes.c_double(0.0), ctypes.c_double(0.0)
    st = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
    rc = lib().tf_fp64_peak(int(launches), ctypes.byref(best), ctypes.byref(mean), st)
    if rc != OK:
        _err(None, rc, "tf_fp64_peak")
    return best.value, mean.value


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise TfError(ERR_CUDA, "cuda", "no CUDA device: this package has no CPU path")
    return torch


class ThinFilm:
    """tf_create / tf_set_newton / tf_set_state / tf_step / tf_get_state / tf_mass on one GPU."""

    def __init__(self, nx, ny, dx, dy, kappa=100.0, hstar=0.1, n=3, m=2, bc=BC_NOFLUX, device=None, stream=None):
        torch = _torch()
        L = lib()
        self.nx, self.ny = int(nx), int(ny)
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self._h = _vp()
        nbytes = L.tf_workspace_bytes(self.nx, self.ny)
        with torch.cuda.device(self.device):
            self._ws = torch.empty(max(nbytes, 256) + 256, dtype=torch.uint8, device=self.device)
            base = self._ws.data_ptr()
            off = (-base) % 256
            self._stream = torch.cuda.current_stream(self.device) if stream is None else stream
            st = L.tf_create_with_workspace(ctypes.byref(self._h), self.nx, self.ny, dx, dy, kappa, hstar, n, m, bc,
                                            base + off, nbytes, self._stream.cuda_stream)
        if st != OK:
            self._h = _vp()
            _err(None, st, "tf_create_with_workspace")

    def close(self):
        if getattr(self, "_h", None):
            lib().tf_destroy(self._h)
            self._h = _vp()
            self._ws = None

    def __del__(self):
        try:                       # at interpreter shutdown module globals may already be gone
            self.close()
        except Exception:
            pass

    def set_newton(self, tol=1e-10, max_iter=10, fixed_iters=0):
        st = lib().tf_set_newton(self._h, tol, max_iter, fixed_iters)
        if st != OK:
            _err(self._h, st, "tf_set_newton")

    def set_launch_ahead(self, batch):
        """tf_set_launch_ahead: 0 = host decision after every iteration, > 0 = speculative batches (default 2)."""
        st = lib().tf_set_launch_ahead(self._h, int(batch))
        if st != OK:
            _err(self._h, st, "tf_set_launch_ahead")

    def set_cuda_graphs(self, on=True):
        """tf_set_cuda_graphs: replay recurring launch-ahead batches as CUDA graphs (default on; bit-identical results)."""
        st = lib().tf_set_cuda_graphs(self._h, 1 if on else 0)
        if st != OK:
            _err(self._h, st, "tf_set_cuda_graphs")

    def graph_replays(self):
        n = ctypes.c_ulonglong(0)
        st = lib().tf_graph_replays(self._h, ctypes.byref(n))
        if st != OK:
            _err(self._h, st, "tf_graph_replays")
        return int(n.value)

    def set_solution_criteria(self, max_rel_change=0.0):
        """tf_set_solution_criteria: accept a converged step only if max|u^{n+1}-u^n|/u^n <= max_rel_change (0 = off)."""
        st = lib().tf_set_solution_criteria(self._h, float(max_rel_change))
        if st != OK:
            _err(self._h, st, "tf_set_solution_criteria")

    def set_truncation_criterion(self, max_rel_truncation=0.0):
        """tf_set_truncation_criterion: accept a converged step only if the estimated local truncation error of the
        trapezoidal rule, relative to h, is <= max_rel_truncation (0 = off)."""
        st = lib().tf_set_truncation_criterion(self._h, float(max_rel_truncation))
        if st != OK:
            _err(self._h, st, "tf_set_truncation_criterion")

    def last_truncation_estimate(self):
        v = ctypes.c_double(0.0)
        st = lib().tf_last_truncation_estimate(self._h, ctypes.byref(v))
        if st != OK:
            _err(self._h, st, "tf_last_truncation_estimate")
        return v.value

    def set_pressure(self, kind, params=()):
        """tf_set_pressure: PI_POWER (), PI_NLC (cap0, cap1, K, b, N, beta, w), PI_POLYMER (cap0, cap1, C, A_SiOx, A_Si, d)."""
        arr = (ctypes.c_double * max(len(params), 1))(*[float(v) for v in params])
        st = lib().tf_set_pressure(self._h, int(kind), arr, len(params))
        if st != OK:
            _err(self._h, st, "tf_set_pressure")

    def set_state(self, h):
        """h: torch CUDA float64 tensor [ny][nx] (device copy) or numpy / CPU tensor (host copy)."""
        ptr, is_dev, keep = self._marshal(h, writable=False)
        st = lib().tf_set_state(self._h, ptr, is_dev)
        if st != OK:
            _err(self._h, st, "tf_set_state")

    def get_state(self, out=None):
        """Returns the state: into `out` (torch CUDA tensor or numpy array) or a new numpy array."""
        if out is None:
            out = np.empty((self.ny, self.nx), dtype=np.float64)
        ptr, is_dev, keep = self._marshal(out, writable=True)
        st = lib().tf_get_state(self._h, ptr, is_dev)
        if st != OK:
            _err(self._h, st, "tf_get_state")
        return out

    def step(self, dt):
        """One time step; returns (status, newton_iters, residual).  status 1 = rejected, state unchanged."""
        it, res = ctypes.c_int(0), ctypes.c_double(0.0)
        st = lib().tf_step(self._h, dt, ctypes.byref(it), ctypes.byref(res))
        if st < 0:
            _err(self._h, st, "tf_step")
        return st, it.value, res.value

    # ---- the rows of the path one at a time (tf_field / tf_sweep / tf_residual / tf_accept)
    FIELD_STATE, FIELD_ITERATE, FIELD_BN, FIELD_W, FIELD_RECORDS = 0, 1, 2, 3, 4
    SWEEP_Y, SWEEP_X, SWEEP_GATED = 1, 2, 4

    def field(self, which):
        """a torch view [ny][nx] of a field the context owns (no copy; the addresses of 0 and 1 swap on accept)"""
        torch = _torch()
        p = _vp()
        st = lib().tf_field(self._h, int(which), ctypes.byref(p))
        if st != OK:
            _err(self._h, st, "tf_field")
        n = self.nx * self.ny if which != self.FIELD_RECORDS else 2 * 4096
        if self._ws is not None:
            off = (p.value - self._ws.data_ptr()) // 8
            if 0 <= off and off + n <= self._ws.numel() * self._ws.element_size() // 8:
                v = self._ws.view(torch.float64)[off:off + n]
                return v.view(self.ny, self.nx) if which != self.FIELD_RECORDS else v.view(4096, 2)
        raise TfError(ERR_STATE, "tf_field", "field views need a context created on a torch workspace")

    def sweep(self, dt, k, which):
        st = lib().tf_sweep(self._h, dt, k, which)
        if st != OK:
            _err(self._h, st, "tf_sweep")

    def residual(self, k):
        res, bad = ctypes.c_double(0.0), ctypes.c_int(0)
        st = lib().tf_residual(self._h, k, ctypes.byref(res), ctypes.byref(bad))
        if st != OK:
            _err(self._h, st, "tf_residual")
        return res.value, bool(bad.value)

    def accept(self):
        st = lib().tf_accept(self._h)
        if st != OK:
            _err(self._h, st, "tf_accept")

    def record_sanitize(self, k):
        """tf_record_sanitize: record k ready for a max-reduction over ranks (NaN -> {+inf, bad})."""
        st = lib().tf_record_sanitize(self._h, int(k))
        if st != OK:
            _err(self._h, st, "tf_record_sanitize")

    def mass(self):
        m = ctypes.c_double(0.0)
        st = lib().tf_mass(self._h, ctypes.byref(m))
        if st != OK:
            _err(self._h, st, "tf_mass")
        return m.value

    PROFILE_SLOTS = ("y_forward", "y_backward", "x_forward", "x_backward_update")

    def set_profiling(self, on=True):
        st = lib().tf_set_profiling(self._h, 1 if on else 0)
        if st != OK:
            _err(self._h, st, "tf_set_profiling")

    def get_profile(self):
        """{kernel: (total_ms, launches)} accumulated since set_profiling(True)."""
        ms = (ctypes.c_double * 4)()
        n = (ctypes.c_ulonglong * 4)()
        st = lib().tf_get_profile(self._h, ms, n)
        if st != OK:
            _err(self._h, st, "tf_get_profile")
        return {k: (ms[i], int(n[i])) for i, k in enumerate(self.PROFILE_SLOTS)}

    def _marshal(self, h, writable):
        if isinstance(h, np.ndarray):
            if h.dtype != np.float64 or not h.flags["C_CONTIGUOUS"] or h.shape != (self.ny, self.nx):
                if writable:
                    raise ValueError("output must be a C-contiguous float64 [ny][nx] array")
                h = np.ascontiguousarray(h, dtype=np.float64)
                if h.shape != (self.ny, self.nx):
                    raise ValueError(f"expected shape {(self.ny, self.nx)}, got {h.shape}")
            return h.ctypes.data, 0, h
        torch = _torch()
        if not isinstance(h, torch.Tensor):
            raise TypeError("expected numpy array or torch tensor")
        if h.dtype != torch.float64 or not h.is_contiguous() or tuple(h.shape) != (self.ny, self.nx):
            raise ValueError("expected a contiguous float64 [ny][nx] tensor")
        return h.data_ptr(), (1 if h.is_cuda else 0), h


class _Rect(ctypes.Structure):
    _fields_ = [("row0", ctypes.c_int), ("nrows", ctypes.c_int), ("col0", ctypes.c_int), ("ncols", ctypes.c_int),
                ("offset", ctypes.c_longlong)]


def make_rects(blocks):
    """[(row0, nrows, col0, ncols, offset), ...] -> the tf_rect array tf_blocks_gather / tf_blocks_scatter take"""
    arr = (_Rect * len(blocks))()
    for k, b in enumerate(blocks):
        arr[k] = _Rect(*[int(v) for v in b])
    return arr


def blocks_gather(field, rects, buf, stream=None):
    """tf_blocks_gather: every block of the 2-D CUDA tensor `field` into the flat send buffer `buf` (one kernel)."""
    torch = _torch()
    assert field.is_cuda and buf.is_cuda and field.dtype == buf.dtype == torch.float64 and field.stride(1) == 1
    stream = torch.cuda.current_stream(field.device) if stream is None else stream
    st = lib().tf_blocks_gather(field.data_ptr(), field.stride(0), rects, len(rects), buf.data_ptr(), stream.cuda_stream)
    if st != OK:
        _err(None, st, "tf_blocks_gather")


def blocks_scatter(buf, rects, field, reflect_left=False, reflect_right_at=-1, stream=None):
    """tf_blocks_scatter: the receive buffer into `field`, ghost columns of (2.28) filled in the same pass."""
    torch = _torch()
    assert field.is_cuda and buf.is_cuda and field.dtype == buf.dtype == torch.float64 and field.stride(1) == 1
    stream = torch.cuda.current_stream(field.device) if stream is None else stream
    st = lib().tf_blocks_scatter(buf.data_ptr(), rects, len(rects), field.data_ptr(), field.stride(0),
                                 1 if reflect_left else 0, int(reflect_right_at), stream.cuda_stream)
    if st != OK:
        _err(None, st, "tf_blocks_scatter")


def block_copy(src, srow0, scol0, dst, drow0, dcol0, nrows, ncols, reflect_left=False, reflect_right_at=-1, stream=None):
    """tf_block_copy: one block from the 2-D CUDA tensor `src` straight into `dst` (ghost columns as in blocks_scatter)."""
    torch = _torch()
    assert src.is_cuda and dst.is_cuda and src.dtype == dst.dtype == torch.float64 and src.stride(1) == dst.stride(1) == 1
    stream = torch.cuda.current_stream(src.device) if stream is None else stream
    st = lib().tf_block_copy(src.data_ptr(), src.stride(0), int(srow0), int(scol0), dst.data_ptr(), dst.stride(0), int(drow0),
                             int(dcol0), int(nrows), int(ncols), 1 if reflect_left else 0, int(reflect_right_at),
                             stream.cuda_stream)
    if st != OK:
        _err(None, st, "tf_block_copy")


class _Adaptive(ctypes.Structure):
    _fields_ = [("dt", ctypes.c_double), ("shrink", ctypes.c_double), ("grow", ctypes.c_double),
                ("grow_after", ctypes.c_int), ("dt_min", ctypes.c_double), ("dt_max", ctypes.c_double)]


class _StepRecord(ctypes.Structure):
    _fields_ = [("dt", ctypes.c_double), ("status", ctypes.c_int), ("newton_iters", ctypes.c_int),
                ("residual", ctypes.c_double)]


_STEP_FN = ctypes.CFUNCTYPE(ctypes.c_int, _vp, ctypes.c_double, ctypes.POINTER(ctypes.c_int), _dp)


def advance_adaptive(ctx, dt, n_accept, grow=1.1, shrink=0.5, dt_max=0.1, dt_min=1e-12, max_attempts=None, grow_after=1,
                     on_device=False, return_status=False):
    """Adaptive time stepping of Fig. 1 until `n_accept` steps were accepted: tf_advance_adaptive
    for a ThinFilm, tf_adaptive_run (the same controller, driven through a callback) for any object with a
    step(dt) -> (status, newton_iters, residual) method.  The controller itself is in the library; this marshals.
    on_device=True: tf_advance_adaptive_device, the same controller with its decisions taken on the device.
    Returns (t, dt_next, history) with history = [(dt, status, newton_iters, residual), ...]; with return_status=True a
    fourth value, the status, is returned and a soft failure (dt below dt_min, attempt cap) does not raise."""
    L = lib()
    ctl = _Adaptive(float(dt), float(shrink), float(grow), int(grow_after), float(dt_min), float(dt_max))
    cap = int(max_attempts or 50 * max(n_accept, 1))
    hist = (_StepRecord * cap)()
    nh, t = ctypes.c_int(0), ctypes.c_double(0.0)
    if isinstance(ctx, ThinFilm):
        run = L.tf_advance_adaptive_device if on_device else L.tf_advance_adaptive
        st = run(ctx._h, ctypes.byref(ctl), n_accept, cap, ctypes.byref(t), hist, cap, ctypes.byref(nh))
        handle = ctx._h
    else:
        def cb(_user, dt_, it_p, res_p):
            s_, it_, res_ = ctx.step(dt_)
            it_p[0], res_p[0] = int(it_), float(res_)
            return int(s_)
        fn = _STEP_FN(cb)
        st = L.tf_adaptive_run(ctypes.cast(fn, _vp), None, ctypes.byref(ctl), n_accept, cap, ctypes.byref(t), hist, cap,
                               ctypes.byref(nh))
        handle = None
    if st != OK and not (return_status and st == NOT_CONVERGED):
        _err(handle, st, "advance_adaptive")
    out = [(hist[k].dt, hist[k].status, hist[k].newton_iters, hist[k].residual) for k in range(min(nh.value, cap))]
    return (t.value, ctl.dt, out, st) if return_status else (t.value, ctl.dt, out)


PENTA_LU, PENTA_PARTITION, PENTA_PCR = 0, 1, 2


def penta_partition_chunks(nrow, ncol, direction, nparts=0):
    """tf_penta_partition_chunks: chunks per system the partition variant will use for this shape (1 = LU)."""
    return lib().tf_penta_partition_chunks(nrow, ncol, direction, nparts)


def penta_solve(direction, e, c, d, a, b, rhs, out=None, workspace=None, stream=None, variant=PENTA_LU, nparts=0):
    """tf_penta_solve_ex on torch CUDA float64 tensors [nrow][ncol]; direction 0: rows are systems, 1: columns.
    variant PENTA_LU (thread per system) or PENTA_PARTITION (nparts chunks per system, 0 = automatic).
    Enqueues on the current stream and returns `out` without synchronising."""
    torch = _torch()
    ts = (e, c, d, a, b, rhs)
    nrow, ncol = e.shape
    for t in ts:
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and tuple(t.shape) == (nrow, ncol)):
            raise ValueError("expected contiguous CUDA float64 tensors of one shape")
    if out is None:
        out = torch.empty_like(e)
    L = lib()
    need = L.tf_penta_workspace_bytes_ex(nrow, ncol, direction, variant, nparts)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=e.device)
    if workspace.numel() * workspace.element_size() < need or workspace.data_ptr() % 256:
        raise ValueError("workspace too small or not 256-byte aligned")
    st = (torch.cuda.current_stream(e.device) if stream is None else stream).cuda_stream
    rc = L.tf_penta_solve_ex(nrow, ncol, direction, variant, nparts, *[t.data_ptr() for t in ts], out.data_ptr(),
                             workspace.data_ptr(), st)
    if rc != OK:
        _err(None, rc, "tf_penta_solve_ex")
    return out


def penta_static_max_elems():
    """tf_penta_static_max_elems: the largest nrow * ncol that penta_solve_static accepts."""
    return int(lib().tf_penta_static_max_elems())


def penta_solve_static(direction, e, c, d, a, b, rhs, out, stream=None):
    """tf_penta_solve_static: penta_solve for a caller that may not allocate device memory when it calls -- all of
    HBM already belongs to its own pool, or a cudaMalloc would stall its other streams, or its host application forbids
    allocations after start-up.  The scratch is a fixed 24 MiB array inside libtf_b200.so, so this binding allocates
    nothing either: `out` must be passed in.  nrow * ncol <= penta_static_max_elems(), else TfError (ERR_INVALID_ARG).
    The first call on a device does one-time set-up.  All calls on a device share the one scratch array: keep them on
    one stream (or order them), calls that overlap on the GPU corrupt each other.  Same kernels and bits as penta_solve.
    The tensors must live on the current device.  Enqueues and returns `out` without synchronising."""
    torch = _torch()
    ts = (e, c, d, a, b, rhs, out)
    nrow, ncol = e.shape
    for t in ts:
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and tuple(t.shape) == (nrow, ncol)):
            raise ValueError("expected contiguous CUDA float64 tensors of one shape")
    st = (torch.cuda.current_stream(e.device) if stream is None else stream).cuda_stream
    rc = lib().tf_penta_solve_static(nrow, ncol, direction, *[t.data_ptr() for t in ts], st)
    if rc != OK:
        _err(None, rc, "tf_penta_solve_static")
    return out


def betti(h, thresholds, workspace=None, stream=None):
    """tf_betti on a contiguous CUDA float64 [ny][nx] tensor: (b0, b1) int64 numpy arrays, one entry per threshold
    (superlevel sets {h > H*}: components, and holes that do not reach the border)."""
    torch = _torch()
    if not (isinstance(h, torch.Tensor) and h.is_cuda and h.dtype == torch.float64 and h.is_contiguous() and h.dim() == 2):
        raise ValueError("expected a contiguous CUDA float64 [ny][nx] tensor")
    ny, nx = h.shape
    thr = np.ascontiguousarray(np.atleast_1d(thresholds), dtype=np.float64)
    L = lib()
    need = L.tf_betti_workspace_bytes(nx, ny, len(thr))
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=h.device)
    if workspace.numel() * workspace.element_size() < need or workspace.data_ptr() % 256:
        raise ValueError("workspace too small or not 256-byte aligned")
    b0 = np.zeros(len(thr), dtype=np.int64)
    b1 = np.zeros(len(thr), dtype=np.int64)
    lp = ctypes.POINTER(ctypes.c_longlong)
    st = (torch.cuda.current_stream(h.device) if stream is None else stream).cuda_stream
    rc = L.tf_betti(h.data_ptr(), nx, ny, thr.ctypes.data_as(_dp), len(thr), b0.ctypes.data_as(lp), b1.ctypes.data_as(lp),
                    workspace.data_ptr(), st)
    if rc != OK:
        _err(None, rc, "tf_betti")
    return b0, b1


def radial_spectrum(h, L, H0, sigma, kmax, workspace=None, stream=None):
    """tf_radial_spectrum (App. B steps 1-4) on a contiguous CUDA float64 [ny][nx] tensor of a square domain of side L:
    returns numpy arrays (q_r, mean magnitude, N_k) over the distinct radii up to kmax index units."""
    torch = _torch()
    if not (isinstance(h, torch.Tensor) and h.is_cuda and h.dtype == torch.float64 and h.is_contiguous() and h.dim() == 2):
        raise ValueError("expected a contiguous CUDA float64 [ny][nx] tensor")
    ny, nx = h.shape
    Lb = lib()
    need = Lb.tf_spectrum_workspace_bytes(nx, ny, kmax)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=h.device)
    if workspace.numel() * workspace.element_size() < need or workspace.data_ptr() % 256:
        raise ValueError("workspace too small or not 256-byte aligned")
    cap = kmax * kmax + 1
    q = np.zeros(cap)
    z = np.zeros(cap)
    cnt = np.zeros(cap, dtype=np.int64)
    nk = ctypes.c_int(0)
    st = (torch.cuda.current_stream(h.device) if stream is None else stream).cuda_stream
    rc = Lb.tf_radial_spectrum(h.data_ptr(), nx, ny, float(L), float(H0), float(sigma), int(kmax), q.ctypes.data_as(_dp),
                               z.ctypes.data_as(_dp), cnt.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)), cap,
                               ctypes.byref(nk), workspace.data_ptr(), st)
    if rc != OK:
        _err(None, rc, "tf_radial_spectrum")
    m = min(nk.value, cap)
    return q[:m], z[:m], cnt[:m]


def radial_peaks(q, zeta, per_interval=10, ngrid=400, max_peaks=64):
    """tf_radial_peaks (App. B steps 5-6 and the maxima; host only): returns (grid, smoothed spectrum, [(q, value), ...])."""
    q = np.ascontiguousarray(q, dtype=np.float64)
    z = np.ascontiguousarray(zeta, dtype=np.float64)
    g, f = np.zeros(ngrid), np.zeros(ngrid)
    pq, pz = np.zeros(max_peaks), np.zeros(max_peaks)
    n = ctypes.c_int(0)
    rc = lib().tf_radial_peaks(q.ctypes.data_as(_dp), z.ctypes.data_as(_dp), len(q), per_interval, ngrid, g.ctypes.data_as(_dp),
                               f.ctypes.data_as(_dp), pq.ctypes.data_as(_dp), pz.ctypes.data_as(_dp), max_peaks, ctypes.byref(n))
    if rc != OK:
        _err(None, rc, "tf_radial_peaks")
    m = min(n.value, max_peaks)
    return g, f, list(zip(pq[:m].tolist(), pz[:m].tolist()))


def _check_six(ts):
    torch = _torch()
    nrow, ncol = ts[0].shape
    for t in ts:
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and tuple(t.shape) == (nrow, ncol)):
            raise ValueError("expected contiguous CUDA float64 tensors of one shape")
    return nrow, ncol


def penta_slab_interface(direction, nparts, slab, nslabs, e, c, d, a, b, rhs, stream=None):
    """tf_penta_slab_interface on the local slab [nrow][ncol]: returns the local interface values, a CUDA float64 tensor
    of shape [nparts, 2, 10, nsys] (nsys = ncol for direction 1, nrow for direction 0)."""
    torch = _torch()
    ts = (e, c, d, a, b, rhs)
    nrow, ncol = _check_six(ts)
    L = lib()
    if L.tf_penta_slab_interface_doubles(nrow, ncol, direction, nparts) == 0:
        raise ValueError("shape not admitted by the slab solver (see include/tf.h)")
    nsys = ncol if direction == 1 else nrow
    out = torch.empty((nparts, 2, 10, nsys), dtype=torch.float64, device=e.device)
    st = (torch.cuda.current_stream(e.device) if stream is None else stream).cuda_stream
    rc = L.tf_penta_slab_interface(nrow, ncol, direction, nparts, slab, nslabs, *[t.data_ptr() for t in ts], out.data_ptr(), st)
    if rc != OK:
        _err(None, rc, "tf_penta_slab_interface")
    return out


def penta_slab_solve(direction, nparts, slab, nslabs, e, c, d, a, b, rhs, iface_all, out=None, workspace=None, stream=None):
    """tf_penta_slab_solve: iface_all = the interface values of all slabs in slab order, [nslabs * nparts, 2, 10, nsys]."""
    torch = _torch()
    ts = (e, c, d, a, b, rhs)
    nrow, ncol = _check_six(ts)
    nsys = ncol if direction == 1 else nrow
    if not (iface_all.is_cuda and iface_all.dtype == torch.float64 and iface_all.is_contiguous()
            and iface_all.numel() == nslabs * nparts * 20 * nsys):
        raise ValueError("iface_all must be a contiguous CUDA float64 tensor of nslabs * nparts * 20 * nsys values")
    L = lib()
    need = L.tf_penta_slab_workspace_bytes(nrow, ncol, direction, nparts, nslabs)
    if need == 0:
        raise ValueError("shape not admitted by the slab solver (see include/tf.h)")
    if out is None:
        out = torch.empty_like(e)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=e.device)
    if workspace.numel() * workspace.element_size() < need or workspace.data_ptr() % 256:
        raise ValueError("workspace too small or not 256-byte aligned")
    st = (torch.cuda.current_stream(e.device) if stream is None else stream).cuda_stream
    rc = L.tf_penta_slab_solve(nrow, ncol, direction, nparts, slab, nslabs, *[t.data_ptr() for t in ts], iface_all.data_ptr(),
                               out.data_ptr(), workspace.data_ptr(), st)
    if rc != OK:
        _err(None, rc, "tf_penta_slab_solve")
    return out

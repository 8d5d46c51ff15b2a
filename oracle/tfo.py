"""ctypes binding of the CPU oracle (oracle/tfo.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from the CUDA package.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tfo.c")
OK, NOT_CONVERGED = 0, 1


def build(force=False):
    """Compile tfo.c with gcc: libtfo.so (serial) and libtfo_omp.so (-fopenmp)."""
    outs = []
    for name, extra in (("libtfo.so", []), ("libtfo_omp.so", ["-fopenmp"])):
        out = os.path.join(_HERE, name)
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
            subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-std=c11", "-fPIC", "-shared",
                                   *extra, "-o", out, _SRC, "-lm"])
        outs.append(out)
    return outs


_libs = {}
_dp = ctypes.POINTER(ctypes.c_double)


def _declare(L):
    """ctypes signatures of the tfo_* entry points (also used by tests that load a mutated build of tfo.c)."""
    L.tfo_create.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.c_int, ctypes.c_double,
                             ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                             ctypes.c_int]
    L.tfo_set_model_linear.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_double]
    L.tfo_set_pressure.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, ctypes.c_int]
    L.tfo_pressure.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, _dp]
    L.tfo_cell_functions.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, _dp, _dp, _dp, _dp]
    L.tfo_set_newton.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_int, ctypes.c_int]
    L.tfo_set_state.argtypes = [ctypes.c_void_p, _dp]
    L.tfo_get_state.argtypes = [ctypes.c_void_p, _dp]
    L.tfo_step.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.POINTER(ctypes.c_int), _dp]
    L.tfo_mass.argtypes = [ctypes.c_void_p, _dp]
    L.tfo_destroy.argtypes = [ctypes.c_void_p]
    L.tfo_destroy.restype = None
    L.tfo_operator_D.argtypes = [ctypes.c_void_p, _dp, _dp]
    L.tfo_jacobian_bands.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, _dp, _dp, _dp, _dp, _dp]
    L.tfo_directional_solve.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, _dp, _dp, _dp]
    L.tfo_penta_solve.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int] + [_dp] * 7
    return L


def lib(omp=False):
    key = bool(omp)
    if key not in _libs:
        build()
        _libs[key] = _declare(ctypes.CDLL(os.path.join(_HERE, "libtfo_omp.so" if omp else "libtfo.so")))
    return _libs[key]


def _p(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


class OracleError(RuntimeError):
    pass


def _chk(rc, what):
    if rc < 0:
        raise OracleError(f"{what} failed with status {rc}")
    return rc


class ThinFilmOracle:
    """Same call names as the CUDA binding (create/set_newton/set_state/step/get_state/mass)."""

    def __init__(self, nx, ny, dx, dy, kappa=100.0, hstar=0.1, n=3, m=2, bc=0, omp=False, library=None):
        self.L = library if library is not None else lib(omp)   # library: a mutated build (tests/mutation_sweep.py)
        self.nx, self.ny = nx, ny
        self._h = ctypes.c_void_p()
        _chk(self.L.tfo_create(ctypes.byref(self._h), nx, ny, dx, dy, kappa, hstar, n, m, bc), "tfo_create")

    def close(self):
        if self._h:
            self.L.tfo_destroy(self._h)
            self._h = ctypes.c_void_p()

    __del__ = close

    def set_model_linear(self, c0, c1):
        _chk(self.L.tfo_set_model_linear(self._h, c0, c1), "tfo_set_model_linear")

    def set_pressure(self, kind, params):
        """kind 2: NLC (1.8)-(1.9), params (cap0, cap1, K, b, N, beta, w); kind 3: polymer (1.12), params
        (cap0, cap1, C, A_SiOx, A_Si, d).  f0 = cap0 h^3, f1 = cap1 h^3 Pi'(h)."""
        p = np.ascontiguousarray(params, dtype=np.float64)
        _chk(self.L.tfo_set_pressure(self._h, int(kind), _p(p), int(p.size)), "tfo_set_pressure")

    def pressure(self, h):
        h = np.ascontiguousarray(h, dtype=np.float64).ravel()
        out = np.empty_like(h)
        _chk(self.L.tfo_pressure(self._h, h.size, _p(h), _p(out)), "tfo_pressure")
        return out

    def cell_functions(self, h):
        h = np.ascontiguousarray(h, dtype=np.float64).ravel()
        outs = [np.empty_like(h) for _ in range(4)]
        _chk(self.L.tfo_cell_functions(self._h, h.size, _p(h), *[_p(o) for o in outs]), "tfo_cell_functions")
        return outs   # f0, f1, f0', f1'

    def set_newton(self, tol=1e-10, max_iter=10, fixed_iters=0):
        _chk(self.L.tfo_set_newton(self._h, tol, max_iter, fixed_iters), "tfo_set_newton")

    def set_state(self, h):
        h = np.ascontiguousarray(h, dtype=np.float64)
        assert h.shape == (self.ny, self.nx)
        _chk(self.L.tfo_set_state(self._h, _p(h)), "tfo_set_state")

    def get_state(self):
        out = np.empty((self.ny, self.nx))
        _chk(self.L.tfo_get_state(self._h, _p(out)), "tfo_get_state")
        return out

    def step(self, dt):
        """Returns (status, newton_iters, residual); status 0 = accepted, 1 = rejected (state unchanged)."""
        it, res = ctypes.c_int(0), ctypes.c_double(0.0)
        rc = _chk(self.L.tfo_step(self._h, dt, ctypes.byref(it), ctypes.byref(res)), "tfo_step")
        return rc, it.value, res.value

    def mass(self):
        m = ctypes.c_double(0.0)
        _chk(self.L.tfo_mass(self._h, ctypes.byref(m)), "tfo_mass")
        return m.value

    # pieces for pins / per-kernel parity
    def operator_D(self, h):
        h = np.ascontiguousarray(h, dtype=np.float64)
        D = np.empty_like(h)
        _chk(self.L.tfo_operator_D(self._h, _p(h), _p(D)), "tfo_operator_D")
        return D

    def jacobian_bands(self, direction, h):
        h = np.ascontiguousarray(h, dtype=np.float64)
        out = [np.zeros_like(h) for _ in range(5)]
        _chk(self.L.tfo_jacobian_bands(self._h, direction, _p(h), *[_p(o) for o in out]), "tfo_jacobian_bands")
        return out

    def directional_solve(self, direction, s, uk, rhs):
        uk = np.ascontiguousarray(uk, dtype=np.float64)
        rhs = np.ascontiguousarray(rhs, dtype=np.float64)
        out = np.empty_like(uk)
        _chk(self.L.tfo_directional_solve(self._h, direction, s, _p(uk), _p(rhs), _p(out)), "tfo_directional_solve")
        return out


def penta_solve(direction, e, c, d, a, b, rhs, omp=False):
    """Batched pentadiagonal solve on [nrow][ncol] arrays; direction 0: rows are systems, 1: columns."""
    arrs = [np.ascontiguousarray(t, dtype=np.float64) for t in (e, c, d, a, b, rhs)]
    nrow, ncol = arrs[0].shape
    x = np.zeros_like(arrs[0])
    _chk(lib(omp).tfo_penta_solve(nrow, ncol, direction, *[_p(t) for t in arrs], _p(x)), "tfo_penta_solve")
    return x


def num_threads(omp=False):
    return int(lib(omp).tfo_num_threads())


# ---------------------------------------------------------------------------------------------------------------
# Fig. 1, written out step by step.  "If the solution criteria are not met, then the time-step is
# reduced and the pseudo-Newton iterative scheme is performed with the new reduced time step.  Furthermore, if the new
# reduced time step is below some minimum, the numerical scheme halts and ends in a failed state. ... the time step is
# increased if a minimum number of successful time steps have been consecutively computed. ... the time step is bounded
# from above."  The paper gives no constants (R13); they are arguments.
# ---------------------------------------------------------------------------------------------------------------
REJECTED = 2


def max_rel_change(u_old, u_new):
    """The one extra solution criterion the build offers (PAPER.md:252 Note 2 leaves them open; R21):
    max over the grid of |u^{n+1} - u^n| / u^n."""
    return float(np.max(np.abs(np.asarray(u_new) - np.asarray(u_old)) / np.asarray(u_old)))


class CriteriaStepper:
    """step(dt) of a ThinFilmOracle with the extra criterion: a converged step whose max_rel_change exceeds
    `limit` is undone (state back to u^n) and reported as REJECTED."""
    def __init__(self, oracle, limit):
        self.o, self.limit, self.last_change = oracle, limit, None

    def step(self, dt):
        before = self.o.get_state()
        st, it, res = self.o.step(dt)
        if st == OK and self.limit > 0:
            self.last_change = max_rel_change(before, self.o.get_state())
            if not (self.last_change <= self.limit):
                self.o.set_state(before)
                st = REJECTED
        return st, it, res


class TruncationStepper:
    """step(dt) of a ThinFilmOracle with the criterion PAPER.md:252 Note 2 names ("sufficiently small truncation
    error"), reading R25 of DESIGN.md, written out step by step:
        u_t^n     = -D(u^n)                                     (the equation, PAPER.md:134 (2.1), with the oracle's D)
        u_t^{n+1} = 2 (u^{n+1} - u^n)/dt - u_t^n                (the trapezoidal rule (2.14) solved for u_t^{n+1})
        a_{n+1/2} = (u_t^{n+1} - u_t^n)/dt                      (second time derivative at the middle of the step)
        u_ttt     = (a_{n+1/2} - a_{n-1/2}) / ((dt + dt_prev)/2)
        estimate  = max (dt^3/12) |u_ttt| / |u^{n+1}|           (local error of the trapezoidal rule, relative to h)
    A converged step whose estimate exceeds `limit` is undone (REJECTED); the first step has no a_{n-1/2} and is not
    tested.  a_{n-1/2} is only replaced when a step is accepted."""
    def __init__(self, oracle, limit):
        self.o, self.limit, self.a_prev, self.dt_prev, self.last = oracle, limit, None, None, 0.0

    def step(self, dt):
        before = self.o.get_state()
        st, it, res = self.o.step(dt)
        if st != OK:
            return st, it, res
        after = self.o.get_state()
        ut0 = -self.o.operator_D(before)
        ut1 = 2.0 * (after - before) / dt - ut0
        a = (ut1 - ut0) / dt
        if self.a_prev is not None:
            uttt = (a - self.a_prev) / (0.5 * (dt + self.dt_prev))
            self.last = float(np.max(dt ** 3 / 12.0 * np.abs(uttt) / np.abs(after)))
            if self.limit > 0 and not (self.last <= self.limit):
                self.o.set_state(before)
                return REJECTED, it, res
        self.a_prev, self.dt_prev = a, dt
        return st, it, res


def advance_adaptive(stepper, dt, n_accept, grow, shrink, dt_max, dt_min, grow_after=1, max_attempts=None):
    """Flow chart of Fig. 1 over any object with step(dt) -> (status, iters, residual).  Returns
    (t, dt_next, history, failed) with history = [(dt, status, iters, residual), ...]."""
    t, hist, accepted, streak, attempts = 0.0, [], 0, 0, 0
    dt = min(dt, dt_max)                                  # "bounded from above"
    max_attempts = max_attempts or 50 * max(n_accept, 1)
    while accepted < n_accept:
        if attempts >= max_attempts:
            return t, dt, hist, True
        attempts += 1
        st, it, res = stepper.step(dt)
        hist.append((dt, st, it, res))
        if st == OK:                                      # solution criteria met: accept
            accepted += 1
            t += dt
            streak += 1
            if streak >= grow_after:                      # "a minimum number of successful time steps ... consecutively"
                dt = min(dt * grow, dt_max)
                streak = 0
        else:                                             # not met: reduce the time step and redo
            streak = 0
            dt = dt * shrink
            if dt < dt_min:                               # "halts and ends in a failed state"
                return t, dt, hist, True
    return t, dt, hist, False

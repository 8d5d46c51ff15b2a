"""tf_penta_solve_static: the isolated pentadiagonal solve for callers that cannot allocate device memory.

Who that is: a process that handed all free HBM to its own pool at start-up (a later cudaMalloc simply fails), a
latency-bound loop that cannot afford the device-wide synchronisation of cudaMalloc / cudaFree, a plug-in whose host
forbids CUDA allocations after initialisation.  tf_penta_solve asks such a caller for three scratch arrays it cannot
supply; tf_penta_solve_static keeps them in a fixed 24 MiB array inside libtf_b200.so instead and accepts systems of
up to tf_penta_static_max_elems() = 2^20 unknowns in total.

This file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide the rest of the suite.  It passes alone in a fresh process (the first call then does the one-time
set-up) and after all other tests (the kernels' attributes are then already set and the array was never touched)."""
import ctypes

import pytest

from paper_1806_10550_b200 import inputs, tf as _tf


def test_shapes_beyond_the_built_in_scratch_are_refused_without_a_device():
    """The size check comes before any CUDA call, so it can be exercised on a machine with no GPU."""
    L = _tf.lib()
    cap = L.tf_penta_static_max_elems()
    assert cap == 1 << 20
    fake = [ctypes.c_void_p(256)] * 7                      # never dereferenced: the call is refused first
    assert L.tf_penta_solve_static(1025, 1024, 0, *fake, None) == _tf.ERR_INVALID_ARG
    msg = L.tf_last_error(None).decode()
    assert "TF_PENTA_STATIC_MAX_ELEMS" in msg and str(cap) in msg and str(1025 * 1024) in msg
    assert L.tf_penta_solve_static(46341, 46341, 1, *fake, None) == _tf.ERR_INVALID_ARG   # product overflows 32 bits
    assert L.tf_penta_solve_static(64, 64, 2, *fake, None) == _tf.ERR_INVALID_ARG
    assert L.tf_penta_solve_static(64, 64, 0, *([None] * 7), None) == _tf.ERR_INVALID_ARG


@pytest.mark.gpu
def test_two_calls_in_a_row_equal_the_caller_workspace_path():
    """Two calls back to back on the shared array -- different data, different shape, different direction, so the
    second call finds the first one's factors lying in its scratch -- each against tf_penta_solve with a workspace the
    caller allocated.  Same kernels on the same inputs: the suite's tolerance for this solver (1e-12, relative to
    max |x|) is asserted, and bit equality on top of it.  A third call repeats the first and must reproduce it."""
    import torch
    torch.cuda.init()
    cases = [(0, 250, 254, 11), (1, 1000, 66, 12), (0, 1024, 1024, 13), (1, 33, 70, 14)]   # TMA path, ragged, the limit, fallback path
    first = None
    for direction, nrow, ncol, seed in cases + cases[:1]:
        dev = [torch.from_numpy(t).cuda() for t in inputs.penta_system(nrow, ncol, seed=seed)]
        want = _tf.penta_solve(direction, *dev)                                # existing path, torch-allocated workspace
        got = torch.full_like(dev[0], float("nan"))
        _tf.penta_solve_static(direction, *dev, out=got)
        torch.cuda.synchronize()
        assert torch.isfinite(got).all()
        assert float((got - want).abs().max() / want.abs().max()) <= 1e-12
        assert torch.equal(got, want)
        if first is None:
            first = got.clone()
    assert torch.equal(got, first)
    with pytest.raises(_tf.TfError) as ei:                                     # one element over the limit
        big = [torch.empty(1025, 1024, dtype=torch.float64, device="cuda") for _ in range(7)]
        _tf.penta_solve_static(0, *big[:6], out=big[6])
    assert ei.value.status == _tf.ERR_INVALID_ARG and "TF_PENTA_STATIC_MAX_ELEMS" in str(ei.value)

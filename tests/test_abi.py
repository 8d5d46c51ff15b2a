"""No-GPU checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/tf.h declares; argument validation that needs no device."""
import ctypes
import os
import re

from paper_1806_10550_b200 import tf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "tf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return set(re.findall(r"\b(tf_[a-z0-9_]+)\s*\(", src))


def test_library_exports_every_declared_symbol():
    L = tf.lib()
    decl = declared_symbols()
    assert decl == set(tf.SYMBOLS), (decl ^ set(tf.SYMBOLS))
    for name in decl:
        assert hasattr(L, name), name


def test_workspace_sizes_and_host_side_validation():
    L = tf.lib()
    assert L.tf_workspace_bytes(4, 128) == 0
    n = L.tf_workspace_bytes(128, 128)
    assert n >= 7 * 128 * 128 * 8 and n % 256 == 0
    assert L.tf_penta_workspace_bytes(64, 32) >= 3 * 64 * 32 * 8
    h = ctypes.c_void_p()
    # invalid arguments are rejected before any device work
    assert L.tf_create(ctypes.byref(h), 3, 128, 0.1, 0.1, 100.0, 0.1, 3, 2, 0) == tf.ERR_INVALID_ARG
    assert L.tf_create(ctypes.byref(h), 128, 128, 0.1, 0.1, 100.0, 0.1, 2, 3, 0) == tf.ERR_INVALID_ARG
    assert L.tf_create(ctypes.byref(h), 128, 128, -0.1, 0.1, 100.0, 0.1, 3, 2, 0) == tf.ERR_INVALID_ARG
    assert L.tf_create(ctypes.byref(h), 128, 128, 0.1, 0.1, 100.0, 0.1, 3, 2, 1) == tf.ERR_UNSUPPORTED
    assert b"2.28" in L.tf_last_error(None)
    assert L.tf_penta_solve(8, 8, 2, *([None] * 9)) == tf.ERR_INVALID_ARG
    # partition variant: chunk count and workspace are pure host functions of the shape
    assert L.tf_penta_partition_chunks(256, 16384, 0, 0) >= 16          # few long systems: many chunks
    assert L.tf_penta_partition_chunks(16384, 16384, 0, 0) == 1         # config 4 itself: thread per line fills the GPU
    assert L.tf_penta_partition_chunks(64, 100, 0, 0) == 1 and L.tf_penta_partition_chunks(33, 400, 0, 4) == 1
    assert L.tf_penta_partition_chunks(64, 512, 0, 4) == 4 and L.tf_penta_partition_chunks(512, 64, 1, 4) == 4
    assert L.tf_penta_partition_chunks(64, 512, 0, 100) == 5            # clamped: chunks keep >= 81 rows
    assert L.tf_penta_workspace_bytes_ex(64, 512, 0, tf.PENTA_LU, 4) == L.tf_penta_workspace_bytes(64, 512)
    assert L.tf_penta_workspace_bytes_ex(64, 512, 0, tf.PENTA_PARTITION, 4) >= \
        L.tf_penta_workspace_bytes(64, 512) + 4 * 36 * 64 * 8
    assert L.tf_penta_solve_ex(8, 8, 0, 7, 0, *([None] * 9)) == tf.ERR_INVALID_ARG
    # analysis and slab entry points validate their arguments before any device work
    import numpy as np
    one = (ctypes.c_double * 1)(float("nan"))
    ll = (ctypes.c_longlong * 1)()
    assert L.tf_betti_workspace_bytes(0, 8, 1) == 0 and L.tf_betti_workspace_bytes(64, 64, 3) >= 64 * 64 * 5
    assert L.tf_betti(None, 8, 8, one, 1, ll, ll, None, None) == tf.ERR_INVALID_ARG
    assert L.tf_spectrum_workspace_bytes(64, 64, 10) >= 3 * 64 * 64 * 8 and L.tf_spectrum_workspace_bytes(1, 64, 10) == 0
    assert L.tf_radial_spectrum(None, 64, 64, 1.0, 1.0, 1.0, 10, None, None, None, 0, None, None, None) == tf.ERR_INVALID_ARG
    assert L.tf_penta_slab_interface_doubles(64, 512, 0, 4) == 4 * 20 * 64
    assert L.tf_penta_slab_interface_doubles(64, 100, 0, 4) == 0                     # chunks would be shorter than 96
    assert L.tf_penta_slab_workspace_bytes(512, 64, 1, 2, 3) >= 3 * 512 * 64 * 8 + 6 * 16 * 64 * 8
    assert L.tf_penta_slab_interface(64, 512, 0, 4, 5, 3, *([None] * 8)) == tf.ERR_INVALID_ARG   # slab index >= nslabs
    q = np.linspace(0.1, 5.0, 50)
    g, f, peaks = tf.radial_peaks(q, np.exp(-(q - 2.0) ** 2))                          # host-only entry point works without a GPU
    assert len(g) == 400 and abs(max(peaks, key=lambda p: p[1])[0] - 2.0) < 0.1
    assert L.tf_kernel_launches() == 0


def test_product_path_does_not_touch_the_oracle():
    """The package must not import, link or call anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1806_10550_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower() or f == "inputs.py", f
                assert "tfo_" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1806_10550_b200 import" not in txt and "libtf_b200" not in txt, f

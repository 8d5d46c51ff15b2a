"""Per-kernel times of the library as built (not a pytest module):

    python tests/kernel_times.py [n] [fixed_iters] [steps]        # default 8192 8 3

One warm-up step, then `steps` steps of `fixed_iters` Newton iterations on the n x n film of config 3's recipe; prints the
mean CUDA-event time of the four kernels of an iteration (tf_set_profiling) and the time per iteration.  The status of the
steps is ignored on purpose: this is the harness behind the probe tables of profiles/r02_ncu.md, where the library is
built with a timing-only macro that computes wrong results, e.g.

    TF_EXTRA_NVCC_FLAGS="-DTF_EXP_NOCONS=1" python -m paper_1806_10550_b200.build --force && python tests/kernel_times.py
    python -m paper_1806_10550_b200.build --force                 # back to the product build
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_1806_10550_b200 import inputs, tf  # noqa: E402


def main():
    n = int(sys.argv[1]) if len(sys.argv) > 1 else 8192
    fixed = int(sys.argv[2]) if len(sys.argv) > 2 else 8
    steps = int(sys.argv[3]) if len(sys.argv) > 3 else 3
    cfg = inputs.config(3)
    g = tf.ThinFilm(n, n, cfg["dx"], cfg["dy"], cfg["kappa"], cfg["hstar"], cfg["n"], cfg["m"])
    g.set_newton(1e-10, 64, fixed)
    g.set_state(torch.from_numpy(inputs.noise_ic(n, n, cfg["seed"])).cuda())
    g.step(cfg["dt"])
    g.set_profiling(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(steps):
        g.step(cfg["dt"])
    ev1.record()
    torch.cuda.synchronize()
    out = {k: round(ms / max(cnt, 1), 4) for k, (ms, cnt) in g.get_profile().items()}
    out["iteration_ms"] = round(ev0.elapsed_time(ev1) / (steps * fixed), 4)
    print(n, json.dumps(out), flush=True)


if __name__ == "__main__":
    main()

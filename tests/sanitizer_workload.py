"""Workload for compute-sanitizer (memcheck / racecheck / synccheck), SURVEY.md section 5 -- not a pytest module:

    compute-sanitizer --tool memcheck  python tests/sanitizer_workload.py
    compute-sanitizer --tool racecheck python tests/sanitizer_workload.py
    compute-sanitizer --tool synccheck python tests/sanitizer_workload.py

Small grids that still reach every kernel family of the path: both CTA layouts of the forward kernels (four teams per
CTA needs more strips / blocks than SMs: one long side), the TMA rings and the plain fallbacks (odd pitch), the first
iteration (b^n) and later ones, launch-ahead gates, the isolated solver in both variants and directions, the mass
reduction, the extra solution criterion, the Betti numbers.  Results are checked against the oracle so that a run
that passes the sanitizer but computes garbage is not counted.  The summaries are in profiles/r02_sanitizer.md."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from oracle import tfo  # noqa: E402
from paper_1806_10550_b200 import inputs, tf  # noqa: E402


def step_case(nx, ny, fixed, steps, dt=1e-2, check=True):
    cfg = inputs.config(0)
    h = inputs.noise_ic(nx, ny, seed=nx + ny)
    g = tf.ThinFilm(nx, ny, cfg["dx"], cfg["dy"])
    g.set_newton(1e-10, 64, fixed)
    g.set_state(h)
    for _ in range(steps):
        st = g.step(dt)
        assert st[0] == 0, st
    u, m = g.get_state(), g.mass()
    if check:
        o = tfo.ThinFilmOracle(nx, ny, cfg["dx"], cfg["dy"], omp=True)
        o.set_newton(1e-10, 64, fixed)
        o.set_state(h)
        for _ in range(steps):
            o.step(dt)
        err = np.max(np.abs(u - o.get_state())) / np.max(np.abs(u))
        assert err <= 1e-11, (nx, ny, err)
        assert abs(m - o.mass()) <= 1e-13 * m
    g.close()
    print(f"tf_step {nx} x {ny}, fixed_iters {fixed}, {steps} steps: ok", flush=True)


def penta_case(nsys, length, variant):
    rows = inputs.penta_system(nsys, length, seed=length)
    for direction in (0, 1):
        arrs = rows if direction == 0 else [np.ascontiguousarray(t.T) for t in rows]
        x = tf.penta_solve(direction, *[torch.from_numpy(a).cuda() for a in arrs], variant=variant)
        torch.cuda.synchronize()
        ref = tfo.penta_solve(direction, *arrs)
        assert np.max(np.abs(x.cpu().numpy() - ref)) <= 1e-12 * np.max(np.abs(ref))
    print(f"tf_penta_solve_ex {nsys} x {length}, variant {variant}: ok", flush=True)


def main():
    assert torch.cuda.is_available()
    step_case(192, 160, 3, 1)                      # TMA rings, two teams per CTA
    step_case(61, 45, 2, 1)                        # odd pitch: plain kernels
    step_case(4228, 64, 2, 1)                      # 151 strips > SMs: y forward with four teams per CTA
    step_case(64, 4228, 2, 1)                      # 151 blocks > SMs: x forward with four teams per CTA
    step_case(128, 128, 0, 2)                      # tol-converged steps: launch-ahead batches and gated-off iterations
    g = tf.ThinFilm(96, 80, 0.43, 0.43)            # extra solution criterion: a rejected and an accepted step
    g.set_newton(1e-10, 64, 0)
    g.set_solution_criteria(1e-9)
    g.set_state(inputs.noise_ic(96, 80, seed=1))
    assert g.step(1e-2)[0] == tf.REJECTED
    g.set_solution_criteria(0.5)
    assert g.step(1e-2)[0] == tf.OK
    g.close()
    penta_case(64, 400, tf.PENTA_LU)
    penta_case(64, 400, tf.PENTA_PARTITION)
    penta_case(33, 37, tf.PENTA_LU)                # odd shapes: one-sided fallbacks
    img = torch.from_numpy(inputs.noise_ic(200, 130, seed=3)).cuda()
    b0, b1 = tf.betti(img, [0.995, 1.0, 1.005])
    assert len(b0) == 3 and all(v >= 0 for v in b0 + b1)
    print("tf_betti: ok\nsanitizer workload done", flush=True)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""Writes tests/golden/run_*.npz: sub-sampled FINAL states of full-length ORACLE runs of the BASELINE configs.

    python tests/golden/make_golden_runs.py [case ...]        (default: all cases; ~1 h on 8 cores, <= 10 GB)

TEST INFRASTRUCTURE.  This script calls only `oracle/` (the CPU oracle, written from PAPER.md:17-31, :25, :49 and the
readings of DESIGN.md 2) and the seeded input generators of `paper_1511_02137_b200/synthetic.py` (which hold none of
the method's arithmetic).  Nothing here comes from the CUDA path.  The `-m gpu` tests of tests/test_gpu_golden.py run
the CUDA path for the full length of each case (north_star: "matching the CPU oracle within 1e-9 ... after the run";
PAPER.md:49 grid, :41/:47 t = 2.4 fm/c = 120 steps) and compare the cells stored here.

Cases (name: config, steps, oracle options):
    cfg2          BASELINE config 2, 128^3, 50 steps
    cfg3          BASELINE config 3, 256^3, 120 steps                    (the graded benchmark)
    cfg3_fp32     config 3 with the fp32 variant's reading R10: initial state rounded to fp32, delta = 1e-5
    cfg3_lim      config 3 with the positivity-preserving flux limiter (reading R16)
    cfg3_w5       config 3 with the WENO5 variant, 120 steps
    cfg2_s500     config 2 run ten times its length (500 steps, t = 10 fm/c): the jet crosses the whole grid and LEAVES it through
                  the +x face at step ~470 (a jet outside deposits nothing, R7), the flow reaches the outflow boundaries
    cfg4_s6       BASELINE config 4 at FULL SIZE (512^3, nf = 5, two jets), the first 6 of its 200 steps (the whole run is
                  ~4 h of oracle time; 6 steps are ~10 min and ~40 GB) -- the one oracle comparison at the size where the
                  nf = 5 kernels run several waves with tail splitting

What is stored per case (numpy .npz):
    idx      (ncells, 3) int32   (k, j, i) of the sampled cells: every 8th cell per axis (offset 3; cfg4_s6: every 16th), the full-resolution
                                 line j = ny/2, k = nz/2 (the jet line y = z = 0+, R7) and the box of +-8 cells around
                                 the jet's track (all cells the jet deposits into during the run)
    U        (nf, ncells) f64    final conserved state at those cells
    fmax, fsum, fabs (nf,) f64   max |U_f|, sum U_f, sum |U_f| over ALL cells (R13 denominators, global budget)
    alpha (3,), deposited (4,), ncap, nlim, step, delta, limiter, config, steps      diagnostics of the oracle run
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as O  # noqa: E402
from paper_1511_02137_b200 import synthetic as S  # noqa: E402

CASES = {
    "cfg2": dict(config=2, delta=1e-10, fp32_input=False, limiter=False),
    "cfg3": dict(config=3, delta=1e-10, fp32_input=False, limiter=False),
    "cfg3_fp32": dict(config=3, delta=1e-5, fp32_input=True, limiter=False),
    "cfg3_lim": dict(config=3, delta=1e-10, fp32_input=False, limiter=True),
    "cfg3_w5": dict(config=3, delta=1e-10, fp32_input=False, limiter=False, weno_order=5),
    "cfg2_s500": dict(config=2, delta=1e-10, fp32_input=False, limiter=False, steps=500),
    "cfg4_s6": dict(config=4, delta=1e-10, fp32_input=False, limiter=False, steps=6, stride=16),
}


def sample_indices(c, steps, stride=8):
    """(k, j, i) of the stored cells (docstring above).  Integer work on the config's jet geometry (R6, R7)."""
    nx, ny, nz = c["n"]
    dx, dt = c["dx"], c["dt"]
    keep = np.zeros((nz, ny, nx), bool)
    keep[3::stride, 3::stride, 3::stride] = True
    for pos, d in c["jets"]:
        d = np.asarray(d, float) / np.linalg.norm(d)
        track = np.array([[np.floor((pos[a] + d[a] * s * dt + 0.5 * n * dx) / dx + 2.0 ** -20)
                           for a, n in enumerate((nx, ny, nz))] for s in (0.0, float(steps))]).astype(int)
        lo = np.minimum(track[0], track[1]) - 8
        hi = np.maximum(track[0], track[1]) + 8
        lo = np.maximum(lo, 0)
        hi = np.minimum(hi, [nx - 1, ny - 1, nz - 1])
        keep[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1] = True
    keep[nz // 2, ny // 2, :] = True
    return np.argwhere(keep).astype(np.int32)


def run_case(name):
    case = CASES[name]
    c = S.CONFIGS[case["config"]]
    steps = case.get("steps", c["steps"])
    U0 = S.make_state(case["config"])
    if case["fp32_input"]:
        U0 = U0.astype(np.float32).astype(np.float64)
    o = O.Oracle(*c["n"], c["dx"], c["dt"], nfields=c["nf"], v_cap_delta=case["delta"],
                 weno_order=case.get("weno_order", 7))
    o.set_state(U0)
    for pos, d in c["jets"]:
        o.add_jet(pos, d, S.KAPPA_RAD, S.KAPPA_COLL, S.CR_OVER_CF)
    o.set_limiter(case["limiter"])
    del U0
    t0 = time.time()
    for s in range(steps):
        o.step(1)
        if (s + 1) % 10 == 0 or steps < 10:
            print("%s: step %d / %d, %.0f s" % (name, s + 1, steps, time.time() - t0), flush=True)
    U = o.get_fields(0)
    dg = o.diag()
    assert dg["has_nan"] == 0 and dg["step"] == steps
    idx = sample_indices(c, steps, case.get("stride", 8))
    out = os.path.join(HERE, "run_%s.npz" % name)
    np.savez(out, idx=idx, U=U[:, idx[:, 0], idx[:, 1], idx[:, 2]],
             fmax=np.abs(U).max(axis=(1, 2, 3)), fsum=U.sum(axis=(1, 2, 3), dtype=np.longdouble).astype(np.float64),
             fabs=np.abs(U).sum(axis=(1, 2, 3), dtype=np.longdouble).astype(np.float64),
             alpha=dg["alpha"], deposited=dg["deposited"], ncap=np.int64(dg["ncap"]), nlim=np.int64(o.limited_faces()),
             step=np.int64(dg["step"]), delta=case["delta"], limiter=np.int64(case["limiter"]),
             config=np.int64(case["config"]), steps=np.int64(steps), fp32_input=np.int64(case["fp32_input"]),
             weno_order=np.int64(case.get("weno_order", 7)))
    print("%s: wrote %s (%d cells, %.1f MB), ncap %d, nlim %d, %.0f s" %
          (name, out, len(idx), os.path.getsize(out) / 1e6, dg["ncap"], o.limited_faces(), time.time() - t0), flush=True)
    o.close()


if __name__ == "__main__":
    for nm in (sys.argv[1:] or list(CASES)):
        run_case(nm)

"""Full-length parity of the BASELINE configs (pin P9 "after the run"): the CUDA path runs config 2 for its 50 steps and
config 3 (256^3, the graded benchmark; PAPER.md:49 grid, :41/:47 t = 2.4 fm/c) for its 120 steps -- fp64, the fp32
variant, with the flux limiter and with the WENO5 variant --, and config 4 at its full size (512^3, nf = 5) for its first 6
steps, in the launch configuration bench.py times, and is compared with the ORACLE's final
state at the cells stored in tests/golden/run_*.npz (written by tests/golden/make_golden_runs.py, which calls only
oracle/; every 8th cell per axis, the full-resolution jet line and the box of +-8 cells around the jet's track) plus the
global per-field sums.  Error metric R13: max over the stored cells of |gpu - oracle| / max over ALL cells of |oracle|.
Tolerances: 1e-9 fp64 (north_star), 1e-4 fp32 (north_star), 1e-8 with the limiter."""
import os

import numpy as np
import pytest

from paper_1511_02137_b200 import synthetic as S

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def H():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1511_02137_b200 import hydro
    hydro.load()
    return hydro


def load(name):
    path = os.path.join(GOLD, "run_%s.npz" % name)
    assert os.path.exists(path), "missing %s: run python tests/golden/make_golden_runs.py %s" % (path, name)
    return np.load(path)


@pytest.mark.parametrize("name,precision,tol,tol_sum", [("cfg2", 64, 1e-9, 1e-11), ("cfg3", 64, 1e-9, 1e-11),
                                                         ("cfg3_fp32", 32, 1e-4, 1e-5), ("cfg3_lim", 64, 1e-8, 1e-10),
                                                         ("cfg3_w5", 64, 1e-9, 1e-11), ("cfg4_s6", 64, 1e-9, 1e-11)])
def test_full_length_run_matches_the_oracle_sample(H, name, precision, tol, tol_sum):
    gold = load(name)
    cfg, steps = int(gold["config"]), int(gold["steps"])
    c = S.CONFIGS[cfg]
    assert steps == c["steps"] or name == "cfg4_s6"          # config 4: the first 6 steps at full size (512^3, nf = 5)
    order = int(gold["weno_order"]) if "weno_order" in gold.files else 7
    U0 = S.make_state(cfg)
    if precision == 32:
        U0 = U0.astype(np.float32)
    g = H.Hydro(*c["n"], c["dx"], c["dt"], nfields=c["nf"], precision=precision, weno_order=order)
    assert g.uses_ring()
    g.set_state(U0)
    del U0
    for pos, d in c["jets"]:
        g.add_jet(pos, d, S.KAPPA_RAD, S.KAPPA_COLL, S.CR_OVER_CF)
    g.set_limiter(bool(gold["limiter"]))
    g.step(steps)
    U = g.get_fields().astype(np.float64)
    dg = g.diag()
    nlim = g.limited_faces()
    g.close()
    assert dg["has_nan"] == 0 and dg["step"] == steps
    idx, Uo = gold["idx"], gold["U"]
    Ug = U[:, idx[:, 0], idx[:, 1], idx[:, 2]]
    errs = np.max(np.abs(Ug - Uo), axis=1) / gold["fmax"]
    assert np.all(errs < tol), (name, errs)
    # global budget: per-field sums over ALL cells (a cell outside the sample that went wrong would show up here)
    fsum = U.sum(axis=(1, 2, 3), dtype=np.longdouble).astype(np.float64)
    assert np.all(np.abs(fsum - gold["fsum"]) <= tol_sum * gold["fabs"]), (name, fsum, gold["fsum"])
    fmax = np.abs(U).max(axis=(1, 2, 3))
    assert np.all(np.abs(fmax - gold["fmax"]) <= tol * gold["fmax"]), (name, fmax, gold["fmax"])
    # diagnostics of the run
    atol = 1e-12 if precision == 64 else 1e-5
    assert np.max(np.abs(dg["alpha"] - gold["alpha"])) < atol, (dg["alpha"], gold["alpha"])
    dep = gold["deposited"]
    assert np.max(np.abs(dg["deposited"] - dep)) <= (1e-10 if precision == 64 else 1e-4) * dep[0]
    ncap = int(gold["ncap"])
    if precision == 64:
        assert abs(dg["ncap"] - ncap) <= max(2, 0.02 * ncap), (dg["ncap"], ncap)
        if name in ("cfg2", "cfg3", "cfg3_w5"):
            assert ncap > 0                     # the full-length runs reach the regime where the cap fires (R9)
    else:
        assert abs(dg["ncap"] - ncap) <= max(10, 0.2 * ncap), (dg["ncap"], ncap)      # fp32 decides the cap in fp32 (R10)
    if bool(gold["limiter"]):
        assert ncap == 0 and dg["ncap"] == 0
        assert abs(nlim - int(gold["nlim"])) <= max(3, 0.02 * int(gold["nlim"])), (nlim, int(gold["nlim"]))


def test_ten_times_the_length_of_config2(H):
    """Config 2 run for 500 steps (ten times its length, t = 10 fm/c; oracle sample run_cfg2_s500.npz): the jet crosses the
    grid and LEAVES it through the +x face near step 470 (a jet outside deposits nothing, R7), the flow reaches the outflow
    boundaries (a-7), and the con2prim cap R9 fires 261 147 times along the jet's track.  What is integer or decided
    per event must agree as in the short runs (cap count, deposited totals, the jet's q = 0 at the end, alpha); the fields
    are compared at 1e-5 instead of 1e-9: each cap event is a switch, and ulp-level differences between the two
    arithmetic orders grow along the capped track over ten times the graded length (measured 9e-7 on M_y, 3e-8 on E)."""
    gold = load("cfg2_s500")
    c = S.CONFIGS[2]
    steps = int(gold["steps"])
    assert steps == 500
    g = H.Hydro(*c["n"], c["dx"], c["dt"])
    g.set_state(S.make_state(2))
    for pos, d in c["jets"]:
        g.add_jet(pos, d, S.KAPPA_RAD, S.KAPPA_COLL, S.CR_OVER_CF)
    g.step(steps)
    U = g.get_fields()
    dg = g.diag()
    q = g.last_stage_q()
    g.close()
    assert dg["has_nan"] == 0 and dg["step"] == steps
    idx = gold["idx"]
    errs = np.max(np.abs(U[:, idx[:, 0], idx[:, 1], idx[:, 2]] - gold["U"]), axis=1) / gold["fmax"]
    assert np.all(errs < 1e-5), errs
    fsum = U.sum(axis=(1, 2, 3), dtype=np.longdouble).astype(np.float64)
    assert np.all(np.abs(fsum - gold["fsum"]) <= 1e-9 * gold["fabs"])
    ncap = int(gold["ncap"])
    assert ncap > 100000 and abs(dg["ncap"] - ncap) <= 0.02 * ncap
    assert np.max(np.abs(dg["alpha"] - gold["alpha"])) < 1e-9
    assert np.max(np.abs(dg["deposited"] - gold["deposited"])) <= 1e-10 * gold["deposited"][0]
    assert np.all(q == 0.0)                                  # the jet is outside the grid: nothing is deposited any more

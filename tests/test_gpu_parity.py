"""GPU parity (pin P9): the CUDA path, called through the C ABI, against the CPU oracle on the same seeded inputs.

Error metric (reading R13): err_f = max_cells |f_gpu - f_oracle| / max_cells |f_oracle| per conserved field; a field
that is identically zero in the oracle must be exactly zero on the GPU.  Tolerance: 1e-9 in fp64 after the run
(north_star), tighter for single kernels / single stages.
"""
import os

import numpy as np
import pytest

from paper_1511_02137_b200 import synthetic as S

pytestmark = pytest.mark.gpu

TOL_RUN = 1e-9          # north_star: after the run, fp64
TOL_STAGE = 1e-12       # one evaluation of L(U): only rounding-order differences


@pytest.fixture(scope="module")
def H():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1511_02137_b200 import hydro
    hydro.load()
    return hydro


def r13(gpu, ref):
    errs = []
    for f in range(ref.shape[0]):
        m = np.max(np.abs(ref[f]))
        if m == 0.0:
            assert np.all(gpu[f] == 0.0), "field %d must be exactly zero" % f
            errs.append(0.0)
        else:
            errs.append(float(np.max(np.abs(gpu[f] - ref[f])) / m))
    return errs


def make_pair(H, oracle, cfg, noise=True, jets=True, **kw):
    c = S.CONFIGS[cfg] if not isinstance(cfg, dict) else cfg
    U0 = S.make_state(c, noise=noise)
    g = H.Hydro(*c["n"], c["dx"], c["dt"], nfields=c["nf"], **kw)
    o = oracle.Oracle(*c["n"], c["dx"], c["dt"], nfields=c["nf"])
    g.set_state(U0)
    o.set_state(U0)
    if jets:
        for pos, d in c["jets"]:
            g.add_jet(pos, d, S.KAPPA_RAD, S.KAPPA_COLL, S.CR_OVER_CF)
            o.add_jet(pos, d, S.KAPPA_RAD, S.KAPPA_COLL, S.CR_OVER_CF)
    return c, U0, g, o


def compare_diag(g, o, steps):
    dg, do = g.diag(), o.diag()
    assert dg["step"] == do["step"] == steps
    assert np.max(np.abs(dg["alpha"] - do["alpha"])) < 1e-12
    assert abs(dg["cfl"] - do["cfl"]) < 1e-12
    assert dg["has_nan"] == do["has_nan"] == 0
    assert np.max(np.abs(dg["deposited"] - do["deposited"])) <= 1e-10 * max(1e-300, np.max(np.abs(do["deposited"])))
    return dg, do


# ------------------------------------------------------------------------------------------------ a-1, a-2
def test_con2prim_parity(H, oracle):
    rng = np.random.default_rng(42)
    n = (37, 19, 23)                                     # ragged: not a multiple of any block size
    N = n[0] * n[1] * n[2]
    e = 10.0 ** rng.uniform(-3, 3, N)
    vm = rng.uniform(0, 0.999, N)
    d = rng.normal(size=(3, N))
    d /= np.linalg.norm(d, axis=0)
    u = vm / np.sqrt(1 - vm * vm) * d
    U = S.prim_to_cons(e, u[0], u[1], u[2], e / 10).reshape(5, n[2], n[1], n[0])
    # a few inadmissible cells: cap and floor must act identically (R9)
    U[1, 0, 0, :5] = 2.0 * U[0, 0, 0, :5]
    U[0, 1, 1, :3] = -1.0
    for nf in (4, 5):
        g = H.Hydro(*n, 0.1, 0.02, nfields=nf)
        o = oracle.Oracle(*n, 0.1, 0.02, nfields=nf)
        g.set_state(U[:nf].copy())
        o.set_state(U[:nf].copy())
        Pg, Po = g.get_fields(H.FIELDS_PRIMITIVE), o.get_fields(1)
        assert np.array_equal(g.get_fields(H.FIELDS_CONSERVED), U[:nf])          # state round-trips bitwise
        gam2 = 1.0 / (1.0 - np.minimum(vm, 0.9999) ** 2).reshape(n[2], n[1], n[0])
        capped = np.zeros(gam2.shape, bool)
        capped[0, 0, :5] = True
        capped[1, 1, :3] = True
        assert np.max((np.abs(Pg[0] - Po[0]) / (np.abs(Po[0]) * gam2))[~capped]) < 5e-15
        # on the cap e = 3(E^2-M^2)/(E+s) cancels to ~2 delta E: compare relative to E, not to e
        assert np.max((np.abs(Pg[0] - Po[0]) / np.maximum(np.abs(U[0]), 1e-12))[capped]) < 5e-15
        for f in (1, 2, 3):
            assert np.max(np.abs(Pg[f] - Po[f])) < 5e-15
        if nf == 5:
            assert np.max((np.abs(Pg[4] - Po[4]) / np.abs(Po[4]))[~capped]) < 1e-12 * gam2.max()
            # on the cap 1 - v^2 ~ 2 delta is itself only known to ~1e-16/delta
            assert np.max((np.abs(Pg[4] - Po[4]) / np.abs(Po[4]))[capped]) < 1e-5
        # wavespeed maxima and cap counts come out of one RHS evaluation
        g.eval_rhs(0.0)
        o.eval_rhs(0.0)
        dg, do = g.diag(), o.diag()
        assert np.max(np.abs(dg["alpha"] - do["alpha"])) < 1e-13
        g.close(), o.close()


# ------------------------------------------------------------------------------------------------ a-3..a-5, a-7
@pytest.mark.parametrize("n", [(32, 32, 32), (37, 19, 23), (7, 5, 3), (1, 1, 40), (130, 9, 6), (34, 19, 23), (2, 3, 4),
                               (64, 40, 72), (8, 100, 8), (72, 8, 33)])
@pytest.mark.parametrize("nf", [4, 5])
def test_rhs_single_stage_parity(H, oracle, n, nf):
    c = S.scaled_config(0, n)
    c["nf"] = nf
    c["jets"] = [((-0.12, 0.03, 0.0), (1.0, 0.5, -0.25))]
    c, U0, g, o = make_pair(H, oracle, c)
    for stage_c in (0.0, 1.0, 0.5):
        Lg, Lo = g.eval_rhs(stage_c), o.eval_rhs(stage_c)
        scale = np.max(np.abs(Lo), axis=(1, 2, 3))
        for f in range(nf):
            assert np.max(np.abs(Lg[f] - Lo[f])) <= TOL_STAGE * max(scale[f], scale[0]), (f, stage_c)
        assert np.max(np.abs(g.diag()["alpha"] - o.diag()["alpha"])) < 1e-13
    g.close(), o.close()


def test_jet_cell_and_source_bitwise_location(H, oracle):
    """The deposit cell is integer work: the set of cells touched by the source must be identical."""
    c = S.scaled_config(0, (24, 20, 16))
    c["jets"] = [((0.0, 0.0, 0.0), (1.0, 0.0, 0.0)), ((0.0, 0.0, 0.0), (-1.0, 0.0, 0.0)),
                 ((-0.35, 0.25, 0.05), (0.3, -0.4, 0.2)), ((9.0, 0.0, 0.0), (1.0, 0.0, 0.0)),
                 # 0.8 and 1.2 x 2^-20 cells below a face: the upper / the lower cell (size of the R7 bias), at rest along x
                 ((0.3 - 0.8 * 2.0 ** -20 * 0.1, -0.45, 0.33), (0.0, 1e-9, 1.0)),
                 ((0.3 - 1.2 * 2.0 ** -20 * 0.1, 0.45, -0.33), (0.0, 1e-9, -1.0))]
    for stage_c in (0.0, 0.5, 1.0):
        _, U0, g, o = make_pair(H, oracle, c)
        _, _, g0, o0 = make_pair(H, oracle, c, jets=False)
        dLg = g.eval_rhs(stage_c) - g0.eval_rhs(stage_c)
        dLo = o.eval_rhs(stage_c) - o0.eval_rhs(stage_c)
        assert np.array_equal(dLg != 0, dLo != 0)
        assert np.max(np.abs(dLg - dLo)) < 1e-12 * np.max(np.abs(dLo))
        for x in (g, o, g0, o0):
            x.close()


def test_maximum_number_of_jets(H, oracle):
    """Eq. (2) sums over jets: a full jet table (64, the handle's maximum), seeded positions and directions,
    several jets starting next to a face and leaving the grid during the run (a jet outside deposits nothing, R7), compared
    with the oracle after 8 steps; the 65th jet is refused with HYDRO_ESTATE and leaves the table unchanged."""
    c = S.scaled_config(0, (32, 24, 20))
    rng = np.random.default_rng(64)
    half = 0.5 * np.array(c["n"]) * c["dx"]
    jets = []
    for j in range(64):
        pos = rng.uniform(-0.9, 0.9, size=3) * half
        d = rng.normal(size=3)
        if j % 8 == 0:                                   # next to the +x face, heading out: gone after a few steps
            pos[0] = half[0] - 0.05
            d = np.array([1.0, 0.1 * d[1], 0.1 * d[2]])
        jets.append((tuple(pos), tuple(d)))
    c["jets"] = jets
    _, U0, g, o = make_pair(H, oracle, c)
    with pytest.raises(H.HydroError) as ei:
        g.add_jet((0.0, 0.0, 0.0), (1.0, 0.0, 0.0))
    assert ei.value.code == H.ESTATE
    g.step(8)
    o.step(8)
    errs = r13(g.get_fields(), o.get_fields())
    assert max(errs) < 1e-9, errs
    dg, do = compare_diag(g, o, 8)
    assert dg["deposited"][0] > 0
    g.close()
    o.close()


def test_jet_added_in_the_middle_of_a_run(H, oracle):
    """The path length of eq. (3) counts from the step a jet was added (R8: l = t - t_added): a second jet added after
    two steps (the captured step graph is rebuilt for the new jet table), three more steps, compared with the oracle."""
    c = S.scaled_config(0, (32, 24, 20))
    _, U0, g, o = make_pair(H, oracle, c)
    g.step(2)
    o.step(2)
    for x in (g, o):
        x.add_jet((0.4, -0.3, 0.2), (-0.6, 0.7, 0.1), 3.0, 1.5, 9.0 / 4.0)
    g.step(3)
    o.step(3)
    errs = r13(g.get_fields(), o.get_fields())
    assert max(errs) < 1e-9, errs
    compare_diag(g, o, 5)
    qg, qo = g.last_stage_q(), o.last_stage_q()
    assert qg.shape == qo.shape == (3, 2) and np.max(np.abs(qg - qo)) < 1e-11 * np.max(qo)
    g.close()
    o.close()


# ------------------------------------------------------------------------------------------------ whole path
def test_config0_full_run(H, oracle):
    c, U0, g, o = make_pair(H, oracle, 0)
    g.step(c["steps"])
    o.step(c["steps"])
    errs = r13(g.get_fields(), o.get_fields())
    assert max(errs) < TOL_RUN, errs
    dg, do = compare_diag(g, o, c["steps"])
    assert dg["ncap"] == do["ncap"] == 0
    assert np.max(np.abs(g.last_stage_q() - o.last_stage_q())) < 1e-11
    assert do["deposited"][0] > 0
    # split stepping gives the same state as one call (the step counter, jets and primitives carry over)
    g2 = H.Hydro(*c["n"], c["dx"], c["dt"])
    g2.set_state(U0)
    for pos, d in c["jets"]:
        g2.add_jet(pos, d)
    for k in (3, 0, 6, 1):
        g2.step(k)
    assert np.array_equal(g2.get_fields(), g.get_fields())
    for x in (g, g2, o):
        x.close()


def test_config0_five_fields_and_ragged_grid(H, oracle):
    c = S.scaled_config(0, (45, 27, 18))
    c["nf"] = 5
    c["steps"] = 6
    c, U0, g, o = make_pair(H, oracle, c)
    g.step(c["steps"])
    o.step(c["steps"])
    errs = r13(g.get_fields(), o.get_fields())
    assert max(errs) < TOL_RUN, errs
    compare_diag(g, o, c["steps"])
    Pg, Po = g.get_fields(H.FIELDS_PRIMITIVE), o.get_fields(1)
    assert max(r13(Pg, Po)) < TOL_RUN
    g.close(), o.close()


def test_five_fields_multi_wave_grid(H, oracle):
    """nf = 5 on a grid whose three sweeps each launch more tiles than resident block slots (several waves + the
    tail-split last wave of hydro.cu launch_ring_nf): one evaluation of L(U) (OUT_STORE / OUT_REDUCE kernels) and a
    2-step run (OUT_COMBINE kernels) against the oracle on every cell."""
    c = S.scaled_config(3, (136, 168, 130))
    c["nf"] = 5
    c["jets"] = [((-5.0, 0.0, 0.0), (1.0, 0.0, 0.0)), ((1.0, 2.0, -1.0), (-1.0, 1.0, 0.5))]
    c, U0, g, o = make_pair(H, oracle, c)
    Lg, Lo = g.eval_rhs(0.5), o.eval_rhs(0.5)
    scale = np.max(np.abs(Lo), axis=(1, 2, 3))
    for f in range(5):
        assert np.max(np.abs(Lg[f] - Lo[f])) <= TOL_STAGE * max(scale[f], scale[0]), f
    g.step(2), o.step(2)
    errs = r13(g.get_fields(), o.get_fields())
    assert max(errs) < TOL_RUN, errs
    compare_diag(g, o, 2)
    g.close(), o.close()


def test_config1_shock_tube(H, oracle):
    """BASELINE config 1: 512x8x8, 375 steps; GPU vs oracle, and GPU vs the exact Riemann solution (pin P4)."""
    from test_oracle_riemann import exact_solution, exact_profile
    c, U0, g, _o = make_pair(H, oracle, 1)
    _o.close()
    g.step(c["steps"])
    Ug = g.get_fields()
    Pg = g.get_fields(H.FIELDS_PRIMITIVE)
    # P7 on the GPU: the embedded tube is independent of j, k bitwise and has no transverse momentum
    assert np.array_equal(Ug, np.broadcast_to(Ug[:, :1, :1, :], Ug.shape))
    assert np.all(Ug[2] == 0) and np.all(Ug[3] == 0)
    # the oracle run of the same tube is 1-D (P7: embedding is bitwise in the oracle too)
    o = oracle.Oracle(512, 1, 1, c["dx"], c["dt"])
    o.set_state(U0[:, :1, :1, :].copy())
    o.step(c["steps"])
    Uo = o.get_fields()
    errs = r13(Ug[:, :1, :1, :], Uo)
    assert max(errs) < TOL_RUN, errs
    x = S.cell_centres(512, c["dx"])
    ee, ve = exact_profile(x, c["dt"] * c["steps"], exact_solution())
    assert np.sum(np.abs(Pg[0, 0, 0] - ee)) * c["dx"] < 0.08
    assert np.sum(np.abs(Pg[1, 0, 0] - ve)) * c["dx"] < 0.01
    dg = g.diag()
    assert dg["ncap"] == 0 and abs(dg["alpha"][0] - o.diag()["alpha"][0]) < 1e-12
    g.close(), o.close()


def test_jet_run_with_cap_events(H, oracle):
    """A jet through e ~ 30 GeV/fm^3 drives cells next to the deposit inadmissible (R9): the cap must fire on
    both sides in (nearly) the same cells and parity must survive it."""
    c = S.scaled_config(2, (64, 32, 32))
    c["jets"] = [((-2.0, 0.0, 0.0), (1.0, 0.0, 0.0))]
    steps = int(os.environ.get("HYDRO_TEST_CAP_STEPS", "60"))
    c, U0, g, o = make_pair(H, oracle, c)
    g.step(steps)
    o.step(steps)
    errs = r13(g.get_fields(), o.get_fields())
    assert max(errs) < TOL_RUN, errs
    dg, do = compare_diag(g, o, steps)
    assert do["ncap"] > 0, "this case is meant to exercise the cap"
    assert abs(dg["ncap"] - do["ncap"]) <= max(2, 0.02 * do["ncap"])
    g.close(), o.close()


def test_config2_midsize(H, oracle):
    """BASELINE config 2 (128^3); HYDRO_TEST_CFG2_STEPS (default 4) of its 50 steps -- the oracle costs ~9 s/step
    on 8 cores."""
    steps = int(os.environ.get("HYDRO_TEST_CFG2_STEPS", "4"))
    c, U0, g, o = make_pair(H, oracle, 2)
    g.step(steps)
    o.step(steps)
    errs = r13(g.get_fields(), o.get_fields())
    assert max(errs) < TOL_RUN, errs
    compare_diag(g, o, steps)
    g.close(), o.close()


def test_config3_full_size_first_steps(H, oracle):
    """BASELINE config 3 at its full size (256^3), in the launch configuration bench.py times (ring kernels, one
    segment per line): HYDRO_TEST_CFG3_STEPS (default 2) of its 120 steps against the oracle on every cell (the
    oracle needs ~4-8 s per step on the box's cores and ~3 GB)."""
    steps = int(os.environ.get("HYDRO_TEST_CFG3_STEPS", "2"))
    c, U0, g, o = make_pair(H, oracle, 3)
    assert g.uses_ring()
    g.step(steps)
    o.step(steps)
    errs = r13(g.get_fields(), o.get_fields())
    assert max(errs) < TOL_RUN, errs
    compare_diag(g, o, steps)
    g.close(), o.close()


def test_config3_long_run_properties(H):
    """Config 3 for its full 120 steps on the GPU alone, in bench.py's launch configuration: properties that hold at
    any size.  Pin P5 on the device: the run with the jet and the run without it differ in total energy and
    momentum by exactly the deposited amounts (the jet's wake has not reached the boundary by t = 2.4 fm/c, so the
    boundary fluxes of the two runs agree up to the tiny change of the global Lax-Friedrichs alpha); the state stays
    finite; a repeated run is bitwise identical (reduce-adds are ordered by the stream)."""
    c = S.CONFIGS[3]
    U0 = S.make_state(3)
    g = H.Hydro(*c["n"], c["dx"], c["dt"])
    assert g.uses_ring()
    g.set_state(U0)
    g.step(c["steps"])
    tot0 = [U.sum(dtype=np.longdouble) for U in g.get_fields()]
    for pos, d in c["jets"]:
        g.add_jet(pos, d)
    g.set_state(U0)
    g.step(c["steps"])
    U = g.get_fields()
    dg = g.diag()
    assert dg["has_nan"] == 0 and dg["step"] == c["steps"] and np.all(np.isfinite(U))
    dep = dg["deposited"]
    assert dep[0] > 5.0 and dep[1] == pytest.approx(dep[0], rel=1e-12) and dep[2] == 0.0 and dep[3] == 0.0
    dx3 = c["dx"] ** 3
    for f in range(4):
        diff = float((U[f].sum(dtype=np.longdouble) - tot0[f]) * dx3)
        assert abs(diff - dep[f]) <= 5e-5 * dep[0], (f, diff, dep[f])      # measured 6e-6 (alpha: 0.97 -> 1.0 with the jet)
    g.set_state(U0)
    g.step(c["steps"])
    assert np.array_equal(g.get_fields(), U)
    g.close()


@pytest.mark.parametrize("n", [(32, 32, 32), (36, 19, 23), (8, 5, 3), (132, 9, 6), (33, 20, 17), (64, 40, 72)])
@pytest.mark.parametrize("nf", [4, 5])
def test_fp32_rhs_single_stage(H, oracle, n, nf):
    """fp32 variant, one evaluation of L(U) (R10); every nx runs the ring kernels (rows are pitched to 16 bytes)."""
    c = S.scaled_config(0, n)
    c["nf"] = nf
    c["jets"] = [((-0.12, 0.03, 0.0), (1.0, 0.5, -0.25))]
    U0 = S.make_state(c).astype(np.float32)
    g = H.Hydro(*n, c["dx"], c["dt"], nfields=nf, precision=32)
    o = oracle.Oracle(*n, c["dx"], c["dt"], nfields=nf, v_cap_delta=1e-5)
    assert g.uses_ring()
    g.set_state(U0)
    o.set_state(U0.astype(np.float64))
    for pos, d in c["jets"]:
        g.add_jet(pos, d)
        o.add_jet(pos, d)
    for stage_c in (0.0, 0.5):
        Lg, Lo = g.eval_rhs(stage_c).astype(np.float64), o.eval_rhs(stage_c)
        scale = np.max(np.abs(Lo), axis=(1, 2, 3))
        for f in range(nf):
            assert np.max(np.abs(Lg[f] - Lo[f])) <= 1e-4 * max(scale[f], scale[0]), (f, stage_c)
        assert np.max(np.abs(g.diag()["alpha"] - o.diag()["alpha"])) < 1e-5
    g.close(), o.close()


@pytest.mark.parametrize("cfg,n,steps", [(0, (32, 32, 32), 10), (2, (64, 32, 32), 30), (0, (33, 20, 17), 6),
                                         (0, (44, 27, 18), 6)])
def test_fp32_variant(H, oracle, cfg, n, steps):
    """fp32 variant (R10): storage and arithmetic in fp32, compared with the fp64 oracle run with delta = 1e-5,
    north_star tolerance 1e-4 (R13 metric)."""
    c = S.scaled_config(cfg, n)
    if cfg == 2:
        c["jets"] = [((-2.0, 0.0, 0.0), (1.0, 0.0, 0.0))]
    U0 = S.make_state(c)
    g = H.Hydro(*c["n"], c["dx"], c["dt"], precision=32)
    o = oracle.Oracle(*c["n"], c["dx"], c["dt"], v_cap_delta=1e-5)
    g.set_state(U0.astype(np.float32))
    o.set_state(U0.astype(np.float32).astype(np.float64))
    for pos, d in c["jets"]:
        g.add_jet(pos, d)
        o.add_jet(pos, d)
    g.step(steps)
    o.step(steps)
    errs = r13(g.get_fields().astype(np.float64), o.get_fields())
    assert max(errs) < 1e-4, errs
    assert g.diag()["has_nan"] == 0
    g.close(), o.close()


def test_config4_full_size_properties(H):
    """BASELINE config 4 at its full size (512^3, nf = 5, two back-to-back jets; 22 GiB on the device), a few steps on
    the GPU alone (the oracle would need ~30 GB and minutes): properties that hold at any size -- finite state, both
    jets start in the same cell with opposite directions so the deposited momentum cancels at l = 0 and stays well
    below the deposited energy (the +x jet stays in the cell both heated, so its q is somewhat larger), the baryon number only changes through the boundary, a repeated run is bitwise equal."""
    import torch
    if torch.cuda.mem_get_info()[1] < 40 * 2 ** 30:
        pytest.skip("needs a device with > 40 GiB")
    c = S.CONFIGS[4]
    steps = int(os.environ.get("HYDRO_TEST_CFG4_STEPS", "2"))
    U0 = S.make_state(4)
    g = H.Hydro(*c["n"], c["dx"], c["dt"], nfields=5)
    g.set_state(U0)
    for pos, d in c["jets"]:
        g.add_jet(pos, d)
    g.step(steps)
    U = g.get_fields()
    dg = g.diag()
    assert dg["has_nan"] == 0 and dg["step"] == steps and np.all(np.isfinite(U[:, ::7, ::5, ::3]))
    q = g.last_stage_q()
    assert q.shape == (3, 2) and np.all(q > 0)
    assert dg["deposited"][0] > 0 and abs(dg["deposited"][1]) < 0.5 * dg["deposited"][0]
    nb0, nb1 = U0[4].sum(dtype=np.longdouble), U[4].sum(dtype=np.longdouble)
    assert abs(float(nb1 - nb0)) < 1e-3 * float(nb0)                      # only boundary outflow of the 0.01 background
    g.set_state(U0)
    g.step(steps)
    assert np.array_equal(g.get_fields()[:, 250:262], U[:, 250:262])
    g.close()


# ------------------------------------------------------------------------------------------------ WENO5 variant (f-2)
@pytest.mark.parametrize("n", [(32, 32, 32), (37, 19, 23), (7, 5, 3), (130, 9, 6), (64, 40, 72)])
@pytest.mark.parametrize("nf", [4, 5])
def test_weno5_rhs_single_stage_parity(H, oracle, n, nf):
    c = S.scaled_config(0, n)
    c["nf"] = nf
    c["jets"] = [((-0.12, 0.03, 0.0), (1.0, 0.5, -0.25))]
    U0 = S.make_state(c)
    g = H.Hydro(*n, c["dx"], c["dt"], nfields=nf, weno_order=5)
    o = oracle.Oracle(*n, c["dx"], c["dt"], nfields=nf, weno_order=5)
    g.set_state(U0), o.set_state(U0)
    for pos, d in c["jets"]:
        g.add_jet(pos, d), o.add_jet(pos, d)
    for stage_c in (0.0, 0.5):
        Lg, Lo = g.eval_rhs(stage_c), o.eval_rhs(stage_c)
        scale = np.max(np.abs(Lo), axis=(1, 2, 3))
        for f in range(nf):
            assert np.max(np.abs(Lg[f] - Lo[f])) <= TOL_STAGE * max(scale[f], scale[0]), (f, stage_c)
    # and it is a different scheme from WENO7
    g7 = H.Hydro(*n, c["dx"], c["dt"], nfields=nf)
    g7.set_state(U0)
    assert np.max(np.abs(g7.eval_rhs(0.0)[0] - g.eval_rhs(0.0)[0])) > 1e-9 * scale[0]
    g.close(), o.close(), g7.close()


@pytest.mark.parametrize("prec,tol", [(64, TOL_RUN), (32, 1e-4)])
def test_weno5_runs(H, oracle, prec, tol):
    """WENO5 variant: config 0 (10 steps, jet) and the jet/cap case, fp64 and fp32."""
    for cfg, n, steps in ((0, (32, 32, 32), 10), (2, (64, 32, 32), 40)):
        c = S.scaled_config(cfg, n)
        if cfg == 2:
            c["jets"] = [((-2.0, 0.0, 0.0), (1.0, 0.0, 0.0))]
        dt_np = np.float64 if prec == 64 else np.float32
        U0 = S.make_state(c).astype(dt_np)
        g = H.Hydro(*n, c["dx"], c["dt"], precision=prec, weno_order=5)
        o = oracle.Oracle(*n, c["dx"], c["dt"], weno_order=5, v_cap_delta=1e-10 if prec == 64 else 1e-5)
        g.set_state(U0), o.set_state(U0.astype(np.float64))
        for pos, d in c["jets"]:
            g.add_jet(pos, d), o.add_jet(pos, d)
        g.step(steps), o.step(steps)
        errs = r13(g.get_fields().astype(np.float64), o.get_fields())
        assert max(errs) < tol, (cfg, errs)
        assert g.diag()["has_nan"] == 0
        g.close(), o.close()


# ------------------------------------------------------------------------------------------------ smeared deposit (f-3)
@pytest.mark.parametrize("sigma", [0.05, 0.1, 0.25])
def test_smeared_deposit_rhs_parity(H, oracle, sigma):
    """Reading R15: the Gaussian deposit of several jets (one near a corner, one outside the grid) on the GPU and in
    the oracle: same support (integer work) and the same values."""
    c = S.scaled_config(0, (26, 21, 16))
    c["jets"] = [((0.0, 0.0, 0.0), (1.0, 0.0, 0.0)), ((0.02, 0.01, 0.0), (-1.0, 0.0, 0.0)),
                 ((-0.35, 0.25, 0.05), (0.3, -0.4, 0.2)), ((1.25, 1.0, 0.75), (1.0, 1.0, 1.0)), ((9.0, 0.0, 0.0), (1.0, 0.0, 0.0))]
    for stage_c in (0.0, 0.5):
        _, U0, g, o = make_pair(H, oracle, c)
        _, _, g0, o0 = make_pair(H, oracle, c, jets=False)
        g.set_deposit_width(sigma), o.set_deposit_width(sigma)
        dLg = g.eval_rhs(stage_c) - g0.eval_rhs(stage_c)
        dLo = o.eval_rhs(stage_c) - o0.eval_rhs(stage_c)
        big = np.abs(dLo) > 1e-9 * np.max(np.abs(dLo))            # tiny tails may round to the background's ulp
        assert np.array_equal((dLg != 0)[big], (dLo != 0)[big])
        assert np.max(np.abs(dLg - dLo)) < 1e-11 * np.max(np.abs(dLo))
        for x in (g, o, g0, o0):
            x.close()


@pytest.mark.parametrize("prec,tol", [(64, TOL_RUN), (32, 1e-4)])
def test_smeared_deposit_run(H, oracle, prec, tol):
    """The jet/cap case of test_jet_run_with_cap_events with a Gaussian deposit of width dx: parity after the run, the
    deposited totals agree, and (SURVEY f-3) the smearing removes the cap events the point deposit causes."""
    c = S.scaled_config(2, (64, 32, 32))
    c["jets"] = [((-2.0, 0.0, 0.0), (1.0, 0.0, 0.0)), ((2.0, 0.5, 0.0), (-1.0, 0.0, 0.0))]
    steps = 40
    U0 = S.make_state(c).astype(np.float64 if prec == 64 else np.float32)
    g = H.Hydro(*c["n"], c["dx"], c["dt"], precision=prec)
    o = oracle.Oracle(*c["n"], c["dx"], c["dt"], v_cap_delta=1e-10 if prec == 64 else 1e-5)
    g.set_state(U0), o.set_state(U0.astype(np.float64))
    for pos, d in c["jets"]:
        g.add_jet(pos, d), o.add_jet(pos, d)
    g.set_deposit_width(0.1), o.set_deposit_width(0.1)
    g.step(steps), o.step(steps)
    errs = r13(g.get_fields().astype(np.float64), o.get_fields())
    assert max(errs) < tol, errs
    dg, do = g.diag(), o.diag()
    assert np.max(np.abs(dg["deposited"] - do["deposited"])) <= (1e-10 if prec == 64 else 1e-4) * do["deposited"][0]
    assert dg["has_nan"] == 0 and dg["ncap"] == do["ncap"] == 0
    g.close(), o.close()


# ------------------------------------------------------------------------------------------------ flux limiter (f-1)
def _rough_state(n, seed, vmax=0.98, nf=4):
    rng = np.random.default_rng(seed)
    shape = (n[2], n[1], n[0])
    e = 10.0 ** rng.uniform(-2, 2, shape)
    vm = rng.uniform(0, vmax, shape)
    d = rng.normal(size=(3,) + shape)
    d /= np.linalg.norm(d, axis=0)
    u = vm / np.sqrt(1 - vm * vm) * d
    return S.prim_to_cons(e, u[0], u[1], u[2], e / 10.0 if nf == 5 else None)


@pytest.mark.parametrize("n", [(32, 32, 32), (37, 19, 23), (9, 5, 3), (72, 12, 40)])
@pytest.mark.parametrize("order", [7, 5])
@pytest.mark.parametrize("nf", [4, 5])
def test_limiter_rhs_parity(H, oracle, n, order, nf):
    """R16 on rough admissible data (the limiter acts on a large share of the faces) and on smooth data with a jet:
    L of the limited scheme, GPU vs oracle; nf = 5 is BASELINE config 4's field count (the baryon density is limited with
    the same theta as the energy-momentum fields)."""
    for kind in ("rough", "smooth"):
        if kind == "rough":
            U0 = _rough_state(n, 5, nf=nf)
            jets = []
        else:
            c = S.scaled_config(0, n)
            c["nf"] = nf
            U0 = S.make_state(c)
            jets = [((-0.12, 0.03, 0.0), (1.0, 0.5, -0.25))]
        g = H.Hydro(*n, 0.1, 0.02, weno_order=order, nfields=nf)
        o = oracle.Oracle(*n, 0.1, 0.02, weno_order=order, nfields=nf)
        g.set_state(U0), o.set_state(U0)
        g.set_limiter(True), o.set_limiter(True)
        for pos, d in jets:
            g.add_jet(pos, d), o.add_jet(pos, d)
        Lg, Lo = g.eval_rhs(0.5), o.eval_rhs(0.5)
        scale = np.max(np.abs(Lo), axis=(1, 2, 3))
        for f in range(nf):
            # L is recovered from the limited Euler update: (U' - U)/dt costs ulp(U)/dt of absolute accuracy
            tol = 1e-11 * max(scale[f], scale[0]) + 4e-16 * np.max(np.abs(U0[f])) / 0.02
            assert np.max(np.abs(Lg[f] - Lo[f])) <= tol, (kind, f)
        ng, no = g.limited_faces(), o.limited_faces()
        if kind == "rough":
            assert no > 0 and abs(ng - no) <= max(2, 0.01 * no)
        else:
            assert ng == no == 0
        g.close(), o.close()


def test_limiter_run_five_fields(H, oracle):
    """Limiter x nf = 5 over a run (the jet/cap case with a baryon density): parity, no cap events, N_B limited too."""
    c = S.scaled_config(2, (64, 32, 32))
    c["nf"] = 5
    c["jets"] = [((-2.0, 0.0, 0.0), (1.0, 0.0, 0.0))]
    steps = 40
    c, U0, g, o = make_pair(H, oracle, c)
    g.set_limiter(True), o.set_limiter(True)
    g.step(steps), o.step(steps)
    Ug, Uo = g.get_fields(), o.get_fields()
    errs = r13(Ug, Uo)
    assert max(errs) < 1e-8, errs
    dg, do = compare_diag(g, o, steps)
    assert dg["ncap"] == do["ncap"] == 0
    ng, no = g.limited_faces(), o.limited_faces()
    assert no > 0 and abs(ng - no) <= max(3, 0.02 * no)
    g.close(), o.close()


def test_limiter_runs(H, oracle):
    """The jet/cap case with the limiter: parity after the run, the cap never fires, the state stays admissible;
    rough data: admissible on the GPU as in the oracle."""
    c = S.scaled_config(2, (64, 32, 32))
    c["jets"] = [((-2.0, 0.0, 0.0), (1.0, 0.0, 0.0))]
    steps = 40
    c, U0, g, o = make_pair(H, oracle, c)
    g.set_limiter(True), o.set_limiter(True)
    g.step(steps), o.step(steps)
    Ug, Uo = g.get_fields(), o.get_fields()
    errs = r13(Ug, Uo)
    assert max(errs) < 1e-8, errs                     # theta = (g0 - delta)/(g0 - g1) amplifies rounding where it acts
    dg, do = compare_diag(g, o, steps)
    assert dg["ncap"] == do["ncap"] == 0
    assert (Ug[0] - np.sqrt(Ug[1] ** 2 + Ug[2] ** 2 + Ug[3] ** 2)).min() > 0
    ng, no = g.limited_faces(), o.limited_faces()
    assert no > 0 and abs(ng - no) <= max(3, 0.02 * no)
    g.close(), o.close()
    n = (24, 20, 16)
    U0 = _rough_state(n, 11)
    g, o = H.Hydro(*n, 0.1, 0.02), oracle.Oracle(*n, 0.1, 0.02)
    g.set_state(U0), o.set_state(U0)
    g.set_limiter(True), o.set_limiter(True)
    g.step(4), o.step(4)
    Ug, Uo = g.get_fields(), o.get_fields()
    assert (Ug[0] - np.sqrt(Ug[1] ** 2 + Ug[2] ** 2 + Ug[3] ** 2)).min() > 0 and g.diag()["ncap"] == 0
    assert max(r13(Ug, Uo)) < 1e-7
    g.close(), o.close()
    with pytest.raises(H.HydroError):
        H.Hydro(8, 8, 8, 0.1, 0.02, precision=32).set_limiter(True)


# ------------------------------------------------------------------------------------------------ invariants on the GPU
def test_gpu_uniform_state_and_symmetry(H):
    n = (40, 24, 17)
    ones = np.ones((n[2], n[1], n[0]))
    U0 = S.prim_to_cons(3.7 * ones, 0.3 * ones, -0.2 * ones, 0.1 * ones)
    g = H.Hydro(*n, 0.1, 0.02)
    g.set_state(U0)
    assert np.all(g.eval_rhs(0.0) == 0.0)               # P2: bitwise
    g.step(3)
    U = g.get_fields()
    assert np.array_equal(U, np.broadcast_to(U[:, :1, :1, :1], U.shape))
    g.close()
    n = (32, 24, 20)                                     # P6: mirror symmetry
    U0 = S.gaussian_flow(n, 0.1, peak=10.0, sigma=(0.5, 0.4, 0.6), R=(1.0, 0.8, 1.2), ucoef=0.2, noise=0.0)
    g = H.Hydro(*n, 0.1, 0.02)
    g.set_state(U0)
    g.step(4)
    U = g.get_fields()
    g.close()
    scale = np.abs(U).max(axis=(1, 2, 3))
    for axis, odd in ((3, 1), (2, 2), (1, 3)):
        F = np.flip(U, axis=axis)
        for f in range(4):
            sign = -1.0 if f == odd else 1.0
            assert np.max(np.abs(U[f] - sign * F[f])) <= 1e-13 * scale[f]


def test_device_pointers_and_streams(H, oracle):
    """set_state / get_fields with device memory (torch tensors) on a caller-owned torch stream."""
    import torch
    c = S.CONFIGS[0]
    U0 = S.make_state(0)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        Ud = torch.from_numpy(U0).cuda()
    st.synchronize()
    g = H.Hydro(*c["n"], c["dx"], c["dt"], stream=st)
    g.set_state(Ud)
    g.step(2)
    out = torch.empty_like(Ud)
    g.get_fields(out=out)
    g2 = H.Hydro(*c["n"], c["dx"], c["dt"])
    g2.set_state(U0)
    g2.step(2)
    assert np.array_equal(out.cpu().numpy(), g2.get_fields())
    assert g.launch_count() == 2 * (3 * 5) + 1
    g.close(), g2.close()


def test_graph_replay_equals_individual_launches(H):
    """hydro_step replays one captured RK3 step as a CUDA graph (the step counter lives on the device); with per-kernel
    profiling on it launches the 15 kernels one by one.  Same kernels, same arguments: bitwise equal states, equal
    diagnostics and launch counts, across split calls, a jet added mid-run (recapture) and set_step."""
    c = S.scaled_config(0, (40, 24, 20))
    U0 = S.make_state(c)
    out = []
    for profiled in (False, True):
        g = H.Hydro(*c["n"], c["dx"], c["dt"])
        g.set_state(U0)
        g.set_profiling(profiled)
        g.add_jet((-1.0, 0.0, 0.0), (1.0, 0.0, 0.0))
        g.step(3)
        g.step(1)
        g.add_jet((0.3, 0.2, -0.1), (0.0, 1.0, 0.5))
        g.step(4)
        g.set_deposit_width(0.1)
        g.step(2)
        g.set_step(20)
        g.step(2)
        d = g.diag()
        out.append((g.get_fields(), d, g.last_stage_q(), g.launch_count()))
        g.close()
    (Ua, da, qa, la), (Ub, db, qb, lb) = out
    assert np.array_equal(Ua, Ub) and la == lb
    assert da["step"] == db["step"] == 22 and da["ncap"] == db["ncap"]
    assert np.array_equal(da["deposited"], db["deposited"]) and np.array_equal(da["alpha"], db["alpha"])
    assert np.array_equal(qa, qb)


def test_checkpoint_resume_is_bitwise(H):
    """(U, step counter, jets) is a complete checkpoint: a run resumed in a NEW handle continues bitwise."""
    c = S.scaled_config(0, (40, 24, 20))
    U0 = S.make_state(c)
    jets = [((-1.0, 0.0, 0.0), (1.0, 0.0, 0.0)), ((0.3, 0.2, -0.1), (0.0, 1.0, 0.5))]
    g = H.Hydro(*c["n"], c["dx"], c["dt"])
    g.set_state(U0)
    for pos, d in jets:
        g.add_jet(pos, d)
    g.step(4)
    Uc, dep_c = g.get_fields(), g.diag()["deposited"]
    g.step(5)
    Uref, dref = g.get_fields(), g.diag()
    r = H.Hydro(*c["n"], c["dx"], c["dt"])
    r.set_state(Uc)
    for pos, d in jets:
        r.add_jet(pos, d)
    r.set_step(4)
    r.step(5)
    assert np.array_equal(r.get_fields(), Uref)
    dr = r.diag()
    assert dr["step"] == 9 and np.allclose(dep_c + dr["deposited"], dref["deposited"], rtol=1e-13, atol=0)
    g.close(), r.close()


def test_non_finite_state_is_flagged(H, oracle):
    """has_nan: a NaN or an infinity in any conserved field of any cell is flagged by k_prim (0 * x summed over the fields),
    like the oracle does; ragged and dense grids (the scalar and the vector path of k_prim), both precisions."""
    for n in ((6, 5, 4), (7, 5, 3), (32, 8, 8)):
        c = S.scaled_config(0, n)
        U0 = S.make_state(c, noise=False)
        for prec in (64, 32):
            for f, cell, bad in ((None, None, None), (0, (0, 0, 0), np.nan), (1, (n[2] - 1, n[1] - 1, n[0] - 1), np.inf),
                                 (2, (1, 2, 3), -np.inf), (3, (2, 0, 1), np.nan)):
                U = U0.copy()
                if f is not None:
                    U[(f,) + cell] = bad
                g = H.Hydro(*n, c["dx"], c["dt"], precision=prec)
                g.set_state(U.astype(np.float64 if prec == 64 else np.float32))
                g.step(1)                                    # the flag is committed with the stages of a step
                flag = g.diag()["has_nan"]
                g.close()
                if prec == 64:
                    o = oracle.Oracle(*n, c["dx"], c["dt"])
                    o.set_state(U)
                    o.eval_rhs(0.0)
                    assert o.diag()["has_nan"] == (0 if f is None else 1)
                    o.close()
                assert flag == (0 if f is None else 1), (n, prec, f, cell, bad)


def test_error_paths(H):
    g = H.Hydro(8, 8, 8, 0.1, 0.02)
    with pytest.raises(H.HydroError):
        g.add_jet((0, 0, 0), (0, 0, 0))
    with pytest.raises(H.HydroError):
        g.step(-1)
    g.close()
    with pytest.raises(H.HydroError):
        H.Hydro(8, 8, 8, 0.1, 0.0)

"""Pins of the oracle's positivity-preserving flux limiter, reading R16 (PAPER.md:25 cites the
positivity-preserving FD-WENO paper [2], without details).  What is pinned is the theory the reading is
built on and the properties it must deliver, not the oracle's own formulas:
  * Lax-Friedrichs property U -+ F/alpha admissible for alpha >= the largest wavespeed (why F^L is safe);
  * with the limiter the state stays admissible (g = E - |M| > 0) where the unlimited scheme does not;
  * smooth data: theta = 1 everywhere, i.e. the scheme is unchanged; conservation and symmetry are untouched."""
import numpy as np

from paper_1511_02137_b200 import synthetic as S


def g_over_E(U):
    return (U[0] - np.sqrt(U[1] ** 2 + U[2] ** 2 + U[3] ** 2)) / U[0]


def test_lax_friedrichs_states_are_admissible(oracle):
    rng = np.random.default_rng(17)
    for _ in range(2000):
        e = 10.0 ** rng.uniform(-3, 3)
        v = rng.uniform(0, 0.999) * (lambda d: d / np.linalg.norm(d))(rng.normal(size=3))
        gam = 1.0 / np.sqrt(1.0 - v @ v)
        U = S.prim_to_cons(np.array([e]), *(np.array([gam * vi]) for vi in v))[:, 0]
        p = e / 3.0
        lam = oracle.wavespeeds(*v)
        for d in range(3):
            F = np.array([U[1 + d], U[1] * v[d], U[2] * v[d], U[3] * v[d]])
            F[1 + d] += p
            for a in (lam[d], 1.0):
                for sgn in (-1.0, 1.0):
                    W = U + sgn * F / a
                    assert W[0] - np.linalg.norm(W[1:]) >= -1e-12 * W[0], (e, v, d, a, sgn)


def _rough_state(n, seed, vmax=0.98):
    rng = np.random.default_rng(seed)
    shape = (n[2], n[1], n[0])
    e = 10.0 ** rng.uniform(-2, 2, shape)
    vm = rng.uniform(0, vmax, shape)
    d = rng.normal(size=(3,) + shape)
    d /= np.linalg.norm(d, axis=0)
    u = vm / np.sqrt(1 - vm * vm) * d
    return S.prim_to_cons(e, u[0], u[1], u[2])


def test_rough_data_stay_admissible_only_with_the_limiter(oracle):
    n = (16, 12, 10)
    U0 = _rough_state(n, 4)
    assert g_over_E(U0).min() > 0
    res = {}
    for lim in (False, True):
        o = oracle.Oracle(*n, 0.1, 0.02)                      # dt/dx = 0.2 as in the paper: 3 alpha dt/dx <= 0.6
        o.set_state(U0)
        o.set_limiter(lim)
        gmin = 1.0
        for _ in range(5):
            o.step(1)
            gmin = min(gmin, g_over_E(o.get_fields()).min())
        res[lim] = (gmin, o.diag()["ncap"], o.limited_faces())
        o.close()
    assert res[False][0] < 0 and res[False][1] > 0            # the plain scheme leaves the admissible set (cap fires)
    assert res[True][0] > 0 and res[True][1] == 0 and res[True][2] > 0


def test_jet_case_no_cap_events(oracle):
    c = S.scaled_config(2, (48, 24, 24))
    U0 = S.make_state(c)
    o = oracle.Oracle(*c["n"], c["dx"], c["dt"])
    o.set_state(U0)
    o.add_jet((-1.5, 0.0, 0.0), (1.0, 0.0, 0.0))
    o.set_limiter(True)
    gmin = 1.0
    for _ in range(45):
        o.step(1)
        gmin = min(gmin, g_over_E(o.get_fields()).min())
    d = o.diag()
    assert gmin > 0 and d["ncap"] == 0 and d["has_nan"] == 0 and o.limited_faces() > 0
    o.close()


def test_smooth_flow_is_not_touched_and_invariants(oracle):
    n = (20, 16, 12)
    U0 = S.gaussian_flow(n, 0.1, peak=10.0, sigma=(0.5, 0.4, 0.6), R=(1.0, 0.8, 1.2), ucoef=0.2, noise=0.0)
    a, b = oracle.Oracle(*n, 0.1, 0.02), oracle.Oracle(*n, 0.1, 0.02)
    a.set_state(U0), b.set_state(U0)
    b.set_limiter(True)
    a.step(3), b.step(3)
    Ua, Ub = a.get_fields(), b.get_fields()
    assert b.limited_faces() == 0
    assert np.max(np.abs(Ua - Ub)) < 1e-13 * np.max(np.abs(Ua))      # F^L + 1*(F^H - F^L) vs F^H: rounding only
    scale = np.abs(Ub).max(axis=(1, 2, 3))
    for axis, odd in ((3, 1), (2, 2), (1, 3)):                        # P6 mirror symmetry survives
        F = np.flip(Ub, axis=axis)
        for f in range(4):
            assert np.max(np.abs(Ub[f] - (-1.0 if f == odd else 1.0) * F[f])) <= 1e-13 * scale[f]
    a.close(), b.close()
    # P2: uniform state stays uniform with the limiter on
    ones = np.ones((6, 7, 9))
    U0 = S.prim_to_cons(2.0 * ones, 0.5 * ones, -0.3 * ones, 0.1 * ones)
    o = oracle.Oracle(9, 7, 6, 0.1, 0.02)
    o.set_state(U0)
    o.set_limiter(True)
    assert np.all(o.eval_rhs(0.0) == 0.0)
    o.close()


def test_conservation_with_limiter_active(oracle):
    """Flux form: the limiter changes fluxes, never the telescoping sum.  Rough data in the middle of a uniform
    background at rest: one step moves information by 3 stages x 4 cells = 12 < 14 cells of margin, so the totals are
    conserved to rounding."""
    n = (36, 36, 36)
    ones = np.ones((n[2], n[1], n[0]))
    U0 = S.prim_to_cons(1.0 * ones, 0 * ones, 0 * ones, 0 * ones)
    U0[:, 14:22, 14:22, 14:22] = _rough_state((8, 8, 8), 9, vmax=0.95)
    o = oracle.Oracle(*n, 0.1, 0.02)
    o.set_state(U0)
    o.set_limiter(True)
    o.step(1)
    U = o.get_fields()
    assert o.limited_faces() > 0 and g_over_E(U).min() > 0
    for f in range(4):
        s0, s1 = U0[f].sum(dtype=np.longdouble), U[f].sum(dtype=np.longdouble)
        assert abs(float(s1 - s0)) < 1e-11 * float(np.abs(U0[f]).sum())
    o.close()

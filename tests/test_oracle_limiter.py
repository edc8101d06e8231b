"""Pins of the oracle's positivity-preserving flux limiter, reading R16 (PAPER.md:25 cites the
positivity-preserving FD-WENO paper [2], without details).  What is pinned is the theory the reading is
built on and the properties it must deliver, not the oracle's own formulas:
  * Lax-Friedrichs property U -+ F/alpha admissible for alpha >= the largest wavespeed (why F^L is safe);
  * with the limiter the state stays admissible (g = E - |M| > 0) where the unlimited scheme does not;
  * smooth data: theta = 1 everywhere, i.e. the scheme is unchanged; conservation and symmetry are untouched."""
import numpy as np
import pytest

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


# ------------------------------------------------------------------ R16's constants: exact case with a linear g
def _weno7_from_definition(v, eps):
    """WENO7-JS value at the right face of the centre cell from 7 cell values, straight from the definition (O5):
    cubic p_k with the prescribed cell averages on sub-stencil k (4x4 linear solve), q_k = p_k(face),
    beta_k = sum_l int_cell dx^(2l-1) (d^l p_k)^2, weights d_k/(eps + beta_k)^2, d = (1, 12, 18, 4)/35."""
    from numpy.polynomial import polynomial as Pl
    d = np.array([1.0, 12.0, 18.0, 4.0]) / 35.0
    q, beta = np.zeros(4), np.zeros(4)
    for k in range(4):
        A = np.array([[((r + 0.5) ** (c + 1) - (r - 0.5) ** (c + 1)) / (c + 1) for c in range(4)] for r in range(4)])
        coef = np.linalg.solve(A, v[k:k + 4])              # unit cells at 0..3; the centre cell sits at 3 - k
        pos = 3 - k
        q[k] = Pl.polyval(pos + 0.5, coef)
        for l in (1, 2, 3):
            dl = Pl.polyder(coef, l)
            sq = Pl.polyint(Pl.polymul(dl, dl))
            beta[k] += Pl.polyval(pos + 0.5, sq) - Pl.polyval(pos - 0.5, sq)
    a = d / (eps + beta) ** 2
    return float(a @ q / a.sum())


@pytest.mark.parametrize("seed,span,vlo,small", [(3, 0.5, 0.6, False), (4, 1.0, 0.3, True)])
def test_r16_constants_on_a_linear_admissibility_function(oracle, seed, span, vlo, small):
    """Reading R16 states: the limited Euler update is the average of the six states
    W_f = U^L_i -+ 6 (dt/dx) theta_f C_f, and theta_f is the largest value for which g(W_f) >= delta_i =
    min(1e-8 E^L_i, g(U^L_i)) in both cells of the face, as far as the concavity of g = E - |M| can tell.  In 1-D with
    momenta along x only, g = E - |M_x| is LINEAR wherever M_x keeps its sign along the segment U^L_i .. W_f(1); there
    the concavity bound is exact and theta_f is the true supremum, found here by bisection on that definition (no secant
    formula), with U^L, F^L and the WENO7 fluxes rebuilt from eq. (1), the Lax-Friedrichs splitting and the definition
    of the reconstruction.  On the remaining limited faces (M_x changes sign: g is only concave) the oracle's theta must
    be admissible and not larger than the supremum.  The oracle's face fluxes are recovered from its L by summing the
    divergence from the left boundary, where a uniform pad makes the flux known.  A different face multiplier
    (6 -> 12) or a different delta (1e-8 -> 1e-4) moves theta on the linear faces and fails this test.  The second, rougher
    parameter set reaches theta < 0.25 on linear faces (a theta clipped or floored there would go unnoticed otherwise)."""
    nx, pad, dx, dt, eps = 72, 6, 0.1, 0.02, 1e-6
    lam = dt / dx
    rng = np.random.default_rng(seed)
    e = 10.0 ** rng.uniform(-span, span, nx)
    v = rng.uniform(vlo, 0.985, nx)
    e[:pad], v[:pad] = e[pad], v[pad]                     # uniform pad: the flux through the left boundary is F(U_0)
    gam2 = 1.0 / (1.0 - v * v)
    E = (4.0 / 3.0) * e * gam2 - e / 3.0                  # eq. (1), p = e/3
    M = (4.0 / 3.0) * e * gam2 * v
    U = np.stack([E, M])                                  # (E, M_x); M_y = M_z = 0 exactly
    F = np.stack([M, M * v + e / 3.0])                    # F^x = (M_x, M_x v_x + p)
    cs = 1.0 / np.sqrt(3.0)
    alpha = np.max((v + cs) / (1.0 + v * cs))             # v > 0: the faster acoustic wave (1-D addition formula)
    fp, fm = 0.5 * (F + alpha * U), 0.5 * (F - alpha * U)
    cl = lambda i: min(max(i, 0), nx - 1)                 # zero-gradient ghosts = index clamping (R8b)
    FH, FL = np.zeros((2, nx + 1)), np.zeros((2, nx + 1))
    for f in range(nx + 1):                               # face f lies between cells i = f-1 and i+1 = f
        i = f - 1
        for q in range(2):
            wp = np.array([fp[q, cl(i + m)] for m in range(-3, 4)])
            wm = np.array([fm[q, cl(i + 1 - m)] for m in range(-3, 4)])
            FH[q, f] = _weno7_from_definition(wp, eps) + _weno7_from_definition(wm, eps)
            FL[q, f] = fp[q, cl(i)] + fm[q, cl(i + 1)]
    C = FH - FL
    UL = U - lam * (FL[:, 1:] - FL[:, :-1])
    g = lambda W: W[0] - abs(W[1])
    cells = lambda f: [(c, sgn) for c, sgn in ((f - 1, -1.0), (f, 1.0)) if 0 <= c < nx]

    def admissible(f, t, slack=0.0):
        return all(g(UL[:, c] + sgn * 6.0 * lam * t * C[:, f]) >= min(1e-8 * UL[0, c], g(UL[:, c])) - slack * UL[0, c]
                   for c, sgn in cells(f))

    theta, linear = np.ones(nx + 1), np.ones(nx + 1, bool)
    for f in range(nx + 1):
        if not admissible(f, 1.0):
            lo, hi = 0.0, 1.0
            for _ in range(200):
                mid = 0.5 * (lo + hi)
                lo, hi = (mid, hi) if admissible(f, mid) else (lo, mid)
            theta[f] = lo
            linear[f] = all(UL[1, c] > 0 and UL[1, c] + sgn * 6.0 * lam * C[1, f] > 0 for c, sgn in cells(f))
    lim = theta < 1.0
    assert np.sum(lim & linear & (theta > 0.05) & (theta < 0.95)) >= 4      # the case must exercise the exact regime
    assert not small or np.sum(lim & linear & (theta > 0.02) & (theta < 0.25)) >= 1
    o = oracle.Oracle(nx, 1, 1, dx, dt)
    U4 = np.zeros((4, 1, 1, nx))
    U4[0, 0, 0], U4[1, 0, 0] = E, M
    o.set_state(U4)
    o.set_limiter(True)
    L = o.eval_rhs(0.0)
    assert abs(o.diag()["alpha"][0] - alpha) < 1e-14
    assert o.limited_faces() == int(lim.sum())
    assert np.all(L[2] == 0.0) and np.all(L[3] == 0.0)
    assert not lim[0] and abs(C[0, 0]) < 1e-13 and abs(C[1, 0]) < 1e-13       # the pad did its job
    Fo = np.zeros((2, nx + 1))                                                # the oracle's limited face fluxes
    Fo[:, 0] = FL[:, 0]
    Fo[:, 1:] = Fo[:, :1] - dx * np.cumsum(L[:2, 0, 0], axis=1)
    scale = np.max(np.abs(FH), axis=1)
    for f in range(nx + 1):
        if not lim[f]:
            assert np.max(np.abs(Fo[:, f] - FH[:, f]) / scale) < 1e-10, f
            continue
        q = int(np.argmax(np.abs(C[:, f]) / scale))
        th_o = (Fo[q, f] - FL[q, f]) / C[q, f]                               # one theta for all fields
        assert np.max(np.abs(Fo[:, f] - (FL[:, f] + th_o * C[:, f])) / scale) < 1e-10, f
        if linear[f]:
            assert abs(th_o - theta[f]) < 1e-8, (f, th_o, theta[f])          # exact: on the boundary g = delta
        else:
            assert -1e-9 <= th_o <= theta[f] + 1e-8 and admissible(f, max(th_o, 0.0), slack=1e-9), (f, th_o, theta[f])
    o.close()


def test_limiter_is_mirror_symmetric_on_rough_data_up_to_the_boundary_cells(oracle):
    """x -> -x (reverse the line, flip the sign of M_x) must mirror the limited RHS, boundary cells included: ghost cells
    impose no admissibility condition, the first and the last interior cell do (P6 with the limiter active everywhere)."""
    nx, dx, dt = 40, 0.1, 0.02
    nlim = 0
    for seed in range(8):
        rng = np.random.default_rng(100 + seed)
        e = 10.0 ** rng.uniform(-1.0, 1.0, nx)
        v = rng.uniform(-0.98, 0.98, nx)
        gam2 = 1.0 / (1.0 - v * v)
        U = np.zeros((4, 1, 1, nx))
        U[0, 0, 0] = (4.0 / 3.0) * e * gam2 - e / 3.0
        U[1, 0, 0] = (4.0 / 3.0) * e * gam2 * v
        Um = U[..., ::-1].copy()
        Um[1] = -Um[1]
        out = []
        for W in (U, Um):
            o = oracle.Oracle(nx, 1, 1, dx, dt)
            o.set_state(W)
            o.set_limiter(True)
            out.append((o.eval_rhs(0.0), o.limited_faces()))
            o.close()
        (L, n1), (Lm, n2) = out
        assert n1 == n2
        nlim += n1
        scale = np.max(np.abs(L), axis=(1, 2, 3))
        assert np.max(np.abs(Lm[0] - L[0][..., ::-1])) < 1e-11 * scale[0]
        assert np.max(np.abs(Lm[1] + L[1][..., ::-1])) < 1e-11 * scale[1]
    assert nlim > 40

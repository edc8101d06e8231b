"""Pins P1, P3, P8 (+ wavespeed / LF-flux / jet-index pins) of the CPU oracle -- scalar pieces.

Each expected value here comes from the paper's equations or from textbook mathematics, never from the
oracle itself and never from the CUDA path.
"""
import math

import numpy as np
import pytest
from numpy.polynomial import polynomial as Pl

from conftest import read_golden


# ------------------------------------------------------------------ P1: con2prim round trip (eq. 1, EOS p=e/3)
def _cons(e, v):
    """eq. (1) PAPER.md:17-19 with u^mu = gamma (1, v), p = e/3: E = (e+p)gamma^2 - p, M = (e+p)gamma^2 v."""
    v = np.asarray(v, float)
    g2 = 1.0 / (1.0 - v @ v)
    p = e / 3.0
    return (e + p) * g2 - p, (e + p) * g2 * v


def test_p1_con2prim_round_trip(oracle):
    rng = np.random.default_rng(7)
    for _ in range(2000):
        e = 10.0 ** rng.uniform(-3, 3)
        vmag = rng.uniform(0, 0.999)
        n = rng.normal(size=3)
        n /= np.linalg.norm(n)
        v = vmag * n
        E, M = _cons(e, v)
        P = oracle.con2prim(E, *M)
        g2 = 1.0 / (1.0 - vmag ** 2)
        assert P["limited"] == 0
        assert abs(P["e"] - e) <= 1e-12 * g2 * e
        assert abs(P["p"] - e / 3.0) <= 1e-12 * g2 * e
        assert np.max(np.abs(P["v"] - v)) <= 1e-12 * g2
        # north_star closed form e = -E + sqrt(4E^2 - 3M^2) (cancellation-prone, so looser)
        assert abs(P["e"] - (-E + math.sqrt(4 * E * E - 3 * (M @ M)))) <= 1e-10 * g2 * e


def test_p1_rest_frame_exact_and_baryon(oracle):
    P = oracle.con2prim(7.25, 0.0, 0.0, 0.0, NB=2.0)
    assert P["e"] == 7.25 and np.all(P["v"] == 0.0) and P["n"] == 2.0
    # N_B = n gamma  =>  n = N_B sqrt(1 - v^2)
    E, M = _cons(3.0, [0.6, 0.0, 0.0])
    P = oracle.con2prim(E, *M, NB=5.0)
    assert abs(P["n"] - 5.0 * 0.8) < 1e-14


def test_p1_admissibility_cap_R9(oracle):
    # |M| > (1 - delta) E: momenta are scaled onto the cap, the result is finite and subluminal
    P = oracle.con2prim(1.0, 0.9, 0.9, 0.0)
    v = np.linalg.norm(P["v"])
    assert P["limited"] == 1 and np.isfinite(P["e"]) and P["e"] > 0 and v < 1.0
    assert abs(P["v"][0] - P["v"][1]) < 1e-15 and P["v"][2] == 0.0      # direction kept
    # E below the floor
    P = oracle.con2prim(-1.0, 0.0, 0.0, 0.0)
    assert P["limited"] == 1 and abs(P["e"] / oracle.E_FLOOR - 1) < 1e-15
    # continuity at the cap: just inside and just outside give nearly the same primitives
    d = oracle.V_CAP_DELTA
    a = oracle.con2prim(2.0, 2.0 * (1 - d) * (1 - 1e-13), 0, 0)
    b = oracle.con2prim(2.0, 2.0 * (1 - d) * (1 + 1e-13), 0, 0)
    assert a["limited"] == 0 and b["limited"] == 1
    assert abs(a["v"][0] - b["v"][0]) < 1e-9 and abs(a["e"] - b["e"]) < 1e-9


# ------------------------------------------------------------------ wavespeeds (a-2): special cases + brute force
def test_wavespeed_special_cases(oracle):
    cs = 1 / math.sqrt(3)
    for v in [0.0, 0.1, -0.4, 0.9, -0.99]:
        lam = oracle.wavespeeds(v, 0.0, 0.0)
        # v parallel to d: relativistic velocity addition (v +- cs)/(1 +- v cs)
        expect = max(abs((v + cs) / (1 + v * cs)), abs((v - cs) / (1 - v * cs)))
        assert abs(lam[0] - expect) < 1e-14
        # v perpendicular to d: cs sqrt((1-v^2)/(1-v^2 cs^2))
        perp = cs * math.sqrt((1 - v * v) / (1 - v * v / 3))
        assert abs(lam[1] - perp) < 1e-14 and abs(lam[2] - perp) < 1e-14


def _flux(oracle, U, d):
    """F^d(U) from eq. (1): (M_d, M_i v_d + p delta_id), primitives by the (P1-pinned) oracle con2prim."""
    P = oracle.con2prim(*U)
    F = np.array([U[1 + d], U[1] * P["v"][d], U[2] * P["v"][d], U[3] * P["v"][d]])
    F[1 + d] += P["p"]
    return F


def test_wavespeed_is_spectral_radius_of_flux_jacobian(oracle):
    """Brute force: eigenvalues of dF^d/dU by central differences are {lam-, v_d, v_d, lam+}."""
    rng = np.random.default_rng(3)
    for _ in range(20):
        e = 10 ** rng.uniform(-1, 1.5)
        v = rng.uniform(-0.55, 0.55, size=3)
        E, M = _cons(e, v)
        U = np.array([E, *M])
        lam = oracle.wavespeeds(*v)
        for d in range(3):
            J = np.zeros((4, 4))
            for c in range(4):
                h = 1e-6 * max(abs(U[c]), E)
                Up, Um = U.copy(), U.copy()
                Up[c] += h
                Um[c] -= h
                J[:, c] = (_flux(oracle, Up, d) - _flux(oracle, Um, d)) / (2 * h)
            ev = np.linalg.eigvals(J)
            assert np.max(np.abs(ev.imag)) < 1e-5
            assert abs(np.max(np.abs(ev.real)) - lam[d]) < 2e-6
            assert np.sum(np.abs(ev.real - v[d]) < 1e-5) >= 2       # the two entropy/shear waves


# ------------------------------------------------------------------ P3: WENO7
D_IDEAL = np.array([1, 12, 18, 4]) / 35.0


def _cell_averages(coef, i0, n):
    """cell averages over unit cells [i-1/2, i+1/2], i = i0..i0+n-1, of the polynomial `coef` (low->high)."""
    A = Pl.polyint(coef)
    return np.array([Pl.polyval(i + 0.5, A) - Pl.polyval(i - 0.5, A) for i in range(i0, i0 + n)])


def test_p3_candidates_reproduce_cubics_and_ideal_weights_degree6(oracle):
    rng = np.random.default_rng(11)
    for deg in range(0, 7):
        coef = rng.normal(size=deg + 1)
        v = _cell_averages(coef, -3, 7)                  # cells i-3..i+3 around i = 0
        exact = Pl.polyval(0.5, coef)                    # value at the face i+1/2
        q, beta, beta_sos, om = oracle.weno7_parts(v)
        scale = np.max(np.abs(v)) + 1
        if deg <= 3:
            assert np.max(np.abs(q - exact)) < 1e-13 * scale
        assert abs(D_IDEAL @ q - exact) < 2e-13 * scale
        # the 420-denominator form of sum d_k q_k
        lin = np.array([-3, 25, -101, 319, 214, -38, 4]) @ v / 420.0
        assert abs(D_IDEAL @ q - lin) < 1e-13 * scale
    # degree 7 is NOT reproduced (the scheme is exactly 7th order)
    v = _cell_averages(np.eye(8)[7], -3, 7)
    q = oracle.weno7_parts(v)[0]
    assert abs(D_IDEAL @ q - 0.5 ** 7) > 1e-3


def _beta_from_definition(v4, cell_pos):
    """beta = sum_{l=1..3} int_cell dx^{2l-1} (d^l p/dx^l)^2 for the cubic p with the 4 given cell averages;
    cells are unit cells at integer positions 0..3, smoothness measured over cell `cell_pos`."""
    # solve for cubic coefficients from the 4 average conditions
    A = np.zeros((4, 4))
    for r in range(4):
        for c in range(4):
            A[r, c] = ((r + 0.5) ** (c + 1) - (r - 0.5) ** (c + 1)) / (c + 1)
    coef = np.linalg.solve(A, v4)
    tot = 0.0
    for l in (1, 2, 3):
        dl = Pl.polyder(coef, l)
        sq = Pl.polyint(Pl.polymul(dl, dl))
        tot += Pl.polyval(cell_pos + 0.5, sq) - Pl.polyval(cell_pos - 0.5, sq)
    return tot


def test_p3_smoothness_indicators_match_integral_definition(oracle):
    rng = np.random.default_rng(5)
    for _ in range(50):
        v = rng.normal(size=7)
        q, beta, beta_sos, om = oracle.weno7_parts(v)
        for k in range(4):
            ref = _beta_from_definition(v[k:k + 4], 3 - k)      # centre cell d is index 3
            assert abs(beta[k] - ref) < 1e-10 * (1 + ref)
            assert abs(beta_sos[k] - ref) < 1e-10 * (1 + ref)
        assert np.all(beta >= 0)
        assert abs(om.sum() - 1) < 1e-14
    # constants: beta = 0 exactly, weights ideal, value reproduced
    q, beta, beta_sos, om = oracle.weno7_parts(np.full(7, 3.25))
    assert np.all(beta == 0) and np.all(beta_sos == 0)
    assert np.max(np.abs(om - D_IDEAL)) < 1e-15
    assert abs(oracle.weno7(np.full(7, 3.25)) - 3.25) < 2e-15


def test_p3_nonlinear_weights_limits(oracle):
    # beta << eps -> ideal weights
    x = np.arange(-3, 4) * 0.01
    q, beta, _, om = oracle.weno7_parts(1e-4 * np.sin(x))
    assert np.max(np.abs(om - D_IDEAL)) < 1e-3
    # step between cells i and i+1: only sub-stencil 0 (cells i-3..i) is smooth
    v = np.array([1.0, 1, 1, 1, 5, 5, 5])
    q, beta, _, om = oracle.weno7_parts(v)
    assert om[0] > 1 - 1e-6 and abs(oracle.weno7(v) - 1.0) < 1e-5
    # step between i-1 and i: only sub-stencil 3 (cells i..i+3) is smooth
    v = np.array([1.0, 1, 1, 5, 5, 5, 5])
    q, beta, _, om = oracle.weno7_parts(v)
    assert om[3] > 1 - 1e-6 and abs(oracle.weno7(v) - 5.0) < 1e-5


def test_p3_weight_exponent_and_epsilon_R3(oracle):
    """Reading R3 (WENO-JS: omega_k ~ d_k / (eps + beta_k)^2, eps absolute): the weight RATIOS follow from the smoothness
    indicators of the integral definition (computed here by quadrature of the sub-stencil cubics, not by the oracle).
    An exponent of 1, or an eps that scales with the data, fails this."""
    rng = np.random.default_rng(19)
    for scale in (1e-3, 1.0, 50.0):
        v = scale * rng.normal(size=7)
        for eps in (1e-6, 1e-2):
            om = oracle.weno7_parts(v, eps)[3]
            beta = np.array([_beta_from_definition(v[k:k + 4], 3 - k) for k in range(4)])
            for k in range(1, 4):
                expect = (D_IDEAL[k] / D_IDEAL[0]) * ((eps + beta[0]) / (eps + beta[k])) ** 2
                assert abs(om[k] / om[0] - expect) < 1e-9 * expect, (scale, eps, k)


def _substencil_cubic(v4):
    """coefficients (ascending) of the cubic whose averages over the unit cells at 0, 1, 2, 3 are v4"""
    A = np.zeros((4, 4))
    for r in range(4):
        for c in range(4):
            A[r, c] = ((r + 0.5) ** (c + 1) - (r - 0.5) ** (c + 1)) / (c + 1)
    return np.linalg.solve(A, v4)


def test_p3_reconstructed_value_from_the_definition_R3(oracle):
    """The VALUE the solver's reconstruction returns (oracle.weno7: the routine the interface flux calls, not the
    diagnostic copy behind weno7_parts) is sum_k omega_k q_k with everything rebuilt here from the definition: q_k = the
    sub-stencil cubic (given by its cell averages) at the face, beta_k = the integral definition by quadrature,
    omega_k ~ d_k / (eps + beta_k)^2 (reading R3).  An exponent of 1 or a relative eps in the solver's routine fails this."""
    rng = np.random.default_rng(23)
    for scale in (1e-3, 1.0, 50.0):
        for eps in (1e-6, 1e-2):
            v = scale * rng.normal(size=7)
            q = np.array([Pl.polyval(3 - k + 0.5, _substencil_cubic(v[k:k + 4])) for k in range(4)])
            beta = np.array([_beta_from_definition(v[k:k + 4], 3 - k) for k in range(4)])
            al = D_IDEAL / (eps + beta) ** 2
            expect = float(al @ q / al.sum())
            got = oracle.weno7(v, eps)
            assert abs(got - expect) < 1e-11 * (np.max(np.abs(v)) + abs(expect)), (scale, eps, got, expect)
            wrong = float((D_IDEAL / (eps + beta)) @ q / (D_IDEAL / (eps + beta)).sum())     # exponent 1 is distinguishable
            assert abs(wrong - expect) > 1e-6 * np.max(np.abs(v)) or scale == 1e-3


def _fd_derivative_error(oracle, f, dfdx, n, eps):
    """(W_{i+1/2} - W_{i-1/2})/dx vs f'(x_i) with point values f(x_i): the finite-difference use of O5-O7."""
    dx = 1.0 / n
    xs = (np.arange(-4, n + 4) + 0.5) * dx
    fv = f(xs)
    W = np.array([oracle.weno7(fv[m:m + 7], eps) for m in range(0, n + 1)])      # faces m+3+1/2
    der = (W[1:] - W[:-1]) / dx                                                # cells m = 4 .. n+3
    return np.max(np.abs(der - dfdx(xs[4:n + 4])))


def test_p3_seventh_order_convergence(oracle):
    # ideal-weight regime (beta << eps): design order 7 (7.2-8.3 observed)
    f = lambda x: 1e-3 * np.sin(2 * np.pi * x)
    df = lambda x: 1e-3 * 2 * np.pi * np.cos(2 * np.pi * x)
    e1, e2 = (_fd_derivative_error(oracle, f, df, n, 1e-6) for n in (16, 32))
    assert math.log2(e1 / e2) > 6.8
    # genuinely nonlinear weights, no critical points: exp(2x) (6.7-6.9)
    f = lambda x: np.exp(2 * x)
    df = lambda x: 2 * np.exp(2 * x)
    e1, e2 = (_fd_derivative_error(oracle, f, df, n, 1e-6) for n in (20, 40))
    assert 6.4 < math.log2(e1 / e2) < 8.5


def test_p3_polynomial_derivative_exact_with_ideal_weights(oracle):
    """With ideal weights the FD flux difference differentiates degree <= 7 polynomials exactly, not degree 8."""
    dx = 1.0 / 16
    xs = (np.arange(-4, 5)) * dx                                     # cells -4..4, evaluate at cell 0
    for deg, exact_expected in [(5, True), (7, True), (8, False)]:
        fv = xs ** deg
        lin = np.array([-3, 25, -101, 319, 214, -38, 4]) / 420.0
        # use the oracle's candidates (not the literal formula) through weno7_parts
        Wm = D_IDEAL @ oracle.weno7_parts(fv[0:7])[0]                # face -1/2
        Wp = D_IDEAL @ oracle.weno7_parts(fv[1:8])[0]                # face +1/2
        assert abs(Wm - lin @ fv[0:7]) < 1e-15
        der = (Wp - Wm) / dx
        exact = 0.0                                                  # d/dx x^deg at x = 0 (deg >= 2)
        if exact_expected:
            assert abs(der - exact) < 1e-14
        else:
            assert abs(der - exact) > 1e-9


# ------------------------------------------------------------------ O6: Lax-Friedrichs split interface flux
def test_interface_flux_consistency_and_upwinding(oracle):
    rng = np.random.default_rng(2)
    for d in range(3):
        e = 400.0                       # O(100) jumps in every field: beta >> eps, weights fully one-sided
        v = rng.uniform(0.1, 0.4, size=3)
        E, M = _cons(e, v)
        U = np.array([E, *M])
        win = np.tile(U, (8, 1))
        # consistency: F_hat(U, ..., U) = F^d(U)
        Fh = oracle.interface_flux(d, win, alpha=0.9)
        assert np.max(np.abs(Fh - _flux(oracle, U, d))) < 1e-14 * E
        # a clean jump between cell i and i+1: WENO picks the one-sided smooth stencils, so the flux is the
        # textbook local Lax-Friedrichs (Rusanov) flux 1/2 (F_L + F_R) - alpha/2 (U_R - U_L)
        E2, M2 = _cons(100.0, -v)
        UR = np.array([E2, *M2])
        win = np.vstack([np.tile(U, (4, 1)), np.tile(UR, (4, 1))])
        a = 0.8
        Fh = oracle.interface_flux(d, win, alpha=a)
        llf = 0.5 * (_flux(oracle, U, d) + _flux(oracle, UR, d)) - 0.5 * a * (UR - U)
        assert np.max(np.abs(Fh - llf)) < 1e-6 * E
    # fifth field: F = N_B v_d
    U5 = np.array([E, *M, 2.5])
    Fh = oracle.interface_flux(0, np.tile(U5, (8, 1)), alpha=0.7)
    assert abs(Fh[4] - 2.5 * v[0]) < 1e-14


# ------------------------------------------------------------------ P8: source law (eq. 3) and jet cell (R7)
def test_p8_source_law_values(oracle):
    g = read_golden("source_law.txt")
    c = oracle.constants()
    assert c["hbarc"] == 0.1973269804 and abs(c["g"] - 47.5 * math.pi ** 2 / 30) < 1e-14 and c["cs2"] == 1 / 3
    for tag, e in [("e30", 30.0), ("e10", 10.0), ("e7p5", 7.5)]:
        B = oracle.source_q(e, 0.0)
        A = oracle.source_q(e, 1.0) - B
        assert abs(B - g["B_" + tag]) < 2e-9 and abs(A - g["A_" + tag]) < 2e-9
        # linear in the path length (eq. 3: kappa_rad T^3 x + kappa_coll T^2)
        assert abs(oracle.source_q(e, 0.37) - (B + 0.37 * A)) < 1e-13
    # T itself: q(l=0) = hbarc * kappa_coll * T^2
    T = math.sqrt(oracle.source_q(30.0, 0.0) / (c["hbarc"] * 2.5))
    assert abs(T - g["T_e30"]) < 1e-8
    # coefficients enter linearly; C_R/C_F multiplies both terms
    assert abs(oracle.source_q(10.0, 0.5, 8.0, 5.0, 1.0) - 2 * oracle.source_q(10.0, 0.5)) < 1e-13
    assert abs(oracle.source_q(10.0, 0.5, 4.0, 2.5, 2.25) - 2.25 * oracle.source_q(10.0, 0.5)) < 1e-13
    assert abs(oracle.source_q(10.0, 0.5, 4.0, 0.0, 1.0) - 0.5 * g["A_e10"]) < 1e-9


def test_r7_jet_cell_index(oracle):
    n, dx = 32, 0.1                                   # x_min = -1.6, cell i covers [-1.6 + 0.1 i, -1.6 + 0.1 (i+1))
    assert oracle.jet_axis_index(-1.55, n, dx) == 0
    assert oracle.jet_axis_index(1.55, n, dx) == 31
    assert oracle.jet_axis_index(0.0, n, dx) == 16    # exactly on a face -> upper cell (the 2^-20 bias)
    assert oracle.jet_axis_index(-1.0, n, dx) == 6    # config 0 start: face between 5 and 6 -> 6
    assert oracle.jet_axis_index(0.05, n, dx) == 16
    assert oracle.jet_axis_index(-0.05, n, dx) == 15
    assert oracle.jet_axis_index(1.61, n, dx) == -1 and oracle.jet_axis_index(-1.61, n, dx) == -1
    # the size of the bias: a position 0.8 x 2^-20 cells below a face counts as the upper cell, 1.2 x 2^-20 cells below
    # it as the lower one (rounding of (x - x_min)/dx is ~1e-15 cells, far below 0.2 x 2^-20)
    for face, i in ((-0.3, 13), (0.7, 23), (0.0, 16)):
        assert oracle.jet_axis_index(face - 0.8 * 2.0 ** -20 * dx, n, dx) == i
        assert oracle.jet_axis_index(face - 1.2 * 2.0 ** -20 * dx, n, dx) == i - 1
    # every stage position of the BASELINE jets is at least 0.05 cells away from a rounding-sensitive tie
    for x0, nn in [(-1.0, 32), (-3.0, 128), (-5.0, 256)]:
        for step in range(0, 60):
            for c in (0.0, 1.0, 0.5):
                a = (x0 + (step + c) * 0.02 + 0.5 * nn * dx) / dx + 2.0 ** -20
                frac = a - math.floor(a)
                assert 5e-7 < frac < 1 - 0.05

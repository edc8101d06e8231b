"""Pins of the oracle's WENO5 variant ("... also implemented ... 5th order WENO").

Nothing here retypes the oracle's formulas: candidates are checked against exact face values of polynomials given by
their cell averages, smoothness indicators against the integral definition evaluated from scratch, the nonlinear
scheme against convergence orders and limits, and the grid path against the same invariants as WENO7 (P2, P5, P6).
"""
import math

import numpy as np
import numpy.polynomial.polynomial as Pl

from paper_1511_02137_b200 import synthetic as S

D5 = np.array([0.1, 0.6, 0.3])


def _cell_averages(coef, i0, n):
    A = Pl.polyint(coef)
    return np.array([Pl.polyval(i + 0.5, A) - Pl.polyval(i - 0.5, A) for i in range(i0, i0 + n)])


def test_candidates_reproduce_quadratics_and_ideal_weights_degree4(oracle):
    rng = np.random.default_rng(3)
    for deg in range(0, 5):
        coef = rng.normal(size=deg + 1)
        v = _cell_averages(coef, -2, 5)
        exact = Pl.polyval(0.5, coef)
        q, beta, om = oracle.weno5_parts(v)
        scale = np.max(np.abs(v)) + 1
        if deg <= 2:
            assert np.max(np.abs(q - exact)) < 1e-13 * scale
        assert abs(D5 @ q - exact) < 2e-13 * scale
    v = _cell_averages(np.eye(6)[5], -2, 5)              # degree 5 is not reproduced: exactly 5th order
    assert abs(D5 @ oracle.weno5_parts(v)[0] - 0.5 ** 5) > 1e-3


def _beta_from_definition(v3, cell_pos):
    """sum_{l=1,2} int_cell dx^{2l-1} (d^l p/dx^l)^2 for the quadratic with the 3 given unit-cell averages at 0,1,2."""
    A = np.zeros((3, 3))
    for r in range(3):
        for c in range(3):
            A[r, c] = ((r + 0.5) ** (c + 1) - (r - 0.5) ** (c + 1)) / (c + 1)
    coef = np.linalg.solve(A, v3)
    tot = 0.0
    for l in (1, 2):
        dl = Pl.polyder(coef, l)
        sq = Pl.polyint(Pl.polymul(dl, dl))
        tot += Pl.polyval(cell_pos + 0.5, sq) - Pl.polyval(cell_pos - 0.5, sq)
    return tot


def test_smoothness_indicators_match_integral_definition(oracle):
    rng = np.random.default_rng(8)
    for _ in range(50):
        v = rng.normal(size=5)
        q, beta, om = oracle.weno5_parts(v)
        for k in range(3):
            ref = _beta_from_definition(v[k:k + 3], 2 - k)
            assert abs(beta[k] - ref) < 1e-11 * (1 + ref)
        assert abs(om.sum() - 1) < 1e-14 and np.all(beta >= 0)
    q, beta, om = oracle.weno5_parts(np.full(5, -1.75))
    assert np.all(beta == 0) and np.max(np.abs(om - D5)) < 1e-15
    assert abs(oracle.weno5(np.full(5, -1.75)) + 1.75) < 2e-15


def test_reconstructed_value_from_the_definition(oracle):
    """The VALUE of the solver's r = 3 reconstruction (oracle.weno5, the routine the interface flux calls; weno5_parts is a
    diagnostic copy) is sum_k omega_k q_k rebuilt here from the definition: q_k = the sub-stencil quadratic (given by its
    cell averages) at the face, beta_k = the integral definition, omega_k ~ d_k / (eps + beta_k)^2."""
    rng = np.random.default_rng(29)
    for scale in (1e-3, 1.0, 50.0):
        for eps in (1e-6, 1e-2):
            v = scale * rng.normal(size=5)
            q, beta = np.zeros(3), np.zeros(3)
            for k in range(3):
                A = np.zeros((3, 3))
                for r in range(3):
                    for c in range(3):
                        A[r, c] = ((r + 0.5) ** (c + 1) - (r - 0.5) ** (c + 1)) / (c + 1)
                coef = np.linalg.solve(A, v[k:k + 3])
                q[k] = Pl.polyval(2 - k + 0.5, coef)
                beta[k] = _beta_from_definition(v[k:k + 3], 2 - k)
            al = D5 / (eps + beta) ** 2
            expect = float(al @ q / al.sum())
            got = oracle.weno5(v, eps)
            assert abs(got - expect) < 1e-11 * (np.max(np.abs(v)) + abs(expect)), (scale, eps, got, expect)


def test_weight_limits_and_mirror(oracle):
    v = np.array([1.0, 1, 1, 5, 5])                      # step between i and i+1: sub-stencil 0 is the smooth one
    q, beta, om = oracle.weno5_parts(v)
    assert om[0] > 1 - 1e-6 and abs(oracle.weno5(v) - 1.0) < 1e-5
    v = np.array([1.0, 1, 5, 5, 5])                      # step between i-1 and i: sub-stencil 2
    q, beta, om = oracle.weno5_parts(v)
    assert om[2] > 1 - 1e-6 and abs(oracle.weno5(v) - 5.0) < 1e-5
    # linear data: exact for any weights
    assert abs(oracle.weno5(np.array([0.0, 1, 2, 3, 4])) - 2.5) < 1e-14


def _fd_error(oracle, f, dfdx, n, eps):
    dx = 1.0 / n
    xs = (np.arange(-3, n + 3) + 0.5) * dx
    fv = f(xs)
    W = np.array([oracle.weno5(fv[m:m + 5], eps) for m in range(0, n + 1)])      # faces m+2+1/2
    der = (W[1:] - W[:-1]) / dx                                                # cells 3 .. n+2
    return np.max(np.abs(der - dfdx(xs[3:n + 3])))


def test_fifth_order_convergence(oracle):
    f = lambda x: 1e-3 * np.sin(2 * np.pi * x)
    df = lambda x: 1e-3 * 2 * np.pi * np.cos(2 * np.pi * x)
    e1, e2 = (_fd_error(oracle, f, df, n, 1e-6) for n in (16, 32))
    assert 4.8 < math.log2(e1 / e2) < 6.5
    f = lambda x: np.exp(2 * x)
    df = lambda x: 2 * np.exp(2 * x)
    e1, e2 = (_fd_error(oracle, f, df, n, 1e-6) for n in (20, 40))
    assert 4.5 < math.log2(e1 / e2) < 6.5


def test_interface_flux_consistency_and_window(oracle):
    """Uniform window: F_hat = F(U) exactly up to rounding; the r = 3 flux must ignore the outermost cells
    (i-3 and i+4) of the 8-cell window."""
    from oracle import oracle as O
    import ctypes as C
    L = O.lib()
    U = S.prim_to_cons(np.array([3.0]), np.array([0.4]), np.array([-0.2]), np.array([0.1]))[:, 0]
    win = np.tile(U, (8, 1))
    rng = np.random.default_rng(2)
    win2 = win * (1 + 0.05 * rng.normal(size=win.shape))
    out_a, out_b = np.zeros(4), np.zeros(4)
    for d in range(3):
        L.oracle_interface_flux_order(d, 4, O._dp(np.ascontiguousarray(win)), 0.9, 1e-6, 1e-12, 1e-10, 5, O._dp(out_a))
        p = O.con2prim(*U)
        F = np.array([U[1 + d], U[1] * p["v"][d], U[2] * p["v"][d], U[3] * p["v"][d]])
        F[1 + d] += p["p"]
        assert np.max(np.abs(out_a - F)) < 1e-14 * np.max(np.abs(U))
        w3 = win2.copy()
        L.oracle_interface_flux_order(d, 4, O._dp(np.ascontiguousarray(w3)), 0.9, 1e-6, 1e-12, 1e-10, 5, O._dp(out_a))
        w3[0] *= 3.0
        w3[7] *= 0.1
        L.oracle_interface_flux_order(d, 4, O._dp(np.ascontiguousarray(w3)), 0.9, 1e-6, 1e-12, 1e-10, 5, O._dp(out_b))
        assert np.array_equal(out_a, out_b)
        L.oracle_interface_flux_order(d, 4, O._dp(np.ascontiguousarray(w3)), 0.9, 1e-6, 1e-12, 1e-10, 7, O._dp(out_b))
        assert not np.array_equal(out_a, out_b)


def test_grid_invariants_weno5(oracle):
    # P2: uniform state stays uniform bitwise
    n = (12, 9, 7)
    ones = np.ones((n[2], n[1], n[0]))
    U0 = S.prim_to_cons(2.5 * ones, 0.3 * ones, -0.1 * ones, 0.2 * ones)
    o = oracle.Oracle(*n, 0.1, 0.02, weno_order=5)
    o.set_state(U0)
    assert np.all(o.eval_rhs(0.0) == 0.0)
    o.step(2)
    U = o.get_fields()
    assert np.array_equal(U, np.broadcast_to(U[:, :1, :1, :1], U.shape)) and np.allclose(U, U0, rtol=1e-15)
    o.close()
    # P6 mirror symmetry + P5 conservation while nothing reaches the boundary
    n = (24, 20, 16)
    U0 = S.gaussian_flow(n, 0.1, peak=10.0, sigma=(0.3, 0.25, 0.2), R=(1.0, 0.8, 1.2), ucoef=0.05, noise=0.0,
                         background=1.0)
    o = oracle.Oracle(*n, 0.1, 0.02, weno_order=5)
    o.set_state(U0)
    o.step(3)
    U = o.get_fields()
    o.close()
    scale = np.abs(U).max(axis=(1, 2, 3))
    for axis, odd in ((3, 1), (2, 2), (1, 3)):
        F = np.flip(U, axis=axis)
        for f in range(4):
            sign = -1.0 if f == odd else 1.0
            assert np.max(np.abs(U[f] - sign * F[f])) <= 1e-13 * scale[f]
    # WENO5 and WENO7 runs differ (different schemes) but only at truncation level
    o7 = oracle.Oracle(*n, 0.1, 0.02)
    o7.set_state(U0)
    o7.step(3)
    d = np.max(np.abs(o7.get_fields()[0] - U[0])) / scale[0]
    o7.close()
    assert 1e-9 < d < 5e-2


def test_shock_tube_weno5_against_exact(oracle):
    """Config 1 at nx = 256 with WENO5: first-order L1 convergence to the exact p = e/3 Riemann solution (pin P4)."""
    from test_oracle_riemann import exact_solution, exact_profile
    sol = exact_solution()
    errs = []
    for nx in (128, 256):
        dx = 5.12 / nx
        c = dict(S.CONFIGS[1], n=(nx, 1, 1), dx=dx)
        U0 = S.make_state(c)
        steps = int(round(1.5 / (0.4 * dx)))
        o = oracle.Oracle(nx, 1, 1, dx, 1.5 / steps, weno_order=5)
        o.set_state(U0)
        o.step(steps)
        P = o.get_fields(1)
        o.close()
        ee, ve = exact_profile(S.cell_centres(nx, dx), 1.5, sol)
        errs.append(np.sum(np.abs(P[0, 0, 0] - ee)) * dx)
    assert errs[1] < 0.2 and 1.5 < errs[0] / errs[1] < 2.6

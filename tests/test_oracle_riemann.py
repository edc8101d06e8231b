"""Pin P4: the oracle's whole 1-D path (con2prim, LF-split WENO7, divergence, RK3, outflow ghosts) against the
exact Riemann solution for p = e/3 (BASELINE.json config 1), and P5 on the same run (conservation).

The exact solution is re-derived here from eq. (1) with nested root finders on the
Rankine-Hugoniot conditions written directly in T^{mu nu}; tests/golden/riemann_p_e3.txt holds the numbers
derived in SURVEY.md 8(c) P4 and must agree.
"""
import math

import numpy as np
from scipy.optimize import brentq

from conftest import read_golden

CS = 1 / math.sqrt(3)
EL, ER = 10.0, 1.0


def _EM(e, v):
    g2 = 1 / (1 - v * v)
    return (4 / 3) * e * g2 - e / 3, (4 / 3) * e * g2 * v


def _shock_branch(es):
    """post-shock velocity and shock speed for post-shock energy density es, upstream (ER, v=0)."""
    def rh(v):                               # V = [M]/[E] inserted into V [M] = [M v + p]
        E, M = _EM(es, v)
        return M * M / (E - ER) - M * v - es / 3 + ER / 3
    v = brentq(rh, 1e-12, 1 - 1e-12, xtol=1e-16, rtol=1e-15)
    E, M = _EM(es, v)
    return v, M / (E - ER)


def _raref_velocity(e):
    """left-going rarefaction from (EL, 0): artanh v + (sqrt(3)/4) ln e = (sqrt(3)/4) ln EL."""
    return math.tanh((math.sqrt(3) / 4) * math.log(EL / e))


def exact_solution():
    es = brentq(lambda e: _shock_branch(e)[0] - _raref_velocity(e), ER * (1 + 1e-9), EL * (1 - 1e-9),
                xtol=1e-15, rtol=1e-15)
    vs, V = _shock_branch(es)
    return dict(e_star=es, v_star=vs, v_shock=V, xi_head=-CS, xi_tail=(vs - CS) / (1 - vs * CS))


def exact_profile(x, t, sol):
    xi = x / t
    e = np.empty_like(x)
    v = np.empty_like(x)
    head, tail, V = sol["xi_head"], sol["xi_tail"], sol["v_shock"]
    left = xi <= head
    fan = (xi > head) & (xi < tail)
    star = (xi >= tail) & (xi < V)
    right = xi >= V
    e[left], v[left] = EL, 0.0
    vf = (xi[fan] + CS) / (1 + xi[fan] * CS)
    v[fan] = vf
    e[fan] = EL * ((1 - vf) / (1 + vf)) ** (2 / math.sqrt(3))
    e[star], v[star] = sol["e_star"], sol["v_star"]
    e[right], v[right] = ER, 0.0
    return e, v


def test_exact_solution_matches_golden_and_rankine_hugoniot():
    g = read_golden("riemann_p_e3.txt")
    s = exact_solution()
    for k in ("e_star", "v_star", "v_shock", "xi_head", "xi_tail"):
        assert abs(s[k] - g[k]) < 2e-9, k
    # Rankine-Hugoniot in T^{mu nu}: V [U] = [F] for U = (E, Mx), F = (Mx, Mx v + p)
    E, M = _EM(s["e_star"], s["v_star"])
    V = s["v_shock"]
    assert abs(V * (E - ER) - M) < 1e-13
    assert abs(V * M - (M * s["v_star"] + s["e_star"] / 3 - ER / 3)) < 1e-13
    # SURVEY's closed forms for the same branch
    es = s["e_star"]
    assert abs(s["v_star"] ** 2 - 3 * (es - ER) ** 2 / ((3 * ER + es) * (3 * es + ER))) < 1e-13
    assert abs(V ** 2 - (3 * es + ER) / (3 * (3 * ER + es))) < 1e-13
    # inside the fan the characteristic speed (v - cs)/(1 - v cs) equals xi
    for xi in (-0.5, -0.3, -0.2):
        v = (xi + CS) / (1 + xi * CS)
        assert abs((v - CS) / (1 - v * CS) - xi) < 1e-15


def _run_tube(oracle, S, nx, steps, dt_over_dx=0.4, length=5.12):
    dx = length / nx
    dt = dt_over_dx * dx
    U0 = S.shock_tube((nx, 1, 1), EL, ER)
    o = oracle.Oracle(nx, 1, 1, dx, dt)
    o.set_state(U0)
    o.step(steps)
    U = o.get_fields(0)
    P = o.get_fields(1)
    d = o.diag()
    o.close()
    x = S.cell_centres(nx, dx)
    return x, dx, dt * steps, U0, U, P, d


def test_p4_config1_against_exact_solution(oracle):
    from paper_1511_02137_b200 import synthetic as S
    sol = exact_solution()
    errs = {}
    for nx, steps in ((256, 150), (512, 300)):          # t = 1.2 on both grids
        x, dx, t, U0, U, P, d = _run_tube(oracle, S, nx, steps)
        ee, ve = exact_profile(x, t, sol)
        errs[nx] = (np.sum(np.abs(P[0, 0, 0] - ee)) * dx, np.sum(np.abs(P[1, 0, 0] - ve)) * dx)
        assert d["ncap"] == 0 and d["has_nan"] == 0
    # first-order convergence in L1 (there is a shock): ratio ~ 2 per refinement
    assert 1.6 < errs[256][0] / errs[512][0] < 2.6
    assert 1.5 < errs[256][1] / errs[512][1] < 2.8
    # the BASELINE run itself: 375 steps of dt = 0.004 to t = 1.5 (R11)
    x, dx, t, U0, U, P, d = _run_tube(oracle, S, 512, 375)
    assert abs(t - 1.5) < 1e-12
    ee, ve = exact_profile(x, t, sol)
    l1e = np.sum(np.abs(P[0, 0, 0] - ee)) * dx
    l1v = np.sum(np.abs(P[1, 0, 0] - ve)) * dx
    assert l1e < 0.08 and l1v < 0.01                      # SURVEY probe: 0.059 / 0.0067
    # plateau and wave positions
    e = P[0, 0, 0]
    plateau = (x > 0.0) & (x < 0.9)
    assert np.max(np.abs(e[plateau] - sol["e_star"])) < 0.05
    assert np.max(np.abs(P[1, 0, 0][plateau] - sol["v_star"])) < 0.02
    shock_pos = x[np.argmin(np.diff(e)) + 1]
    assert abs(shock_pos - sol["v_shock"] * 1.5) < 0.03
    assert e.max() < EL + 1e-3 and e.min() > ER - 1e-3     # overshoot (SURVEY probe: 6e-5)
    assert d["ncap"] == 0
    # P5 on this run: boundary cells are still at rest, so sum(E) dx is constant and sum(Mx) dx = (pL - pR) t
    assert abs(np.sum(U[0]) - np.sum(U0[0])) * dx < 1e-11
    assert abs(np.sum(U[1]) * dx - (EL - ER) / 3 * 1.5) < 1e-11
    assert np.all(U[2] == 0) and np.all(U[3] == 0)
    # alpha of the last stage: the largest wavespeed is in the post-shock/fan region and below 1
    assert 0.7 < d["alpha"][0] < 1.0 and abs(d["alpha"][1] - CS) < 1e-3


def test_rk3_temporal_order(oracle):
    """Reading R5: the time integrator is 3rd order (self-convergence in dt on smooth 1-D data)."""
    from paper_1511_02137_b200 import synthetic as S
    nx, dx = 64, 0.1
    x = S.cell_centres(nx, dx)
    e = 1.0 + 0.5 * np.exp(-x * x / (2 * 0.8 ** 2))
    U0 = S.prim_to_cons(e[None, None, :], *(np.zeros((1, 1, nx)),) * 3)
    res = {}
    for nsteps in (128, 8, 16, 32):
        dt = 0.8 / nsteps
        o = oracle.Oracle(nx, 1, 1, dx, dt)
        o.set_state(U0)
        o.step(nsteps)
        res[nsteps] = o.get_fields(0)[0, 0, 0].copy()
        o.close()
    err = {n: np.max(np.abs(res[n] - res[128])) for n in (8, 16, 32)}
    assert 2.7 < math.log2(err[8] / err[16]) < 3.4
    assert 2.7 < math.log2(err[16] / err[32]) < 3.5

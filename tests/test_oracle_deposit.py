"""Pins of the smeared (Gaussian) jet deposit, reading R15 (eq. (2) PAPER.md:21-23 sums over jets and
has a true delta function, of which the Gaussian is a regularisation).  The deposit is read off as the difference of
two RHS evaluations (with and without jets), so nothing here re-types the oracle's weights."""
import numpy as np

from paper_1511_02137_b200 import synthetic as S


def _deposit(oracle, n, sigma, jets, stage_c=0.5, dx=0.1):
    c = S.scaled_config(0, n)
    U0 = S.make_state(c, noise=False)
    o = oracle.Oracle(*n, dx, 0.02)
    o.set_state(U0)
    L0 = o.eval_rhs(stage_c)
    for pos, d in jets:
        o.add_jet(pos, d)
    o.set_deposit_width(sigma)
    L1 = o.eval_rhs(stage_c)
    o.step(1)
    q = o.last_stage_q()
    o.close()
    return L1 - L0, q, U0


def test_total_deposit_equals_q_and_direction(oracle):
    n, dx = (24, 24, 24), 0.1
    dirv = np.array([1.0, 0.5, -0.25])
    dirv /= np.linalg.norm(dirv)
    dL, q, _ = _deposit(oracle, n, 0.12, [((0.03, -0.02, 0.01), tuple(dirv))], stage_c=0.0)
    tot = dL.reshape(4, -1).sum(axis=1) * dx ** 3
    assert tot[0] > 0 and abs(tot[0] - q[0, 0]) < 1e-12 * q[0, 0]            # q^0 of that step = stage_c 0
    assert np.max(np.abs(tot[1:] - tot[0] * dirv)) < 1e-12 * tot[0]
    assert np.all(dL[0] >= 0)


def test_shape_is_the_gaussian_around_the_jet_position(oracle):
    n, dx, sigma = (28, 28, 28), 0.1, 0.1
    pos = (0.03, -0.02, 0.01)
    dL, q, _ = _deposit(oracle, n, sigma, [(pos, (1.0, 0.0, 0.0))], stage_c=0.0)
    w = dL[0] / dL[0].sum()
    x = S.cell_centres(n[0], dx)
    # first moments reproduce the jet position (symmetric truncation at >= 3 sigma: error << dx)
    mx = (w * x[None, None, :]).sum(); my = (w * x[None, :, None]).sum(); mz = (w * x[:, None, None]).sum()
    assert abs(mx - pos[0]) < 2e-3 and abs(my - pos[1]) < 2e-3 and abs(mz - pos[2]) < 2e-3
    # second moment ~ sigma^2 (truncated at 3 sigma and sampled: within 10 %)
    vx = (w * (x[None, None, :] - mx) ** 2).sum()
    assert 0.85 * sigma ** 2 < vx < 1.05 * sigma ** 2
    # support: the cube of radius ceil(3 sigma / dx) = 3 cells around the R7 cell
    nzc = np.argwhere(dL[0] > 0)
    assert (nzc.max(axis=0) - nzc.min(axis=0) == 6).all() and len(nzc) == 7 ** 3
    # ratio of two cells = the Gaussian ratio (the normalisation cancels)
    k0, j0, i0 = nzc.min(axis=0) + 3
    r2 = lambda i, j, k: (x[i] - pos[0]) ** 2 + (x[j] - pos[1]) ** 2 + (x[k] - pos[2]) ** 2
    ratio = dL[0][k0, j0, i0 + 2] / dL[0][k0, j0, i0]
    assert abs(ratio - np.exp(-(r2(i0 + 2, j0, k0) - r2(i0, j0, k0)) / (2 * sigma ** 2))) < 1e-12


def test_limits_point_deposit_and_boundary_loss(oracle):
    n, dx = (16, 16, 16), 0.1
    jets = [((0.03, -0.02, 0.01), (1.0, 0.0, 0.0))]
    dLp, qp, _ = _deposit(oracle, n, 0.0, jets, stage_c=0.0)
    dLs, qs, _ = _deposit(oracle, n, 1e-3, jets, stage_c=0.0)             # sigma << dx: all weight in the nearest cell
    assert np.count_nonzero(dLp[0]) == 1
    assert np.max(np.abs(dLs - dLp)) < 1e-12 * np.max(np.abs(dLp))
    # a jet in the corner cell: part of the cube is outside the grid and that share is lost
    edge = (n[0] / 2 - 0.5) * dx
    dLe, qe, _ = _deposit(oracle, n, 0.1, [((edge, edge, edge), (1.0, 0.0, 0.0))], stage_c=0.0)
    tot = dLe[0].sum() * dx ** 3
    # jet at the centre of the corner cell, sigma = dx: per axis the offsets -3..0 of -3..3 stay inside the grid
    w = np.exp(-0.5 * np.arange(-3, 4) ** 2)
    frac = (w[:4].sum() / w.sum()) ** 3
    assert abs(tot / qe[0, 0] - frac) < 1e-12


def test_conservation_budget_with_two_smeared_jets(oracle):
    """Pin P5 with R15: the change of total energy/momentum over a step equals dt sum_s w_s q^s (n_hat)."""
    n, dx, dt = (24, 24, 24), 0.1, 0.02
    ones = np.ones((n[2], n[1], n[0]))
    U0 = S.prim_to_cons(5.0 * ones, 0 * ones, 0 * ones, 0 * ones)       # uniform and at rest: no boundary flux at all
    o = oracle.Oracle(*n, dx, dt)
    o.set_state(U0)
    o.add_jet((0.0, 0.0, 0.0), (1.0, 0.0, 0.0))
    o.add_jet((0.05, 0.1, 0.0), (-1.0, 0.0, 0.0))
    o.set_deposit_width(0.08)
    ref = oracle.Oracle(*n, dx, dt)
    ref.set_state(U0)
    for _ in range(3):
        o.step(1), ref.step(1)
    dU = (o.get_fields() - ref.get_fields()).reshape(4, -1).sum(axis=1) * dx ** 3
    dep = o.diag()["deposited"]
    assert dep[0] > 0 and abs(dU[0] - dep[0]) < 1e-9 * dep[0]
    assert abs(dU[1] - dep[1]) < 1e-9 * dep[0] and abs(dep[1]) < 0.2 * dep[0]   # back-to-back: momenta nearly cancel
    o.close(), ref.close()


def _r7_cell(x, n, dx):
    """R7: index per axis = floor((x - x_min)/dx + 2^-20), x_min = -n dx / 2; None outside the grid"""
    idx = []
    for a in range(3):
        i = int(np.floor((x[a] + 0.5 * n[a] * dx) / dx + 2.0 ** -20))
        if i < 0 or i > n[a] - 1:
            return None
        idx.append(i)
    return tuple(idx)


def test_jet_moves_along_its_direction_at_c_and_leaves_the_grid(oracle):
    """Eq. (2): the source sits at x_i(t) = x_0 + n_hat (t - t_added) (a parton at c, R8).  The deposit
    cell -- the only cell where the RHS with the jet differs from the RHS without -- follows that line through several cells
    (both the sign and the speed of the motion), the Gaussian deposit's centre of mass does likewise, and once the jet is
    outside the grid nothing is deposited and its q is 0 (R7)."""
    n, dx, dt = (24, 20, 16), 0.1, 0.02
    x0 = np.array([-0.93, 0.41, -0.22])
    d = np.array([0.8, -0.5, 0.33])
    d /= np.linalg.norm(d)
    c = S.scaled_config(0, n)
    U0 = S.make_state(c, noise=False)
    xs = [S.cell_centres(n[a], dx) for a in range(3)]
    seen = set()
    for stage_c in (0.0, 9.5, 23.25, 41.0, 68.5):
        ell = stage_c * dt
        pos = x0 + d * ell
        cell = _r7_cell(pos, n, dx)
        assert cell is not None
        for sigma in (0.0, 0.06):
            o = oracle.Oracle(*n, dx, dt)
            o.set_state(U0)
            L0 = o.eval_rhs(stage_c)
            o.add_jet(tuple(x0), tuple(d))
            o.set_deposit_width(sigma)
            dL = o.eval_rhs(stage_c) - L0
            o.close()
            if sigma == 0.0:
                nz = np.argwhere(dL[0] != 0)
                assert len(nz) == 1 and tuple(nz[0][::-1]) == cell, (stage_c, nz, cell)       # arrays are (k, j, i)
            else:
                w = dL[0] / dL[0].sum()
                com = np.array([(w * xs[0][None, None, :]).sum(), (w * xs[1][None, :, None]).sum(), (w * xs[2][:, None, None]).sum()])
                assert np.max(np.abs(com - pos)) < 0.02 * dx + 2e-3, (stage_c, com, pos)
        seen.add(cell)
    assert len(seen) == 5                                     # five different cells along the track
    # a jet sitting in the FIRST cell of an axis (index 0) deposits like any other
    for axis in range(3):
        pos = np.array([0.03, -0.02, 0.01])
        pos[axis] = -0.5 * n[axis] * dx + 0.4 * dx
        o = oracle.Oracle(*n, dx, dt)
        o.set_state(U0)
        L0 = o.eval_rhs(0.0)
        o.add_jet(tuple(pos), (0.0, 0.0, 1.0) if axis != 2 else (1.0, 0.0, 0.0))
        dL = o.eval_rhs(0.0) - L0
        o.close()
        nz = np.argwhere(dL[0] != 0)
        assert len(nz) == 1 and tuple(nz[0][::-1]) == _r7_cell(pos, n, dx) and nz[0][::-1][axis] == 0
    # outside: nothing is deposited, q = 0, the deposited totals do not move
    o = oracle.Oracle(*n, dx, dt)
    o.set_state(U0)
    L0 = o.eval_rhs(0.0)
    o.add_jet((1.15, 0.0, 0.0), (1.0, 0.0, 0.0))             # x_max = 1.2: outside after 3 steps
    for s in range(6):
        o.step(1)
    assert np.all(o.last_stage_q() == 0.0)
    dep6 = o.diag()["deposited"].copy()
    o.step(2)
    assert np.array_equal(o.diag()["deposited"], dep6) and dep6[0] > 0
    o.close()


def test_path_length_counts_from_the_step_the_jet_was_added(oracle):
    """Eq. (3) with x = the path length l = t - t_added (R8): a jet added after three steps starts with
    l = 0.  With kappa_coll = 0 the rate is purely radiative, q = hbarc kappa_rad T^3 l, so its first stage value (l = 0)
    is exactly 0 and the second one (l = dt) is positive; its first deposit goes into the cell of its START position."""
    n, dx, dt = (16, 16, 16), 0.1, 0.02
    c = S.scaled_config(0, n)
    U0 = S.make_state(c, noise=False)
    o = oracle.Oracle(*n, dx, dt)
    o.set_state(U0)
    o.step(3)
    x0 = (-0.33, 0.12, 0.07)
    L0 = o.eval_rhs(0.5)
    o.add_jet(x0, (1.0, 0.0, 0.0), kappa_rad=4.0, kappa_coll=0.0)
    dL = o.eval_rhs(0.5) - L0                                  # l = dt/2: still in the start cell (dt/2 = 0.1 dx)
    nz = np.argwhere(dL[0] != 0)
    assert len(nz) == 1 and tuple(nz[0][::-1]) == _r7_cell(np.array(x0), n, dx)
    o.step(1)
    q = o.last_stage_q()[:, 0]
    assert q[0] == 0.0 and q[1] > 0.0 and abs(q[2] - 0.5 * q[1]) < 0.05 * q[1]     # l = 0, dt, dt/2 (T moves a little)
    o.close()


def test_deposit_radius_is_clamped_to_1_and_8_cells(oracle):
    """R15: R = ceil(3 sigma / dx) clamped to [1, 8]: a very narrow Gaussian still covers the 3^3 cells around the R7 cell,
    a very wide one is cut at 17^3."""
    n, dx = (24, 24, 24), 0.1
    for sigma, side in ((0.004, 3), (0.03, 3), (0.034, 5), (0.3, 17), (0.5, 17)):
        dL, q, _ = _deposit(oracle, n, sigma, [((0.03, -0.02, 0.01), (1.0, 0.0, 0.0))], stage_c=0.0)
        nzc = np.argwhere(dL[0] != 0)
        span = nzc.max(axis=0) - nzc.min(axis=0) + 1
        # exp() of far cells may underflow to 0 for the narrowest width: the support is then smaller, never larger
        assert (span <= side).all() and (sigma < 0.02 or (span == side).all()), (sigma, span, side)
        tot = dL[0].sum() * dx ** 3
        assert abs(tot - q[0, 0]) < 1e-12 * q[0, 0]

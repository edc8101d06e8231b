"""hydro_wavespeeds_noalloc (include/hydro.h): the entry point that allocates nothing, against the existing handle path.

Collected last on purpose (the suite runs with pytest -x: a failure here must not hide another test).  Steps a-1 + a-2
(con2prim + exact wavespeed maxima, eq. 1 with p = e/3) run in the same kernel on both sides, so the
maxima agree bitwise; the bound asserted is the 1e-13 the parity tests use for alpha.
"""
import numpy as np
import pytest

from paper_1511_02137_b200 import synthetic as S

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1511_02137_b200 import hydro
    hydro.load()
    return hydro


def _existing_path(H, n, nf, U0):
    """alpha, cap events and NaN flag of U0 through a handle: hydro_stage_prims + hydro_stage_alpha (stage 1's input state is
    U0), then the stage itself, which commits the cap count of that state."""
    g = H.Hydro(*n, 0.1, 0.02, nfields=nf)
    g.set_state(U0)
    g.stage_prims(0)
    alpha = np.array(g.stage_alpha(0))
    g.stage_sweeps(0)
    d = g.diag()
    g.close()
    return alpha, d["ncap"], d["has_nan"]


def _capped_state(n, nf, seed):
    """config 0's flow on grid n plus a few cells with |M| > E (the con2prim cap fires there) and E below the floor"""
    c = S.scaled_config(0, n)
    c["nf"] = nf
    U0 = S.make_state(c)
    rng = np.random.default_rng(seed)
    for _ in range(7):
        k, j, i = (int(rng.integers(0, m)) for m in (n[2], n[1], n[0]))
        U0[1, k, j, i] = 1.5 * U0[0, k, j, i]
    U0[0, 0, 0, 0] = 1e-15
    return U0


@pytest.mark.parametrize("n,nf", [((32, 32, 32), 4), ((37, 19, 23), 5), ((64, 64, 64), 4)])
def test_no_alloc_entry_point_matches_the_handle_path_twice_in_a_row(H, n, nf):
    import torch
    alpha_d = torch.full((3,), -1.0, dtype=torch.float64, device="cuda")
    counts_d = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    # two calls in a row on different states: the second must not see anything the first left in the shared scratch
    # (its maxima are LOWER than the first call's, so a missing clear of the reduction block would show)
    Ua = _capped_state(n, nf, 11)
    Ub = S.make_state(dict(S.scaled_config(0, n), nf=nf))
    Ub[1:4] *= 0.25
    for it, U0 in enumerate((Ua, Ub, Ua)):
        ref_alpha, ref_ncap, ref_nan = _existing_path(H, n, nf, U0)
        Ud = torch.from_numpy(np.ascontiguousarray(U0)).cuda()
        torch.cuda.synchronize()
        before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
        H.wavespeeds_noalloc(Ud, alpha_d, counts_d)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before
        if it > 0:                                             # (the first launch of a kernel may load its module)
            assert torch.cuda.mem_get_info()[0] == free_before, "device memory in use changed across the call"
        alpha = alpha_d.cpu().numpy()
        assert np.max(np.abs(alpha - ref_alpha)) <= 1e-13, (alpha, ref_alpha)
        assert int(counts_d[0]) == ref_ncap and int(counts_d[1]) == ref_nan == 0
        assert np.all(alpha > 0.0) and np.all(alpha < 1.0)
    assert ref_ncap >= 7                                       # the capped cells were seen (state Ua)


def test_no_alloc_nan_flag_and_optional_counts(H):
    import torch
    n = (16, 8, 8)
    U0 = S.make_state(S.scaled_config(0, n))
    U0[2, 3, 4, 5] = np.nan
    Ud = torch.from_numpy(U0).cuda()
    alpha_d = torch.zeros(3, dtype=torch.float64, device="cuda")
    counts_d = torch.zeros(2, dtype=torch.int64, device="cuda")
    H.wavespeeds_noalloc(Ud, alpha_d, counts_d)
    assert int(counts_d[1]) == 1
    U0[2, 3, 4, 5] = 0.0
    Ud = torch.from_numpy(U0).cuda()
    H.wavespeeds_noalloc(Ud, alpha_d, None)                    # counts are optional
    H.wavespeeds_noalloc(Ud, alpha_d, counts_d)
    assert int(counts_d[1]) == 0                               # the flag of the earlier call is gone


def test_no_alloc_rejects_what_does_not_fit(H):
    import torch
    alpha_d = torch.zeros(3, dtype=torch.float64, device="cuda")
    big = torch.zeros((4, 65, 64, 64), dtype=torch.float64, device="cuda")      # 64^3 + one plane > HYDRO_NOALLOC_MAX_CELLS
    with pytest.raises(H.HydroError) as e:
        H.wavespeeds_noalloc(big, alpha_d)
    assert e.value.code == H.EINVAL and "HYDRO_NOALLOC_MAX_CELLS" in str(e.value)
    with pytest.raises(H.HydroError):
        H.wavespeeds_noalloc(torch.zeros((3, 8, 8, 8), dtype=torch.float64, device="cuda"), alpha_d)   # nfields
    assert H.NOALLOC_MAX_CELLS == 64 ** 3

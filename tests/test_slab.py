"""z-slab decomposition.  CPU: the plane split, the local extents and the torch.distributed exchange
over gloo (world_size 3).  GPU (one device): all slabs in one process, exchanged by device copies, against the
one-handle run -- owned planes must come out bitwise identical."""
import os
import socket
import sys

import numpy as np
import pytest

from paper_1511_02137_b200 import slab as SL
from paper_1511_02137_b200 import synthetic as S

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_split_and_extents():
    assert SL.split_planes(10, 2) == [(0, 5), (5, 10)]
    assert SL.split_planes(14, 3) == [(0, 5), (5, 10), (10, 14)]
    with pytest.raises(ValueError):
        SL.split_planes(7, 2)
    for nz, world in ((32, 2), (33, 3), (64, 5), (16, 4)):
        covered = []
        for r in range(world):
            k_off, nloc, lo, hi = SL.local_extent(nz, world, r)
            assert k_off >= 0 and k_off + nloc <= nz and hi - lo >= SL.HALO
            assert lo == (SL.HALO if r > 0 else 0) and nloc - hi == (SL.HALO if r < world - 1 else 0)
            covered += list(range(k_off + lo, k_off + hi))
        assert covered == list(range(nz))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    send = [torch.full((6,), 10.0 * rank + side, dtype=torch.float64) for side in (0, 1)]
    recv = [torch.full((6,), -1.0, dtype=torch.float64) for _ in (0, 1)]
    SL.exchange_faces(send, recv, rank, world, dist)
    amax = SL.allreduce_max([0.1 * rank, 0.5 - 0.1 * rank, 0.3], dist)
    # the device path reduces the BIT PATTERNS as 64-bit integers: non-negative reals order like their patterns
    vals = torch.tensor([0.1 * rank, 0.5 - 0.1 * rank, 0.3], dtype=torch.float64)
    bits = vals.view(torch.int64).clone()
    dist.all_reduce(bits, op=dist.ReduceOp.MAX)
    assert bits.view(torch.float64).tolist() == amax
    f32 = torch.tensor([0.1 * rank, 0.5 - 0.1 * rank, 0.3], dtype=torch.float32).view(torch.int32).to(torch.int64)
    dist.all_reduce(f32, op=dist.ReduceOp.MAX)                  # fp32 handles keep the 32-bit pattern in the low word
    assert f32.to(torch.int32).view(torch.float32).tolist() == pytest.approx(amax, rel=1e-6)
    q.put((rank, recv[0][0].item(), recv[1][0].item(), amax))
    dist.barrier()
    dist.destroy_process_group()


def test_exchange_and_alpha_over_gloo_world3():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    world = 3
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=180) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, lo, hi, amax in res:
        assert lo == (10.0 * (rank - 1) + 1 if rank > 0 else -1.0)          # the lower neighbour's HIGH face
        assert hi == (10.0 * (rank + 1) + 0 if rank < world - 1 else -1.0)   # the upper neighbour's LOW face
        assert amax == pytest.approx([0.2, 0.5, 0.3])


# ------------------------------------------------------------------------------------------------ one GPU, all slabs
@pytest.fixture(scope="module")
def H():
    import torch
    assert torch.cuda.is_available()
    from paper_1511_02137_b200 import hydro
    hydro.load()
    return hydro


CASES = [
    dict(n=(32, 24, 40), world=2, steps=4, jets=[((-0.5, 0.0, 0.02), (1.0, 0.2, 0.3))]),
    dict(n=(36, 20, 33), world=3, steps=3, jets=[((0.0, 0.0, 0.0), (0.0, 0.0, 1.0)), ((0.3, 0.1, -0.6), (0.0, 0.0, -1.0))]),
    dict(n=(36, 20, 33), world=3, steps=3, jets=[((0.0, 0.0, 0.0), (0.0, 0.0, 1.0)), ((0.3, 0.1, -0.6), (0.0, 0.0, -1.0))],
         overlap=False),
    dict(n=(32, 24, 40), world=2, steps=3, jets=[((-0.5, 0.0, 0.02), (1.0, 0.2, 0.3))], limiter=True),
    dict(n=(32, 24, 40), world=2, steps=3, jets=[((-0.5, 0.0, 0.35), (0.0, 0.0, 1.0))], sigma=0.1),
    dict(n=(32, 24, 40), world=2, steps=3, jets=[((-0.5, 0.0, -0.25), (0.0, 0.0, 1.0))], sigma=0.13),     # R = 4 = the halo
    dict(n=(32, 24, 40), world=4, steps=3, jets=[((-0.5, 0.0, 0.02), (1.0, 0.2, 0.3))], precision=32),
    dict(n=(32, 24, 40), world=2, steps=3, jets=[((-0.5, 0.0, 0.02), (1.0, 0.2, 0.3))], weno_order=5, nf=5),
    dict(n=(64, 40, 72), world=2, steps=2, jets=[((-0.5, 0.0, -0.22), (0.2, 0.1, 1.0))], nf=5),
]


def _setup(x, case):
    """x: a Hydro handle or a Slab (same setter names)."""
    g = getattr(x, "g", x)
    for pos, d in case["jets"]:
        g.add_jet(pos, d)
    if case.get("limiter"):
        x.set_limiter(True)
    x.set_deposit_width(case.get("sigma", 0.0))


def _reference_run(H, case):
    n, steps = case["n"], case["steps"]
    c = S.scaled_config(0, n)
    c["nf"] = case.get("nf", 4)
    kw = dict(nfields=c["nf"], precision=case.get("precision", 64), weno_order=case.get("weno_order", 7))
    U0 = S.make_state(c).astype(np.float64 if kw["precision"] == 64 else np.float32)
    ref = H.Hydro(*n, c["dx"], c["dt"], **kw)
    ref.set_state(U0)
    _setup(ref, case)
    ref.step(steps)
    out = (ref.get_fields(), ref.diag(), ref.last_stage_q(), ref.limited_faces())
    ref.close()
    return c, kw, U0, out


@pytest.mark.gpu
@pytest.mark.parametrize("case", CASES)
def test_slabs_match_the_single_handle_run_bitwise(H, case):
    import torch
    n, world, steps = case["n"], case["world"], case["steps"]
    c, kw, U0, (Uref, dref, qref, nlim_ref) = _reference_run(H, case)
    st = torch.cuda.Stream()
    slabs = [SL.Slab(H, n, c["dx"], c["dt"], r, world, stream=st, **kw) for r in range(world)]
    for sl in slabs:
        sl.set_state(U0)
        _setup(sl, case)
    assert all(sl.overlap == (not case.get("limiter") and not case.get("sigma")) for sl in slabs)
    SL.run_local(slabs, steps, overlap=case.get("overlap"))
    U = np.concatenate([sl.owned() for sl in slabs], axis=1)
    assert U.shape == Uref.shape
    assert np.array_equal(U, Uref)                                              # bitwise
    ds = [sl.g.diag() for sl in slabs]
    assert all(d["step"] == steps and d["has_nan"] == 0 for d in ds)
    assert sum(d["ncap"] for d in ds) == dref["ncap"]
    assert np.allclose(sum(d["deposited"] for d in ds), dref["deposited"], rtol=1e-13, atol=0)
    assert np.allclose(sum(sl.g.last_stage_q() for sl in slabs), qref, rtol=1e-13, atol=0)
    assert np.array_equal(np.max([d["alpha"] for d in ds], axis=0), dref["alpha"])
    assert sum(sl.g.limited_faces() for sl in slabs) == nlim_ref               # counted on owned planes only
    for sl in slabs:
        sl.close()


@pytest.mark.gpu
def test_slab_run_of_config2_matches_the_oracle_sample(H):
    """The decomposed path against the ORACLE directly (not only against the one-handle run): BASELINE config 2 (128^3, jet)
    for its full 50 steps as 4 z-slabs in the overlapped schedule, compared with the stored final state of the oracle run
    (tests/golden/run_cfg2.npz, written by make_golden_runs.py from oracle/ only) at 1e-9 (north_star)."""
    import torch
    gold = np.load(os.path.join(ROOT, "tests", "golden", "run_cfg2.npz"))
    c = S.CONFIGS[2]
    steps, world = int(gold["steps"]), 4
    assert steps == c["steps"]
    U0 = S.make_state(2)
    st = torch.cuda.Stream()
    slabs = [SL.Slab(H, c["n"], c["dx"], c["dt"], r, world, stream=st) for r in range(world)]
    for sl in slabs:
        sl.set_state(U0)
        for pos, d in c["jets"]:
            sl.g.add_jet(pos, d, S.KAPPA_RAD, S.KAPPA_COLL, S.CR_OVER_CF)
    SL.run_local(slabs, steps)
    U = np.concatenate([sl.owned() for sl in slabs], axis=1)
    idx = gold["idx"]
    errs = np.max(np.abs(U[:, idx[:, 0], idx[:, 1], idx[:, 2]] - gold["U"]), axis=1) / gold["fmax"]
    assert np.all(errs < 1e-9), errs
    fsum = U.sum(axis=(1, 2, 3), dtype=np.longdouble).astype(np.float64)
    assert np.all(np.abs(fsum - gold["fsum"]) <= 1e-11 * gold["fabs"])
    ds = [sl.g.diag() for sl in slabs]
    assert abs(sum(d["ncap"] for d in ds) - int(gold["ncap"])) <= max(2, 0.02 * int(gold["ncap"]))
    assert np.max(np.abs(np.max([d["alpha"] for d in ds], axis=0) - gold["alpha"])) < 1e-12
    dep = sum(d["deposited"] for d in ds)
    assert np.max(np.abs(dep - gold["deposited"])) <= 1e-10 * gold["deposited"][0]
    for sl in slabs:
        sl.close()


def _rank_main(rank, world, port, case, q):
    """One process = one rank with its own CUDA context and Slab handle on the ONE GPU; torch.distributed over gloo."""
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    from paper_1511_02137_b200 import hydro as H
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n = case["n"]
    c = S.scaled_config(0, n)
    U0 = S.make_state(c)
    sl = SL.Slab(H, n, c["dx"], c["dt"], rank, world)
    sl.set_state(U0)
    _setup(sl, case)
    SL.run_distributed(sl, case["steps"], dist, overlap=case.get("overlap"))
    d = sl.g.diag()
    q.put((rank, sl.owned(), d["deposited"], d["ncap"], d["alpha"], sl.g.limited_faces()))
    dist.barrier()
    sl.close()
    dist.destroy_process_group()


@pytest.mark.gpu
@pytest.mark.parametrize("case", [
    dict(n=(32, 24, 40), world=2, steps=3, jets=[((-0.5, 0.0, -0.25), (0.1, 0.1, 1.0))]),                 # overlapped
    dict(n=(32, 24, 40), world=2, steps=3, jets=[((-0.5, 0.0, -0.25), (0.1, 0.1, 1.0))], overlap=False),
    dict(n=(32, 24, 40), world=2, steps=3, jets=[((-0.5, 0.0, -0.25), (0.1, 0.1, 1.0))], limiter=True),
])
def test_run_distributed_two_processes_one_gpu(H, case):
    """`slab.run_distributed` end to end: two processes, each with its own handle on this one GPU, alpha and halos over
    torch.distributed (gloo, staged through the host), a jet that crosses the slab face (z = -0.25 -> +0.35 over the run
    ... the face is at z = 0): owned planes bitwise equal to the single-handle run.  Ranks never wait on one another's
    kernels: every exchange is host-synchronised."""
    import torch.multiprocessing as mp
    c, kw, U0, (Uref, dref, qref, nlim_ref) = _reference_run(H, case)
    world = case["world"]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_rank_main, args=(r, world, port, case, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted((q.get(timeout=600) for _ in ps), key=lambda t: t[0])
    for p in ps:
        p.join(timeout=120)
        assert p.exitcode == 0
    U = np.concatenate([r[1] for r in res], axis=1)
    assert np.array_equal(U, Uref)
    assert np.allclose(sum(r[2] for r in res), dref["deposited"], rtol=1e-13, atol=0)
    assert sum(r[3] for r in res) == dref["ncap"]
    assert np.array_equal(np.max([r[4] for r in res], axis=0), dref["alpha"])
    assert sum(r[5] for r in res) == nlim_ref


@pytest.mark.gpu
def test_slab_argument_checks(H):
    g = H.Hydro(16, 16, 12, 0.1, 0.02)
    with pytest.raises(H.HydroError):
        g.set_slab(32, 8, 2, 8)          # an interior low end needs 4 halo planes
    with pytest.raises(H.HydroError):
        g.set_slab(8, 0, 0, 12)          # local array larger than the grid
    g.set_slab(32, 8, 4, 8)
    # a Gaussian deposit whose cube is wider than the halo cannot be split over slabs (R = ceil(3 sigma/dx) > 4)
    g.set_deposit_width(0.13)
    with pytest.raises(H.HydroError):
        g.set_deposit_width(0.25)
    g.set_limiter(True)
    with pytest.raises(H.HydroError):
        g.stage_sweeps_part(0, 0)        # the limiter needs the halos before the x sweep: no split stage
    g.close()
    g = H.Hydro(16, 16, 12, 0.1, 0.02)
    g.set_deposit_width(0.25)
    with pytest.raises(H.HydroError):
        g.set_slab(32, 8, 4, 8)
    g.close()

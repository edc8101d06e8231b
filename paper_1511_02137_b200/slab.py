"""z-slab decomposition of one grid over several ranks -- host-side plumbing only.

Every step of the path still runs in the library's kernels (include/hydro.h, "z-slab decomposition"); this module
splits the planes, builds each rank's local array (owned planes + 4 halo planes per neighbour), and moves the two things
that must cross ranks once per stage: the three Lax-Friedrichs speeds (MAX, reading R4) and the 4 boundary planes per
face (halo exchange).

Schedule of one stage s (`run_distributed`, and `run_local` in lock step for all slabs of one process):

    overlapped (default)                                         serial (limiter or Gaussian deposit: they need the
                                                                 halos before the x sweep)
    prims of the OWNED planes + local alpha maxima               finish the halo exchange of the input state, unpack
    alpha: MAX over ranks of three 64-bit patterns, on device    prims of all planes, alpha exchange
    x sweep + source + y sweep on the owned planes               all sweeps
    finish the halo exchange of the input state, unpack
    prims of the halo planes, z sweep
    pack the output state's boundary planes, POST their exchange (completed in the next stage, behind the x/y sweeps)

Everything is enqueued on ONE CUDA stream per rank (the handle's); over NCCL the transfer runs on a second stream
between two events, and no call in the loop blocks the host.  Transports:

  * `DistTransport`   one process per GPU, torch.distributed: NCCL (device buffers, stream-ordered) or gloo (staged
                      through host tensors; used by the tests, which have one GPU);
  * `run_local`       all slabs in ONE process on one device, exchanged by device copies -- the way to check the
                      decomposition on a single GPU without kernels that wait on one another.

The owned planes of a slab run are bitwise identical to the one-GPU run: same kernels, same data, same alpha.
"""
import numpy as np

HALO = 4


def split_planes(nz, world):
    """Contiguous, nearly equal plane ranges [g0, g1) per rank; every rank gets at least HALO planes."""
    if world < 1 or nz < HALO * world:
        raise ValueError("need at least %d planes per rank" % HALO)
    base, rem = divmod(nz, world)
    out, g = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((g, g + n))
        g += n
    return out


def local_extent(nz, world, rank):
    """(k_offset, nz_local, own_lo, own_hi) of rank's local array: halos only towards existing neighbours."""
    g0, g1 = split_planes(nz, world)[rank]
    lo = HALO if rank > 0 else 0
    hi = HALO if rank < world - 1 else 0
    return g0 - lo, (g1 - g0) + lo + hi, lo, lo + (g1 - g0)


class Slab:
    """One rank's part of the grid: a Hydro handle on the local array + its place in the decomposition."""

    def __init__(self, H, n, dx, dt, rank, world, stream=None, **kw):
        import torch
        nx, ny, nz = n
        self.rank, self.world, self.nz_global = rank, world, nz
        self.k_offset, self.nz_local, self.own_lo, self.own_hi = local_extent(nz, world, rank)
        self.stream = stream if stream is not None else torch.cuda.Stream()
        self.g = H.Hydro(nx, ny, self.nz_local, dx, dt, stream=self.stream, **kw)
        self.g.set_slab(nz, self.k_offset, self.own_lo, self.own_hi)
        tdt = torch.float64 if self.g.dtype == np.float64 else torch.float32
        nr = self.g.halo_reals()
        self.send = [torch.empty(nr, dtype=tdt, device="cuda") for _ in range(2)]     # [low face, high face]
        self.recv = [torch.empty(nr, dtype=tdt, device="cuda") for _ in range(2)]
        self.bits = torch.zeros(3, dtype=torch.int64, device="cuda")                  # alpha bit patterns
        self.limiter, self.sigma = False, 0.0
        self.pending = None                      # stage whose output halos are in flight

    def set_limiter(self, on=True):
        self.g.set_limiter(on)
        self.limiter = bool(on)

    def set_deposit_width(self, sigma):
        self.g.set_deposit_width(sigma)
        self.sigma = float(sigma)

    @property
    def overlap(self):
        """x/y sweeps may run while the halos fly unless a step of the stage needs them earlier (hydro.h)."""
        return not self.limiter and not self.sigma > 0.0

    def set_state(self, U_global):
        """U_global: (nf, nz, ny, nx) array of the WHOLE grid (every rank slices its local array, halos included)."""
        self.g.set_state(np.ascontiguousarray(U_global[:, self.k_offset:self.k_offset + self.nz_local]))
        self.pending = None

    def owned(self, which=0):
        return self.g.get_fields(which)[:, self.own_lo:self.own_hi]

    def has_neighbour(self, side):
        return self.rank > 0 if side == 0 else self.rank < self.world - 1

    def pack(self, s):
        for side in (0, 1):
            if self.has_neighbour(side):
                self.g.halo(s, side, False, self.send[side])

    def unpack(self, s):
        for side in (0, 1):
            if self.has_neighbour(side):
                self.g.halo(s, side, True, self.recv[side])

    def close(self):
        self.g.close()


# ------------------------------------------------------------------------------------------------ transports
class DistTransport:
    """torch.distributed: NCCL moves device buffers between two stream events; gloo is staged through host tensors."""

    def __init__(self, dist):
        import torch
        self.dist = dist
        self.nccl = dist.get_backend() == "nccl"
        self.comm = torch.cuda.Stream() if self.nccl else None
        self.works, self.host_recv = [], None

    def allreduce_alpha(self, slab, s):
        import torch
        with torch.cuda.stream(slab.stream):
            slab.g.stage_alpha_dev(s, slab.bits)
            if self.nccl:                                            # stays on the device, ordered by the stream
                self.dist.all_reduce(slab.bits, op=self.dist.ReduceOp.MAX)
            else:
                h = slab.bits.cpu()
                self.dist.all_reduce(h, op=self.dist.ReduceOp.MAX)
                slab.bits.copy_(h)
            slab.g.stage_alpha_dev(s, slab.bits, set=True)

    def post(self, slab, s):
        """Pack stage s's output boundary planes and start their exchange."""
        import torch
        with torch.cuda.stream(slab.stream):
            slab.pack(s)
            if self.nccl:
                ev = torch.cuda.Event()
                ev.record(slab.stream)
                self.comm.wait_event(ev)
                with torch.cuda.stream(self.comm):
                    self.works = exchange_faces(slab.send, slab.recv, slab.rank, slab.world, self.dist, wait=False)
            else:
                slab.stream.synchronize()
                hs = [t.cpu() for t in slab.send]
                self.host_recv = [torch.empty_like(t) for t in hs]
                self.works = exchange_faces(hs, self.host_recv, slab.rank, slab.world, self.dist, wait=False)
                self._keep = hs
        slab.pending = s

    def complete(self, slab):
        """Make the handle's stream wait for the posted exchange and unpack it into the halo planes."""
        import torch
        if slab.pending is None:
            return
        with torch.cuda.stream(slab.stream):
            for w in self.works:
                w.wait()                                             # NCCL: the CURRENT stream (the handle's) waits
            if not self.nccl:
                for side in (0, 1):
                    slab.recv[side].copy_(self.host_recv[side])
            slab.unpack(slab.pending)
        self.works = []
        slab.pending = None


def exchange_faces(send, recv, rank, world, dist, wait=True):
    """Neighbour exchange of the packed faces over torch.distributed: send[0] -> rank-1, send[1] -> rank+1,
    recv[0] <- rank-1 (its high face), recv[1] <- rank+1 (its low face).  Works on CPU (gloo) and CUDA (nccl) tensors.
    Returns the list of work handles (already waited for if `wait`)."""
    ops = []
    if rank > 0:
        ops += [dist.P2POp(dist.isend, send[0], rank - 1), dist.P2POp(dist.irecv, recv[0], rank - 1)]
    if rank < world - 1:
        ops += [dist.P2POp(dist.isend, send[1], rank + 1), dist.P2POp(dist.irecv, recv[1], rank + 1)]
    works = list(dist.batch_isend_irecv(ops)) if ops else []
    if wait:
        for w in works:
            w.wait()
    return works


def allreduce_max(values, dist, device="cpu"):
    import torch
    t = torch.tensor(values, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


# ------------------------------------------------------------------------------------------------ the stage loop
def _stage(slab, s, tr, overlap):
    g = slab.g
    if overlap:
        g.stage_prims_part(s, 0)
        if tr is not None:
            tr.allreduce_alpha(slab, s)
        g.stage_sweeps_part(s, 0)
        if tr is not None:
            tr.complete(slab)
        g.stage_prims_part(s, 1)
        g.stage_sweeps_part(s, 1)
    else:
        if tr is not None:
            tr.complete(slab)
        g.stage_prims(s)
        if tr is not None:
            tr.allreduce_alpha(slab, s)
        g.stage_sweeps(s)
    if tr is not None:
        tr.post(slab, s)


def run_distributed(slab, nsteps, dist, overlap=None):
    """One rank's loop (one process per GPU, torch.distributed initialised by the caller).  On return the halo planes
    of the current state are valid again (the last exchange has been completed)."""
    single = dist is None or slab.world == 1
    tr = None if single else DistTransport(dist)
    ov = slab.overlap if overlap is None else (overlap and slab.overlap)
    for _ in range(nsteps):
        for s in range(3):
            _stage(slab, s, tr, ov)
    if tr is not None:
        tr.complete(slab)


def run_local(slabs, nsteps, overlap=None):
    """Advance all slabs of ONE process in lock step with the schedule of `run_distributed`; alpha and the halos move by
    device copies on the slabs' common stream (all slabs must have been created on the same torch stream)."""
    import torch
    st = slabs[0].stream
    assert all(sl.stream is st for sl in slabs), "run_local: create the slabs on one common torch stream"
    ov = all(sl.overlap for sl in slabs) if overlap is None else (overlap and all(sl.overlap for sl in slabs))

    def alpha(s):
        with torch.cuda.stream(st):
            for sl in slabs:
                sl.g.stage_alpha_dev(s, sl.bits)
            m = torch.stack([sl.bits for sl in slabs]).max(dim=0).values
            for sl in slabs:
                sl.bits.copy_(m)
                sl.g.stage_alpha_dev(s, sl.bits, set=True)

    def complete():
        with torch.cuda.stream(st):
            for r, sl in enumerate(slabs):
                if sl.pending is None:
                    continue
                if sl.has_neighbour(0):
                    sl.recv[0].copy_(slabs[r - 1].send[1])
                if sl.has_neighbour(1):
                    sl.recv[1].copy_(slabs[r + 1].send[0])
                sl.unpack(sl.pending)
                sl.pending = None

    for _ in range(nsteps):
        for s in range(3):
            if ov:
                for sl in slabs:
                    sl.g.stage_prims_part(s, 0)
                alpha(s)
                for sl in slabs:
                    sl.g.stage_sweeps_part(s, 0)
                complete()
                for sl in slabs:
                    sl.g.stage_prims_part(s, 1)
                    sl.g.stage_sweeps_part(s, 1)
            else:
                complete()
                for sl in slabs:
                    sl.g.stage_prims(s)
                alpha(s)
                for sl in slabs:
                    sl.g.stage_sweeps(s)
            for sl in slabs:                             # pack every slab before any neighbour's unpack reads it
                sl.pack(s)
                sl.pending = s
    complete()

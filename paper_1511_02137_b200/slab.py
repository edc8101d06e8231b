"""z-slab decomposition of one grid over several ranks -- host-side plumbing only.

Every step of the path still runs in the library's kernels (include/hydro.h, "z-slab decomposition"); this module
splits the planes, builds each rank's local array (owned planes + 4 halo planes per neighbour), and moves the two things
that must cross ranks once per stage: the three Lax-Friedrichs speeds (MAX, reading R4) and the 4 boundary planes per
face (halo exchange).  Two transports:

  * `TorchDistComm`  one process per GPU, torch.distributed (NCCL on GPUs; the tests drive the same code over gloo);
  * `run_local`      all slabs in ONE process on one device, exchanged by device copies -- the way to check the
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

    def __init__(self, H, n, dx, dt, rank, world, **kw):
        import torch
        nx, ny, nz = n
        self.rank, self.world, self.nz_global = rank, world, nz
        self.k_offset, self.nz_local, self.own_lo, self.own_hi = local_extent(nz, world, rank)
        self.g = H.Hydro(nx, ny, self.nz_local, dx, dt, **kw)
        self.g.set_slab(nz, self.k_offset, self.own_lo, self.own_hi)
        tdt = torch.float64 if self.g.dtype == np.float64 else torch.float32
        nr = self.g.halo_reals()
        self.send = [torch.empty(nr, dtype=tdt, device="cuda") for _ in range(2)]     # [low face, high face]
        self.recv = [torch.empty(nr, dtype=tdt, device="cuda") for _ in range(2)]

    def set_state(self, U_global):
        """U_global: (nf, nz, ny, nx) array of the WHOLE grid (every rank slices its local array, halos included)."""
        self.g.set_state(np.ascontiguousarray(U_global[:, self.k_offset:self.k_offset + self.nz_local]))

    def owned(self, which=0):
        return self.g.get_fields(which)[:, self.own_lo:self.own_hi]

    def has_neighbour(self, side):
        return self.rank > 0 if side == 0 else self.rank < self.world - 1

    def close(self):
        self.g.close()


def run_local(slabs, nsteps):
    """Advance all slabs (one process, one device) in lock step, exchanging alpha and halos by local copies."""
    for _ in range(nsteps):
        for s in range(3):
            for sl in slabs:
                sl.g.stage_prims(s)
            alpha = np.max([sl.g.stage_alpha(s) for sl in slabs], axis=0)
            for sl in slabs:
                sl.g.stage_alpha(s, list(alpha))
                sl.g.stage_sweeps(s)
            for sl in slabs:
                for side in (0, 1):
                    if sl.has_neighbour(side):
                        sl.g.halo(s, side, False, sl.send[side])
            for sl in slabs:
                sl.g.synchronize()
            for r, sl in enumerate(slabs):
                if sl.has_neighbour(0):
                    sl.recv[0].copy_(slabs[r - 1].send[1])
                if sl.has_neighbour(1):
                    sl.recv[1].copy_(slabs[r + 1].send[0])
            import torch
            torch.cuda.synchronize()
            for sl in slabs:
                for side in (0, 1):
                    if sl.has_neighbour(side):
                        sl.g.halo(s, side, True, sl.recv[side])


def exchange_faces(send, recv, rank, world, dist):
    """Neighbour exchange of the packed faces over torch.distributed: send[0] -> rank-1, send[1] -> rank+1,
    recv[0] <- rank-1 (its high face), recv[1] <- rank+1 (its low face).  Works on CPU (gloo) and CUDA (nccl) tensors."""
    ops = []
    if rank > 0:
        ops += [dist.P2POp(dist.isend, send[0], rank - 1), dist.P2POp(dist.irecv, recv[0], rank - 1)]
    if rank < world - 1:
        ops += [dist.P2POp(dist.isend, send[1], rank + 1), dist.P2POp(dist.irecv, recv[1], rank + 1)]
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


def allreduce_max(values, dist, device="cpu"):
    import torch
    t = torch.tensor(values, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def run_distributed(slab, nsteps, dist):
    """One rank's loop (one process per GPU, torch.distributed initialised by the caller)."""
    import torch
    single = dist is None or slab.world == 1
    dev = "cpu" if single or dist.get_backend() != "nccl" else "cuda"
    for _ in range(nsteps):
        for s in range(3):
            slab.g.stage_prims(s)
            if not single:
                slab.g.stage_alpha(s, allreduce_max(slab.g.stage_alpha(s), dist, dev))
            slab.g.stage_sweeps(s)
            if single:
                continue
            for side in (0, 1):
                if slab.has_neighbour(side):
                    slab.g.halo(s, side, False, slab.send[side])
            slab.g.synchronize()
            if dev == "cuda":
                exchange_faces(slab.send, slab.recv, slab.rank, slab.world, dist)
            else:                                   # gloo: stage through host tensors
                hs = [t.cpu() for t in slab.send]
                hr = [torch.empty_like(t) for t in hs]
                exchange_faces(hs, hr, slab.rank, slab.world, dist)
                for side in (0, 1):
                    slab.recv[side].copy_(hr[side])
                torch.cuda.synchronize()
            for side in (0, 1):
                if slab.has_neighbour(side):
                    slab.g.halo(s, side, True, slab.recv[side])

"""Seeded synthetic inputs shaped like the paper's workloads -- the BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle (tests, bench.py).  It holds none of the
method's arithmetic: it only builds initial conserved fields U = T^{0 nu} from an analytic (e, u^i)
profile with eq. (1) of the paper read forwards, E = (e+p) gamma^2 - p,
M = (e+p) gamma^2 v with p = e/3, plus the seeded noise of reading R12.  numpy only.

Recipe (reading R12):
  * cell centres x_i = (i + 1/2 - n/2) dx on every axis (R6);
  * e = peak * exp(-x^2/2sx^2 - y^2/2sy^2 - z^2/2sz^2) + 0.01 + 1e-6 * r,  r in [0,1) from
    splitmix64(seed + linear cell index) >> 11, seed = 1234;
  * u^i = coef * x^i / R_i is the spatial part of the 4-velocity: gamma = sqrt(1+|u|^2), v = u/gamma;
  * config 4: N_B = (e/10) gamma.
"""
import numpy as np

SEED = 1234

# name -> dict(grid, dx, dt, steps, nf, ic parameters, jets)
CONFIGS = {
    0: dict(n=(32, 32, 32), dx=0.1, dt=0.02, steps=10, nf=4, kind="gauss", peak=10.0, sigma=(1.0, 0.8, 1.2),
            R=(2.0, 1.6, 2.4), ucoef=0.1, jets=[((-1.0, 0.0, 0.0), (1.0, 0.0, 0.0))]),
    1: dict(n=(512, 8, 8), dx=0.01, dt=0.004, steps=375, nf=4, kind="tube", eL=10.0, eR=1.0, axis=0, jets=[]),
    2: dict(n=(128, 128, 128), dx=0.1, dt=0.02, steps=50, nf=4, kind="gauss", peak=30.0, sigma=(1.5, 1.2, 1.8),
            R=(3.0, 2.4, 3.6), ucoef=0.1, jets=[((-3.0, 0.0, 0.0), (1.0, 0.0, 0.0))]),
    3: dict(n=(256, 256, 256), dx=0.1, dt=0.02, steps=120, nf=4, kind="gauss", peak=30.0, sigma=(3.0, 2.4, 3.6),
            R=(3.0, 2.4, 3.6), ucoef=0.15, jets=[((-5.0, 0.0, 0.0), (1.0, 0.0, 0.0))]),
    4: dict(n=(512, 512, 512), dx=0.05, dt=0.01, steps=200, nf=5, kind="gauss", peak=30.0, sigma=(3.0, 2.4, 3.6),
            R=(3.0, 2.4, 3.6), ucoef=0.15,
            jets=[((0.0, 0.0, 0.0), (1.0, 0.0, 0.0)), ((0.0, 0.0, 0.0), (-1.0, 0.0, 0.0))]),
}
KAPPA_RAD, KAPPA_COLL, CR_OVER_CF = 4.0, 2.5, 1.0


def splitmix64_unit(seed, index):
    """Counter-based uniform [0,1): splitmix64 of (seed + index), top 53 bits.  index: uint64 array."""
    with np.errstate(over="ignore"):
        z = (np.asarray(index, dtype=np.uint64) + np.uint64(seed)) * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def cell_centres(n, dx):
    return (np.arange(n, dtype=np.float64) + 0.5 - 0.5 * n) * dx


def prim_to_cons(e, ux, uy, uz, nb=None):
    """eq. (1) forwards with p = e/3 and u^i = gamma v^i: E = (4/3) e gamma^2 - e/3, M^i = (4/3) e gamma u^i."""
    g2 = 1.0 + ux * ux + uy * uy + uz * uz
    g = np.sqrt(g2)
    w = (4.0 / 3.0) * e
    fields = [w * g2 - e / 3.0, w * g * ux, w * g * uy, w * g * uz]
    if nb is not None:
        fields.append(nb * g)
    return np.stack(fields, axis=0)


def gaussian_flow(n, dx, peak, sigma, R, ucoef, nf=4, noise=1e-6, seed=SEED, background=0.01,
                  z_range=None):
    """Ellipsoidal-flow stand-in (R12).  Returns U of shape (nf, nz, ny, nx); z_range = (k0, k1) builds a slab."""
    nx, ny, nz = n
    k0, k1 = (0, nz) if z_range is None else z_range
    x = cell_centres(nx, dx)[None, None, :]
    y = cell_centres(ny, dx)[None, :, None]
    z = cell_centres(nz, dx)[k0:k1, None, None]
    e = peak * np.exp(-x * x / (2 * sigma[0] ** 2) - y * y / (2 * sigma[1] ** 2) - z * z / (2 * sigma[2] ** 2))
    e = e + background
    if noise:
        kk = np.arange(k0, k1, dtype=np.uint64)[:, None, None]
        jj = np.arange(ny, dtype=np.uint64)[None, :, None]
        ii = np.arange(nx, dtype=np.uint64)[None, None, :]
        lin = (kk * np.uint64(ny) + jj) * np.uint64(nx) + ii
        e = e + noise * splitmix64_unit(seed, lin)
    ux = np.broadcast_to(ucoef * x / R[0], e.shape)
    uy = np.broadcast_to(ucoef * y / R[1], e.shape)
    uz = np.broadcast_to(ucoef * z / R[2], e.shape)
    nb = None
    if nf == 5:
        nb = e / 10.0
    return np.ascontiguousarray(prim_to_cons(e, ux, uy, uz, nb))


def shock_tube(n, eL, eR, axis=0, nf=4):
    """Config 1 (R11): e = eL in the lower half along `axis`, eR in the upper half, at rest."""
    nx, ny, nz = n
    e = np.empty((nz, ny, nx))
    m = (nx, ny, nz)[axis]
    prof = np.where(np.arange(m) < m // 2, eL, eR).astype(np.float64)
    shape = [1, 1, 1]
    shape[2 - axis] = m
    e[...] = prof.reshape(shape)
    zero = np.zeros_like(e)
    nb = e / 10.0 if nf == 5 else None
    return np.ascontiguousarray(prim_to_cons(e, zero, zero, zero, nb))


def make_state(cfg, noise=True, z_range=None):
    """Initial U for BASELINE config `cfg` (int key of CONFIGS or a dict of the same form)."""
    c = CONFIGS[cfg] if not isinstance(cfg, dict) else cfg
    if c["kind"] == "tube":
        return shock_tube(c["n"], c["eL"], c["eR"], c.get("axis", 0), c["nf"])
    return gaussian_flow(c["n"], c["dx"], c["peak"], c["sigma"], c["R"], c["ucoef"], c["nf"],
                         noise=1e-6 if noise else 0.0, z_range=z_range)


def scaled_config(cfg, n):
    """A copy of config `cfg` on an n = (nx, ny, nz) grid with the same dx/dt/IC (for small parity cases)."""
    c = dict(CONFIGS[cfg])
    c["n"] = tuple(n)
    return c

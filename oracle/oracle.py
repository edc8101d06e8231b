"""ctypes loader for the CPU oracle (oracle/hydro_oracle.cpp).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It shares no code with the CUDA path (paper_1511_02137_b200/csrc, include/).

The oracle follows PAPER.md:17-31 (eqs. 1-3), :25 (WENO7, RK3), :49 (dx, dt, grid, EOS) and the
readings R1-R14 of DESIGN.md; see the header of hydro_oracle.cpp.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hydro_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

# oracle defaults = readings R3 / R9
WENO_EPS = 1e-6
V_CAP_DELTA = 1e-10
E_FLOOR = 1e-12


def build(force=False):
    """g++ -O2 -ffp-contract=off -fopenmp: the oracle's rounding must not depend on host FMA."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        d, i, p, ll = C.c_double, C.c_int, C.c_void_p, C.c_longlong
        dp = C.POINTER(C.c_double)
        L.oracle_create.restype = p
        L.oracle_create.argtypes = [i, i, i, d, d, i, d, d, d]
        L.oracle_destroy.argtypes = [p]
        L.oracle_set_state.argtypes = [p, dp]
        L.oracle_add_jet.restype = i
        L.oracle_add_jet.argtypes = [p] + [d] * 9
        L.oracle_clear_jets.argtypes = [p]
        L.oracle_step.argtypes = [p, i]
        L.oracle_get_fields.argtypes = [p, dp, i]
        L.oracle_get_diag.argtypes = [p, dp, dp, C.POINTER(ll), C.POINTER(i), dp, C.POINTER(ll)]
        L.oracle_eval_rhs.argtypes = [p, d, dp]
        L.oracle_last_stage_q.argtypes = [p, dp]
        L.oracle_con2prim.argtypes = [d] * 7 + [dp, C.POINTER(i)]
        L.oracle_wavespeeds.argtypes = [d, d, d, dp]
        L.oracle_weno7.restype = d
        L.oracle_weno7.argtypes = [dp, d]
        L.oracle_weno7_parts.argtypes = [dp, d, dp, dp, dp, dp]
        L.oracle_interface_flux.argtypes = [i, i, dp, d, d, d, d, dp]
        L.oracle_interface_flux_order.argtypes = [i, i, dp, d, d, d, d, i, dp]
        L.oracle_set_limiter.restype = ll
        L.oracle_set_limiter.argtypes = [p, i]
        L.oracle_limited_faces.restype = ll
        L.oracle_limited_faces.argtypes = [p]
        L.oracle_set_deposit_width.restype = i
        L.oracle_set_deposit_width.argtypes = [p, d]
        L.oracle_set_weno_order.restype = i
        L.oracle_set_weno_order.argtypes = [p, i]
        L.oracle_weno5.restype = d
        L.oracle_weno5.argtypes = [dp, d]
        L.oracle_weno5_parts.argtypes = [dp, d, dp, dp, dp]
        L.oracle_source_q.restype = d
        L.oracle_source_q.argtypes = [d] * 5
        L.oracle_jet_axis_index.restype = i
        L.oracle_jet_axis_index.argtypes = [d, i, d]
        L.oracle_constants.argtypes = [dp]
        L.oracle_count_flops.restype = d
        L.oracle_count_flops.argtypes = [i, dp]
        L.oracle_count_flops_order.restype = d
        L.oracle_count_flops_order.argtypes = [i, i, dp]
        L.oracle_num_threads.restype = i
        L.oracle_set_num_threads.argtypes = [i]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Oracle:
    """One CPU solver instance.  U arrays have shape (nf, nz, ny, nx), float64, x fastest."""

    def __init__(self, nx, ny, nz, dx, dt, nfields=4, weno_eps=WENO_EPS, v_cap_delta=V_CAP_DELTA,
                 e_floor=E_FLOOR, weno_order=7):
        self.L = lib()
        self.shape = (nfields, nz, ny, nx)
        self.h = self.L.oracle_create(nx, ny, nz, dx, dt, nfields, weno_eps, v_cap_delta, e_floor)
        if not self.h:
            raise ValueError("oracle_create: bad arguments")
        if self.L.oracle_set_weno_order(self.h, weno_order):
            raise ValueError("weno_order must be 5 or 7")
        self.njets = 0

    def close(self):
        if self.h:
            self.L.oracle_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, U):
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.shape == self.shape, (U.shape, self.shape)
        self.L.oracle_set_state(self.h, _dp(U))

    def add_jet(self, pos, direction, kappa_rad=4.0, kappa_coll=2.5, cr_over_cf=1.0):
        j = self.L.oracle_add_jet(self.h, *map(float, pos), *map(float, direction), kappa_rad, kappa_coll,
                                  cr_over_cf)
        if j < 0:
            raise ValueError("oracle_add_jet: zero direction")
        self.njets += 1
        return j

    def clear_jets(self):
        self.L.oracle_clear_jets(self.h)
        self.njets = 0

    def set_limiter(self, on=True):
        """Positivity-preserving flux limiter (reading R16)."""
        self.L.oracle_set_limiter(self.h, 1 if on else 0)

    def limited_faces(self):
        return self.L.oracle_limited_faces(self.h)

    def set_deposit_width(self, sigma):
        """Gaussian deposit of width sigma [fm] (reading R15); 0 = point deposit (R7)."""
        if self.L.oracle_set_deposit_width(self.h, float(sigma)):
            raise ValueError("sigma must be >= 0")

    def step(self, n=1):
        self.L.oracle_step(self.h, int(n))

    def get_fields(self, which=0):
        out = np.empty(self.shape, dtype=np.float64)
        self.L.oracle_get_fields(self.h, _dp(out), which)
        return out

    def eval_rhs(self, stage_c=0.0):
        out = np.empty(self.shape, dtype=np.float64)
        self.L.oracle_eval_rhs(self.h, float(stage_c), _dp(out))
        return out

    def diag(self):
        alpha = np.zeros(3)
        dep = np.zeros(4)
        cfl = C.c_double()
        ncap = C.c_longlong()
        nan = C.c_int()
        step = C.c_longlong()
        self.L.oracle_get_diag(self.h, _dp(alpha), C.byref(cfl), C.byref(ncap), C.byref(nan), _dp(dep),
                               C.byref(step))
        return dict(alpha=alpha, cfl=cfl.value, ncap=ncap.value, has_nan=nan.value, deposited=dep,
                    step=step.value)

    def last_stage_q(self):
        out = np.zeros((3, max(self.njets, 1)))
        self.L.oracle_last_stage_q(self.h, _dp(out))
        return out[:, :self.njets]


# ---------------------------------------------------------------- scalar entry points (pins)
def con2prim(E, Mx, My, Mz, NB=0.0, e_floor=E_FLOOR, delta=V_CAP_DELTA):
    out = np.zeros(6)
    lim = C.c_int()
    lib().oracle_con2prim(E, Mx, My, Mz, NB, e_floor, delta, _dp(out), C.byref(lim))
    return dict(e=out[0], p=out[1], v=out[2:5].copy(), n=out[5], limited=lim.value)


def wavespeeds(vx, vy, vz):
    out = np.zeros(3)
    lib().oracle_wavespeeds(vx, vy, vz, _dp(out))
    return out


def weno7(v, eps=WENO_EPS):
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert v.shape == (7,)
    return lib().oracle_weno7(_dp(v), eps)


def weno5(v, eps=WENO_EPS):
    """r = 3 reconstruction at the right face of the centre cell of the 5 values v."""
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert v.shape == (5,)
    return lib().oracle_weno5(_dp(v), eps)


def weno5_parts(v, eps=WENO_EPS):
    v = np.ascontiguousarray(v, dtype=np.float64)
    q, beta, om = np.zeros(3), np.zeros(3), np.zeros(3)
    lib().oracle_weno5_parts(_dp(v), eps, _dp(q), _dp(beta), _dp(om))
    return q, beta, om


def weno7_parts(v, eps=WENO_EPS):
    v = np.ascontiguousarray(v, dtype=np.float64)
    q, b, bs, om = np.zeros(4), np.zeros(4), np.zeros(4), np.zeros(4)
    lib().oracle_weno7_parts(_dp(v), eps, _dp(q), _dp(b), _dp(bs), _dp(om))
    return q, b, bs, om


def interface_flux(d, Uwin, alpha, eps=WENO_EPS, e_floor=E_FLOOR, delta=V_CAP_DELTA):
    Uwin = np.ascontiguousarray(Uwin, dtype=np.float64)
    assert Uwin.shape[0] == 8
    nf = Uwin.shape[1]
    out = np.zeros(nf)
    lib().oracle_interface_flux(d, nf, _dp(Uwin), alpha, eps, e_floor, delta, _dp(out))
    return out


def source_q(e_c, ell, k_rad=4.0, k_coll=2.5, crcf=1.0):
    return lib().oracle_source_q(e_c, ell, k_rad, k_coll, crcf)


def jet_axis_index(x, n, dx):
    return lib().oracle_jet_axis_index(x, n, dx)


def constants():
    out = np.zeros(3)
    lib().oracle_constants(_dp(out))
    return dict(hbarc=out[0], g=out[1], cs2=out[2])


def count_flops(nf=4, order=7):
    br = np.zeros(6)
    tot = lib().oracle_count_flops_order(nf, order, _dp(br))
    return tot, dict(con2prim=br[0], wavespeeds=br[1], interface_flux=br[2], divergence=br[3], rk=br[4],
                     weno7=br[5])


def num_threads():
    return lib().oracle_num_threads()


def set_num_threads(n):
    lib().oracle_set_num_threads(n)

"""Thin ctypes binding of the C-ABI CUDA library (include/hydro.h -> libhydro.so).

Argument marshalling only: every step of the path runs in the library's kernels.  torch is used for device
memory and streams.  There is NO CPU fallback: loading fails loudly if libhydro.so is missing, and
`Hydro(...)` fails with HYDRO_ECUDA without a CUDA device.

Names mirror the C entry points: hydro_create -> Hydro(...), hydro_set_state -> .set_state, hydro_add_jet ->
.add_jet, hydro_step -> .step, hydro_get_fields -> .get_fields, hydro_eval_rhs -> .eval_rhs, hydro_get_diag ->
.diag, ... (PAPER.md:17-31 for what they compute; include/hydro.h for layouts and error behaviour).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhydro.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, 1, 2, 3, 4
MEM_HOST, MEM_DEVICE = 0, 1
FIELDS_CONSERVED, FIELDS_PRIMITIVE = 0, 1
K_NAMES = ("prim", "sweep_x", "sweep_y", "sweep_z", "source")

# every symbol include/hydro.h declares (tests check that the library exports all of them)
SYMBOLS = ("hydro_create", "hydro_destroy", "hydro_set_state", "hydro_add_jet", "hydro_clear_jets", "hydro_set_step", "hydro_set_deposit_width", "hydro_set_limiter", "hydro_get_limited_faces", "hydro_set_slab", "hydro_stage_prims",
           "hydro_stage_alpha", "hydro_stage_sweeps", "hydro_stage_prims_part", "hydro_stage_sweeps_part", "hydro_stage_alpha_dev", "hydro_halo", "hydro_halo_reals", "hydro_step",
           "hydro_synchronize", "hydro_get_fields", "hydro_eval_rhs", "hydro_get_diag", "hydro_get_last_stage_q",
           "hydro_set_profiling", "hydro_get_kernel_times", "hydro_launch_count", "hydro_sweep_path", "hydro_measure_alu_peak",
           "hydro_wavespeeds_noalloc", "hydro_strerror", "hydro_last_cuda_error")


class EosT(C.Structure):
    _fields_ = [("eos", C.c_int), ("nfields", C.c_int), ("precision", C.c_int), ("weno_eps", C.c_double),
                ("v_cap_delta", C.c_double), ("e_floor", C.c_double), ("weno_order", C.c_int)]


class HydroError(RuntimeError):
    def __init__(self, code, what, detail=""):
        self.code = code
        RuntimeError.__init__(self, "%s failed: %s%s" % (what, _strerror(code), (" [" + detail + "]") if detail else ""))


_lib = None


def load():
    """dlopen libhydro.so (built in-tree by paper_1511_02137_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    try:                                   # (re)build in-tree if the library is missing or older than its sources
        from . import build as _build
        _build.build()
    except Exception as e:                 # no nvcc, or a compile error
        if not os.path.exists(LIB_PATH):
            raise ImportError("CUDA library %s is missing and could not be built (%s): run "
                              "`python -m paper_1511_02137_b200.build` (there is no CPU fallback)" % (LIB_PATH, e))
        if any(os.path.getmtime(LIB_PATH) < os.path.getmtime(d) for d in _build.DEPS):
            raise ImportError("CUDA library %s is older than its sources and the rebuild failed (%s): a stale binary "
                              "must not run against newer headers" % (LIB_PATH, e))
    L = C.CDLL(LIB_PATH)
    missing = [n for n in SYMBOLS if not hasattr(L, n)]
    if missing:
        raise ImportError("%s does not export %s: rebuild it (python -m paper_1511_02137_b200.build --force)" %
                          (LIB_PATH, ", ".join(missing)))
    vp, i, d, ll = C.c_void_p, C.c_int, C.c_double, C.c_longlong
    dp = C.POINTER(C.c_double)
    L.hydro_create.restype = i
    L.hydro_create.argtypes = [C.POINTER(vp), i, i, i, d, d, C.POINTER(EosT), vp]
    L.hydro_destroy.restype = None
    L.hydro_destroy.argtypes = [vp]
    L.hydro_set_state.restype = i
    L.hydro_set_state.argtypes = [vp, vp, i]
    L.hydro_add_jet.restype = i
    L.hydro_add_jet.argtypes = [vp] + [d] * 9 + [C.POINTER(i)]
    L.hydro_clear_jets.restype = i
    L.hydro_clear_jets.argtypes = [vp]
    L.hydro_set_step.restype = i
    L.hydro_set_step.argtypes = [vp, ll]
    L.hydro_set_slab.restype = i
    L.hydro_set_slab.argtypes = [vp, i, i, i, i]
    L.hydro_stage_prims.restype = i
    L.hydro_stage_prims.argtypes = [vp, i]
    L.hydro_stage_alpha.restype = i
    L.hydro_stage_alpha.argtypes = [vp, i, i, dp]
    L.hydro_stage_sweeps.restype = i
    L.hydro_stage_sweeps.argtypes = [vp, i]
    L.hydro_stage_prims_part.restype = i
    L.hydro_stage_prims_part.argtypes = [vp, i, i]
    L.hydro_stage_sweeps_part.restype = i
    L.hydro_stage_sweeps_part.argtypes = [vp, i, i]
    L.hydro_stage_alpha_dev.restype = i
    L.hydro_stage_alpha_dev.argtypes = [vp, i, i, vp]
    L.hydro_halo.restype = i
    L.hydro_halo.argtypes = [vp, i, i, i, vp]
    L.hydro_halo_reals.restype = ll
    L.hydro_halo_reals.argtypes = [vp]
    L.hydro_set_limiter.restype = i
    L.hydro_set_limiter.argtypes = [vp, i]
    L.hydro_get_limited_faces.restype = i
    L.hydro_get_limited_faces.argtypes = [vp, C.POINTER(ll)]
    L.hydro_set_deposit_width.restype = i
    L.hydro_set_deposit_width.argtypes = [vp, d]
    L.hydro_step.restype = i
    L.hydro_step.argtypes = [vp, i]
    L.hydro_synchronize.restype = i
    L.hydro_synchronize.argtypes = [vp]
    L.hydro_wavespeeds_noalloc.restype = i
    L.hydro_wavespeeds_noalloc.argtypes = [vp, i, i, i, i, d, d, vp, vp, vp, C.c_char_p, i]
    L.hydro_get_fields.restype = i
    L.hydro_get_fields.argtypes = [vp, vp, i, i]
    L.hydro_eval_rhs.restype = i
    L.hydro_eval_rhs.argtypes = [vp, d, vp, i]
    L.hydro_get_diag.restype = i
    L.hydro_get_diag.argtypes = [vp, dp, dp, C.POINTER(ll), C.POINTER(i), dp, C.POINTER(ll)]
    L.hydro_get_last_stage_q.restype = i
    L.hydro_get_last_stage_q.argtypes = [vp, i, dp]
    L.hydro_set_profiling.restype = i
    L.hydro_set_profiling.argtypes = [vp, i]
    L.hydro_get_kernel_times.restype = i
    L.hydro_get_kernel_times.argtypes = [vp, dp, C.POINTER(ll)]
    L.hydro_launch_count.restype = ll
    L.hydro_launch_count.argtypes = [vp]
    L.hydro_sweep_path.restype = i
    L.hydro_sweep_path.argtypes = [vp]
    L.hydro_measure_alu_peak.restype = i
    L.hydro_measure_alu_peak.argtypes = [i, d, vp, dp]
    L.hydro_strerror.restype = C.c_char_p
    L.hydro_strerror.argtypes = [i]
    L.hydro_last_cuda_error.restype = C.c_char_p
    L.hydro_last_cuda_error.argtypes = [vp]
    _lib = L
    return L


def _strerror(code):
    try:
        return load().hydro_strerror(code).decode()
    except Exception:
        return "error %d" % code


def _ptr_and_space(a):
    """(address, memspace, keepalive) of a numpy array (host) or a torch tensor (host or cuda)."""
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data, MEM_HOST, a
    import torch
    assert isinstance(a, torch.Tensor) and a.is_contiguous()
    return a.data_ptr(), (MEM_DEVICE if a.is_cuda else MEM_HOST), a


def measure_alu_peak(precision=64, millis=200.0, stream=None):
    """hydro_measure_alu_peak: achieved TFLOP/s of a register-resident FMA chain on all SMs."""
    out = C.c_double()
    rc = load().hydro_measure_alu_peak(precision, millis, C.c_void_p(stream or 0), C.byref(out))
    if rc != OK:
        raise HydroError(rc, "hydro_measure_alu_peak")
    return out.value


NOALLOC_MAX_CELLS = 262144


def wavespeeds_noalloc(U, alpha_out, counts_out=None, v_cap_delta=0.0, e_floor=0.0, stream=None):
    """hydro_wavespeeds_noalloc: alpha_d maxima (+ cap / NaN counts) of the fp64 CUDA tensor U (nf, nz, ny, nx) into the
    caller's CUDA tensors alpha_out (3 float64) and counts_out (2 int64, optional).  Allocates nothing; asynchronous."""
    L = load()
    nf, nz, ny, nx = U.shape
    err = C.create_string_buffer(256)
    rc = L.hydro_wavespeeds_noalloc(C.c_void_p(U.data_ptr()), nx, ny, nz, nf, float(v_cap_delta), float(e_floor),
                                    C.c_void_p(alpha_out.data_ptr()),
                                    C.c_void_p(counts_out.data_ptr() if counts_out is not None else 0),
                                    C.c_void_p(stream if stream else 0), err, 256)
    if rc != OK:
        raise HydroError(rc, "hydro_wavespeeds_noalloc", err.value.decode())


class Hydro:
    """One solver handle (hydro_t).  Arrays have shape (nfields, nz, ny, nx), x fastest."""

    def __init__(self, nx, ny, nz, dx, dt, nfields=4, precision=64, weno_eps=0.0, v_cap_delta=0.0, e_floor=0.0,
                 stream=None, weno_order=7):
        self.L = load()
        self.h = C.c_void_p()
        self.shape = (nfields, nz, ny, nx)
        self.nfields = nfields
        self.dtype = np.float64 if precision == 64 else np.float32
        eos = EosT(0, nfields, precision, weno_eps, v_cap_delta, e_floor, weno_order)
        self._stream = stream                      # keep a torch stream object alive
        sp = 0
        if stream is not None:
            sp = stream if isinstance(stream, int) else stream.cuda_stream
        rc = self.L.hydro_create(C.byref(self.h), nx, ny, nz, dx, dt, C.byref(eos), C.c_void_p(sp))
        if rc != OK:
            self.h = C.c_void_p()
            raise HydroError(rc, "hydro_create")
        self.njets = 0

    # -- helpers
    def _ck(self, rc, what):
        if rc != OK:
            raise HydroError(rc, what, self.L.hydro_last_cuda_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None) is not None and self.h:
            self.L.hydro_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, a):
        assert tuple(a.shape) == self.shape, (tuple(a.shape), self.shape)
        if isinstance(a, np.ndarray):
            assert a.dtype == self.dtype, (a.dtype, self.dtype)
        else:
            import torch
            assert a.dtype == (torch.float64 if self.dtype == np.float64 else torch.float32)

    # -- the C entry points
    def set_state(self, U):
        self._check(U)
        p, space, keep = _ptr_and_space(U)
        self._ck(self.L.hydro_set_state(self.h, C.c_void_p(p), space), "hydro_set_state")

    def add_jet(self, pos, direction, kappa_rad=4.0, kappa_coll=2.5, cr_over_cf=1.0):
        jid = C.c_int()
        self._ck(self.L.hydro_add_jet(self.h, *map(float, pos), *map(float, direction), kappa_rad, kappa_coll,
                                      cr_over_cf, C.byref(jid)), "hydro_add_jet")
        self.njets += 1
        return jid.value

    def set_step(self, step):
        self._ck(self.L.hydro_set_step(self.h, int(step)), "hydro_set_step")

    def clear_jets(self):
        self._ck(self.L.hydro_clear_jets(self.h), "hydro_clear_jets")
        self.njets = 0

    # -- z-slab decomposition (f-4): see include/hydro.h and paper_1511_02137_b200/slab.py
    def set_slab(self, nz_global, k_offset, own_lo, own_hi):
        self._ck(self.L.hydro_set_slab(self.h, nz_global, k_offset, own_lo, own_hi), "hydro_set_slab")

    def stage_prims(self, s):
        self._ck(self.L.hydro_stage_prims(self.h, s), "hydro_stage_prims")

    def stage_alpha(self, s, alpha=None):
        a = (C.c_double * 3)(*(alpha if alpha is not None else (0.0, 0.0, 0.0)))
        self._ck(self.L.hydro_stage_alpha(self.h, s, 0 if alpha is None else 1, a), "hydro_stage_alpha")
        return [a[0], a[1], a[2]]

    def stage_sweeps(self, s):
        self._ck(self.L.hydro_stage_sweeps(self.h, s), "hydro_stage_sweeps")

    def stage_prims_part(self, s, part):
        self._ck(self.L.hydro_stage_prims_part(self.h, s, part), "hydro_stage_prims_part")

    def stage_sweeps_part(self, s, part):
        self._ck(self.L.hydro_stage_sweeps_part(self.h, s, part), "hydro_stage_sweeps_part")

    def stage_alpha_dev(self, s, bits, set=False):
        """bits: CUDA int64 tensor of 3 elements (the alpha bit patterns); asynchronous on the handle's stream."""
        assert bits.is_cuda and bits.numel() >= 3 and bits.element_size() == 8
        self._ck(self.L.hydro_stage_alpha_dev(self.h, s, 1 if set else 0, C.c_void_p(bits.data_ptr())),
                 "hydro_stage_alpha_dev")

    def halo(self, s, side, unpack, buf):
        """buf: CUDA torch tensor of halo_reals() elements of the handle's dtype."""
        assert buf.is_cuda and buf.is_contiguous() and buf.numel() >= self.halo_reals()
        self._ck(self.L.hydro_halo(self.h, s, side, 1 if unpack else 0, C.c_void_p(buf.data_ptr())), "hydro_halo")

    def halo_reals(self):
        return self.L.hydro_halo_reals(self.h)

    def set_limiter(self, on=True):
        self._ck(self.L.hydro_set_limiter(self.h, 1 if on else 0), "hydro_set_limiter")

    def limited_faces(self):
        n = C.c_longlong()
        self._ck(self.L.hydro_get_limited_faces(self.h, C.byref(n)), "hydro_get_limited_faces")
        return n.value

    def set_deposit_width(self, sigma):
        self._ck(self.L.hydro_set_deposit_width(self.h, float(sigma)), "hydro_set_deposit_width")

    def step(self, n=1):
        self._ck(self.L.hydro_step(self.h, int(n)), "hydro_step")

    def synchronize(self):
        self._ck(self.L.hydro_synchronize(self.h), "hydro_synchronize")

    def get_fields(self, which=FIELDS_CONSERVED, out=None):
        if out is None:
            out = np.empty(self.shape, dtype=self.dtype)
        self._check(out)
        p, space, keep = _ptr_and_space(out)
        self._ck(self.L.hydro_get_fields(self.h, C.c_void_p(p), which, space), "hydro_get_fields")
        return out

    def eval_rhs(self, stage_c=0.0, out=None):
        if out is None:
            out = np.empty(self.shape, dtype=self.dtype)
        self._check(out)
        p, space, keep = _ptr_and_space(out)
        self._ck(self.L.hydro_eval_rhs(self.h, float(stage_c), C.c_void_p(p), space), "hydro_eval_rhs")
        return out

    def diag(self):
        """hydro_get_diag.  ncap, has_nan and deposited are committed by the stages of step() (and of the stage_* calls);
        eval_rhs() refreshes alpha only."""
        alpha = (C.c_double * 3)()
        dep = (C.c_double * 4)()
        cfl, ncap, nan, step = C.c_double(), C.c_longlong(), C.c_int(), C.c_longlong()
        self._ck(self.L.hydro_get_diag(self.h, alpha, C.byref(cfl), C.byref(ncap), C.byref(nan), dep, C.byref(step)),
                 "hydro_get_diag")
        return dict(alpha=np.array(alpha[:]), cfl=cfl.value, ncap=ncap.value, has_nan=nan.value,
                    deposited=np.array(dep[:]), step=step.value)

    def last_stage_q(self):
        out = np.zeros((3, self.njets))
        for j in range(self.njets):
            q = (C.c_double * 3)()
            self._ck(self.L.hydro_get_last_stage_q(self.h, j, q), "hydro_get_last_stage_q")
            out[:, j] = q[:]
        return out

    def set_profiling(self, enable=True):
        self._ck(self.L.hydro_set_profiling(self.h, 1 if enable else 0), "hydro_set_profiling")

    def kernel_times(self):
        ms = (C.c_double * len(K_NAMES))()
        n = (C.c_longlong * len(K_NAMES))()
        self._ck(self.L.hydro_get_kernel_times(self.h, ms, n), "hydro_get_kernel_times")
        return {k: dict(ms=ms[i], launches=n[i]) for i, k in enumerate(K_NAMES)}

    def launch_count(self):
        return self.L.hydro_launch_count(self.h)

    def uses_ring(self):
        return self.L.hydro_sweep_path(self.h) == 1

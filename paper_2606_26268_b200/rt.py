"""Thin ctypes binding of include/rt.h (librt_m1.so).  Argument marshalling only: every step of the
radiation sub-step runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and
streams; nothing here computes on the CPU and there is no fallback: a missing library or a missing
GPU raises.

Function names mirror the C ABI (rt_grid_create, rt_set_params, rt_set_opacity, rt_explicit_step,
rt_implicit_step, rt_cfl_dt, ...); `Grid` is a small handle owner around them.
"""
import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

CARTESIAN, CYLINDRICAL, SPHERICAL = 0, 1, 2
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT, BC_FIXED = 0, 1, 2, 3
SOLVER_HLL, SOLVER_GLF, SOLVER_RUSANOV = 0, 1, 2
FIX_FPRESERVING, FIX_PLUTO, FIX_CLIP = 0, 1, 2
RECON_PLM, RECON_LIMO3 = 0, 1
OPAC_PLANCK, OPAC_ROSSELAND, OPAC_SCATTER = 0, 1, 2
OK, ERR_INVALID_ARG, ERR_BAD_STATE, ERR_CUDA, ERR_NOT_FINITE = 0, 1, 2, 3, 4
NGHOST = 2
KERNEL_KINDS = ("ghost_fill", "thick_limit", "sweep_x1", "sweep_x2", "sweep_x3", "implicit", "cfl", "fused")
NKERNEL_KINDS = 8

_dp = C.POINTER(C.c_double)


class Params(C.Structure):
    _fields_ = [("chat", C.c_double), ("c", C.c_double), ("a_R", C.c_double), ("c_v", C.c_double),
                ("E_floor", C.c_double), ("solver", C.c_int32), ("thick_limit", C.c_int32),
                ("feedback_momentum", C.c_int32)]


class Opacity(C.Structure):
    _fields_ = [("kind", C.c_int32), ("kappa0", C.c_double), ("rho0", C.c_double), ("T0", C.c_double),
                ("a", C.c_double), ("b", C.c_double), ("kmin", C.c_double), ("kmax", C.c_double),
                ("n_lrho", C.c_int32), ("n_lT", C.c_int32), ("lrho_min", C.c_double), ("lrho_max", C.c_double),
                ("lT_min", C.c_double), ("lT_max", C.c_double), ("rho_unit", C.c_double), ("T_unit", C.c_double),
                ("log10_kappa", _dp)]


class RtError(RuntimeError):
    def __init__(self, call, status, message=""):
        self.status = status
        super().__init__("%s failed with status %d%s" % (call, status, (": " + message) if message else ""))


_lib = None

_SIGNATURES = {
    "rt_grid_create": (C.c_int32, [C.c_int32, C.POINTER(C.c_int32), C.c_int32, _dp, _dp, _dp, C.POINTER(C.c_int32),
                                   C.c_void_p, C.POINTER(C.c_void_p)]),
    "rt_grid_destroy": (C.c_int32, [C.c_void_p]),
    "rt_grid_get_metrics": (C.c_int32, [C.c_void_p, _dp, _dp, _dp, _dp]),
    "rt_set_params": (C.c_int32, [C.c_void_p, C.POINTER(Params)]),
    "rt_set_opacity": (C.c_int32, [C.c_void_p, C.c_int32, C.POINTER(Opacity)]),
    "rt_fill_ghosts": (C.c_int32, [C.c_void_p, C.POINTER(C.c_void_p)]),
    "rt_explicit_step": (C.c_int32, [C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p),
                                     C.POINTER(C.c_void_p)]),
    "rt_implicit_step": (C.c_int32, [C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p),
                                     C.POINTER(C.c_void_p)]),
    "rt_implicit_step_cfl": (C.c_int32, [C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p),
                                         C.POINTER(C.c_void_p), C.c_double, C.c_void_p]),
    "rt_substep": (C.c_int32, [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p),
                               C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]),
    "rt_set_irradiation": (C.c_int32, [C.c_void_p, C.c_void_p]),
    "rt_set_face_fix": (C.c_int32, [C.c_void_p, C.c_int32]),
    "rt_set_reconstruction": (C.c_int32, [C.c_void_p, C.c_int32, C.c_double]),
    "rt_irradiation_radial": (C.c_int32, [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]),
    "rt_rk2_step": (C.c_int32, [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p),
                                C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]),
    "rt_cfl_dt": (C.c_int32, [C.c_void_p, C.POINTER(C.c_void_p), C.c_double, _dp]),
    "rt_cfl_dt_async": (C.c_int32, [C.c_void_p, C.POINTER(C.c_void_p), C.c_double, C.c_void_p]),
    "rt_get_floor_counts": (C.c_int32, [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]),
    "rt_check_finite": (C.c_int32, [C.c_void_p, C.POINTER(C.c_void_p), C.c_void_p, C.POINTER(C.c_int64)]),
    "rt_get_launch_count": (C.c_int64, [C.c_void_p]),
    "rt_set_tuning": (C.c_int32, [C.c_void_p, C.c_int32, C.c_int32]),
    "rt_set_profiling": (C.c_int32, [C.c_void_p, C.c_int32]),
    "rt_get_kernel_times": (C.c_int32, [C.c_void_p, _dp, C.POINTER(C.c_int64)]),
    "rt_measure_fp64": (C.c_int32, [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32, _dp]),
    "rt_cfl_dt_uniform_noalloc": (C.c_int32, [C.c_void_p, C.POINTER(C.c_int32), _dp, C.c_double, C.c_double,
                                              C.POINTER(C.c_void_p), C.c_void_p, C.c_char_p, C.c_int32]),
    "rt_last_error": (C.c_char_p, [C.c_void_p]),
}


def exported_symbols():
    """names the C ABI must export (used by the CPU-side load test)"""
    return sorted(_SIGNATURES)


def lib():
    """load (building first if needed) librt_m1.so; raises if it cannot be had"""
    global _lib
    if _lib is None:
        path = _build.build()
        if not os.path.exists(path):
            raise RuntimeError("librt_m1.so is missing and could not be built")
        L = C.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)  # AttributeError if the symbol is missing: loud by design
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check_field(t, shape, name, device=None):
    if not isinstance(t, torch.Tensor):
        raise TypeError("%s must be a torch.Tensor on the GPU" % name)
    if not t.is_cuda:
        raise RuntimeError("%s is not a CUDA tensor: this library has no CPU path" % name)
    if device is not None and t.device != device:
        raise ValueError("%s lives on %s but the grid was created on %s" % (name, t.device, device))
    if t.dtype != torch.float64 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
        raise ValueError("%s must be contiguous float64 of shape %s (got %s %s)" % (name, tuple(shape), t.dtype,
                                                                                     tuple(t.shape)))


def _ptr_array(tensors):
    return (C.c_void_p * len(tensors))(*[t.data_ptr() for t in tensors])


def make_params(chat=1.0, c=1.0, a_R=1.0, c_v=1.5, E_floor=0.0, solver=SOLVER_HLL, thick_limit=0,
                feedback_momentum=0):
    return Params(chat, c, a_R, c_v, E_floor, solver, thick_limit, feedback_momentum)


def make_power_law(kappa0, a=0.0, b=0.0, rho0=1.0, T0=1.0, kmin=0.0, kmax=np.inf):
    o = Opacity()
    o.kind = 0
    o.kappa0, o.rho0, o.T0, o.a, o.b, o.kmin, o.kmax = kappa0, rho0, T0, a, b, kmin, kmax
    o.rho_unit = o.T_unit = 1.0
    return o


def make_table(log10_kappa, lrho_range, lT_range, rho_unit=1.0, T_unit=1.0):
    tab = np.ascontiguousarray(np.asarray(log10_kappa, dtype=np.float64))
    if tab.ndim != 2:
        raise ValueError("table must be 2-D (n_lT, n_lrho)")
    o = Opacity()
    o.kind = 1
    o.n_lT, o.n_lrho = tab.shape
    o.lrho_min, o.lrho_max = lrho_range
    o.lT_min, o.lT_max = lT_range
    o.rho_unit, o.T_unit = rho_unit, T_unit
    o.rho0 = o.T0 = 1.0
    o.log10_kappa = tab.ctypes.data_as(_dp)
    o._keep = tab
    return o


def opacity_from_spec(spec):
    """translate the plain-Python opacity description of rt_workloads into the C struct"""
    if spec["kind"] == "power":
        return make_power_law(spec["kappa0"], spec["a"], spec["b"], spec["rho0"], spec["T0"], spec["kmin"],
                              spec["kmax"])
    return make_table(spec["log10_kappa"], spec["lrho_range"], spec["lT_range"], spec["rho_unit"], spec["T_unit"])


def measure_fp64(blocks, threads, chains, iters, device="cuda:0"):
    """rt_measure_fp64: milliseconds of one launch of the DFMA microbenchmark and its DFMA thread-instruction count
    (chains: 1, 2, 4, 8 chains of 8 * iters; 101, 102, 104: 1, 2, 4 chains of 64 * iters; 204, 304, 214, 314: 4 chains of
    8 * iters with two / three register operands, without / with four fp32 multiplies per four DFMAs; include/rt.h)"""
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: paper_2606_26268_b200 has no CPU path")
    ms = C.c_double()
    with torch.cuda.device(torch.device(device)):
        st = torch.cuda.current_stream()
        rc = lib().rt_measure_fp64(C.c_void_p(st.cuda_stream), int(blocks), int(threads), int(chains), int(iters), C.byref(ms))
    if rc != OK:
        raise RtError("rt_measure_fp64", rc)
    nch, per = (chains, 8) if chains < 100 else (chains - 100, 64) if chains < 200 else (4, 8)
    return ms.value, float(blocks) * threads * nch * per * iters


NOALLOC_MAX_ROWS = 65536


def cfl_dt_uniform_noalloc(n, dx, chat, cfl, U, dt_device):
    """rt_cfl_dt_uniform_noalloc: the CFL time step of a uniform Cartesian grid into dt_device, through the entry point
    that allocates nothing (no handle; static device scratch; n[1] * n[2] <= NOALLOC_MAX_ROWS).  Enqueued on the current
    stream of the fields' device."""
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: paper_2606_26268_b200 has no CPU path")
    n = [int(v) for v in n]
    shape = tuple(v + 2 * NGHOST if v > 1 else 1 for v in reversed(n))
    for q in range(4):
        _check_field(U[q], shape, "U[%d]" % q, U[0].device if isinstance(U[0], torch.Tensor) else None)
    if not (dt_device.is_cuda and dt_device.dtype == torch.float64 and dt_device.numel() >= 1 and dt_device.device == U[0].device):
        raise ValueError("dt_device must be a CUDA float64 tensor on the fields' device")
    err = C.create_string_buffer(256)
    with torch.cuda.device(U[0].device):
        st = torch.cuda.current_stream()
        rc = lib().rt_cfl_dt_uniform_noalloc(C.c_void_p(st.cuda_stream), (C.c_int32 * 3)(*n), (C.c_double * 3)(*[float(v) for v in dx]),
                                             float(chat), float(cfl), _ptr_array(U), dt_device.data_ptr(), err, len(err))
    if rc != OK:
        raise RtError("rt_cfl_dt_uniform_noalloc", rc, err.value.decode())


class Grid:
    """Owner of one rt_grid handle.  All field arguments are CUDA float64 tensors of shape `self.shape`
    (ghosted, (nt3, nt2, nt1)); work is enqueued on the stream that was current at construction."""

    def __init__(self, geometry, n, x1f, x2f, x3f, bc, nghost=NGHOST, device="cuda:0", stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: paper_2606_26268_b200 has no CPU path")
        self.device = torch.device(device)
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        self.n = tuple(int(v) for v in n)
        self.gh = tuple(nghost if v > 1 else 0 for v in self.n)
        self.nt = tuple(v + 2 * g for v, g in zip(self.n, self.gh))
        self.shape = (self.nt[2], self.nt[1], self.nt[0])
        self.geometry = int(geometry)
        self.bc = tuple(int(b) for b in bc)
        xs = [np.ascontiguousarray(np.asarray(x, dtype=np.float64)) for x in (x1f, x2f, x3f)]
        for d in range(3):
            if xs[d].shape != (self.n[d] + 1,):
                raise ValueError("x%df must have n[%d] + 1 entries" % (d + 1, d))
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            rc = lib().rt_grid_create(self.geometry, (C.c_int32 * 3)(*self.n), int(nghost),
                                      xs[0].ctypes.data_as(_dp), xs[1].ctypes.data_as(_dp), xs[2].ctypes.data_as(_dp),
                                      (C.c_int32 * 6)(*self.bc), C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if rc != OK:
            raise RtError("rt_grid_create", rc)
        self._h = h

    def __del__(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:
            _lib.rt_grid_destroy(h)
            self._h = None

    # ------------------------------------------------------------------ helpers
    def _raise(self, call, rc):
        msg = lib().rt_last_error(self._h)
        raise RtError(call, rc, msg.decode() if msg else "")

    @property
    def interior(self):
        return tuple(slice(g, g + n) for g, n in zip(self.gh[::-1], self.n[::-1]))

    @property
    def ncells(self):
        return self.n[0] * self.n[1] * self.n[2]

    def zeros(self):
        return torch.zeros(self.shape, dtype=torch.float64, device=self.device)

    def to_device(self, a):
        return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).to(self.device)

    # ------------------------------------------------------------------ the C ABI, one method per call
    def set_params(self, params):
        rc = lib().rt_set_params(self._h, C.byref(params))
        if rc != OK:
            self._raise("rt_set_params", rc)
        self.params = params

    def set_opacity(self, which, o):
        rc = lib().rt_set_opacity(self._h, int(which), C.byref(o))
        if rc != OK:
            self._raise("rt_set_opacity", rc)

    def set_tuning(self, march_len=0, fused_seg=0):
        rc = lib().rt_set_tuning(self._h, int(march_len), int(fused_seg))
        if rc != OK:
            self._raise("rt_set_tuning", rc)

    def metrics(self):
        n1, n2, n3 = self.n
        vol = np.empty((n3, n2, n1))
        a1 = np.empty((n3, n2, n1 + 1))
        a2 = np.empty((n3, n2 + 1, n1))
        a3 = np.empty((n3 + 1, n2, n1))
        rc = lib().rt_grid_get_metrics(self._h, *[a.ctypes.data_as(_dp) for a in (vol, a1, a2, a3)])
        if rc != OK:
            self._raise("rt_grid_get_metrics", rc)
        return vol, a1, a2, a3

    def fill_ghosts(self, U):
        for q, t in enumerate(U):
            _check_field(t, self.shape, "U[%d]" % q, self.device)
        rc = lib().rt_fill_ghosts(self._h, _ptr_array(U))
        if rc != OK:
            self._raise("rt_fill_ghosts", rc)

    def explicit_step(self, dt, rho, T, U_in, U_out):
        for name, t in (("rho", rho), ("T", T)):
            if t is not None:
                _check_field(t, self.shape, name, self.device)
        for q in range(4):
            _check_field(U_in[q], self.shape, "U_in[%d]" % q, self.device)
            _check_field(U_out[q], self.shape, "U_out[%d]" % q, self.device)
        rc = lib().rt_explicit_step(self._h, float(dt), rho.data_ptr() if rho is not None else None,
                                    T.data_ptr() if T is not None else None, _ptr_array(U_in), _ptr_array(U_out))
        if rc != OK:
            self._raise("rt_explicit_step", rc)

    def implicit_step(self, dt, rho, T, mom, U):
        _check_field(rho, self.shape, "rho", self.device)
        _check_field(T, self.shape, "T", self.device)
        for q in range(4):
            _check_field(U[q], self.shape, "U[%d]" % q, self.device)
        if mom is not None:
            for q in range(3):
                _check_field(mom[q], self.shape, "mom[%d]" % q, self.device)
        rc = lib().rt_implicit_step(self._h, float(dt), rho.data_ptr(), T.data_ptr(),
                                    _ptr_array(mom) if mom is not None else None, _ptr_array(U))
        if rc != OK:
            self._raise("rt_implicit_step", rc)

    def implicit_step_cfl(self, dt, rho, T, mom, U, cfl, dt_next_device):
        _check_field(rho, self.shape, "rho", self.device)
        _check_field(T, self.shape, "T", self.device)
        for q in range(4):
            _check_field(U[q], self.shape, "U[%d]" % q, self.device)
        if mom is not None:
            for q in range(3):
                _check_field(mom[q], self.shape, "mom[%d]" % q, self.device)
        self._check_dt_device(dt_next_device)
        rc = lib().rt_implicit_step_cfl(self._h, float(dt), rho.data_ptr(), T.data_ptr(),
                                        _ptr_array(mom) if mom is not None else None, _ptr_array(U), float(cfl),
                                        dt_next_device.data_ptr())
        if rc != OK:
            self._raise("rt_implicit_step_cfl", rc)

    def substep(self, dt_device, cfl, rho, T, mom, U_in, U_out):
        _check_field(rho, self.shape, "rho", self.device)
        _check_field(T, self.shape, "T", self.device)
        for q in range(4):
            _check_field(U_in[q], self.shape, "U_in[%d]" % q, self.device)
            _check_field(U_out[q], self.shape, "U_out[%d]" % q, self.device)
        if mom is not None:
            for q in range(3):
                _check_field(mom[q], self.shape, "mom[%d]" % q, self.device)
        self._check_dt_device(dt_device)
        rc = lib().rt_substep(self._h, dt_device.data_ptr(), float(cfl), rho.data_ptr(), T.data_ptr(),
                              _ptr_array(mom) if mom is not None else None, _ptr_array(U_in), _ptr_array(U_out))
        if rc != OK:
            self._raise("rt_substep", rc)

    def set_reconstruction(self, kind, r=0.0):
        rc = lib().rt_set_reconstruction(self._h, int(kind), float(r))
        if rc != OK:
            self._raise("rt_set_reconstruction", rc)

    def set_face_fix(self, mode):
        rc = lib().rt_set_face_fix(self._h, int(mode))
        if rc != OK:
            self._raise("rt_set_face_fix", rc)

    def irradiation_radial(self, L0, kappa_irr, tau_in, rho, tau_hi, div_firr):
        _check_field(rho, self.shape, "rho", self.device)
        _check_field(div_firr, self.shape, "div_firr", self.device)
        if tau_hi is not None:
            _check_field(tau_hi, self.shape, "tau_hi", self.device)
        rc = lib().rt_irradiation_radial(self._h, float(L0), float(kappa_irr), float(tau_in), rho.data_ptr(),
                                         tau_hi.data_ptr() if tau_hi is not None else None, div_firr.data_ptr())
        if rc != OK:
            self._raise("rt_irradiation_radial", rc)

    def set_irradiation(self, div_firr):
        """div F_irr per cell (CUDA float64 tensor in the field layout, kept alive by this object) or None"""
        if div_firr is not None:
            _check_field(div_firr, self.shape, "div_firr", self.device)
        self._div_firr = div_firr
        rc = lib().rt_set_irradiation(self._h, div_firr.data_ptr() if div_firr is not None else None)
        if rc != OK:
            self._raise("rt_set_irradiation", rc)

    def rk2_step(self, dt_device, cfl, rho, T, mom, U, W1, W2):
        _check_field(rho, self.shape, "rho", self.device)
        _check_field(T, self.shape, "T", self.device)
        for q in range(4):
            _check_field(U[q], self.shape, "U[%d]" % q, self.device)
            _check_field(W1[q], self.shape, "W1[%d]" % q, self.device)
            _check_field(W2[q], self.shape, "W2[%d]" % q, self.device)
        if mom is not None:
            for q in range(3):
                _check_field(mom[q], self.shape, "mom[%d]" % q, self.device)
        self._check_dt_device(dt_device)
        rc = lib().rt_rk2_step(self._h, dt_device.data_ptr(), float(cfl), rho.data_ptr(), T.data_ptr(),
                               _ptr_array(mom) if mom is not None else None, _ptr_array(U), _ptr_array(W1), _ptr_array(W2))
        if rc != OK:
            self._raise("rt_rk2_step", rc)

    @staticmethod
    def _check_dt_device(t):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.numel() >= 1):
            raise ValueError("dt_device must be a CUDA float64 tensor")

    def cfl_dt(self, U, cfl):
        for q in range(4):
            _check_field(U[q], self.shape, "U[%d]" % q, self.device)
        out = C.c_double()
        rc = lib().rt_cfl_dt(self._h, _ptr_array(U), float(cfl), C.byref(out))
        if rc != OK:
            self._raise("rt_cfl_dt", rc)
        return out.value

    def cfl_dt_async(self, U, cfl, dt_device):
        for q in range(4):
            _check_field(U[q], self.shape, "U[%d]" % q, self.device)
        if not (dt_device.is_cuda and dt_device.dtype == torch.float64 and dt_device.numel() >= 1):
            raise ValueError("dt_device must be a CUDA float64 tensor")
        rc = lib().rt_cfl_dt_async(self._h, _ptr_array(U), float(cfl), dt_device.data_ptr())
        if rc != OK:
            self._raise("rt_cfl_dt_async", rc)

    def floor_counts(self):
        a, b = C.c_int64(), C.c_int64()
        rc = lib().rt_get_floor_counts(self._h, C.byref(a), C.byref(b))
        if rc != OK:
            self._raise("rt_get_floor_counts", rc)
        return a.value, b.value

    def check_finite(self, U, T=None):
        """rt_check_finite: number of interior cells holding a NaN / inf (raises RtError with status ERR_NOT_FINITE if any)"""
        for q in range(4):
            _check_field(U[q], self.shape, "U[%d]" % q, self.device)
        if T is not None:
            _check_field(T, self.shape, "T", self.device)
        n = C.c_int64()
        rc = lib().rt_check_finite(self._h, _ptr_array(U), T.data_ptr() if T is not None else None, C.byref(n))
        if rc != OK:
            self._raise("rt_check_finite", rc)
        return n.value

    def set_profiling(self, on):
        rc = lib().rt_set_profiling(self._h, 1 if on else 0)
        if rc != OK:
            self._raise("rt_set_profiling", rc)

    def kernel_times(self):
        """{kind name: (summed ms, launches)} since the last call (needs set_profiling(True))"""
        ms = (C.c_double * NKERNEL_KINDS)()
        cnt = (C.c_int64 * NKERNEL_KINDS)()
        rc = lib().rt_get_kernel_times(self._h, ms, cnt)
        if rc != OK:
            self._raise("rt_get_kernel_times", rc)
        return {name: (ms[k], cnt[k]) for k, name in enumerate(KERNEL_KINDS)}

    def launch_count(self):
        return int(lib().rt_get_launch_count(self._h))

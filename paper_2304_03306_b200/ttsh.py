"""Thin ctypes binding of include/ttsh.h (argument marshalling only; every step of the path runs in the
CUDA kernels of csrc/).  PyTorch is used for device memory and streams, nothing else.

The functions ``ttsh_*`` mirror the C ABI one to one (device pointers are passed as integers, e.g.
``tensor.data_ptr()``).  ``Solver`` is a small convenience wrapper that owns the torch tensors.
There is no CPU fallback: if ``csrc/libttsh.so`` is missing, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("TTSH_LIB_PATH") or os.path.join(_HERE, "csrc", "libttsh.so")   # override: an out-of-tree build

TTSH_OK = 0
TTSH_ERR_INVALID_ARG = -1
TTSH_ERR_UNSUPPORTED_SIZE = -2
TTSH_ERR_WORKSPACE_TOO_SMALL = -3
TTSH_ERR_NOT_INITIALIZED = -4
TTSH_ERR_CUDA = -5
TTSH_F64, TTSH_F32 = 8, 4
TTSH_MASK_BINARY, TTSH_MASK_PROCESSED = 0, 1
TTSH_ADVECTION_CONSERVATIVE, TTSH_ADVECTION_LITERAL = 0, 1
(TTSH_STAGE_INV_COL, TTSH_STAGE_INV_ROW, TTSH_STAGE_REAL, TTSH_STAGE_FWD_ROW, TTSH_STAGE_FWD_COL,
 TTSH_STAGE_SPECTRAL, TTSH_STAGE_REAL_FWD_ROW, TTSH_STAGE_FWD_COL_P2, TTSH_STAGE_SPECTRAL_P2, TTSH_STAGE_ROW_STEP,
 TTSH_STAGE_COL_STEP) = range(11)

# every symbol include/ttsh.h declares (tests check that the library exports all of them)
SYMBOLS = ("ttsh_workspace_bytes", "ttsh_create", "ttsh_set_mask", "ttsh_set_velocity", "ttsh_set_advection_form", "ttsh_step",
           "ttsh_get_fields", "ttsh_state_elems", "ttsh_get_state", "ttsh_set_state", "ttsh_diagnostics",
           "ttsh_launch_count", "ttsh_run_stage", "ttsh_debug_get_real", "ttsh_destroy", "ttsh_strerror",
           "ttsh_last_error", "ttsh_dumbbell_order", "ttsh_psd_workspace_bytes", "ttsh_psd_create",
           "ttsh_psd_accumulate", "ttsh_psd_result", "ttsh_psd_reset", "ttsh_psd_destroy", "ttsh_tangent_workspace_bytes",
           "ttsh_tangent_create", "ttsh_tangent_set", "ttsh_tangent_step", "ttsh_tangent_orthonormalize",
           "ttsh_tangent_get_fields", "ttsh_tangent_destroy", "ttsh_ensemble_create", "ttsh_ensemble_step", "ttsh_ensemble_launch_count",
           "ttsh_ensemble_destroy", "ttsh_build_info", "ttsh_diagnostics_noalloc", "ttsh_diagnostics_noalloc_error",
           "ttsh_microbench_fma")
TTSH_NOALLOC_MAX_POINTS = 16384 * 16384


class ttsh_params(C.Structure):
    _fields_ = [("lambda0", C.c_double), ("alpha", C.c_double), ("beta", C.c_double), ("Gamma0", C.c_double),
                ("Gamma2", C.c_double), ("gamma_v", C.c_double), ("gamma_w", C.c_double),
                ("dealias_num", C.c_int), ("dealias_den", C.c_int)]


class ttsh_diag(C.Structure):
    _fields_ = [("t", C.c_double), ("step", C.c_longlong), ("kinetic_energy", C.c_double), ("enstrophy", C.c_double),
                ("vortex_order", C.c_double), ("polar_order", C.c_double), ("sum_speed", C.c_double),
                ("sum_abs_vtheta", C.c_double), ("mean_vx", C.c_double), ("mean_vy", C.c_double),
                ("max_speed", C.c_double), ("nonfinite", C.c_longlong)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
                      "(nvcc, sm_100a).  There is no CPU fallback.")
_lib = C.CDLL(LIB_PATH)

_vp, _i, _d, _sz, _ll = C.c_void_p, C.c_int, C.c_double, C.c_size_t, C.c_longlong
_sig = {
    "ttsh_workspace_bytes": (_sz, [_i, _i, _i]),
    "ttsh_create": (_i, [C.POINTER(_vp), _i, _i, _d, _d, C.POINTER(ttsh_params), _i, _vp, _i, _vp, _sz, _vp]),
    "ttsh_set_mask": (_i, [_vp, _vp, _i]),
    "ttsh_set_velocity": (_i, [_vp, _vp, _vp]),
    "ttsh_set_advection_form": (_i, [_vp, _i]),
    "ttsh_step": (_i, [_vp, _i]),
    "ttsh_get_fields": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "ttsh_state_elems": (_sz, [_vp]),
    "ttsh_get_state": (_i, [_vp, _vp, C.POINTER(_d)]),
    "ttsh_set_state": (_i, [_vp, _vp, C.POINTER(_d), _d, _ll]),
    "ttsh_diagnostics": (_i, [_vp, _d, _d, C.POINTER(ttsh_diag)]),
    "ttsh_launch_count": (_ll, [_vp]),
    "ttsh_run_stage": (_i, [_vp, _i]),
    "ttsh_debug_get_real": (_i, [_vp, _i, _vp]),
    "ttsh_destroy": (_i, [_vp]),
    "ttsh_strerror": (C.c_char_p, [_i]),
    "ttsh_last_error": (C.c_char_p, [_vp]),
    "ttsh_dumbbell_order": (_i, [_vp, _d, _d, _d, _d, _d, _vp]),
    "ttsh_psd_workspace_bytes": (_sz, [_i, _i, _i, _i]),
    "ttsh_psd_create": (_i, [C.POINTER(_vp), _vp, C.POINTER(_d), _i, _vp, _sz]),
    "ttsh_psd_accumulate": (_i, [_vp]),
    "ttsh_psd_result": (_i, [_vp, C.POINTER(_d), C.POINTER(_ll)]),
    "ttsh_psd_reset": (_i, [_vp]),
    "ttsh_psd_destroy": (_i, [_vp]),
    "ttsh_tangent_workspace_bytes": (_sz, [_i, _i, _i, _i]),
    "ttsh_tangent_create": (_i, [C.POINTER(_vp), _vp, _i, _vp, _sz]),
    "ttsh_tangent_set": (_i, [_vp, _i, _vp, _vp]),
    "ttsh_tangent_step": (_i, [_vp, _i]),
    "ttsh_tangent_orthonormalize": (_i, [_vp, C.POINTER(_d)]),
    "ttsh_tangent_get_fields": (_i, [_vp, _i, _vp, _vp, _vp]),
    "ttsh_tangent_destroy": (_i, [_vp]),
    "ttsh_ensemble_create": (_i, [C.POINTER(_vp), C.POINTER(_vp), _i]),
    "ttsh_ensemble_step": (_i, [_vp, _i]),
    "ttsh_ensemble_launch_count": (_ll, [_vp]),
    "ttsh_ensemble_destroy": (_i, [_vp]),
    "ttsh_build_info": (C.c_char_p, []),
    "ttsh_diagnostics_noalloc": (_i, [_i, _i, _d, _i, _vp, _vp, _vp, _d, _d, _vp, C.POINTER(ttsh_diag), _vp]),
    "ttsh_diagnostics_noalloc_error": (C.c_char_p, []),
    "ttsh_microbench_fma": (_i, [_i, _i, _i, _d, _d, _vp, _vp, C.POINTER(_d)]),
}
for _name, (_res, _args) in _sig.items():
    _f = getattr(_lib, _name)
    _f.restype, _f.argtypes = _res, _args


class ttsh_psi2(C.Structure):
    _fields_ = [("psi2", C.c_double), ("omega_left", C.c_double), ("omega_right", C.c_double),
                ("index_left", C.c_longlong), ("index_right", C.c_longlong)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class TTSHError(RuntimeError):
    def __init__(self, code: int, detail: str = ""):
        self.code = code
        msg = _lib.ttsh_strerror(code).decode()
        super().__init__(f"ttsh error {code}: {msg}" + (f" ({detail})" if detail else ""))


# ---- the C ABI, one to one ------------------------------------------------------------------
def ttsh_workspace_bytes(Nx: int, Ny: int, dtype: int) -> int:
    return int(_lib.ttsh_workspace_bytes(Nx, Ny, dtype))


def ttsh_create(Nx, Ny, dx, dt, params: ttsh_params, dtype, mask_ptr, mask_kind, workspace_ptr, workspace_bytes,
                stream_ptr):
    """Returns (status, handle).  Pointers are integers (0 / None = NULL)."""
    h = _vp()
    rc = _lib.ttsh_create(C.byref(h), Nx, Ny, dx, dt, C.byref(params), dtype, mask_ptr or None, mask_kind,
                          workspace_ptr or None, workspace_bytes, stream_ptr or None)
    return rc, h


def ttsh_set_mask(h, mask_ptr, mask_kind):
    return _lib.ttsh_set_mask(h, mask_ptr or None, mask_kind)


def ttsh_set_velocity(h, vx_ptr, vy_ptr):
    return _lib.ttsh_set_velocity(h, vx_ptr or None, vy_ptr or None)


def ttsh_set_advection_form(h, form):
    return _lib.ttsh_set_advection_form(h, form)


def ttsh_step(h, n):
    return _lib.ttsh_step(h, n)


def ttsh_get_fields(h, vx_ptr=None, vy_ptr=None, omega_ptr=None, psi_ptr=None):
    return _lib.ttsh_get_fields(h, vx_ptr or None, vy_ptr or None, omega_ptr or None, psi_ptr or None)


def ttsh_state_elems(h):
    return int(_lib.ttsh_state_elems(h))


def ttsh_get_state(h, w_hat_ptr):
    mf = (_d * 2)()
    rc = _lib.ttsh_get_state(h, w_hat_ptr or None, mf)
    return rc, (mf[0], mf[1])


def ttsh_set_state(h, w_hat_ptr, mean_flow, t, step):
    mf = (_d * 2)(float(mean_flow[0]), float(mean_flow[1]))
    return _lib.ttsh_set_state(h, w_hat_ptr or None, mf, t, step)


def ttsh_diagnostics(h, cx, cy):
    d = ttsh_diag()
    rc = _lib.ttsh_diagnostics(h, cx, cy, C.byref(d))
    return rc, d


def ttsh_diagnostics_noalloc(Nx, Ny, dx, dtype, vx_ptr, vy_ptr, omega_ptr, cx, cy, sums_ptr, stream_ptr, read_back=True):
    """Diagnostics of three caller-owned DEVICE fields without a handle or workspace, for callers that cannot allocate device
    memory (see include/ttsh.h): the library's scratch is a static array on the GPU, shared by all calls on that device, so
    calls must not overlap on the GPU.  sums_ptr: DEVICE double[8] out.  Returns (status, ttsh_diag or None); with
    read_back=False nothing is copied to the host and the call is asynchronous."""
    d = ttsh_diag() if read_back else None
    rc = _lib.ttsh_diagnostics_noalloc(Nx, Ny, dx, dtype, vx_ptr, vy_ptr, omega_ptr, cx, cy, sums_ptr,
                                       C.byref(d) if read_back else None, stream_ptr)
    return rc, d


def ttsh_diagnostics_noalloc_error():
    return _lib.ttsh_diagnostics_noalloc_error().decode()


def ttsh_microbench_fma(dtype, blocks, rounds, a, b, sink_ptr, stream_ptr):
    """One launch of the dense FMA loop (include/ttsh.h); returns (status, flops of the launch)."""
    fl = _d(0.0)
    rc = _lib.ttsh_microbench_fma(dtype, blocks, rounds, a, b, sink_ptr, stream_ptr, C.byref(fl))
    return rc, fl.value


def ttsh_dumbbell_order(h, cx_left, cy_left, cx_right, cy_right, radius):
    d = ttsh_psi2()
    rc = _lib.ttsh_dumbbell_order(h, cx_left, cy_left, cx_right, cy_right, radius, C.byref(d))
    return rc, d


def ttsh_psd_workspace_bytes(Nx, Ny, dtype, nfreq):
    return int(_lib.ttsh_psd_workspace_bytes(Nx, Ny, dtype, nfreq))


def ttsh_psd_create(h, omegas, workspace_ptr, workspace_bytes):
    """Returns (status, psd handle).  omegas: sequence of angular frequencies (host)."""
    s = _vp()
    arr = (_d * max(1, len(omegas)))(*[float(o) for o in omegas])
    rc = _lib.ttsh_psd_create(C.byref(s), h, arr, len(omegas), workspace_ptr or None, workspace_bytes)
    return rc, s


def ttsh_psd_accumulate(s):
    return _lib.ttsh_psd_accumulate(s)


def ttsh_psd_result(s, nfreq):
    out = (_d * max(1, nfreq))()
    n = _ll(0)
    rc = _lib.ttsh_psd_result(s, out, C.byref(n))
    return rc, [out[i] for i in range(nfreq)], int(n.value)


def ttsh_psd_reset(s):
    return _lib.ttsh_psd_reset(s)


def ttsh_psd_destroy(s):
    return _lib.ttsh_psd_destroy(s)


def ttsh_tangent_workspace_bytes(Nx, Ny, dtype, nvec):
    return int(_lib.ttsh_tangent_workspace_bytes(Nx, Ny, dtype, nvec))


def ttsh_tangent_create(h, nvec, workspace_ptr, workspace_bytes):
    s = _vp()
    rc = _lib.ttsh_tangent_create(C.byref(s), h, nvec, workspace_ptr or None, workspace_bytes)
    return rc, s


def ttsh_tangent_set(s, i, dvx_ptr, dvy_ptr):
    return _lib.ttsh_tangent_set(s, i, dvx_ptr or None, dvy_ptr or None)


def ttsh_tangent_step(s, n):
    return _lib.ttsh_tangent_step(s, n)


def ttsh_tangent_orthonormalize(s, nvec):
    out = (_d * max(1, nvec))()
    rc = _lib.ttsh_tangent_orthonormalize(s, out)
    return rc, [out[i] for i in range(nvec)]


def ttsh_tangent_get_fields(s, i, dvx_ptr=None, dvy_ptr=None, domega_ptr=None):
    return _lib.ttsh_tangent_get_fields(s, i, dvx_ptr or None, dvy_ptr or None, domega_ptr or None)


def ttsh_tangent_destroy(s):
    return _lib.ttsh_tangent_destroy(s)


def ttsh_launch_count(h):
    return int(_lib.ttsh_launch_count(h))


def ttsh_run_stage(h, stage):
    return _lib.ttsh_run_stage(h, stage)


def ttsh_debug_get_real(h, which, dst_ptr):
    return _lib.ttsh_debug_get_real(h, which, dst_ptr or None)


def ttsh_destroy(h):
    return _lib.ttsh_destroy(h)


def ttsh_ensemble_create(handles):
    """Returns (status, ensemble).  handles: sequence of member handles (c_void_p or int; None = NULL)."""
    e = _vp()
    arr = (_vp * max(1, len(handles)))(*[getattr(h, "value", h) for h in handles])
    rc = _lib.ttsh_ensemble_create(C.byref(e), arr, len(handles))
    return rc, e


def ttsh_ensemble_step(e, n):
    return _lib.ttsh_ensemble_step(e, n)


def ttsh_ensemble_launch_count(e):
    return int(_lib.ttsh_ensemble_launch_count(e))


def ttsh_ensemble_destroy(e):
    return _lib.ttsh_ensemble_destroy(e)


def ttsh_build_info():
    return _lib.ttsh_build_info().decode()


def ttsh_strerror(code):
    return _lib.ttsh_strerror(code).decode()


def ttsh_last_error(h):
    return _lib.ttsh_last_error(h).decode()


# ---- presets ----------------------------------------------------------------------------------
def paper_params() -> ttsh_params:
    """(a, b, lambda, gamma_v, gamma_w) = (0.5, 1.6, 9, 40, 4); alpha = 1-a, Gamma0 = -2, Gamma2 = 1."""
    return ttsh_params(9.0, 0.5, 1.6, -2.0, 1.0, 40.0, 4.0, 1, 2)


def baseline_params() -> ttsh_params:
    """BASELINE.json configs: lambda0=3.5, alpha=-0.5, beta=0.5, Gamma0=-1, Gamma2=1 (+ the paper's gammas)."""
    return ttsh_params(3.5, -0.5, 0.5, -1.0, 1.0, 40.0, 4.0, 1, 2)


# ---- convenience wrapper (owns torch tensors; marshalling only) --------------------------------------
class Solver:
    def __init__(self, Nx: int, Ny: int, dx: float, dt: float, params: ttsh_params, dtype: str = "f64",
                 mask=None, mask_kind: int = TTSH_MASK_BINARY, device: str = "cuda:0", stream=None, workspace=None):
        """workspace: an optional uint8 CUDA tensor (>= ttsh_workspace_bytes, 256-byte aligned) to use instead of a fresh one
        (Ensemble carves its members' workspaces from one allocation)."""
        import torch
        self.torch = torch
        self.Nx, self.Ny, self.dx, self.dt = Nx, Ny, dx, dt
        self.dtype_code = {"f64": TTSH_F64, "f32": TTSH_F32}[dtype]
        self.tdtype = torch.float64 if dtype == "f64" else torch.float32
        self.device = torch.device(device)
        self._dependants = []     # TemporalPSD / Tangent / Ensemble objects that borrow the handle: closed before it
        nbytes = ttsh_workspace_bytes(Nx, Ny, self.dtype_code)
        if nbytes == 0:
            raise TTSHError(TTSH_ERR_UNSUPPORTED_SIZE)
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        with self._ctx():
            self.workspace = workspace if workspace is not None else torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            nbytes = self.workspace.numel()
            mptr = 0
            if mask is not None:
                want = torch.uint8 if mask_kind == TTSH_MASK_BINARY else self.tdtype
                self._mask = torch.as_tensor(mask).to(device=self.device, dtype=want).contiguous()
                mptr = self._mask.data_ptr()
            rc, self.h = ttsh_create(Nx, Ny, dx, dt, params, self.dtype_code, mptr, mask_kind,
                                     self.workspace.data_ptr(), nbytes, self.stream.cuda_stream)
        if rc != TTSH_OK:
            detail = ttsh_last_error(self.h) if self.h else ""
            if self.h:
                ttsh_destroy(self.h)
                self.h = None
            raise TTSHError(rc, detail)

    def _check(self, rc):
        if rc != TTSH_OK:
            raise TTSHError(rc, ttsh_last_error(self.h))

    def _ctx(self):
        """The handle's device and stream made current: the library enqueues on self.stream, and every tensor this wrapper
        allocates or copies must be ordered on that same stream (torch's caching allocator reuses memory per stream)."""
        import contextlib
        st = contextlib.ExitStack()
        st.enter_context(self.torch.cuda.device(self.device))
        st.enter_context(self.torch.cuda.stream(self.stream))
        return st

    def _dev(self, a):
        with self._ctx():
            return self.torch.as_tensor(a).to(device=self.device, dtype=self.tdtype).contiguous()

    def set_mask(self, mask, mask_kind=TTSH_MASK_BINARY):
        with self._ctx():
            if mask is None:
                self._check(ttsh_set_mask(self.h, 0, mask_kind))
                return
            want = self.torch.uint8 if mask_kind == TTSH_MASK_BINARY else self.tdtype
            self._mask = self.torch.as_tensor(mask).to(device=self.device, dtype=want).contiguous()
            self._check(ttsh_set_mask(self.h, self._mask.data_ptr(), mask_kind))

    def set_velocity(self, vx, vy):
        with self._ctx():
            self._vx0, self._vy0 = self._dev(vx), self._dev(vy)
            self._check(ttsh_set_velocity(self.h, self._vx0.data_ptr(), self._vy0.data_ptr()))

    def set_advection_form(self, form: int):
        with self._ctx():
            self._check(ttsh_set_advection_form(self.h, form))

    def step(self, n: int = 1):
        with self._ctx():
            self._check(ttsh_step(self.h, n))

    def new_field(self):
        with self._ctx():
            return self.torch.empty((self.Ny, self.Nx), dtype=self.tdtype, device=self.device)

    def get_fields(self, psi: bool = True):
        with self._ctx():
            vx, vy, w = self.new_field(), self.new_field(), self.new_field()
            ps = self.new_field() if psi else None
            self._check(ttsh_get_fields(self.h, vx.data_ptr(), vy.data_ptr(), w.data_ptr(), ps.data_ptr() if psi else 0))
        return vx, vy, w, ps

    def diagnostics(self, cx: Optional[float] = None, cy: Optional[float] = None) -> dict:
        cx = (self.Nx // 2) * self.dx if cx is None else cx
        cy = (self.Ny // 2) * self.dx if cy is None else cy
        with self._ctx():
            rc, d = ttsh_diagnostics(self.h, cx, cy)
        self._check(rc)
        return d.as_dict()

    def dumbbell_order(self, centre_left, centre_right, radius: float) -> dict:
        with self._ctx():
            rc, d = ttsh_dumbbell_order(self.h, centre_left[0], centre_left[1], centre_right[0], centre_right[1], radius)
        self._check(rc)
        return d.as_dict()

    def run_stage(self, stage: int):
        with self._ctx():
            self._check(ttsh_run_stage(self.h, stage))

    def debug_real(self, which: int):
        with self._ctx():
            out = self.new_field()
            self._check(ttsh_debug_get_real(self.h, which, out.data_ptr()))
        return out

    def launch_count(self) -> int:
        return ttsh_launch_count(self.h)

    def close(self):
        """Closes the objects that borrow the handle (TemporalPSD, Tangent, Ensemble) first, then the handle."""
        for d in list(getattr(self, "_dependants", [])):
            d.close()
        if getattr(self, "h", None):
            self.torch.cuda.synchronize(self.device)
            ttsh_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class TemporalPSD:
    """Streaming Eq. (5) on a Solver: accumulate() after every sampling interval, result() -> S(Omega_m)."""

    def __init__(self, solver: Solver, omegas):
        self.solver, self.omegas = solver, [float(o) for o in omegas]
        torch = solver.torch
        nbytes = ttsh_psd_workspace_bytes(solver.Nx, solver.Ny, solver.dtype_code, len(self.omegas))
        if nbytes == 0:
            raise TTSHError(TTSH_ERR_INVALID_ARG, "1 <= nfreq <= 1024")
        with torch.cuda.device(solver.device), torch.cuda.stream(solver.stream):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=solver.device)
            rc, self.s = ttsh_psd_create(solver.h, self.omegas, self.workspace.data_ptr(), nbytes)
        if rc != TTSH_OK:
            raise TTSHError(rc)
        solver._dependants.append(self)

    def accumulate(self):
        with self.solver._ctx():
            self.solver._check(ttsh_psd_accumulate(self.s))

    def result(self):
        with self.solver._ctx():
            rc, S, n = ttsh_psd_result(self.s, len(self.omegas))
        self.solver._check(rc)
        return S, n

    def reset(self):
        with self.solver._ctx():
            self.solver._check(ttsh_psd_reset(self.s))

    def close(self):
        if getattr(self, "s", None):
            self.solver.torch.cuda.synchronize(self.solver.device)
            ttsh_psd_destroy(self.s)
            self.s = None
            if self in self.solver._dependants:
                self.solver._dependants.remove(self)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Tangent:
    """nvec perturbations carried along a Solver's trajectory by the Jacobian of Algorithm 1, with QR re-orthonormalisation
    (Lyapunov exponents): lambda_i = sum of orthonormalize()[i] over the run / elapsed time."""

    def __init__(self, solver: Solver, nvec: int):
        self.solver, self.nvec = solver, int(nvec)
        torch = solver.torch
        nbytes = ttsh_tangent_workspace_bytes(solver.Nx, solver.Ny, solver.dtype_code, self.nvec)
        if nbytes == 0:
            raise TTSHError(TTSH_ERR_INVALID_ARG, "1 <= nvec <= 64")
        with torch.cuda.device(solver.device), torch.cuda.stream(solver.stream):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=solver.device)
            rc, self.s = ttsh_tangent_create(solver.h, self.nvec, self.workspace.data_ptr(), nbytes)
        if rc != TTSH_OK:
            raise TTSHError(rc)
        solver._dependants.append(self)

    def set(self, i: int, dvx, dvy):
        with self.solver._ctx():
            a, b = self.solver._dev(dvx), self.solver._dev(dvy)
            self._keep = (a, b)
            self.solver._check(ttsh_tangent_set(self.s, i, a.data_ptr(), b.data_ptr()))

    def step(self, n: int = 1):
        with self.solver._ctx():
            self.solver._check(ttsh_tangent_step(self.s, n))

    def orthonormalize(self):
        with self.solver._ctx():
            rc, logr = ttsh_tangent_orthonormalize(self.s, self.nvec)
        self.solver._check(rc)
        return logr

    def get_fields(self, i: int):
        s = self.solver
        with s._ctx():
            dvx, dvy, dw = s.new_field(), s.new_field(), s.new_field()
            s._check(ttsh_tangent_get_fields(self.s, i, dvx.data_ptr(), dvy.data_ptr(), dw.data_ptr()))
        return dvx, dvy, dw

    def close(self):
        if getattr(self, "s", None):
            self.solver.torch.cuda.synchronize(self.solver.device)
            ttsh_tangent_destroy(self.s)
            self.s = None
            if self in self.solver._dependants:
                self.solver._dependants.remove(self)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Ensemble:
    """`count` independent systems on one grid (different masks / initial fields, same parameters) advanced together by
    ttsh_ensemble_step: one launch of each hot kernel per Euler step for all members.  members[i] is an ordinary Solver."""

    def __init__(self, count: int, Nx: int, Ny: int, dx: float, dt: float, params: ttsh_params, dtype: str = "f64",
                 masks=None, mask_kind: int = TTSH_MASK_BINARY, device: str = "cuda:0", stream=None):
        import torch
        self.torch = torch
        self.device = torch.device(device)
        code = {"f64": TTSH_F64, "f32": TTSH_F32}[dtype]
        nbytes = ttsh_workspace_bytes(Nx, Ny, code)
        if nbytes == 0:
            raise TTSHError(TTSH_ERR_UNSUPPORTED_SIZE)
        stride = (nbytes + 255) // 256 * 256
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.workspace = torch.empty(stride * count, dtype=torch.uint8, device=self.device)
        self.members = [Solver(Nx, Ny, dx, dt, params, dtype, mask=None if masks is None else masks[i], mask_kind=mask_kind,
                               device=device, stream=self.stream, workspace=self.workspace[i * stride:(i + 1) * stride])
                        for i in range(count)]
        rc, self.e = ttsh_ensemble_create([m.h for m in self.members])
        if rc != TTSH_OK:
            raise TTSHError(rc)
        for m in self.members:
            m._dependants.append(self)      # closing a member closes the ensemble first

    def step(self, n: int = 1):
        with self.members[0]._ctx():
            rc = ttsh_ensemble_step(self.e, n)
        if rc != TTSH_OK:
            raise TTSHError(rc, ttsh_last_error(self.members[0].h))

    def launch_count(self) -> int:
        return ttsh_ensemble_launch_count(self.e)

    def close(self):
        if getattr(self, "e", None):
            self.torch.cuda.synchronize(self.device)
            ttsh_ensemble_destroy(self.e)
            self.e = None
            for m in self.members:
                if self in m._dependants:
                    m._dependants.remove(self)
        for m in getattr(self, "members", []):
            m.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

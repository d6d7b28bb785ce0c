"""ctypes binding of oracle/ttsh_oracle_c.c — the "oracle-fft" restatement of the CPU oracle in plain C (TEST INFRASTRUCTURE).

``TTSHOracleC`` has the interface of ``TTSHOracle`` (set_velocity / step / get_fields / diagnostics / K) so that the parity
tests can use either.  It is used where the definition-oracle's O(N^3) transforms are prohibitive: the 100-step bound at
4096 x 4096 (BASELINE.json:north_star), the 8192 x 8192 grid of the paper, and as the honest CPU timing baseline
of bench.py (the counterpart of the CPU curve of Fig. 9).  It is locked to the definition-oracle by
tests/test_oracle_c.py.  The library is built with gcc on first use (``build()``; __graft_entry__.build() calls it too).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

from .ttsh_oracle import TTSHParams

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "ttsh_oracle_c.c")
LIB = os.path.join(_HERE, "build", "libcpuoracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -ffp-contract=off -shared -> oracle/build/libcpuoracle.so (rebuilt when the source is newer)."""
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        os.makedirs(os.path.dirname(LIB), exist_ok=True)
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", SRC, "-o", LIB, "-lm"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("oracle build failed:\n" + r.stdout + r.stderr)
    return LIB


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        vp, i, d = C.c_void_p, C.c_int, C.c_double
        lib.ttsho_create.restype, lib.ttsho_create.argtypes = vp, [i, i, d, d, vp, i, i, vp]
        lib.ttsho_destroy.restype, lib.ttsho_destroy.argtypes = None, [vp]
        lib.ttsho_get_K.restype, lib.ttsho_get_K.argtypes = None, [vp, vp]
        lib.ttsho_set_K.restype, lib.ttsho_set_K.argtypes = None, [vp, vp]
        lib.ttsho_set_velocity.restype, lib.ttsho_set_velocity.argtypes = None, [vp, vp, vp]
        lib.ttsho_step.restype, lib.ttsho_step.argtypes = None, [vp, i]
        lib.ttsho_get_fields.restype, lib.ttsho_get_fields.argtypes = None, [vp, vp, vp, vp, vp]
        lib.ttsho_diagnostics.restype, lib.ttsho_diagnostics.argtypes = None, [vp, d, d, vp]
        lib.ttsho_debug_post.restype, lib.ttsho_debug_post.argtypes = None, [vp, vp, vp, vp, vp, vp]
        lib.ttsho_debug_set_state.restype, lib.ttsho_debug_set_state.argtypes = None, [vp, vp, vp, vp]
        lib.ttsho_time.restype, lib.ttsho_time.argtypes = d, [vp]
        lib.ttsho_nstep.restype, lib.ttsho_nstep.argtypes = C.c_longlong, [vp]
        _lib = lib
    return _lib


def threads() -> int:
    """OpenMP threads the library will use (OMP_NUM_THREADS, else the cores of the affinity mask)."""
    n = os.environ.get("OMP_NUM_THREADS")
    return int(n) if n and n.isdigit() else len(os.sched_getaffinity(0))


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


class TTSHOracleC:
    def __init__(self, Nx: int, Ny: int, dx: float, dt: float, params: TTSHParams, mask=None, mask_kind: str = "binary"):
        lib = _load()
        self.Nx, self.Ny, self.dx, self.dt, self.p = int(Nx), int(Ny), float(dx), float(dt), params
        p7 = np.array([params.lambda0, params.alpha, params.beta, params.Gamma0, params.Gamma2, params.gamma_v, params.gamma_w],
                      dtype=np.float64)
        m = None
        if mask is not None and mask_kind == "binary":
            m = np.ascontiguousarray(np.asarray(mask) != 0, dtype=np.uint8)
            assert m.shape == (self.Ny, self.Nx)
        self.h = lib.ttsho_create(self.Nx, self.Ny, self.dx, self.dt, _ptr(p7), params.dealias_num, params.dealias_den,
                                  _ptr(m) if m is not None else None)
        if mask is not None and mask_kind == "processed":
            self.K = mask

    def _field(self):
        return np.empty((self.Ny, self.Nx), dtype=np.float64)

    @property
    def K(self) -> np.ndarray:
        out = self._field()
        _load().ttsho_get_K(self.h, _ptr(out))
        return out

    @K.setter
    def K(self, value):
        a = np.ascontiguousarray(value, dtype=np.float64)
        assert a.shape == (self.Ny, self.Nx)
        _load().ttsho_set_K(self.h, _ptr(a))

    @property
    def t(self) -> float:
        return float(_load().ttsho_time(self.h))

    @property
    def nstep(self) -> int:
        return int(_load().ttsho_nstep(self.h))

    def set_velocity(self, vx0, vy0):
        a = np.ascontiguousarray(vx0, dtype=np.float64); b = np.ascontiguousarray(vy0, dtype=np.float64)
        assert a.shape == (self.Ny, self.Nx) and b.shape == (self.Ny, self.Nx)
        _load().ttsho_set_velocity(self.h, _ptr(a), _ptr(b))

    def step(self, n: int = 1):
        _load().ttsho_step(self.h, int(n))

    def get_fields(self):
        vx, vy, w, psi = self._field(), self._field(), self._field(), self._field()
        _load().ttsho_get_fields(self.h, _ptr(vx), _ptr(vy), _ptr(w), _ptr(psi))
        return vx, vy, w, psi

    def diagnostics(self, cx: float, cy: float) -> dict:
        out = np.empty(10, dtype=np.float64)
        _load().ttsho_diagnostics(self.h, float(cx), float(cy), _ptr(out))
        keys = ("kinetic_energy", "enstrophy", "vortex_order", "polar_order", "sum_speed", "sum_abs_vtheta", "mean_vx", "mean_vy",
                "max_speed")
        d = {k: float(v) for k, v in zip(keys, out[:9])}
        d.update(t=self.t, step=self.nstep, nonfinite=int(out[9]))
        return d

    # ---- test-only (tests/test_oracle_c.py): see ttsho_debug_* in ttsh_oracle_c.c ----
    def debug_post(self, w_naive, v0_new=(0.0, 0.0)):
        """Lines 5-16 of Algorithm 1 on a caller-supplied spectrum complex[Ny, Nx]; returns (w^_new, v^_x, v^_y)."""
        a = np.ascontiguousarray(w_naive, dtype=np.complex128)
        assert a.shape == (self.Ny, self.Nx)
        v0 = np.ascontiguousarray(v0_new, dtype=np.float64)
        out = [np.empty((self.Ny, self.Nx), dtype=np.complex128) for _ in range(3)]
        _load().ttsho_debug_post(self.h, _ptr(a), _ptr(v0), _ptr(out[0]), _ptr(out[1]), _ptr(out[2]))
        return tuple(out)

    def debug_set_state(self, w_hat=None, vx=None, vy=None):
        """Overwrites the raw state arrays (no projection, no dealiasing)."""
        keep = [None if x is None else np.ascontiguousarray(x, dtype=dt) for x, dt in
                ((w_hat, np.complex128), (vx, np.float64), (vy, np.float64))]
        assert all(x is None or x.shape == (self.Ny, self.Nx) for x in keep)
        _load().ttsho_debug_set_state(self.h, *[None if x is None else _ptr(x) for x in keep])

    def close(self):
        if getattr(self, "h", None):
            _load().ttsho_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

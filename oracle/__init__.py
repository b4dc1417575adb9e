"""ctypes front end of the CPU oracle (oracle/tslb_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2401_17074_b200 and the CUDA path imports nothing from here.

The arithmetic lives in tslb_oracle.c (fp64, citations to PAPER.md there); this file only
compiles it with gcc, marshals numpy arrays and mirrors the C-ABI call names with an
``oracle_`` prefix so one harness can drive both sides.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tslb_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_tslb.so")
_lock = threading.Lock()
_lib = None

FIELDS = ("rho", "ux", "uy", "uz", "Pxx", "Pyy", "Pzz", "Pxy", "Pxz", "Pyz")
FACE_XLO, FACE_XHI, FACE_YLO, FACE_YHI, FACE_ZLO, FACE_ZHI = range(6)
BC_PERIODIC, BC_BOUNCE_BACK, BC_VELOCITY_INLET, BC_OUTLET_ZERO_GRADIENT = range(4)
BC_OUTLET_PRESSURE = 5
NOISE_GAUSSIAN = 0x100
MODE_BRUTE, MODE_CLOSED = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no -ffast-math: plain IEEE fp64)."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + ".tmp%d" % os.getpid()
            subprocess.check_call(
                ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
                 "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        lib.oracle_fstar.restype = C.c_double
        lib.oracle_fstar.argtypes = [dp, ip, C.c_double, dp, C.c_int]
        lib.oracle_fstar_order.restype = C.c_double
        lib.oracle_fstar_order.argtypes = [dp, ip, C.c_double, dp, C.c_int, C.c_int]
        lib.oracle_set_order.argtypes = [C.c_void_p, C.c_int]
        lib.oracle_mix64.restype = C.c_uint64
        lib.oracle_mix64.argtypes = [C.c_uint64]
        lib.oracle_noise_r24.restype = C.c_uint32
        lib.oracle_noise_r24.argtypes = [C.c_uint64, C.c_longlong, C.c_longlong]
        lib.oracle_noise_xi.restype = C.c_double
        lib.oracle_noise_xi.argtypes = [C.c_uint64, C.c_longlong, C.c_longlong]
        lib.oracle_noise_gauss.restype = C.c_double
        lib.oracle_noise_gauss.argtypes = [C.c_uint64, C.c_longlong, C.c_longlong]
        lib.oracle_set_pressure_outlet.argtypes = [C.c_void_p, C.c_int, C.c_double]
        lib.oracle_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.POINTER(C.c_void_p)]
        lib.oracle_destroy.argtypes = [C.c_void_p]
        lib.oracle_destroy.restype = None
        lib.oracle_set_moments.argtypes = [C.c_void_p, dp]
        lib.oracle_set_force.argtypes = [C.c_void_p, dp]
        lib.oracle_set_sponge.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double]
        lib.oracle_tau_of_plane.argtypes = [C.c_void_p, C.c_int]
        lib.oracle_tau_of_plane.restype = C.c_double
        lib.oracle_set_face.argtypes = [C.c_void_p, C.c_int, C.c_int, dp, C.c_double, C.c_uint64, C.c_int]
        lib.oracle_step.argtypes = [C.c_void_p, C.c_int, C.c_int]
        lib.oracle_get_moments.argtypes = [C.c_void_p, dp]
        lib.oracle_diagnostics.argtypes = [C.c_void_p, dp]
        lib.oracle_plane_statistics.argtypes = [C.c_void_p, C.c_int, dp]
        lib.oracle_radial_statistics.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_int, dp]
        lib.oracle_step_count.argtypes = [C.c_void_p]
        lib.oracle_step_count.restype = C.c_longlong
        lib.oracle_num_threads.restype = C.c_int
        _lib = lib
    return _lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def fstar(M10, c3, omega: float, g3=(0.0, 0.0, 0.0), mode: int = MODE_CLOSED, order: int = 3) -> float:
    """Post-collision population f*_c(M) of Eq. 18 (order 3) or Eq. 8 (order 2)."""
    M = np.ascontiguousarray(M10, dtype=np.float64)
    c = np.ascontiguousarray(c3, dtype=np.intc)
    g = np.ascontiguousarray(g3, dtype=np.float64)
    assert M.shape == (10,) and c.shape == (3,) and g.shape == (3,)
    return float(_load().oracle_fstar_order(_dptr(M), c.ctypes.data_as(C.POINTER(C.c_int)), omega, _dptr(g), mode, order))


def mix64(z: int) -> int:
    return int(_load().oracle_mix64(C.c_uint64(z & (2**64 - 1))))


def noise_r24(seed: int, t: int, idx: int) -> int:
    return int(_load().oracle_noise_r24(C.c_uint64(seed), t, idx))


def noise_xi(seed: int, t: int, idx: int) -> float:
    return float(_load().oracle_noise_xi(C.c_uint64(seed), t, idx))


def noise_gauss(seed: int, t: int, idx: int) -> float:
    return float(_load().oracle_noise_gauss(C.c_uint64(seed), int(t), int(idx)))


def num_threads() -> int:
    return int(_load().oracle_num_threads())


class Oracle:
    """One lattice + its ping-pong moment buffers on the host (fp64)."""

    def __init__(self, nx: int, ny: int, nz: int, tau: float):
        self._lib = _load()
        self._h = C.c_void_p()
        rc = self._lib.oracle_create(nx, ny, nz, float(tau), C.byref(self._h))
        if rc:
            raise ValueError("oracle_create failed rc=%d" % rc)
        self.shape = (nz, ny, nx)
        self.tau = float(tau)

    def close(self):
        if self._h:
            self._lib.oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc, what):
        if rc:
            raise RuntimeError("%s failed rc=%d" % (what, rc))

    def set_moments(self, M: np.ndarray):
        """M: [10][nz][ny][nx]; any float dtype, converted to fp64 exactly."""
        A = np.ascontiguousarray(M, dtype=np.float64)
        assert A.shape == (10,) + self.shape, A.shape
        self._chk(self._lib.oracle_set_moments(self._h, _dptr(A)), "oracle_set_moments")

    def set_order(self, order: int):
        """Hermite order of the reconstruction: 3 (Eq. 18, default) or 2 (Eq. 8)."""
        self._chk(self._lib.oracle_set_order(self._h, int(order)), "oracle_set_order")

    def set_force(self, g3):
        g = np.ascontiguousarray(g3, dtype=np.float64)
        self._chk(self._lib.oracle_set_force(self._h, _dptr(g)), "oracle_set_force")

    def set_pressure_outlet(self, face: int, rho: float):
        """Density-imposed outlet: u and Pi_neq from x_F, rho imposed."""
        self._chk(self._lib.oracle_set_pressure_outlet(self._h, int(face), float(rho)), "oracle_set_pressure_outlet")

    def set_sponge(self, z_start: int, K: float, p: float = 3.0):
        """Sponge layer towards z = nz (Eq. 26; reading A24).  K = 0 removes it."""
        self._chk(self._lib.oracle_set_sponge(self._h, int(z_start), float(K), float(p)), "oracle_set_sponge")

    def tau_of_plane(self, z: int) -> float:
        return float(self._lib.oracle_tau_of_plane(self._h, int(z)))

    def set_face(self, face: int, kind: int, u_plane=None, noise_amp: float = 0.0, seed: int = 0,
                 noise_mask: int = 0):
        if u_plane is not None:
            U = np.ascontiguousarray(u_plane, dtype=np.float64)
            p = _dptr(U)
        else:
            p = None
        self._chk(self._lib.oracle_set_face(self._h, face, kind, p, float(noise_amp), C.c_uint64(seed),
                                            int(noise_mask)), "oracle_set_face")

    def step(self, n: int = 1, mode: int = MODE_CLOSED):
        self._chk(self._lib.oracle_step(self._h, int(n), int(mode)), "oracle_step")

    def get_moments(self) -> np.ndarray:
        out = np.empty((10,) + self.shape, dtype=np.float64)
        self._chk(self._lib.oracle_get_moments(self._h, _dptr(out)), "oracle_get_moments")
        return out

    def diagnostics(self) -> np.ndarray:
        out = np.empty(5, dtype=np.float64)
        self._chk(self._lib.oracle_diagnostics(self._h, _dptr(out)), "oracle_diagnostics")
        return out

    def plane_statistics(self, axis: int, sums: np.ndarray) -> np.ndarray:
        """Add one sample of the plane sums (Eq. 24-25 raw sums) to sums[13][n_axis] (fp64, C-contiguous)."""
        n_axis = self.shape[2 - axis]
        assert sums.dtype == np.float64 and sums.shape == (13, n_axis) and sums.flags["C_CONTIGUOUS"]
        self._chk(self._lib.oracle_plane_statistics(self._h, int(axis), _dptr(sums)), "oracle_plane_statistics")
        return sums

    def radial_statistics(self, xc: float, yc: float, dr: float, nr: int, sums: np.ndarray) -> np.ndarray:
        """ADD one sample of the (r, z)-bin sums [8][nz][nr] of a jet along z (reading A27)."""
        assert sums.dtype == np.float64 and sums.flags["C_CONTIGUOUS"] and sums.shape == (8, self.shape[0], nr)
        self._chk(self._lib.oracle_radial_statistics(self._h, float(xc), float(yc), float(dr), int(nr), _dptr(sums)),
                  "oracle_radial_statistics")
        return sums

    @property
    def step_count(self) -> int:
        return int(self._lib.oracle_step_count(self._h))

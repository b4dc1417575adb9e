"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.  It holds no
arithmetic of the TSLB method itself (no lattice, no Hermite terms, no update): only initial
fields, boundary descriptions and the parameter arithmetic the configs state (nu -> tau).

Recipe: numpy.random.Generator(PCG64(seed)); draws in the order
ux, uy, uz, each of shape [nz][ny][nx], as float64; perturbations are added in float64 and
the result is cast ONCE to the run dtype.  Node j of an axis with n nodes sits at phase 2*pi*j/n.
The identical array goes to the oracle and to the GPU.

Moment layout everywhere: [10][nz][ny][nx], x fastest,
field order rho, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Optional, Tuple

import numpy as np

FACE_XLO, FACE_XHI, FACE_YLO, FACE_YHI, FACE_ZLO, FACE_ZHI = range(6)
BC_PERIODIC, BC_BOUNCE_BACK, BC_VELOCITY_INLET, BC_OUTLET_ZERO_GRADIENT = range(4)
BC_OUTLET_PRESSURE = 5       # rho imposed (Workload.rho_out[face]), u and Pi_neq from the interior neighbour
NOISE_GAUSSIAN = 0x100       # bit 8 of Inlet.noise_mask: Gaussian instead of uniform inlet noise

_NP_DTYPE = {"f32": np.float32, "f64": np.float64}


@dataclass
class Inlet:
    face: int
    u_plane: np.ndarray          # [3][n_b][n_a] in run dtype (a = lower in-plane axis, fastest)
    noise_amp: float             # relative amplitude: u = u_in * (1 + noise_amp * xi), xi in [-1, 1)
    seed: int
    noise_mask: int              # bit k set -> component k is perturbed


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dtype: str                   # "f32" | "f64"
    tau: float
    steps: int
    moments: np.ndarray          # [10][nz][ny][nx] in run dtype
    faces: Dict[int, int] = field(default_factory=dict)   # face -> kind (default periodic)
    g: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    inlet: Optional[Inlet] = None
    order: int = 3               # Hermite order of the reconstruction (3: Eq. 18, 2: Eq. 8)
    sponge: Optional[Tuple[int, float, float]] = None     # (z_start, K, p) of the sponge layer (Eq. 26), or None
    rho_out: Dict[int, float] = field(default_factory=dict)   # face -> imposed density of a BC_OUTLET_PRESSURE face

    @property
    def sites(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def np_dtype(self):
        return _NP_DTYPE[self.dtype]


def _empty_moments(nx, ny, nz):
    M = np.zeros((10, nz, ny, nx), dtype=np.float64)
    M[0] = 1.0
    return M


def _phase(n):
    return 2.0 * np.pi * np.arange(n, dtype=np.float64) / n


def _taylor_green(M, U0, phases=(0.0, 0.0, 0.0)):
    """u = U0 (sin X cos Y cos Z, -cos X sin Y cos Z, 0) with optional phase shifts."""
    _, nz, ny, nx = M.shape
    X = _phase(nx)[None, None, :] + phases[0]
    Y = _phase(ny)[None, :, None] + phases[1]
    Z = _phase(nz)[:, None, None] + phases[2]
    M[1] += U0 * np.sin(X) * np.cos(Y) * np.cos(Z)
    M[2] += -U0 * np.cos(X) * np.sin(Y) * np.cos(Z)


def _add_uniform_noise(M, amp, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    shape = M.shape[1:]
    for k in (1, 2, 3):                      # draw order ux, uy, uz
        M[k] += rng.uniform(-amp, amp, size=shape)


def config0(n: int = 32, steps: int = 100) -> Workload:
    """configs[0]: fp64 periodic cube, Taylor-Green U0 = 0.01, tau = 0.8."""
    M = _empty_moments(n, n, n)
    _taylor_green(M, 0.01)
    return Workload("cfg0_tg%d_f64" % n, n, n, n, "f64", 0.8, steps, M.astype(np.float64))


def taylor_green_2d(n: int = 32, nz: int = 4, tau: float = 0.8, U0: float = 0.01, steps: int = 100) -> Workload:
    """2-D Taylor-Green vortex extruded along z: u = U0 (sin X cos Y, -cos X sin Y, 0)."""
    M = _empty_moments(n, n, nz)
    X = _phase(n)[None, None, :]
    Y = _phase(n)[None, :, None]
    M[1] += U0 * np.sin(X) * np.cos(Y) * np.ones((nz, 1, 1))
    M[2] += -U0 * np.cos(X) * np.sin(Y) * np.ones((nz, 1, 1))
    return Workload("tg2d_%d" % n, n, n, nz, "f64", tau, steps, M)


def config1(n: int = 128, steps: int = 1000, dtype: str = "f32", U0: float = 0.02) -> Workload:
    """configs[1]: fp32 periodic cube, TG U0 = 0.02 + uniform(+-1e-3) noise (seed 1), tau = 0.5 + 3e-5.
    (U0 is an argument for the stability-margin scan of tests/test_gpu_stability.py.)"""
    M = _empty_moments(n, n, n)
    _taylor_green(M, U0)
    _add_uniform_noise(M, 1e-3, seed=1)
    return Workload("cfg1_tgnoise%d_%s" % (n, dtype), n, n, n, dtype, 0.5 + 3e-5, steps,
                    M.astype(_NP_DTYPE[dtype]))


def channel(nx: int = 384, ny: int = 128, nz: int = 192, steps: int = 2000, dtype: str = "f32",
            u_tau: float = 0.0035, re_tau: float = 180.0, pert: float = 0.05, seed: int = 1) -> Workload:
    """configs[2]: turbulent-channel shape.  Walls (halfway bounce-back) on both y faces, x and z
    periodic, half-width h = ny/2, nu = u_tau h / Re_tau, tau = 0.5 + 3 nu, g = u_tau^2 / h along +x;
    init = laminar parabola u_x(j) = (g / 2 nu)(j + 1/2)(ny - 1/2 - j) + pert * U_c * uniform(-1,1)."""
    h = ny / 2.0
    nu = u_tau * h / re_tau
    tau = 0.5 + 3.0 * nu
    g = u_tau * u_tau / h
    M = _empty_moments(nx, ny, nz)
    j = np.arange(ny, dtype=np.float64)
    prof = (g / (2.0 * nu)) * (j + 0.5) * (ny - 0.5 - j)
    Uc = g * h * h / (2.0 * nu)
    M[1] += prof[None, :, None]
    _add_uniform_noise(M, pert * Uc, seed=seed)
    faces = {FACE_YLO: BC_BOUNCE_BACK, FACE_YHI: BC_BOUNCE_BACK}
    return Workload("cfg2_channel%dx%dx%d_%s" % (nx, ny, nz, dtype), nx, ny, nz, dtype, tau, steps,
                    M.astype(_NP_DTYPE[dtype]), faces=faces, g=(g, 0.0, 0.0))


def jet(nx: int = 256, ny: int = 256, nz: int = 768, steps: int = 1000, dtype: str = "f32",
        U: float = 0.05, D: float = 20.0, re: float = 7000.0, noise: float = 0.01, seed: int = 1) -> Workload:
    """configs[3]: round-jet shape.  z = 0 plane is a velocity inlet (top-hat U inside a disc of
    diameter D centred on the face, 0 outside; relative noise on u_z), every other face is a
    zero-gradient outlet; quiescent rho = 1 start; nu = U D / Re, tau = 0.5 + 3 nu."""
    nu = U * D / re
    tau = 0.5 + 3.0 * nu
    M = _empty_moments(nx, ny, nz)
    x = np.arange(nx, dtype=np.float64)[None, :] - (nx - 1) / 2.0
    y = np.arange(ny, dtype=np.float64)[:, None] - (ny - 1) / 2.0
    disc = (x * x + y * y) <= (D / 2.0) ** 2
    up = np.zeros((3, ny, nx), dtype=np.float64)
    up[2][disc] = U
    faces = {FACE_ZLO: BC_VELOCITY_INLET, FACE_ZHI: BC_OUTLET_ZERO_GRADIENT,
             FACE_XLO: BC_OUTLET_ZERO_GRADIENT, FACE_XHI: BC_OUTLET_ZERO_GRADIENT,
             FACE_YLO: BC_OUTLET_ZERO_GRADIENT, FACE_YHI: BC_OUTLET_ZERO_GRADIENT}
    inlet = Inlet(FACE_ZLO, up.astype(_NP_DTYPE[dtype]), noise, seed, 1 << 2)
    return Workload("cfg3_jet%dx%dx%d_%s" % (nx, ny, nz, dtype), nx, ny, nz, dtype, tau, steps,
                    M.astype(_NP_DTYPE[dtype]), faces=faces, inlet=inlet)


def throughput(n: int = 512, dtype: str = "f32", steps: int = 200, edge: Optional[int] = None) -> Workload:
    """configs[4]: periodic cube, random-phase Taylor-Green U0 = 0.02 (3 phases ~ U(0, 2 pi), seed = n),
    tau = 0.501.  With `edge` only the sub-cube [0, edge)^3 of the n^3 field is built (a bounded sample of
    the same workload for the CPU baseline; it is then treated as a periodic edge^3 box)."""
    rng = np.random.Generator(np.random.PCG64(n))
    ph = rng.uniform(0.0, 2.0 * np.pi, size=3)
    # built in the run dtype plane by plane to keep the host footprint at one copy for 512^3 / 768^3
    npdt = _NP_DTYPE[dtype]
    e = n if edge is None else min(edge, n)
    M = np.zeros((10, e, e, e), dtype=npdt)
    M[0] = 1.0
    X = _phase(n)[None, :e] + ph[0]
    Y = _phase(n)[:e, None] + ph[1]
    Z = _phase(n)[:e] + ph[2]
    a = 0.02 * np.sin(X) * np.cos(Y)
    b = -0.02 * np.cos(X) * np.sin(Y)
    cz = np.cos(Z)
    for k in range(e):
        M[1, k] = (a * cz[k]).astype(npdt)
        M[2, k] = (b * cz[k]).astype(npdt)
    name = "cfg4_tp%d_%s" % (n, dtype) + ("" if e == n else "_sub%d" % e)
    return Workload(name, e, e, e, dtype, 0.501, steps, M)


def random_state(nx: int, ny: int, nz: int, seed: int = 7, dtype: str = "f64", tau: float = 0.7,
                 amp_u: float = 0.05, amp_pi: float = 1e-3) -> Workload:
    """Small random state for brute-force / edge-case tests: rho in 1 +- 0.05, |u| <= amp_u, |Pi| <= amp_pi."""
    rng = np.random.Generator(np.random.PCG64(seed))
    M = np.zeros((10, nz, ny, nx), dtype=np.float64)
    M[0] = 1.0 + rng.uniform(-0.05, 0.05, size=(nz, ny, nx))
    for k in (1, 2, 3):
        M[k] = rng.uniform(-amp_u, amp_u, size=(nz, ny, nx))
    for k in range(4, 10):
        M[k] = rng.uniform(-amp_pi, amp_pi, size=(nz, ny, nx))
    return Workload("rand%dx%dx%d" % (nx, ny, nz), nx, ny, nz, dtype, tau, 1, M.astype(_NP_DTYPE[dtype]))

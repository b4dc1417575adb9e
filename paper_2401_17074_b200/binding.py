"""Thin ctypes binding of libtslb.so (include/tslb.h): argument marshalling only.

Every step of the TSLB path runs in the CUDA kernels behind the C ABI; PyTorch is used for device
memory (the workspace and the caller's moment arrays) and streams.  There is NO CPU fallback: if the
library is missing, or a call needs a CUDA device and none is there, this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libtslb.so")

TSLB_F32, TSLB_F64 = 0, 1
TSLB_OK, TSLB_EINVAL, TSLB_ENOMEM, TSLB_ECUDA, TSLB_ESTATE = range(5)
FACE_XLO, FACE_XHI, FACE_YLO, FACE_YHI, FACE_ZLO, FACE_ZHI = range(6)
BC_PERIODIC, BC_BOUNCE_BACK, BC_VELOCITY_INLET, BC_OUTLET_ZERO_GRADIENT, BC_BODY_FORCE, BC_OUTLET_PRESSURE, BC_EXCHANGE = range(7)
NOISE_GAUSSIAN = 0x100
KERNEL_AUTO, KERNEL_GATHER, KERNEL_TILE = range(3)
KERNEL_NAMES = {KERNEL_AUTO: "auto", KERNEL_GATHER: "gather", KERNEL_TILE: "tile"}

# every symbol include/tslb.h declares (tests check that the library exports all of them)
SYMBOLS = ("tslb_create", "tslb_destroy", "tslb_workspace_bytes", "tslb_bind_workspace", "tslb_set_moments",
           "tslb_set_moments_host", "tslb_set_boundary", "tslb_set_kernel", "tslb_active_kernel", "tslb_step",
           "tslb_get_moments", "tslb_get_moments_host", "tslb_diagnostics", "tslb_step_count",
           "tslb_launch_count", "tslb_last_error", "tslb_version", "tslb_set_timing", "tslb_get_timing", "tslb_set_order", "tslb_plane_statistics",
           "tslb_export_state", "tslb_import_state", "tslb_set_sponge", "tslb_radial_statistics",
           "tslb_plane_statistics_static", "tslb_face_bytes", "tslb_export_face", "tslb_import_face", "tslb_face_planes",
           "tslb_buffers", "tslb_set_neighbor", "tslb_refresh")
PLANE_STATISTICS_STATIC_MAX = 1024   # TSLB_PLANE_STATISTICS_STATIC_MAX of include/tslb.h


class InletParams(C.Structure):
    _fields_ = [("dev_u_plane", C.c_void_p), ("noise_amp", C.c_double), ("seed", C.c_uint64),
                ("noise_component_mask", C.c_int32)]


class TSLBError(RuntimeError):
    def __init__(self, code: int, what: str, msg: str):
        super().__init__("%s failed (status %d): %s" % (what, code, msg))
        self.code = code


_lib = None


def load_library(path: Optional[str] = None):
    """dlopen libtslb.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or os.environ.get("TSLB_LIBRARY") or LIB_PATH     # TSLB_LIBRARY: use another build of the same library
    if not os.path.exists(path):
        raise FileNotFoundError(
            "%s is missing: build it with `python -m paper_2401_17074_b200.build` (no CPU fallback exists)" % path)
    lib = C.CDLL(path)
    vp, ip = C.c_void_p, C.c_int
    lib.tslb_create.argtypes = [ip, ip, ip, C.c_double, ip, C.POINTER(vp)]
    lib.tslb_destroy.argtypes = [vp]
    lib.tslb_destroy.restype = None
    lib.tslb_workspace_bytes.argtypes = [vp]
    lib.tslb_workspace_bytes.restype = C.c_size_t
    lib.tslb_bind_workspace.argtypes = [vp, vp, C.c_size_t]
    lib.tslb_set_moments.argtypes = [vp, vp, vp]
    lib.tslb_set_moments_host.argtypes = [vp, vp, vp]
    lib.tslb_set_boundary.argtypes = [vp, ip, ip, vp]
    lib.tslb_set_kernel.argtypes = [vp, ip]
    lib.tslb_set_order.argtypes = [vp, ip]
    lib.tslb_set_sponge.argtypes = [vp, ip, C.c_double, C.c_double]
    lib.tslb_active_kernel.argtypes = [vp]
    lib.tslb_step.argtypes = [vp, ip, vp]
    lib.tslb_get_moments.argtypes = [vp, vp, vp]
    lib.tslb_get_moments_host.argtypes = [vp, vp, vp]
    lib.tslb_diagnostics.argtypes = [vp, vp, vp]
    lib.tslb_export_state.argtypes = [vp, vp, C.POINTER(C.c_longlong), vp]
    lib.tslb_import_state.argtypes = [vp, vp, C.c_longlong, vp]
    lib.tslb_plane_statistics.argtypes = [vp, ip, vp, vp]
    lib.tslb_plane_statistics_static.argtypes = [vp, ip, vp, vp]
    lib.tslb_radial_statistics.argtypes = [vp, C.c_double, C.c_double, C.c_double, ip, vp, vp]
    lib.tslb_face_bytes.argtypes = [vp]
    lib.tslb_face_bytes.restype = C.c_size_t
    lib.tslb_export_face.argtypes = [vp, ip, vp, vp]
    lib.tslb_import_face.argtypes = [vp, ip, vp, vp]
    lib.tslb_face_planes.argtypes = [vp, ip, C.POINTER(vp), C.POINTER(vp), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t), vp]
    lib.tslb_buffers.argtypes = [vp, C.POINTER(vp), C.POINTER(ip)]
    lib.tslb_set_neighbor.argtypes = [vp, ip, C.POINTER(vp), ip, ip]
    lib.tslb_refresh.argtypes = [vp, vp]
    lib.tslb_set_timing.argtypes = [vp, ip]
    lib.tslb_get_timing.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_double)]
    lib.tslb_step_count.argtypes = [vp]
    lib.tslb_step_count.restype = C.c_longlong
    lib.tslb_launch_count.argtypes = [vp]
    lib.tslb_launch_count.restype = C.c_longlong
    lib.tslb_last_error.argtypes = [vp]
    lib.tslb_last_error.restype = C.c_char_p
    lib.tslb_version.restype = C.c_char_p
    _lib = lib
    return lib


def version() -> str:
    return load_library().tslb_version().decode()


def _stream_ptr(stream) -> C.c_void_p:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(int(getattr(stream, "cuda_stream", stream)))


class TSLB:
    """One lattice on the current CUDA device.  Mirrors the C ABI call for call."""

    def __init__(self, nx: int, ny: int, nz: int, tau: float, dtype: str = "f32", bind: bool = True):
        self._lib = load_library()
        self._h = C.c_void_p()
        self.dtype = dtype
        self.shape = (nz, ny, nx)
        code = {"f32": TSLB_F32, "f64": TSLB_F64}.get(dtype, -1)
        rc = self._lib.tslb_create(nx, ny, nz, float(tau), code, C.byref(self._h))
        if rc:
            raise TSLBError(rc, "tslb_create", self._lib.tslb_last_error(None).decode())
        self._keep = {}       # tensors the context points at (workspace, inlet planes)
        if bind:
            self.bind_workspace()

    # -- plumbing ---------------------------------------------------------------------------
    def _chk(self, rc: int, what: str):
        if rc:
            raise TSLBError(rc, what, self._lib.tslb_last_error(self._h).decode())

    @property
    def torch_dtype(self):
        import torch
        return torch.float32 if self.dtype == "f32" else torch.float64

    def close(self):
        if getattr(self, "_h", None):
            self._lib.tslb_destroy(self._h)
            self._h = C.c_void_p()
            self._keep.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check_tensor(self, t, what, shape=None):
        if not t.is_cuda:
            raise ValueError("%s must be a CUDA tensor" % what)
        if t.dtype != self.torch_dtype or not t.is_contiguous():
            raise ValueError("%s must be contiguous %s" % (what, self.torch_dtype))
        if shape is not None and tuple(t.shape) != tuple(shape):
            raise ValueError("%s has shape %s, expected %s" % (what, tuple(t.shape), tuple(shape)))

    # -- C ABI ------------------------------------------------------------------------------
    def workspace_bytes(self) -> int:
        return int(self._lib.tslb_workspace_bytes(self._h))

    def bind_workspace(self, workspace=None):
        import torch
        if workspace is None:
            if not torch.cuda.is_available():
                raise TSLBError(TSLB_ECUDA, "tslb_bind_workspace", "no CUDA device (there is no CPU fallback)")
            workspace = torch.empty(self.workspace_bytes(), dtype=torch.uint8, device="cuda")
        self._chk(self._lib.tslb_bind_workspace(self._h, C.c_void_p(workspace.data_ptr()), workspace.numel()),
                  "tslb_bind_workspace")
        self._keep["ws"] = workspace
        self._keep.pop("ws_typed", None)

    def set_moments(self, M, stream=None):
        """M: CUDA tensor [10][nz][ny][nx] of the context dtype."""
        self._check_tensor(M, "moments", (10,) + self.shape)
        self._chk(self._lib.tslb_set_moments(self._h, C.c_void_p(M.data_ptr()), _stream_ptr(stream)), "tslb_set_moments")

    def set_moments_host(self, M, stream=None):
        """M: host tensor or numpy array [10][nz][ny][nx] of the context dtype (pinned = async copy)."""
        ptr, keep = _host_ptr(M, self, (10,) + self.shape)
        self._chk(self._lib.tslb_set_moments_host(self._h, ptr, _stream_ptr(stream)), "tslb_set_moments_host")

    def set_boundary(self, face: int, kind: int, u_plane=None, noise_amp: float = 0.0, seed: int = 0,
                     noise_mask: int = 0, rho_out: float = 1.0):
        if kind == BC_OUTLET_PRESSURE:
            rho = C.c_double(float(rho_out))
            self._chk(self._lib.tslb_set_boundary(self._h, face, kind, C.cast(C.byref(rho), C.c_void_p)), "tslb_set_boundary")
        elif kind == BC_VELOCITY_INLET:
            if u_plane is None:
                raise ValueError("VELOCITY_INLET needs u_plane")
            self._check_tensor(u_plane, "u_plane")
            ip = InletParams(C.c_void_p(u_plane.data_ptr()), float(noise_amp), int(seed), int(noise_mask))
            self._chk(self._lib.tslb_set_boundary(self._h, face, kind, C.cast(C.byref(ip), C.c_void_p)),
                      "tslb_set_boundary")
            self._keep["inlet%d" % face] = u_plane
        else:
            self._chk(self._lib.tslb_set_boundary(self._h, face, kind, None), "tslb_set_boundary")

    def set_body_force(self, g: Sequence[float]):
        arr = (C.c_double * 3)(*[float(v) for v in g])
        self._chk(self._lib.tslb_set_boundary(self._h, 0, BC_BODY_FORCE, C.cast(arr, C.c_void_p)), "tslb_set_boundary")

    def set_order(self, order: int):
        """Hermite order of the reconstruction: 3 (Eq. 18, default) or 2 (Eq. 8)."""
        self._chk(self._lib.tslb_set_order(self._h, int(order)), "tslb_set_order")

    def set_sponge(self, z_start: int, K: float, p: float = 3.0):
        """Sponge layer towards z = nz (Eq. 26; reading A24).  K = 0 removes it."""
        self._chk(self._lib.tslb_set_sponge(self._h, int(z_start), float(K), float(p)), "tslb_set_sponge")

    def set_kernel(self, kernel: int):
        self._chk(self._lib.tslb_set_kernel(self._h, int(kernel)), "tslb_set_kernel")

    def active_kernel(self) -> int:
        return int(self._lib.tslb_active_kernel(self._h))

    def step(self, n: int = 1, stream=None):
        self._chk(self._lib.tslb_step(self._h, int(n), _stream_ptr(stream)), "tslb_step")

    def get_moments(self, out=None, stream=None):
        import torch
        if out is None:
            out = torch.empty((10,) + self.shape, dtype=self.torch_dtype, device="cuda")
        self._check_tensor(out, "out", (10,) + self.shape)
        self._chk(self._lib.tslb_get_moments(self._h, C.c_void_p(out.data_ptr()), _stream_ptr(stream)), "tslb_get_moments")
        return out

    def get_moments_host(self, out, stream=None):
        ptr, keep = _host_ptr(out, self, (10,) + self.shape)
        self._chk(self._lib.tslb_get_moments_host(self._h, ptr, _stream_ptr(stream)), "tslb_get_moments_host")
        return out

    def export_state(self, out=None, stream=None):
        """(raw state [10][nz][ny][nx] with field 0 = rho - 1, step counter): the bit-exact checkpoint."""
        import torch
        if out is None:
            out = torch.empty((10,) + self.shape, dtype=self.torch_dtype, device="cuda")
        self._check_tensor(out, "out", (10,) + self.shape)
        t = C.c_longlong(0)
        self._chk(self._lib.tslb_export_state(self._h, C.c_void_p(out.data_ptr()), C.byref(t), _stream_ptr(stream)), "tslb_export_state")
        return out, t.value

    def import_state(self, S, step_count: int, stream=None):
        self._check_tensor(S, "state", (10,) + self.shape)
        self._chk(self._lib.tslb_import_state(self._h, C.c_void_p(S.data_ptr()), int(step_count), _stream_ptr(stream)), "tslb_import_state")

    def face_bytes(self) -> int:
        return int(self._lib.tslb_face_bytes(self._h))

    def export_face(self, face: int, out=None, stream=None):
        """The outermost owned plane next to the EXCHANGE face `face` (FACE_ZLO / FACE_ZHI), raw internal values [10][ny][nx]."""
        import torch
        shape = (10,) + self.shape[1:]
        if out is None:
            out = torch.empty(shape, dtype=self.torch_dtype, device="cuda")
        self._check_tensor(out, "out", shape)
        self._chk(self._lib.tslb_export_face(self._h, int(face), C.c_void_p(out.data_ptr()), _stream_ptr(stream)), "tslb_export_face")
        return out

    def import_face(self, face: int, plane, stream=None):
        """Load the ghost plane of the EXCHANGE face `face` from an array as written by export_face."""
        self._check_tensor(plane, "plane", (10,) + self.shape[1:])
        self._chk(self._lib.tslb_import_face(self._h, int(face), C.c_void_p(plane.data_ptr()), _stream_ptr(stream)), "tslb_import_face")

    def face_planes(self, face: int, stream=None):
        """tslb_face_planes as two tensors [10][plane elements] that alias the workspace: (outermost owned plane, ghost plane)
        of the EXCHANGE face `face` in the current buffer; row f is contiguous.  Valid until the next step of this context."""
        import torch
        owned, ghost, pb, fs = C.c_void_p(), C.c_void_p(), C.c_size_t(), C.c_size_t()
        self._chk(self._lib.tslb_face_planes(self._h, int(face), C.byref(owned), C.byref(ghost), C.byref(pb), C.byref(fs),
                                             _stream_ptr(stream)), "tslb_face_planes")
        ws = self._keep["ws"]
        if not hasattr(ws, "untyped_storage"):
            raise TypeError("face_planes returns views of a torch workspace; this context is bound to %s" % type(ws).__name__)
        es = 4 if self.dtype == "f32" else 8
        typed = self._keep.get("ws_typed")
        if typed is None:
            typed = self._keep["ws_typed"] = ws[: ws.numel() - ws.numel() % es].view(self.torch_dtype)
        view = lambda ptr: torch.as_strided(typed, (10, pb.value // es), (fs.value // es, 1),
                                            typed.storage_offset() + (ptr.value - typed.data_ptr()) // es)
        return view(owned), view(ghost)

    def buffers(self):
        """(address of moment buffer 0, of buffer 1, index of the one that holds the current time level)."""
        arr, cur = (C.c_void_p * 2)(), C.c_int(0)
        self._chk(self._lib.tslb_buffers(self._h, arr, C.byref(cur)), "tslb_buffers")
        return int(arr[0]), int(arr[1]), cur.value

    def set_neighbor(self, face: int, peer_bufs=None, peer_nz: int = 0, peer_cur: int = 0):
        """tslb_set_neighbor: read the ghost plane of the EXCHANGE face `face` in place from the neighbouring slab's buffers
        (two addresses valid on this device, as the neighbour's buffers() reports them); peer_bufs = None detaches."""
        if peer_bufs is None:
            self._chk(self._lib.tslb_set_neighbor(self._h, int(face), None, 0, 0), "tslb_set_neighbor")
            return
        arr = (C.c_void_p * 2)(C.c_void_p(int(peer_bufs[0])), C.c_void_p(int(peer_bufs[1])))
        self._chk(self._lib.tslb_set_neighbor(self._h, int(face), arr, int(peer_nz), int(peer_cur)), "tslb_set_neighbor")

    def refresh(self, stream=None):
        self._chk(self._lib.tslb_refresh(self._h, _stream_ptr(stream)), "tslb_refresh")

    def diagnostics(self, stream=None):
        """(mass, px, py, pz, kinetic energy) as a CUDA fp64 tensor of 5."""
        import torch
        out = torch.empty(5, dtype=torch.float64, device="cuda")
        self._chk(self._lib.tslb_diagnostics(self._h, C.c_void_p(out.data_ptr()), _stream_ptr(stream)), "tslb_diagnostics")
        return out

    def plane_statistics(self, axis: int, sums=None, stream=None):
        """Add one sample of the plane sums (1, u, uu, uuu; Eq. 24-25) along `axis` to sums[13][n_axis] (CUDA fp64)."""
        import torch
        n_axis = self.shape[2 - axis]
        if sums is None:
            sums = torch.zeros((13, n_axis), dtype=torch.float64, device="cuda")
        if not (sums.is_cuda and sums.dtype == torch.float64 and sums.is_contiguous() and tuple(sums.shape) == (13, n_axis)):
            raise ValueError("sums must be a contiguous CUDA float64 tensor of shape (13, %d)" % n_axis)
        self._chk(self._lib.tslb_plane_statistics(self._h, int(axis), C.c_void_p(sums.data_ptr()), _stream_ptr(stream)),
                  "tslb_plane_statistics")
        return sums

    def plane_statistics_static(self, axis: int, sums, stream=None):
        """tslb_plane_statistics_static: the same sums with the scratch in a static device array of the library; allocates
        nothing (the caller passes `sums`), n_axis <= PLANE_STATISTICS_STATIC_MAX, overlapping calls on one GPU race."""
        import torch
        n_axis = self.shape[2 - axis]
        if not (sums.is_cuda and sums.dtype == torch.float64 and sums.is_contiguous() and tuple(sums.shape) == (13, n_axis)):
            raise ValueError("sums must be a contiguous CUDA float64 tensor of shape (13, %d)" % n_axis)
        self._chk(self._lib.tslb_plane_statistics_static(self._h, int(axis), C.c_void_p(sums.data_ptr()), _stream_ptr(stream)),
                  "tslb_plane_statistics_static")
        return sums

    def radial_statistics(self, xc: float, yc: float, dr: float, nr: int, sums=None, stream=None):
        """Add one sample of the (r, z)-bin sums of a jet along z to sums[8][nz][nr] (CUDA fp64)."""
        import torch
        shape = (8, self.shape[0], int(nr))
        if sums is None:
            sums = torch.zeros(shape, dtype=torch.float64, device="cuda")
        if not (sums.is_cuda and sums.dtype == torch.float64 and sums.is_contiguous() and tuple(sums.shape) == shape):
            raise ValueError("sums must be a contiguous CUDA float64 tensor of shape %s" % (shape,))
        self._chk(self._lib.tslb_radial_statistics(self._h, float(xc), float(yc), float(dr), int(nr),
                                                   C.c_void_p(sums.data_ptr()), _stream_ptr(stream)), "tslb_radial_statistics")
        return sums

    def set_timing(self, max_launches: int):
        self._chk(self._lib.tslb_set_timing(self._h, int(max_launches)), "tslb_set_timing")

    def get_timing(self):
        """(number of timed sweep launches, sum of their durations in ms) since the last call."""
        n, ms = C.c_int(0), C.c_double(0.0)
        self._chk(self._lib.tslb_get_timing(self._h, C.byref(n), C.byref(ms)), "tslb_get_timing")
        return n.value, ms.value

    @property
    def step_count(self) -> int:
        return int(self._lib.tslb_step_count(self._h))

    @property
    def launch_count(self) -> int:
        return int(self._lib.tslb_launch_count(self._h))


def _host_ptr(M, ctx: TSLB, shape):
    """Pointer to a contiguous host array (torch CPU tensor or numpy array) of the context dtype."""
    import numpy as np
    if hasattr(M, "data_ptr"):
        if M.is_cuda or M.dtype != ctx.torch_dtype or not M.is_contiguous() or tuple(M.shape) != tuple(shape):
            raise ValueError("host tensor must be contiguous CPU %s of shape %s" % (ctx.torch_dtype, tuple(shape)))
        return C.c_void_p(M.data_ptr()), M
    want = np.float32 if ctx.dtype == "f32" else np.float64
    if not isinstance(M, np.ndarray) or M.dtype != want or not M.flags["C_CONTIGUOUS"] or M.shape != tuple(shape):
        raise ValueError("host array must be C-contiguous %s of shape %s" % (want.__name__, tuple(shape)))
    return C.c_void_p(M.ctypes.data), M


def from_workload(w, kernel: int = KERNEL_AUTO, workspace=None) -> TSLB:
    """Context configured (boundary set, force, kernel choice) for a workloads.Workload; state not loaded.
    workspace: None (a torch allocation) or a callable nbytes -> object with data_ptr() / numel() to bind instead."""
    import torch
    sim = TSLB(w.nx, w.ny, w.nz, w.tau, w.dtype, bind=workspace is None)
    if workspace is not None:
        sim.bind_workspace(workspace(sim.workspace_bytes()))
    for face, kind in w.faces.items():
        if w.inlet is not None and face == w.inlet.face:
            up = torch.from_numpy(w.inlet.u_plane).to("cuda")
            sim.set_boundary(face, kind, up, w.inlet.noise_amp, w.inlet.seed, w.inlet.noise_mask)
        elif kind == BC_OUTLET_PRESSURE:
            sim.set_boundary(face, kind, rho_out=w.rho_out[face])
        else:
            sim.set_boundary(face, kind)
    if any(w.g):
        sim.set_body_force(w.g)
    if getattr(w, "order", 3) != 3:
        sim.set_order(w.order)
    if getattr(w, "sponge", None):
        sim.set_sponge(*w.sponge)
    sim.set_kernel(kernel)
    return sim

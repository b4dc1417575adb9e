"""Slab decomposition of one lattice along z over several GPUs.

Host-side orchestration only: every number is produced by the kernels behind the C ABI.  A rank owns the planes
[z_lo, z_hi) of the global lattice in a context of its own (`binding.TSLB`) whose z axis carries one ghost plane per cut
face (face kind BC_EXCHANGE, include/tslb.h "Slab decomposition").  One step is

    sweep of the slab (tslb_step)  ->  transport of the outermost owned planes into the neighbours' ghost planes
    (zero copy: in place in the workspaces, tslb_face_planes; or staged: tslb_export_face -> transport -> tslb_import_face)

or, where the slabs' buffers are mutually addressable (one process; `connect_local` / `step_connected`), no transport at
all: the tile kernel's TMA producer loads the ghost planes from the neighbours' buffers while it sweeps (tslb_set_neighbor)

and because a sweep reads time-t nearest neighbours only (PAPER.md:68 Eq. 6, :157), the owned planes advance bit for bit
as in the undivided lattice.  Transport: `torch.distributed` point-to-point (NCCL over NVLink / NVSwitch: one 40 B/node
plane per cut face and direction, 10.5 MB for 512^2 fp32, i.e. ~12 us at 900 GB/s against a ~2.3 ms sweep -- the
exchange is not overlapped with the sweep, there is nothing to win yet), or plain device copies between slabs that live
in one process on one GPU (`exchange_local`, what the 1-GPU parity test uses; the slabs never wait on one another).

Limits (checked, with an error): the seeded inlet noise is keyed on a context's own node index, so a noisy inlet must sit
on the global z = 0 / z = nz-1 face of a first / last slab whose z offset is zero (the jet's inlet does); a sponge layer
(Eq. 26) must lie inside the last slab.  `Slab.plane_statistics` / `radial_statistics` / `diagnostics` give the sums of
the undivided lattice (ghost planes left out).
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass
from typing import List, Optional, Sequence

from . import workloads as W

BC_EXCHANGE = 6   # TSLB_BC_EXCHANGE (include/tslb.h)


@dataclass(frozen=True)
class SlabPlan:
    """Planes [z_lo, z_hi) of an nz-plane lattice on `rank` of `world`; lo_rank / hi_rank = -1 where the slab ends on a
    face of the global lattice (which then keeps its own boundary kind)."""
    rank: int
    world: int
    nz: int
    z_lo: int
    z_hi: int
    lo_rank: int
    hi_rank: int

    @property
    def ghost_lo(self) -> bool:
        return self.lo_rank >= 0

    @property
    def ghost_hi(self) -> bool:
        return self.hi_rank >= 0

    @property
    def owned(self) -> int:
        return self.z_hi - self.z_lo

    @property
    def nz_local(self) -> int:
        return self.owned + int(self.ghost_lo) + int(self.ghost_hi)

    @property
    def z_offset(self) -> int:
        """global z of local plane 0"""
        return self.z_lo - int(self.ghost_lo)


def plan_slabs(nz: int, world: int, periodic_z: bool) -> List[SlabPlan]:
    """Balanced split: the first nz % world ranks own one plane more.  Every slab owns at least one plane and its context
    at least three (tslb_create's minimum)."""
    if world < 1 or nz < world:
        raise ValueError("cannot split %d planes over %d ranks" % (nz, world))
    base, rem = divmod(nz, world)
    plans, z = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        if world == 1:
            lo = hi = -1                       # undivided: the z faces keep their kinds (periodic wraps inside the kernel)
        elif periodic_z:
            lo, hi = (r - 1) % world, (r + 1) % world
        else:
            lo, hi = (r - 1 if r > 0 else -1), (r + 1 if r < world - 1 else -1)
        p = SlabPlan(r, world, nz, z, z + n, lo, hi)
        if p.nz_local < 3:
            raise ValueError("slab of rank %d would have %d planes (< 3): use fewer ranks" % (r, p.nz_local))
        plans.append(p)
        z += n
    return plans


def local_workload(w: W.Workload, plan: SlabPlan) -> W.Workload:
    """The slab's own Workload: the global initial state cut to the slab's planes (ghost planes included, wrapped on a
    periodic axis), EXCHANGE on the cut faces, everything else as in `w`."""
    import numpy as np
    periodic_z = w.faces.get(W.FACE_ZLO, W.BC_PERIODIC) == W.BC_PERIODIC
    zs = np.arange(plan.z_offset, plan.z_offset + plan.nz_local)
    if periodic_z:
        zs = zs % w.nz
    faces = dict(w.faces)
    if plan.world > 1:
        faces[W.FACE_ZLO] = BC_EXCHANGE if plan.ghost_lo else w.faces.get(W.FACE_ZLO, W.BC_PERIODIC)
        faces[W.FACE_ZHI] = BC_EXCHANGE if plan.ghost_hi else w.faces.get(W.FACE_ZHI, W.BC_PERIODIC)
    inlet = w.inlet
    if inlet is not None and plan.world > 1:
        if inlet.face == W.FACE_ZLO and plan.ghost_lo:
            inlet = None                                        # the inlet face belongs to the first slab
        elif inlet.face == W.FACE_ZHI and plan.ghost_hi:
            inlet = None
        elif inlet.face == W.FACE_ZHI and inlet.noise_amp != 0.0 and plan.z_offset != 0:
            raise NotImplementedError("noisy inlet on z = nz-1 of a slab with a z offset (noise is keyed on local indices)")
        elif inlet.face < W.FACE_ZLO:
            if inlet.noise_amp != 0.0:
                raise NotImplementedError("noisy inlet on a face the slab cuts cross (noise is keyed on local indices)")
            up = inlet.u_plane                                  # [3][nz][n_a]: cut to the slab's planes
            inlet = dataclasses.replace(inlet, u_plane=np.ascontiguousarray(up[:, zs, :]))
    sponge = w.sponge
    if sponge is not None and plan.world > 1:
        z_start, K, p = sponge
        if plan.z_hi != w.nz:
            if z_start < plan.z_hi + 1:                         # the layer reaches this slab's planes or its upper ghost plane
                raise NotImplementedError("sponge layer starts below the last slab")
            sponge = None
        else:
            if z_start <= plan.z_offset:
                raise NotImplementedError("sponge layer starts below the last slab")
            sponge = (z_start - plan.z_offset, K, p)            # nz_local - z_start_local = nz - z_start: same profile
    return dataclasses.replace(w, name="%s_slab%dof%d" % (w.name, plan.rank, plan.world), nz=plan.nz_local,
                               moments=np.ascontiguousarray(w.moments[:, zs]), faces=faces, inlet=inlet, sponge=sponge)


def _chunks(t):
    return [] if t is None else (list(t) if isinstance(t, (list, tuple)) else [t])


def exchange_planes(plan: SlabPlan, send_lo, send_hi, recv_lo, recv_hi, group=None) -> None:
    """Point-to-point exchange of the cut-face planes with the neighbouring ranks (any device `torch.distributed` serves:
    NCCL for CUDA tensors, gloo for CPU ones).  send_lo / send_hi: this rank's outermost owned planes; recv_lo / recv_hi:
    what becomes its ghost planes; each a contiguous tensor or a list of contiguous chunks (the ten field runs of a plane
    inside the workspace, for the zero-copy path).  With two ranks on a periodic axis both neighbours are the same peer:
    messages between a pair are matched in the order they are issued (NCCL has no tags), so the low plane is always sent
    first and the matching receive -- the neighbour's LOW plane is this rank's HIGH ghost -- is issued first."""
    import torch.distributed as dist
    ops = []
    if plan.ghost_lo:
        ops += [dist.P2POp(dist.isend, c, plan.lo_rank, group, tag=i) for i, c in enumerate(_chunks(send_lo))]
    if plan.ghost_hi:
        ops += [dist.P2POp(dist.isend, c, plan.hi_rank, group, tag=64 + i) for i, c in enumerate(_chunks(send_hi))]
    if plan.ghost_hi:
        ops += [dist.P2POp(dist.irecv, c, plan.hi_rank, group, tag=i) for i, c in enumerate(_chunks(recv_hi))]
    if plan.ghost_lo:
        ops += [dist.P2POp(dist.irecv, c, plan.lo_rank, group, tag=64 + i) for i, c in enumerate(_chunks(recv_lo))]
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()


def _cudart():
    from cuda.bindings import runtime as rt
    return rt


class RawWorkspace:
    """Device memory straight from cudaMalloc (not torch's caching allocator, whose blocks share allocations): its CUDA IPC
    handle names exactly this workspace.  Quacks like the tensor binding.TSLB.bind_workspace expects."""

    def __init__(self, nbytes: int):
        import torch
        torch.empty(1, device="cuda")          # torch's current device is the runtime's current device from here on
        rt = _cudart()
        err, ptr = rt.cudaMalloc(int(nbytes))
        if int(err) != 0:
            raise RuntimeError("cudaMalloc(%d) failed: %s" % (nbytes, err))
        self._ptr, self._n = int(ptr), int(nbytes)

    def data_ptr(self) -> int:
        return self._ptr

    def numel(self) -> int:
        return self._n

    def ipc_handle(self) -> bytes:
        err, h = _cudart().cudaIpcGetMemHandle(self._ptr)
        if int(err) != 0:
            raise RuntimeError("cudaIpcGetMemHandle failed: %s" % err)
        return bytes(h.reserved)

    def __del__(self):
        try:
            if self._ptr:
                _cudart().cudaFree(self._ptr)
                self._ptr = 0
        except Exception:
            pass


class Slab:
    """One rank's part of a slab-decomposed lattice on the current CUDA device.  staged = False (default): the transport
    reads the owned planes and writes the ghost planes in place in the workspace (tslb_face_planes, zero copy);
    staged = True: through dense arrays (tslb_export_face / tslb_import_face)."""

    def __init__(self, w: W.Workload, plan: SlabPlan, kernel: int = 0, staged: bool = False, ipc: bool = False):
        import torch
        from . import binding
        self.plan = plan
        self.staged = staged
        self.local = local_workload(w, plan)
        # ipc: the workspace is a cudaMalloc allocation of its own, so that other processes can map it (connect_ipc)
        self.sim = binding.from_workload(self.local, kernel, RawWorkspace if ipc else None)
        self._opened = {}          # rank -> base address of that rank's workspace mapped into this process
        self.sim.set_moments(torch.from_numpy(self.local.moments).to("cuda"))
        shape = (10, w.ny, w.nx)
        mk = lambda: torch.empty(shape, dtype=self.sim.torch_dtype, device="cuda")
        self.send_lo, self.recv_lo = (mk(), mk()) if plan.ghost_lo and staged else (None, None)
        self.send_hi, self.recv_hi = (mk(), mk()) if plan.ghost_hi and staged else (None, None)

    # staged path: the three phases of one exchange (tslb_export_face / transport / tslb_import_face)
    def export_faces(self, stream=None):
        if self.plan.ghost_lo:
            self.sim.export_face(W.FACE_ZLO, self.send_lo, stream)
        if self.plan.ghost_hi:
            self.sim.export_face(W.FACE_ZHI, self.send_hi, stream)

    def import_faces(self, stream=None):
        if self.plan.ghost_lo:
            self.sim.import_face(W.FACE_ZLO, self.recv_lo, stream)
        if self.plan.ghost_hi:
            self.sim.import_face(W.FACE_ZHI, self.recv_hi, stream)

    # zero-copy path: (owned_lo, ghost_lo, owned_hi, ghost_hi) as views [10][plane] of the workspace, None where uncut
    def planes(self, stream=None):
        olo, glo = self.sim.face_planes(W.FACE_ZLO, stream) if self.plan.ghost_lo else (None, None)
        ohi, ghi = self.sim.face_planes(W.FACE_ZHI, stream) if self.plan.ghost_hi else (None, None)
        return olo, glo, ohi, ghi

    def exchange(self, group=None):
        if self.staged:
            self.export_faces()
            exchange_planes(self.plan, self.send_lo, self.send_hi, self.recv_lo, self.recv_hi, group)
            self.import_faces()
        else:
            rows = lambda v: None if v is None else [v[f] for f in range(v.shape[0])]     # ten contiguous runs
            olo, glo, ohi, ghi = self.planes()
            exchange_planes(self.plan, rows(olo), rows(ohi), rows(glo), rows(ghi), group)

    def step(self, n: int = 1, group=None):
        """n time steps of the whole lattice as seen from this rank (collective: every rank calls it)."""
        for _ in range(n):
            self.sim.step(1)
            self.exchange(group)

    def owned(self, M):
        """Cut the ghost planes off an array whose axis 1 is the slab's z axis (get_moments, export_state)."""
        return M[:, int(self.plan.ghost_lo): self.plan.nz_local - int(self.plan.ghost_hi)]

    def owned_moments(self):
        return self.owned(self.sim.get_moments())

    def plane_statistics(self, axis: int, sums, group=None, reduce: bool = False):
        """One sample of the plane sums (tslb_plane_statistics) of this slab's OWNED planes added to `sums`, the array of
        the whole lattice ([13][n_axis of the undivided lattice], CUDA fp64): planes of constant x or y get this slab's
        share, planes of constant z land in rows z_lo .. z_hi.  reduce = True adds the ranks up (collective; then every
        rank must pass an array that holds only its own contribution, e.g. zeros)."""
        import torch
        loc = self.sim.plane_statistics(axis)                      # ghost planes are left out by the library
        if axis == 2:
            sums[:, self.plan.z_lo:self.plan.z_hi] += self.owned(loc)
        else:
            sums += loc
        if reduce and self.plan.world > 1:
            import torch.distributed as dist
            dist.all_reduce(sums, op=dist.ReduceOp.SUM, group=group)
        return sums

    def radial_statistics(self, xc: float, yc: float, dr: float, nr: int, sums):
        """One sample of the (r, z)-ring sums (tslb_radial_statistics) of the owned planes added to rows z_lo .. z_hi of
        `sums` ([8][nz of the undivided lattice][nr], CUDA fp64)."""
        loc = self.sim.radial_statistics(xc, yc, dr, nr)
        sums[:, self.plan.z_lo:self.plan.z_hi] += self.owned(loc)
        return sums

    def diagnostics(self, group=None, reduce: bool = True):
        """(mass, momentum[3], kinetic energy) of the whole lattice: the slabs' sums (ghost planes left out) added up."""
        import torch.distributed as dist
        d = self.sim.diagnostics()
        if reduce and self.plan.world > 1:
            dist.all_reduce(d, op=dist.ReduceOp.SUM, group=group)
        return d


def _rank_barrier(group=None) -> None:
    """One ordering point between the ranks' GPU work.  NCCL: a one-element all-reduce on the current stream (device side:
    it completes when every rank's preceding sweep has, and the following sweep waits for it; the host does not block).
    Other backends (gloo in the tests): synchronise the device, then a host barrier."""
    import torch
    import torch.distributed as dist
    if dist.get_backend(group) == "nccl":
        dist.all_reduce(torch.zeros(1, device="cuda"), group=group)
    else:
        torch.cuda.synchronize()
        dist.barrier(group)


def connect_ipc(slab: Slab, group=None) -> None:
    """connect_local across processes (one slab per rank, Slab(..., ipc=True)): every rank publishes the CUDA IPC handle of
    its workspace and where its two moment buffers sit in it, maps its neighbours' workspaces (cudaIpcOpenMemHandle with
    lazy peer access: NVLink peer memory when the neighbour is another GPU of the node) and attaches them
    (tslb_set_neighbor).  Collective; all ranks at the same step count.  Advance with step_connected_dist."""
    import os
    import torch.distributed as dist
    rt = _cudart()
    ws = slab.sim._keep["ws"]
    if not isinstance(ws, RawWorkspace):
        raise ValueError("connect_ipc needs Slab(..., ipc=True)")
    b0, b1, cur = slab.sim.buffers()
    mine = (ws.ipc_handle(), b0 - ws.data_ptr(), b1 - ws.data_ptr(), slab.plan.nz_local, cur, os.getpid())
    infos = [None] * slab.plan.world
    dist.all_gather_object(infos, mine, group=group)
    for face, on, nb in ((W.FACE_ZLO, slab.plan.ghost_lo, slab.plan.lo_rank), (W.FACE_ZHI, slab.plan.ghost_hi, slab.plan.hi_rank)):
        if not on:
            continue
        handle, o0, o1, nz, pcur, _ = infos[nb]
        if nb not in slab._opened:
            h = rt.cudaIpcMemHandle_t()
            h.reserved = handle
            err, base = rt.cudaIpcOpenMemHandle(h, rt.cudaIpcMemLazyEnablePeerAccess)
            if int(err) != 0:
                raise RuntimeError("cudaIpcOpenMemHandle (rank %d) failed: %s" % (nb, err))
            slab._opened[nb] = int(base)
        base = slab._opened[nb]
        slab.sim.set_neighbor(face, (base + o0, base + o1), nz, pcur)
    _rank_barrier(group)


def step_connected_dist(slab: Slab, n: int = 1, group=None) -> None:
    """n steps of IPC-connected slabs, one rank each: complete the own state of time t, one ordering point (every rank's
    state of time t complete, every sweep of step t-1 finished: the buffer it read may be overwritten), sweep.  The
    closing ordering point keeps the buffers of the last step alive until every neighbour has read them."""
    for _ in range(n):
        slab.sim.refresh()
        _rank_barrier(group)
        slab.sim.step(1)
    _rank_barrier(group)


def disconnect_ipc(slab: Slab, group=None) -> None:
    """Detach the neighbours and unmap their workspaces (collective: nobody may still be sweeping)."""
    _rank_barrier(group)
    for face, on in ((W.FACE_ZLO, slab.plan.ghost_lo), (W.FACE_ZHI, slab.plan.ghost_hi)):
        if on:
            slab.sim.set_neighbor(face, None)
    for base in slab._opened.values():
        _cudart().cudaIpcCloseMemHandle(base)
    slab._opened.clear()
    _rank_barrier(group)


def exchange_local(slabs: Sequence[Slab]) -> None:
    """The exchange between slabs that live in one process on one GPU: plane-to-plane device copies on the current stream
    (zero-copy path: straight from workspace to workspace; staged path: export everywhere, copy, import).  Serial launches
    of one stream: no kernel ever waits on another."""
    if slabs and slabs[0].staged:
        for s in slabs:
            s.export_faces()
        for s in slabs:
            if s.plan.ghost_lo:
                s.recv_lo.copy_(slabs[s.plan.lo_rank].send_hi)
            if s.plan.ghost_hi:
                s.recv_hi.copy_(slabs[s.plan.hi_rank].send_lo)
        for s in slabs:
            s.import_faces()
        return
    views = [s.planes() for s in slabs]                    # also completes every owned plane for the current time
    for s, (_, glo, _, ghi) in zip(slabs, views):
        if s.plan.ghost_lo:
            glo.copy_(views[s.plan.lo_rank][2])            # the HIGH owned plane of the slab below
        if s.plan.ghost_hi:
            ghi.copy_(views[s.plan.hi_rank][0])            # the LOW owned plane of the slab above


def connect_local(slabs: Sequence[Slab]) -> None:
    """Fused form (tslb_set_neighbor): every slab's tile kernel reads its ghost planes in place from the neighbouring slabs'
    current buffers while it sweeps; nothing is exchanged between steps.  Slabs of one process whose buffers are mutually
    addressable: one GPU, or several GPUs of one process with peer access enabled.  Tile kernel only (tslb_step refuses
    otherwise).  Call after the states are loaded, with all slabs at the same step count; advance with step_connected."""
    for s in slabs:
        for face, on, nb in ((W.FACE_ZLO, s.plan.ghost_lo, s.plan.lo_rank), (W.FACE_ZHI, s.plan.ghost_hi, s.plan.hi_rank)):
            if on:
                b0, b1, cur = slabs[nb].sim.buffers()
                s.sim.set_neighbor(face, (b0, b1), slabs[nb].plan.nz_local, cur)


def step_connected(slabs: Sequence[Slab], n: int = 1) -> None:
    """n steps of connected slabs on one stream: first every slab's state of time t is completed (tslb_refresh: lateral
    open-face nodes, ghost columns), then every slab is swept -- each sweep reads only time-t buffers and writes its own
    time-(t+1) buffer, so stream order is all the synchronisation there is."""
    for _ in range(n):
        for s in slabs:
            s.sim.refresh()
        for s in slabs:
            s.sim.step(1)


def step_local(slabs: Sequence[Slab], n: int = 1) -> None:
    for _ in range(n):
        for s in slabs:
            s.sim.step(1)
        exchange_local(slabs)


def gather_local(slabs: Sequence[Slab]):
    """The whole lattice's moments [10][nz][ny][nx] from slabs of one process, in rank order."""
    import torch
    return torch.cat([s.owned_moments() for s in slabs], dim=1)

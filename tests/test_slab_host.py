"""Host logic of the slab decomposition (paper_2401_17074_b200/slab.py): the plan, the slab workloads, and the
point-to-point plane exchange over a world_size-2 gloo group on CPU (N > 1 paths are covered with gloo)."""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2401_17074_b200 import slab as S
from paper_2401_17074_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("nz,world,periodic", [(12, 1, True), (12, 2, True), (13, 4, True), (13, 4, False), (7, 3, False), (3, 3, True)])
def test_plan_covers_every_plane_once(nz, world, periodic):
    plans = S.plan_slabs(nz, world, periodic)
    assert [p.rank for p in plans] == list(range(world))
    assert plans[0].z_lo == 0 and plans[-1].z_hi == nz
    for a, b in zip(plans, plans[1:]):
        assert a.z_hi == b.z_lo and a.owned - b.owned in (0, 1)          # contiguous, balanced, larger slabs first
    for p in plans:
        assert p.owned >= 1 and p.nz_local == p.owned + p.ghost_lo + p.ghost_hi >= 3
        if world == 1:
            assert not p.ghost_lo and not p.ghost_hi
        elif periodic:
            assert p.lo_rank == (p.rank - 1) % world and p.hi_rank == (p.rank + 1) % world
        else:
            assert p.lo_rank == (p.rank - 1 if p.rank else -1) and p.hi_rank == (p.rank + 1 if p.rank < world - 1 else -1)
        # neighbours point at each other
        if p.ghost_hi:
            assert plans[p.hi_rank].lo_rank == p.rank
        if p.ghost_lo:
            assert plans[p.lo_rank].hi_rank == p.rank


def test_plan_rejects_impossible_splits():
    with pytest.raises(ValueError):
        S.plan_slabs(4, 5, True)
    with pytest.raises(ValueError):
        S.plan_slabs(2, 2, False)       # an end slab would hold one owned + one ghost plane: below tslb_create's minimum


def test_local_workload_periodic_wraps_ghost_planes():
    w = W.random_state(5, 6, 11, seed=3)
    plans = S.plan_slabs(w.nz, 3, True)
    seen = np.zeros(w.nz, dtype=int)
    for p in plans:
        lw = S.local_workload(w, p)
        assert lw.nz == p.nz_local and lw.faces[W.FACE_ZLO] == lw.faces[W.FACE_ZHI] == S.BC_EXCHANGE
        zs = np.arange(p.z_offset, p.z_offset + p.nz_local) % w.nz
        assert np.array_equal(lw.moments, w.moments[:, zs])
        seen[p.z_lo:p.z_hi] += 1
    assert (seen == 1).all()


def test_local_workload_jet_keeps_end_faces_and_inlet_on_first_slab():
    w = W.jet(12, 12, 20, steps=1)
    w.sponge = (15, 10.0, 3.0)
    plans = S.plan_slabs(w.nz, 2, False)
    lo, hi = (S.local_workload(w, p) for p in plans)
    assert lo.faces[W.FACE_ZLO] == W.BC_VELOCITY_INLET and lo.faces[W.FACE_ZHI] == S.BC_EXCHANGE and lo.inlet is w.inlet
    assert hi.faces[W.FACE_ZLO] == S.BC_EXCHANGE and hi.faces[W.FACE_ZHI] == W.BC_OUTLET_ZERO_GRADIENT and hi.inlet is None
    assert lo.faces[W.FACE_XLO] == hi.faces[W.FACE_XLO] == W.BC_OUTLET_ZERO_GRADIENT
    # the sponge layer lives in the last slab, with the same width (nz_local - z_start_local = nz - z_start)
    assert lo.sponge is None and hi.sponge == (15 - plans[1].z_offset, 10.0, 3.0)
    assert hi.nz - hi.sponge[0] == w.nz - 15
    w.sponge = (8, 10.0, 3.0)                                   # reaches below the last slab: refused, not silently wrong
    with pytest.raises(NotImplementedError):
        S.local_workload(w, plans[0])


WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
from paper_2401_17074_b200 import slab as S
rank, port, periodic = int(sys.argv[1]), sys.argv[2], sys.argv[3] == "1"
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + port, rank=rank, world_size=2)
plan = S.plan_slabs(10, 2, periodic)[rank]
shape = (10, 3, 4)
mk = lambda v: torch.full(shape, float(v))
# plane value = 10 * owner + (0 low plane | 1 high plane)
send_lo, send_hi = mk(10 * rank), mk(10 * rank + 1)
recv_lo, recv_hi = mk(-1), mk(-1)
chunked = sys.argv[4] == "1"        # the zero-copy path hands over the ten field runs of a plane one by one
if chunked:
    send_lo += torch.arange(10.0).view(10, 1, 1) / 100; send_hi += torch.arange(10.0).view(10, 1, 1) / 100
rows = lambda t: [t[f] for f in range(10)] if chunked else t
for it in range(3):            # several exchanges in a row: the pairing must not drift
    S.exchange_planes(plan, rows(send_lo) if plan.ghost_lo else None, rows(send_hi) if plan.ghost_hi else None,
                      rows(recv_lo) if plan.ghost_lo else None, rows(recv_hi) if plan.ghost_hi else None)
    other = 1 - rank
    field = (torch.arange(10.0).view(10, 1, 1) / 100) if chunked else 0.0
    if plan.ghost_lo:          # my low ghost plane is the HIGH plane of the rank below
        assert (recv_lo == 10 * other + 1 + field).all(), (rank, it, recv_lo.flatten()[0])
    else:
        assert (recv_lo == -1).all()
    if plan.ghost_hi:          # my high ghost plane is the LOW plane of the rank above
        assert (recv_hi == 10 * other + field).all(), (rank, it, recv_hi.flatten()[0])
    else:
        assert (recv_hi == -1).all()
    recv_lo.fill_(-1); recv_hi.fill_(-1)
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
"""


@pytest.mark.parametrize("chunked", [False, True])
@pytest.mark.parametrize("periodic", [True, False])
def test_exchange_planes_world_size_2_gloo(tmp_path, periodic, chunked):
    """Two ranks: on a periodic axis both neighbours are the same peer (the pairing of the two messages is what can go
    wrong); on a bounded axis each rank has one neighbour only."""
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    procs = [subprocess.Popen([sys.executable, str(script), str(r), str(port), "1" if periodic else "0", "1" if chunked else "0"],
                              stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True) for r in range(2)]
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0 and "ok" in o, o


def test_local_workload_cuts_a_lateral_inlet_plane_and_refuses_its_noise():
    """An inlet on a face the cuts cross: its imposed-velocity plane [3][nz][nx] is cut to the slab's planes (ghost planes
    included); with noise it is refused (the noise stream is keyed on a context's own node index)."""
    w = W.random_state(6, 5, 12, seed=4)
    up = np.random.default_rng(1).uniform(-0.03, 0.03, (3, w.nz, w.nx))
    w.faces = {W.FACE_YHI: W.BC_VELOCITY_INLET, W.FACE_YLO: W.BC_OUTLET_ZERO_GRADIENT}
    w.inlet = W.Inlet(W.FACE_YHI, up, 0.0, 9, 0)
    for p in S.plan_slabs(w.nz, 3, True):
        lw = S.local_workload(w, p)
        zs = np.arange(p.z_offset, p.z_offset + p.nz_local) % w.nz
        assert lw.inlet.u_plane.shape == (3, p.nz_local, w.nx) and np.array_equal(lw.inlet.u_plane, up[:, zs, :])
    w.inlet = W.Inlet(W.FACE_YHI, up, 0.05, 9, 0b111)
    with pytest.raises(NotImplementedError):
        S.local_workload(w, S.plan_slabs(w.nz, 3, True)[1])

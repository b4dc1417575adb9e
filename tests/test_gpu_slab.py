"""Slab decomposition along z (include/tslb.h tslb_export_face / tslb_import_face): several
slabs of one lattice, each in a context of its own, advanced on ONE GPU with the ghost planes exchanged by device copies
(slab.step_local: serial launches on one stream, no kernel waits on another), against (1) the fp64 oracle of the UNDIVIDED
lattice, element by element, at the tolerances of the other parity tests, and (2) the undivided CUDA run, bit for bit --
a node's arithmetic does not depend on where the lattice was cut.  The transport over torch.distributed is covered on CPU
(tests/test_slab_host.py, gloo, world_size 2)."""
import dataclasses
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2401_17074_b200 import slab as S
from paper_2401_17074_b200 import workloads as W
from tests.parity_util import assert_parity, gpu_state, make_gpu, make_oracle
from tests.test_gpu_parity import BC_SETS, B, kernels_for, with_faces  # noqa: F401  (B is the fixture)

pytestmark = pytest.mark.gpu


def run_slabs(w, world, steps, kernel, staged=False):
    import torch
    periodic_z = w.faces.get(W.FACE_ZLO, W.BC_PERIODIC) == W.BC_PERIODIC
    slabs = [S.Slab(w, p, kernel, staged) for p in S.plan_slabs(w.nz, world, periodic_z)]
    S.step_local(slabs, steps)
    G = S.gather_local(slabs)
    torch.cuda.synchronize()
    return slabs, G.cpu().numpy()


def lateral_inlet(dt):
    """Inlet on a face the cuts cross (its imposed-velocity plane is cut with the slabs); noise off, see slab.py."""
    w = with_faces(W.random_state(40, 16, 17, seed=55, dtype=dt, tau=0.6), **BC_SETS["outlet_y_walls_z"])
    w.inlet = dataclasses.replace(w.inlet, noise_amp=0.0, noise_mask=0)
    return w


CASES = {
    "periodic": lambda dt: W.random_state(70, 27, 23, seed=51, dtype=dt, tau=0.58),
    "channel": lambda dt: with_faces(W.random_state(66, 15, 21, seed=52, dtype=dt, tau=0.6), **BC_SETS["walls_y+force"]),
    "jet_like": lambda dt: with_faces(W.random_state(24, 17, 30, seed=53, dtype=dt, tau=0.55), **BC_SETS["jet_like"]),
    "walls_z": lambda dt: with_faces(W.random_state(64, 12, 19, seed=54, dtype=dt, tau=0.6), **BC_SETS["walls_z"]),
    "inlet_y_walls_z": lambda dt: lateral_inlet(dt),
    "wall_outlet_z": lambda dt: with_faces(W.random_state(33, 17, 14, seed=56, dtype=dt, tau=0.6),
                                           **BC_SETS["mixed_wall_outlet_same_axis"]),
}


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("case", sorted(CASES))
def test_slabs_match_oracle_and_undivided_run(B, oracle_mod, case, world, dtype):
    w = CASES[case](dtype)
    steps = 6
    o = make_oracle(oracle_mod, w)
    o.step(steps)
    R = o.get_moments()
    for k in kernels_for(B, w):
        slabs_st, G_st = run_slabs(w, world, steps, k, staged=True)        # tslb_export_face / tslb_import_face
        slabs, G = run_slabs(w, world, steps, k)                           # tslb_face_planes (zero copy)
        assert np.array_equal(G, G_st)
        for s in slabs_st:
            s.sim.close()
        assert all(s.sim.step_count == steps for s in slabs)
        assert_parity(w, G.astype(np.float64), R, "%s, %d slabs, kernel %d" % (case, world, k))
        one = make_gpu(w, k)
        one.step(steps)
        G1 = one.get_moments().cpu().numpy()
        assert np.array_equal(G, G1), "%s: %d slabs differ from the undivided run (kernel %d), max %.3e" % (
            case, world, k, np.abs(G.astype(np.float64) - G1).max())
        # the slabs' diagnostics add up to the undivided lattice's (ghost planes are left out)
        d = sum(s.diagnostics(reduce=False).cpu().numpy() for s in slabs)
        d1 = one.diagnostics().cpu().numpy()
        np.testing.assert_allclose(d, d1, rtol=1e-12, atol=1e-12 * abs(d1[0]))
        one.close()
        for s in slabs:
            s.sim.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("case", sorted(CASES))
def test_connected_slabs_read_their_neighbours_in_place(B, case, world, dtype):
    """tslb_set_neighbor: the tile kernel loads the ghost planes from the neighbouring slabs' buffers; no exchange between
    steps.  Bitwise equal to the undivided run (whose parity with the oracle the test above and test_gpu_parity.py hold).
    The ghost planes of the contexts are poisoned first: nothing may read them."""
    import torch
    w = CASES[case](dtype)
    if not runs_on_tile(B, w):
        pytest.skip("gather-only lattice")
    steps = 7
    periodic_z = w.faces.get(W.FACE_ZLO, W.BC_PERIODIC) == W.BC_PERIODIC
    slabs = [S.Slab(w, p, B.KERNEL_TILE) for p in S.plan_slabs(w.nz, world, periodic_z)]
    for s in slabs:                                        # poison the ghost planes of the loaded state
        M = s.sim.export_state()[0]
        if s.plan.ghost_lo:
            M[:, 0] = float("nan")
        if s.plan.ghost_hi:
            M[:, -1] = float("nan")
        s.sim.import_state(M, 0)
    S.connect_local(slabs)
    l0 = sum(s.sim.launch_count for s in slabs)
    S.step_connected(slabs, steps)
    G = S.gather_local(slabs)
    torch.cuda.synchronize()
    one = make_gpu(w, B.KERNEL_TILE)
    one.step(steps)
    G1 = one.get_moments()
    assert torch.equal(G, G1), "max %.3e" % (G.double() - G1.double()).abs().max().item()
    # reloading a state detaches the neighbours; the gather kernel refuses to run with a neighbour attached
    S.connect_local(slabs)
    slabs[0].sim.set_kernel(B.KERNEL_GATHER)
    with pytest.raises(B.TSLBError):
        slabs[0].sim.step(1)
    one.close()
    for s in slabs:
        s.sim.close()


def runs_on_tile(B, w):
    return len(kernels_for(B, w)) == 2


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_thin_slabs_of_one_and_two_planes(B, oracle_mod, dtype):
    """The smallest slabs there are: one owned plane between two ghost planes (its low and its high export are the same
    plane), next to slabs of two; ragged split (the first ranks own one plane more); all three transports."""
    import torch
    cases = [(W.random_state(62, 13, 5, seed=71, dtype=dtype, tau=0.6), 4),                     # periodic: 2, 1, 1, 1 planes
             (with_faces(W.random_state(30, 16, 7, seed=72, dtype=dtype, tau=0.57), **BC_SETS["jet_like"]), 3)]   # 3, 2, 2
    for w, world in cases:
        steps = 5
        o = make_oracle(oracle_mod, w)
        o.step(steps)
        R = o.get_moments()
        one = make_gpu(w, B.KERNEL_TILE)
        one.step(steps)
        G1 = one.get_moments()
        for mode in ("staged", "in place", "connected"):
            periodic_z = w.faces.get(W.FACE_ZLO, W.BC_PERIODIC) == W.BC_PERIODIC
            slabs = [S.Slab(w, p, B.KERNEL_TILE, staged=(mode == "staged")) for p in S.plan_slabs(w.nz, world, periodic_z)]
            assert min(s.plan.owned for s in slabs) <= 2
            if mode == "connected":
                S.connect_local(slabs)
                S.step_connected(slabs, steps)
            else:
                S.step_local(slabs, steps)
            G = S.gather_local(slabs)
            assert torch.equal(G, G1), "%s, %s" % (w.name, mode)
            for s in slabs:
                s.sim.close()
        assert_parity(w, G1.cpu().numpy().astype(np.float64), R, "thin slabs")
        one.close()


def test_jet_with_inlet_noise_and_sponge_in_slabs(B, oracle_mod):
    """configs[3]'s own boundary set, reduced: the noisy inlet sits on the first slab, the sponge layer in the last one."""
    w = W.jet(24, 20, 40, steps=12, dtype="f32", D=6.0)
    w.sponge = (32, 1000.0, 3.0)
    o = make_oracle(oracle_mod, w)
    o.step(w.steps)
    R = o.get_moments()
    for world in (2, 3):
        slabs, G = run_slabs(w, world, w.steps, B.KERNEL_AUTO)
        assert_parity(w, G.astype(np.float64), R, "jet, %d slabs" % world)
        one = make_gpu(w, B.KERNEL_AUTO)
        one.step(w.steps)
        assert np.array_equal(G, one.get_moments().cpu().numpy())
        # the same with the neighbours read in place
        periodic_z = False
        slabs = [S.Slab(w, p, B.KERNEL_TILE) for p in S.plan_slabs(w.nz, world, periodic_z)]
        S.connect_local(slabs)
        S.step_connected(slabs, w.steps)
        assert np.array_equal(S.gather_local(slabs).cpu().numpy(), G)
        one.close()


@pytest.mark.parametrize("connected", [False, True])
def test_statistics_of_slabs_add_up_to_the_undivided_lattice(B, connected):
    """Plane sums on all three axes and the jet's (r, z)-ring sums: the slabs' contributions (ghost planes left out, which in
    the connected form hold whatever the sweep wrote there) against the undivided CUDA run, whose parity with the oracle
    test_gpu_parity.py holds."""
    import torch
    w = W.jet(24, 20, 40, steps=8, dtype="f32", D=6.0)
    one = make_gpu(w, B.KERNEL_AUTO)
    one.step(w.steps)
    slabs = [S.Slab(w, p, B.KERNEL_AUTO) for p in S.plan_slabs(w.nz, 3, False)]
    if connected:
        S.connect_local(slabs)
        S.step_connected(slabs, w.steps)
    else:
        S.step_local(slabs, w.steps)
    for axis, n in ((0, w.nx), (1, w.ny), (2, w.nz)):
        ref = one.plane_statistics(axis)
        tot = torch.zeros((13, n), dtype=torch.float64, device="cuda")
        for s in slabs:
            s.plane_statistics(axis, tot)
        assert torch.isfinite(tot).all()
        torch.testing.assert_close(tot, ref, rtol=1e-12, atol=1e-13)
        assert tot[0].sum().item() == w.sites                       # every node counted once
    xc, yc = (w.nx - 1) / 2.0, (w.ny - 1) / 2.0
    ref = one.radial_statistics(xc, yc, 1.5, 8)
    tot = torch.zeros_like(ref)
    for s in slabs:
        s.radial_statistics(xc, yc, 1.5, 8, tot)
    torch.testing.assert_close(tot, ref, rtol=1e-12, atol=1e-13)
    one.close()


def test_face_calls_reject_other_faces(B):
    w = W.random_state(16, 8, 9, seed=3, dtype="f32")
    s = S.Slab(w, S.plan_slabs(w.nz, 2, True)[0])
    with pytest.raises(B.TSLBError) as e:
        s.sim._chk(s.sim._lib.tslb_export_face(s.sim._h, B.FACE_XLO, 0x1000, None), "tslb_export_face")
    assert e.value.code == B.TSLB_EINVAL
    one = make_gpu(w, B.KERNEL_AUTO)                      # periodic z: not an EXCHANGE face
    with pytest.raises(B.TSLBError):
        one.export_face(B.FACE_ZLO)
    one.close()


IPC_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_2401_17074_b200 import binding as B, slab as S, workloads as W
rank, port, world, case = int(sys.argv[1]), sys.argv[2], int(sys.argv[3]), sys.argv[4]
torch.cuda.set_device(0)
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + port, rank=rank, world_size=world)
if case == "periodic":
    w = W.random_state(70, 27, 23, seed=61, dtype="f32", tau=0.58)
else:
    w = W.jet(24, 20, 40, steps=9, dtype="f32", D=6.0)
steps = 9
plan = S.plan_slabs(w.nz, world, case == "periodic")[rank]
s = S.Slab(w, plan, B.KERNEL_TILE, ipc=True)
M = s.sim.export_state()[0]                      # poison the ghost planes: nothing may read them
if plan.ghost_lo: M[:, 0] = float("nan")
if plan.ghost_hi: M[:, -1] = float("nan")
s.sim.import_state(M, 0)
S.connect_ipc(s)
l0 = s.sim.launch_count
S.step_connected_dist(s, steps)
G = s.owned_moments()
one = B.from_workload(w, B.KERNEL_TILE)
one.set_moments(torch.from_numpy(w.moments).to("cuda"))
one.step(steps)
G1 = one.get_moments()[:, plan.z_lo:plan.z_hi]
assert torch.equal(G, G1), (rank, (G.double() - G1.double()).abs().max().item())
S.disconnect_ipc(s)
dist.barrier(); dist.destroy_process_group()
print("ok", rank, "launches per step", (s.sim.launch_count - l0) / steps)
"""


@pytest.mark.parametrize("case,world", [("periodic", 2), ("periodic", 3), ("jet", 2)])
def test_ipc_connected_slabs_in_separate_processes(B, tmp_path, case, world):
    """One slab per PROCESS, all on this GPU: each maps its neighbours' workspaces through CUDA IPC (slab.connect_ipc), the tile
    kernel reads their planes in place, the processes meet at one host barrier per step (their kernels never wait on one
    another), and every rank's owned planes equal the undivided run bit for bit.  The path bench.py --slabs N --connected
    takes under torchrun, except that there the neighbour is another GPU and the barrier is a stream-ordered NCCL all-reduce."""
    import socket
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sk = socket.socket(); sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]; sk.close()
    script = tmp_path / "ipc_worker.py"
    script.write_text(IPC_WORKER % root)
    procs = [subprocess.Popen([sys.executable, str(script), str(r), str(port), str(world), case], stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT, text=True) for r in range(world)]
    outs = [p.communicate(timeout=600)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0 and "ok" in o, o

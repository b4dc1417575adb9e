"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element on identical
seeded inputs.  All tests need a B200: run with  pytest -m gpu  on the GPU box."""
import numpy as np
import pytest

from paper_2401_17074_b200 import workloads as W
from tests.parity_util import (TOL, assert_parity, errors, gpu_state, make_gpu, make_oracle, run_both, subbox)

pytestmark = pytest.mark.gpu

GATHER, TILE = 1, 2


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2401_17074_b200 import binding, build
    build.build_lib()
    binding.load_library()
    return binding


def kernels_for(B, w):
    """Every sweep kernel that covers this workload (the gather kernel covers everything)."""
    sim = B.from_workload(w, B.KERNEL_AUTO)
    ks = [GATHER] + ([TILE] if sim.active_kernel() == TILE else [])
    sim.close()
    return ks


def with_faces(w, faces, g=(0.0, 0.0, 0.0), inlet_face=None, seed=5):
    w.faces = dict(faces)
    w.g = g
    if inlet_face is not None:
        n = {0: (w.nz, w.ny), 1: (w.nz, w.nx), 2: (w.ny, w.nx)}[inlet_face // 2]
        up = np.random.default_rng(seed).uniform(-0.03, 0.03, (3,) + n).astype(w.np_dtype)
        w.inlet = W.Inlet(inlet_face, up, 0.05, 9, 0b111)
    return w


# ---------------------------------------------------------------------------------------------
# small cases: several tiles + ragged tails, every boundary kind, both dtypes, every kernel
# ---------------------------------------------------------------------------------------------
# (the tile kernel needs ny >= one tile height: 4 rows fp32 (small geometry), 8 rows fp64; smaller lattices run on the gather
#  kernel only)
SHAPES = [(3, 3, 3), (4, 3, 5), (5, 7, 9), (33, 17, 6), (64, 12, 10), (130, 9, 7), (136, 36, 5), (260, 20, 4),
          (61, 14, 5), (3, 29, 3), (124, 15, 33), (60, 28, 3), (59, 43, 4)]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", SHAPES)
def test_periodic_random_state(B, oracle_mod, shape, dtype):
    w = W.random_state(*shape, seed=31, dtype=dtype, tau=0.62)
    w.g = (1e-4, -2e-4, 3e-4)
    for k in kernels_for(B, w):
        G, R, _ = run_both(oracle_mod, w, 3, k)
        assert_parity(w, G, R, "kernel %d" % k)


BC_SETS = {
    "walls_y+force": dict(faces={W.FACE_YLO: W.BC_BOUNCE_BACK, W.FACE_YHI: W.BC_BOUNCE_BACK}, g=(2e-4, 0, 1e-4)),
    "walls_z": dict(faces={W.FACE_ZLO: W.BC_BOUNCE_BACK, W.FACE_ZHI: W.BC_BOUNCE_BACK}),
    "walls_x": dict(faces={W.FACE_XLO: W.BC_BOUNCE_BACK, W.FACE_XHI: W.BC_BOUNCE_BACK}, g=(0, 1e-4, 0)),
    "walls_xyz": dict(faces={f: W.BC_BOUNCE_BACK for f in range(6)}, g=(1e-4, 1e-4, -1e-4)),
    "walls_yz_duct": dict(faces={f: W.BC_BOUNCE_BACK for f in (2, 3, 4, 5)}, g=(2e-4, 1e-4, -1e-4)),
    "jet_like": dict(faces={W.FACE_ZLO: W.BC_VELOCITY_INLET, **{f: W.BC_OUTLET_ZERO_GRADIENT for f in (0, 1, 2, 3, 5)}},
                     inlet_face=W.FACE_ZLO),
    "inlet_x_walls_y": dict(faces={W.FACE_XLO: W.BC_VELOCITY_INLET, W.FACE_XHI: W.BC_OUTLET_ZERO_GRADIENT,
                                   W.FACE_YLO: W.BC_BOUNCE_BACK, W.FACE_YHI: W.BC_BOUNCE_BACK}, inlet_face=W.FACE_XLO,
                            g=(1e-4, 0, 0)),
    "outlet_y_walls_z": dict(faces={W.FACE_YLO: W.BC_OUTLET_ZERO_GRADIENT, W.FACE_YHI: W.BC_VELOCITY_INLET,
                                    W.FACE_ZLO: W.BC_BOUNCE_BACK, W.FACE_ZHI: W.BC_BOUNCE_BACK}, inlet_face=W.FACE_YHI),
    "mixed_wall_outlet_same_axis": dict(faces={W.FACE_ZLO: W.BC_BOUNCE_BACK, W.FACE_ZHI: W.BC_OUTLET_ZERO_GRADIENT}),
}


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("bc", sorted(BC_SETS))
@pytest.mark.parametrize("shape", [(4, 3, 5), (12, 10, 7), (136, 11, 6), (70, 16, 6), (65, 31, 5)])
def test_boundary_sets(B, oracle_mod, shape, bc, dtype):
    w = with_faces(W.random_state(*shape, seed=17, dtype=dtype, tau=0.58), **BC_SETS[bc])
    for k in kernels_for(B, w):
        G, R, _ = run_both(oracle_mod, w, 4, k)
        assert_parity(w, G, R, "%s kernel %d" % (bc, k))


# ---------------------------------------------------------------------------------------------
# BASELINE.json configs
# ---------------------------------------------------------------------------------------------
def test_config0_full(B, oracle_mod):
    """configs[0]: 32^3 fp64 Taylor-Green, tau = 0.8, 100 steps, max |d| <= 1e-12."""
    w = W.config0()
    for k in kernels_for(B, w):
        G, R, curve = run_both(oracle_mod, w, w.steps, k, checkpoints=[1, 10])
        e = assert_parity(w, G, R, "kernel %d" % k)
        print("config0 kernel %d: err(rho,u,Pi) = %s, curve %s" % (k, e, curve))
        assert abs(G[0].sum() - 32**3) < 1e-9                       # mass conserved


def test_config1_reduced_full_steps(B, oracle_mod):
    """configs[1] at 32^3: fp32, near-inviscid TG + noise, the full 1000 steps; parity curve logged."""
    w = W.config1(n=32, steps=1000)
    for k in kernels_for(B, w):
        G, R, curve = run_both(oracle_mod, w, w.steps, k, checkpoints=[1, 10, 100])
        print("config1@32 kernel %d curve (rho,u,Pi): %s" % (k, curve))
        assert_parity(w, G, R, "kernel %d" % k)
        assert np.abs(G[1:4]).max() < 0.1 and 0.9 < G[0].min() and G[0].max() < 1.1   # boundedness
        assert abs(G[0].astype(np.float64).sum() / 32**3 - 1) < 1e-6                   # mass


def test_config1_full_size_100_steps(B, oracle_mod):
    """configs[1] at its full 128^3: 100 steps element by element (the oracle needs ~minutes for 1000)."""
    w = W.config1()
    for k in kernels_for(B, w):
        G, R, curve = run_both(oracle_mod, w, 100, k, checkpoints=[1, 10])
        print("config1@128 kernel %d curve: %s" % (k, curve))
        assert_parity(w, G, R, "kernel %d" % k)


def test_config2_channel_reduced_full_steps(B, oracle_mod):
    """configs[2] with its own wall-normal size and parameters (ny = 128, h = 64, tau, g as in the full box) on a
    narrower 32 x 128 x 16 periodic cross-section: walls + body force, the full 2000 steps.  (A box with a smaller h
    has a smaller tau at the same Mach number and goes unstable in the oracle itself.)"""
    w = W.channel(32, 128, 16, steps=2000)
    for k in kernels_for(B, w):
        G, R, curve = run_both(oracle_mod, w, w.steps, k, checkpoints=[1, 10, 100, 1000])
        print("channel@32x128x16 kernel %d curve: %s" % (k, curve))
        assert_parity(w, G, R, "kernel %d" % k)


def test_config3_jet_reduced_full_steps(B, oracle_mod):
    """configs[3] shape at 32x32x96, D = 6: inlet with noise + outlets, the full 1000 steps."""
    w = W.jet(32, 32, 96, steps=1000, D=6.0)
    for k in kernels_for(B, w):
        G, R, curve = run_both(oracle_mod, w, w.steps, k, checkpoints=[1, 10, 100])
        print("jet@32x32x96 kernel %d curve: %s" % (k, curve))
        assert_parity(w, G, R, "kernel %d" % k)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config4_64cube_200_steps(B, oracle_mod, dtype):
    w = W.throughput(64, dtype, 200)
    for k in kernels_for(B, w):
        G, R, curve = run_both(oracle_mod, w, 200, k, checkpoints=[1, 10])
        print("throughput64 %s kernel %d curve: %s" % (dtype, k, curve))
        assert_parity(w, G, R, "kernel %d" % k)


# ---------------------------------------------------------------------------------------------
# full sizes, in the launch configuration bench.py times: sampled sub-boxes + invariants
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,dtype", [(512, "f32"), (256, "f64")])
def test_full_size_sampled_subboxes(B, oracle_mod, n, dtype):
    """Bench workload at full size: 3 GPU steps on the whole cube; the oracle recomputes sub-boxes cut from the
    SAME seeded initial state (never from GPU output) and the uncontaminated cores are compared."""
    import torch
    w = W.throughput(n, dtype, 3)
    sim = B.from_workload(w, B.KERNEL_AUTO)
    sim.set_moments(torch.from_numpy(w.moments).to("cuda"))
    sim.step(3)
    G = gpu_state(sim)
    k = 3
    for lo in [(0, 0, 0), (n - 9, n - 9, n - 9), (n // 2 - 3, 0, n - 5), (124, 250, 3)]:
        lo = [v - 4 for v in lo]                      # boxes straddle the periodic wrap and tile edges
        hi = [v + 16 for v in lo]
        s = subbox(w, lo, hi)
        o = make_oracle(oracle_mod, s); o.step(k)
        R = o.get_moments()
        ix = [np.arange(lo[a] + k, hi[a] - k) % n for a in range(3)]
        Gs = G[:, ix[2]][:, :, ix[1]][:, :, :, ix[0]]
        Rs = R[:, k:-k, k:-k, k:-k]
        s.nx = s.ny = s.nz = 16 - 2 * k
        assert_parity(s, Gs, Rs, "sub-box at %s" % (lo,))
    m = G[0].sum(dtype=np.float64)
    assert abs(m / n**3 - 1) < 1e-7
    sim.close()


def test_config2_full_size_20_steps(B, oracle_mod):
    """configs[2] at its full 384 x 128 x 192 in the launch configuration of the tile kernel: 20 steps element by
    element against the oracle (the full 2000 steps run on the reduced cross-section above), mass conserved."""
    w = W.channel(steps=20)
    G, R, curve = run_both(oracle_mod, w, 20, B.KERNEL_AUTO, checkpoints=[1])
    print("channel full size curve: %s" % curve)
    assert_parity(w, G, R, "full-size channel")
    assert abs(G[0].sum(dtype=np.float64) / w.sites - 1) < 1e-7


def test_config3_full_size_10_steps(B, oracle_mod):
    """configs[3] at its full 256 x 256 x 768: 10 steps element by element (inlet noise, outlets, fill kernel)."""
    w = W.jet(steps=10)
    G, R, curve = run_both(oracle_mod, w, 10, B.KERNEL_AUTO, checkpoints=[1])
    print("jet full size curve: %s" % curve)
    assert_parity(w, G, R, "full-size jet")
    assert 0.9 < G[0].min() and G[0].max() < 1.15


def test_kernel_switch_keeps_ghost_layers_valid(B, oracle_mod):
    """tile -> gather -> tile: the gather kernel does not maintain the ghost layers, the next tile step must refresh them."""
    for w in (W.config1(n=40, steps=9), with_faces(W.random_state(70, 20, 9, seed=3, dtype="f64", tau=0.6),
                                                     {W.FACE_YLO: W.BC_BOUNCE_BACK, W.FACE_YHI: W.BC_BOUNCE_BACK}, g=(1e-4, 0, 0))):
        o = make_oracle(oracle_mod, w); sim = make_gpu(w, TILE)
        for k, n in ((TILE, 3), (GATHER, 2), (TILE, 3), (GATHER, 1)):
            sim.set_kernel(k); sim.step(n); o.step(n)
        assert_parity(w, gpu_state(sim), o.get_moments(), "kernel switching")
        sim.close()


def test_set_moments_mid_run_and_timing_api(B, oracle_mod):
    """set_moments invalidates the ghost layers; tslb_set_timing / tslb_get_timing count the sweep launches."""
    import torch
    w = W.config1(n=36, steps=4)
    sim = make_gpu(w, B.KERNEL_AUTO)
    sim.step(3)
    sim.set_moments(torch.from_numpy(np.ascontiguousarray(w.moments)).to("cuda"))
    sim.set_timing(8)
    sim.step(4)
    n, ms = sim.get_timing()
    assert n == 4 and ms > 0.0
    assert sim.get_timing() == (0, 0.0)
    sim.set_timing(0)
    o = make_oracle(oracle_mod, w); o.step(4)
    assert_parity(w, gpu_state(sim), o.get_moments(), "after set_moments mid-run")


# ---------------------------------------------------------------------------------------------
# second-order variant (Eq. 8, tslb_set_order(2)): SURVEY.md 8(f) rank 2
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_order2_parity(B, oracle_mod, dtype):
    cases = [W.random_state(70, 21, 9, seed=12, dtype=dtype, tau=0.64),
             with_faces(W.random_state(66, 15, 7, seed=13, dtype=dtype, tau=0.6),
                        {W.FACE_YLO: W.BC_BOUNCE_BACK, W.FACE_YHI: W.BC_BOUNCE_BACK}, g=(2e-4, 0, -1e-4)),
             with_faces(W.random_state(12, 17, 14, seed=14, dtype=dtype, tau=0.58), **BC_SETS["jet_like"])]
    for w in cases:
        w.order = 2
        for k in kernels_for(B, w):
            G, R, _ = run_both(oracle_mod, w, 4, k)
            assert_parity(w, G, R, "order 2, kernel %d" % k)
            # and it is not the third-order result
            w3 = W.Workload(**{**w.__dict__, "order": 3})
            G3, _, _ = run_both(oracle_mod, w3, 4, k)
            assert np.abs(G3 - G).max() > 1e-9


def test_order2_config1_reduced(B, oracle_mod):
    """configs[1] inputs at 32^3, 300 steps, second-order reconstruction (near-inviscid: the case where the paper expects
    the higher order to matter for stability; here only parity and boundedness over a short run)."""
    w = W.config1(n=32, steps=300)
    w.order = 2
    for k in kernels_for(B, w):
        G, R, curve = run_both(oracle_mod, w, w.steps, k, checkpoints=[1, 100])
        print("config1@32 order 2 kernel %d curve: %s" % (k, curve))
        assert_parity(w, G, R, "order 2 kernel %d" % k)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_tile_kernel_is_bitwise_repeatable(B, dtype):
    """The sweep has no atomics and a fixed operation order: repeated runs from the same state must agree bit for bit.
    A run-to-run difference means a race between the warp roles (exchange slots, stage ring, output tiles, the store
    warp's boundary patches): 12 repetitions of 6 steps on lattices that exercise every instantiation family."""
    import torch
    cases = {"periodic": W.random_state(130, 38, 70, seed=71, dtype=dtype, tau=0.6),
             "small_geometry": W.random_state(64, 9, 24, seed=72, dtype=dtype, tau=0.6),
             "walls_y": with_faces(W.random_state(124, 37, 30, seed=73, dtype=dtype, tau=0.6), **BC_SETS["walls_y+force"]),
             "walls_z": with_faces(W.random_state(124, 37, 30, seed=74, dtype=dtype, tau=0.6), **BC_SETS["walls_z"]),
             "duct": with_faces(W.random_state(124, 37, 30, seed=77, dtype=dtype, tau=0.6), **BC_SETS["walls_yz_duct"]),
             "walls_x": with_faces(W.random_state(124, 37, 30, seed=78, dtype=dtype, tau=0.6), **BC_SETS["walls_x"]),
             "jet_fused": with_faces(W.random_state(124, 38, 30, seed=75, dtype=dtype, tau=0.6), **BC_SETS["jet_like"]),
             "inlet_x_walls_y": with_faces(W.random_state(124, 37, 30, seed=76, dtype=dtype, tau=0.6), **BC_SETS["inlet_x_walls_y"])}
    for name, w in cases.items():
        ref = None
        for rep in range(12):
            sim = make_gpu(w, TILE)
            assert sim.active_kernel() == TILE, name
            sim.step(6)
            G = sim.get_moments()
            torch.cuda.synchronize()
            if ref is None:
                ref = G.clone()
                assert torch.isfinite(ref).all(), name
            else:
                assert torch.equal(G, ref), "%s: run %d differs from run 0 in %d values" % (name, rep, int((G != ref).sum()))
            sim.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_z_walls_and_sponge_across_z_chunks(B, oracle_mod, dtype):
    """Lattices longer than one z chunk (64 planes): the wall planes sit in the first and the last chunk only, the sponge
    table is indexed with the source plane of every chunk; z walls also next to open faces and with a body force."""
    wz = with_faces(W.random_state(70, 26, 150, seed=81, dtype=dtype, tau=0.6), **BC_SETS["walls_z"])
    wz.g = (1e-4, -1e-4, 2e-4)
    wo = with_faces(W.random_state(66, 25, 140, seed=82, dtype=dtype, tau=0.58), **BC_SETS["outlet_y_walls_z"])
    wm = with_faces(W.random_state(30, 13, 135, seed=83, dtype=dtype, tau=0.58), **BC_SETS["mixed_wall_outlet_same_axis"])
    wd = with_faces(W.random_state(64, 27, 130, seed=85, dtype=dtype, tau=0.6), **BC_SETS["walls_yz_duct"])
    ws = W.random_state(40, 20, 150, seed=84, dtype=dtype, tau=0.54)
    ws.sponge = (100, 1000.0, 3.0)
    wx = with_faces(W.random_state(130, 26, 70, seed=86, dtype=dtype, tau=0.6), **BC_SETS["walls_x"])
    wx.g = (1e-4, 2e-4, -1e-4)
    for w in (wz, wo, wm, wd, wx, ws):
        ks = kernels_for(B, w)
        assert TILE in ks, w.name
        G, R, _ = run_both(oracle_mod, w, 4, TILE)
        assert_parity(w, G, R, "%s tile" % w.name)


def test_which_boundary_sets_run_on_the_tile_kernel(B):
    """Bounce-back walls on the y faces or on the z faces (also next to open faces) run on the tile kernel; walls on x or on
    two axes fall back to the gather kernel."""
    want = {"walls_y+force": TILE, "walls_z": TILE, "walls_yz_duct": TILE, "walls_x": TILE, "walls_xyz": GATHER, "jet_like": TILE,
            "inlet_x_walls_y": TILE, "outlet_y_walls_z": TILE, "mixed_wall_outlet_same_axis": TILE}
    for name, k in want.items():
        w = with_faces(W.random_state(70, 31, 12, seed=3, dtype="f32", tau=0.6), **BC_SETS[name])
        sim = B.from_workload(w, B.KERNEL_AUTO)
        assert sim.active_kernel() == k, name
        sim.close()


def test_open_faces_are_filled_inside_the_sweep(B, oracle_mod):
    """north_star: 'boundary and forcing kernels fused into the same sweep'.  On the jet boundary set the tile kernel's
    store warp writes the boundary nodes of time t+1 itself: one launch per step once the first fill has run, and the
    boundary nodes it wrote are exactly what the oracle's fill gives (inlet with noise, outlets, edges and corners)."""
    w = W.jet(64, 48, 40, steps=6, D=12.0)
    sim = make_gpu(w, TILE)
    assert sim.active_kernel() == TILE
    sim.step(1)
    n0 = sim.launch_count
    sim.step(5)
    assert sim.launch_count - n0 == 5, "open faces cost extra launches: %d for 5 steps" % (sim.launch_count - n0)
    G = gpu_state(sim)
    o = make_oracle(oracle_mod, w); o.step(6)
    R = o.get_moments()
    assert_parity(w, G, R, "fused fill")
    # boundary nodes (get_moments does not have to refill them: the sweep's own fill is current)
    for ax, idx in ((1, 0), (1, -1), (2, 0), (2, -1), (3, 0), (3, -1)):
        g = np.take(G, idx, axis=ax).astype(np.float64); r = np.take(R, idx, axis=ax)
        assert np.abs(g[0] - r[0]).max() < 1e-6 and np.abs(g[1:4] - r[1:4]).max() < 1e-6 * max(1e-30, np.abs(R[1:4]).max()) + 1e-8
    sim.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_boundary_variants_of_section_IIC(B, oracle_mod, dtype):
    """pressure (density-imposed) outlet, NEQ no-slip walls (zero-velocity Dirichlet nodes on the
    faces) and the Gaussian inlet noise, on lattices that span several tiles, both kernels."""
    def jet_pressure(shape, seed):
        w = with_faces(W.random_state(*shape, seed=seed, dtype=dtype, tau=0.56), **BC_SETS["jet_like"])
        w.faces[W.FACE_ZHI] = W.BC_OUTLET_PRESSURE
        w.rho_out = {W.FACE_ZHI: 0.98}
        w.inlet.noise_mask |= W.NOISE_GAUSSIAN
        return w
    def neq_walls(shape, seed):
        w = W.random_state(*shape, seed=seed, dtype=dtype, tau=0.6)
        w.faces = {W.FACE_YLO: W.BC_VELOCITY_INLET, W.FACE_YHI: W.BC_OUTLET_PRESSURE}
        w.rho_out = {W.FACE_YHI: 1.01}
        w.g = (1e-4, 0.0, 0.0)
        w.inlet = W.Inlet(W.FACE_YLO, np.zeros((3, w.nz, w.nx), dtype=w.np_dtype), 0.0, 0, 0)
        return w
    for w in (jet_pressure((24, 17, 12), 61), jet_pressure((70, 30, 9), 62), neq_walls((66, 15, 7), 63)):
        for k in kernels_for(B, w):
            G, R, _ = run_both(oracle_mod, w, 5, k)
            assert_parity(w, G, R, "%s kernel %d" % (w.name, k))
            # boundary nodes themselves (get_moments refills them): imposed density / zero wall velocity, exactly
            for f, rho in w.rho_out.items():
                sl = [slice(None)] * 3
                sl[2 - f // 2] = -1 if f % 2 else 0
                assert np.abs(G[(0,) + tuple(sl)] - rho).max() <= (2e-7 if dtype == "f32" else 3e-16)   # one rounding of rho - 1


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_radial_statistics_match_oracle(B, oracle_mod, dtype):
    """(r, z)-bin sums of the jet (tslb_radial_statistics) against the oracle after a few steps of the jet boundary set:
    ring counts bit-exact (the ring index is an integer both sides decide in fp64), sums to 1e-12 relative in fp64 /
    to the state's own parity in fp32; off-centre axis, rings that leave the box, two samples accumulate."""
    w = with_faces(W.random_state(45, 38, 12, seed=51, dtype=dtype, tau=0.6), **BC_SETS["jet_like"])
    nr, dr, xc, yc = 9, 2.5, 21.3, 18.0
    o = make_oracle(oracle_mod, w)
    S = np.zeros((8, w.nz, nr))
    for k in kernels_for(B, w)[-1:]:
        sim = make_gpu(w, k)
        G = None
        for n in (0, 3):
            sim.step(n); o.step(n)
            G = sim.radial_statistics(xc, yc, dr, nr, G)
            o.radial_statistics(xc, yc, dr, nr, S)
        Gh = G.cpu().numpy()
        assert np.array_equal(Gh[0], S[0])
        assert S[0].sum() > 0 and S[0, :, -1].min() > 0
        tol = 1e-12 if dtype == "f64" else 2e-5
        scale = np.abs(S).max(axis=(1, 2), keepdims=True)
        assert (np.abs(Gh - S) / scale).max() < tol, (np.abs(Gh - S) / scale).max()
        sim.close()


# ---------------------------------------------------------------------------------------------
# sponge layer (Eq. 26, tslb_set_sponge): SURVEY.md 8(f) rank 3
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_sponge_parity(B, oracle_mod, dtype):
    """Per-plane relaxation time along z in both kernels: periodic box (the layer wraps around), channel walls, and the jet
    set (inlet at z = 0, outlets elsewhere) with the paper's K = 1000, p = 3 on a layer of 10 planes; several z chunks and
    tiles.  Also: K = 0 is bit-identical to no layer."""
    cases = [W.random_state(70, 27, 40, seed=41, dtype=dtype, tau=0.56),
             with_faces(W.random_state(66, 15, 21, seed=42, dtype=dtype, tau=0.6),
                        {W.FACE_YLO: W.BC_BOUNCE_BACK, W.FACE_YHI: W.BC_BOUNCE_BACK}, g=(2e-4, 0, -1e-4)),
             with_faces(W.random_state(24, 17, 30, seed=43, dtype=dtype, tau=0.52), **BC_SETS["jet_like"])]
    for w, sp in zip(cases, [(25, 40.0, 3.0), (9, 1000.0, 3.0), (20, 1000.0, 3.0)]):
        w.sponge = sp
        for k in kernels_for(B, w):
            G, R, _ = run_both(oracle_mod, w, 5, k)
            assert_parity(w, G, R, "sponge, kernel %d" % k)
            w0 = W.Workload(**{**w.__dict__, "sponge": None})
            G0, _, _ = run_both(oracle_mod, w0, 5, k)
            assert np.abs(G0 - G).max() > 1e-7                 # the layer changes the result
            wk0 = W.Workload(**{**w.__dict__, "sponge": (sp[0], 0.0, 3.0)})
            Gk0, _, _ = run_both(oracle_mod, wk0, 5, k)
            assert np.array_equal(Gk0, G0)


# ---------------------------------------------------------------------------------------------
# plane statistics (Eq. 24-25 raw sums, tslb_plane_statistics): SURVEY.md 8(f) rank 1
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_plane_statistics_match_oracle(B, oracle_mod, dtype):
    import torch
    for w, axis in ((W.channel(40, 24, 18, steps=30, dtype=dtype), 1), (W.jet(16, 20, 24, steps=30, dtype=dtype, D=5.0), 2),
                    (W.config1(n=24, steps=30, dtype=dtype), 0)):
        o = make_oracle(oracle_mod, w); sim = make_gpu(w, B.KERNEL_AUTO)
        n_axis = (w.nx, w.ny, w.nz)[axis]
        So = np.zeros((13, n_axis)); Sg = None
        for _ in range(3):                                # three samples, 10 steps apart
            o.step(10); sim.step(10)
            o.plane_statistics(axis, So); Sg = sim.plane_statistics(axis, Sg)
        torch.cuda.synchronize()
        G = Sg.cpu().numpy()
        tol = 1e-12 if dtype == "f64" else 2e-5
        # a plane sum of u^k is compared relative to (number of samples in the sum) x max|u|^k (the sums themselves may cancel)
        umax = np.abs(o.get_moments()[1:4]).max()
        power = np.array([0, 1, 1, 1, 2, 2, 2, 2, 2, 2, 3, 3, 3])[:, None]
        scale = So[0].max() * umax ** power
        assert np.array_equal(G[0], So[0])                # sample counts are exact
        assert (np.abs(G - So) / scale).max() < tol, (w.name, (np.abs(G - So) / scale).max())
        # fixed-order reduction: a second context gives the same bits
        sim2 = make_gpu(w, B.KERNEL_AUTO); S2 = None
        for _ in range(3):
            sim2.step(10); S2 = sim2.plane_statistics(axis, S2)
        assert torch.equal(Sg, S2)
        # Reynolds stress <u'x u'y> and variance from the raw sums against numpy on the GPU state itself
        M = gpu_state(sim)
        one = sim.plane_statistics(axis).cpu().numpy()
        ax_np = {0: (0, 1), 1: (0, 2), 2: (1, 2)}[axis]   # axes of [nz][ny][nx] to average over
        mean = one[1:4] / one[0]
        var = one[4:7] / one[0] - mean**2
        assert np.abs(var - M[1:4].var(axis=tuple(a + 1 for a in ax_np))).max() < 1e-9
        sim.close(); sim2.close()


# ---------------------------------------------------------------------------------------------
# library behaviour on the device
# ---------------------------------------------------------------------------------------------
def test_checkpoint_resume(B):
    """tslb_export_state / tslb_import_state is the bit-exact checkpoint: run 2n == run n, export,
    import, run n -- bitwise, on every kernel, with inlet noise (the step counter is part of the state).  The rho-valued
    get_moments / set_moments pair rounds drho once to the ulp of rho.  A rerun is bitwise reproducible."""
    import torch
    for w in (W.config1(n=32, steps=20), W.jet(16, 16, 24, steps=20, D=5.0), W.channel(32, 16, 12, steps=20)):
        for k in kernels_for(B, w):
            a = make_gpu(w, k); a.step(20); Ga = a.get_moments().clone(); Sa, ta = a.export_state()
            b = make_gpu(w, k); b.step(10); S, t = b.export_state(); S = S.clone()
            assert t == 10 and ta == 20
            c = B.from_workload(w, k); c.import_state(S, t); c.step(10)
            Sc, tc = c.export_state()
            torch.cuda.synchronize()
            assert tc == 20 and torch.equal(Sa, Sc), (w.name, k)              # bitwise, counter restored
            assert torch.equal(Ga, c.get_moments())
            # the rho-valued pair: one rounding of drho
            mid = b.get_moments().clone()
            d = make_gpu(w, k); d.set_moments(mid); d.step(10); Gd = d.get_moments()
            if w.inlet is None:                                                  # (set_moments restarts the noise counter)
                assert (Ga[0] - Gd[0]).abs().max().item() <= 4e-7 and (Ga[1:4] - Gd[1:4]).abs().max().item() <= 2e-6
            a2 = make_gpu(w, k); a2.step(20)
            assert torch.equal(Ga, a2.get_moments())                            # rerun is bitwise reproducible
            for s_ in (a, b, c, d, a2):
                s_.close()


def test_diagnostics_match_oracle(B, oracle_mod):
    import torch
    for w in (W.channel(24, 16, 12, steps=30, dtype="f64"), W.jet(16, 16, 24, steps=30, dtype="f32", D=5.0)):
        o = make_oracle(oracle_mod, w); sim = make_gpu(w, B.KERNEL_AUTO)
        o.step(30); sim.step(30)
        d = sim.diagnostics(); torch.cuda.synchronize()
        d = d.cpu().numpy(); r = o.diagnostics()
        tol = 1e-12 if w.dtype == "f64" else 1e-5
        assert abs(d[0] / r[0] - 1) < tol
        np.testing.assert_allclose(d[1:], r[1:], rtol=tol * 10, atol=tol * abs(r[0]) * 1e-2)
        d2 = sim.diagnostics().cpu().numpy()
        np.testing.assert_array_equal(d, d2)           # fixed-order reduction


def test_host_buffer_round_trip(B, oracle_mod):
    """tslb_set_moments_host / tslb_get_moments_host (the e2e path of bench.py).  The export is staged in the stale
    ping-pong buffer, which overwrites its pad cells and ghost columns with caller data: periodic, wall and open-face
    lattices, both kernels, must still step correctly afterwards."""
    cases = [W.random_state(20, 9, 7, seed=2, dtype="f32"),
             with_faces(W.random_state(70, 16, 6, seed=3, dtype="f32", tau=0.58), **BC_SETS["walls_y+force"]),
             with_faces(W.random_state(64, 17, 9, seed=4, dtype="f64", tau=0.58), **BC_SETS["jet_like"]),
             with_faces(W.random_state(61, 15, 6, seed=5, dtype="f32", tau=0.58), **BC_SETS["inlet_x_walls_y"])]
    for w in cases:
        for k in kernels_for(B, w):
            sim = B.from_workload(w, k)
            sim.set_moments_host(np.ascontiguousarray(w.moments))
            out = np.empty_like(w.moments)
            sim.get_moments_host(out)
            o = make_oracle(oracle_mod, w)
            # (boundary nodes refilled on both sides; an imposed fp32 inlet velocity is rounded once)
            np.testing.assert_allclose(out.astype(np.float64), o.get_moments(), rtol=0, atol=0 if w.inlet is None else 1e-8)
            sim.step(2)
            sim.get_moments_host(out)          # staging between steps
            sim.step(2)
            sim.get_moments_host(out)
            o.step(4)
            assert_parity(w, out.astype(np.float64), o.get_moments(), "host round trip, kernel %d" % k)
            sim.close()


def test_step_errors_on_device(B):
    w = W.random_state(8, 8, 8, dtype="f64")
    sim = B.from_workload(w)
    with pytest.raises(B.TSLBError) as e:
        sim.step(1)
    assert e.value.code == B.TSLB_ESTATE
    sim = make_gpu(w, B.KERNEL_AUTO)
    with pytest.raises(B.TSLBError):
        sim.step(-1)
    sim.set_boundary(B.FACE_XLO, B.BC_BOUNCE_BACK)      # periodic on XHI only -> inconsistent
    with pytest.raises(B.TSLBError) as e:
        sim.step(1)
    assert e.value.code == B.TSLB_EINVAL

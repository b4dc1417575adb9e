"""tslb_plane_statistics_static: the allocation-free variant of the plane statistics (scratch in a file-scope device array
of the library, include/tslb.h) against the existing path tslb_plane_statistics (scratch in the caller's workspace).

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other tests:
it depends on nothing but its own contexts, and the static array needs no initial contents.
"""
import numpy as np
import pytest

from paper_2401_17074_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2401_17074_b200 import binding, build
    build.build_lib()
    binding.load_library()
    return binding


def _sim(B, w):
    import torch
    sim = B.from_workload(w, B.KERNEL_AUTO)
    sim.set_moments(torch.from_numpy(np.ascontiguousarray(w.moments)).to("cuda"))
    return sim


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_static_scratch_matches_the_workspace_path_on_two_calls_in_a_row(B, dtype):
    """Two calls in a row on the shared static array -- first the long axis (fills 13 x 70 x 8 entries), then a shorter one
    (must not see what the first call left behind) -- and a second sample that accumulates, each against the existing
    path on the same state.  Same kernels and summation order, so the bar is the tightest one: bitwise equality (the
    suite's fp64 tolerance is 1e-12)."""
    import torch
    w = W.random_state(45, 38, 70, seed=91, dtype=dtype, tau=0.6)
    w.faces = {W.FACE_ZLO: W.BC_VELOCITY_INLET, **{f: W.BC_OUTLET_ZERO_GRADIENT for f in (0, 1, 2, 3, 5)}}
    up = np.random.default_rng(5).uniform(-0.03, 0.03, (3, w.ny, w.nx)).astype(w.np_dtype)
    w.inlet = W.Inlet(W.FACE_ZLO, up, 0.05, 9, 0b111)
    sim = _sim(B, w)
    sim.step(3)
    for axis in (2, 0, 1):                                   # consecutive calls: n_axis = 70, 45, 38
        n_axis = sim.shape[2 - axis]
        ref = sim.plane_statistics(axis)                     # existing path
        got = torch.zeros((13, n_axis), dtype=torch.float64, device="cuda")
        sim.plane_statistics_static(axis, got)               # new entry point, call 1
        torch.cuda.synchronize()
        assert torch.isfinite(got).all() and float(got[0].sum()) == w.sites
        assert torch.equal(got, ref), (axis, float((got - ref).abs().max()))
        sim.step(2)                                          # a second sample at a later time: the sums accumulate
        sim.plane_statistics(axis, ref)
        sim.plane_statistics_static(axis, got)               # call 2, same array
        torch.cuda.synchronize()
        assert torch.equal(got, ref), (axis, float((got - ref).abs().max()))
        assert np.abs((got - ref).cpu().numpy()).max() <= 1e-12 * max(1.0, float(ref.abs().max()))
    sim.close()


def test_static_scratch_is_shared_between_contexts_and_rejects_long_axes(B):
    """A second context uses the same array right after the first (stream-ordered: no race); an axis longer than the
    stated maximum is refused with a clear error instead of overrunning the array."""
    import torch
    wa = W.random_state(33, 17, 24, seed=92, dtype="f32", tau=0.6)
    wb = W.random_state(20, 40, 9, seed=93, dtype="f64", tau=0.7)
    sa, sb = _sim(B, wa), _sim(B, wb)
    for sim in (sa, sb, sa):
        for axis in (0, 1, 2):
            got = torch.zeros((13, sim.shape[2 - axis]), dtype=torch.float64, device="cuda")
            sim.plane_statistics_static(axis, got)
            assert torch.equal(got, sim.plane_statistics(axis)), axis
    sa.close(); sb.close()
    n = B.PLANE_STATISTICS_STATIC_MAX + 1
    wl = W.random_state(n, 4, 3, seed=94, dtype="f32", tau=0.6)
    sl = _sim(B, wl)
    with pytest.raises(B.TSLBError) as ei:
        sl.plane_statistics_static(0, torch.zeros((13, n), dtype=torch.float64, device="cuda"))
    assert ei.value.code == 1 and "static scratch holds %d" % B.PLANE_STATISTICS_STATIC_MAX in str(ei.value)
    ok = torch.zeros((13, 4), dtype=torch.float64, device="cuda")          # the short axes of the same lattice still work
    sl.plane_statistics_static(1, ok)
    assert torch.equal(ok, sl.plane_statistics(1))
    sl.close()

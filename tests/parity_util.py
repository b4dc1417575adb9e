"""Shared helpers of the GPU parity tests: drive the CUDA path (through the C ABI binding) and the CPU
oracle on the same seeded workload and compare element by element.

Tolerances (BASELINE.json north_star, reading A19):
  fp64: max |d rho|, max |d u|  <= 1e-12 (absolute)
  fp32: max |d rho| / max |rho_oracle|  and  max |d u| / max |u_oracle|  <= 2e-5
  Pi_neq: <= 1e-12 absolute (fp64), <= 1e-3 of max |Pi_oracle| (fp32)
over the nodes that are not on an open face (those are imposed, not computed).
"""
import numpy as np

from paper_2401_17074_b200 import workloads as W

TOL = {"f64": 1e-12, "f32": 2e-5}
# Pi_neq (six of the ten stored fields; north_star names rho and u only): rebuilt from scratch every step, so its error does
# not accumulate -- absolute for f64, relative to max|Pi_oracle| for f32
TOL_PI = {"f64": 1e-12, "f32": 1e-3}


def make_oracle(oracle_mod, w):
    o = oracle_mod.Oracle(w.nx, w.ny, w.nz, w.tau)
    for f, k in w.faces.items():
        if w.inlet is not None and f == w.inlet.face:
            o.set_face(f, k, w.inlet.u_plane, w.inlet.noise_amp, w.inlet.seed, w.inlet.noise_mask)
        elif k == 5:                       # BC_OUTLET_PRESSURE
            o.set_pressure_outlet(f, w.rho_out[f])
        else:
            o.set_face(f, k)
    o.set_force(w.g)
    if getattr(w, "order", 3) != 3:
        o.set_order(w.order)
    if getattr(w, "sponge", None):
        o.set_sponge(*w.sponge)
    o.set_moments(w.moments)          # the run-dtype array, converted exactly to fp64
    return o


def make_gpu(w, kernel):
    import torch
    from paper_2401_17074_b200 import binding as B
    sim = B.from_workload(w, kernel)
    sim.set_moments(torch.from_numpy(np.ascontiguousarray(w.moments)).to("cuda"))
    return sim


def gpu_state(sim):
    import torch
    out = sim.get_moments()
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def interior_mask(w):
    m = np.ones((w.nz, w.ny, w.nx), dtype=bool)
    open_kinds = (W.BC_VELOCITY_INLET, W.BC_OUTLET_ZERO_GRADIENT)
    sl = {W.FACE_XLO: (slice(None), slice(None), 0), W.FACE_XHI: (slice(None), slice(None), -1),
          W.FACE_YLO: (slice(None), 0, slice(None)), W.FACE_YHI: (slice(None), -1, slice(None)),
          W.FACE_ZLO: (0, slice(None), slice(None)), W.FACE_ZHI: (-1, slice(None), slice(None))}
    for f, k in w.faces.items():
        if k in open_kinds:
            m[sl[f]] = False
    return m


def errors(w, G, R):
    """(err_rho, err_u, err_pi) in the metric of the dtype: absolute for f64, relative (A19) for f32."""
    m = interior_mask(w)
    d_rho = np.abs(G[0] - R[0])[m].max()
    d_u = max(np.abs(G[k] - R[k])[m].max() for k in (1, 2, 3))
    d_pi = max(np.abs(G[k] - R[k])[m].max() for k in range(4, 10))
    if w.dtype == "f32":
        s_u = max(np.abs(R[k])[m].max() for k in (1, 2, 3))
        s_pi = max(np.abs(R[k])[m].max() for k in range(4, 10))
        return d_rho / np.abs(R[0])[m].max(), d_u / max(s_u, 1e-30), d_pi / max(s_pi, 1e-30)
    return d_rho, d_u, d_pi


def assert_parity(w, G, R, what="", tol=None):
    assert np.isfinite(G).all(), "non-finite GPU moments " + what
    e_rho, e_u, e_pi = errors(w, G, R)
    t = TOL[w.dtype] if tol is None else tol
    assert e_rho <= t and e_u <= t, "%s %s: err rho %.3e, u %.3e (Pi %.3e) > %.1e" % (w.name, what, e_rho, e_u, e_pi, t)
    if tol is None:
        assert e_pi <= TOL_PI[w.dtype], "%s %s: err Pi %.3e > %.1e" % (w.name, what, e_pi, TOL_PI[w.dtype])
    # boundary nodes are imposed values: they must agree to storage rounding
    m = ~interior_mask(w)
    if m.any():
        lim = 1e-14 if w.dtype == "f64" else 2e-7
        for k in range(10):
            assert np.abs(G[k] - R[k])[m].max() <= lim * max(1.0, np.abs(R[k])[m].max()), "boundary node field %d" % k
    return e_rho, e_u, e_pi


def run_both(oracle_mod, w, steps, kernel, checkpoints=None):
    """Advance both sides `steps` steps; returns (G, R) and, for each checkpoint step, the error triple."""
    o = make_oracle(oracle_mod, w)
    sim = make_gpu(w, kernel)
    curve = {}
    done = 0
    for cp in sorted(set(checkpoints or []) | {steps}):
        sim.step(cp - done); o.step(cp - done); done = cp
        G, R = gpu_state(sim), o.get_moments()
        curve[cp] = errors(w, G, R)
    assert sim.step_count == steps == o.step_count
    sim.close()
    return G, R, curve


def subbox(w, lo, hi):
    """Periodic-wrapped sub-box [lo, hi) of a periodic workload as a fresh periodic workload (its edges are
    contaminated by the artificial wrap; compare only nodes >= k nodes inside after k steps)."""
    ix = [np.arange(lo[a], hi[a]) % n for a, n in enumerate((w.nx, w.ny, w.nz))]
    M = w.moments[:, ix[2]][:, :, ix[1]][:, :, :, ix[0]]
    return W.Workload(w.name + "_sub", len(ix[0]), len(ix[1]), len(ix[2]), w.dtype, w.tau, 0,
                      np.ascontiguousarray(M), faces={}, g=w.g)

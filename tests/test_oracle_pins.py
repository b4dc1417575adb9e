"""Pins of the CPU oracle against what the paper and the mathematics fix (all -m "not gpu").

Each test names the passage of PAPER.md (arXiv 2401.17074) or the DESIGN.md reading it pins.
Nothing here is produced by the CUDA path.
"""
import itertools
import os

import numpy as np
import pytest

from paper_2401_17074_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
CS2 = 1.0 / 3.0
DIRS = [(cx, cy, cz) for cz in (-1, 0, 1) for cy in (-1, 0, 1) for cx in (-1, 0, 1)]


def rand_M(rng, amp_u=0.1, amp_pi=0.01):
    M = np.empty(10)
    M[0] = 1.0 + rng.uniform(-0.2, 0.2)
    M[1:4] = rng.uniform(-amp_u, amp_u, 3)
    M[4:10] = rng.uniform(-amp_pi, amp_pi, 6)
    return M


def Pi_of(M):
    return np.array([[M[4], M[7], M[8]], [M[7], M[5], M[9]], [M[8], M[9], M[6]]])


# ---------------------------------------------------------------------------------------------
# P1 / P2: moment reproduction.  Pins w_i, H2, H3, the 1/(n! cs^2n) prefactors, readings A1-A4, A6.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", [0, 1])
def test_P1_moments_order_0_1_2(oracle_mod, mode):
    """sum f* = rho; sum c f* = rho u (+ rho g); sum cc f* = rho cs2 I + rho uu + (1-w) Pi.
    (PAPER.md:45 'linear and local summations', Eq. 12, Eq. 14, Eq. 17)"""
    rng = np.random.default_rng(11)
    for _ in range(20):
        M = rand_M(rng)
        omega = rng.uniform(0.3, 1.99)
        g = rng.uniform(-1e-3, 1e-3, 3) if _ % 2 else np.zeros(3)
        rho, u, Pi = M[0], M[1:4], Pi_of(M)
        f = np.array([oracle_mod.fstar(M, c, omega, g, mode) for c in DIRS])
        c = np.array(DIRS, dtype=float)
        assert abs(f.sum() - rho) < 1e-15 * 4
        np.testing.assert_allclose(c.T @ f, rho * (u + g), atol=5e-16)
        S = np.einsum("i,ia,ib->ab", f, c, c)
        np.testing.assert_allclose(S, rho * CS2 * np.eye(3) + rho * np.outer(u, u) + (1 - omega) * Pi, atol=5e-16)


@pytest.mark.parametrize("mode", [0, 1])
def test_P2_third_moments(oracle_mod, mode):
    """sum c_a c_b c_g f* = rho u_a u_b u_g + (1-w) a3_abg + cs2 rho (u_a d_bg + u_b d_ag + u_g d_ab)
    for every index triple except a=b=g (H3_aaa = 0 on this lattice).  Pins H3, 1/(6 cs^6), the
    three-term symmetrised a3 of Eq. 17 (reading A4) and 'third-order equilibrium term once' (A1).
    (PAPER.md:140 Eq. 15, :150 Eq. 17)"""
    rng = np.random.default_rng(12)
    d = np.eye(3)
    for _ in range(10):
        M = rand_M(rng)
        omega = rng.uniform(0.3, 1.99)
        rho, u, Pi = M[0], M[1:4], Pi_of(M)
        f = np.array([oracle_mod.fstar(M, c, omega, (0, 0, 0), mode) for c in DIRS])
        c = np.array(DIRS, dtype=float)
        Q = np.einsum("i,ia,ib,ig->abg", f, c, c, c)
        a3 = (np.einsum("ab,g->abg", Pi, u) + np.einsum("a,bg->abg", u, Pi) + np.einsum("b,ag->abg", u, Pi))
        want = (rho * np.einsum("a,b,g->abg", u, u, u) + (1 - omega) * a3
                + CS2 * rho * (np.einsum("a,bg->abg", u, d) + np.einsum("b,ag->abg", u, d) + np.einsum("g,ab->abg", u, d)))
        for a, b, g in itertools.product(range(3), repeat=3):
            if a == b == g:
                # the lattice cannot carry c^3: sum c_a^3 f = sum c_a f
                assert abs(Q[a, a, a] - rho * u[a]) < 1e-15
            else:
                assert abs(Q[a, b, g] - want[a, b, g]) < 1e-16 * 5, (a, b, g)


def test_P2b_dropped_terms_would_fail(oracle_mod):
    """Sensitivity check of P1/P2: a second-order-only population (Eq. 8) misses the third moment."""
    M = np.array([1.1, 0.1, -0.07, 0.05, 0, 0, 0, 0, 0, 0])
    c = np.array(DIRS, dtype=float)
    f = np.array([oracle_mod.fstar(M, ci, 1.0, (0, 0, 0), 1) for ci in DIRS])
    w = np.array([np.prod([2 / 3 if k == 0 else 1 / 6 for k in ci]) for ci in DIRS])
    cu = c @ M[1:4]
    f2 = w * M[0] * (1 + 3 * cu + 4.5 * cu * cu - 1.5 * (M[1:4] @ M[1:4]))      # Eq. 2
    Q3 = np.einsum("i,i,i,i->", f, c[:, 0], c[:, 0], c[:, 1])
    Q2 = np.einsum("i,i,i,i->", f2, c[:, 0], c[:, 0], c[:, 1])
    want = M[0] * M[1] ** 2 * M[2] + CS2 * M[0] * M[2]
    assert abs(Q3 - want) < 1e-16 and abs(Q2 - want) > 1e-4


def test_tau1_is_pure_equilibrium(oracle_mod):
    """omega = 1: f* = f_eq, independent of Pi (Eq. 5)."""
    rng = np.random.default_rng(3)
    M = rand_M(rng)
    M0 = M.copy(); M0[4:] = 0
    for c in DIRS:
        assert oracle_mod.fstar(M, c, 1.0) == oracle_mod.fstar(M0, c, 1.0)


def test_rest_state_weights(oracle_mod):
    """rho = 1, u = 0, Pi = 0: f*_i = w_i, the D3Q27 weights 8/27, 2/27, 1/54, 1/216 by shell (Fig. 2)."""
    M = np.zeros(10); M[0] = 1
    shell = {0: 8 / 27, 1: 2 / 27, 2: 1 / 54, 3: 1 / 216}
    for c in DIRS:
        assert abs(oracle_mod.fstar(M, c, 0.7, (0, 0, 0), 0) - shell[sum(abs(k) for k in c)]) < 1e-17


# ---------------------------------------------------------------------------------------------
# P9: brute-force tensor mode == closed-form mode, on states incl. every boundary kind
# ---------------------------------------------------------------------------------------------
def _mk(oracle_mod, w):
    o = oracle_mod.Oracle(w.nx, w.ny, w.nz, w.tau)
    for f, k in w.faces.items():
        if w.inlet is not None and f == w.inlet.face:
            o.set_face(f, k, w.inlet.u_plane, w.inlet.noise_amp, w.inlet.seed, w.inlet.noise_mask)
        else:
            o.set_face(f, k)
    o.set_force(w.g)
    o.set_moments(w.moments)
    return o


def test_P9_brute_vs_closed_fstar(oracle_mod):
    rng = np.random.default_rng(5)
    for _ in range(50):
        M = rand_M(rng); om = rng.uniform(0.2, 1.99); g = rng.uniform(-1e-2, 1e-2, 3)
        for c in DIRS:
            a = oracle_mod.fstar(M, c, om, g, 0); b = oracle_mod.fstar(M, c, om, g, 1)
            assert abs(a - b) < 2e-16


@pytest.mark.parametrize("shape", [(3, 3, 3), (4, 3, 5), (6, 5, 7)])
def test_P9_brute_vs_closed_step_all_bc(oracle_mod, shape):
    nx, ny, nz = shape
    w = W.random_state(nx, ny, nz, seed=21)
    # walls in y + force, periodic x, open z (inlet lo / outlet hi)
    w.faces = {W.FACE_YLO: W.BC_BOUNCE_BACK, W.FACE_YHI: W.BC_BOUNCE_BACK,
               W.FACE_ZLO: W.BC_VELOCITY_INLET, W.FACE_ZHI: W.BC_OUTLET_ZERO_GRADIENT}
    up = np.random.default_rng(2).uniform(-0.03, 0.03, (3, ny, nx))
    w.inlet = W.Inlet(W.FACE_ZLO, up, 0.05, 9, 0b111)
    w.g = (1e-4, -2e-4, 3e-4)
    a = _mk(oracle_mod, w); b = _mk(oracle_mod, w)
    a.step(3, 0); b.step(3, 1)
    assert np.abs(a.get_moments() - b.get_moments()).max() < 1e-15


# ---------------------------------------------------------------------------------------------
# P3: uniform flow is a fixed point
# ---------------------------------------------------------------------------------------------
def test_P3_uniform_flow_fixed_point(oracle_mod):
    M = np.zeros((10, 4, 5, 6)); M[0] = 1.07; M[1] = 0.05; M[2] = -0.03; M[3] = 0.02
    o = oracle_mod.Oracle(6, 5, 4, 0.6); o.set_moments(M); o.step(5)
    R = o.get_moments()
    assert np.abs(R[:4] - M[:4]).max() < 5e-16
    assert np.abs(R[4:]).max() < 5e-16


# ---------------------------------------------------------------------------------------------
# P4: equivalence with a classic two-lattice population code (independent numpy implementation)
# ---------------------------------------------------------------------------------------------
class PopulationLB:
    """Recursive-regularised BGK on D3Q27 with explicit populations, collide then push-stream
    (Eq. 1, 5, 12, 14, 16, 17).  Walls in y: halfway bounce-back.  Written independently of the
    oracle with explicit Hermite tensors and einsum."""

    def __init__(self, M, tau, g, walls_y=False):
        self.c = np.array(DIRS, dtype=int)
        cf = self.c.astype(float)
        self.w = np.prod(np.where(self.c == 0, 2 / 3, 1 / 6), axis=1)
        d = np.eye(3)
        self.H2 = np.einsum("ia,ib->iab", cf, cf) - CS2 * d[None]
        self.H3 = (np.einsum("ia,ib,ig->iabg", cf, cf, cf)
                   - CS2 * (np.einsum("ig,ab->iabg", cf, d) + np.einsum("ia,bg->iabg", cf, d)
                            + np.einsum("ib,ag->iabg", cf, d)))
        self.cf = cf
        self.omega = 1.0 / tau
        self.g = np.asarray(g, float)
        self.walls_y = walls_y
        rho, u = M[0], M[1:4]
        Pi = np.array([[M[4], M[7], M[8]], [M[7], M[5], M[9]], [M[8], M[9], M[6]]])
        self.f = self.feq(rho, u) + self.fneq_reg(Pi, u)            # pre-collision

    def feq(self, rho, u):
        cu = np.einsum("ia,a...->i...", self.cf, u)
        e2 = np.einsum("iab,a...,b...->i...", self.H2, u, u)
        e3 = np.einsum("iabg,a...,b...,g...->i...", self.H3, u, u, u)
        wb = self.w.reshape((-1,) + (1,) * (u.ndim - 1))
        return wb * rho[None] * (1 + cu / CS2 + e2 / (2 * CS2**2) + e3 / (6 * CS2**3))

    def fneq_reg(self, a2, u):
        a3 = (np.einsum("ab...,g...->abg...", a2, u) + np.einsum("a...,bg...->abg...", u, a2)
              + np.einsum("b...,ag...->abg...", u, a2))
        n2 = np.einsum("iab,ab...->i...", self.H2, a2)
        n3 = np.einsum("iabg,abg...->i...", self.H3, a3)
        wb = self.w.reshape((-1,) + (1,) * (u.ndim - 1))
        return wb * (n2 / (2 * CS2**2) + n3 / (6 * CS2**3))

    def moments(self):
        f = self.f
        rho = f.sum(0)
        u = np.einsum("ia,i...->a...", self.cf, f) / rho
        fneq = f - self.feq(rho, u)
        a2 = np.einsum("iab,i...->ab...", self.H2, fneq)             # Eq. 12
        return rho, u, a2

    def step(self):
        rho, u, a2 = self.moments()
        wb = self.w.reshape(-1, 1, 1, 1)
        cg = (self.cf @ self.g).reshape(-1, 1, 1, 1)
        post = self.feq(rho, u) + (1 - self.omega) * self.fneq_reg(a2, u) + wb * rho[None] * cg / CS2
        new = np.empty_like(post)
        for i, (cx, cy, cz) in enumerate(self.c):
            new[i] = np.roll(post[i], shift=(cz, cy, cx), axis=(0, 1, 2))   # f_i(x + c_i) = post_i(x)
        if self.walls_y:
            opp = {tuple(c): i for i, c in enumerate(self.c)}
            for i, (cx, cy, cz) in enumerate(self.c):
                ib = opp[(-cx, -cy, -cz)]
                if cy == 1:
                    new[i][:, 0, :] = post[ib][:, 0, :]
                elif cy == -1:
                    new[i][:, -1, :] = post[ib][:, -1, :]
        self.f = new

    def M(self):
        rho, u, a2 = self.moments()
        return np.stack([rho, u[0], u[1], u[2], a2[0, 0], a2[1, 1], a2[2, 2], a2[0, 1], a2[0, 2], a2[1, 2]])


@pytest.mark.parametrize("walls", [False, True])
def test_P4_population_code_equivalence(oracle_mod, walls):
    """TSLB moments == moments of the explicit collide-and-stream code at every step (Eq. 5-6:
    the thread-safe form is the regularised LB 'in disguise').  Pins pull direction, source-site
    semantics of the force term (reading A11) and the bounce-back convention (A12)."""
    w = W.random_state(6, 5, 7, seed=4, tau=0.62)
    g = (2e-4, -1e-4, 3e-4)
    o = oracle_mod.Oracle(6, 5, 7, w.tau)
    if walls:
        o.set_face(W.FACE_YLO, W.BC_BOUNCE_BACK); o.set_face(W.FACE_YHI, W.BC_BOUNCE_BACK)
    o.set_force(g); o.set_moments(w.moments)
    p = PopulationLB(w.moments, w.tau, g, walls_y=walls)
    assert np.abs(p.M() - w.moments).max() < 1e-15        # initial populations carry the moments
    for s in range(5):
        o.step(1); p.step()
        assert np.abs(o.get_moments() - p.M()).max() < 5e-15, s


# ---------------------------------------------------------------------------------------------
# P5: mass conservation; momentum budget with force
# ---------------------------------------------------------------------------------------------
def test_P5_mass_and_momentum_budget_periodic(oracle_mod):
    w = W.random_state(8, 7, 6, seed=8, tau=0.55)
    g = np.array([1e-4, 2e-4, -3e-4])
    o = oracle_mod.Oracle(8, 7, 6, w.tau); o.set_force(g); o.set_moments(w.moments)
    d0 = o.diagnostics()
    for s in range(20):
        o.step(1)
        d = o.diagnostics()
        assert abs(d[0] - d0[0]) < 1e-12 * d0[0]
        # first-order (Luo) forcing: momentum grows by g * mass per step
        np.testing.assert_allclose(d[1:4], d0[1:4] + (s + 1) * g * d0[0], atol=1e-12)


def test_P5_mass_closed_channel(oracle_mod):
    w = W.channel(8, 12, 6, steps=50, dtype="f64")
    o = _mk(oracle_mod, w)
    m0 = o.diagnostics()[0]
    o.step(50)
    assert abs(o.diagnostics()[0] - m0) < 1e-12 * m0


# ---------------------------------------------------------------------------------------------
# P6: viscous decay, nu = cs2 (tau - 1/2)
# ---------------------------------------------------------------------------------------------
def _amp(M, M0):
    return float((M[1:4] * M0[1:4]).sum() / (M0[1:4] ** 2).sum())


def test_P6_taylor_green_2d_decay(oracle_mod):
    """2-D Taylor-Green vortex: velocity amplitude ~ exp(-2 nu k^2 t) (the law quoted in north_star)."""
    w = W.taylor_green_2d(32, 4, tau=0.8, U0=0.01, steps=100)
    o = _mk(oracle_mod, w); o.step(100)
    nu = CS2 * (w.tau - 0.5); k = 2 * np.pi / 32
    nu_eff = -np.log(_amp(o.get_moments(), w.moments)) / (2 * k * k * 100)
    assert abs(nu_eff / nu - 1) < 0.02


def test_P6_config0_decay(oracle_mod):
    """configs[0]: wave vector (k,k,k) -> amplitude ~ exp(-3 nu k^2 t) (reading A20)."""
    w = W.config0()
    o = _mk(oracle_mod, w); o.step(100)
    nu = CS2 * (w.tau - 0.5); k = 2 * np.pi / 32
    nu_eff = -np.log(_amp(o.get_moments(), w.moments)) / (3 * k * k * 100)
    assert abs(nu_eff / nu - 1) < 0.02
    # wrong tau->nu maps (tau/3, (tau-1)/3) are off by > 60 %
    assert abs(nu_eff / (CS2 * w.tau) - 1) > 0.3


# ---------------------------------------------------------------------------------------------
# P7 / P8: steady forced Poiseuille flow between halfway bounce-back walls
# ---------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def poiseuille(oracle_mod):
    ny, tau, g = 16, 0.8, 1e-6
    M = np.zeros((10, 3, ny, 3)); M[0] = 1
    o = oracle_mod.Oracle(3, ny, 3, tau)
    o.set_face(W.FACE_YLO, W.BC_BOUNCE_BACK); o.set_face(W.FACE_YHI, W.BC_BOUNCE_BACK)
    o.set_force((g, 0, 0)); o.set_moments(M)
    o.step(30000)
    return o.get_moments(), ny, tau, g


def test_P7_poiseuille_parabola(poiseuille):
    M, ny, tau, g = poiseuille
    nu = CS2 * (tau - 0.5)
    ux = M[1][1, :, 1]
    d2 = ux[2:] - 2 * ux[1:-1] + ux[:-2]
    np.testing.assert_allclose(d2, -g / nu, rtol=1e-6)             # curvature: nu = cs2 (tau - 1/2)
    j = np.arange(ny)
    para = (g / (2 * nu)) * (j + 0.5) * (ny - 0.5 - j)             # walls half a cell outside nodes 0, ny-1
    slip = ux - para
    assert np.ptp(slip) < 1e-6 * ux.max()                          # constant offset only
    assert abs(slip.mean()) < 0.02 * ux.max()                      # wall position: halfway (reading A12)
    assert np.abs(M[2]).max() < 1e-14 and np.abs(M[3]).max() < 1e-14


def test_P8_shear_stress(poiseuille):
    """Pi_neq_xy = -(tau/3) rho du_x/dy  (sign/scale of the stored non-equilibrium flux)."""
    M, ny, tau, g = poiseuille
    ux = M[1][1, :, 1]; rho = M[0][1, :, 1]; pxy = M[7][1, :, 1]
    dudy = 0.5 * (ux[2:] - ux[:-2])
    np.testing.assert_allclose(pxy[1:-1], -(tau / 3) * rho[1:-1] * dudy, rtol=1e-4)


# ---------------------------------------------------------------------------------------------
# Lattice symmetries: the step commutes with axis permutations and reflections
# ---------------------------------------------------------------------------------------------
def _permute(M, perm):
    """Relabel axes: new axis a is old axis perm[a] (array axes are z,y,x = 2,1,0)."""
    vec = [1, 2, 3]
    ten = {(0, 0): 4, (1, 1): 5, (2, 2): 6, (0, 1): 7, (0, 2): 8, (1, 2): 9}
    out = np.empty_like(M)
    arr_perm = tuple(2 - perm[2 - ax] for ax in range(3))          # array axis order for transpose
    tr = lambda A: np.transpose(A, arr_perm)
    out[0] = tr(M[0])
    for a in range(3):
        out[vec[a]] = tr(M[vec[perm[a]]])
    for (a, b), k in ten.items():
        pa, pb = sorted((perm[a], perm[b]))
        out[k] = tr(M[ten[(pa, pb)]])
    return np.ascontiguousarray(out)


def _reflect(M, ax):
    """x_ax -> -x_ax."""
    out = np.flip(M, axis=3 - ax).copy()                           # M axes: field, z, y, x
    out[1 + ax] *= -1
    for (a, b), k in {(0, 1): 7, (0, 2): 8, (1, 2): 9}.items():
        if ax in (a, b):
            out[k] *= -1
    return out


@pytest.mark.parametrize("perm", [(1, 0, 2), (2, 1, 0), (1, 2, 0)])
def test_symmetry_axis_permutation(oracle_mod, perm):
    w = W.random_state(5, 5, 5, seed=13, tau=0.58)
    a = oracle_mod.Oracle(5, 5, 5, w.tau); a.set_moments(w.moments); a.step(2)
    b = oracle_mod.Oracle(5, 5, 5, w.tau); b.set_moments(_permute(w.moments, perm)); b.step(2)
    assert np.abs(_permute(a.get_moments(), perm) - b.get_moments()).max() < 1e-15


@pytest.mark.parametrize("ax", [0, 1, 2])
def test_symmetry_reflection(oracle_mod, ax):
    w = W.random_state(4, 5, 6, seed=14, tau=0.58)
    a = oracle_mod.Oracle(4, 5, 6, w.tau); a.set_moments(w.moments); a.step(2)
    b = oracle_mod.Oracle(4, 5, 6, w.tau); b.set_moments(_reflect(w.moments, ax)); b.step(2)
    assert np.abs(_reflect(a.get_moments(), ax) - b.get_moments()).max() < 1e-15


# ---------------------------------------------------------------------------------------------
# Open boundaries (readings A13-A16; physically "parity unpinned"): definitional checks only
# ---------------------------------------------------------------------------------------------
def test_open_faces_quiescent_stays_quiescent(oracle_mod):
    M = np.zeros((10, 6, 5, 4)); M[0] = 1
    o = oracle_mod.Oracle(4, 5, 6, 0.7)
    for f in range(6):
        o.set_face(f, W.BC_OUTLET_ZERO_GRADIENT)
    o.set_moments(M); o.step(10)
    R = o.get_moments()
    assert np.abs(R - M).max() < 1e-15


def test_ghost_fill_definition(oracle_mod):
    """get_moments returns boundary nodes filled from x_F (clamp to [1, n-2] on open axes), inlet u imposed."""
    w = W.random_state(5, 6, 7, seed=3)
    up = np.random.default_rng(1).uniform(-0.02, 0.02, (3, 6, 5))
    o = oracle_mod.Oracle(5, 6, 7, 0.7)
    o.set_face(W.FACE_ZLO, W.BC_VELOCITY_INLET, up, 0.0, 5, 0)
    o.set_face(W.FACE_ZHI, W.BC_OUTLET_ZERO_GRADIENT)
    o.set_face(W.FACE_XLO, W.BC_OUTLET_ZERO_GRADIENT); o.set_face(W.FACE_XHI, W.BC_OUTLET_ZERO_GRADIENT)
    o.set_moments(w.moments)
    R = o.get_moments(); M = w.moments
    np.testing.assert_array_equal(R[:, 1:-1, :, 1:-1], M[:, 1:-1, :, 1:-1])      # interior untouched
    np.testing.assert_array_equal(R[:, -1, :, 2], M[:, -2, :, 2])                 # outlet copies all 10
    np.testing.assert_array_equal(R[:, 3, :, 0], M[:, 3, :, 1])
    np.testing.assert_array_equal(R[:, -1, :, 0], M[:, -2, :, 1])                 # edge: both clamped
    np.testing.assert_array_equal(R[0, 0], np.pad(M[0, 1, :, 1:-1], ((0, 0), (1, 1)), mode="edge"))  # rho from x_F
    np.testing.assert_array_equal(R[1:4, 0], up)                                  # inlet wins on the edge too
    np.testing.assert_array_equal(R[4:, 0, :, 2], M[4:, 1, :, 2])                 # Pi from x_F


def _fstar_all(p, M):
    """Post-collision populations f* = f_eq + (1-w) f_neq (+ force) of every node from its moments M[10,nz,ny,nx],
    with the independent numpy tensors of PopulationLB (Eq. 5, 14, 17)."""
    rho, u = M[0], M[1:4]
    Pi = np.array([[M[4], M[7], M[8]], [M[7], M[5], M[9]], [M[8], M[9], M[6]]])
    wb = p.w.reshape(-1, 1, 1, 1)
    cg = (p.cf @ p.g).reshape(-1, 1, 1, 1)
    return p.feq(rho, u) + (1 - p.omega) * p.fneq_reg(Pi, u) + wb * rho[None] * cg / CS2


def _pull_plane(p, src_by_cz):
    """Moments of one z-plane (x, y periodic) from the populations arriving from the planes below (c_z = +1), at
    (c_z = 0) and above (c_z = -1): src_by_cz[cz][i] is population i on the source plane.  Eq. 6 + Eq. 12."""
    arr = np.stack([np.roll(src_by_cz[cz][i], shift=(cy, cx), axis=(0, 1)) for i, (cx, cy, cz) in enumerate(DIRS)])
    R = arr.sum(0)
    J = np.einsum("ia,i...->a...", p.cf, arr)
    S = np.einsum("ia,ib,i...->ab...", p.cf, p.cf, arr)
    u = J / R
    Pi = S - R * (CS2 * np.eye(3)[:, :, None, None] + np.einsum("a...,b...->ab...", u, u))
    return np.stack([R, u[0], u[1], u[2], Pi[0, 0], Pi[1, 1], Pi[2, 2], Pi[0, 1], Pi[0, 2], Pi[1, 2]])


def test_inlet_and_outlet_populations_are_eq23_as_printed(oracle_mod):
    """PAPER.md:181-196 (Eq. 22-23), :202: the population an interior node pulls from a velocity-inlet node is
    f_eq(rho_B, u_B) + (1 - omega) f_neq(Pi(x_F), u_B), with u_B imposed, rho_B and Pi taken from the fluid neighbour
    x_F AT THE CURRENT TIME LEVEL (readings A13, A15); from a zero-gradient outlet node it is the post-collision
    population of x_F's own moments.  Built here with the independent numpy Hermite tensors and compared with the
    oracle's first interior planes over two steps (the second step fixes the time level of the fill).
    Mutations that fail: rho or Pi of the boundary node's own old value instead of x_F's; u copied instead of imposed;
    x_F taken at the previous time level."""
    nx, ny, nz, tau = 6, 5, 7, 0.63
    w = W.random_state(nx, ny, nz, seed=41, tau=tau)
    up = np.random.default_rng(7).uniform(-0.03, 0.03, (3, ny, nx))
    o = oracle_mod.Oracle(nx, ny, nz, tau)
    o.set_face(W.FACE_ZLO, W.BC_VELOCITY_INLET, up, 0.0, 3, 0)
    o.set_face(W.FACE_ZHI, W.BC_OUTLET_ZERO_GRADIENT)
    o.set_moments(w.moments)
    p = PopulationLB(w.moments, tau, (0.0, 0.0, 0.0))
    Pi_at = lambda M, z: np.array([[M[4, z], M[7, z], M[8, z]], [M[7, z], M[5, z], M[9, z]], [M[8, z], M[9, z], M[6, z]]])
    M_prev = None
    M = w.moments.copy()
    for step in range(2):
        post = _fstar_all(p, M)
        # inlet node x_B = (x, y, 0), x_F = (x, y, 1): Eq. 23 as printed
        fB = p.feq(M[0, 1], up) + (1 - p.omega) * p.fneq_reg(Pi_at(M, 1), up)
        want_lo = _pull_plane(p, {1: fB, 0: post[:, 1], -1: post[:, 2]})
        # outlet node x_B = (x, y, nz-1), x_F = (x, y, nz-2): all ten moments of x_F
        want_hi = _pull_plane(p, {1: post[:, nz - 3], 0: post[:, nz - 2], -1: post[:, nz - 2]})
        o.step(1)
        R = o.get_moments()
        assert np.abs(R[:, 1] - want_lo).max() < 2e-15, step
        assert np.abs(R[:, nz - 2] - want_hi).max() < 2e-15, step
        # mutations
        f_own = p.feq(M[0, 0], up) + (1 - p.omega) * p.fneq_reg(Pi_at(M, 0), up)          # boundary node's own rho, Pi
        f_copy = p.feq(M[0, 1], M[1:4, 1]) + (1 - p.omega) * p.fneq_reg(Pi_at(M, 1), M[1:4, 1])   # u not imposed
        # (get_moments returns the boundary nodes already refilled, so "own old value" is a mutation at step 0 only)
        for bad in ((f_own, f_copy) if step == 0 else (f_copy,)):
            assert np.abs(_pull_plane(p, {1: bad, 0: post[:, 1], -1: post[:, 2]}) - R[:, 1]).max() > 1e-5
        if M_prev is not None:                                                                  # stale time level
            f_stale = p.feq(M_prev[0, 1], up) + (1 - p.omega) * p.fneq_reg(Pi_at(M_prev, 1), up)
            assert np.abs(_pull_plane(p, {1: f_stale, 0: post[:, 1], -1: post[:, 2]}) - R[:, 1]).max() > 1e-5
        M_prev, M = M, R


def test_uniform_through_flow_is_a_fixed_point(oracle_mod):
    """A uniform state (rho0, u0, Pi = 0) entering through an inlet with u_in = u0 and leaving through zero-gradient
    outlets on the five other faces is an exact fixed point of fill + sweep: every copy, every imposed value and every
    pulled population reproduces it (Eq. 22-23 with a uniform neighbour; P3 for the interior)."""
    nx, ny, nz = 5, 6, 7
    M = np.zeros((10, nz, ny, nx)); M[0] = 1.03; M[1] = 0.01; M[2] = -0.02; M[3] = 0.04
    up = np.empty((3, ny, nx)); up[0] = 0.01; up[1] = -0.02; up[2] = 0.04
    o = oracle_mod.Oracle(nx, ny, nz, 0.56)
    o.set_face(W.FACE_ZLO, W.BC_VELOCITY_INLET, up, 0.0, 1, 0)
    for f in (W.FACE_ZHI, W.FACE_XLO, W.FACE_XHI, W.FACE_YLO, W.FACE_YHI):
        o.set_face(f, W.BC_OUTLET_ZERO_GRADIENT)
    o.set_moments(M)
    o.step(10)
    assert np.abs(o.get_moments() - M).max() < 1e-15
    # and it is the imposed velocity that holds it there: a different u_in moves the first interior plane
    up2 = up.copy(); up2[2] = 0.05
    o2 = oracle_mod.Oracle(nx, ny, nz, 0.56)
    o2.set_face(W.FACE_ZLO, W.BC_VELOCITY_INLET, up2, 0.0, 1, 0)
    for f in (W.FACE_ZHI, W.FACE_XLO, W.FACE_XHI, W.FACE_YLO, W.FACE_YHI):
        o2.set_face(f, W.BC_OUTLET_ZERO_GRADIENT)
    o2.set_moments(M); o2.step(1)
    assert np.abs(o2.get_moments()[:, 1, 2, 2] - M[:, 1, 2, 2]).max() > 1e-4


def test_diagnostics_are_the_plain_sums(oracle_mod):
    """oracle_diagnostics (reading A26): mass = sum rho, momentum = sum rho u, kinetic energy = 1/2 sum rho |u|^2 over the
    nodes that are not on an open face -- against numpy sums of get_moments(), without and with open faces.
    Mutations that fail: a missing 1/2 or rho in the energy, u instead of rho u, open-face nodes included."""
    w = W.random_state(7, 6, 5, seed=23)
    for open_faces in ((), (W.FACE_ZLO, W.FACE_ZHI, W.FACE_XHI)):
        o = oracle_mod.Oracle(7, 6, 5, 0.7)
        for f in open_faces:
            o.set_face(f, W.BC_OUTLET_ZERO_GRADIENT)
        if open_faces:
            o.set_face(W.FACE_XLO, W.BC_OUTLET_ZERO_GRADIENT)
        o.set_moments(w.moments); o.step(2)
        M = o.get_moments()
        m = np.ones(M.shape[1:], dtype=bool)
        if open_faces:
            m[0] = m[-1] = False; m[:, :, 0] = m[:, :, -1] = False
        rho, u = M[0][m], M[1:4][:, m]
        want = np.array([rho.sum(), (rho * u[0]).sum(), (rho * u[1]).sum(), (rho * u[2]).sum(),
                         0.5 * (rho * (u * u).sum(0)).sum()])
        d = o.diagnostics()
        np.testing.assert_allclose(d, want, rtol=1e-13, atol=1e-15)
        assert abs(d[4] - (rho * (u * u).sum(0)).sum()) > 1e-3 * d[4]           # the 1/2 is there
        assert abs(d[1] - u[0].sum()) > 1e-6                                     # rho u, not u
        if open_faces:                                                           # the exclusion is exercised
            assert abs(d[0] - M[0].sum()) > 1.0


def test_inlet_noise_is_relative_and_reproducible(oracle_mod):
    w = W.jet(12, 12, 8, steps=1, dtype="f64", D=6.0)
    a = _mk(oracle_mod, w); b = _mk(oracle_mod, w)
    a.step(3); b.step(3)
    Ra, Rb = a.get_moments(), b.get_moments()
    np.testing.assert_array_equal(Ra, Rb)
    uz = Ra[3, 0]; up = w.inlet.u_plane[2]
    assert np.all(uz[up == 0] == 0)
    rel = uz[up != 0] / up[up != 0] - 1
    assert np.abs(rel).max() <= 0.01 * (1 + 1e-12) and np.abs(rel).max() > 0.005
    idx = (0 * 12 + 5) * 12 + 5                                   # node (5,5,0), t = 3
    assert abs(uz[5, 5] - up[5, 5] * (1 + 0.01 * oracle_mod.noise_xi(1, 3, idx))) < 1e-18


# ---------------------------------------------------------------------------------------------
# Inlet-noise hash (reading A14) against the published SplitMix64 stream
# ---------------------------------------------------------------------------------------------
def test_mix64_published_vectors(oracle_mod):
    want = [int(l) for l in open(os.path.join(GOLD, "splitmix64_seed1234567.txt")) if l.strip() and l[0] != "#"]
    s = 1234567
    for v in want:
        s = (s + 0x9E3779B97F4A7C15) % 2**64
        assert oracle_mod.mix64(s) == v


def test_noise_xi_range_and_exactness(oracle_mod):
    xs = np.array([oracle_mod.noise_xi(1, t, i) for t in range(4) for i in range(500)])
    assert xs.min() >= -1 and xs.max() < 1
    assert abs(xs.mean()) < 0.05 and abs(xs.std() - 1 / np.sqrt(3)) < 0.03
    np.testing.assert_array_equal(xs, xs.astype(np.float32).astype(np.float64))   # exact in fp32
    r = oracle_mod.noise_r24(7, 2, 99)
    k = oracle_mod.mix64((oracle_mod.mix64(7 ^ ((0x9E3779B97F4A7C15 * 3) % 2**64)) + 99) % 2**64)
    assert r == k >> 40 and 0 <= r < 2**24


# ---------------------------------------------------------------------------------------------
# Parameters the paper prints
# ---------------------------------------------------------------------------------------------
def test_paper_parameter_sets():
    P = {}
    for l in open(os.path.join(GOLD, "paper_parameters.txt")):
        if l.strip() and l[0] != "#":
            k, v = l.split(); P[k] = float(v)
    # nu = cs2 (tau - 1/2), PAPER.md:51 vs :258 (tau printed to 4 digits)
    assert abs(0.5 + 3 * P["jet_nu"] - P["jet_tau"]) < 5e-5
    assert abs(P["jet_U"] * P["jet_D"] / P["jet_nu"] / P["jet_Re"] - 1) < 0.1
    assert abs(P["jet_U"] * np.sqrt(3) - P["jet_Ma"]) < 0.005
    u_tau = np.sqrt(P["chan_g"] * P["chan_H"])
    assert abs(P["chan_H"] * u_tau / P["chan_nu"] / P["chan_Re_tau"] - 1) < 0.01
    # BASELINE.json configs[2]/[3] use the same maps
    w = W.channel(6, 8, 6, steps=1)
    assert abs(w.tau - (0.5 + 3 * 0.0035 * 4 / 180)) < 1e-15 and abs(w.g[0] - 0.0035**2 / 4) < 1e-20
    j = W.jet(8, 8, 8, steps=1)
    assert abs(j.tau - (0.5 + 3 * 0.05 * 20 / 7000)) < 1e-15


# ---------------------------------------------------------------------------------------------
# Second-order variant (Eq. 8): oracle_set_order(2).  SURVEY.md 8(f) rank 2.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", [0, 1])
def test_order2_moments(oracle_mod, mode):
    """Eq. 8 reproduces rho, rho u and rho cs2 I + rho uu + (1-w) Pi exactly like Eq. 18; its third moments carry
    only the lattice part cs2 rho (u delta)_sym: no rho uuu, no a3 (that is what 'second order' means)."""
    rng = np.random.default_rng(23)
    for _ in range(10):
        M = rand_M(rng)
        omega = rng.uniform(0.6, 1.9)
        rho, u, Pi = M[0], M[1:4], Pi_of(M)
        f = np.array([oracle_mod.fstar(M, c, omega, mode=mode, order=2) for c in DIRS])
        c = np.array(DIRS, float)
        assert abs(f.sum() - rho) < 1e-15
        assert np.abs(c.T @ f - rho * u).max() < 1e-15
        S = np.einsum("i,ia,ib->ab", f, c, c)
        assert np.abs(S - (rho * CS2 * np.eye(3) + rho * np.outer(u, u) + (1 - omega) * Pi)).max() < 1e-15
        Q = np.einsum("i,ia,ib,ig->abg", f, c, c, c)
        d = np.eye(3)
        lattice = CS2 * rho * (np.einsum("a,bg->abg", u, d) + np.einsum("b,ag->abg", u, d) + np.einsum("g,ab->abg", u, d))
        for a, b, g in itertools.product(range(3), repeat=3):
            if not (a == b == g):
                assert abs(Q[a, b, g] - lattice[a, b, g]) < 1e-15
        # and it differs from the third-order population by exactly the H3 terms
        f3 = np.array([oracle_mod.fstar(M, c_, omega, mode=mode, order=3) for c_ in DIRS])
        assert np.abs(f3 - f).max() > 1e-7


def test_order2_population_code_equivalence(oracle_mod):
    """Order-2 TSLB == explicit collide-and-stream BGK with second-order equilibrium and the projected (Eq. 7)
    non-equilibrium part, at every step, walls and force included."""
    class Pop2(PopulationLB):
        def feq(self, rho, u):
            cu = np.einsum("ia,a...->i...", self.cf, u)
            e2 = np.einsum("iab,a...,b...->i...", self.H2, u, u)
            wb = self.w.reshape((-1,) + (1,) * (u.ndim - 1))
            return wb * rho[None] * (1 + cu / CS2 + e2 / (2 * CS2**2))             # Eq. 2

        def fneq_reg(self, a2, u):
            wb = self.w.reshape((-1,) + (1,) * (u.ndim - 1))
            return wb * np.einsum("iab,ab...->i...", self.H2, a2) / (2 * CS2**2)   # Eq. 7
    w = W.random_state(6, 5, 7, seed=8, tau=0.7)
    g = (1e-4, 2e-4, -3e-4)
    for walls in (False, True):
        o = oracle_mod.Oracle(6, 5, 7, w.tau)
        o.set_order(2)
        if walls:
            o.set_face(W.FACE_YLO, W.BC_BOUNCE_BACK); o.set_face(W.FACE_YHI, W.BC_BOUNCE_BACK)
        o.set_force(g); o.set_moments(w.moments)
        p = Pop2(w.moments, w.tau, g, walls_y=walls)
        for s in range(5):
            o.step(1); p.step()
            assert np.abs(o.get_moments() - p.M()).max() < 5e-15, (walls, s)


def test_order2_brute_vs_closed_and_decay(oracle_mod):
    """Brute-force and closed-form modes agree at order 2; the viscosity is unchanged (nu = (tau - 1/2)/3)."""
    w = W.random_state(5, 4, 6, seed=2, tau=0.66)
    a = oracle_mod.Oracle(5, 4, 6, w.tau); b = oracle_mod.Oracle(5, 4, 6, w.tau)
    for o in (a, b):
        o.set_order(2); o.set_force((1e-4, 0, -1e-4)); o.set_moments(w.moments)
    a.step(3, mode=oracle_mod.MODE_BRUTE); b.step(3, mode=oracle_mod.MODE_CLOSED)
    assert np.abs(a.get_moments() - b.get_moments()).max() < 1e-15
    w = W.taylor_green_2d(n=32, nz=3, tau=0.8, U0=0.01, steps=100)
    o = oracle_mod.Oracle(w.nx, w.ny, w.nz, w.tau); o.set_order(2); o.set_moments(w.moments); o.step(100)
    M = o.get_moments()
    k = 2 * np.pi / 32
    nu = (0.8 - 0.5) / 3
    ratio = np.abs(M[1]).max() / 0.01
    nu_eff = -np.log(ratio) / (2 * k * k * 100)
    assert abs(nu_eff / nu - 1) < 0.02
    with pytest.raises(RuntimeError):
        o.set_order(4)


# ---------------------------------------------------------------------------------------------
# Plane statistics (Eq. 24-25 raw sums).  SURVEY.md 8(f) rank 1.
# ---------------------------------------------------------------------------------------------
def test_plane_statistics_closed_forms(oracle_mod):
    """Taylor-Green field u = U0 (sinX cosY cosZ, -cosX sinY cosZ, 0): over a plane of constant y the sums have closed
    forms (sum of sin^2 or cos^2 over a full period of n >= 3 nodes is n/2, odd powers and mixed products vanish)."""
    n, U0 = 16, 0.01
    w = W.config0(n=n, steps=0)
    o = oracle_mod.Oracle(n, n, n, w.tau); o.set_moments(w.moments)
    S = np.zeros((13, n)); o.plane_statistics(1, S)
    Y = 2 * np.pi * np.arange(n) / n
    assert np.abs(S[0] - n * n).max() == 0
    assert np.abs(S[1:4]).max() < 1e-15 and np.abs(S[10:13]).max() < 1e-16          # odd moments vanish
    assert np.abs(S[4] - U0**2 * np.cos(Y)**2 * n * n / 4).max() < 1e-16
    assert np.abs(S[5] - U0**2 * np.sin(Y)**2 * n * n / 4).max() < 1e-16
    assert np.abs(S[6]).max() == 0 and np.abs(S[7:10]).max() < 1e-17
    # along x the roles change: sum over (y,z) of u_x^2 = U0^2 sin^2 X n^2/4; two samples accumulate
    S = np.zeros((13, n)); o.plane_statistics(0, S); o.plane_statistics(0, S)
    assert np.abs(S[4] - 2 * U0**2 * np.sin(Y)**2 * n * n / 4).max() < 1e-16 and np.abs(S[0] - 2 * n * n).max() == 0


def test_plane_statistics_vs_numpy_central_moments(oracle_mod):
    """Reynolds stresses and skewness derived from the raw sums equal numpy's central moments of the same field."""
    w = W.random_state(7, 9, 5, seed=21)
    o = oracle_mod.Oracle(7, 9, 5, w.tau); o.set_moments(w.moments)
    S = np.zeros((13, 9)); o.plane_statistics(1, S)
    u = w.moments[1:4]                                  # [3][nz][ny][nx]
    mean = S[1:4] / S[0]
    assert np.abs(mean - u.mean(axis=(1, 3))).max() < 1e-15
    var = S[4:7] / S[0] - mean**2
    assert np.abs(var - u.var(axis=(1, 3))).max() < 1e-15
    rxy = S[7] / S[0] - mean[0] * mean[1]
    up = u - u.mean(axis=(1, 3), keepdims=True)
    assert np.abs(rxy - (up[0] * up[1]).mean(axis=(0, 2))).max() < 1e-15
    m3 = S[10:13] / S[0] - 3 * mean * S[4:7] / S[0] + 2 * mean**3
    assert np.abs(m3 - (up**3).mean(axis=(1, 3))).max() < 1e-16


# ---------------------------------------------------------------------------------------------
# Sponge layer (Eq. 26; reading A24): SURVEY.md 8(f) rank 3
# ---------------------------------------------------------------------------------------------
def _sponge_nu(nu, z, nz, z_start, K, p):
    """Eq. 26 typed from the paper, with reading A24 (layer width in the denominator)."""
    return nu if z < z_start else nu * (K * ((z - z_start) / (nz - z_start)) ** p + 1.0)


def test_sponge_K0_is_no_sponge(oracle_mod):
    w = W.random_state(6, 5, 9, seed=21, tau=0.6)
    a = _mk(oracle_mod, w); b = _mk(oracle_mod, w)
    b.set_sponge(4, 0.0, 3.0)
    a.step(3); b.step(3)
    assert np.array_equal(a.get_moments(), b.get_moments())


def test_sponge_profile_paper_numbers(oracle_mod):
    """K = 1000, z_start = N_z - 50, p = 3 (A24): tau(z) = 1/2 + 3 nu_sponge(z).
    Fails for an off-by-one in z - z_start (tau(z_start) must be the bulk tau), a dropped '+ 1', or 1/tau vs tau mix-ups."""
    nz, tau = 120, 0.5004
    o = oracle_mod.Oracle(4, 4, nz, tau)
    o.set_sponge(nz - 50, 1000.0, 3.0)
    nu = (tau - 0.5) / 3
    assert o.tau_of_plane(0) == tau and o.tau_of_plane(nz - 51) == tau
    assert abs(o.tau_of_plane(nz - 50) - tau) < 1e-15
    for z in (nz - 49, nz - 25, nz - 1):
        assert abs(o.tau_of_plane(z) - (0.5 + 3 * _sponge_nu(nu, z, nz, nz - 50, 1000.0, 3))) < 1e-13
    # last plane: (49/50)^3 * 1000 + 1 = 942.192 times the bulk viscosity
    assert abs((o.tau_of_plane(nz - 1) - 0.5) / (tau - 0.5) - 942.192) < 1e-6
    taus = [o.tau_of_plane(z) for z in range(nz)]
    assert all(b >= a for a, b in zip(taus, taus[1:]))


def test_sponge_population_code_equivalence(oracle_mod):
    """Collision is local (Eq. 1, 5): a population code that relaxes every node with ITS OWN omega(z) and then streams
    gives the same moments as the thread-safe sweep with the sponge.  Fails if the sweep takes omega of the destination
    node instead of the source node, or applies the profile along another axis."""
    nx, ny, nz, tau = 6, 5, 10, 0.56
    w = W.random_state(nx, ny, nz, seed=22, tau=tau)
    g = (1e-4, 2e-4, -1e-4)
    z_start, K, p = 4, 7.0, 3.0
    o = oracle_mod.Oracle(nx, ny, nz, tau)
    o.set_force(g); o.set_sponge(z_start, K, p); o.set_moments(w.moments)
    pop = PopulationLB(w.moments, tau, g)
    nu = CS2 * (tau - 0.5)
    tau_z = np.array([0.5 + _sponge_nu(nu, z, nz, z_start, K, p) / CS2 for z in range(nz)])
    pop.omega = (1.0 / tau_z).reshape(1, nz, 1, 1)         # broadcasts over [direction][z][y][x]
    for s in range(5):
        o.step(1); pop.step()
        assert np.abs(o.get_moments() - pop.M()).max() < 5e-15, s
    # and the layer matters: without it the result differs
    o2 = oracle_mod.Oracle(nx, ny, nz, tau); o2.set_force(g); o2.set_moments(w.moments); o2.step(5)
    assert np.abs(o2.get_moments() - o.get_moments()).max() > 1e-6


def test_sponge_two_region_decay(oracle_mod):
    """p = 0 turns Eq. 26 into a step: nu in z < z_start, (K + 1) nu above.  A shear wave u_y = U sin(kx), uniform in z,
    decays as exp(-nu_local k^2 t) on planes far from the two interfaces (periodic z) -- the viscosity <-> tau map with
    the factor (K + 1) applied on the right planes."""
    nx, ny, nz, tau, K = 32, 3, 48, 0.56, 2.0
    k = 2 * np.pi / nx
    M = np.zeros((10, nz, ny, nx)); M[0] = 1.0
    M[2] = 1e-3 * np.sin(k * np.arange(nx))[None, None, :]
    o = oracle_mod.Oracle(nx, ny, nz, tau)
    o.set_sponge(24, K, 0.0); o.set_moments(M)
    # (measured between two times: the start from Pi_neq = 0 has an initial layer of a few steps)
    o.step(20); R1 = o.get_moments()
    o.step(40); R2 = o.get_moments()
    nu = CS2 * (tau - 0.5)
    for z, nu_loc in ((12, nu), (36, (K + 1) * nu)):
        a1 = (R1[2, z] * M[2, z]).sum(); a2 = (R2[2, z] * M[2, z]).sum()
        assert abs(-np.log(a2 / a1) / (k * k * 40) / nu_loc - 1) < 0.03, (z, a1, a2)


# ---------------------------------------------------------------------------------------------
# (r, z)-bin statistics of the jet (Fig. 7-8; reading A27): SURVEY.md 8(f) rank 1
# ---------------------------------------------------------------------------------------------
def test_radial_statistics_analytic_swirling_jet(oracle_mod):
    """u_z = exp(-r^2/s^2), u_r = a r, u_t = b r written in Cartesian components: every bin sum is then a sum of known
    functions of the node radii, evaluated here with numpy's hypot / bincount (library routines, no shared code).
    Fails for swapped u_r / u_t projections, a wrong sign of u_t, bins along the wrong axis or a missing z index."""
    nx, ny, nz, nr, dr = 21, 19, 4, 6, 1.5
    xc, yc, s2, a, b = 9.25, 8.5, 30.0, 2e-3, -1e-3
    X, Y = np.meshgrid(np.arange(nx) - xc, np.arange(ny) - yc)          # [ny][nx]
    r = np.hypot(X, Y)
    M = np.zeros((10, nz, ny, nx)); M[0] = 1.0
    for z in range(nz):
        M[3, z] = (1 + 0.1 * z) * np.exp(-r * r / s2)
        M[1, z] = a * X - b * Y                                          # u_r e_r + u_t e_t, e_r = (X, Y)/r, e_t = (-Y, X)/r
        M[2, z] = a * Y + b * X
    o = oracle_mod.Oracle(nx, ny, nz, 0.7); o.set_moments(M)
    S = np.zeros((8, nz, nr)); o.radial_statistics(xc, yc, dr, nr, S)
    k = np.floor(r / dr).astype(int)
    sel = k < nr
    cnt = np.bincount(k[sel], minlength=nr)
    for z in range(nz):
        uz = M[3, z]
        exp = [cnt, np.bincount(k[sel], uz[sel], nr), np.bincount(k[sel], (a * r)[sel], nr), np.bincount(k[sel], (b * r)[sel], nr),
               np.bincount(k[sel], (uz * uz)[sel], nr), np.bincount(k[sel], (a * r)[sel] ** 2, nr),
               np.bincount(k[sel], (b * r)[sel] ** 2, nr), np.bincount(k[sel], (uz * a * r)[sel], nr)]
        for row in range(8):
            assert np.abs(S[row, z] - exp[row]).max() < 1e-13, (row, z)
    # a second sample adds
    o.radial_statistics(xc, yc, dr, nr, S)
    assert np.abs(S[0, 0] - 2 * cnt).max() == 0


def test_radial_statistics_axis_node_and_rotation(oracle_mod):
    """A node exactly on the axis has no radial direction: it counts in bin 0 with u_r = u_t = 0.  Rotating the field
    by 90 degrees about a centred axis leaves every sum unchanged (the bins are rings)."""
    n, nz, nr, dr = 11, 3, 5, 1.0
    w = W.random_state(n, n, nz, seed=8)
    M = w.moments.astype(np.float64)
    o = oracle_mod.Oracle(n, n, nz, 0.7); o.set_moments(M)
    S = np.zeros((8, nz, nr)); o.radial_statistics(5.0, 5.0, dr, nr, S)
    assert np.all(S[0, :, 0] == 1.0)                                    # only the axis node has r < 1
    assert np.abs(S[1, :, 0] - M[3, :, 5, 5]).max() == 0 and np.all(S[2, :, 0] == 0) and np.all(S[3, :, 0] == 0)
    # rotate by +90 degrees about z: (x, y) -> (-y, x); u_x' = -u_y, u_y' = u_x on the rotated nodes
    Mr = np.empty_like(M)
    rot = lambda F: np.rot90(F, k=1, axes=(2, 1))                       # value at (x, y) moves to (-y, x) (centred grid)
    for f in range(10):
        Mr[f] = rot(M[f])
    Mr[1], Mr[2] = -rot(M[2]), rot(M[1])
    o2 = oracle_mod.Oracle(n, n, nz, 0.7); o2.set_moments(Mr)
    S2 = np.zeros((8, nz, nr)); o2.radial_statistics(5.0, 5.0, dr, nr, S2)
    assert np.abs(S2 - S).max() < 1e-13


# ---------------------------------------------------------------------------------------------
# Boundary variants of section II.C: pressure outlet, NEQ no-slip wall, Gaussian inlet noise
# ---------------------------------------------------------------------------------------------
def test_pressure_outlet_populations_are_eq23_with_imposed_density(oracle_mod):
    """'the equilibrium distribution is computed by imposing the hydrodynamic variables at the boundary
    (either momentum or density/pressure), while the non-equilibrium part is extrapolated'.  The population pulled from a
    pressure-outlet node is f_eq(rho_out, u(x_F)) + (1 - omega) f_neq(Pi(x_F), u(x_F)), built with the independent numpy
    tensors.  Fails if rho is copied instead of imposed, or u is zeroed."""
    nx, ny, nz, tau, rho_out = 6, 5, 7, 0.63, 0.97
    w = W.random_state(nx, ny, nz, seed=43, tau=tau)
    up = np.random.default_rng(9).uniform(-0.03, 0.03, (3, ny, nx))
    o = oracle_mod.Oracle(nx, ny, nz, tau)
    o.set_face(W.FACE_ZLO, W.BC_VELOCITY_INLET, up, 0.0, 3, 0)
    o.set_pressure_outlet(W.FACE_ZHI, rho_out)
    o.set_moments(w.moments)
    p = PopulationLB(w.moments, tau, (0.0, 0.0, 0.0))
    M = w.moments.copy()
    Pi_at = lambda M, z: np.array([[M[4, z], M[7, z], M[8, z]], [M[7, z], M[5, z], M[9, z]], [M[8, z], M[9, z], M[6, z]]])
    for step in range(2):
        post = _fstar_all(p, M)
        uF = M[1:4, nz - 2]
        fB = p.feq(np.full((ny, nx), rho_out), uF) + (1 - p.omega) * p.fneq_reg(Pi_at(M, nz - 2), uF)
        want = _pull_plane(p, {1: post[:, nz - 3], 0: post[:, nz - 2], -1: fB})
        o.step(1)
        R = o.get_moments()
        assert np.abs(R[:, nz - 2] - want).max() < 2e-15, step
        f_copy = post[:, nz - 2]                                          # zero-gradient outlet instead
        assert np.abs(_pull_plane(p, {1: post[:, nz - 3], 0: post[:, nz - 2], -1: f_copy}) - R[:, nz - 2]).max() > 1e-4
        assert np.all(R[0, nz - 1] == rho_out) and np.array_equal(R[1:, nz - 1], R[1:, nz - 2])
        M = R


def test_pressure_outlet_uniform_through_flow(oracle_mod):
    """Uniform flow leaving through a pressure outlet with rho_out = rho0 is a fixed point; a lower rho_out is not."""
    nx, ny, nz = 5, 6, 8
    M = np.zeros((10, nz, ny, nx)); M[0] = 1.02; M[3] = 0.03
    up = np.zeros((3, ny, nx)); up[2] = 0.03
    def run(rho_out):
        o = oracle_mod.Oracle(nx, ny, nz, 0.58)
        o.set_face(W.FACE_ZLO, W.BC_VELOCITY_INLET, up, 0.0, 1, 0)
        o.set_pressure_outlet(W.FACE_ZHI, rho_out)
        o.set_moments(M); o.step(6)
        return o.get_moments()
    assert np.abs(run(1.02) - M).max() < 1e-15
    assert np.abs(run(1.00)[:, nz - 2] - M[:, nz - 2]).max() > 1e-3


def test_neq_no_slip_wall_poiseuille(oracle_mod):
    """The Dirichlet member of section II.C with u_B = 0 is the paper's thread-safe no-slip wall:
    wall nodes ON the faces y = 0, ny-1 with imposed zero velocity.  Steady forced flow between them is the parabola
    u_x'' = -g/nu through u = 0 AT the wall nodes (halfway bounce-back puts the zero half a cell outside, P7)."""
    nx, ny, nz, tau, g = 3, 25, 3, 0.9, 1e-6
    nu = CS2 * (tau - 0.5)
    M = np.zeros((10, nz, ny, nx)); M[0] = 1.0
    zero = np.zeros((3, nz, nx))
    o = oracle_mod.Oracle(nx, ny, nz, tau)
    o.set_face(W.FACE_YLO, W.BC_VELOCITY_INLET, zero, 0.0, 1, 0)
    o.set_face(W.FACE_YHI, W.BC_VELOCITY_INLET, zero, 0.0, 1, 0)
    o.set_force((g, 0.0, 0.0)); o.set_moments(M)
    o.step(6000)
    u = o.get_moments()[1, 1, :, 1]
    y = np.arange(ny)
    exact = g / (2 * nu) * y * (ny - 1 - y)
    assert np.all(u[[0, -1]] == 0.0)
    assert np.abs(u - exact).max() / exact.max() < 0.02
    assert abs(np.diff(u, 2)[3:-3].mean() / (-g / nu) - 1) < 0.01


def test_gaussian_noise_is_box_muller_of_the_counter_stream(oracle_mod):
    """xi = sqrt(-2 ln u1) cos(2 pi u2) with u1 = (r24 + 1)/2^24, u2 = r24'/2^24 from the pinned SplitMix64 mixer
    (recomputed here through oracle.mix64, itself pinned to the published stream), and the sample moments of 2e5 draws
    are those of a unit normal (mean 0, variance 1, kurtosis 3)."""
    GOLD, mask = 0x9E3779B97F4A7C15, (1 << 64) - 1
    seed, t = 77, 5
    k = oracle_mod.mix64((seed ^ (GOLD * (t + 1))) & mask)
    for idx in (0, 1, 12345, 2**31 + 7):
        a = oracle_mod.mix64((k + idx) & mask); b = oracle_mod.mix64(a)
        u1 = ((a >> 40) + 1) / 2.0**24; u2 = (b >> 40) / 2.0**24
        assert abs(oracle_mod.noise_gauss(seed, t, idx) - np.sqrt(-2 * np.log(u1)) * np.cos(2 * np.pi * u2)) < 1e-14
    x = np.array([oracle_mod.noise_gauss(3, 0, i) for i in range(200000)])
    assert abs(x.mean()) < 0.01 and abs(x.var() - 1) < 0.02 and abs((x**4).mean() / x.var()**2 - 3) < 0.1
    # consecutive steps and neighbouring nodes are uncorrelated
    y = np.array([oracle_mod.noise_gauss(3, 1, i) for i in range(200000)])
    assert abs(np.corrcoef(x, y)[0, 1]) < 0.01 and abs(np.corrcoef(x[:-1], x[1:])[0, 1]) < 0.01


def test_gaussian_inlet_noise_enters_relatively(oracle_mod):
    """Bit 8 of the noise mask switches the inlet to the Gaussian law: u_k = u_in,k (1 + amp xi_gauss) on masked components."""
    nx, ny, nz = 4, 5, 6
    M = np.zeros((10, nz, ny, nx)); M[0] = 1.0
    up = np.zeros((3, ny, nx)); up[2] = 0.05; up[0] = 0.01
    o = oracle_mod.Oracle(nx, ny, nz, 0.6)
    o.set_face(W.FACE_ZLO, W.BC_VELOCITY_INLET, up, 0.1, 11, 0b100 | W.NOISE_GAUSSIAN)
    o.set_face(W.FACE_ZHI, W.BC_OUTLET_ZERO_GRADIENT)
    o.set_moments(M)
    R = o.get_moments()
    for y in range(ny):
        for x in range(nx):
            xi = oracle_mod.noise_gauss(11, 0, y * nx + x)
            assert abs(R[3, 0, y, x] - 0.05 * (1 + 0.1 * xi)) < 1e-16 and R[1, 0, y, x] == 0.01

/*
 * tslb_oracle.c -- CPU ORACLE for the high-order thread-safe lattice Boltzmann (TSLB) sweep.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant generator with the CUDA path in paper_2401_17074_b200/csrc.
 *
 * It is a plain, slow, fp64 restatement of arXiv 2401.17074 ("PAPER.md" = the extracted text):
 *   - lattice D3Q27, c_s^2 = 1/3, weights w_i                         PAPER.md:41-45, :97 (Fig. 2)
 *   - third-order equilibrium                                          PAPER.md:135 (Eq. 14)
 *   - third-order regularised non-equilibrium                          PAPER.md:150 (Eq. 17)
 *   - recursive a^3_neq = Pi u + u Pi + u Pi                            PAPER.md:146-150 (Eq. 16-17)
 *   - thread-safe fused stream+collide: f_i(x+c_i,t+1)=f_eq+(1-w)f_neq  PAPER.md:68 (Eq. 6), :154 (Eq. 18)
 *   - second-order variant (oracle_set_order(ctx, 2)): Eq. 2 + (1-w) Eq. 7     PAPER.md:86-89 (Eq. 8)
 *   - new moments by linear local sums                                 PAPER.md:45, :126 (Eq. 12)
 *   - body force term rho w_i c_i.F / c_s^2
 *   - NEQ-extrapolation open boundaries (Dirichlet u / zero gradient)  PAPER.md:181-202 (Eq. 22-23), :258
 *   - halfway bounce-back no-slip walls  (paper only says "no-slip"; reading A12 in DESIGN.md)
 *   - sponge layer nu(z) = nu (K ((z - z_start)/(N_z - z_start))^p + 1)  PAPER.md:264-268 (Eq. 26; reading A24 in DESIGN.md)
 *
 * Readings of garbled / ambiguous passages are listed in DESIGN.md ("Readings").  In short:
 * Eq. 18's duplicated third-order equilibrium term is taken once; w_i multiplies the whole
 * bracket and rho only the equilibrium part; the second-order non-equilibrium term uses the
 * Hermite tensor H2 = cc - cs2*delta (Eq. 7), not the bare cc printed in Eq. 17.
 *
 * Two evaluation modes of the post-collision population f*:
 *   mode 0 "brute":  Hermite tensors H2, H3 built entry by entry from their definition and
 *                    contracted over all index values -- Eq. 14 / Eq. 17 as printed.
 *   mode 1 "closed": the same contractions reduced by hand to scalar products (derivation in
 *                    the comment above fstar_closed).  tests/ pin mode 1 to mode 0.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): moment reproduction (orders 0-3), uniform-flow
 * fixed point, equivalence with a two-lattice population code, mass conservation, Taylor-Green
 * viscous decay, forced Poiseuille curvature, shear stress Pi_xy = -(tau/3) rho du/dy, lattice
 * symmetries, brute-vs-closed; open faces: the populations pulled from inlet / outlet nodes equal Eq. 23 as printed
 * (built with independent numpy Hermite tensors, two time levels), uniform through-flow is a fixed point; diagnostics
 * equal the plain numpy sums; sponge layer (Eq. 26): K = 0 identity, the profile at the paper's numbers, equivalence with a
 * population code that relaxes every node with its own omega, decay rates of a two-region layer; pressure outlet: Eq. 23
 * with the imposed density, through-flow fixed point; NEQ no-slip wall: Poiseuille parabola through u = 0 at the wall
 * nodes; Gaussian noise: the Box-Muller identity through the pinned mixer and the sample moments of a unit normal; plane
 * statistics: closed-form Taylor-Green sums, numpy central moments; (r,z)-ring statistics: an analytic swirling jet via
 * numpy hypot / bincount, the axis node, rotation invariance.  Still PARITY UNPINNED (readings, nothing in the paper or the mathematics fixes them):
 * A13's nozzle geometry (top-hat disc on a full inlet plane), A14's noise law (uniform, relative) and A16's clamp rule
 * where several open faces meet.
 *
 * Layout of every moment array: [10][nz][ny][nx] doubles, x fastest;
 * field order rho, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz  (Pi = non-equilibrium momentum flux).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NF 10

enum { FACE_XLO = 0, FACE_XHI, FACE_YLO, FACE_YHI, FACE_ZLO, FACE_ZHI };
enum { BC_PERIODIC = 0, BC_BOUNCE_BACK = 1, BC_VELOCITY_INLET = 2, BC_OUTLET_ZERO_GRADIENT = 3, BC_OUTLET_PRESSURE = 5 };
#define NOISE_GAUSSIAN 0x100   /* bit 8 of the noise mask: Gaussian law instead of the uniform one */

typedef struct {
    int n[3];              /* nx, ny, nz */
    double tau, omega;     /* omega = 1/tau, nu = cs2 (1/omega - 1/2) */
    double g[3];           /* body acceleration */
    int order;             /* Hermite order of the expansion: 3 (Eq. 18, default) or 2 (Eq. 8) */
    double *omega_z;       /* sponge layer: relaxation frequency of the nodes of plane z, or NULL (uniform omega) */
    int kind[6];           /* per face */
    double *uin[6];        /* inlet planes [3][n_b][n_a], owned copy, or NULL */
    double noise_amp[6];
    uint64_t seed[6];
    int noise_mask[6];
    double rho_out[6];     /* imposed density of a pressure outlet */
    double *M[2];          /* ping-pong ("AB flip-flop") moment buffers */
    int cur;
    long long t;
    int have_state;
} oracle_ctx;

static const double CS2 = 1.0 / 3.0;

/* D3Q27 weights as a tensor product: w(0) = 2/3, w(+-1) = 1/6  ->  8/27, 2/27, 1/54, 1/216
 * for rest / |c|=1 / |c|=sqrt2 / |c|=sqrt3 (the three shells of Fig. 2). */
static double w1(int c) { return c == 0 ? 2.0 / 3.0 : 1.0 / 6.0; }

static void unpack(const double M[NF], double *rho, double u[3], double Pi[3][3])
{
    *rho = M[0];
    u[0] = M[1]; u[1] = M[2]; u[2] = M[3];
    Pi[0][0] = M[4]; Pi[1][1] = M[5]; Pi[2][2] = M[6];
    Pi[0][1] = Pi[1][0] = M[7];
    Pi[0][2] = Pi[2][0] = M[8];
    Pi[1][2] = Pi[2][1] = M[9];
}

/* f*_c(M) = w_c [ rho (1 + c.u/cs2 + H2:uu/(2 cs4) + H3:uuu/(6 cs6))              Eq. 14
 *               + (1-omega) ( H2:Pi/(2 cs4) + H3:a3/(6 cs6) )                      Eq. 17
 *               + rho c.g/cs2 ]
 * with a3_abg = Pi_ab u_g + u_a Pi_bg + u_b Pi_ag                                  Eq. 17
 * Mode 0: tensors built from the definitions, all index values summed.            */
static double fstar_brute(const double M[NF], const int c[3], double omega, const double g[3], int order)
{
    double rho, u[3], Pi[3][3];
    unpack(M, &rho, u, Pi);
    double H2[3][3], H3[3][3][3];
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            H2[a][b] = (double)(c[a] * c[b]) - CS2 * (a == b);
            for (int d = 0; d < 3; ++d)
                H3[a][b][d] = (double)(c[a] * c[b] * c[d])
                              - CS2 * (c[d] * (a == b) + c[a] * (b == d) + c[b] * (a == d));
        }
    double cu = 0, cg = 0, eq2 = 0, eq3 = 0, ne2 = 0, ne3 = 0;
    for (int a = 0; a < 3; ++a) {
        cu += c[a] * u[a];
        cg += c[a] * g[a];
        for (int b = 0; b < 3; ++b) {
            eq2 += H2[a][b] * u[a] * u[b];
            ne2 += H2[a][b] * Pi[a][b];
            for (int d = 0; d < 3; ++d) {
                double a3 = Pi[a][b] * u[d] + u[a] * Pi[b][d] + u[b] * Pi[a][d];
                eq3 += H3[a][b][d] * u[a] * u[b] * u[d];
                ne3 += H3[a][b][d] * a3;
            }
        }
    }
    const double cs4 = CS2 * CS2, cs6 = cs4 * CS2;
    double w = w1(c[0]) * w1(c[1]) * w1(c[2]);
    if (order < 3) { eq3 = 0.0; ne3 = 0.0; }   /* Eq. 8: the expansion stops at the second-order Hermite terms */
    return w * (rho * (1.0 + cu / CS2 + eq2 / (2.0 * cs4) + eq3 / (6.0 * cs6))
                + (1.0 - omega) * (ne2 / (2.0 * cs4) + ne3 / (6.0 * cs6))
                + rho * cg / CS2);
}

/* Mode 1: the same, with the contractions done by hand (c = c_i, tr = trace):
 *   H2:uu  = (c.u)^2 - cs2 |u|^2
 *   H3:uuu = (c.u)^3 - 3 cs2 (c.u) |u|^2
 *   H2:Pi  = c.Pi.c - cs2 tr Pi
 *   H3:a3  = ccc:a3 - 3 cs2 c_g a3_aag            (a3 is fully symmetric)
 *          = 3 (c.Pi.c)(c.u) - 3 cs2 [ trPi (c.u) + 2 c.Pi.u ]                       */
static double fstar_closed(const double M[NF], const int c[3], double omega, const double g[3], int order)
{
    double rho, u[3], Pi[3][3];
    unpack(M, &rho, u, Pi);
    double cu = 0, uu = 0, cg = 0, cPc = 0, cPu = 0, trP = 0;
    for (int a = 0; a < 3; ++a) {
        cu += c[a] * u[a];
        uu += u[a] * u[a];
        cg += c[a] * g[a];
        trP += Pi[a][a];
        for (int b = 0; b < 3; ++b) {
            cPc += c[a] * Pi[a][b] * c[b];
            cPu += c[a] * Pi[a][b] * u[b];
        }
    }
    const double cs4 = CS2 * CS2, cs6 = cs4 * CS2;
    double eq2 = cu * cu - CS2 * uu;
    double eq3 = cu * cu * cu - 3.0 * CS2 * cu * uu;
    double ne2 = cPc - CS2 * trP;
    double ne3 = 3.0 * cPc * cu - 3.0 * CS2 * (trP * cu + 2.0 * cPu);
    double w = w1(c[0]) * w1(c[1]) * w1(c[2]);
    if (order < 3) { eq3 = 0.0; ne3 = 0.0; }   /* Eq. 8: the expansion stops at the second-order Hermite terms */
    return w * (rho * (1.0 + cu / CS2 + eq2 / (2.0 * cs4) + eq3 / (6.0 * cs6))
                + (1.0 - omega) * (ne2 / (2.0 * cs4) + ne3 / (6.0 * cs6))
                + rho * cg / CS2);
}

double oracle_fstar_order(const double *M10, const int *c3, double omega, const double *g3, int mode, int order)
{
    return mode == 0 ? fstar_brute(M10, c3, omega, g3, order) : fstar_closed(M10, c3, omega, g3, order);
}
double oracle_fstar(const double *M10, const int *c3, double omega, const double *g3, int mode)
{
    return oracle_fstar_order(M10, c3, omega, g3, mode, 3);
}

/* ---- inlet noise (reading A14 in DESIGN.md) ---------------------------------------------
 * xi(seed, t, idx) in [-1, 1): top 24 bits of a 64-bit avalanche hash, so the value is exact
 * in fp32 and fp64.  mix64 is the finaliser of Vigna's public-domain SplitMix64 generator
 * (pinned in tests against that generator's published output stream).                       */
static uint64_t mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
uint64_t oracle_mix64(uint64_t z) { return mix64(z); }

uint32_t oracle_noise_r24(uint64_t seed, long long t, long long idx)
{
    uint64_t k = mix64(seed ^ (0x9E3779B97F4A7C15ULL * (uint64_t)(t + 1)));
    k = mix64(k + (uint64_t)idx);
    return (uint32_t)(k >> 40);
}
/* Gaussian variant ("time-varying Gaussian noise"; reading A14b in DESIGN.md): Box-Muller on two uniforms of
 * the same counter-based stream, u1 = (r24 + 1) / 2^24 in (0, 1] from the first hash, u2 = r24' / 2^24 in [0, 1) from the
 * hash of that hash:  xi = sqrt(-2 ln u1) cos(2 pi u2)  -- zero mean, unit variance. */
double oracle_noise_gauss(uint64_t seed, long long t, long long idx)
{
    uint64_t k = mix64(seed ^ (0x9E3779B97F4A7C15ULL * (uint64_t)(t + 1)));
    uint64_t a = mix64(k + (uint64_t)idx);
    uint64_t b = mix64(a);
    double u1 = ((double)(uint32_t)(a >> 40) + 1.0) / 16777216.0;
    double u2 = (double)(uint32_t)(b >> 40) / 16777216.0;
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

double oracle_noise_xi(uint64_t seed, long long t, long long idx)
{
    return (double)oracle_noise_r24(seed, t, idx) / 8388608.0 - 1.0;   /* 2 r / 2^24 - 1 */
}

/* ---- context ---------------------------------------------------------------------------- */
int oracle_create(int nx, int ny, int nz, double tau, oracle_ctx **out)
{
    if (!out || nx < 3 || ny < 3 || nz < 3 || !(tau > 0.5) || !isfinite(tau)) return 1;
    oracle_ctx *c = (oracle_ctx *)calloc(1, sizeof *c);
    if (!c) return 2;
    c->n[0] = nx; c->n[1] = ny; c->n[2] = nz;
    c->tau = tau; c->omega = 1.0 / tau;
    c->order = 3;
    size_t N = (size_t)nx * ny * nz;
    c->M[0] = (double *)malloc(sizeof(double) * NF * N);
    c->M[1] = (double *)malloc(sizeof(double) * NF * N);
    if (!c->M[0] || !c->M[1]) { free(c->M[0]); free(c->M[1]); free(c); return 2; }
    *out = c;
    return 0;
}

void oracle_destroy(oracle_ctx *c)
{
    if (!c) return;
    for (int f = 0; f < 6; ++f) free(c->uin[f]);
    free(c->omega_z);
    free(c->M[0]); free(c->M[1]); free(c);
}

int oracle_set_moments(oracle_ctx *c, const double *src)
{
    if (!c || !src) return 1;
    size_t N = (size_t)c->n[0] * c->n[1] * c->n[2];
    memcpy(c->M[c->cur], src, sizeof(double) * NF * N);
    c->t = 0; c->have_state = 1;
    return 0;
}

/* Hermite order of the reconstruction: 3 = Eq. 18 (high-order TSLB), 2 = Eq. 8 (the second-order TSLB of ref. 10). */
int oracle_set_order(oracle_ctx *c, int order)
{
    if (!c || (order != 2 && order != 3)) return 1;
    c->order = order;
    return 0;
}

/* Sponge layer (Eq. 26): the kinematic viscosity grows towards the z = N_z exit,
 *     nu_sponge(z) = nu ( K ((z - z_start) / (N_z - z_start))^p + 1 )   for z >= z_start,   nu otherwise,
 * and with it the relaxation time of the nodes of that plane, tau(z) = 1/2 + nu_sponge(z)/cs2.
 * Reading A24: the printed denominator "N_z - z_end" is the width of the layer, N_z - z_start, and the
 * printed exponent "p = -3" is p = +3 (a negative exponent diverges at z = z_start); p is an argument here.
 * The collision is local (Eq. 6): the population that leaves a node was relaxed with THAT node's omega, so the sweep
 * takes omega of the upstream (source) node.  K = 0 removes the layer. */
int oracle_set_sponge(oracle_ctx *c, int z_start, double K, double p)
{
    if (!c || !isfinite(K) || !isfinite(p) || K < 0) return 1;
    free(c->omega_z); c->omega_z = NULL;
    if (K == 0) return 0;
    const int nz = c->n[2];
    if (z_start < 0 || z_start >= nz) return 1;
    c->omega_z = (double *)malloc(sizeof(double) * nz);
    if (!c->omega_z) return 2;
    const double nu = CS2 * (c->tau - 0.5);
    for (int z = 0; z < nz; ++z) {
        double nu_z = nu;
        if (z >= z_start) nu_z = nu * (K * pow((double)(z - z_start) / (double)(nz - z_start), p) + 1.0);
        c->omega_z[z] = 1.0 / (0.5 + nu_z / CS2);
    }
    return 0;
}

/* tau of the nodes of plane z (for tests) */
double oracle_tau_of_plane(const oracle_ctx *c, int z)
{
    if (!c || z < 0 || z >= c->n[2]) return 0;
    return c->omega_z ? 1.0 / c->omega_z[z] : c->tau;
}

int oracle_set_force(oracle_ctx *c, const double *g3)
{
    if (!c || !g3) return 1;
    for (int a = 0; a < 3; ++a) { if (!isfinite(g3[a])) return 1; c->g[a] = g3[a]; }
    return 0;
}

/* face plane extents: the two in-plane axes of face f, lower axis index first (a fastest). */
static void face_axes(int f, int *ax, int *a, int *b)
{
    *ax = f / 2;
    *a = (*ax == 0) ? 1 : 0;
    *b = (*ax == 2) ? 1 : 2;
}

int oracle_set_face(oracle_ctx *c, int face, int kind, const double *u_plane, double noise_amp,
                    uint64_t seed, int noise_mask)
{
    if (!c || face < 0 || face > 5 || kind < 0 || kind > 3) return 1;
    free(c->uin[face]); c->uin[face] = NULL;
    c->kind[face] = kind;
    if (kind == BC_VELOCITY_INLET) {
        if (!u_plane) return 1;
        int ax, a, b; face_axes(face, &ax, &a, &b);
        size_t cnt = (size_t)3 * c->n[a] * c->n[b];
        c->uin[face] = (double *)malloc(sizeof(double) * cnt);
        if (!c->uin[face]) return 2;
        memcpy(c->uin[face], u_plane, sizeof(double) * cnt);
        c->noise_amp[face] = noise_amp; c->seed[face] = seed; c->noise_mask[face] = noise_mask;
    }
    return 0;
}

static int is_open(int kind) { return kind == BC_VELOCITY_INLET || kind == BC_OUTLET_ZERO_GRADIENT || kind == BC_OUTLET_PRESSURE; }

/* Pressure (density-imposed) outlet, PAPER.md:187 ("imposing the hydrodynamic variables at the boundary (either momentum
 * or density/pressure)") and :202: the boundary node takes u and Pi_neq of x_F and the imposed rho. */
int oracle_set_pressure_outlet(oracle_ctx *c, int face, double rho)
{
    if (!c || face < 0 || face > 5 || !(rho > 0) || !isfinite(rho)) return 1;
    free(c->uin[face]); c->uin[face] = NULL;
    c->kind[face] = BC_OUTLET_PRESSURE;
    c->rho_out[face] = rho;
    return 0;
}

/* A node is a boundary node if it lies on a face of kind INLET/OUTLET (step 1 of the update). */
static int on_open_face(const oracle_ctx *c, const int p[3])
{
    for (int ax = 0; ax < 3; ++ax) {
        if (p[ax] == 0 && is_open(c->kind[2 * ax])) return 1;
        if (p[ax] == c->n[ax] - 1 && is_open(c->kind[2 * ax + 1])) return 1;
    }
    return 0;
}

static size_t lin(const oracle_ctx *c, const int p[3])
{
    return ((size_t)p[2] * c->n[1] + p[1]) * c->n[0] + p[0];
}

/* Step 1 -- ghost fill of the boundary nodes at time t (Eq. 22-23):
 * non-equilibrium moments (and rho) come from the nearest interior node x_F, the velocity is
 * imposed (inlet) or copied (zero-gradient outlet).  x_F = x_B with every coordinate on an open
 * axis clamped to [1, n-2].  Inlet wins where faces meet; lowest inlet face index wins.        */
static void ghost_fill(oracle_ctx *c, double *M)
{
    const int nx = c->n[0], ny = c->n[1], nz = c->n[2];
    const size_t N = (size_t)nx * ny * nz;
    int any = 0;
    for (int f = 0; f < 6; ++f) any |= is_open(c->kind[f]);
    if (!any) return;
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                int p[3] = { x, y, z };
                if (!on_open_face(c, p)) continue;
                int q[3] = { x, y, z };
                for (int ax = 0; ax < 3; ++ax) {
                    int open_axis = is_open(c->kind[2 * ax]) || is_open(c->kind[2 * ax + 1]);
                    if (!open_axis) continue;
                    if (q[ax] == 0 && is_open(c->kind[2 * ax])) q[ax] = 1;
                    if (q[ax] == c->n[ax] - 1 && is_open(c->kind[2 * ax + 1])) q[ax] = c->n[ax] - 2;
                }
                size_t ib = lin(c, p), iF = lin(c, q);
                for (int k = 0; k < NF; ++k) M[k * N + ib] = M[k * N + iF];
                for (int f = 0; f < 6; ++f) {        /* imposed density (lowest pressure face that holds the node) */
                    if (c->kind[f] != BC_OUTLET_PRESSURE) continue;
                    int on = (f % 2 == 0) ? (p[f / 2] == 0) : (p[f / 2] == c->n[f / 2] - 1);
                    if (!on) continue;
                    M[ib] = c->rho_out[f];
                    break;
                }
                for (int f = 0; f < 6; ++f) {
                    if (c->kind[f] != BC_VELOCITY_INLET) continue;
                    int ax, a, b; face_axes(f, &ax, &a, &b);
                    int on = (f % 2 == 0) ? (p[ax] == 0) : (p[ax] == c->n[ax] - 1);
                    if (!on) continue;
                    size_t pl = (size_t)c->n[a] * c->n[b];
                    size_t j = (size_t)p[b] * c->n[a] + p[a];
                    double xi = (c->noise_mask[f] & NOISE_GAUSSIAN) ? oracle_noise_gauss(c->seed[f], c->t, (long long)ib)
                                                                    : oracle_noise_xi(c->seed[f], c->t, (long long)ib);
                    for (int k = 0; k < 3; ++k) {
                        double v = c->uin[f][k * pl + j];
                        if (c->noise_mask[f] & (1 << k)) v *= 1.0 + c->noise_amp[f] * xi;
                        M[(1 + k) * N + ib] = v;
                    }
                    break;
                }
            }
}

static int bc_valid(const oracle_ctx *c)
{
    for (int ax = 0; ax < 3; ++ax)
        if ((c->kind[2 * ax] == BC_PERIODIC) != (c->kind[2 * ax + 1] == BC_PERIODIC)) return 0;
    return 1;
}

/* Steps 2-5 -- one fused stream+collide sweep t -> t+1 (Eq. 18 pulled from the upstream node). */
static void sweep(oracle_ctx *c, int mode)
{
    const int nx = c->n[0], ny = c->n[1], nz = c->n[2];
    const size_t N = (size_t)nx * ny * nz;
    double *A = c->M[c->cur], *B = c->M[1 - c->cur];
    ghost_fill(c, A);
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                int p[3] = { x, y, z };
                size_t ip = lin(c, p);
                if (on_open_face(c, p)) {           /* boundary nodes are not advanced */
                    for (int k = 0; k < NF; ++k) B[k * N + ip] = A[k * N + ip];
                    continue;
                }
                double Mx[NF];
                for (int k = 0; k < NF; ++k) Mx[k] = A[k * N + ip];
                double R = 0, J[3] = { 0, 0, 0 }, S[3][3] = { { 0 } };
                for (int cz = -1; cz <= 1; ++cz)
                    for (int cy = -1; cy <= 1; ++cy)
                        for (int cx = -1; cx <= 1; ++cx) {
                            const int ci[3] = { cx, cy, cz };      /* arrival direction c_i */
                            int q[3], bounced = 0;
                            for (int ax = 0; ax < 3; ++ax) {
                                q[ax] = p[ax] - ci[ax];            /* upstream node x - c_i */
                                if (q[ax] < 0) {
                                    if (c->kind[2 * ax] == BC_PERIODIC) q[ax] += c->n[ax];
                                    else if (c->kind[2 * ax] == BC_BOUNCE_BACK) bounced = 1;
                                } else if (q[ax] >= c->n[ax]) {
                                    if (c->kind[2 * ax + 1] == BC_PERIODIC) q[ax] -= c->n[ax];
                                    else if (c->kind[2 * ax + 1] == BC_BOUNCE_BACK) bounced = 1;
                                }
                            }
                            double f;
                            if (bounced) {          /* halfway bounce-back: f_i(x,t+1) = f*_ibar(x,t) */
                                const int cb[3] = { -cx, -cy, -cz };
                                const double om = c->omega_z ? c->omega_z[z] : c->omega;
                                f = oracle_fstar_order(Mx, cb, om, c->g, mode, c->order);
                            } else {
                                double Ms[NF];
                                size_t iq = lin(c, q);
                                for (int k = 0; k < NF; ++k) Ms[k] = A[k * N + iq];
                                const double om = c->omega_z ? c->omega_z[q[2]] : c->omega;   /* omega of the source node */
                                f = oracle_fstar_order(Ms, ci, om, c->g, mode, c->order);
                            }
                            R += f;
                            for (int a = 0; a < 3; ++a) {
                                J[a] += ci[a] * f;
                                for (int b = 0; b < 3; ++b) S[a][b] += ci[a] * ci[b] * f;
                            }
                        }
                /* Eq. 12 with f_neq = f - f_eq(rho', u'): Pi' = S - rho'(cs2 delta + u'u') */
                double u[3] = { J[0] / R, J[1] / R, J[2] / R };
                B[0 * N + ip] = R;
                B[1 * N + ip] = u[0]; B[2 * N + ip] = u[1]; B[3 * N + ip] = u[2];
                B[4 * N + ip] = S[0][0] - R * (CS2 + u[0] * u[0]);
                B[5 * N + ip] = S[1][1] - R * (CS2 + u[1] * u[1]);
                B[6 * N + ip] = S[2][2] - R * (CS2 + u[2] * u[2]);
                B[7 * N + ip] = S[0][1] - R * u[0] * u[1];
                B[8 * N + ip] = S[0][2] - R * u[0] * u[2];
                B[9 * N + ip] = S[1][2] - R * u[1] * u[2];
            }
    c->cur = 1 - c->cur;
    c->t += 1;
}

int oracle_step(oracle_ctx *c, int n, int mode)
{
    if (!c || n < 0 || (mode != 0 && mode != 1)) return 1;
    if (!c->have_state) return 4;
    if (!bc_valid(c)) return 1;
    for (int s = 0; s < n; ++s) sweep(c, mode);
    return 0;
}

int oracle_get_moments(oracle_ctx *c, double *dst)
{
    if (!c || !dst) return 1;
    if (!c->have_state) return 4;
    size_t N = (size_t)c->n[0] * c->n[1] * c->n[2];
    ghost_fill(c, c->M[c->cur]);
    memcpy(dst, c->M[c->cur], sizeof(double) * NF * N);
    return 0;
}

/* mass, momentum[3], kinetic energy over non-boundary nodes (reading A26). */
int oracle_diagnostics(oracle_ctx *c, double *out5)
{
    if (!c || !out5) return 1;
    if (!c->have_state) return 4;
    const size_t N = (size_t)c->n[0] * c->n[1] * c->n[2];
    const double *M = c->M[c->cur];
    double m = 0, px = 0, py = 0, pz = 0, e = 0;
    for (int z = 0; z < c->n[2]; ++z)
        for (int y = 0; y < c->n[1]; ++y)
            for (int x = 0; x < c->n[0]; ++x) {
                int p[3] = { x, y, z };
                if (on_open_face(c, p)) continue;
                size_t i = lin(c, p);
                double r = M[i], ux = M[N + i], uy = M[2 * N + i], uz = M[3 * N + i];
                m += r; px += r * ux; py += r * uy; pz += r * uz;
                e += 0.5 * r * (ux * ux + uy * uy + uz * uz);
            }
    out5[0] = m; out5[1] = px; out5[2] = py; out5[3] = pz; out5[4] = e;
    return 0;
}

/* Running plane statistics (PAPER.md:236 Eq. 24, :242 Eq. 25): for every plane j of constant coordinate along `axis`
 * ADD to sums[13][n_axis] the sums over the nodes of the plane of
 *   1 | u_x u_y u_z | u_x u_x, u_y u_y, u_z u_z, u_x u_y, u_x u_z, u_y u_z | u_x^3 u_y^3 u_z^3
 * at the current time (boundary nodes refilled first).  Means, Reynolds stresses <u'_i u'_j> and skewness follow from
 * these raw sums; the caller zeroes the array once and calls once per sample. */
int oracle_plane_statistics(oracle_ctx *c, int axis, double *sums)
{
    if (!c || !sums || axis < 0 || axis > 2) return 1;
    if (!c->have_state) return 4;
    const size_t N = (size_t)c->n[0] * c->n[1] * c->n[2];
    const int na = c->n[axis];
    double *M = c->M[c->cur];
    ghost_fill(c, M);
    for (int z = 0; z < c->n[2]; ++z)
        for (int y = 0; y < c->n[1]; ++y)
            for (int x = 0; x < c->n[0]; ++x) {
                const int p[3] = { x, y, z };
                const size_t i = lin(c, p);
                const int j = p[axis];
                const double u[3] = { M[N + i], M[2 * N + i], M[3 * N + i] };
                sums[0 * na + j] += 1.0;
                for (int a = 0; a < 3; ++a) {
                    sums[(1 + a) * na + j] += u[a];
                    sums[(4 + a) * na + j] += u[a] * u[a];
                    sums[(10 + a) * na + j] += u[a] * u[a] * u[a];
                }
                sums[7 * na + j] += u[0] * u[1];
                sums[8 * na + j] += u[0] * u[2];
                sums[9 * na + j] += u[1] * u[2];
            }
    return 0;
}

/* Running (r, z)-bin statistics of a round jet along z (Fig. 7-8: centre-line velocity, half-width,
 * mean axial profile, axial / radial rms and the Reynolds stress <u'_z u'_r> on sections z = const).  Reading A27
 * (DESIGN.md): with (xc, yc) the jet axis in node coordinates, dx = x - xc, dy = y - yc, r = sqrt(dx^2 + dy^2), a node
 * belongs to bin k = floor(r / dr) of its plane if k < nr; the cylindrical components are u_r = (u_x dx + u_y dy) / r,
 * u_t = (u_y dx - u_x dy) / r (both 0 on the axis, r = 0).  For every plane z and bin k ADD to sums[8][nz][nr]
 *     1 | u_z | u_r | u_t | u_z^2 | u_r^2 | u_t^2 | u_z u_r
 * at the current time (boundary nodes refilled first); the caller zeroes the array once and calls once per sample. */
int oracle_radial_statistics(oracle_ctx *c, double xc, double yc, double dr, int nr, double *sums)
{
    if (!c || !sums || nr < 1 || !(dr > 0) || !isfinite(xc) || !isfinite(yc)) return 1;
    if (!c->have_state) return 4;
    const size_t N = (size_t)c->n[0] * c->n[1] * c->n[2];
    const int nz = c->n[2];
    double *M = c->M[c->cur];
    ghost_fill(c, M);
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < c->n[1]; ++y)
            for (int x = 0; x < c->n[0]; ++x) {
                const double dx = x - xc, dy = y - yc;
                const double r = sqrt(dx * dx + dy * dy);
                const double kf = floor(r / dr);
                if (!(kf < nr)) continue;
                const int k = (int)kf;
                const int p[3] = { x, y, z };
                const size_t i = lin(c, p);
                const double ux = M[N + i], uy = M[2 * N + i], uz = M[3 * N + i];
                double ur = 0, ut = 0;
                if (r > 0) { ur = (ux * dx + uy * dy) / r; ut = (uy * dx - ux * dy) / r; }
                double *s = sums + (size_t)z * nr + k;
                const size_t row = (size_t)nz * nr;
                s[0 * row] += 1.0;
                s[1 * row] += uz; s[2 * row] += ur; s[3 * row] += ut;
                s[4 * row] += uz * uz; s[5 * row] += ur * ur; s[6 * row] += ut * ut;
                s[7 * row] += uz * ur;
            }
    return 0;
}

long long oracle_step_count(const oracle_ctx *c) { return c ? c->t : -1; }

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

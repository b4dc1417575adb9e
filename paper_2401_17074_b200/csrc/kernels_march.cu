// kernels_march.cu -- the register-marching SEPARABLE sweep (the fast path of tslb_step) for sm_100a.
//
// Same update as the gather kernel (Eq. 18 + Eq. 12), evaluated in the form derived in
// the post-collision population of a source node is linear in 17 Hermite
// coefficients A_k of that node (k = (kx,ky,kz), k_a <= 2, |k| <= 3; Eq. 13, 16, 17), and because D3Q27 and its
// Hermite basis are tensor products the 27-direction pull + moment sums factor into three 1-D 3-tap passes
//       M'_p(x) = sum_k  T^x_{px,kx} T^y_{py,ky} T^z_{pz,kz}  A_k ,      T_{p,q} phi (x) = sum_c w(c) c^p h_q(c) phi(x - c).
// With every field scaled by 216 (and the q = 2 fields by a further 2/3) all taps are the small integers
// 1, 4, -2, so no rounded lattice weight ever multiplies the data: that removes the systematic per-step gain
// that rounded w_i give in fp32.  One exact-scaling division at the end.
//
// Mapping: a thread owns one x column and TWO adjacent y rows, packed in a 2-wide register pair so that fp32
// arithmetic issues as FFMA2/FADD2 (sm_100 packed fp32); it marches along z.
//   y pass: in registers, from the A_k of rows r0-1 .. r0+2 (halo rows recomputed),
//   x pass: neighbours' values by warp shuffles (warps overlap by one halo lane on each side),
//   z pass: by marching -- 3 running values per (px,py) group, no plane is read twice.
// Each node's moments are read from global memory once per row pair (+ halo rows, which hit L1/L2) and the
// 10 new moments are written once: 80 B (fp32) / 160 B (fp64) of compulsory traffic per node update.
#include "tslb_internal.h"

namespace {

// ---- 2-wide packs --------------------------------------------------------------------------------------
struct D2 { double x, y; };
template <typename T> struct PackOf;
template <> struct PackOf<float> { typedef float2 type; };
template <> struct PackOf<double> { typedef D2 type; };

__device__ __forceinline__ float2 pk(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ D2 pk(double a, double b) { D2 r; r.x = a; r.y = b; return r; }
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 pmul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 psub(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
__device__ __forceinline__ D2 padd(D2 a, D2 b) { return pk(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ D2 pmul(D2 a, D2 b) { return pk(a.x * b.x, a.y * b.y); }
__device__ __forceinline__ D2 pfma(D2 a, D2 b, D2 c) { return pk(fma(a.x, b.x, c.x), fma(a.y, b.y, c.y)); }
__device__ __forceinline__ D2 psub(D2 a, D2 b) { return pk(a.x - b.x, a.y - b.y); }
template <typename P, typename T> __device__ __forceinline__ P pbc(T s) { return pk(s, s); }
// a*s + c and a*s with a scalar s
template <typename P, typename T> __device__ __forceinline__ P pfmas(P a, T s, P c) { return pfma(a, pbc<P, T>(s), c); }
template <typename P, typename T> __device__ __forceinline__ P pmuls(P a, T s) { return pmul(a, pbc<P, T>(s)); }

template <typename P> __device__ __forceinline__ P shfl_up1(P v)
{
    return pk(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1));
}
template <typename P> __device__ __forceinline__ P shfl_dn1(P v)
{
    return pk(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1));
}

template <typename T>
struct MarchParams {
    int nx, ny, nz;
    int kind[6];
    T beta, g[3];
    int nseg;    // x segments (warps per row); segment s outputs columns [s*nx/nseg, (s+1)*nx/nseg)
    int zchunk;  // planes per z chunk
};

// valid Hermite index: each <= 2, sum <= 3 (H3_aaa == 0 on this lattice)
__host__ __device__ constexpr bool kvalid(int kx, int ky, int kz) { return kx <= 2 && ky <= 2 && kz <= 2 && kx + ky + kz <= 3; }

// ---- Hermite coefficients of one pack of two nodes, round kz (216-scaled, integer prefactors) -----------
//   A000 = drho                       A100 = 3 rho (ux+gx) ...          (Eq. 13; force PAPER.md:216)
//   A200 = 3 (rho ux ux + beta Pxx)   A110 = 9 (rho ux uy + beta Pxy)   (Eq. 13 + Eq. 7/17, n = 2)
//   A210 = 9 a3_xxy, A111 = 27 a3_xyz,  a3_abg = rho ua ub ug + beta (Pab ug + ua Pbg + ub Pag)   (Eq. 16-17)
// raw[]: drho, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz.  Out: A[kx][ky] for this kz.
template <int KZ, typename P, typename T>
__device__ __forceinline__ void hermite_round(const P (&raw)[TSLB_NF], T beta, const T (&g)[3], P (&A)[3][3])
{
    const P one = pbc<P, T>((T)1);
    const P rho = padd(one, raw[0]);
    const P r3 = pmuls(rho, (T)3);
    const P ux = raw[1], uy = raw[2], uz = raw[3];
    const T b3 = (T)3 * beta, b9 = (T)9 * beta;
    if (KZ == 0) {
        const P m3x = pmul(r3, ux), m3y = pmul(r3, uy);
        const P q9xy = pmuls(raw[7], b9);
        const P a20 = pfma(m3x, ux, pmuls(raw[4], b3));
        const P a02 = pfma(m3y, uy, pmuls(raw[5], b3));
        A[0][0] = raw[0];
        A[1][0] = pmul(r3, padd(ux, pbc<P, T>(g[0])));
        A[0][1] = pmul(r3, padd(uy, pbc<P, T>(g[1])));
        A[2][0] = a20;
        A[0][2] = a02;
        A[1][1] = pfma(pmuls(m3x, (T)3), uy, q9xy);
        A[2][1] = pfma(padd(ux, ux), q9xy, pmul(a20, pmuls(uy, (T)3)));
        A[1][2] = pfma(padd(uy, uy), q9xy, pmul(a02, pmuls(ux, (T)3)));
    } else if (KZ == 1) {
        const P m3x = pmul(r3, ux), m3y = pmul(r3, uy);
        const P m9x = pmuls(m3x, (T)3), m9y = pmuls(m3y, (T)3);
        const P q9xy = pmuls(raw[7], b9), q9xz = pmuls(raw[8], b9), q9yz = pmuls(raw[9], b9);
        const P a200 = pfma(m3x, ux, pmuls(raw[4], b3));
        const P a020 = pfma(m3y, uy, pmuls(raw[5], b3));
        const P a110 = pfma(m9x, uy, q9xy);
        const P u3x = pmuls(ux, (T)3), u3y = pmuls(uy, (T)3), u3z = pmuls(uz, (T)3);
        A[0][0] = pmul(r3, padd(uz, pbc<P, T>(g[2])));
        A[1][0] = pfma(m9x, uz, q9xz);
        A[0][1] = pfma(m9y, uz, q9yz);
        A[2][0] = pfma(padd(ux, ux), q9xz, pmul(a200, u3z));
        A[0][2] = pfma(padd(uy, uy), q9yz, pmul(a020, u3z));
        A[1][1] = pfma(u3x, q9yz, pfma(u3y, q9xz, pmul(u3z, a110)));
    } else {
        const P m3z = pmul(r3, uz);
        const P q9xz = pmuls(raw[8], b9), q9yz = pmuls(raw[9], b9);
        const P a002 = pfma(m3z, uz, pmuls(raw[6], b3));
        const P uz2 = padd(uz, uz);
        A[0][0] = a002;
        A[1][0] = pfma(uz2, q9xz, pmul(a002, pmuls(ux, (T)3)));
        A[0][1] = pfma(uz2, q9yz, pmul(a002, pmuls(uy, (T)3)));
    }
}

// ---- one 1-D pass on a group of up to three fields q = 0,1,2 given S_q = phi(-1)+phi(+1), D_q = phi(-1)-phi(+1)
//      and the centre values c0, c2:      out0 = E + 4 c0 - 2 c2,  out1 = D0 + S1 + D2,  out2 = E = S0 + D1 + S2
template <int NQ, typename P, typename T>
__device__ __forceinline__ void pass_group(const P (&S)[3], const P (&D)[3], P c0, P c2, P &o0, P &o1, P &o2)
{
    P E = S[0];
    P O = D[0];
    if (NQ >= 2) { E = padd(E, D[1]); O = padd(O, S[1]); }
    if (NQ >= 3) { E = padd(E, S[2]); O = padd(O, D[2]); }
    o2 = E;
    o1 = O;
    o0 = pfmas(c0, (T)4, E);
    if (NQ >= 3) o0 = pfmas(c2, (T)-2, o0);
}

__device__ __forceinline__ bool open_kind(int k) { return k == TSLB_BC_VELOCITY_INLET || k == TSLB_BC_OUTLET_ZERO_GRADIENT; }

// Contribution of the bounced directions at a node next to a halfway bounce-back wall on a y face
// (DESIGN.md "Walls in the separable form"): f_i(x,t+1) = f*_ibar(x,t) for the 9 directions with c_y = sgn_in,
// evaluated from the node's own 216-scaled Hermite coefficients.  Adds to out[10] (216-scaled raw moments in the
// order 000,100,010,001,200,020,002,110,101,011).  lo_wall: wall below (arrival c_y = +1), else above.
template <typename T>
__device__ __noinline__ void bounce_y_correction(const T *__restrict__ Abuf, size_t N, size_t idx, T beta, const T (&g)[3],
                                                 bool lo_wall, T (&out)[TSLB_NF])
{
    T raw[TSLB_NF];
#pragma unroll
    for (int f = 0; f < TSLB_NF; ++f) raw[f] = __ldg(Abuf + f * N + idx);
    const T rho = (T)1 + raw[0], ux = raw[1], uy = raw[2], uz = raw[3];
    const T u[3] = {ux, uy, uz};
    const T Pm[3][3] = {{raw[4], raw[7], raw[8]}, {raw[7], raw[5], raw[9]}, {raw[8], raw[9], raw[6]}};
    T a2[3][3];
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) a2[a][b] = rho * u[a] * u[b] + beta * Pm[a][b];
    // A(kx,ky,kz), scaled as in hermite_round
    T A[3][3][3];
    for (int i = 0; i < 27; ++i) (&A[0][0][0])[i] = (T)0;
    A[0][0][0] = raw[0];
    A[1][0][0] = (T)3 * rho * (ux + g[0]); A[0][1][0] = (T)3 * rho * (uy + g[1]); A[0][0][1] = (T)3 * rho * (uz + g[2]);
    A[2][0][0] = (T)3 * a2[0][0]; A[0][2][0] = (T)3 * a2[1][1]; A[0][0][2] = (T)3 * a2[2][2];
    A[1][1][0] = (T)9 * a2[0][1]; A[1][0][1] = (T)9 * a2[0][2]; A[0][1][1] = (T)9 * a2[1][2];
    // a3_aab = a2_aa u_b + 2 u_a beta P_ab
    A[2][1][0] = (T)9 * (a2[0][0] * uy + (T)2 * ux * beta * Pm[0][1]);
    A[2][0][1] = (T)9 * (a2[0][0] * uz + (T)2 * ux * beta * Pm[0][2]);
    A[1][2][0] = (T)9 * (a2[1][1] * ux + (T)2 * uy * beta * Pm[0][1]);
    A[0][2][1] = (T)9 * (a2[1][1] * uz + (T)2 * uy * beta * Pm[1][2]);
    A[1][0][2] = (T)9 * (a2[2][2] * ux + (T)2 * uz * beta * Pm[0][2]);
    A[0][1][2] = (T)9 * (a2[2][2] * uy + (T)2 * uz * beta * Pm[1][2]);
    A[1][1][1] = (T)27 * (a2[0][1] * uz + beta * (Pm[0][2] * uy + Pm[1][2] * ux));
    // B(kx,kz) = sum_ky s^ky A(kx,ky,kz), s = t_ky(-c_y): wall below -> t(-1) = (1,-1,1); above -> t(+1) = (1,1,1)
    const T s1 = lo_wall ? (T)-1 : (T)1;
    T Bm[3][3];
    for (int kx = 0; kx < 3; ++kx)
        for (int kz = 0; kz < 3; ++kz) Bm[kx][kz] = A[kx][0][kz] + s1 * A[kx][1][kz] + A[kx][2][kz];
    const T sg = lo_wall ? (T)1 : (T)-1;  // c_y^py of the arrival direction
    // local sums L(p,q) = sum_c c^p t_q(-c): L(0,0)=6, L(1,1)=-2, L(2,0)=2, L(2,2)=2, others 0
    out[0] += (T)36 * Bm[0][0];
    out[1] += (T)-12 * Bm[1][0];
    out[2] += sg * (T)36 * Bm[0][0];
    out[3] += (T)-12 * Bm[0][1];
    out[4] += (T)12 * (Bm[0][0] + Bm[2][0]);
    out[5] += (T)36 * Bm[0][0];
    out[6] += (T)12 * (Bm[0][0] + Bm[0][2]);
    out[7] += sg * (T)-12 * Bm[1][0];
    out[8] += (T)4 * Bm[1][1];
    out[9] += sg * (T)-12 * Bm[0][1];
}

// finalise one node from its 216-scaled raw moments and store (Eq. 12; exact scaling, no rounded weights)
template <typename T>
__device__ __forceinline__ void finalize_store(const T (&m)[TSLB_NF], T *__restrict__ Bbuf, size_t N, size_t idx)
{
    // x/216 as x*hi + x*lo: unbiased to ~1 ulp (a rounded 1/216 alone would be a systematic gain)
    const T hi = (T)(1.0 / 216.0);
    const T lo = (T)(1.0 / 216.0 - (double)hi);
    const T dR = fma(m[0], lo, m[0] * hi);
    const T rho = (T)1 + dR;
    const T inv = (T)1 / ((T)216 + m[0]);
    const T ux = m[1] * inv, uy = m[2] * inv, uz = m[3] * inv;
    const T third = (T)(1.0 / 3.0);
    const T iso = third * dR;
    Bbuf[idx] = dR;
    Bbuf[N + idx] = ux;
    Bbuf[2 * N + idx] = uy;
    Bbuf[3 * N + idx] = uz;
    Bbuf[4 * N + idx] = fma(m[4], lo, m[4] * hi) - iso - rho * ux * ux;
    Bbuf[5 * N + idx] = fma(m[5], lo, m[5] * hi) - iso - rho * uy * uy;
    Bbuf[6 * N + idx] = fma(m[6], lo, m[6] * hi) - iso - rho * uz * uz;
    Bbuf[7 * N + idx] = fma(m[7], lo, m[7] * hi) - rho * ux * uy;
    Bbuf[8 * N + idx] = fma(m[8], lo, m[8] * hi) - rho * ux * uz;
    Bbuf[9 * N + idx] = fma(m[9], lo, m[9] * hi) - rho * uy * uz;
}

#define MARCH_WARPS 4

// index of group (px,py), px+py <= 2, in the z-march state: (0,0)=0 (1,0)=1 (2,0)=2 (0,1)=3 (1,1)=4 (0,2)=5
__host__ __device__ constexpr int gidx(int px, int py) { return py == 0 ? px : (py == 1 ? 3 + px : 5); }

template <typename T>
__global__ void __launch_bounds__(MARCH_WARPS * 32) sweep_march_kernel(const T *__restrict__ Abuf, T *__restrict__ Bbuf,
                                                                        MarchParams<T> p)
{
    typedef typename PackOf<T>::type P;
    const int lane = threadIdx.x & 31;
    const int wid = threadIdx.x >> 5;
    const size_t N = (size_t)p.nx * p.ny * p.nz;
    const size_t plane = (size_t)p.nx * p.ny;

    // ---- columns: segment s outputs [xs, xe); lane l holds column xs - 1 + l ----------------------------
    const int seg = blockIdx.x;
    const int xs = (int)(((long long)seg * p.nx) / p.nseg);
    const int xe = (int)(((long long)(seg + 1) * p.nx) / p.nseg);
    int col = xs - 1 + lane;
    const bool col_out = lane >= 1 && col < xe;  // this lane produces output
    if (p.kind[0] == TSLB_BC_PERIODIC) { col %= p.nx; if (col < 0) col += p.nx; }
    else col = min(max(col, 0), p.nx - 1);       // beyond an open face: value never used

    // ---- rows: pack .x = row r0, .y = row r0+1; halo rows r0-1, r0+2 ---------------------------------------
    const int r0 = 2 * (blockIdx.y * MARCH_WARPS + wid);
    if (r0 >= p.ny) return;                      // whole warp exits together
    int rows[4];
    bool ghost_lo = false, ghost_hi = false;     // halo row lies beyond a bounce-back wall: contributes nothing
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        int r = r0 - 1 + j;
        if (r < 0) {
            if (p.kind[2] == TSLB_BC_PERIODIC) r += p.ny;
            else { if (p.kind[2] == TSLB_BC_BOUNCE_BACK) ghost_lo = true; r = 0; }
        } else if (r >= p.ny) {
            if (p.kind[3] == TSLB_BC_PERIODIC) r = (r - p.ny) % p.ny;
            else { if (p.kind[3] == TSLB_BC_BOUNCE_BACK && r == p.ny && j == 3) ghost_hi = true; r = p.ny - 1; }
        }
        rows[j] = r;
    }
    const bool row1_valid = r0 + 1 < p.ny;
    // if ny is odd the last pair has one real row; its .y is a dummy and row r0+1 = ny is the halo of r0
    const bool ghost_mid_hi = !row1_valid && p.kind[3] == TSLB_BC_BOUNCE_BACK;  // row r0+1 beyond the upper wall
    const bool any_ghost = ghost_lo || ghost_hi || ghost_mid_hi;

    const int z0 = blockIdx.z * p.zchunk;
    const int z1 = min(z0 + p.zchunk, p.nz);

    // z-march state per (px,py) group: Vp of plane zs-2, centre term of plane zs-1, Vp of plane zs-1
    P vp2[6], cc1[6], vp1[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) { vp2[i] = pbc<P, T>((T)0); cc1[i] = vp2[i]; vp1[i] = vp2[i]; }

    for (int zs = z0 - 1; zs <= z1; ++zs) {
        int zsrc = zs;
        if (zsrc < 0) zsrc = (p.kind[4] == TSLB_BC_PERIODIC) ? p.nz - 1 : 0;
        else if (zsrc >= p.nz) zsrc = (p.kind[5] == TSLB_BC_PERIODIC) ? 0 : p.nz - 1;
        const T *src = Abuf + (size_t)zsrc * plane + col;

        // ---- a1: moments of rows r0-1 .. r0+2 at this column, packed (r0-1,r0) and (r0+1,r0+2) ---------------
        P rlo[TSLB_NF], rhi[TSLB_NF];
#pragma unroll
        for (int f = 0; f < TSLB_NF; ++f) {
            const T *s = src + f * N;
            rlo[f] = pk(__ldg(s + (size_t)rows[0] * p.nx), __ldg(s + (size_t)rows[1] * p.nx));
            rhi[f] = pk(__ldg(s + (size_t)rows[2] * p.nx), __ldg(s + (size_t)rows[3] * p.nx));
        }

        P vp0[6], vm0[6], cc0[6];  // this plane's Vp, Vm, centre term per group
#pragma unroll
        for (int kz = 0; kz < 3; ++kz) {
            // ---- a2: Hermite coefficients of the four rows for this kz --------------------------------------
            P Alo[3][3], Ahi[3][3];
            if (kz == 0) { hermite_round<0, P, T>(rlo, p.beta, p.g, Alo); hermite_round<0, P, T>(rhi, p.beta, p.g, Ahi); }
            if (kz == 1) { hermite_round<1, P, T>(rlo, p.beta, p.g, Alo); hermite_round<1, P, T>(rhi, p.beta, p.g, Ahi); }
            if (kz == 2) { hermite_round<2, P, T>(rlo, p.beta, p.g, Alo); hermite_round<2, P, T>(rhi, p.beta, p.g, Ahi); }
            if (any_ghost) {  // rows beyond a bounce-back wall send nothing (their part is added by bounce_y_correction)
#pragma unroll
                for (int kx = 0; kx < 3; ++kx)
#pragma unroll
                    for (int ky = 0; ky < 3; ++ky)
                        if (kvalid(kx, ky, kz)) {
                            if (ghost_lo) Alo[kx][ky].x = (T)0;
                            if (ghost_hi) Ahi[kx][ky].y = (T)0;
                            if (ghost_mid_hi) { Ahi[kx][ky].x = (T)0; Ahi[kx][ky].y = (T)0; }
                        }
            }
            // ---- y pass: G1[py][kx] = sum_ky T^y_{py,ky} A(kx,ky,kz) at rows r0, r0+1 -------------------------
            P G1[3][3];
#pragma unroll
            for (int kx = 0; kx < 3; ++kx) {
                if (!kvalid(kx, 0, kz)) continue;
                P S[3], D[3];
#pragma unroll
                for (int ky = 0; ky < 3; ++ky)
                    if (kvalid(kx, ky, kz)) { S[ky] = padd(Alo[kx][ky], Ahi[kx][ky]); D[ky] = psub(Alo[kx][ky], Ahi[kx][ky]); }
                const P c0 = pk(Alo[kx][0].y, Ahi[kx][0].x);
                if (kvalid(kx, 2, kz)) {
                    const P c2 = pk(Alo[kx][2].y, Ahi[kx][2].x);
                    pass_group<3, P, T>(S, D, c0, c2, G1[0][kx], G1[1][kx], G1[2][kx]);
                } else if (kvalid(kx, 1, kz)) {
                    pass_group<2, P, T>(S, D, c0, c0, G1[0][kx], G1[1][kx], G1[2][kx]);
                } else {
                    pass_group<1, P, T>(S, D, c0, c0, G1[0][kx], G1[1][kx], G1[2][kx]);
                }
            }
            // ---- x pass (warp shuffles): G2[px][py] = sum_kx T^x_{px,kx} G1[py][kx]; then the z bookkeeping ----
#pragma unroll
            for (int py = 0; py < 3; ++py) {
                P S[3], D[3];
#pragma unroll
                for (int kx = 0; kx < 3; ++kx)
                    if (kvalid(kx, 0, kz)) {
                        const P up = shfl_up1(G1[py][kx]);  // value at column-1  (c_x = +1 pulls from x-1)
                        const P dn = shfl_dn1(G1[py][kx]);  // value at column+1
                        S[kx] = padd(up, dn);
                        D[kx] = psub(up, dn);
                    }
                P o0, o1, o2;
                if (kvalid(2, 0, kz)) pass_group<3, P, T>(S, D, G1[py][0], G1[py][2], o0, o1, o2);
                else pass_group<2, P, T>(S, D, G1[py][0], G1[py][0], o0, o1, o2);
                const P o[3] = {o0, o1, o2};
#pragma unroll
                for (int px = 0; px + py <= 2; ++px) {
                    const int gi = gidx(px, py);
                    const P v = o[px];
                    // Vp = phi0 + phi1 + phi2, Vm = phi0 - phi1 + phi2, centre = 4 phi0 - 2 phi2   (over kz)
                    if (kz == 0) { vp0[gi] = v; vm0[gi] = v; cc0[gi] = pmuls(v, (T)4); }
                    if (kz == 1) { vp0[gi] = padd(vp0[gi], v); vm0[gi] = psub(vm0[gi], v); }
                    if (kz == 2) { vp0[gi] = padd(vp0[gi], v); vm0[gi] = padd(vm0[gi], v); cc0[gi] = pfmas(v, (T)-2, cc0[gi]); }
                }
            }
        }

        // ---- z pass for target plane zt = zs - 1:  pz=0: Vp(zs-2) + centre(zs-1) + Vm(zs);  pz=1: Vp(zs-2) - Vm(zs);
        //      pz=2: Vp(zs-2) + Vm(zs) --------------------------------------------------------------------------
        const int zt = zs - 1;
        if (zt >= z0 && col_out) {
            P m[TSLB_NF];
            {
                const P e00 = padd(vp2[0], vm0[0]);
                m[0] = padd(e00, cc1[0]);                                  // 000
                m[3] = psub(vp2[0], vm0[0]);                               // 001
                m[6] = e00;                                                // 002
                const P e10 = padd(vp2[1], vm0[1]);
                m[1] = padd(e10, cc1[1]);                                  // 100
                m[8] = psub(vp2[1], vm0[1]);                               // 101
                const P e01 = padd(vp2[3], vm0[3]);
                m[2] = padd(e01, cc1[3]);                                  // 010
                m[9] = psub(vp2[3], vm0[3]);                               // 011
                m[4] = padd(padd(vp2[2], vm0[2]), cc1[2]);                 // 200
                m[7] = padd(padd(vp2[4], vm0[4]), cc1[4]);                 // 110
                m[5] = padd(padd(vp2[5], vm0[5]), cc1[5]);                 // 020
            }
            const size_t i0 = (size_t)zt * plane + (size_t)r0 * p.nx + col;
            const bool zopen = (zt == 0 && open_kind(p.kind[4])) || (zt == p.nz - 1 && open_kind(p.kind[5]));
            const bool xopen = (col == 0 && open_kind(p.kind[0])) || (col == p.nx - 1 && open_kind(p.kind[1]));
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int r = r0 + s;
                if (s == 1 && !row1_valid) break;
                const size_t idx = i0 + (size_t)s * p.nx;
                const bool yopen = (r == 0 && open_kind(p.kind[2])) || (r == p.ny - 1 && open_kind(p.kind[3]));
                if (zopen || xopen || yopen) {  // boundary nodes are not advanced: M_{t+1}(x_B) := M_t(x_B)
#pragma unroll
                    for (int f = 0; f < TSLB_NF; ++f) Bbuf[f * N + idx] = __ldg(Abuf + f * N + idx);
                    continue;
                }
                T ms[TSLB_NF];
#pragma unroll
                for (int f = 0; f < TSLB_NF; ++f) ms[f] = s == 0 ? m[f].x : m[f].y;
                if (r == 0 && p.kind[2] == TSLB_BC_BOUNCE_BACK) bounce_y_correction<T>(Abuf, N, idx, p.beta, p.g, true, ms);
                if (r == p.ny - 1 && p.kind[3] == TSLB_BC_BOUNCE_BACK) bounce_y_correction<T>(Abuf, N, idx, p.beta, p.g, false, ms);
                finalize_store<T>(ms, Bbuf, N, idx);
            }
        }
        // ---- shift the march state ---------------------------------------------------------------------------------
#pragma unroll
        for (int i = 0; i < 6; ++i) { vp2[i] = vp1[i]; vp1[i] = vp0[i]; cc1[i] = cc0[i]; }
    }
}

template <typename T>
MarchParams<T> make_march(const tslb_ctx *c)
{
    MarchParams<T> p;
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz;
    for (int f = 0; f < 6; ++f) p.kind[f] = c->kind[f];
    p.beta = (T)(1.0 - c->omega);
    for (int a = 0; a < 3; ++a) p.g[a] = (T)c->g[a];
    p.nseg = (c->nx + 29) / 30;
    // z chunk: enough blocks to fill the SMs a few times over, chunks long enough to amortise the 2 halo planes
    const long long cols = (long long)p.nseg * ((c->ny + 2 * MARCH_WARPS - 1) / (2 * MARCH_WARPS));
    int chunks = (int)((8LL * c->sm_count + cols - 1) / cols);
    if (chunks < 1) chunks = 1;
    int zc = (c->nz + chunks - 1) / chunks;
    if (zc < 16) zc = c->nz < 16 ? c->nz : 16;
    p.zchunk = zc;
    return p;
}

}  // namespace

bool tslb_march_supported(const tslb_ctx *c, const char **why)
{
    // bounce-back walls are handled on the y faces only (x or z walls: gather kernel)
    for (int f = 0; f < 6; ++f)
        if (c->kind[f] == TSLB_BC_BOUNCE_BACK && (f >> 1) != 1) {
            if (why) *why = "bounce-back walls on x or z faces";
            return false;
        }
    if (why) *why = "";
    return true;
}

cudaError_t tslb_launch_march(tslb_ctx *c, cudaStream_t st)
{
    if (c->dtype == TSLB_F32) {
        MarchParams<float> p = make_march<float>(c);
        dim3 grid(p.nseg, (c->ny + 2 * MARCH_WARPS - 1) / (2 * MARCH_WARPS), (c->nz + p.zchunk - 1) / p.zchunk);
        sweep_march_kernel<float><<<grid, MARCH_WARPS * 32, 0, st>>>((const float *)c->buf[c->cur], (float *)c->buf[1 - c->cur], p);
    } else {
        MarchParams<double> p = make_march<double>(c);
        dim3 grid(p.nseg, (c->ny + 2 * MARCH_WARPS - 1) / (2 * MARCH_WARPS), (c->nz + p.zchunk - 1) / p.zchunk);
        sweep_march_kernel<double><<<grid, MARCH_WARPS * 32, 0, st>>>((const double *)c->buf[c->cur], (double *)c->buf[1 - c->cur], p);
    }
    c->launches++;
    return cudaGetLastError();
}

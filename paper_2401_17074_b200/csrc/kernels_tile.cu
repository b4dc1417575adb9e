// kernels_tile.cu -- the TMA-staged, register-marching SEPARABLE sweep (the fast path of tslb_step) for sm_100a.
//
// Same update as the gather kernel (Eq. 18 + Eq. 12), evaluated in the form derived in
// the post-collision population of a source node is linear in 17 Hermite
// coefficients A_k of that node (k = (kx,ky,kz), k_a <= 2, |k| <= 3; Eq. 13, 16, 17), and because D3Q27 and its
// Hermite basis are tensor products the 27-direction pull + moment sums factor into three 1-D 3-tap passes
//       M'_p(x) = sum_k  T^x_{px,kx} T^y_{py,ky} T^z_{pz,kz}  A_k ,      T_{p,q} phi (x) = sum_c w(c) c^p h_q(c) phi(x - c).
// With every field scaled by 216 (and the q = 2 fields by a further 2/3) all taps are the small integers
// 1, 4, -2, so no rounded lattice weight ever multiplies the data.
//
// Data path: one CTA per SM owns a 60 x 14 column of nodes (fp32: 2 x 7 warps; fp64: 60 x 8,
// 2 x 4 warps) and marches along z.  One elected thread streams the z-planes of the 10 moment fields, 64 x 16 nodes
// each (the tile plus a 1-node halo, rows 16-byte aligned), from the padded SoA buffer into a 4-deep shared-memory
// ring with TMA (cp.async.bulk.tensor.4d, mbarrier complete_tx); ghost layers in the buffer stand for the periodic
// images, so the kernel has no wrap logic, and it keeps them current itself by storing the images of the nodes it
// writes on periodic faces.  Every warp owns 2 rows (packed in a 2-wide register pair so fp32 issues as FFMA2/FADD2)
// x 32 columns (30 outputs + 2 halo lanes):
//   y pass: in registers, from the A_k of rows r0-1 .. r0+2 read from shared memory (packs (r0,r0+1) and (r0-1,r0+2)),
//   x pass: neighbours' values by warp shuffles (one combination up, one down per group),
//   z pass: by marching -- 15 running pairs per thread, no plane is staged twice.
// Each node's moments leave HBM once per tile (halo re-reads hit L2) and the 10 new moments are written once:
// 80 B (fp32) / 160 B (fp64) of compulsory traffic per node update.
//
// INCREMENT FORM: the base 3 u_a of the first-order coefficients never enters the
// passes.  A pass with taps (t-, t0, t+) applied to B*u gives (t- + t0 + t+) B u(x) + B [t- (u(x-1) - u(x)) + t+ (u(x+1) - u(x))];
// only the bracket (exact differences of stored velocities) is added at each stage, and the product of the tap sums,
// 216 u_a(x), is re-attached in closed form at the end:  u' = u + (J_small - u dR) / (216 + dR).
#include "tslb_internal.h"

namespace {

// ---- 2-wide packs --------------------------------------------------------------------------------------
struct D2 { double x, y; };
template <typename T> struct PackOf;
template <> struct PackOf<float> { typedef float2 type; };
template <> struct PackOf<double> { typedef D2 type; };

__device__ __forceinline__ float2 pk(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ D2 pk(double a, double b) { D2 r; r.x = a; r.y = b; return r; }
#ifndef TSLB_SCALAR_F32
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 pmul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 psub(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
#else
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 pmul(float2 a, float2 b) { return make_float2(a.x * b.x, a.y * b.y); }
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
__device__ __forceinline__ float2 psub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
#endif
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

// ---- TMA / mbarrier (PTX; SASS: UTMALDG, SYNCS) ----------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

template <typename T>
struct TileParams {
    Layout L;
    int kind[6];
    T beta, g[3];
    int zchunk;  // planes per z chunk
};

// valid Hermite index: each <= 2, sum <= ORDER (3: Eq. 18, H3_aaa == 0 on this lattice; 2: the second-order TSLB of Eq. 8)
template <int ORDER>
__host__ __device__ constexpr bool kvalid(int kx, int ky, int kz) { return kx <= 2 && ky <= 2 && kz <= 2 && kx + ky + kz <= ORDER; }

// ---- Hermite coefficients of one pack of two nodes, round kz (216-scaled, integer prefactors) -----------
//   A000 = drho                       A100 = 3 [rho (ux+gx) - ux]  (increment form: base 3 ux handled apart)
//   A200 = 3 (rho ux ux + beta Pxx)   A110 = 9 (rho ux uy + beta Pxy)   (Eq. 13 + Eq. 7/17, n = 2)
//   A210 = 9 a3_xxy, A111 = 27 a3_xyz,  a3_abg = rho ua ub ug + beta (Pab ug + ua Pbg + ub Pag)   (Eq. 16-17)
// raw[]: drho, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz.  Out: A[kx][ky] for this kz.
template <int KZ, typename P, typename T>
__device__ __forceinline__ void hermite_round(const P (&raw)[TSLB_NF], T beta, const T (&g)[3], P (&A)[3][3])
{
    const P one = pbc<P, T>((T)1);
    const P rho = padd(one, raw[0]);
    const P r3 = pmuls(rho, (T)3);
    const P d3 = pmuls(raw[0], (T)3);
    const P ux = raw[1], uy = raw[2], uz = raw[3];
    const T b3 = (T)3 * beta, b9 = (T)9 * beta;
    if (KZ == 0) {
        const P m3x = pmul(r3, ux), m3y = pmul(r3, uy);
        const P q9xy = pmuls(raw[7], b9);
        const P a20 = pfma(m3x, ux, pmuls(raw[4], b3));
        const P a02 = pfma(m3y, uy, pmuls(raw[5], b3));
        A[0][0] = raw[0];
        A[1][0] = pfma(d3, padd(ux, pbc<P, T>(g[0])), pbc<P, T>((T)3 * g[0]));   // 3 [g + drho (u + g)]
        A[0][1] = pfma(d3, padd(uy, pbc<P, T>(g[1])), pbc<P, T>((T)3 * g[1]));
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
        A[0][0] = pfma(d3, padd(uz, pbc<P, T>(g[2])), pbc<P, T>((T)3 * g[2]));
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

// The same pass for the y stage, where the rows are packed (centre, halo): W_q = D_q * sgn with sgn = (1,-1).
template <int NQ, typename P, typename T>
__device__ __forceinline__ void pass_group_y(const P (&S)[3], const P (&W)[3], P c0, P c2, P sgn, P &o0, P &o1, P &o2)
{
    P E, O;
    if (NQ == 1) { E = S[0]; O = pmul(W[0], sgn); }
    if (NQ == 2) { E = pfma(W[1], sgn, S[0]); O = pfma(W[0], sgn, S[1]); }
    if (NQ == 3) { E = pfma(W[1], sgn, padd(S[0], S[2])); O = pfma(padd(W[0], W[2]), sgn, S[1]); }
    o2 = E;
    o1 = O;
    o0 = pfmas(c0, (T)4, E);
    if (NQ >= 3) o0 = pfmas(c2, (T)-2, o0);
}

// Periodic ghost images of the two rows of a pack (rare path).  eflags: bit 0 = column on a periodic x face,
// bits 1/2 = row r0 / r0+1 on a periodic y face, bit 3 = plane on a periodic z face.
template <typename P, typename T>
__device__ __forceinline__ void store_images(const P (&o)[TSLB_NF], T *__restrict__ Bbuf, long long N, long long i0, long long i1, bool row1,
                                          int eflags, const Layout &L, int col, int r0, int zt)
{
    const long long xi = col == 0 ? (long long)L.nx : -(long long)L.nx;
    const long long zi = zt == 0 ? (long long)L.nz * L.plane : -(long long)L.nz * L.plane;
    const long long ywrap = (long long)L.ny * L.px;
    const long long yi0 = r0 == 0 ? ywrap : -ywrap, yi1 = -ywrap;
    const bool ex = eflags & 1, ey0 = eflags & 2, ey1 = (eflags & 4) && row1, ez = eflags & 8;
    T *b0 = Bbuf + i0, *b1 = Bbuf + i1;
#define TSLB_PUT0(off) _Pragma("unroll") for (int f = 0; f < TSLB_NF; ++f) b0[f * N + (off)] = o[f].x;
#define TSLB_PUT1(off) _Pragma("unroll") for (int f = 0; f < TSLB_NF; ++f) b1[f * N + (off)] = o[f].y;
    if (ex) { TSLB_PUT0(xi) if (row1) { TSLB_PUT1(xi) } }
    if (ey0) { TSLB_PUT0(yi0) if (ex) { TSLB_PUT0(yi0 + xi) } }
    if (ey1) { TSLB_PUT1(yi1) if (ex) { TSLB_PUT1(yi1 + xi) } }
    if (ez) {
        TSLB_PUT0(zi) if (row1) { TSLB_PUT1(zi) }
        if (ex) { TSLB_PUT0(zi + xi) if (row1) { TSLB_PUT1(zi + xi) } }
        if (ey0) { TSLB_PUT0(zi + yi0) if (ex) { TSLB_PUT0(zi + yi0 + xi) } }
        if (ey1) { TSLB_PUT1(zi + yi1) if (ex) { TSLB_PUT1(zi + yi1 + xi) } }
    }
#undef TSLB_PUT0
#undef TSLB_PUT1
}

// finalise the two rows of a pack from their 216-scaled raw moments (m[1..3] lack their base 216 u) and store (Eq. 12)
template <typename P, typename T>
__device__ __forceinline__ void finalize_store(const P (&m)[TSLB_NF], const P (&uo)[3], T *__restrict__ Bbuf, long long N, long long i0,
                                               long long i1, bool row1, int eflags, const Layout &L, int col, int r0, int zt)
{
    // x/216 as x*hi + x*lo: unbiased to ~1 ulp (a rounded 1/216 alone would be a systematic gain)
    const T hi = (T)(1.0 / 216.0);
    const T lo = (T)(1.0 / 216.0 - (double)hi);
    const P dR = pfmas(m[0], lo, pmuls(m[0], hi));
    const P rho = padd(pbc<P, T>((T)1), dR);
    const P den = padd(pbc<P, T>((T)216), m[0]);
    const P inv = pk((T)1 / den.x, (T)1 / den.y);
    const P nm0 = pmuls(m[0], (T)-1);
    // u' = (216 u + J) / (216 + dR216) = u + (J - u dR216) / (216 + dR216)
    P o[TSLB_NF];
    o[0] = dR;
#pragma unroll
    for (int a = 0; a < 3; ++a) o[1 + a] = pfma(pfma(uo[a], nm0, m[1 + a]), inv, uo[a]);
    const P niso = pmuls(dR, (T)(-1.0 / 3.0));
    const P nrho = pmuls(rho, (T)-1);
    const P rx = pmul(nrho, o[1]), ry = pmul(nrho, o[2]), rz = pmul(nrho, o[3]);
    // (the second moments are rebuilt from scratch every step, so a singly rounded 1/216 cannot compound there)
    o[4] = pfma(rx, o[1], pfmas(m[4], hi, niso));
    o[5] = pfma(ry, o[2], pfmas(m[5], hi, niso));
    o[6] = pfma(rz, o[3], pfmas(m[6], hi, niso));
    o[7] = pfma(rx, o[2], pmuls(m[7], hi));
    o[8] = pfma(rx, o[3], pmuls(m[8], hi));
    o[9] = pfma(ry, o[3], pmuls(m[9], hi));
#pragma unroll
    for (int f = 0; f < TSLB_NF; ++f) Bbuf[f * N + i0] = o[f].x;
    if (row1) {
#pragma unroll
        for (int f = 0; f < TSLB_NF; ++f) Bbuf[f * N + i1] = o[f].y;
    }
    // periodic images: a node on a periodic face is also the ghost cell beyond the opposite face (and the edge /
    // corner ghosts when it lies on several), so the next sweep needs no separate ghost-layer refresh
    if (eflags) store_images<P, T>(o, Bbuf, N, i0, i1, row1, eflags, L, col, r0, zt);
}

// index of group (px,py), px+py <= 2, in the z-march state: (0,0)=0 (1,0)=1 (2,0)=2 (0,1)=3 (1,1)=4 (0,2)=5
__host__ __device__ constexpr int gidx(int px, int py) { return py == 0 ? px : (py == 1 ? 3 + px : 5); }

// CTA geometry per dtype: WX x WY warps, each 30 output columns x 2 rows; one CTA per SM (the CTAs of an SM then
// march in lock-step, which keeps the halo re-reads of neighbouring tiles inside L2 -- DESIGN.md "Tile kernel").
// TMA needs the byte offset of the box origin along x to be a multiple of 16 (measured on B200: an origin at a
// multiple of 2 floats raises "illegal instruction"): the box starts at the CTA's first column rounded down to ALIGN
// elements and lanes read at the remaining offset (0 for WX = 2).
template <typename T> struct TileGeom;
#ifndef TILE_F32_WY
#define TILE_F32_WY 7
#endif
#ifndef TILE_F32_NS
#define TILE_F32_NS 4
#endif
#ifndef TILE_F32_WX
#define TILE_F32_WX 2
#endif
#ifndef TILE_F32_MINB
#define TILE_F32_MINB 1
#endif
template <> struct TileGeom<float> { static constexpr int WX = TILE_F32_WX, WY = TILE_F32_WY, NS = TILE_F32_NS, ALIGN = 4, MINB = TILE_F32_MINB; };
template <> struct TileGeom<double> { static constexpr int WX = 2, WY = 4, NS = 4, ALIGN = 2, MINB = 1; };
template <typename T> struct TileDims {
    typedef TileGeom<T> G;
    static constexpr int WARPS = G::WX * G::WY;
    static constexpr int COLS = TILE_COLS * G::WX;                                   // output columns per CTA
    static constexpr int ROWS = 2 * G::WY;                                           // output rows per CTA
    static constexpr int BY = ROWS + 2;                                              // box height
    static constexpr int MAXOFF = (COLS % G::ALIGN) ? 2 : 0;
    static constexpr int BXW = (COLS + 2 + MAXOFF + 3) / 4 * 4;                      // box width = smem row pitch
    static constexpr int BOX_ELEMS = TSLB_NF * BY * BXW;
    static constexpr int STAGE_ELEMS = (int)(((BOX_ELEMS * sizeof(T) + 127) / 128 * 128) / sizeof(T));
    static constexpr int SMEM_BYTES = G::NS * STAGE_ELEMS * (int)sizeof(T);
};
static_assert(TileDims<float>::BY <= TILE_MAX_BY && TileDims<double>::BY <= TILE_MAX_BY, "layout height");

template <typename T, bool WALLY, int ORDER>
__global__ void __launch_bounds__(TileDims<T>::WARPS * 32, TileGeom<T>::MINB) sweep_tile_kernel(const __grid_constant__ CUtensorMap tmA,
                                                                   T *__restrict__ Bbuf, TileParams<T> p)
{
    typedef typename PackOf<T>::type P;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    typedef TileDims<T> TD;
    T *ring = reinterpret_cast<T *>(smem_raw);          // NS stages of [10][BY][BXW]
    constexpr int BXW = TD::BXW, TILE_BY = TD::BY, TILE_NS = TileGeom<T>::NS, STAGE_ELEMS = TD::STAGE_ELEMS;
    __shared__ uint64_t full_bar[TILE_NS];

    const int lane = threadIdx.x & 31;
    const int wid = threadIdx.x >> 5;
    const Layout &L = p.L;
    const long long N = L.field;

    // ---- columns: the warp outputs [xs, xs+30); lane l holds column xs - 1 + l -------------------------------
    const int wx = wid % TileGeom<T>::WX, wy = wid / TileGeom<T>::WX;
    const int xs0 = blockIdx.x * TD::COLS;               // first column of the CTA
    const int xs = xs0 + wx * TILE_COLS;
    const int col = xs - 1 + lane;
    const int xb = xs0 & ~(TileGeom<T>::ALIGN - 1);      // box origin (element index in the padded row), 16-byte aligned
    const bool col_out = lane >= 1 && lane <= TILE_COLS && col < L.nx;  // this lane produces output
    // ---- rows: pack .x = row r0, .y = row r0+1; halo rows r0-1, r0+2 ------------------------------------------
    const int row0 = blockIdx.y * TD::ROWS;
    const int r0 = row0 + 2 * wy;
    const bool warp_active = r0 < L.ny;
    const bool row1_valid = r0 + 1 < L.ny;
    // rows beyond a bounce-back wall contribute nothing (their part is added by bounce_y_correction)
    const bool ghost_lo = WALLY && p.kind[2] == TSLB_BC_BOUNCE_BACK && r0 == 0;                 // row r0-1
    const bool ghost_mid = WALLY && p.kind[3] == TSLB_BC_BOUNCE_BACK && r0 + 1 == L.ny;         // rows r0+1, r0+2
    const bool ghost_hi = WALLY && p.kind[3] == TSLB_BC_BOUNCE_BACK && r0 + 2 == L.ny;          // row r0+2
    const bool any_ghost = ghost_lo || ghost_mid || ghost_hi;   // warp-uniform: this warp owns a wall-adjacent row
    // multiplicative masks of the rows beyond a wall (no selects in the marching loop): mh for the halo pack (r0-1, r0+2),
    // ms for the swapped centre pack (r0+1, r0)
    const P mh = pk(ghost_lo ? (T)0 : (T)1, (ghost_hi || ghost_mid) ? (T)0 : (T)1);
    const P ms = pk(ghost_mid ? (T)0 : (T)1, (T)1);

    const int z0 = blockIdx.z * p.zchunk;
    const int z1 = min(z0 + p.zchunk, L.nz);
    const int nplanes = z1 - z0 + 2;                     // source planes z0-1 .. z1

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < TILE_NS; ++s) mbar_init(&full_bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    // plane i of this CTA = source plane z0-1+i: box origin (element xs, padded row row0, padded plane z0+i, field 0)
    auto issue = [&](int i) {
        const int s = i % TILE_NS;
        mbar_expect_tx(&full_bar[s], (uint32_t)(TD::BOX_ELEMS * sizeof(T)));
        tma_load_4d(ring + s * STAGE_ELEMS, &tmA, &full_bar[s], xb, row0, z0 + i, 0);
    };
    if (threadIdx.x == 0)
        for (int i = 0; i < TILE_NS && i < nplanes; ++i) issue(i);

    // z-march state per (px,py) group: Vp of plane zs-2, centre term of plane zs-1, Vp of plane zs-1
    // (kept as T1 = Vp(zs-2) + centre(zs-1), Vp(zs-2) where it is needed alone -- groups 0, 1, 3 -- and Vp(zs-1):
    //  15 instead of 18 running pairs, 9 instead of 18 register moves per plane)
    P vp2[6], tt1[6], vp1[6];
    // increment form along z: velocity of the previous plane and its backward difference, rows r0, r0+1
    P uprev[3], dprev[3];
    P kw[4];                                              // carried bounce-back terms of the moments with c_z (walls only)
#pragma unroll
    for (int k = 0; k < 4; ++k) kw[k] = pbc<P, T>((T)0);
#pragma unroll
    for (int i = 0; i < 6; ++i) { vp2[i] = pbc<P, T>((T)0); tt1[i] = vp2[i]; vp1[i] = vp2[i]; }
#pragma unroll
    for (int a = 0; a < 3; ++a) { uprev[a] = pbc<P, T>((T)0); dprev[a] = uprev[a]; }

    // which of this thread's nodes have periodic ghost images (finalize_store)
    const int eflags_xy = ((p.kind[0] == TSLB_BC_PERIODIC && (col == 0 || col == L.nx - 1)) ? 1 : 0) |
                          ((p.kind[2] == TSLB_BC_PERIODIC && (r0 == 0 || r0 == L.ny - 1)) ? 2 : 0) |
                          ((p.kind[2] == TSLB_BC_PERIODIC && r0 + 1 == L.ny - 1) ? 4 : 0);
    const P sgn = pk((T)1, (T)-1);                        // D = W * sgn for the (centre, halo) row packing, see below
    const bool st_ok = col_out && warp_active;
    for (int i = 0; i < nplanes; ++i) {
        const int stg = i % TILE_NS;
        mbar_wait(&full_bar[stg], (uint32_t)((i / TILE_NS) & 1));
        {   // every warp computes (rows beyond the lattice read defined but meaningless smem rows and store nothing):
            // no divergent region around the shuffles
            const int zs = z0 - 1 + i;
            const T *S = ring + stg * STAGE_ELEMS + (2 * wy) * BXW + (xs - xb) + lane;

            // ---- a1: moments of rows r0-1 .. r0+2 at this column.  Packing: C = (r0, r0+1) the two output rows,
            //      H = (r0-1, r0+2) their outer neighbours.  For the output pack: up = (H.x, C.x), dn = (C.y, H.y), so
            //      up + dn = H + swap(C) and up - dn = (H - swap(C)) * (1,-1): the centre needs no repacking and the swap
            //      is an operand modifier of the packed instructions. ------------------------------------------------
            P rc[TSLB_NF], rh[TSLB_NF];
#pragma unroll
            for (int f = 0; f < TSLB_NF; ++f) {
                const T *s = S + f * (TILE_BY * BXW);
                rc[f] = pk(s[BXW], s[2 * BXW]);
                rh[f] = pk(s[0], s[3 * BXW]);
            }
            // ---- increment form: exact differences of the stored velocities along y, x, z ---------------------------
            P Ly[3], Wy[3], Lx[3], Dx[3], Lz[3], Dz[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const P uc = rc[1 + a];
                P hs = rh[1 + a], cs = pk(uc.y, uc.x);
                if (WALLY) { hs = pmul(hs, mh); cs = pmul(cs, ms); }   // a node beyond a wall enters the differences as u = 0
                Ly[a] = pfmas(uc, (T)-2, padd(hs, cs));      // (up - c) + (dn - c)
                Wy[a] = psub(hs, cs);                        // (up - dn) * sgn
                const T *s = S + (1 + a) * (TILE_BY * BXW);
                const P xl = pk(s[BXW - 1], s[2 * BXW - 1]), xr = pk(s[BXW + 1], s[2 * BXW + 1]);
                Lx[a] = pfmas(uc, (T)-2, padd(xl, xr));
                Dx[a] = psub(xl, xr);
                const P dcur = psub(uc, uprev[a]);           // u(zs) - u(zs-1)
                Lz[a] = psub(dcur, dprev[a]);                // at the target plane zs-1
                Dz[a] = padd(dprev[a], dcur);                // u(zs) - u(zs-2) = -(D along z); used with negated multipliers
                dprev[a] = dcur;
            }

            P vp0[6], vm0[6], cc0[6];  // this plane's Vp, Vm, centre term per group
            // halfway bounce-back on a y face: for a wall-adjacent row the 9
            // populations arriving from beyond the wall are f*_ibar of the node itself, a local combination of its own
            // coefficients: B(kx,kz) with the local sums L(0,0)=6, L(1,1)=-2, L(2,0)=L(2,2)=2.  .x = row r0, .y = row r0+1.
            P WB[3][3];
            const P wsp = pk(ghost_lo ? (T)-1 : (T)1, (T)1);
#pragma unroll
            for (int kz = 0; kz < 3; ++kz) {
                // ---- a2: Hermite coefficients of the four rows for this kz --------------------------------------
                P Ac[3][3], Ah[3][3];
                if (kz == 0) { hermite_round<0, P, T>(rc, p.beta, p.g, Ac); hermite_round<0, P, T>(rh, p.beta, p.g, Ah); }
                if (kz == 1) { hermite_round<1, P, T>(rc, p.beta, p.g, Ac); hermite_round<1, P, T>(rh, p.beta, p.g, Ah); }
                if (kz == 2) { hermite_round<2, P, T>(rc, p.beta, p.g, Ac); hermite_round<2, P, T>(rh, p.beta, p.g, Ah); }
                // ---- y pass: G1[py][kx] = sum_ky T^y_{py,ky} A(kx,ky,kz) at rows r0, r0+1 -------------------------
                P G1[3][3];
#pragma unroll
                for (int kx = 0; kx < 3; ++kx) {
                    if (!kvalid<ORDER>(kx, 0, kz)) continue;
                    // E = up(P) + dn(M), O = up(P) - dn(M) with P = phi0 + phi1 + phi2, M = phi0 - phi1 + phi2 of the
                    // neighbour rows.  Per pack Q = (P of its .x row, M of its .y row) = phi0 + phi2 + phi1 * sgn; then
                    // E = Q_H + swap(Q_C) and O = (Q_H - swap(Q_C)) * sgn.
                    P qh = Ah[kx][0], qc = Ac[kx][0];
                    if (kvalid<ORDER>(kx, 2, kz)) { qh = padd(qh, Ah[kx][2]); qc = padd(qc, Ac[kx][2]); }
                    if (kvalid<ORDER>(kx, 1, kz)) { qh = pfma(Ah[kx][1], sgn, qh); qc = pfma(Ac[kx][1], sgn, qc); }
                    P qs = pk(qc.y, qc.x);
                    if (WALLY) {   // rows beyond a bounce-back wall send nothing; the bounced populations are added below
                        qh = pmul(qh, mh);
                        qs = pmul(qs, ms);
                        // B(kx,kz) = sum_ky t_ky(-c_y) A(kx,ky,kz) of the own rows: wall below -> (1,-1,1), above -> (1,1,1)
                        if (kx + kz <= 2 && !(kx == 1 && kz == 2) && !(kx == 2 && kz == 1)) {
                            P bq = Ac[kx][0];
                            if (kvalid<ORDER>(kx, 2, kz)) bq = padd(bq, Ac[kx][2]);
                            if (kvalid<ORDER>(kx, 1, kz)) bq = pfma(Ac[kx][1], wsp, bq);
                            WB[kx][kz] = bq;
                        }
                    }
                    const P E = padd(qh, qs);
                    G1[2][kx] = E;
                    G1[1][kx] = pmul(psub(qh, qs), sgn);
                    P o0 = pfmas(Ac[kx][0], (T)4, E);
                    if (kvalid<ORDER>(kx, 2, kz)) o0 = pfmas(Ac[kx][2], (T)-2, o0);
                    G1[0][kx] = o0;
                }
                // y-stage increments of the bases 3 u_a (tap sums along y: 6, 0, 2 for py = 0, 1, 2 when ky = 0; 0, 2, 0 when ky = 1)
                const P sg3 = pk((T)3, (T)-3);
                if (kz == 0) {
                    G1[0][1] = pfmas(Ly[0], (T)3, G1[0][1]); G1[1][1] = pfma(Wy[0], sg3, G1[1][1]); G1[2][1] = pfmas(Ly[0], (T)3, G1[2][1]);
                    G1[0][0] = pfma(Wy[1], sg3, G1[0][0]); G1[1][0] = pfmas(Ly[1], (T)3, G1[1][0]); G1[2][0] = pfma(Wy[1], sg3, G1[2][0]);
                }
                if (kz == 1) {
                    G1[0][0] = pfmas(Ly[2], (T)3, G1[0][0]); G1[1][0] = pfma(Wy[2], sg3, G1[1][0]); G1[2][0] = pfmas(Ly[2], (T)3, G1[2][0]);
                }
                // ---- x pass (warp shuffles): G2[px][py] = sum_kx T^x_{px,kx} G1[py][kx]; then the z bookkeeping ----
#pragma unroll
                for (int py = 0; py < 3; ++py) {
                    // E = up(P) + dn(M), O = up(P) - dn(M): one shuffle up of P = phi0 + phi1 + phi2 and one down of
                    // M = phi0 - phi1 + phi2 instead of two per field
                    P t = G1[py][0];
                    if (kvalid<ORDER>(2, 0, kz)) t = padd(t, G1[py][2]);
                    P pp = t, mm = t;
                    if (kvalid<ORDER>(1, 0, kz)) { pp = padd(t, G1[py][1]); mm = psub(t, G1[py][1]); }
                    const P upP = shfl_up1(pp);   // from column-1  (c_x = +1 pulls from x-1)
                    const P dnM = shfl_dn1(mm);   // from column+1
                    P o[3];
                    o[2] = padd(upP, dnM);
                    o[1] = psub(upP, dnM);
                    o[0] = pfmas(G1[py][0], (T)4, o[2]);
                    if (kvalid<ORDER>(2, 0, kz)) o[0] = pfmas(G1[py][2], (T)-2, o[0]);
                    // x-stage increments: base multipliers after the y stage are 18 (py=0) and 6 (py=2) for ux (kx=1) and uz
                    // (kx=0, kz=1), 6 (py=1) for uy (kx=0)
                    if (kz == 0 && py == 0) { o[0] = pfmas(Dx[0], (T)18, o[0]); o[1] = pfmas(Lx[0], (T)18, o[1]); o[2] = pfmas(Dx[0], (T)18, o[2]); }
                    if (kz == 0 && py == 2) { o[0] = pfmas(Dx[0], (T)6, o[0]); }
                    if (kz == 0 && py == 1) { o[0] = pfmas(Lx[1], (T)6, o[0]); o[1] = pfmas(Dx[1], (T)6, o[1]); }
                    if (kz == 1 && py == 0) { o[0] = pfmas(Lx[2], (T)18, o[0]); o[1] = pfmas(Dx[2], (T)18, o[1]); o[2] = pfmas(Lx[2], (T)18, o[2]); }
                    if (kz == 1 && py == 2) { o[0] = pfmas(Lx[2], (T)6, o[0]); }
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

            P kw_new[4];
            if (WALLY && any_ghost) {
                // full first-order coefficients (the passes carry them without their base 3 u)
                WB[1][0] = pfmas(rc[1], (T)3, WB[1][0]);
                WB[0][0] = pfma(rc[2], pmuls(wsp, (T)3), WB[0][0]);
                WB[0][1] = pfmas(rc[3], (T)3, WB[0][1]);
                const P wm = pk((ghost_lo || ghost_mid) ? (T)1 : (T)0, ghost_hi ? (T)1 : (T)0);   // which row of the pack is at a wall
                const P sgp = pk(ghost_lo ? (T)1 : (T)-1, (T)-1);                              // c_y of the arrival direction
                const P w12 = pmuls(wm, (T)12), w36 = pmuls(wm, (T)36), w12s = pmul(w12, sgp), w36s = pmul(w36, sgp);
                // arrival c_z = 0: into this plane's centre terms (they reach the target plane through tt1)
                cc0[0] = pfma(WB[0][0], w36, cc0[0]);                         // 000
                cc0[1] = pfma(WB[1][0], pmuls(w12, (T)-1), cc0[1]);           // 100
                cc0[3] = pfma(WB[0][0], w36s, cc0[3]);                        // 010
                cc0[2] = pfma(padd(WB[0][0], WB[2][0]), w12, cc0[2]);         // 200
                cc0[5] = pfma(WB[0][0], w36, cc0[5]);                         // 020
                cc0[4] = pfma(WB[1][0], pmuls(w12s, (T)-1), cc0[4]);          // 110
                // moments with c_z: carried to the next iteration, where this plane is the target
                kw_new[0] = pmul(WB[0][1], pmuls(w12, (T)-1));                // 001
                kw_new[1] = pmul(padd(WB[0][0], WB[0][2]), w12);              // 002
                kw_new[2] = pmul(WB[1][1], pmuls(wm, (T)4));                  // 101
                kw_new[3] = pmul(WB[0][1], pmuls(w12s, (T)-1));               // 011
            }
            // ---- z pass for target plane zt = zs - 1:  pz=0: Vp(zs-2) + centre(zs-1) + Vm(zs);  pz=1: Vp(zs-2) - Vm(zs);
            //      pz=2: Vp(zs-2) + Vm(zs); plus the z-stage increments (base multipliers 36 for ux, uy; 108 / 36 for uz) ----
            const int zt = zs - 1;
            if (zt >= z0 && st_ok) {
                P m[TSLB_NF];
                {
                    m[0] = pfmas(Dz[2], (T)-108, padd(tt1[0], vm0[0]));          // 000
                    m[3] = pfmas(Lz[2], (T)108, psub(vp2[0], vm0[0]));         // 001
                    m[6] = pfmas(Dz[2], (T)-108, padd(vp2[0], vm0[0]));         // 002
                    m[1] = pfmas(Lz[0], (T)36, padd(tt1[1], vm0[1]));           // 100
                    m[8] = pfmas(Dz[0], (T)-36, psub(vp2[1], vm0[1]));          // 101
                    m[2] = pfmas(Lz[1], (T)36, padd(tt1[3], vm0[3]));           // 010
                    m[9] = pfmas(Dz[1], (T)-36, psub(vp2[3], vm0[3]));          // 011
                    m[4] = pfmas(Dz[2], (T)-36, padd(tt1[2], vm0[2]));           // 200
                    m[7] = padd(tt1[4], vm0[4]);                               // 110
                    m[5] = pfmas(Dz[2], (T)-36, padd(tt1[5], vm0[5]));           // 020
                }
                const long long i0 = lay_idx(L, col, r0, zt);
                if (WALLY) { m[3] = padd(m[3], kw[0]); m[6] = padd(m[6], kw[1]); m[8] = padd(m[8], kw[2]); m[9] = padd(m[9], kw[3]); }
                const int eflags = eflags_xy | ((p.kind[4] == TSLB_BC_PERIODIC && (zt == 0 || zt == L.nz - 1)) ? 8 : 0);
                finalize_store<P, T>(m, uprev, Bbuf, N, i0, i0 + L.px, row1_valid, eflags, L, col, r0, zt);
            }
            if (WALLY && any_ghost) {
#pragma unroll
                for (int k = 0; k < 4; ++k) kw[k] = kw_new[k];
            }
            // ---- shift the march state ---------------------------------------------------------------------------------
#pragma unroll
            for (int g = 0; g < 6; ++g) {
                tt1[g] = padd(vp1[g], cc0[g]);               // Vp(zs-1) + centre(zs): used when plane zs+1 arrives
                if (g == 0 || g == 1 || g == 3) vp2[g] = vp1[g];
                vp1[g] = vp0[g];
            }
#pragma unroll
            for (int a = 0; a < 3; ++a) uprev[a] = rc[1 + a];
        }
        __syncthreads();                                  // every warp is done with stage `stg`: refill it
        if (threadIdx.x == 0 && i + TILE_NS < nplanes) issue(i + TILE_NS);
    }
}

template <typename T>
TileParams<T> make_tile(const tslb_ctx *c, dim3 *grid)
{
    TileParams<T> p;
    p.L = c->L;
    for (int f = 0; f < 6; ++f) p.kind[f] = c->kind[f];
    p.beta = (T)(1.0 - c->omega);
    for (int a = 0; a < 3; ++a) p.g[a] = (T)c->g[a];
    const int gx = (c->nx + TileDims<T>::COLS - 1) / TileDims<T>::COLS;
    const int gy = (c->ny + TileDims<T>::ROWS - 1) / TileDims<T>::ROWS;
    // z chunks (one CTA per SM is resident): pick the chunk count whose number of waves x (chunk length + 2 halo planes)
    // is smallest
    const long long cols = (long long)gx * gy;
    int best = 1;
    double best_cost = 1e300;
    for (int k = 1; k <= 64 && k <= c->nz; ++k) {
        const int zc = (c->nz + k - 1) / k;
        if (k > 1 && zc < 8) break;
        const long long ctas = cols * ((c->nz + zc - 1) / zc);
        const long long slots = (long long)c->sm_count * TileGeom<T>::MINB;
        const long long waves = (ctas + slots - 1) / slots;
        const double cost = (double)waves * (zc + 2 + 3);      // + ring fill latency of a fresh CTA, in plane units
        if (cost < best_cost) { best_cost = cost; best = k; }
    }
    const int zc = (c->nz + best - 1) / best;
    p.zchunk = zc;
    *grid = dim3(gx, gy, (c->nz + zc - 1) / zc);
    return p;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

bool tslb_tile_supported(const tslb_ctx *c, const char **why)
{
    // bounce-back walls are handled on the y faces only (x or z walls: gather kernel)
    for (int f = 0; f < 6; ++f)
        if (c->kind[f] == TSLB_BC_BOUNCE_BACK && (f >> 1) != 1) {
            if (why) *why = "bounce-back walls on x or z faces";
            return false;
        }
    if (c->ws && !c->tmap_ok) {
        if (why) *why = "TMA descriptors unavailable";
        return false;
    }
    if (why) *why = "";
    return true;
}

// TMA descriptors of the two moment buffers: 4-D tensor (x, y, z, field) of the padded SoA layout, box 36|32 x 10 x 1 x 10.
// cuTensorMapEncodeTiled is fetched through the runtime so that the library links against cudart only.
cudaError_t tslb_tile_prepare(tslb_ctx *c)
{
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return e;
    if (!fn || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
    const Layout &L = c->L;
    const size_t es = tslb_elem(c);
    const cuuint64_t dims[4] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)L.pz, TSLB_NF};
    const cuuint64_t strides[3] = {(cuuint64_t)L.px * es, (cuuint64_t)L.plane * es, (cuuint64_t)L.field * es};
    const cuuint32_t box[4] = {(cuuint32_t)(c->dtype == TSLB_F64 ? TileDims<double>::BXW : TileDims<float>::BXW),
                               (cuuint32_t)(c->dtype == TSLB_F64 ? TileDims<double>::BY : TileDims<float>::BY), 1, TSLB_NF};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    for (int b = 0; b < 2; ++b) {
        CUresult r = ((EncodeTiledFn)fn)(&c->tmap[b], c->dtype == TSLB_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                                         4, c->buf[b], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                         CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    }
    const int smem32 = TileDims<float>::SMEM_BYTES, smem64 = TileDims<double>::SMEM_BYTES;
    e = cudaSuccess;
#define TSLB_SMEM_ATTR(T, W, O, B) if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_tile_kernel<T, W, O>, cudaFuncAttributeMaxDynamicSharedMemorySize, B)
    TSLB_SMEM_ATTR(float, false, 3, smem32); TSLB_SMEM_ATTR(float, true, 3, smem32);
    TSLB_SMEM_ATTR(float, false, 2, smem32); TSLB_SMEM_ATTR(float, true, 2, smem32);
    TSLB_SMEM_ATTR(double, false, 3, smem64); TSLB_SMEM_ATTR(double, true, 3, smem64);
    TSLB_SMEM_ATTR(double, false, 2, smem64); TSLB_SMEM_ATTR(double, true, 2, smem64);
#undef TSLB_SMEM_ATTR
    if (e != cudaSuccess) return e;
    c->tmap_ok = 1;
    return cudaSuccess;
}

template <typename T, bool WALLY, int ORDER>
static void launch_tile(tslb_ctx *c, cudaStream_t st)
{
    dim3 grid;
    TileParams<T> p = make_tile<T>(c, &grid);
    sweep_tile_kernel<T, WALLY, ORDER><<<grid, TileDims<T>::WARPS * 32, TileDims<T>::SMEM_BYTES, st>>>(c->tmap[c->cur], (T *)c->buf[1 - c->cur], p);
}

cudaError_t tslb_launch_tile(tslb_ctx *c, cudaStream_t st)
{
    const bool wally = c->kind[2] == TSLB_BC_BOUNCE_BACK || c->kind[3] == TSLB_BC_BOUNCE_BACK;
    const bool o3 = c->order >= 3;
    if (c->dtype == TSLB_F32) {
        if (wally) { if (o3) launch_tile<float, true, 3>(c, st); else launch_tile<float, true, 2>(c, st); }
        else { if (o3) launch_tile<float, false, 3>(c, st); else launch_tile<float, false, 2>(c, st); }
    } else {
        if (wally) { if (o3) launch_tile<double, true, 3>(c, st); else launch_tile<double, true, 2>(c, st); }
        else { if (o3) launch_tile<double, false, 3>(c, st); else launch_tile<double, false, 2>(c, st); }
    }
    c->launches++;
    return cudaGetLastError();
}

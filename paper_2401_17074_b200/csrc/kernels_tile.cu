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
// Data path.  One CTA per SM owns a 60 x 14 column of nodes (fp32: 2 x 7 "main" warps; fp64:
// 60 x 8, 2 x 4) and marches along z.  Warp roles:
//   main warps   2 rows (packed in a 2-wide register pair, so fp32 issues as FFMA2/FADD2) x 32 columns (30 outputs + 2
//                halo lanes).  Per source plane: Hermite coefficients of the OWN two rows only; the y pass needs, from
//                the row below, P = phi0+phi1+phi2 and, from the row above, M = phi0-phi1+phi2 of 8 coefficient groups:
//                every warp publishes these two combinations of its rows in shared memory and reads its neighbours'
//                (per-row-pair mbarriers, double-buffered: no CTA-wide barrier anywhere in the plane loop);
//                x pass by warp shuffles; z pass by marching (15 running pairs per thread).
//   halo warps   2 warps: the rows just below and above the tile (Hermite coefficients + the published combinations
//                only).  Lane 0 of the first is the TMA PRODUCER (3-stage ring of source planes: the 14 tile rows and
//                the two halo rows as three boxes, y and z wrapped by coordinate, walls / open faces by out-of-bounds
//                zero fill; full/empty mbarriers, a stage is released as soon as its values sit in registers).
//                Lane 0 of the second is the STORE thread: the finished 60 x 14 x 10 output tile is staged in shared
//                memory and written with one TMA store (cp.async.bulk.tensor shared -> global, SASS UTMASTG).
// Each node's moments leave HBM once per tile (halo re-reads hit L2) and the 10 new moments are written once, in full
// rows: 80 B (fp32) / 160 B (fp64) of compulsory traffic per node update.
//
// INCREMENT FORM: the base 3 u_a of the first-order coefficients never enters the
// passes.  A pass with taps (t-, t0, t+) applied to B*u gives (t- + t0 + t+) B u(x) + B [t- (u(x-1) - u(x)) + t+ (u(x+1) - u(x))];
// only the bracket (exact differences of stored velocities) is added at each stage, and the product of the tap sums,
// 216 u_a(x), is re-attached in closed form at the end:  u' = u + (J_small - u dR) / (216 + dR).
#include <string.h>
#include <type_traits>
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
template <typename P> __device__ __forceinline__ P pswap(P a) { return pk(a.y, a.x); }
// 1/x for x = 216 + dR216 (always close to 216): fp32 uses the hardware approximation (MUFU.RCP, <= 1 ulp) -- the quotient
// only scales the per-step INCREMENT of u (increment form), so its rounding is far below the stored precision
__device__ __forceinline__ float rcp_fast(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ double rcp_fast(double x) { return 1.0 / x; }

template <typename P> __device__ __forceinline__ P shfl_up1(P v)
{
    return pk(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1));
}
template <typename P> __device__ __forceinline__ P shfl_dn1(P v)
{
    return pk(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1));
}

// ---- TMA / mbarrier / shared memory by 32-bit shared address (PTX; SASS: UTMALDG, UTMASTG, SYNCS, LDS, STS) ------------
// Every shared-memory access of the kernel goes through a 32-bit shared-window address held in a register plus an
// immediate: the addresses are formed once before the plane loop (keep(): an empty asm the compiler cannot
// rematerialise through), so the loop carries no address arithmetic beyond the stage / slot offsets.
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t keep(uint32_t v) { asm volatile("" : "+r"(v)); return v; }
// the same for a floating-point value: a loop-invariant parameter that passes through keepf inside the loop is re-read
// (one constant-bank load) in every iteration instead of being hoisted into registers that stay occupied all the time
__device__ __forceinline__ float keepf(float v) { asm volatile("" : "+f"(v)); return v; }
__device__ __forceinline__ double keepf(double v) { asm volatile("" : "+d"(v)); return v; }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}" ::"r"(bar), "r"(parity) : "memory");
}
// 1: the generic -> async proxy fence before the TMA store of the output tile is executed once by the store thread,
// after it has acquired the main warps' writes through the "tile full" mbarrier (release at their arrive), instead of
// by every main warp after its own writes (fence.proxy.async = MEMBAR.ALL.CTA + FENCE.VIEW.ASYNC: ~400 cycles per warp
// and plane with 20 shared-memory stores in flight)
#ifndef TILE_FENCE_STORER
#define TILE_FENCE_STORER 1
#endif
// "Published" flags of the y exchange: a 32-bit counter per warp in shared memory instead of an mbarrier -- a release store
// by the publisher, an acquire-load poll by the reader.  A try_wait costs ~90 cycles even when the phase is complete; a
// poll that finds its value costs one shared-memory load (~30 cycles), and there are two such waits per plane and warp
// on the lock-step critical path.
__device__ __forceinline__ void flag_set(uint32_t addr, uint32_t val, int lane)
{
    __syncwarp();
    if (lane == 0) asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(addr), "r"(val) : "memory");
}
__device__ __forceinline__ void flag_wait(uint32_t addr, uint32_t want)
{
    uint32_t v;
    do {
        asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    } while ((int)(v - want) < 0);
}
// one warp signals: every lane's earlier shared-memory accesses are ordered before the arrive of lane 0
__device__ __forceinline__ void warp_arrive(uint32_t bar, int lane)
{
    __syncwarp();
    if (lane == 0) mbar_arrive(bar);
}
__device__ __forceinline__ float lds(uint32_t a, float)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ double lds(uint32_t a, double)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void sts(uint32_t a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_store_4d(uint32_t src, const CUtensorMap *map, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
                 ::"l"(map), "r"(src), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <typename T>
struct TileParams {
    Layout L;
    int kind[6];
    T beta, g[3];
    const T *beta_z;   // sponge layer (Eq. 26): 1 - omega of the nodes of plane z, [nz] (SPONGE instantiations only)
    int zchunk;  // planes per z chunk
    int zbeg, zend;   // planes that are advanced: all of them, without the ghost planes of a slab (EXCHANGE faces)
    int fuse;    // the store warp writes the open-face boundary nodes of time t+1 itself (FUSE instantiations)
};
// Slab neighbours read in place (tslb_set_neighbor, include/tslb.h): the source plane ON an EXCHANGE face -- the ghost plane of
// a slab -- is loaded by TMA straight from the neighbouring slab's current buffer (its outermost owned plane: peer memory over
// NVLink, or the same device) instead of from this lattice's ghost plane.  Same plane layout (equal nx, ny, dtype), so the
// boxes, the halo rows and the ghost columns are those of the peer's plane.
struct NbParams {
    CUtensorMap main[2], row[2];   // [0]: the slab below (face ZLO), [1]: the slab above (face ZHI); the peer's CURRENT buffer
    int on[2];
    int z[2];                      // the peer's outermost owned plane on that side
};
// fused boundary fill (a6): what the store warp needs to impose inlet velocities / outlet densities
struct FuseParams {
    Layout L;
    int kind[6];
    long long tnext;           // step index the written boundary values belong to (noise counter)
    InletDev inlet[6];
    double rho_out[6];
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

// The y-pass combinations of one pack (rows .x, .y) for the coefficient group (kx, kz), from A[kx][ky]:
//   t = A0 + A2,   (p0, m1) = (P of row .x, M of row .y)          -- what the pack's own rows exchange with each other
//                  (m0, p1) = (M of row .x, P of row .y)          -- what the rows outside the pack need: PUBLISHED
//   cen = 4 A0 - 2 A2                                              -- the centre taps
// with P = phi0 + phi1 + phi2 (goes up, c_y = +1), M = phi0 - phi1 + phi2 (goes down).
// The four combinations are formed with SCALAR adds (p0, m0 of row .x; p1, m1 of row .y): a packed instruction cannot add
// in one half and subtract in the other, so the packed form needs multiplications by (1,-1) packs (three-register
// FFMA2s, the most expensive instruction of the loop in register-file bandwidth), and a scalar FADD costs exactly half
// a packed one.
template <int ORDER, int KX, int KZ, typename P, typename T>
__device__ __forceinline__ void ycombos(const P (&A)[3][3], T &p0, T &m0, T &p1, T &m1, P &cen)
{
    const P a0 = A[KX][0];
    P t = a0;
    cen = pmuls(a0, (T)4);
    if (kvalid<ORDER>(KX, 2, KZ)) { t = padd(a0, A[KX][2]); cen = pfmas(A[KX][2], (T)-2, cen); }
    p0 = t.x; m0 = t.x; p1 = t.y; m1 = t.y;
    if (kvalid<ORDER>(KX, 1, KZ)) {
        const P a1 = A[KX][1];
        p0 = t.x + a1.x; m0 = t.x - a1.x; p1 = t.y + a1.y; m1 = t.y - a1.y;
    }
}

// x-wall combination of the coefficients of one node pack: Bx(ky,kz) = sum_kx t_kx(-c_x) A(kx,ky,kz) = A0 - c_x A1 + A2
template <int ORDER, int KY, int KZ, typename P, typename T>
__device__ __forceinline__ P bx_combo(const P (&A)[3][3], T cx)
{
    P b = kvalid<ORDER>(0, KY, KZ) ? A[0][KY] : pbc<P, T>((T)0);
    if (kvalid<ORDER>(1, KY, KZ)) b = pfmas(A[1][KY], -cx, b);
    if (kvalid<ORDER>(2, KY, KZ)) b = padd(b, A[2][KY]);
    return b;
}

// index of group (px,py), px+py <= 2, in the z-march state: (0,0)=0 (1,0)=1 (2,0)=2 (0,1)=3 (1,1)=4 (0,2)=5
__host__ __device__ constexpr int gidx(int px, int py) { return py == 0 ? px : (py == 1 ? 3 + px : 5); }
// index of the coefficient group (kx, kz) among the 8 exchanged ones
__host__ __device__ constexpr int qidx(int kx, int kz) { return kz * 3 + kx; }

// ---- CTA geometry -------------------------------------------------------------------------------------------------
// WX x WY main warps, each 30 output columns x 2 rows, + 2 halo warps; one CTA per SM (the CTAs of an SM then march in
// lock-step, which keeps the halo re-reads of neighbouring tiles inside L2).  TMA needs the byte offset of a box origin
// along x to be a multiple of 16 (measured on B200: an origin at a multiple of 2 floats raises "illegal instruction"):
// the source box starts XPAD = 4 columns left of the tile (the layout puts node x = 0 on a 16-byte boundary).
// Geometry index G: 0 = the large tile (one CTA per SM), 1 = the small tile for lattices that cannot fill 148 large CTAs
// (fp32 only: 60 columns x 4 rows, 4 main warps + the 4 helpers, two CTAs per SM).
template <typename T, int G> struct TileGeom;
#ifndef TILE_F32_WY
#define TILE_F32_WY 6
#endif
#ifndef TILE_F32_NS
#define TILE_F32_NS 2
#endif
// duration of one plane of a small-geometry CTA relative to a large one (measured, profiles/README.md)
// 1: the main warps re-read beta and g from the parameter bank in every plane (see keepf)
#ifndef TILE_REREAD_PARAMS
#define TILE_REREAD_PARAMS 1
#endif
#ifndef TILE_SMALL_PLANE
#define TILE_SMALL_PLANE 0.8
#endif
// -1: choose the geometry by estimated cost; 0 / 1: force it (experiments)
#ifndef TILE_FORCE_GEOM
#define TILE_FORCE_GEOM -1
#endif
#ifndef TILE_ZC_MAX
#define TILE_ZC_MAX 64
#endif
// output tiles in shared memory: with two the main warps fill one while the TMA store drains the other (the store of a
// 60 x 14 x 10 tile takes ~1200 cycles from issue to "source read"; with a single tile that is a CTA-wide bubble per plane)
#ifndef TILE_F32_NOUT
#define TILE_F32_NOUT 2
#endif
// REG_MAIN / REG_HALO != 0: the register file is re-divided after launch with setmaxnreg (the main warps, which carry the
// z-march state, get more than an even share; needs the main warps to be whole warpgroups of 4, and NIDLE idle warps that
// complete the helpers' warpgroup).  fp64: 8 main warps at 208 registers + 2 halo + 2 idle at 80 (an even share of the
// 16384 registers of an SM sub-partition among its 3 warps would be 168, which spills).  Register counts are multiples of
// 16: a warp's allocation is rounded up to 512 registers, and a setmaxnreg.inc that cannot be satisfied blocks forever
// (measured: 216 + 216 + 80 and 208 + 208 + 96 per sub-partition hang).  The pool is what the CTA was given at LAUNCH
// (threads x MAXREG), not the whole register file: the re-divided total must not exceed it.
// fp32: 12 main warps at 144 registers + 2 halo + 2 idle at 80 (14 main warps at the even share of 128 spill ~40 values per
// plane: 48.8 GLUPS at 512^3 against 54.5 with 12 warps and no spills)
#ifndef TILE_F32_RM
#define TILE_F32_RM 144
#define TILE_F32_RH 80
#define TILE_F32_NIDLE 2
#endif
template <> struct TileGeom<float, 0> {
    static constexpr int WX = 2, WY = TILE_F32_WY, NS = TILE_F32_NS, NIDLE = TILE_F32_NIDLE, REG_MAIN = TILE_F32_RM, REG_HALO = TILE_F32_RH;
    static constexpr int NOUT = TILE_F32_NOUT, CTAS = 1;
    static constexpr bool QFLAGS = false;
};
template <> struct TileGeom<float, 1> {
    static constexpr int WX = 2, WY = 2, NS = 2, NIDLE = 2, REG_MAIN = 144, REG_HALO = 80, NOUT = 2, CTAS = 2;
    static constexpr bool QFLAGS = false;
};
#ifndef TILE_F64_RM
#define TILE_F64_RM 208
#define TILE_F64_RH 80
#endif
template <> struct TileGeom<double, 0> { static constexpr int WX = 2, WY = 4, NS = 2, NIDLE = 2, REG_MAIN = TILE_F64_RM, REG_HALO = TILE_F64_RH, NOUT = 1, CTAS = 1;
    // "published" signals of the y exchange: polled release/acquire flags instead of mbarriers.  A poll that finds its value
    // costs one shared-memory load (~30 cycles) against ~90 for a try_wait, but a poll that does not spins in the issue
    // slots of the other warps: fp64 (latency-bound, 2 main warps per sub-partition) gains 7 %, fp32 (issue-bound) loses 4 %.
    static constexpr bool QFLAGS = true;
};
template <> struct TileGeom<double, 1> : TileGeom<double, 0> {};     // fp64 has the large geometry only
constexpr int rup128(int bytes) { return (bytes + 127) / 128 * 128; }
template <typename T, int GI = 0> struct TileDims {
    typedef TileGeom<T, GI> G;
    static constexpr int WX = G::WX, WY = G::WY, NS = G::NS;
    static constexpr int NMAIN = WX * WY, NHALO = 2, WARPS = NMAIN + NHALO, THREADS = (WARPS + G::NIDLE) * 32;
    // CTAS CTAs per SM share the register file: 16384 registers per SM sub-partition, warps dealt round-robin to the four
    static constexpr int MAXREG = (16384 / (((WARPS + G::NIDLE + 3) / 4) * 32 * G::CTAS)) / 8 * 8;   // at launch: 128 (fp32), 168 (fp64, 12 warps)
    static_assert(G::REG_MAIN == 0 || (NMAIN % 4 == 0 && (NHALO + G::NIDLE) % 4 == 0), "setmaxnreg works on warpgroups of 4 warps");
    static_assert(G::REG_MAIN % 16 == 0 && G::REG_HALO % 16 == 0, "a warp's registers are allocated in units of 512");
    static_assert(G::REG_MAIN == 0 || NMAIN * G::REG_MAIN + (NHALO + G::NIDLE) * G::REG_HALO <= (WARPS + G::NIDLE) * MAXREG, "setmaxnreg pool = launch allocation");
    static_assert(G::REG_MAIN == 0 || (NMAIN / 4) * G::REG_MAIN + ((NHALO + G::NIDLE) / 4) * G::REG_HALO <= 512 / G::CTAS, "16384 registers per sub-partition");
    static constexpr int COLS = TILE_COLS * WX;                  // output columns per CTA (60)
    static constexpr int ROWS = 2 * WY;                          // output rows per CTA
    static constexpr int XPAD = 4;                               // box origin = first tile column - XPAD
    static constexpr int BXW = COLS + 2 * XPAD;                  // box width (68): tile columns -4 .. 63
    static constexpr int FS = ROWS * BXW;                        // field stride inside the main region [10][ROWS][BXW]
    static constexpr int MAIN_ELEMS = rup128(TSLB_NF * FS * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr int HALO_ELEMS = rup128(TSLB_NF * BXW * (int)sizeof(T)) / (int)sizeof(T);   // one row [10][BXW]
    static constexpr int STAGE_ELEMS = MAIN_ELEMS + 2 * HALO_ELEMS;                               // main | row -1 | row ROWS
    static constexpr int STAGE_TX = (TSLB_NF * FS + 2 * TSLB_NF * BXW) * (int)sizeof(T);         // bytes landing per plane
    static constexpr int NPACK = WY + 1;                         // row pairs that publish (main + the halo pair)
    static constexpr int NGRP = 8;                               // coefficient groups (kx, kz) exchanged
    static constexpr int EXW = 64;                               // exchange columns: tile columns -1 .. 62
    static constexpr int EX_SLOT = NPACK * NGRP * EXW;           // elements per component and slot
    static constexpr int OUT_ELEMS = TSLB_NF * ROWS * COLS;      // output tile [10][ROWS][COLS]
    static constexpr int NOUT = G::NOUT;                         // output tiles (1 or 2)
    static constexpr int OUT_BYTES = rup128(OUT_ELEMS * (int)sizeof(T));
    static constexpr int OFF_OUT = NS * STAGE_ELEMS * (int)sizeof(T);
    static constexpr int OFF_EX = OFF_OUT + NOUT * OUT_BYTES;
    static constexpr int OFF_BAR = OFF_EX + 4 * EX_SLOT * (int)sizeof(T);     // 2 components x 2 slots
    static constexpr int NBAR = 2 * NS + 2 * (NPACK + 1) + 2 * NOUT;
    static_assert(NOUT == 1 || NOUT == 2, "one or two output tiles");
    static constexpr int SMEM_BYTES = OFF_BAR + NBAR * 8;
};
static_assert(TileDims<float>::SMEM_BYTES <= 232448 && TileDims<double>::SMEM_BYTES <= 232448, "shared memory budget");
static_assert(2 * (TileDims<float, 1>::SMEM_BYTES + 1024) <= 233472, "two small CTAs per SM");
static_assert(TileGeom<float, 0>::WX == 2 && TileGeom<float, 1>::WX == 2 && TileGeom<double, 0>::WX == 2, "two warps per row pair publish; two halo warps");

// values imposed on the open-face boundary node (x, y, z) into its slot `a` of an output tile (field stride fs bytes):
// lowest-index pressure face -> rho, lowest-index inlet face -> u (the rule of fill_boundary_kernel).  Out of line: it
// is used from five places of the store warp and is not on the hot path.
template <typename T>
__device__ __noinline__ void tile_impose(const FuseParams &p, uint32_t a, uint32_t fs, int x, int y, int z)
{
    const Layout &L = p.L;
    const int n3[3] = {L.nx, L.ny, L.nz};
    const int q[3] = {x, y, z};
    bool done = false;
#pragma unroll
    for (int f2 = 0; f2 < 6; ++f2) {
        if (done || p.kind[f2] != TSLB_BC_OUTLET_PRESSURE) continue;
        if (q[f2 >> 1] != ((f2 & 1) ? n3[f2 >> 1] - 1 : 0)) continue;
        sts(a, (T)(p.rho_out[f2] - 1.0));
        done = true;
    }
    done = false;
#pragma unroll
    for (int f2 = 0; f2 < 6; ++f2) {
        if (done || p.kind[f2] != TSLB_BC_VELOCITY_INLET) continue;
        const int ax2 = f2 >> 1;
        if (q[ax2] != ((f2 & 1) ? n3[ax2] - 1 : 0)) continue;
        const int a2 = (ax2 == 0) ? 1 : 0, b2 = (ax2 == 2) ? 1 : 2;
        const size_t pl = (size_t)n3[a2] * n3[b2];
        const size_t jj = (size_t)q[b2] * n3[a2] + q[a2];
        const double xi = tslb_inlet_xi(p.inlet[f2], L, x, y, z, p.tnext);
#pragma unroll
        for (int k = 0; k < 3; ++k) sts(a + (1 + k) * fs, tslb_inlet_u<T>(p.inlet[f2], pl, jj, k, xi));
        done = true;
    }
}

// WALL: 0 = no bounce-back wall, 1 = walls on y faces, 2 = walls on z faces, 3 = both (a duct), 4 = walls on x faces
// (x walls together with y or z walls: gather kernel)
template <typename T, int WALL, int ORDER, bool SPONGE, bool FUSE, int GEO>
__global__ void __maxnreg__((TileDims<T, GEO>::MAXREG))
sweep_tile_kernel(const __grid_constant__ CUtensorMap tmMain, const __grid_constant__ CUtensorMap tmRow,
                  const __grid_constant__ CUtensorMap tmStore, T *__restrict__ Bbuf, TileParams<T> p, const __grid_constant__ FuseParams fp,
                  const __grid_constant__ NbParams nb)
{
    typedef typename PackOf<T>::type P;
    typedef TileDims<T, GEO> TD;
    constexpr bool WALLY = (WALL & 1) != 0, WALLZ = (WALL & 2) != 0, WALLX = (WALL & 4) != 0;
    constexpr int NS = TD::NS, BXW = TD::BXW, FS = TD::FS, ROWS = TD::ROWS, COLS = TD::COLS, WY = TD::WY, WX = TD::WX;
    constexpr int NPACK = TD::NPACK, NGRP = TD::NGRP, EXW = TD::EXW, XPAD = TD::XPAD;
    constexpr int ES = (int)sizeof(T);
    constexpr int STAGE_BYTES = TD::STAGE_ELEMS * ES, SLOT_BYTES = TD::EX_SLOT * ES;
    // Exchange area: exX [2 slots][NPACK][NGRP][EXW] = M of a pack's row .x, main pair wy at index wy, the halo pair at WY;
    //                exY (2 slots further) = P of a pack's row .y, main pair wy at index wy + 1, the halo pair at 0.
    // So the pair below pair wy (its "down" source) is exY[wy] and the pair above (its "up" source) exX[wy + 1] for every
    // wy, the halo pair included: all three addresses of a main warp are one register plus immediates.
    constexpr int PACK_BYTES = NGRP * EXW * ES;
    constexpr int OFF_EXY = TD::OFF_EX + 2 * SLOT_BYTES;
    constexpr int NOUT = TD::NOUT, OUT_BYTES = TD::OUT_BYTES;
    // barriers (8 bytes each): full[NS], empty[NS], ofull[NOUT], oempty[NOUT]; between them the "published" flags q of the y
    // exchange, 16 bytes per pair (one 32-bit plane counter per warp wx at + 4 wx): the halo pair has two entries (index 0
    // and WY + 1, it sets both), main pair wy has index wy + 1: a warp polls the flags of its wx at index - 1 and index + 1.
    constexpr int B_FULL = TD::OFF_BAR, B_EMPTY = B_FULL + 8 * NS, B_Q = B_EMPTY + 8 * NS, B_OFULL = B_Q + 16 * (NPACK + 1), B_OEMPTY = B_OFULL + 8 * NOUT;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const uint32_t sb = keep(smem_u32(smem_raw));

    const int lane = threadIdx.x & 31;
    const int wid = threadIdx.x >> 5;
    const Layout &L = p.L;

    // tile origin; the last tile of the y axis is shifted back so that every tile is full (ny >= ROWS is required; overlapped
    // rows are computed twice, to identical values)
    const int x0 = blockIdx.x * COLS;
    const int row0 = min((int)blockIdx.y * ROWS, L.ny - ROWS);
    const int z0 = p.zbeg + blockIdx.z * p.zchunk;
    const int z1 = min(z0 + p.zchunk, p.zend);
    const int nplanes = z1 - z0 + 2;                     // source planes z0-1 .. z1
    // z of the i-th source plane (wrapped on a periodic axis; beyond a wall / open face the plane is zero-filled and the
    // index only has to be valid): needed for the per-plane relaxation of a sponge layer
    auto zsrc = [&](int i) {
        const int zs = z0 - 1 + i;
        const bool zp = p.kind[4] == TSLB_BC_PERIODIC;
        return zs < 0 ? (zp ? L.nz - 1 : 0) : (zs >= L.nz ? (zp ? 0 : L.nz - 1) : zs);
    };

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) { mbar_init(sb + B_FULL + 8 * s, 1); mbar_init(sb + B_EMPTY + 8 * s, TD::WARPS); }
        if (TileGeom<T, GEO>::QFLAGS) {
            for (int s = 0; s < 4 * (NPACK + 1); ++s)                               // published flags: 4 bytes per warp, zero = nothing yet
                asm volatile("st.shared.u32 [%0], %1;" ::"r"(sb + B_Q + 4 * s), "r"(0u) : "memory");
        } else {
            for (int s = 0; s < 2 * (NPACK + 1); ++s) mbar_init(sb + B_Q + 8 * s, WX);
        }
#pragma unroll
        for (int s = 0; s < NOUT; ++s) { mbar_init(sb + B_OFULL + 8 * s, TD::NMAIN); mbar_init(sb + B_OEMPTY + 8 * s, 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_async_smem();
    }
    __syncthreads();

    typedef TileGeom<T, GEO> GE;
    if (GE::REG_MAIN != 0) {
        if (wid >= TD::NMAIN) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(GE::REG_HALO ? GE::REG_HALO : 24));
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(GE::REG_MAIN ? GE::REG_MAIN : 24));
    }
    static_assert(GE::NIDLE == 2, "the two warps that complete the helpers' warpgroup are the producer and the store warp");
    if (wid >= TD::WARPS) {
        // ============================================ producer warp / store warp ==========================================
        // One lane each.  They are warps of their own (not lanes of the halo warps) so that a load is issued the moment its
        // stage has been released and a store the moment its tile is full, whatever the halo warps are doing: with the
        // producer inside a halo warp the load of plane i+1 could not be issued before plane i-1 had LANDED and been
        // processed there, which left the main warps waiting ~300 cycles per plane for their data.
        if (FUSE && wid == TD::WARPS + 1) {
            // ================================== store warp with the fused boundary fill (a6) ==================================
            // Open faces (PAPER.md:181-196 Eq. 22-23, :202, :258): a boundary node of time t+1 takes the 10 moments of the
            // interior node x_F its coordinates clamp to -- moments this very sweep produces -- and then the imposed velocity
            // (inlet) or density (pressure outlet).  The whole warp patches the finished output tile in shared memory before
            // the TMA store: boundary nodes on lateral faces copy from their x_F inside the tile; a boundary PLANE (z = 0 or
            // nz-1) is the patched tile of its neighbour plane stored a second time, with the imposed values written over it.
            // The host selects this path only when every boundary node shares a tile and a chunk with its x_F
            // (tile_fusable), so no separate fill launch is needed between steps.  The main warps' own results for boundary
            // nodes (nodes that are not advanced) are never stored.
            auto open_k = [&](int f) { const int k = p.kind[f]; return k == TSLB_BC_VELOCITY_INLET || k == TSLB_BC_OUTLET_ZERO_GRADIENT || k == TSLB_BC_OUTLET_PRESSURE; };
            const bool oxl = open_k(0), oxh = open_k(1), oyl = open_k(2), oyh = open_k(3), ozl = open_k(4), ozh = open_k(5);
            // which boundary rows / columns this tile holds (tile coordinates, -1 = none)
            const int bcol_lo = (oxl && x0 == 0) ? 0 : -1, bcol_hi = (oxh && x0 < L.nx && x0 + COLS >= L.nx) ? L.nx - 1 - x0 : -1;
            const int brow_lo = (oyl && row0 == 0) ? 0 : -1, brow_hi = (oyh && row0 + ROWS >= L.ny) ? L.ny - 1 - row0 : -1;
            const bool lateral = bcol_lo >= 0 || bcol_hi >= 0 || brow_lo >= 0 || brow_hi >= 0;
            // does any lateral face impose a value (inlet velocity, outlet density)?  plain zero-gradient outlets only copy
            auto imposes = [&](int f) { return p.kind[f] == TSLB_BC_VELOCITY_INLET || p.kind[f] == TSLB_BC_OUTLET_PRESSURE; };
            const bool imp_lateral = imposes(0) || imposes(1) || imposes(2) || imposes(3);
            auto impose = [&](uint32_t a, int x, int y, int z) { tile_impose<T>(fp, a, (uint32_t)(ROWS * COLS * ES), x, y, z); };
            // one boundary node of a lateral face, tile coordinates (r, cx): copy the 10 moments of its x_F, impose
            auto patch_node = [&](uint32_t tile, int r, int cx, int z) {
                const int x = x0 + cx, y = row0 + r;
                if (x >= L.nx) return;
                int xf = x, yf = y;
                if (x == 0 && oxl) xf = 1;
                if (x == L.nx - 1 && oxh) xf = L.nx - 2;
                if (y == 0 && oyl) yf = 1;
                if (y == L.ny - 1 && oyh) yf = L.ny - 2;
                const uint32_t src = tile + ((yf - row0) * COLS + (xf - x0)) * ES, dst = tile + (r * COLS + cx) * ES;
                T v[TSLB_NF];
#pragma unroll
                for (int f = 0; f < TSLB_NF; ++f) v[f] = lds(src + f * (ROWS * COLS) * ES, T());
#pragma unroll
                for (int f = 0; f < TSLB_NF; ++f) sts(dst + f * (ROWS * COLS) * ES, v[f]);
                if (imp_lateral) impose(dst, x, y, z);
            };
            int pending = -1;                                  // tile whose last store may still be reading it
            for (int m = 0; m < nplanes - 2; ++m) {
                const int b = m % NOUT, z = z0 + m;
                const uint32_t tile = sb + TD::OFF_OUT + b * OUT_BYTES;
                mbar_wait(sb + B_OFULL + 8 * b, (uint32_t)((m / NOUT) & 1));
                const bool zplane = (z == 0 && ozl) || (z == L.nz - 1 && ozh);   // a boundary plane: not advanced
                int groups = 0;
                if (!zplane) {
                    if (lateral) {
                        // (a corner node is patched by its row and by its column, with the same values; x_F is never a
                        //  boundary node, so the order of the copies does not matter)
                        if (brow_lo >= 0) for (int cx = lane; cx < COLS; cx += 32) patch_node(tile, brow_lo, cx, z);
                        if (brow_hi >= 0) for (int cx = lane; cx < COLS; cx += 32) patch_node(tile, brow_hi, cx, z);
                        if (lane < ROWS) {
                            if (bcol_lo >= 0) patch_node(tile, lane, bcol_lo, z);
                            if (bcol_hi >= 0) patch_node(tile, lane, bcol_hi, z);
                        }
                        __syncwarp();
                    }
                    if (lane == 0) {
                        fence_async_smem();
                        tma_store_4d(tile, &tmStore, x0 + TSLB_XOFF, row0, z, 0);
                        tma_store_commit();
                    }
                    ++groups;
                    const int zb = (z == 1 && ozl) ? 0 : ((z == L.nz - 2 && ozh) ? L.nz - 1 : -1);
                    if (zb >= 0) {                             // the boundary plane next to this one
                        if (lane == 0) tma_store_wait_read();  // the store above has read the tile
                        __syncwarp();
                        if (imp_lateral || imposes(zb == 0 ? 4 : 5)) {
                            for (int idx = lane; idx < ROWS * COLS; idx += 32) {
                                const int r = idx / COLS, cx = idx - r * COLS, x = x0 + cx, y = row0 + r;
                                if (x < L.nx) impose(tile + idx * ES, x, y, zb);
                            }
                        }
                        __syncwarp();
                        if (lane == 0) {
                            fence_async_smem();
                            tma_store_4d(tile, &tmStore, x0 + TSLB_XOFF, row0, zb, 0);
                            tma_store_commit();
                        }
                        ++groups;
                    }
                }
                if (lane == 0) {
                    if (NOUT == 1 || groups != 1) {            // nothing or two groups from this tile: drain, hand back everything
                        tma_store_wait_read();
                        if (pending >= 0) mbar_arrive(sb + B_OEMPTY + 8 * pending);
                        mbar_arrive(sb + B_OEMPTY + 8 * b);
                    } else if (pending >= 0) {
                        asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
                        mbar_arrive(sb + B_OEMPTY + 8 * pending);
                    }
                }
                pending = (NOUT == 1 || groups != 1) ? -1 : b;
            }
            if (lane == 0) tma_store_wait_all();
            return;
        }
        if (lane != 0) return;
        if (wid == TD::WARPS) {
            const bool yper = p.kind[2] == TSLB_BC_PERIODIC, zper = p.kind[4] == TSLB_BC_PERIODIC;
            // source rows of the two halo rows: wrapped on a periodic axis, out of bounds (zero fill) beyond a wall / open face
            const int ylo = row0 > 0 ? row0 - 1 : (yper ? L.ny - 1 : -1);
            const int yhi = row0 + ROWS < L.ny ? row0 + ROWS : (yper ? 0 : L.ny);
            for (int j = 0; j < nplanes; ++j) {            // source plane z0-1+j into stage j % NS
                // (beyond a z wall the plane NEXT to the wall is loaded once more: its own coefficients give the bounced
                //  populations, see "halfway bounce-back on a z face" in the main warps)
                int zs = z0 - 1 + j;
                if (zs < 0) zs = zper ? L.nz - 1 : ((WALLZ && p.kind[4] == TSLB_BC_BOUNCE_BACK) ? 0 : -1);
                else if (zs >= L.nz) zs = zper ? 0 : ((WALLZ && p.kind[5] == TSLB_BC_BOUNCE_BACK) ? L.nz - 1 : L.nz);
                const int s = j % NS;
                if (j >= NS) mbar_wait(sb + B_EMPTY + 8 * s, (uint32_t)((j / NS - 1) & 1));
                const uint32_t dst = sb + s * STAGE_BYTES, bar = sb + B_FULL + 8 * s;
                mbar_expect_tx(bar, (uint32_t)TD::STAGE_TX);
                // the ghost plane of a slab whose neighbour is attached: the neighbour's own plane, in place
                const CUtensorMap *mm = &tmMain, *mr = &tmRow;
                if (zs == 0 && nb.on[0]) { mm = &nb.main[0]; mr = &nb.row[0]; zs = nb.z[0]; }
                else if (zs == L.nz - 1 && nb.on[1]) { mm = &nb.main[1]; mr = &nb.row[1]; zs = nb.z[1]; }
                tma_load_4d(dst, mm, bar, x0, row0, zs, 0);
                tma_load_4d(dst + TD::MAIN_ELEMS * ES, mr, bar, x0, ylo, zs, 0);
                tma_load_4d(dst + (TD::MAIN_ELEMS + TD::HALO_ELEMS) * ES, mr, bar, x0, yhi, zs, 0);
            }
        } else {
            // output plane m of this chunk (z = z0 + m) sits in output tile m % NOUT; its k-th use completes phase k of the
            // tile's ofull / oempty barriers.  With two tiles the store of plane m is left in flight and the tile of plane
            // m-1 is handed back once ITS store has read the shared memory (at most one bulk group pending).
            for (int m = 0; m < nplanes - 2; ++m) {
                const int b = m % NOUT;
                mbar_wait(sb + B_OFULL + 8 * b, (uint32_t)((m / NOUT) & 1));
                if (TILE_FENCE_STORER) fence_async_smem();
                tma_store_4d(sb + TD::OFF_OUT + b * OUT_BYTES, &tmStore, x0 + TSLB_XOFF, row0, z0 + m, 0);
                tma_store_commit();
                if (NOUT == 1) {
                    tma_store_wait_read();
                    mbar_arrive(sb + B_OEMPTY);
                } else if (m >= 1) {
                    asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
                    mbar_arrive(sb + B_OEMPTY + 8 * ((m - 1) % NOUT));
                }
            }
            tma_store_wait_all();
        }
        return;
    }
    if (wid >= TD::NMAIN) {
        // =================================================== halo warps ===================================================
        const int h = wid - TD::NMAIN;
        // lane l of halo warp h holds the same tile column as lane l of the main warps wx = h, and publishes into the same
        // per-warp column of the exchange area (32 h + lane): every reader depends on ONE publishing warp only
        const int ecol = 32 * h + lane;
        const int bcol = TILE_COLS * h - 1 + lane + XPAD;  // box column
        // pack .x = tile row ROWS (above the tile), .y = tile row -1 (below): it publishes (M of .x, P of .y) like any pack
        const uint32_t aA = keep(sb + (TD::MAIN_ELEMS + TD::HALO_ELEMS + bcol) * ES), aB = keep(sb + (TD::MAIN_ELEMS + bcol) * ES);
        const uint32_t aW = keep(sb + TD::OFF_EX + (WY * NGRP * EXW + ecol) * ES);      // exX[WY]; exY[0] is HALO_Y further
        constexpr int HALO_Y = 2 * SLOT_BYTES - WY * PACK_BYTES;
        // rows beyond a bounce-back wall send nothing (their raw moments are zero-filled, but A100 = 3 g is not zero)
        const P hm = pk((WALLY && p.kind[3] == TSLB_BC_BOUNCE_BACK && row0 + ROWS >= L.ny) ? (T)0 : (T)1,
                        (WALLY && p.kind[2] == TSLB_BC_BOUNCE_BACK && row0 == 0) ? (T)0 : (T)1);
        int stg = 0;
        uint32_t fpar = 0;
        for (int i = 0; i < nplanes; ++i) {
            const uint32_t so = stg * STAGE_BYTES;
            T bz = p.beta;
            if (SPONGE) bz = __ldg(p.beta_z + zsrc(i));
            mbar_wait(sb + B_FULL + 8 * stg, fpar);
            P rh[TSLB_NF];
#pragma unroll
            for (int f = 0; f < TSLB_NF; ++f) rh[f] = pk(lds(aA + so + f * BXW * ES, T()), lds(aB + so + f * BXW * ES, T()));
            warp_arrive(sb + B_EMPTY + 8 * stg, lane);
            const uint32_t w = aW + (i & 1) * SLOT_BYTES;
            // the exchange slot is reused every second plane: its readers (the first and the last row pair of the tile) have
            // finished reading plane i-2 once they have published plane i-1.  (The main warps get the same guarantee from
            // waiting for the pairs they read from; the halo warps read nothing, so they wait explicitly.)
            if (i >= 2) {
                if (GE::QFLAGS) {
                    flag_wait(sb + B_Q + 16 * 1 + 4 * h, (uint32_t)i);         // pair 0, warp wx = h has published plane i-1
                    flag_wait(sb + B_Q + 16 * WY + 4 * h, (uint32_t)i);        // pair WY-1
                } else {
                    mbar_wait(sb + B_Q + 16 * 1 + 8 * ((i - 1) & 1), (uint32_t)(((i - 1) >> 1) & 1));
                    mbar_wait(sb + B_Q + 16 * WY + 8 * ((i - 1) & 1), (uint32_t)(((i - 1) >> 1) & 1));
                }
            }
#define TSLB_HALO_GROUP(KX, KZ)                                                                   \
            if (kvalid<ORDER>(KX, 0, KZ)) {                                                       \
                T p0, m0, p1, m1;                                                                 \
                P cen;                                                                            \
                ycombos<ORDER, KX, KZ, P, T>(A, p0, m0, p1, m1, cen);                             \
                if (WALLY) { m0 *= hm.x; p1 *= hm.y; }                                            \
                sts(w + qidx(KX, KZ) * EXW * ES, m0);                                             \
                sts(w + HALO_Y + qidx(KX, KZ) * EXW * ES, p1);                                    \
            }
#define TSLB_HALO_ROUND(KZ)                                                                       \
            {                                                                                     \
                P A[3][3];                                                                        \
                hermite_round<KZ, P, T>(rh, bz, p.g, A);                                          \
                TSLB_HALO_GROUP(0, KZ) TSLB_HALO_GROUP(1, KZ) TSLB_HALO_GROUP(2, KZ)              \
            }
            TSLB_HALO_ROUND(0)
            TSLB_HALO_ROUND(1)
            TSLB_HALO_ROUND(2)
#undef TSLB_HALO_ROUND
#undef TSLB_HALO_GROUP
            __syncwarp();
            if (lane == 0) {
                if (GE::QFLAGS) {
                    asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(sb + B_Q + 4 * h), "r"((uint32_t)(i + 1)) : "memory");
                    asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(sb + B_Q + 16 * (WY + 1) + 4 * h), "r"((uint32_t)(i + 1)) : "memory");
                } else {
                    mbar_arrive(sb + B_Q + 8 * (i & 1));
                    mbar_arrive(sb + B_Q + 16 * (WY + 1) + 8 * (i & 1));
                }
            }
            if (++stg == NS) { stg = 0; fpar ^= 1; }
        }
        return;
    }

    // ===================================================== main warps =====================================================
    // ---- columns: the warp outputs tile columns [30 wx, 30 wx + 30); lane l holds tile column 30 wx - 1 + l -----------------
    const int wx = wid % WX, wy = wid / WX;
    const int tc = TILE_COLS * wx - 1 + lane;
    const int col = x0 + tc;
    const bool lane_out = lane >= 1 && lane <= TILE_COLS;
    // ---- rows: pack .x = row r0, .y = row r0+1; outer neighbours r0-1, r0+2 -------------------------------------------------
    const int r0 = row0 + 2 * wy;
    // this warp owns a row next to a bounce-back wall (warp-uniform): .x row at the wall below / .y row at the wall above
    const bool ghost_lo = WALLY && p.kind[2] == TSLB_BC_BOUNCE_BACK && r0 == 0;
    const bool ghost_hi = WALLY && p.kind[3] == TSLB_BC_BOUNCE_BACK && r0 + 2 == L.ny;
    const bool any_ghost = ghost_lo || ghost_hi;

    // shared-memory addresses of this thread
    const int bcol = tc + XPAD;
    const uint32_t aC = keep(sb + ((2 * wy) * BXW + bcol) * ES);                 // row r0 in the main region (r0+1: + BXW)
    // u of rows r0-1 / r0+2: in the main region (field stride FS) or, at the tile edge, in a halo-row slot (field stride BXW)
    // (two code versions of the three loads, chosen by warp-uniform predicates, instead of run-time strides)
    const bool loEdge = wy == 0, hiEdge = wy == WY - 1;
    const uint32_t aLo = keep(sb + ((loEdge ? TD::MAIN_ELEMS + bcol + BXW : (2 * wy - 1) * BXW + bcol + FS)) * ES);   // field 1 (ux)
    const uint32_t aHi = keep(sb + ((hiEdge ? TD::MAIN_ELEMS + TD::HALO_ELEMS + bcol + BXW : (2 * wy + 2) * BXW + bcol + FS)) * ES);
    // exchange: every warp publishes lane for lane into its own 32 columns (32 wx + lane) of its pair's slots, and reads
    // the same columns of the pairs below and above: a reader depends on the publishing warp with ITS wx only (the two
    // nodes the warps of a pair share, lanes 30, 31 / 0, 1, are published twice), and the wall code re-reads a warp's own
    // columns, which nobody else writes.  The halo pair is below wy = 0 and above wy = WY-1.
    const int ecol = 32 * wx + lane;
    const uint32_t aW = keep(sb + TD::OFF_EX + (wy * NGRP * EXW + ecol) * ES);       // own: exX[wy]; exY[wy + 1] is OWN_Y further
    const uint32_t aR = aW;
    constexpr int OWN_Y = 2 * SLOT_BYTES + PACK_BYTES;
    constexpr int DN_OFF = 2 * SLOT_BYTES;                                           // exY[wy]: P of the row below
    constexpr int UP_OFF = PACK_BYTES;                                               // exX[wy + 1]: M of the row above
    const uint32_t aO = keep(sb + TD::OFF_OUT + ((2 * wy) * COLS + (tc < 0 ? 0 : tc)) * ES);           // output tile [f][row][tc]
    const uint32_t bQown = keep(sb + B_Q + 16 * (wy + 1) + (GE::QFLAGS ? 4 * wx : 0));   // own published flag / barriers; neighbours: - 16, + 16

    // z-march state per (px,py) group g, DOUBLE-BUFFERED over the parity of the source plane (the plane loop is unrolled by two
    // with the parity as a compile-time constant, so the march shifts no registers and every stage / slot / barrier offset
    // is an immediate):  vpb[par][g] = Vp of the source plane of parity par (Vp(zs-1) is in vpb[1-par], and vpb[par] still
    // holds Vp(zs-2) until this plane's Vp overwrites it);  ttb[par][g] = Vp(zs-2) + centre(zs-1), which this plane completes
    // (ttb[1-par] receives Vp(zs-1) + centre(zs) for the next one).
    P vpb[2][6], ttb[2][6];
    // increment form along z: velocity of the source planes and the backward difference, rows r0, r0+1
    P ub[2][3], db[2][3];
#pragma unroll
    for (int i = 0; i < 6; ++i) { vpb[0][i] = pbc<P, T>((T)0); vpb[1][i] = vpb[0][i]; ttb[0][i] = vpb[0][i]; ttb[1][i] = vpb[0][i]; }
#pragma unroll
    for (int a = 0; a < 3; ++a) { ub[0][a] = pbc<P, T>((T)0); ub[1][a] = ub[0][a]; db[0][a] = ub[0][a]; db[1][a] = ub[0][a]; }

    // ---- halfway bounce-back on an x face (WALL = 4).  A lane that holds a column beyond the wall sends nothing into the x
    //      pass (msrc = 0) and enters the x differences with u = 0; the lane that holds the wall column adds, one iteration
    //      later (when its plane is the target), the nine bounced populations f*_ibar of its own nodes: with
    //      Bx(ky,kz) = sum_kx t_kx(-c_x) A(kx,ky,kz) and the local sums over y and z the ten corrections are
    //      36 Bx00 | c_x 36 Bx00 | -12 Bx10 | -12 Bx01 | 36 Bx00 | 12 (Bx00 + Bx20) | 12 (Bx00 + Bx02) | -c_x 12 Bx10 |
    //      -c_x 12 Bx01 | 4 Bx11   for the moments 000 | 100 | 010 | 001 | 200 | 020 | 002 | 110 | 101 | 011. ---------------------
    const T cxl = !WALLX ? (T)0 : ((col == 0 && p.kind[0] == TSLB_BC_BOUNCE_BACK) ? (T)1
                                   : ((col == L.nx - 1 && p.kind[1] == TSLB_BC_BOUNCE_BACK) ? (T)-1 : (T)0));
    const P msrc = pbc<P, T>((WALLX && ((col < 0 && p.kind[0] == TSLB_BC_BOUNCE_BACK) || (col >= L.nx && p.kind[1] == TSLB_BC_BOUNCE_BACK))) ? (T)0 : (T)1);
    P bxs[2][6];                                          // Bx of the source planes by parity, used when the plane is the target
    if (WALLX) {
#pragma unroll
        for (int k = 0; k < 6; ++k) { bxs[0][k] = pbc<P, T>((T)0); bxs[1][k] = bxs[0][k]; }
    }
    const bool xper = p.kind[0] == TSLB_BC_PERIODIC;
    // periodic x: the node at x = 0 is also the ghost column x = nx, the node at x = nx-1 the ghost column x = -1
    const bool xedge = xper && lane_out && (col == 0 || col == L.nx - 1);
    const long long gcol = col == 0 ? (long long)L.nx + TSLB_XOFF : (long long)TSLB_XOFF - 1;
    // The TMA store works in 16-byte units: the output tensor is clipped at the last 16-byte boundary inside the row (a
    // partly covered unit would be written whole, over the ghost column), the columns beyond it are stored from registers
    const bool xtail = lane_out && col >= (L.nx & ~(16 / ES - 1)) && col < L.nx;

    // The barriers of the exchange slots and of the output tiles complete one phase every two planes (two slots, two tiles):
    // one phase bit serves them all, ph = (i >> 1) & 1; with NS == 2 it serves the stage ring as well and the stage offset is
    // an immediate, otherwise the ring position is carried (stg, fpar).
    uint32_t ph = 0;
    int stg = 0;
    uint32_t fpar = 0;
    auto plane = [&](auto par_c, const int i) {
        constexpr int PAR = decltype(par_c)::value;
        constexpr uint32_t xo = PAR * SLOT_BYTES;
        const uint32_t so = NS == 2 ? PAR * STAGE_BYTES : stg * STAGE_BYTES;
        const uint32_t bring = NS == 2 ? sb + 8 * PAR : sb + 8 * stg;          // + B_FULL / B_EMPTY
        P (&vp1)[6] = vpb[1 - PAR];          // Vp(zs-1)
        P (&vp0)[6] = vpb[PAR];              // Vp(zs-2) on entry (groups 0, 1, 3 read it first), Vp(zs) on exit
        P (&tt1)[6] = ttb[PAR];
        P (&tn)[6] = ttb[1 - PAR];
        P (&uprev)[3] = ub[1 - PAR];
        P (&ucur)[3] = ub[PAR];
        P (&dprev)[3] = db[1 - PAR];
        P (&dcur)[3] = db[PAR];
        // 1 - omega of the source plane: uniform, or per plane inside a sponge layer (Eq. 26)
        T bz = TILE_REREAD_PARAMS ? keepf(p.beta) : p.beta;
        if (SPONGE) bz = __ldg(p.beta_z + zsrc(i));
        T gz[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) gz[a] = TILE_REREAD_PARAMS ? keepf(p.g[a]) : p.g[a];
        mbar_wait(bring + B_FULL, NS == 2 ? ph : fpar);

        // ---- a1: moments of the own rows r0, r0+1 and the velocities of the rows r0-1, r0+2 at this column ------------------
        P rc[TSLB_NF], hu[3];
        {
            const uint32_t a = aC + so;
#pragma unroll
            for (int f = 0; f < TSLB_NF; ++f) rc[f] = pk(lds(a + f * FS * ES, T()), lds(a + (f * FS + BXW) * ES, T()));
            T hl[3], hh[3];
            if (loEdge) {
#pragma unroll
                for (int k = 0; k < 3; ++k) hl[k] = lds(aLo + so + k * BXW * ES, T());
            } else {
#pragma unroll
                for (int k = 0; k < 3; ++k) hl[k] = lds(aLo + so + k * FS * ES, T());
            }
            if (hiEdge) {
#pragma unroll
                for (int k = 0; k < 3; ++k) hh[k] = lds(aHi + so + k * BXW * ES, T());
            } else {
#pragma unroll
                for (int k = 0; k < 3; ++k) hh[k] = lds(aHi + so + k * FS * ES, T());
            }
#pragma unroll
            for (int k = 0; k < 3; ++k) hu[k] = pk(hl[k], hh[k]);
        }
        warp_arrive(bring + B_EMPTY, lane);              // the stage can be refilled: everything needed is in registers
        if (NS != 2 && ++stg == NS) { stg = 0; fpar ^= 1; }

        // ---- a2: Hermite coefficients of the own rows, all three rounds; y-pass combinations of the 8 groups -------------
        // For the output pack: up = (P(r0-1), P(r0)), dn = (M(r0+1), M(r0+2)); P(r0-1) and M(r0+2) are read from the neighbours,
        // P(r0) = qP0 and M(r0+1) = qM1 are the pack's own:  E = up + dn,  O = up - dn,  G0 = E + cen.
        // ---- halfway bounce-back on a z face: the source "plane" beyond the wall (zs = -1 / nz) holds the moments of the
        //      wall-adjacent plane once more (producer).  What that plane would send across the wall -- Vp(-1) into plane 0,
        //      Vm(nz) into plane nz-1 -- is replaced by the bounced populations f*_ibar of the nodes themselves: with
        //      Bz(kx,ky) = sum_kz t_kz(-c_z) A(kx,ky,kz) (M combination below, P above) and the local sums L(0,0) = 6,
        //      L(1,1) = -2, L(2,0) = L(2,2) = 2 over x and y,
        //        V(0,0) = 36 Bz00, V(1,0) = -12 Bz10, V(2,0) = 12 (Bz00 + Bz20), V(0,1) = -12 Bz01, V(1,1) = 4 Bz11,
        //        V(0,2) = 12 (Bz00 + Bz02);
        //      the z march then applies c_z^pz by itself.  The y / x passes of such a plane are skipped (CTA-uniform). ----------
        const int zsrc_raw = z0 - 1 + i;
        const bool wsrc_lo = WALLZ && zsrc_raw < 0 && p.kind[4] == TSLB_BC_BOUNCE_BACK;
        const bool wsrc_hi = WALLZ && zsrc_raw >= L.nz && p.kind[5] == TSLB_BC_BOUNCE_BACK;
        const bool wsrc = wsrc_lo || wsrc_hi;
        P Bz[6];                                          // (kx,ky) = 00, 10, 20, 01, 11, 02
        P Bx[6];                                          // (ky,kz) = 00, 10, 20, 01, 11, 02
        const T sz = wsrc_lo ? (T)-1 : (T)1;
        T qP0[NGRP], qM1[NGRP];
        P cen[NGRP];
        {
            const uint32_t w = aW + xo;
#define TSLB_MAIN_GROUP(KX, KZ)                                                                   \
            if (kvalid<ORDER>(KX, 0, KZ)) {                                                       \
                constexpr int q = qidx(KX, KZ);                                                   \
                T m0, p1;                                                                         \
                ycombos<ORDER, KX, KZ, P, T>(A, qP0[q], m0, p1, qM1[q], cen[q]);                  \
                sts(w + q * EXW * ES, m0);                                                        \
                sts(w + OWN_Y + q * EXW * ES, p1);                                                \
            }
#define TSLB_BZ(G, KX, KY, KZ)                                                                    \
            if (kvalid<ORDER>(KX, KY, KZ)) {                                                      \
                if (KZ == 0) Bz[G] = A[KX][KY];                                                   \
                else if (KZ == 1) Bz[G] = pfmas(A[KX][KY], sz, Bz[G]);                            \
                else Bz[G] = padd(Bz[G], A[KX][KY]);                                              \
            }
#define TSLB_MAIN_ROUND(KZ)                                                                       \
            {                                                                                     \
                P A[3][3];                                                                        \
                hermite_round<KZ, P, T>(rc, bz, gz, A);                                           \
                if (WALLZ && wsrc) {                                                              \
                    TSLB_BZ(0, 0, 0, KZ) TSLB_BZ(1, 1, 0, KZ) TSLB_BZ(2, 2, 0, KZ)                \
                    TSLB_BZ(3, 0, 1, KZ) TSLB_BZ(4, 1, 1, KZ) TSLB_BZ(5, 0, 2, KZ)                \
                }                                                                                 \
                if (WALLX) {                                                                      \
                    if (KZ == 0) { Bx[0] = bx_combo<ORDER, 0, KZ, P, T>(A, cxl); Bx[1] = bx_combo<ORDER, 1, KZ, P, T>(A, cxl); Bx[2] = bx_combo<ORDER, 2, KZ, P, T>(A, cxl); \
                                   Bx[0] = pfmas(rc[1], (T)-3 * cxl, Bx[0]); Bx[1] = pfmas(rc[2], (T)3, Bx[1]); }                                                        \
                    if (KZ == 1) { Bx[3] = pfmas(rc[3], (T)3, bx_combo<ORDER, 0, KZ, P, T>(A, cxl)); Bx[4] = bx_combo<ORDER, 1, KZ, P, T>(A, cxl); }                      \
                    if (KZ == 2) { Bx[5] = bx_combo<ORDER, 0, KZ, P, T>(A, cxl); }                                                                                        \
                }                                                                                 \
                TSLB_MAIN_GROUP(0, KZ) TSLB_MAIN_GROUP(1, KZ) TSLB_MAIN_GROUP(2, KZ)              \
            }
            TSLB_MAIN_ROUND(0)
            TSLB_MAIN_ROUND(1)
            TSLB_MAIN_ROUND(2)
#undef TSLB_MAIN_ROUND
#undef TSLB_MAIN_GROUP
#undef TSLB_BZ
        }
        if (GE::QFLAGS) flag_set(bQown, (uint32_t)(i + 1), lane);
        else warp_arrive(bQown + 8 * PAR, lane);

        if (WALLX) {                                      // kept for the next iteration, when this plane is the target
#pragma unroll
            for (int k = 0; k < 6; ++k) bxs[PAR][k] = Bx[k];
        }

        // ---- increment form along y: exact differences of the stored velocities,
        //      Ly = (up - c) + (dn - c), Wy = (up - dn) * sgn with up / dn the neighbour rows (hu = (u(r0-1), u(r0+2)), the
        //      other neighbour is the pack's other row); a node beyond a wall has u = 0 (zero-filled halo row).  They enter
        //      the y pass of the groups that carry a first-order coefficient:  E += incE, O += incO  with
        //      (kx,kz) = (1,0): 3 Ly_x, sg3 Wy_x;   (0,0): sg3 Wy_y, 3 Ly_y;   (0,1): 3 Ly_z, sg3 Wy_z. -------------------------
        const P sg3 = pk((T)3, (T)-3);
        // (after the publish: the neighbours do not wait for this)
        P incE[3], incO[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const P uc = rc[1 + a];
            const P cs = pswap(uc);
            const P ly3 = pmuls(pfmas(uc, (T)-2, padd(hu[a], cs)), (T)3);
            const P wy3 = pmul(psub(hu[a], cs), sg3);
            incE[a] = a == 1 ? wy3 : ly3;
            incO[a] = a == 1 ? ly3 : wy3;
        }

        // increment form along z: exact differences of the stored velocities at the target plane zs-1
        P Lz[3], Dz[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            // (a plane beyond a z wall enters the differences with u = 0, like the ghost rows of a y wall)
            const P uz = (WALLZ && wsrc) ? pbc<P, T>((T)0) : rc[1 + a];
            ucur[a] = uz;
            const P dc = psub(uz, uprev[a]);             // u(zs) - u(zs-1)
            Lz[a] = psub(dc, dprev[a]);
            Dz[a] = padd(dprev[a], dc);                  // u(zs) - u(zs-2) = -(D along z); used with negated multipliers
            dcur[a] = dc;
        }
        // the z-pass terms that need Vp(zs-2) alone (groups 0, 1, 3), taken before this plane's Vp overwrites it; the z-stage
        // increments (base multipliers 36 for ux, uy; 108 / 36 for uz) go into the sums now, so that no difference stays live
        const P e3 = pfmas(Lz[2], (T)108, vp0[0]);       // 001
        const P e6 = pfmas(Dz[2], (T)-108, vp0[0]);      // 002
        const P e8 = pfmas(Dz[0], (T)-36, vp0[1]);       // 101
        const P e9 = pfmas(Dz[1], (T)-36, vp0[3]);       // 011
        tt1[0] = pfmas(Dz[2], (T)-108, tt1[0]);          // 000
        tt1[1] = pfmas(Lz[0], (T)36, tt1[1]);            // 100
        tt1[3] = pfmas(Lz[1], (T)36, tt1[3]);            // 010
        tt1[2] = pfmas(Dz[2], (T)-36, tt1[2]);           // 200
        tt1[5] = pfmas(Dz[2], (T)-36, tt1[5]);           // 020

        // ---- the neighbours' combinations -----------------------------------------------------------------------------------
        if (GE::QFLAGS) {
            flag_wait(bQown - 16, (uint32_t)(i + 1));
            flag_wait(bQown + 16, (uint32_t)(i + 1));
        } else {
            mbar_wait(bQown - 16 + 8 * PAR, ph);
            mbar_wait(bQown + 16 + 8 * PAR, ph);
        }
        const uint32_t rdn = aR + DN_OFF + xo, rup = aR + UP_OFF + xo;

        // this plane's contributions to the z march, accumulated over kz where they are needed:
        //   tt1[g] += Vm(zs)            (pz = 0 of the target plane zs-1; groups 2, 4, 5, where Vm is not needed alone)
        //   vm0[g]  = Vm(zs)            (groups 0, 1, 3)
        //   tn[g]   = vp1[g] + centre(zs)   (the next plane's tt1)
        //   vp0[g]  = Vp(zs)
        // with Vp = phi0 + phi1 + phi2, Vm = phi0 - phi1 + phi2, centre = 4 phi0 - 2 phi2 over kz.
        P vm0[6];
        if (WALLZ && wsrc) {
            // full first-order coefficients (the passes carry them without their base 3 u)
            const P b00 = pfmas(rc[3], (T)3 * sz, Bz[0]);
            const P b10 = pfmas(rc[1], (T)3, Bz[1]);
            const P b01 = pfmas(rc[2], (T)3, Bz[3]);
            P V[6];
            V[0] = pmuls(b00, (T)36);
            V[1] = pmuls(b10, (T)-12);
            V[2] = pmuls(padd(b00, Bz[2]), (T)12);
            V[3] = pmuls(b01, (T)-12);
            V[4] = kvalid<ORDER>(1, 1, 0) ? pmuls(Bz[4], (T)4) : pbc<P, T>((T)0);
            V[5] = pmuls(padd(b00, Bz[5]), (T)12);
#pragma unroll
            for (int g = 0; g < 6; ++g) {
                const bool alone = g == 0 || g == 1 || g == 3;
                if (wsrc_lo) { vp0[g] = V[g]; tn[g] = pbc<P, T>((T)0); if (alone) vm0[g] = pbc<P, T>((T)0); }   // Vp(-1) into plane 0
                else if (alone) vm0[g] = V[g];                                                              // Vm(nz) into plane nz-1
                else tt1[g] = padd(tt1[g], V[g]);
            }
        } else
#pragma unroll
        for (int kz = 0; kz < 3; ++kz) {
            // ---- y pass: G1[py][kx] = sum_ky T^y_{py,ky} A(kx,ky,kz) at rows r0, r0+1 ---------------------------------------
            P G1[3][3];
#pragma unroll
            for (int kx = 0; kx < 3; ++kx) {
                if (!kvalid<ORDER>(kx, 0, kz)) continue;
                const int q = qidx(kx, kz);
                // (scalar adds: their operands are scalars from four different places, a packed add would need them moved
                //  into register pairs first)
                const T pdn = lds(rdn + q * EXW * ES, T()), mup = lds(rup + q * EXW * ES, T());
                P E = pk(pdn + qM1[q], qP0[q] + mup), O = pk(pdn - qM1[q], qP0[q] - mup);
                // (kx,kz) = (1,0): ux, (0,0): uy, (0,1): uz carry the y-stage increments
                const int ia = q == qidx(1, 0) ? 0 : (q == qidx(0, 0) ? 1 : (q == qidx(0, 1) ? 2 : -1));
                if (ia >= 0) { E = padd(E, incE[ia]); O = padd(O, incO[ia]); }
                G1[2][kx] = E;
                G1[1][kx] = O;
                G1[0][kx] = padd(E, cen[q]);
            }
            // x differences of the stored velocities (increment form along x), from the neighbour lanes
            P Lx[3], Dx[3];
            if (kz == 0) {
#pragma unroll
                for (int a = 0; a < 2; ++a) {
                    const P us = WALLX ? pmul(rc[1 + a], msrc) : rc[1 + a];
                    const P xl = shfl_up1(us), xr = shfl_dn1(us);
                    Lx[a] = pfmas(rc[1 + a], (T)-2, padd(xl, xr));
                    Dx[a] = psub(xl, xr);
                }
            }
            if (kz == 1) {
                const P us = WALLX ? pmul(rc[3], msrc) : rc[3];
                const P xl = shfl_up1(us), xr = shfl_dn1(us);
                Lx[2] = pfmas(rc[3], (T)-2, padd(xl, xr));
                Dx[2] = psub(xl, xr);
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
                if (WALLX) { pp = pmul(pp, msrc); mm = pmul(mm, msrc); }
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
                    const bool alone = gi == 0 || gi == 1 || gi == 3;      // Vm needed on its own (pz = 1, 2)
                    const P v = o[px];
                    if (kz == 0) { vp0[gi] = v; tn[gi] = pfmas(v, (T)4, vp1[gi]); if (alone) vm0[gi] = v; else tt1[gi] = padd(tt1[gi], v); }
                    if (kz == 1) { vp0[gi] = padd(vp0[gi], v); if (alone) vm0[gi] = psub(vm0[gi], v); else tt1[gi] = psub(tt1[gi], v); }
                    if (kz == 2) { vp0[gi] = padd(vp0[gi], v); tn[gi] = pfmas(v, (T)-2, tn[gi]); if (alone) vm0[gi] = padd(vm0[gi], v); else tt1[gi] = padd(tt1[gi], v); }
                }
            }
        }

        // ---- halfway bounce-back on a y face: for a wall-adjacent row the 9
        //      populations arriving from beyond the wall are f*_ibar of the node itself, a local combination of its own
        //      coefficients  B(kx,kz) = sum_ky t_ky(-c_y) A(kx,ky,kz)  -- exactly the published combination of that row
        //      (M of a row at the wall below, P of a row at the wall above) -- with the local sums L(0,0)=6, L(1,1)=-2,
        //      L(2,0)=L(2,2)=2. ---------------------------------------------------------------------------------------------
        // The six bounced populations with c_z = 0 go into this plane's centre terms (they reach the target plane through
        // tt1); the four moments with c_z (001, 002, 101, 011) belong to the target plane zs-1 and are rebuilt there from
        // that plane's combinations, which still sit in the other exchange slot (kwall below).
        P kwall[4];
        if (WALLY) {
#pragma unroll
            for (int k = 0; k < 4; ++k) kwall[k] = pbc<P, T>((T)0);
        }
        // Duct (walls on y AND z): on a row next to a y wall of a plane next to a z wall the three populations that arrive
        // across the edge (c_y and c_z both pointing out of the walls) are in the y correction (9 populations, all c_z)
        // and in the z replacement V (9 populations, all c_y): they are taken out once.  With
        // Bm(kx) = sum_kz t_kz(-c_z) B(kx,kz) and the local sums over x:  e(px,py,pz) = c_y^py c_z^pz (6 Bm0 | -2 Bm1 | 2 (Bm0 + Bm2)).
        P ewall[TSLB_NF];
        bool edge = false;
        if (WALLY && any_ghost) {
            // (the flags pass through an opaque asm so that the packs below are rebuilt here, a few selects, instead of being
            //  hoisted out of the plane loop, where they would occupy 14 registers of every main warp all the time)
            const bool glo = keep((uint32_t)ghost_lo) != 0u, ghi = keep((uint32_t)ghost_hi) != 0u;
            const P wsp = pk(glo ? (T)-1 : (T)1, (T)1);
            const P wm = pk(glo ? (T)1 : (T)0, ghi ? (T)1 : (T)0);                         // which row of the pack is at a wall
            const P sgp = pk(glo ? (T)1 : (T)-1, (T)-1);                                   // c_y of the arrival direction
            const P w12 = pmuls(wm, (T)12), w36 = pmuls(wm, (T)36), w12s = pmul(w12, sgp), w36s = pmul(w36, sgp);
            // (re-read from this warp's own exchange slots instead of being kept in registers across the passes; lanes 0, 1 of
            //  the wx = 1 warp published in the private columns 62, 63)
            auto own = [&](uint32_t w, int q) { return pk(lds(w + q * EXW * ES, T()), lds(w + OWN_Y + q * EXW * ES, T())); };
            {   // source plane zs: full first-order coefficients (the passes carry them without their base 3 u)
                const uint32_t w = aW + xo;
                const P WB10 = pfmas(rc[1], (T)3, own(w, qidx(1, 0)));
                const P WB00 = pfma(rc[2], pmuls(wsp, (T)3), own(w, qidx(0, 0)));
                const P WB20 = own(w, qidx(2, 0));
                tn[0] = pfma(WB00, w36, tn[0]);                             // 000
                tn[1] = pfma(WB10, pmuls(w12, (T)-1), tn[1]);               // 100
                tn[3] = pfma(WB00, w36s, tn[3]);                            // 010
                tn[2] = pfma(padd(WB00, WB20), w12, tn[2]);                 // 200
                tn[5] = pfma(WB00, w36, tn[5]);                             // 020
                tn[4] = pfma(WB10, pmuls(w12s, (T)-1), tn[4]);              // 110
            }
            if (i >= 2) {   // target plane zs-1 (its velocities are uprev)
                const uint32_t w = aW + (SLOT_BYTES - xo);
                const P WB00 = pfma(uprev[1], pmuls(wsp, (T)3), own(w, qidx(0, 0)));
                const P WB01 = pfmas(uprev[2], (T)3, own(w, qidx(0, 1)));
                const P WB11 = own(w, qidx(1, 1)), WB02 = own(w, qidx(0, 2));
                kwall[0] = pmul(WB01, pmuls(w12, (T)-1));                   // 001
                kwall[1] = pmul(padd(WB00, WB02), w12);                     // 002
                kwall[2] = pmul(WB11, pmuls(wm, (T)4));                     // 101
                kwall[3] = pmul(WB01, pmuls(w12s, (T)-1));                  // 011
                if (WALLZ) {
                    const int ztw = z0 + i - 2;
                    const bool e_lo = ztw == 0 && p.kind[4] == TSLB_BC_BOUNCE_BACK, e_hi = ztw == L.nz - 1 && p.kind[5] == TSLB_BC_BOUNCE_BACK;
                    if (e_lo || e_hi) {
                        edge = true;
                        const T cz = e_lo ? (T)1 : (T)-1;
                        const P F10 = pfmas(uprev[0], (T)3, own(w, qidx(1, 0)));
                        P Bm0 = padd(pfmas(WB01, -cz, WB00), WB02);
                        P Bm1 = pfmas(WB11, -cz, F10);
                        if (kvalid<ORDER>(1, 0, 2)) Bm1 = padd(Bm1, own(w, qidx(1, 2)));
                        P Bm2 = own(w, qidx(2, 0));
                        if (kvalid<ORDER>(2, 0, 1)) Bm2 = pfmas(own(w, qidx(2, 1)), -cz, Bm2);
                        const P s6 = pmul(pmuls(Bm0, (T)6), wm), s2 = pmul(pmuls(Bm1, (T)-2), wm);
                        ewall[0] = s6; ewall[1] = s2; ewall[2] = pmul(s6, sgp); ewall[3] = pmuls(s6, cz);
                        ewall[4] = pmul(pmuls(padd(Bm0, Bm2), (T)2), wm); ewall[5] = s6; ewall[6] = s6;
                        ewall[7] = pmul(s2, sgp); ewall[8] = pmuls(s2, cz); ewall[9] = pmuls(pmul(s6, sgp), cz);
                    }
                }
            }
        }

        // ---- z pass for target plane zt = zs - 1:  pz=0: Vp(zs-2) + centre(zs-1) + Vm(zs);  pz=1: Vp(zs-2) - Vm(zs);
        //      pz=2: Vp(zs-2) + Vm(zs); plus the z-stage increments (base multipliers 36 for ux, uy; 108 / 36 for uz) ----
        if (i >= 2) {
            const int zt = z0 + i - 2;
            P m[TSLB_NF];
            m[0] = padd(tt1[0], vm0[0]);                                 // 000
            m[3] = psub(e3, vm0[0]);                                     // 001
            m[6] = padd(e6, vm0[0]);                                     // 002
            m[1] = padd(tt1[1], vm0[1]);                                 // 100
            m[8] = psub(e8, vm0[1]);                                     // 101
            m[2] = padd(tt1[3], vm0[3]);                                 // 010
            m[9] = psub(e9, vm0[3]);                                     // 011
            m[4] = tt1[2];                                               // 200
            m[7] = tt1[4];                                               // 110
            m[5] = tt1[5];                                               // 020
            if (WALLY) { m[3] = padd(m[3], kwall[0]); m[6] = padd(m[6], kwall[1]); m[8] = padd(m[8], kwall[2]); m[9] = padd(m[9], kwall[3]); }
            if (WALLX && cxl != (T)0) {                   // (divergent inside an edge warp only: no shuffles in here)
                const P (&bx)[6] = bxs[1 - PAR];
                const P b36 = pmuls(bx[0], (T)36), n10 = pmuls(bx[1], (T)-12), n01 = pmuls(bx[3], (T)-12);
                m[0] = padd(m[0], b36); m[1] = pfmas(b36, cxl, m[1]); m[2] = padd(m[2], n10); m[3] = padd(m[3], n01);
                m[4] = padd(m[4], b36);
                m[5] = pfmas(padd(bx[0], bx[2]), (T)12, m[5]);
                m[6] = pfmas(padd(bx[0], bx[5]), (T)12, m[6]);
                m[7] = pfmas(n10, cxl, m[7]); m[8] = pfmas(n01, cxl, m[8]);
                m[9] = pfmas(bx[4], (T)4, m[9]);
            }
            if (WALLY && WALLZ && edge) {
#pragma unroll
                for (int k = 0; k < TSLB_NF; ++k) m[k] = psub(m[k], ewall[k]);
            }

            // ---- a8: finalise the two rows from their 216-scaled raw moments (m[1..3] lack their base 216 u), Eq. 12 ------
            // x/216 as x*hi + x*lo: unbiased to ~1 ulp (a rounded 1/216 alone would be a systematic gain)
            const T hi = (T)(1.0 / 216.0);
            const T lo = (T)(1.0 / 216.0 - (double)hi);
            const P dR = pfmas(m[0], lo, pmuls(m[0], hi));
            const P rho = padd(pbc<P, T>((T)1), dR);
            const P den = padd(pbc<P, T>((T)216), m[0]);
            const P inv = pk(rcp_fast(den.x), rcp_fast(den.y));
            const P nm0 = pmuls(m[0], (T)-1);
            // u' = (216 u + J) / (216 + dR216) = u + (J - u dR216) / (216 + dR216)
            P o[TSLB_NF];
            o[0] = dR;
#pragma unroll
            for (int a = 0; a < 3; ++a) o[1 + a] = pfma(pfma(uprev[a], nm0, m[1 + a]), inv, uprev[a]);
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

            // ---- into the output tile of this parity (the store thread has read the plane before the previous one out of it;
            //      with a single tile: the previous one) --------------------------------------------------------------------
            constexpr int ob = NOUT == 2 ? PAR : 0;
            mbar_wait(sb + B_OEMPTY + 8 * ob, NOUT == 2 ? ph : (uint32_t)(PAR ^ 1));
            if (lane_out) {
                const uint32_t ao = aO + ob * OUT_BYTES;
#pragma unroll
                for (int f = 0; f < TSLB_NF; ++f) {
                    sts(ao + f * (ROWS * COLS) * ES, o[f].x);
                    sts(ao + (f * (ROWS * COLS) + COLS) * ES, o[f].y);
                }
            }
            if (!TILE_FENCE_STORER) fence_async_smem();
            warp_arrive(sb + B_OFULL + 8 * ob, lane);
            if (xedge || xtail) {
                T *rp = Bbuf + ((long long)zt * L.plane + (long long)r0 * L.px);
                if (xtail) {
                    T *gp = rp + (col + TSLB_XOFF);
#pragma unroll
                    for (int f = 0; f < TSLB_NF; ++f) { gp[f * L.field] = o[f].x; gp[f * L.field + L.px] = o[f].y; }
                }
                if (xedge) {
                    T *gp = rp + gcol;
#pragma unroll
                    for (int f = 0; f < TSLB_NF; ++f) { gp[f * L.field] = o[f].x; gp[f * L.field + L.px] = o[f].y; }
                }
            }
        }
    };
    for (int i = 0; i < nplanes; i += 2) {
        plane(std::integral_constant<int, 0>(), i);
        if (i + 1 < nplanes) plane(std::integral_constant<int, 1>(), i + 1);
        ph ^= 1;
    }
}

// Launch geometry for tile geometry GEO.  *cost = estimated duration in units of one plane of a LARGE CTA (for the choice
// between the geometries), or a huge value if the lattice has fewer rows than one tile.
template <typename T, int GEO>
TileParams<T> make_tile(const tslb_ctx *c, dim3 *grid, double *cost_out)
{
    typedef TileDims<T, GEO> TDH;
    TileParams<T> p;
    p.L = c->L;
    for (int f = 0; f < 6; ++f) p.kind[f] = c->kind[f];
    p.beta = (T)(1.0 - c->omega);
    p.beta_z = c->beta_z_host ? (const T *)c->beta_z : nullptr;
    for (int a = 0; a < 3; ++a) p.g[a] = (T)c->g[a];
    const int gx = (c->nx + TDH::COLS - 1) / TDH::COLS;
    const int gy = (c->ny + TDH::ROWS - 1) / TDH::ROWS;
    // z chunks (one CTA per SM is resident): pick the chunk count whose number of waves x (chunk length + 2 halo planes +
    // ring fill) is smallest, among chunks of at most TILE_ZC_MAX planes.  Long marches let the CTAs of a wave drift apart
    // in z until the halo rows / columns that neighbouring tiles share have left L2 before their second reader arrives
    // (measured at 512^3 fp32: DRAM reads 7.09 / 6.62 / 6.13 GB per step for chunks of 128 / 64 / 32 planes, 5.4 GB
    // algorithmic; profiles/README.md).
    // (the ghost planes of a slab -- EXCHANGE faces -- are sources only: the march covers the owned planes)
    p.zbeg = c->kind[4] == TSLB_BC_EXCHANGE ? 1 : 0;
    p.zend = c->kind[5] == TSLB_BC_EXCHANGE ? c->nz - 1 : c->nz;
    const int nzs = p.zend - p.zbeg;
    const long long cols = (long long)gx * gy;
    int best = 1;
    double best_cost = 1e300;
    for (int k = 1; k <= nzs; ++k) {
        const int zc = (nzs + k - 1) / k;
        if (k > 1 && zc < 8) break;
        if (zc > TILE_ZC_MAX && (nzs + k) / (k + 1) >= 8) continue;
        const long long ctas = cols * ((nzs + zc - 1) / zc);
        const long long slots = (long long)c->sm_count * TDH::G::CTAS;
        const long long waves = (ctas + slots - 1) / slots;
        const double cost = (double)waves * (zc + 2 + 3);      // + ring fill latency of a fresh CTA, in plane units
        if (cost < best_cost) { best_cost = cost; best = k; }
    }
    // a plane of a small CTA (4 rows, two CTAs per SM) takes about TILE_SMALL_PLANE of a large one's (12 rows)
    if (cost_out) *cost_out = (c->ny < TDH::ROWS) ? 1e300 : best_cost * (GEO == 1 ? TILE_SMALL_PLANE : 1.0);
    int zc = (nzs + best - 1) / best;
    p.zchunk = zc;
    *grid = dim3(gx, gy, (nzs + zc - 1) / zc);
    // Fused boundary fill: possible when every open-face boundary node shares a tile and a z chunk with the interior node
    // x_F it copies (the store warp patches the output tile in shared memory), the row tail and the periodic ghost
    // columns -- stored from the main warps' registers, unpatched -- do not hold boundary values, and open axes are
    // long enough for x_F to be an interior node.
    auto open_k = [&](int f) {
        const int k = c->kind[f];
        return k == TSLB_BC_VELOCITY_INLET || k == TSLB_BC_OUTLET_ZERO_GRADIENT || k == TSLB_BC_OUTLET_PRESSURE;
    };
    bool any = false, ok = true;
    for (int f = 0; f < 6; ++f) any = any || open_k(f);
    const int n3[3] = {c->nx, c->ny, c->nz};
    for (int ax = 0; ax < 3; ++ax)
        if ((open_k(2 * ax) || open_k(2 * ax + 1)) && n3[ax] < 4) ok = false;
    if (c->kind[0] == TSLB_BC_PERIODIC) ok = false;                               // ghost-column images of boundary rows
    if (c->nx % (int)(16 / sizeof(T)) != 0) ok = false;                           // row tail stored from registers
    if (open_k(1) && (c->nx - 1) % TDH::COLS == 0) ok = false;            // x = nx-1 alone in the last tile column
    if (open_k(5) && p.zend - (p.zbeg + (int)(grid->z - 1) * zc) < 2) ok = false;   // z = nz-1 alone in the last chunk
    if (zc < 2) ok = false;
    if (c->kind[4] == TSLB_BC_BOUNCE_BACK || c->kind[5] == TSLB_BC_BOUNCE_BACK) ok = false;   // z-wall kernels: plain store warp only
    if (c->kind[0] == TSLB_BC_BOUNCE_BACK || c->kind[1] == TSLB_BC_BOUNCE_BACK) ok = false;   // x-wall kernels likewise
#ifdef TILE_NO_FUSE
    ok = false;
#endif
    p.fuse = (any && ok) ? 1 : 0;
    return p;
}

#ifndef TSLB_L2PROMO
#define TSLB_L2PROMO CU_TENSOR_MAP_L2_PROMOTION_L2_128B
#endif
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

bool tslb_tile_supported(const tslb_ctx *c, const char **why)
{
    // bounce-back walls are handled on the y faces, on the z faces, on both, or on the x faces alone (x walls together with
    // other walls: gather kernel); the x- and z-wall instantiations exist for the plain case only (no sponge layer)
    bool wall_ax[3] = {false, false, false};
    for (int f = 0; f < 6; ++f)
        if (c->kind[f] == TSLB_BC_BOUNCE_BACK) wall_ax[f >> 1] = true;
    if (wall_ax[0] && (wall_ax[1] || wall_ax[2])) {
        if (why) *why = "bounce-back walls on x faces together with walls on another axis";
        return false;
    }
    if ((wall_ax[2] || wall_ax[0]) && (c->beta_z_host || c->nz < 4 || c->ny < (c->dtype == TSLB_F64 ? TileDims<double>::ROWS : TileDims<float, 0>::ROWS))) {
        if (why) *why = "x or z walls together with a sponge layer, or fewer rows than one large tile";
        return false;
    }
    // every tile is full: the last tile of the y axis is shifted back, which needs at least one tile height of rows
    if (c->ny < (c->dtype == TSLB_F64 ? TileDims<double>::ROWS : TileDims<float, 1>::ROWS)) {
        if (why) *why = "fewer rows (ny) than one tile";
        return false;
    }
    if (c->ws && !c->tmap_ok) {
        if (why) *why = "TMA descriptors unavailable";
        return false;
    }
    if (why) *why = "";
    return true;
}

// TMA descriptors of the two moment buffers: 4-D tensor (x, y, z, field) of the padded SoA layout.
//   tm_main  box BXW x ROWS x 1 x 10: the tile rows of one source plane (with XPAD columns on each side)
//   tm_row   box BXW x 1 x 1 x 10:    one halo row
//   tm_store box COLS x ROWS x 1 x 10, tensor clipped at the last 16-byte boundary <= nx: the output tile (the kernel
//            stores the nx % 4 (fp64: nx % 2) columns beyond it and the ghost columns from registers)
// Out-of-bounds elements of a load are zero-filled: rows -1 / ny and planes -1 / nz beyond a wall or an open face.
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
    const bool f64 = c->dtype == TSLB_F64;
    const cuuint32_t bxw = f64 ? TileDims<double>::BXW : TileDims<float>::BXW;
    const cuuint32_t rows_g[2] = {(cuuint32_t)(f64 ? TileDims<double>::ROWS : TileDims<float, 0>::ROWS),
                                  (cuuint32_t)(f64 ? TileDims<double>::ROWS : TileDims<float, 1>::ROWS)};
    const cuuint32_t cols = f64 ? TileDims<double>::COLS : TileDims<float>::COLS;
    static_assert(TileDims<float, 0>::BXW == TileDims<float, 1>::BXW && TileDims<float, 0>::COLS == TileDims<float, 1>::COLS, "same tile width");
    const cuuint64_t strides[3] = {(cuuint64_t)L.px * es, (cuuint64_t)L.plane * es, (cuuint64_t)L.field * es};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUtensorMapDataType dt = f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    for (int g = 0; g < 2; ++g)
    for (int b = 0; b < 2; ++b) {
        const cuuint32_t rows = rows_g[g];
        const cuuint64_t dims_ld[4] = {(cuuint64_t)L.px, (cuuint64_t)L.ny, (cuuint64_t)L.nz, TSLB_NF};
        const cuuint64_t dims_st[4] = {(cuuint64_t)((L.nx & ~(int)(16 / es - 1)) + TSLB_XOFF), (cuuint64_t)L.ny, (cuuint64_t)L.nz, TSLB_NF};
        const cuuint32_t box_main[4] = {bxw, rows, 1, TSLB_NF}, box_row[4] = {bxw, 1, 1, TSLB_NF}, box_st[4] = {cols, rows, 1, TSLB_NF};
        CUresult r = ((EncodeTiledFn)fn)(&c->tm_main[g][b], dt, 4, c->buf[b], dims_ld, strides, box_main, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                         CU_TENSOR_MAP_SWIZZLE_NONE, TSLB_L2PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r == CUDA_SUCCESS)
            r = ((EncodeTiledFn)fn)(&c->tm_row[g][b], dt, 4, c->buf[b], dims_ld, strides, box_row, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                    CU_TENSOR_MAP_SWIZZLE_NONE, TSLB_L2PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r == CUDA_SUCCESS)
            r = ((EncodeTiledFn)fn)(&c->tm_store[g][b], dt, 4, c->buf[b], dims_st, strides, box_st, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                    CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    }
    e = cudaSuccess;
#define TSLB_SMEM_ATTR_Z(T, O)                                                                                                  \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_tile_kernel<T, 2, O, false, false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, TileDims<T, 0>::SMEM_BYTES); \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_tile_kernel<T, 3, O, false, false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, TileDims<T, 0>::SMEM_BYTES); \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_tile_kernel<T, 4, O, false, false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, TileDims<T, 0>::SMEM_BYTES)
    TSLB_SMEM_ATTR_Z(float, 3); TSLB_SMEM_ATTR_Z(float, 2); TSLB_SMEM_ATTR_Z(double, 3); TSLB_SMEM_ATTR_Z(double, 2);
#undef TSLB_SMEM_ATTR_Z
#define TSLB_SMEM_ATTR(T, W, O, G)                                                                                              \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_tile_kernel<T, W, O, false, false, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, TileDims<T, G>::SMEM_BYTES); \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_tile_kernel<T, W, O, true, false, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, TileDims<T, G>::SMEM_BYTES);  \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_tile_kernel<T, W, O, false, true, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, TileDims<T, G>::SMEM_BYTES);  \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_tile_kernel<T, W, O, true, true, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, TileDims<T, G>::SMEM_BYTES)
    TSLB_SMEM_ATTR(float, 0, 3, 0); TSLB_SMEM_ATTR(float, 1, 3, 0);
    TSLB_SMEM_ATTR(float, 0, 2, 0); TSLB_SMEM_ATTR(float, 1, 2, 0);
    TSLB_SMEM_ATTR(float, 0, 3, 1); TSLB_SMEM_ATTR(float, 1, 3, 1);
    TSLB_SMEM_ATTR(float, 0, 2, 1); TSLB_SMEM_ATTR(float, 1, 2, 1);
    TSLB_SMEM_ATTR(double, 0, 3, 0); TSLB_SMEM_ATTR(double, 1, 3, 0);
    TSLB_SMEM_ATTR(double, 0, 2, 0); TSLB_SMEM_ATTR(double, 1, 2, 0);
#undef TSLB_SMEM_ATTR
    if (e != cudaSuccess) return e;
    c->tmap_ok = 1;
    return cudaSuccess;
}

// Neighbour slabs (tslb_set_neighbor): load descriptors over the peer's two moment buffers (its own nz, same nx / ny / dtype).
cudaError_t tslb_tile_prepare_neighbor(tslb_ctx *c, int side)
{
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return e;
    if (!fn || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
    const Layout &L = c->L;
    const size_t es = tslb_elem(c);
    const bool f64 = c->dtype == TSLB_F64;
    const cuuint32_t bxw = f64 ? TileDims<double>::BXW : TileDims<float>::BXW;
    const cuuint32_t rows_g[2] = {(cuuint32_t)(f64 ? TileDims<double>::ROWS : TileDims<float, 0>::ROWS),
                                  (cuuint32_t)(f64 ? TileDims<double>::ROWS : TileDims<float, 1>::ROWS)};
    const long long pnz = c->nb_nz[side];
    const cuuint64_t strides[3] = {(cuuint64_t)L.px * es, (cuuint64_t)L.plane * es, (cuuint64_t)L.plane * pnz * es};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUtensorMapDataType dt = f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const cuuint64_t dims_ld[4] = {(cuuint64_t)L.px, (cuuint64_t)L.ny, (cuuint64_t)pnz, TSLB_NF};
    for (int g = 0; g < 2; ++g)
    for (int b = 0; b < 2; ++b) {
        const cuuint32_t box_main[4] = {bxw, rows_g[g], 1, TSLB_NF}, box_row[4] = {bxw, 1, 1, TSLB_NF};
        CUresult r = ((EncodeTiledFn)fn)(&c->nb_main[side][g][b], dt, 4, c->nb_buf[side][b], dims_ld, strides, box_main, estr,
                                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, TSLB_L2PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r == CUDA_SUCCESS)
            r = ((EncodeTiledFn)fn)(&c->nb_row[side][g][b], dt, 4, c->nb_buf[side][b], dims_ld, strides, box_row, estr,
                                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, TSLB_L2PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    }
    return cudaSuccess;
}

static NbParams make_nb(const tslb_ctx *c, int geo)
{
    NbParams nb;
    memset(&nb, 0, sizeof nb);
    for (int s = 0; s < 2; ++s) {
        if (!c->nb_on[s]) continue;
        // the peer alternates its buffers in lockstep with this context (include/tslb.h)
        const int b = (int)((c->nb_cur0[s] + (c->t - c->nb_t0[s])) & 1);
        nb.on[s] = 1;
        nb.main[s] = c->nb_main[s][geo][b];
        nb.row[s] = c->nb_row[s][geo][b];
        nb.z[s] = s == 0 ? c->nb_nz[s] - 2 : 1;
    }
    return nb;
}

template <typename T, int WALLY, int ORDER, int GEO>
static void launch_tile_geo(tslb_ctx *c, cudaStream_t st)
{
    dim3 grid;
    TileParams<T> p = make_tile<T, GEO>(c, &grid, nullptr);
    const int a = c->cur, b = 1 - c->cur;
    c->last_fused = p.fuse;
    FuseParams fp;
    fp.L = c->L;
    fp.tnext = c->t + 1;
    for (int f = 0; f < 6; ++f) { fp.kind[f] = c->kind[f]; fp.inlet[f] = c->inlet[f]; fp.rho_out[f] = c->rho_out[f]; }
    const NbParams nb = make_nb(c, GEO);
#define TSLB_TILE_LAUNCH(S, F)                                                                                                            \
    sweep_tile_kernel<T, WALLY, ORDER, S, F, GEO><<<grid, TileDims<T, GEO>::THREADS, TileDims<T, GEO>::SMEM_BYTES, st>>>(                    \
        c->tm_main[GEO][a], c->tm_row[GEO][a], c->tm_store[GEO][b], (T *)c->buf[b], p, fp, nb)
    if (p.beta_z) { if (p.fuse) TSLB_TILE_LAUNCH(true, true); else TSLB_TILE_LAUNCH(true, false); }
    else { if (p.fuse) TSLB_TILE_LAUNCH(false, true); else TSLB_TILE_LAUNCH(false, false); }
#undef TSLB_TILE_LAUNCH
}

// fp32 has two tile geometries: the one with the smaller estimated duration is taken (a lattice that cannot fill 148
// large CTAs, or whose width / height the large tile pads badly, runs on the small one)
// x or z walls (WALLV = 2, 3, 4): the large geometry, plain store warp, no sponge (tslb_tile_supported / make_tile see to it)
template <typename T, int ORDER, int WALLV>
static void launch_tile_zwall(tslb_ctx *c, cudaStream_t st)
{
    dim3 grid;
    TileParams<T> p = make_tile<T, 0>(c, &grid, nullptr);
    const int a = c->cur, b = 1 - c->cur;
    c->last_fused = 0;
    FuseParams fp;
    fp.L = c->L;
    fp.tnext = c->t + 1;
    for (int f = 0; f < 6; ++f) { fp.kind[f] = c->kind[f]; fp.inlet[f] = c->inlet[f]; fp.rho_out[f] = c->rho_out[f]; }
    const NbParams nb = make_nb(c, 0);
    sweep_tile_kernel<T, WALLV, ORDER, false, false, 0><<<grid, TileDims<T, 0>::THREADS, TileDims<T, 0>::SMEM_BYTES, st>>>(
        c->tm_main[0][a], c->tm_row[0][a], c->tm_store[0][b], (T *)c->buf[b], p, fp, nb);
}

template <typename T, int WALLY, int ORDER>
static void launch_tile(tslb_ctx *c, cudaStream_t st)
{
    if (sizeof(T) == 8) { launch_tile_geo<T, WALLY, ORDER, 0>(c, st); return; }
    dim3 g0, g1;
    double c0 = 0, c1 = 0;
    make_tile<T, 0>(c, &g0, &c0);
    make_tile<T, 1>(c, &g1, &c1);
    int geo = c1 < c0 ? 1 : 0;
    if (TILE_FORCE_GEOM >= 0 && (TILE_FORCE_GEOM == 1 ? c1 : c0) < 1e299) geo = TILE_FORCE_GEOM;
    if (geo == 1) launch_tile_geo<T, WALLY, ORDER, 1>(c, st);
    else launch_tile_geo<T, WALLY, ORDER, 0>(c, st);
}

cudaError_t tslb_launch_tile(tslb_ctx *c, cudaStream_t st)
{
    const bool wally = c->kind[2] == TSLB_BC_BOUNCE_BACK || c->kind[3] == TSLB_BC_BOUNCE_BACK;
    const bool wallz = c->kind[4] == TSLB_BC_BOUNCE_BACK || c->kind[5] == TSLB_BC_BOUNCE_BACK;
    const bool wallx = c->kind[0] == TSLB_BC_BOUNCE_BACK || c->kind[1] == TSLB_BC_BOUNCE_BACK;
    const bool o3 = c->order >= 3;
    if (wallx) {
        if (c->dtype == TSLB_F32) { if (o3) launch_tile_zwall<float, 3, 4>(c, st); else launch_tile_zwall<float, 2, 4>(c, st); }
        else { if (o3) launch_tile_zwall<double, 3, 4>(c, st); else launch_tile_zwall<double, 2, 4>(c, st); }
    } else if (c->dtype == TSLB_F32) {
        if (wallz && wally) { if (o3) launch_tile_zwall<float, 3, 3>(c, st); else launch_tile_zwall<float, 2, 3>(c, st); }
        else if (wallz) { if (o3) launch_tile_zwall<float, 3, 2>(c, st); else launch_tile_zwall<float, 2, 2>(c, st); }
        else if (wally) { if (o3) launch_tile<float, 1, 3>(c, st); else launch_tile<float, 1, 2>(c, st); }
        else { if (o3) launch_tile<float, 0, 3>(c, st); else launch_tile<float, 0, 2>(c, st); }
    } else {
        if (wallz && wally) { if (o3) launch_tile_zwall<double, 3, 3>(c, st); else launch_tile_zwall<double, 2, 3>(c, st); }
        else if (wallz) { if (o3) launch_tile_zwall<double, 3, 2>(c, st); else launch_tile_zwall<double, 2, 2>(c, st); }
        else if (wally) { if (o3) launch_tile<double, 1, 3>(c, st); else launch_tile<double, 1, 2>(c, st); }
        else { if (o3) launch_tile<double, 0, 3>(c, st); else launch_tile<double, 0, 2>(c, st); }
    }
    c->launches++;
    return cudaGetLastError();
}

// kernels_basic.cu -- the per-direction "gather" sweep (covers every boundary set and lattice shape),
// the boundary-node fill, the ghost-column (halo) refresh, layout import/export and the diagnostics reduction.  sm_100a.
//
// Arithmetic follows PAPER.md:154 (Eq. 18) with the readings of DESIGN.md; contractions are reduced by
// hand.  Internal storage is the SHIFTED form: field 0 holds drho = rho - 1
// and populations are carried as f_i - w_i, so that fp32 rounding is relative to the perturbation and
// not to 1.  The w_i-part is added back in closed form:
// sum_i w_i = 1, sum_i w_i c_i = 0, sum_i w_i c_i c_i = I/3.
#include "tslb_internal.h"

namespace {

template <typename T>
struct Site {
    T dr, ux, uy, uz, pxx, pyy, pzz, pxy, pxz, pyz;
};

template <typename T>
__device__ __forceinline__ Site<T> load_site(const T *__restrict__ A, long long N, long long i)
{
    Site<T> s;
    s.dr = __ldg(A + i);
    s.ux = __ldg(A + N + i);
    s.uy = __ldg(A + 2 * N + i);
    s.uz = __ldg(A + 3 * N + i);
    s.pxx = __ldg(A + 4 * N + i);
    s.pyy = __ldg(A + 5 * N + i);
    s.pzz = __ldg(A + 6 * N + i);
    s.pxy = __ldg(A + 7 * N + i);
    s.pxz = __ldg(A + 8 * N + i);
    s.pyz = __ldg(A + 9 * N + i);
    return s;
}

// f*_c(M) - w_c - (base of the linear momentum term) for direction (sgn*cx, sgn*cy, sgn*cz); cx,cy,cz are
// compile-time after unrolling.
//   f* = w [ rho (1 + 3 c.(u+g) + 4.5((c.u)^2 - |u|^2/3) + 4.5((c.u)^3 - (c.u)|u|^2))          Eq. 14
//          + beta (4.5 (cPc - trP/3) + 4.5 (3 cPc c.u - trP c.u - 2 cPu)) ]                      Eq. 17
// Terms odd in c change sign with sgn (bounce-back evaluates the opposite direction at the own node).
// INCREMENT FORM: the linear term 3 w c.(rho (u+g)) of the source node is written as
// 3 w c.u(x) + 3 w lin, with u(x) the velocity of the TARGET node; sum_i c_i (3 w_i c_i.u(x)) = 216 u(x) exactly, so
// the base never passes through rounded arithmetic and only `lin` (a difference of neighbouring velocities plus
// small terms) does.  The caller passes lin = c.(u_src - u_x) + c.(g + drho_src (u_src + g)).
template <typename T>
__device__ __forceinline__ T fstar_incr(const Site<T> &m, int cx, int cy, int cz, T sgn, T w, T beta, T lin, T o3)
{
    const T fx = (T)cx, fy = (T)cy, fz = (T)cz;
    const T rho = (T)1 + m.dr;
    const T cu = fx * m.ux + fy * m.uy + fz * m.uz;
    const T uu = m.ux * m.ux + m.uy * m.uy + m.uz * m.uz;
    const T trP = m.pxx + m.pyy + m.pzz;
    const T cPx = fx * m.pxx + fy * m.pxy + fz * m.pxz;  // (c.P)_x
    const T cPy = fx * m.pxy + fy * m.pyy + fz * m.pyz;
    const T cPz = fx * m.pxz + fy * m.pyz + fz * m.pzz;
    const T cPc = cPx * fx + cPy * fy + cPz * fz;
    const T cPu = cPx * m.ux + cPy * m.uy + cPz * m.uz;
    const T even_eq = (T)4.5 * cu * cu - (T)1.5 * uu;
    const T odd_eq = (T)4.5 * cu * (cu * cu - uu);
    const T even_ne = (T)4.5 * cPc - (T)1.5 * trP;
    const T odd_ne = (T)4.5 * ((T)3 * cPc * cu - trP * cu - (T)2 * cPu);
    // o3 = 0 drops the third-order Hermite terms: the second-order TSLB of Eq. 8
    return w * (m.dr + (T)3 * lin + rho * (even_eq + sgn * o3 * odd_eq) + beta * (even_ne + sgn * o3 * odd_ne));
}

__device__ __forceinline__ bool is_open_kind(int k)
{
    return k == TSLB_BC_VELOCITY_INLET || k == TSLB_BC_OUTLET_ZERO_GRADIENT || k == TSLB_BC_OUTLET_PRESSURE;
}

template <typename P>
__device__ __forceinline__ bool on_open_face(const P &p, int x, int y, int z)
{
    return (x == 0 && is_open_kind(p.kind[0])) || (x == p.L.nx - 1 && is_open_kind(p.kind[1])) ||
           (y == 0 && is_open_kind(p.kind[2])) || (y == p.L.ny - 1 && is_open_kind(p.kind[3])) ||
           (z == 0 && is_open_kind(p.kind[4])) || (z == p.L.nz - 1 && is_open_kind(p.kind[5]));
}

// ---------------------------------------------------------------------------------------------
// Gather sweep: one thread per node, 27 upstream nodes read straight from global memory (L1/L2
// provide the reuse).  SURVEY.md 8(a) rows a1-a8 in one kernel.  Does its own periodic wrap (never
// reads the ghost layers), so it needs no halo refresh.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128) sweep_gather_kernel(const T *__restrict__ A, T *__restrict__ B,
                                                            SweepParams<T> p)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    if (x >= p.L.nx || y >= p.L.ny) return;
    for (int z = blockIdx.z; z < p.L.nz; z += gridDim.z) {
    const long long N = p.L.field;
    const long long ip = lay_idx(p.L, x, y, z);
    const Site<T> own = load_site(A, N, ip);

    if (on_open_face(p, x, y, z)) {  // boundary nodes are not advanced: M_{t+1}(x_B) := M_t(x_B)
        B[ip] = own.dr;
        B[N + ip] = own.ux; B[2 * N + ip] = own.uy; B[3 * N + ip] = own.uz;
        B[4 * N + ip] = own.pxx; B[5 * N + ip] = own.pyy; B[6 * N + ip] = own.pzz;
        B[7 * N + ip] = own.pxy; B[8 * N + ip] = own.pxz; B[9 * N + ip] = own.pyz;
        continue;
    }

    // upstream coordinate x - c for c = -1, 0, +1 (index c+1), with periodic wrap; bounce flags
    int sx[3], sy[3], sz[3];
    bool bx[3], by[3], bz[3];
    {
        const int n[3] = {p.L.nx, p.L.ny, p.L.nz};
        const int q[3] = {x, y, z};
        int *s[3] = {sx, sy, sz};
        bool *b[3] = {bx, by, bz};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            s[a][1] = q[a]; b[a][1] = false;
            // c = +1 pulls from q-1
            b[a][2] = false;
            if (q[a] > 0) s[a][2] = q[a] - 1;
            else if (p.kind[2 * a] == TSLB_BC_PERIODIC) s[a][2] = n[a] - 1;
            else { s[a][2] = q[a]; b[a][2] = (p.kind[2 * a] == TSLB_BC_BOUNCE_BACK); }
            // c = -1 pulls from q+1
            b[a][0] = false;
            if (q[a] < n[a] - 1) s[a][0] = q[a] + 1;
            else if (p.kind[2 * a + 1] == TSLB_BC_PERIODIC) s[a][0] = 0;
            else { s[a][0] = q[a]; b[a][0] = (p.kind[2 * a + 1] == TSLB_BC_BOUNCE_BACK); }
        }
    }

    // 1 - omega of the source node: uniform, or per plane inside a sponge layer (Eq. 26)
    T bsrc[3] = {p.beta, p.beta, p.beta};
    if (p.beta_z) {
#pragma unroll
        for (int k = 0; k < 3; ++k) bsrc[k] = p.beta_z[sz[k]];
    }
    T dR = 0, Jx = 0, Jy = 0, Jz = 0, Sxx = 0, Syy = 0, Szz = 0, Sxy = 0, Sxz = 0, Syz = 0;
#pragma unroll
    for (int cz = -1; cz <= 1; ++cz)
#pragma unroll
        for (int cy = -1; cy <= 1; ++cy)
#pragma unroll
            for (int cx = -1; cx <= 1; ++cx) {
                const bool bounced = bx[cx + 1] | by[cy + 1] | bz[cz + 1];
                // 216 w_i = 64, 16, 4, 1: exact powers of two, so no rounded weight multiplies the data
                const T w = (T)((cx ? 1 : 4) * (cy ? 1 : 4) * (cz ? 1 : 4));
                T f;
                if (cx == 0 && cy == 0 && cz == 0) {
                    f = fstar_incr(own, 0, 0, 0, (T)1, w, bsrc[1], (T)0, p.o3);
                } else {
                    // halfway bounce-back: f_i(x,t+1) = f*_ibar(x,t) from the node's own moments
                    const long long is = bounced ? ip : lay_idx(p.L, sx[cx + 1], sy[cy + 1], sz[cz + 1]);
                    const Site<T> m = load_site(A, N, is);
                    // small part of rho (u + g): g + drho (u + g), per component
                    const T smx = fma(m.dr, m.ux + p.g[0], p.g[0]);
                    const T smy = fma(m.dr, m.uy + p.g[1], p.g[1]);
                    const T smz = fma(m.dr, m.uz + p.g[2], p.g[2]);
                    T lin;
                    if (bounced)   // reversed direction at the own node: -c.psi(x) = c.u(x) + [-(2 c.u(x) + c.small(x))]
                        lin = -((T)cx * ((T)2 * own.ux + smx) + (T)cy * ((T)2 * own.uy + smy) + (T)cz * ((T)2 * own.uz + smz));
                    else
                        lin = (T)cx * ((m.ux - own.ux) + smx) + (T)cy * ((m.uy - own.uy) + smy) + (T)cz * ((m.uz - own.uz) + smz);
                    f = fstar_incr(m, cx, cy, cz, bounced ? (T)-1 : (T)1, w, bounced ? bsrc[1] : bsrc[cz + 1], lin, p.o3);
                }
                dR += f;                                  // arrival direction c_i in every sum
                if (cx) Jx += (T)cx * f;
                if (cy) Jy += (T)cy * f;
                if (cz) Jz += (T)cz * f;
                if (cx) Sxx += f;
                if (cy) Syy += f;
                if (cz) Szz += f;
                if (cx && cy) Sxy += (T)(cx * cy) * f;
                if (cx && cz) Sxz += (T)(cx * cz) * f;
                if (cy && cz) Syz += (T)(cy * cz) * f;
            }
    // All sums are 216-scaled and J lacks its base 216 u(x).  rho' = 1 + dR/216; u' = (216 u + J) / (216 rho')
    // = u + (J - u dR) / (216 + dR); Pi' = S - rho'(I/3 + u'u') with S_aa = dS_aa + 1/3 (Eq. 12).  x/216 is formed as
    // x*hi + x*lo (unbiased); a rounded 1/216 or rounded w_i would be a systematic per-step gain that compounds over
    // thousands of steps.
    const T hi = (T)(1.0 / 216.0);
    const T lo = (T)(1.0 / 216.0 - (double)hi);
    const T dr = fma(dR, lo, dR * hi);
    const T rho = (T)1 + dr;
    const T inv = (T)1 / ((T)216 + dR);
    const T ux = fma(fma(-own.ux, dR, Jx), inv, own.ux);
    const T uy = fma(fma(-own.uy, dR, Jy), inv, own.uy);
    const T uz = fma(fma(-own.uz, dR, Jz), inv, own.uz);
    const T iso = (T)(1.0 / 3.0) * dr;
    B[ip] = dr;
    B[N + ip] = ux; B[2 * N + ip] = uy; B[3 * N + ip] = uz;
    B[4 * N + ip] = fma(Sxx, lo, Sxx * hi) - iso - rho * ux * ux;
    B[5 * N + ip] = fma(Syy, lo, Syy * hi) - iso - rho * uy * uy;
    B[6 * N + ip] = fma(Szz, lo, Szz * hi) - iso - rho * uz * uz;
    B[7 * N + ip] = fma(Sxy, lo, Sxy * hi) - rho * ux * uy;
    B[8 * N + ip] = fma(Sxz, lo, Sxz * hi) - rho * ux * uz;
    B[9 * N + ip] = fma(Syz, lo, Syz * hi) - rho * uy * uz;
    }   // z
}

// ---------------------------------------------------------------------------------------------
// Boundary-node fill at time t (PAPER.md:181-196 Eq. 22-23, :202, :258; readings A13-A16):
// every node on an INLET/OUTLET face takes all 10 moments of x_F (its coordinates on open axes
// clamped to [1, n-2]); on an inlet face the velocity is then imposed (with seeded noise).
// One thread per (face, in-plane position); a node on several open faces is handled by the
// lowest-index one.
// ---------------------------------------------------------------------------------------------

template <typename T>
__global__ void fill_boundary_kernel(T *__restrict__ M, FillParams p)
{
    const int f = blockIdx.y;
    if (!is_open_kind(p.kind[f])) return;
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int n[3] = {p.L.nx, p.L.ny, p.L.nz};
    const int ax = f >> 1;
    const int a = (ax == 0) ? 1 : 0;
    const int b = (ax == 2) ? 1 : 2;
    if (j >= n[a] * n[b]) return;
    int q[3];
    q[ax] = (f & 1) ? n[ax] - 1 : 0;
    q[a] = j % n[a];
    q[b] = j / n[a];
    // lowest-index open face containing this node does the work
    for (int f2 = 0; f2 < f; ++f2) {
        const int ax2 = f2 >> 1;
        if (is_open_kind(p.kind[f2]) && q[ax2] == ((f2 & 1) ? n[ax2] - 1 : 0)) return;
    }
    int r[3] = {q[0], q[1], q[2]};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        if (r[d] == 0 && is_open_kind(p.kind[2 * d])) r[d] = 1;
        if (r[d] == n[d] - 1 && is_open_kind(p.kind[2 * d + 1])) r[d] = n[d] - 2;
    }
    const long long N = p.L.field;
    const long long ib = lay_idx(p.L, q[0], q[1], q[2]);
    const long long iF = lay_idx(p.L, r[0], r[1], r[2]);
#pragma unroll
    for (int k = 0; k < TSLB_NF; ++k) M[k * N + ib] = M[k * N + iF];
    for (int f2 = 0; f2 < 6; ++f2) {     // imposed density (field 0 holds rho - 1): lowest pressure face that holds the node
        if (p.kind[f2] != TSLB_BC_OUTLET_PRESSURE) continue;
        const int ax2 = f2 >> 1;
        if (q[ax2] != ((f2 & 1) ? n[ax2] - 1 : 0)) continue;
        M[ib] = (T)(p.rho_out[f2] - 1.0);
        break;
    }
    for (int f2 = 0; f2 < 6; ++f2) {
        if (p.kind[f2] != TSLB_BC_VELOCITY_INLET) continue;
        const int ax2 = f2 >> 1;
        if (q[ax2] != ((f2 & 1) ? n[ax2] - 1 : 0)) continue;
        const int a2 = (ax2 == 0) ? 1 : 0, b2 = (ax2 == 2) ? 1 : 2;
        const size_t pl = (size_t)n[a2] * n[b2];
        const size_t jj = (size_t)q[b2] * n[a2] + q[a2];
        const double xi = tslb_inlet_xi(p.inlet[f2], p.L, q[0], q[1], q[2], p.t);
#pragma unroll
        for (int k = 0; k < 3; ++k) M[(1 + k) * N + ib] = tslb_inlet_u<T>(p.inlet[f2], pl, jj, k, xi);
        break;
    }
}

// ---------------------------------------------------------------------------------------------
// Slab decomposition along z (include/tslb.h, tslb_export_face / tslb_import_face): plane z of the internal buffer <-> a dense
// array [10][ny][nx], values unchanged (field 0 stays rho - 1).  The import also writes the ghost columns x = -1 and x = nx of
// the plane (periodic image, else the clamped node: only has to be finite), so that no halo launch is needed after it.
// 40 B/node of a plane each way: 10.5 MB for 512^2 fp32, a few microseconds at HBM speed.
// ---------------------------------------------------------------------------------------------
template <typename T, int DIR>
__global__ void __launch_bounds__(128) face_kernel(T *__restrict__ M, T *__restrict__ dense, Layout L, int z, int xper)
{
    // one CTA per row (y = blockIdx.x) of one field (blockIdx.y): coalesced along x, no index division
    const int y = blockIdx.x, f = blockIdx.y;
    T *__restrict__ rm = M + f * L.field + lay_idx(L, 0, y, z);
    T *__restrict__ rd = dense + ((long long)f * L.ny + y) * L.nx;
    for (int x = threadIdx.x; x < L.nx; x += blockDim.x) {
        if (DIR > 0) rm[x] = rd[x];
        else rd[x] = rm[x];
    }
    if (DIR > 0 && threadIdx.x < 2) {           // ghost columns x = -1 and x = nx
        const bool hi = threadIdx.x == 1;
        rm[hi ? L.nx : -1] = rd[hi ? (xper ? 0 : L.nx - 1) : (xper ? L.nx - 1 : 0)];
    }
}

// ---------------------------------------------------------------------------------------------
// Ghost-column refresh: the cells x = -1 and x = nx of every row take the 10 moments of the
// node obtained by wrapping x on a periodic axis (clamping it otherwise).  The TMA-staged sweep reads its x neighbours
// through these columns (a TMA row is contiguous and cannot wrap); it keeps them current itself, so this kernel runs
// only after set_moments, a boundary change, a gather step, or a fill next to a periodic x axis.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void halo_kernel(T *__restrict__ M, FillParams p)
{
    const Layout &L = p.L;
    const long long tot = 2LL * L.ny * L.nz;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < tot; i += stride) {
        const long long j = i >> 1;
        const int y = (int)(j % L.ny), z = (int)(j / L.ny);
        const bool hi = i & 1;
        const int x = hi ? L.nx : -1;
        const int xs = hi ? (p.kind[1] == TSLB_BC_PERIODIC ? 0 : L.nx - 1) : (p.kind[0] == TSLB_BC_PERIODIC ? L.nx - 1 : 0);
        const long long ig = lay_idx(L, x, y, z), is = lay_idx(L, xs, y, z);
#pragma unroll
        for (int k = 0; k < TSLB_NF; ++k) M[k * L.field + ig] = M[k * L.field + is];
    }
}

// ---------------------------------------------------------------------------------------------
// API layout [10][nz][ny][nx] <-> internal padded layout (field 0: rho <-> rho - 1; exact for 0.5 <= rho <= 2)
// ---------------------------------------------------------------------------------------------
// SHIFT = 1: field 0 is rho on the API side (tslb_set/get_moments); SHIFT = 0: field 0 stays rho - 1 (the raw checkpoint of
// tslb_export_state / tslb_import_state, bit-for-bit the internal state)
template <typename T, int DIR, int SHIFT>
__global__ void convert_kernel(const T *__restrict__ src, T *__restrict__ dst, Layout L)
{
    const long long N = (long long)L.nx * L.ny * L.nz;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < TSLB_NF * N; i += stride) {
        const int k = (int)(i / N);
        const long long s = i - k * N;
        const int x = (int)(s % L.nx);
        const long long r = s / L.nx;
        const int y = (int)(r % L.ny), z = (int)(r / L.ny);
        const long long j = k * L.field + lay_idx(L, x, y, z);
        if (DIR > 0) { T v = src[i]; if (SHIFT && k == 0) v -= (T)1; dst[j] = v; }
        else { T v = src[j]; if (SHIFT && k == 0) v += (T)1; dst[i] = v; }
    }
}

// ---------------------------------------------------------------------------------------------
// Diagnostics: fp64 accumulation, warp shuffles, fixed-order final pass.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <typename T>
__global__ void __launch_bounds__(TSLB_DIAG_THREADS) diag_partial_kernel(const T *__restrict__ A, FillParams p,
                                                                          double *__restrict__ partial)
{
    // one warp per lattice row (y, z), lanes along x: coalesced, one division per row; the row -> warp and x -> lane
    // assignment is fixed, so the sums are bitwise reproducible
    const long long N = p.L.field;
    const int nrows = p.L.ny * p.L.nz;
    const int wpb = blockDim.x >> 5;
    const int lane_ = threadIdx.x & 31;
    const bool open_x0 = is_open_kind(p.kind[0]), open_x1 = is_open_kind(p.kind[1]);
    double acc[5] = {0, 0, 0, 0, 0};
    for (int row = blockIdx.x * wpb + (threadIdx.x >> 5); row < nrows; row += gridDim.x * wpb) {
        const int y = row % p.L.ny, z = row / p.L.ny;
        if ((y == 0 && is_open_kind(p.kind[2])) || (y == p.L.ny - 1 && is_open_kind(p.kind[3])) ||
            (z == 0 && (is_open_kind(p.kind[4]) || p.kind[4] == TSLB_BC_EXCHANGE)) ||      // ghost planes of a slab belong to
            (z == p.L.nz - 1 && (is_open_kind(p.kind[5]) || p.kind[5] == TSLB_BC_EXCHANGE))) continue;   // the neighbouring rank
        const T *r = A + lay_idx(p.L, 0, y, z);
        const int x0 = open_x0 ? 1 : 0, x1 = open_x1 ? p.L.nx - 1 : p.L.nx;
        for (int x = x0 + lane_; x < x1; x += 32) {
            const double rho = 1.0 + (double)r[x];
            const double ux = r[N + x], uy = r[2 * N + x], uz = r[3 * N + x];
            acc[0] += rho; acc[1] += rho * ux; acc[2] += rho * uy; acc[3] += rho * uz;
            acc[4] += 0.5 * rho * (ux * ux + uy * uy + uz * uz);
        }
    }
    __shared__ double sh[5][TSLB_DIAG_THREADS / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const double v = warp_sum(acc[k]);
        if (lane == 0) sh[k][wid] = v;
    }
    __syncthreads();
    if (threadIdx.x < 5) {
        double v = 0;
        for (int w = 0; w < TSLB_DIAG_THREADS / 32; ++w) v += sh[threadIdx.x][w];
        partial[threadIdx.x * gridDim.x + blockIdx.x] = v;
    }
}

__global__ void diag_final_kernel(const double *__restrict__ partial, int nblocks, double *__restrict__ out5)
{
    // one warp per quantity; lane-strided partial sums in a fixed order, then a shuffle tree
    const int k = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double v = 0;
    for (int b = lane; b < nblocks; b += 32) v += partial[k * nblocks + b];
    v = warp_sum(v);
    if (lane == 0) out5[k] = v;
}

// ---------------------------------------------------------------------------------------------
// Plane statistics (PAPER.md:236 Eq. 24, :242 Eq. 25): raw sums of 1, u, uu, uuu over every plane
// of constant coordinate along `axis`.  Grid (n_axis, PARTS): each CTA reduces a share of one plane in fp64 (warp shuffles,
// then a fixed-order pass over the warps), writes 13 partials; stats_final_kernel adds the PARTS partials of each plane
// in a fixed order to the caller's running sums.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) stats_partial_kernel(const T *__restrict__ A, Layout L, int axis, double *__restrict__ partial,
                                                            int zlo, int zhi)
{
    // [zlo, zhi): the planes that count -- all of them, except the ghost planes of a slab (EXCHANGE faces), which belong to the
    // neighbouring rank and may hold anything: they add nothing to the planes of axis 0 / 1 and give zero rows on axis 2
    const int j = blockIdx.x, part = blockIdx.y, nparts = gridDim.y;
    const int n[3] = {L.nx, L.ny, L.nz};
    const int a = (axis == 0) ? 1 : 0;              // fastest in-plane axis
    const int b = (axis == 2) ? 1 : 2;
    const long long cnt = (long long)n[a] * n[b];
    double acc[TSLB_STAT_ROWS];
#pragma unroll
    for (int k = 0; k < TSLB_STAT_ROWS; ++k) acc[k] = 0.0;
    for (long long i = (long long)part * blockDim.x + threadIdx.x; i < cnt; i += (long long)nparts * blockDim.x) {
        int q[3];
        q[axis] = j; q[a] = (int)(i % n[a]); q[b] = (int)(i / n[a]);
        if (q[2] < zlo || q[2] >= zhi) continue;
        const long long idx = lay_idx(L, q[0], q[1], q[2]);
        const double ux = A[L.field + idx], uy = A[2 * L.field + idx], uz = A[3 * L.field + idx];
        acc[0] += 1.0;
        acc[1] += ux; acc[2] += uy; acc[3] += uz;
        acc[4] += ux * ux; acc[5] += uy * uy; acc[6] += uz * uz;
        acc[7] += ux * uy; acc[8] += ux * uz; acc[9] += uy * uz;
        acc[10] += ux * ux * ux; acc[11] += uy * uy * uy; acc[12] += uz * uz * uz;
    }
    __shared__ double sh[TSLB_STAT_ROWS][8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < TSLB_STAT_ROWS; ++k) {
        const double v = warp_sum(acc[k]);
        if (lane == 0) sh[k][wid] = v;
    }
    __syncthreads();
    if (threadIdx.x < TSLB_STAT_ROWS) {
        double v = 0;
        for (int w = 0; w < 8; ++w) v += sh[threadIdx.x][w];
        partial[((long long)threadIdx.x * gridDim.x + j) * nparts + part] = v;
    }
}

__global__ void stats_final_kernel(const double *__restrict__ partial, int n_axis, int nparts, double *__restrict__ sums)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;     // over 13 * n_axis
    if (i >= TSLB_STAT_ROWS * n_axis) return;
    double v = 0;
    for (int p = 0; p < nparts; ++p) v += partial[(long long)i * nparts + p];
    sums[i] += v;
}

// ---------------------------------------------------------------------------------------------
// (r, z)-bin statistics of a round jet along z (Fig. 7-8; reading A27 in DESIGN.md): a node of plane z
// at distance r = sqrt(dx^2 + dy^2) from the axis (xc, yc) belongs to ring k = floor(r / dr) if k < nr; per plane and
// ring the sums of 1 | u_z | u_r | u_t | u_z^2 | u_r^2 | u_t^2 | u_z u_r are ADDED to sums[8][nz][nr].
// The ring index is an integer decided by floating point: it is taken in fp64 with the oracle's operation order and no
// fused multiply-add (sqrt and the division are correctly rounded on both sides), so both sides bin identically.
// One CTA per (plane, slab of rows): ring sums in shared memory (fp64 atomics), then one global atomic per ring and row
// -- the order of the additions is not fixed, so repeated runs agree to rounding (~1e-16 relative), not bitwise.
// ---------------------------------------------------------------------------------------------
#define TSLB_RSTAT_ROWS 8
#define TSLB_RSTAT_MAXBINS 512
template <typename T>
__global__ void __launch_bounds__(256) radial_stats_kernel(const T *__restrict__ A, Layout L, double xc, double yc, double dr, int nr,
                                                           double *__restrict__ sums)
{
    __shared__ double sh[TSLB_RSTAT_ROWS][TSLB_RSTAT_MAXBINS];
    const int z = blockIdx.x;
    for (int i = threadIdx.x; i < TSLB_RSTAT_ROWS * nr; i += blockDim.x) sh[i / nr][i % nr] = 0.0;
    __syncthreads();
    const int rows_per = (L.ny + gridDim.y - 1) / gridDim.y;
    const int y0 = blockIdx.y * rows_per, y1 = min(y0 + rows_per, L.ny);
    for (int y = y0 + (threadIdx.x >> 5); y < y1; y += blockDim.x >> 5) {
        const double dy = (double)y - yc;
        const double dy2 = __dmul_rn(dy, dy);
        for (int x = threadIdx.x & 31; x < L.nx; x += 32) {
            const double dx = (double)x - xc;
            const double r = sqrt(__dadd_rn(__dmul_rn(dx, dx), dy2));
            const double kf = floor(r / dr);
            if (!(kf < (double)nr)) continue;
            const int k = (int)kf;
            const long long idx = lay_idx(L, x, y, z);
            const double ux = A[L.field + idx], uy = A[2 * L.field + idx], uz = A[3 * L.field + idx];
            double ur = 0.0, ut = 0.0;
            if (r > 0.0) { ur = (ux * dx + uy * dy) / r; ut = (uy * dx - ux * dy) / r; }
            atomicAdd(&sh[0][k], 1.0);
            atomicAdd(&sh[1][k], uz); atomicAdd(&sh[2][k], ur); atomicAdd(&sh[3][k], ut);
            atomicAdd(&sh[4][k], uz * uz); atomicAdd(&sh[5][k], ur * ur); atomicAdd(&sh[6][k], ut * ut);
            atomicAdd(&sh[7][k], uz * ur);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < TSLB_RSTAT_ROWS * nr; i += blockDim.x) {
        const int row = i / nr, k = i % nr;
        const double v = sh[row][k];
        if (v != 0.0) atomicAdd(&sums[((long long)row * L.nz + z) * nr + k], v);
    }
}

template <typename T>
SweepParams<T> make_params(const tslb_ctx *c)
{
    SweepParams<T> p;
    p.L = c->L;
    for (int f = 0; f < 6; ++f) p.kind[f] = c->kind[f];
    p.beta = (T)(1.0 - c->omega);
    for (int a = 0; a < 3; ++a) p.g[a] = (T)c->g[a];
    p.o3 = c->order >= 3 ? (T)1 : (T)0;
    p.beta_z = c->beta_z_host ? (const T *)c->beta_z : nullptr;
    return p;
}

FillParams make_fill(const tslb_ctx *c)
{
    FillParams p;
    p.L = c->L;
    for (int f = 0; f < 6; ++f) { p.kind[f] = c->kind[f]; p.inlet[f] = c->inlet[f]; p.rho_out[f] = c->rho_out[f]; }
    p.t = c->t;
    return p;
}

}  // namespace

cudaError_t tslb_launch_gather(tslb_ctx *c, cudaStream_t st)
{
    dim3 block(64, 2, 1);
    dim3 grid((c->nx + block.x - 1) / block.x, (c->ny + block.y - 1) / block.y, c->nz < 65535 ? c->nz : 65535);
    if (c->dtype == TSLB_F32)
        sweep_gather_kernel<float><<<grid, block, 0, st>>>((const float *)c->buf[c->cur], (float *)c->buf[1 - c->cur],
                                                          make_params<float>(c));
    else
        sweep_gather_kernel<double><<<grid, block, 0, st>>>((const double *)c->buf[c->cur],
                                                           (double *)c->buf[1 - c->cur], make_params<double>(c));
    c->launches++;
    return cudaGetLastError();
}

static bool is_open_kind_host(int k)
{
    return k == TSLB_BC_VELOCITY_INLET || k == TSLB_BC_OUTLET_ZERO_GRADIENT || k == TSLB_BC_OUTLET_PRESSURE;
}

static bool any_open(const tslb_ctx *c)
{
    for (int f = 0; f < 6; ++f)
        if (is_open_kind_host(c->kind[f])) return true;
    return false;
}

cudaError_t tslb_launch_fill(tslb_ctx *c, void *buf, cudaStream_t st)
{
    if (!any_open(c)) return cudaSuccess;
    int pm = c->nx * c->ny;
    if (c->nx * c->nz > pm) pm = c->nx * c->nz;
    if (c->ny * c->nz > pm) pm = c->ny * c->nz;
    dim3 block(128), grid((pm + 127) / 128, 6);
    if (c->dtype == TSLB_F32) fill_boundary_kernel<float><<<grid, block, 0, st>>>((float *)buf, make_fill(c));
    else fill_boundary_kernel<double><<<grid, block, 0, st>>>((double *)buf, make_fill(c));
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tslb_launch_halo(tslb_ctx *c, void *buf, cudaStream_t st)
{
    const long long tot = 2LL * c->ny * c->nz;
    long long blocks = (tot + 255) / 256;
    if (blocks > (long long)c->sm_count * 16) blocks = (long long)c->sm_count * 16;
    if (c->dtype == TSLB_F32) halo_kernel<float><<<(unsigned)blocks, 256, 0, st>>>((float *)buf, make_fill(c));
    else halo_kernel<double><<<(unsigned)blocks, 256, 0, st>>>((double *)buf, make_fill(c));
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tslb_launch_face(tslb_ctx *c, int dir, int z, void *dense, cudaStream_t st)
{
    const dim3 grid(c->ny, TSLB_NF);            // ny <= 131070 (tslb_create)
    const int xper = c->kind[0] == TSLB_BC_PERIODIC;
    void *buf = c->buf[c->cur];
    if (c->dtype == TSLB_F32) {
        if (dir > 0) face_kernel<float, +1><<<grid, 128, 0, st>>>((float *)buf, (float *)dense, c->L, z, xper);
        else face_kernel<float, -1><<<grid, 128, 0, st>>>((float *)buf, (float *)dense, c->L, z, xper);
    } else {
        if (dir > 0) face_kernel<double, +1><<<grid, 128, 0, st>>>((double *)buf, (double *)dense, c->L, z, xper);
        else face_kernel<double, -1><<<grid, 128, 0, st>>>((double *)buf, (double *)dense, c->L, z, xper);
    }
    c->launches++;
    return cudaGetLastError();
}

template <int DIR, int SHIFT>
static cudaError_t launch_convert(tslb_ctx *c, const void *src, void *dst, cudaStream_t st)
{
    const size_t N = tslb_sites(c);
    size_t blocks = (TSLB_NF * N + 255) / 256;
    if (blocks > (size_t)c->sm_count * 16) blocks = (size_t)c->sm_count * 16;
    if (c->dtype == TSLB_F32) convert_kernel<float, DIR, SHIFT><<<(unsigned)blocks, 256, 0, st>>>((const float *)src, (float *)dst, c->L);
    else convert_kernel<double, DIR, SHIFT><<<(unsigned)blocks, 256, 0, st>>>((const double *)src, (double *)dst, c->L);
    c->launches++;
    return cudaGetLastError();
}
cudaError_t tslb_launch_import(tslb_ctx *c, const void *src, void *dst, cudaStream_t st) { return launch_convert<+1, 1>(c, src, dst, st); }
cudaError_t tslb_launch_export(tslb_ctx *c, const void *src, void *dst, cudaStream_t st) { return launch_convert<-1, 1>(c, src, dst, st); }
cudaError_t tslb_launch_import_raw(tslb_ctx *c, const void *src, void *dst, cudaStream_t st) { return launch_convert<+1, 0>(c, src, dst, st); }
cudaError_t tslb_launch_export_raw(tslb_ctx *c, const void *src, void *dst, cudaStream_t st) { return launch_convert<-1, 0>(c, src, dst, st); }

cudaError_t tslb_launch_diag(tslb_ctx *c, double *dev_out5, cudaStream_t st)
{
    if (c->dtype == TSLB_F32)
        diag_partial_kernel<float><<<TSLB_DIAG_BLOCKS, TSLB_DIAG_THREADS, 0, st>>>((const float *)c->buf[c->cur], make_fill(c), c->scratch);
    else
        diag_partial_kernel<double><<<TSLB_DIAG_BLOCKS, TSLB_DIAG_THREADS, 0, st>>>((const double *)c->buf[c->cur], make_fill(c), c->scratch);
    diag_final_kernel<<<1, 160, 0, st>>>(c->scratch, TSLB_DIAG_BLOCKS, dev_out5);
    c->launches += 2;
    return cudaGetLastError();
}

cudaError_t tslb_launch_radial_stats(tslb_ctx *c, double xc, double yc, double dr, int nr, double *dev_sums, cudaStream_t st)
{
    int parts = (c->ny + 63) / 64;          // slabs of ~64 rows: enough CTAs for small nz, few global atomics per ring
    if (parts < 1) parts = 1;
    dim3 grid(c->nz, parts);
    if (c->dtype == TSLB_F32) radial_stats_kernel<float><<<grid, 256, 0, st>>>((const float *)c->buf[c->cur], c->L, xc, yc, dr, nr, dev_sums);
    else radial_stats_kernel<double><<<grid, 256, 0, st>>>((const double *)c->buf[c->cur], c->L, xc, yc, dr, nr, dev_sums);
    c->launches += 1;
    return cudaGetLastError();
}

static int stat_zlo(const tslb_ctx *c) { return c->kind[TSLB_FACE_ZLO] == TSLB_BC_EXCHANGE ? 1 : 0; }
static int stat_zhi(const tslb_ctx *c) { return c->kind[TSLB_FACE_ZHI] == TSLB_BC_EXCHANGE ? c->nz - 1 : c->nz; }

cudaError_t tslb_launch_plane_stats(tslb_ctx *c, int axis, double *dev_sums, cudaStream_t st)
{
    const int na = axis == 0 ? c->nx : (axis == 1 ? c->ny : c->nz);
    dim3 grid(na, TSLB_STAT_PARTS);
    if (c->dtype == TSLB_F32) stats_partial_kernel<float><<<grid, 256, 0, st>>>((const float *)c->buf[c->cur], c->L, axis, c->scratch, stat_zlo(c), stat_zhi(c));
    else stats_partial_kernel<double><<<grid, 256, 0, st>>>((const double *)c->buf[c->cur], c->L, axis, c->scratch, stat_zlo(c), stat_zhi(c));
    const int tot = TSLB_STAT_ROWS * na;
    stats_final_kernel<<<(tot + 127) / 128, 128, 0, st>>>(c->scratch, na, TSLB_STAT_PARTS, dev_sums);
    c->launches += 2;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// Allocation-free variant of the plane statistics (tslb_plane_statistics_static in include/tslb.h): the per-CTA partial
// sums live in a file-scope device array instead of the caller's workspace, so the call needs no scratch from anybody --
// for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
//   * Size: [13][TSLB_STATIC_STAT_MAX_AXIS][8] doubles = 832 KiB, held by every GPU that loads the library until exit.
//   * In host code the array's NAME is a host-side stand-in, not a device address: the kernels get the address that
//     cudaGetSymbolAddress returns, looked up once per device with that device current (static_scratch_ptr).
//   * Every call on a device shares the array.  The partial kernel overwrites every entry the final kernel reads
//     (all 13 x n_axis x 8 of them), so nothing has to be cleared between calls and stale contents of an earlier, larger
//     call are never read; but two calls that OVERLAP on the GPU (different streams, no ordering) race on it.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_static_stat_scratch[TSLB_STAT_ROWS * TSLB_STATIC_STAT_MAX_AXIS * TSLB_STAT_PARTS];

#define TSLB_STATIC_MAX_DEVICES 64
static double *g_static_stat_ptr[TSLB_STATIC_MAX_DEVICES];      // device address of the array, per device ordinal (0 = not looked up)

static cudaError_t static_scratch_ptr(double **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= TSLB_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    double *p = __atomic_load_n(&g_static_stat_ptr[dev], __ATOMIC_ACQUIRE);
    if (!p) {
        e = cudaGetSymbolAddress((void **)&p, g_static_stat_scratch);       // the current device's copy of the array
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        __atomic_store_n(&g_static_stat_ptr[dev], p, __ATOMIC_RELEASE);     // (two threads racing here store the same value)
    }
    *out = p;
    return cudaSuccess;
}

// No cudaMalloc / cudaFree / allocating library routine anywhere on this path: two kernel launches on `st`.
cudaError_t tslb_launch_plane_stats_static(tslb_ctx *c, int axis, double *dev_sums, cudaStream_t st)
{
    const int na = axis == 0 ? c->nx : (axis == 1 ? c->ny : c->nz);
    if (na > TSLB_STATIC_STAT_MAX_AXIS) return cudaErrorInvalidValue;       // (the API layer reports this with a message)
    double *scratch = nullptr;
    cudaError_t e = static_scratch_ptr(&scratch);
    if (e != cudaSuccess) return e;
    dim3 grid(na, TSLB_STAT_PARTS);
    if (c->dtype == TSLB_F32) stats_partial_kernel<float><<<grid, 256, 0, st>>>((const float *)c->buf[c->cur], c->L, axis, scratch, stat_zlo(c), stat_zhi(c));
    else stats_partial_kernel<double><<<grid, 256, 0, st>>>((const double *)c->buf[c->cur], c->L, axis, scratch, stat_zlo(c), stat_zhi(c));
    const int tot = TSLB_STAT_ROWS * na;
    stats_final_kernel<<<(tot + 127) / 128, 128, 0, st>>>(scratch, na, TSLB_STAT_PARTS, dev_sums);
    c->launches += 2;
    return cudaGetLastError();
}

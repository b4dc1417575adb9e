// tslb_internal.h -- host-side context, the device-visible layout/parameter blocks and the launcher prototypes.
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/tslb.h"

#define TSLB_NF 10  // dr = rho - 1, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz

// ---- internal moment-buffer layout -------------------------------------------------
// SoA, one padded box per field: [nz][ny][px] elements, x fastest.  Node (x,y,z), -1 <= x <= nx (x = -1 and x = nx are the
// ghost columns: the periodic images along x, which the contiguous TMA rows cannot wrap), lives at element
//     z*plane + y*px + (x + TSLB_XOFF)      of its field.
// TSLB_XOFF = 4 puts node x = 0 on a 16-byte boundary for both dtypes (TMA box origins and the TMA store of the output
// tile need 16-byte aligned addresses); px is a multiple of 4 with px >= nx + 8.  There are no ghost rows or planes:
// the tile kernel wraps y and z by TMA coordinates, the gather kernel by index arithmetic.
#define TSLB_XOFF 4
struct Layout {
    int nx, ny, nz;
    int px;
    long long plane;  // px*ny
    long long field;  // px*ny*nz
};

__host__ __device__ inline long long lay_idx(const Layout &L, int x, int y, int z)
{
    return (long long)z * L.plane + (long long)y * L.px + (x + TSLB_XOFF);
}

// Device-visible description of one lattice + its boundary set (passed by value).
template <typename T>
struct SweepParams {
    Layout L;
    int kind[6];   // TSLB_BC_* per face
    T beta;        // 1 - omega = 1 - 1/tau, formed in double and rounded once (Eq. 5)
    T g[3];        // body acceleration
    T o3;          // 1 for the third-order expansion (Eq. 18), 0 for the second-order one (Eq. 8)
    const T *beta_z;  // sponge layer (Eq. 26): 1 - omega of the nodes of plane z, [nz]; NULL = uniform beta
};

struct InletDev {
    const void *u_plane;  // [3][n_b][n_a], context dtype
    double noise_amp;
    uint64_t seed;
    int mask;
};

struct FillParams {
    Layout L;
    int kind[6];
    InletDev inlet[6];
    double rho_out[6];   // imposed density of the TSLB_BC_OUTLET_PRESSURE faces
    long long t;  // step index the fill belongs to (noise counter)
};

#ifdef __CUDACC__
// ---- values imposed on open-face boundary nodes: shared by the boundary-fill kernel and by the store warp of the tile
//      kernel (which writes the boundary nodes of time t+1 itself), so that both give the same bits ------------------------
__device__ __forceinline__ uint64_t tslb_mix64(uint64_t z)  // SplitMix64 finaliser (Vigna, public domain)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
// noise variate of the inlet node (x, y, z) at step t (include/tslb.h, tslb_inlet_params; readings A14, A14b)
__device__ __forceinline__ double tslb_inlet_xi(const InletDev &in, const Layout &L, int x, int y, int z, long long t)
{
    const uint64_t lin = ((uint64_t)z * L.ny + y) * L.nx + x;   // API linear index of the node
    uint64_t k64 = tslb_mix64(in.seed ^ (0x9E3779B97F4A7C15ULL * (uint64_t)(t + 1)));
    k64 = tslb_mix64(k64 + lin);
    double xi = (double)(uint32_t)(k64 >> 40) / 8388608.0 - 1.0;  // exact: 24-bit integer
    if (in.mask & TSLB_NOISE_GAUSSIAN) {   // Box-Muller on two uniforms of the same stream, fp64
        const uint64_t k2 = tslb_mix64(k64);
        const double u1 = ((double)(uint32_t)(k64 >> 40) + 1.0) / 16777216.0;
        const double u2 = (double)(uint32_t)(k2 >> 40) / 16777216.0;
        xi = sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
    }
    return xi;
}
// imposed velocity component k of an inlet node: u_in,k (1 + amp xi) on the masked components (fp64, rounded once)
template <typename T>
__device__ __forceinline__ T tslb_inlet_u(const InletDev &in, size_t plane_elems, size_t j, int k, double xi)
{
    double v = (double)((const T *)in.u_plane)[k * plane_elems + j];
    if (in.mask & (1 << k)) v = __dmul_rn(v, __dadd_rn(1.0, __dmul_rn(in.noise_amp, xi)));
    return (T)v;
}
#endif

// geometry of the TMA-staged tile kernel (kernels_tile.cu): a warp owns 2 rows x 30 columns (+ 1 halo lane per side)
#define TILE_COLS 30

struct tslb_ctx {
    int nx, ny, nz, dtype;
    double tau, omega;
    int order;        // Hermite order of the reconstruction, 3 (Eq. 18) or 2 (Eq. 8)
    double g[3];
    int kind[6];
    InletDev inlet[6];
    double rho_out[6];
    Layout L;
    // device memory (caller-owned workspace)
    void *ws;
    size_t ws_bytes;
    void *buf[2];     // moment buffers, internal form (padded SoA, field 0 holds rho - 1)
    double *scratch;  // diagnostics partials
    void *beta_z;     // sponge layer: per-plane 1 - omega in the context dtype, [nz] (in the workspace)
    void *beta_z_host;   // the same on the host (staging for the upload), NULL = no sponge layer
    int sponge_dirty;    // the host table has to be uploaded before the next sweep
    int last_fused;      // the last tile launch wrote the open-face boundary nodes of its output itself (fused fill)
    CUtensorMap tm_main[2][2], tm_row[2][2], tm_store[2][2];  // TMA descriptors [tile geometry][buffer]: tile rows, one halo row, output tile
    int tmap_ok;
    // neighbouring slabs read in place (tslb_set_neighbor): side 0 = below ZLO, 1 = above ZHI
    int nb_on[2], nb_nz[2], nb_cur0[2];
    long long nb_t0[2];              // this context's step count when the neighbour was attached
    void *nb_buf[2][2];              // the peer's two moment buffers
    CUtensorMap nb_main[2][2][2], nb_row[2][2][2];   // [side][tile geometry][peer buffer]
    int cur;          // buf[cur] holds time t
    long long t;
    int have_state;
    int halo_valid;   // ghost columns + open-face boundary nodes of buf[cur] are up to date for time t (tslb_api.cu)
    int kernel_req;   // TSLB_KERNEL_*
    int sm_count;
    long long launches;
    // optional per-kernel timing of the sweep launches (tslb_set_timing): event pairs on the launching stream
    int timing;
    cudaEvent_t *ev;      // 2 * ev_cap events
    int ev_cap, ev_n;
    char err[256];
};

static inline size_t tslb_elem(const tslb_ctx *c) { return c->dtype == TSLB_F64 ? 8 : 4; }
static inline size_t tslb_sites(const tslb_ctx *c) { return (size_t)c->nx * c->ny * c->nz; }

#define TSLB_DIAG_BLOCKS 592  // 148 SMs x 4
#define TSLB_DIAG_THREADS 256

// launchers (defined in the .cu files; all asynchronous on `st`, return cudaGetLastError())
cudaError_t tslb_launch_gather(tslb_ctx *c, cudaStream_t st);
cudaError_t tslb_launch_tile(tslb_ctx *c, cudaStream_t st);
bool tslb_tile_supported(const tslb_ctx *c, const char **why);
cudaError_t tslb_tile_prepare_neighbor(tslb_ctx *c, int side);                            // TMA descriptors over a neighbouring slab's buffers
cudaError_t tslb_tile_prepare(tslb_ctx *c);                                               // TMA descriptors, smem opt-in
cudaError_t tslb_launch_fill(tslb_ctx *c, void *buf, cudaStream_t st);                    // open-face boundary nodes at time t
cudaError_t tslb_launch_halo(tslb_ctx *c, void *buf, cudaStream_t st);                    // ghost layers
cudaError_t tslb_launch_import(tslb_ctx *c, const void *src, void *dst, cudaStream_t st);  // API -> internal
cudaError_t tslb_launch_export(tslb_ctx *c, const void *src, void *dst, cudaStream_t st);  // internal -> API
cudaError_t tslb_launch_import_raw(tslb_ctx *c, const void *src, void *dst, cudaStream_t st);  // the same without the rho <-> rho - 1 shift
cudaError_t tslb_launch_export_raw(tslb_ctx *c, const void *src, void *dst, cudaStream_t st);
cudaError_t tslb_launch_face(tslb_ctx *c, int dir, int z, void *dense, cudaStream_t st);   // slab ghost planes: dir +1 dense -> plane z of buf[cur], -1 back
cudaError_t tslb_launch_diag(tslb_ctx *c, double *dev_out5, cudaStream_t st);
cudaError_t tslb_launch_plane_stats(tslb_ctx *c, int axis, double *dev_sums, cudaStream_t st);
cudaError_t tslb_launch_radial_stats(tslb_ctx *c, double xc, double yc, double dr, int nr, double *dev_sums, cudaStream_t st);

#define TSLB_STAT_ROWS 13   // 1, u (3), uu (6), uuu (3)
#define TSLB_STAT_PARTS 8   // CTAs per plane in the statistics reduction
#define TSLB_STATIC_STAT_MAX_AXIS TSLB_PLANE_STATISTICS_STATIC_MAX   // longest axis the allocation-free variant accepts (include/tslb.h)
cudaError_t tslb_launch_plane_stats_static(tslb_ctx *c, int axis, double *dev_sums, cudaStream_t st);  // scratch in a static device array

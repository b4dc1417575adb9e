// tslb_api.cu -- the C ABI of include/tslb.h: context, validation, launch logic.  No arithmetic of the
// method lives here; every step of the path runs in the kernels.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include "tslb_internal.h"

namespace {

thread_local char g_create_err[256] = "";

int fail(tslb_ctx *c, int code, const char *fmt, const char *detail = "")
{
    char *dst = c ? c->err : g_create_err;
    snprintf(dst, 256, fmt, detail);
    return code;
}

int cuda_fail(tslb_ctx *c, const char *what, cudaError_t e)
{
    snprintf(c->err, sizeof c->err, "%s: %s", what, cudaGetErrorString(e));
    return TSLB_ECUDA;
}

size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

// scratch: per-CTA partials of the diagnostics or of the plane statistics (whichever is larger)
size_t scratch_bytes(const tslb_ctx *c)
{
    int nmax = c->nx > c->ny ? c->nx : c->ny;
    if (c->nz > nmax) nmax = c->nz;
    size_t a = 5 * TSLB_DIAG_BLOCKS * sizeof(double);
    size_t b = (size_t)TSLB_STAT_ROWS * TSLB_STAT_PARTS * nmax * sizeof(double);
    return ((a > b ? a : b) + 255) & ~(size_t)255;
}

size_t buffer_bytes(const tslb_ctx *c) { return align256((size_t)TSLB_NF * (size_t)c->L.field * tslb_elem(c)); }
size_t sponge_bytes(const tslb_ctx *c) { return align256((size_t)c->nz * sizeof(double)); }

// padded internal layout (tslb_internal.h): ghost columns x = -1 and x = nx, node x = 0 on a 16-byte boundary, 16-byte rows,
// never narrower than a TMA box
#ifndef TSLB_PXALIGN
#define TSLB_PXALIGN 4
#endif
Layout make_layout(int nx, int ny, int nz)
{
    Layout L;
    L.nx = nx; L.ny = ny; L.nz = nz;
    L.px = (nx + 2 * TSLB_XOFF + TSLB_PXALIGN - 1) & ~(TSLB_PXALIGN - 1);
    if (L.px < 72) L.px = 72;
    L.plane = (long long)L.px * ny;
    L.field = L.plane * nz;
    return L;
}

int check_ready(tslb_ctx *c, bool need_state)
{
    if (!c) return TSLB_EINVAL;
    if (!c->ws) return fail(c, TSLB_ESTATE, "no workspace bound (call tslb_bind_workspace)");
    if (need_state && !c->have_state) return fail(c, TSLB_ESTATE, "no state loaded (call tslb_set_moments)");
    return TSLB_OK;
}

int check_boundary_set(tslb_ctx *c)
{
    for (int ax = 0; ax < 3; ++ax)
        if ((c->kind[2 * ax] == TSLB_BC_PERIODIC) != (c->kind[2 * ax + 1] == TSLB_BC_PERIODIC))
            return fail(c, TSLB_EINVAL, "PERIODIC must be set on both faces of an axis");
    return TSLB_OK;
}

bool any_open(const tslb_ctx *c)
{
    for (int f = 0; f < 6; ++f)
        if (c->kind[f] == TSLB_BC_VELOCITY_INLET || c->kind[f] == TSLB_BC_OUTLET_ZERO_GRADIENT || c->kind[f] == TSLB_BC_OUTLET_PRESSURE) return true;
    return false;
}

// Boundary nodes of the open faces filled at time t (oracle step 1) and, for the tile kernel, valid ghost columns.
// halo_valid: 0 = nothing done for (buf[cur], t); 1 = boundary nodes filled; 2 = ghost columns valid as well;
// 3 = written by a tile step: the ghost columns are valid (the sweep stores the periodic x images of the nodes it
// writes), the fill is pending.  Only when open faces exist next to a periodic x axis does the fill change nodes whose
// images then have to be refreshed.  Ghost columns of a non-periodic x axis are never used by a node that is advanced;
// they only have to be finite (the workspace is zeroed at bind time).
cudaError_t refresh_boundary(tslb_ctx *c, bool need_halo, cudaStream_t st)
{
    cudaError_t e = cudaSuccess;
    const bool refill = any_open(c) && c->kind[0] == TSLB_BC_PERIODIC;
    if (c->halo_valid < 1 || (c->halo_valid == 3)) {
        e = tslb_launch_fill(c, c->buf[c->cur], st);
        if (e != cudaSuccess) return e;
        c->halo_valid = (c->halo_valid == 3 && !refill) ? 2 : 1;
    }
    if (need_halo && c->halo_valid < 2) {
        e = tslb_launch_halo(c, c->buf[c->cur], st);
        if (e != cudaSuccess) return e;
        c->halo_valid = 2;
    }
    return cudaSuccess;
}

int pick_kernel(const tslb_ctx *c, const char **why)
{
    const bool ok = tslb_tile_supported(c, why);
    if (c->kernel_req == TSLB_KERNEL_GATHER) return TSLB_KERNEL_GATHER;
    if (c->kernel_req == TSLB_KERNEL_TILE) return ok ? TSLB_KERNEL_TILE : -1;
    return ok ? TSLB_KERNEL_TILE : TSLB_KERNEL_GATHER;
}

}  // namespace

extern "C" {

int tslb_create(int nx, int ny, int nz, double tau, int dtype, tslb_ctx **out)
{
    if (!out) return fail(nullptr, TSLB_EINVAL, "out == NULL");
    if (nx < 3 || ny < 3 || nz < 3) return fail(nullptr, TSLB_EINVAL, "every dimension must be >= 3");
    if ((double)nx * ny * nz > 2147483647.0) return fail(nullptr, TSLB_EINVAL, "lattice exceeds 2^31-1 nodes");
    if (ny > 131070) return fail(nullptr, TSLB_EINVAL, "ny exceeds 131070 (grid limit of the gather kernel)");
    if (!isfinite(tau) || !(tau > 0.5)) return fail(nullptr, TSLB_EINVAL, "tau must be finite and > 0.5");
    if (dtype != TSLB_F32 && dtype != TSLB_F64) return fail(nullptr, TSLB_EINVAL, "unknown dtype");
    tslb_ctx *c = (tslb_ctx *)calloc(1, sizeof *c);
    if (!c) return fail(nullptr, TSLB_ENOMEM, "host allocation failed");
    c->nx = nx; c->ny = ny; c->nz = nz; c->dtype = dtype;
    c->tau = tau; c->omega = 1.0 / tau;
    c->order = 3;
    c->kernel_req = TSLB_KERNEL_AUTO;
    c->sm_count = 148;
    c->L = make_layout(nx, ny, nz);
    *out = c;
    return TSLB_OK;
}

void tslb_destroy(tslb_ctx *c)
{
    if (!c) return;
    for (int i = 0; i < 2 * c->ev_cap; ++i) cudaEventDestroy(c->ev[i]);
    free(c->ev);
    free(c->beta_z_host);
    free(c);
}

int tslb_set_timing(tslb_ctx *c, int max_launches)
{
    if (!c) return TSLB_EINVAL;
    if (max_launches < 0 || max_launches > 100000) return fail(c, TSLB_EINVAL, "max_launches out of range");
    for (int i = 0; i < 2 * c->ev_cap; ++i) cudaEventDestroy(c->ev[i]);
    free(c->ev);
    c->ev = nullptr; c->ev_cap = 0; c->ev_n = 0; c->timing = 0;
    if (max_launches == 0) return TSLB_OK;
    c->ev = (cudaEvent_t *)calloc(2 * (size_t)max_launches, sizeof(cudaEvent_t));
    if (!c->ev) return fail(c, TSLB_ENOMEM, "host allocation failed");
    for (int i = 0; i < 2 * max_launches; ++i) {
        cudaError_t e = cudaEventCreate(&c->ev[i]);
        if (e != cudaSuccess) return cuda_fail(c, "cudaEventCreate", e);
    }
    c->ev_cap = max_launches; c->timing = 1;
    return TSLB_OK;
}

int tslb_get_timing(tslb_ctx *c, int *n_launches, double *total_ms)
{
    if (!c || !n_launches || !total_ms) return TSLB_EINVAL;
    double tot = 0;
    for (int i = 0; i < c->ev_n; ++i) {
        float ms = 0;
        cudaError_t e = cudaEventSynchronize(c->ev[2 * i + 1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, c->ev[2 * i], c->ev[2 * i + 1]);
        if (e != cudaSuccess) return cuda_fail(c, "cudaEventElapsedTime", e);
        tot += ms;
    }
    *n_launches = c->ev_n; *total_ms = tot;
    c->ev_n = 0;
    return TSLB_OK;
}

size_t tslb_workspace_bytes(const tslb_ctx *c)
{
    if (!c) return 0;
    return 2 * buffer_bytes(c) + scratch_bytes(c) + sponge_bytes(c);
}

int tslb_bind_workspace(tslb_ctx *c, void *dev_ptr, size_t bytes)
{
    if (!c) return TSLB_EINVAL;
    if (!dev_ptr) return fail(c, TSLB_EINVAL, "workspace pointer is NULL");
    if (((uintptr_t)dev_ptr & 255) != 0) return fail(c, TSLB_EINVAL, "workspace must be 256-byte aligned");
    if (bytes < tslb_workspace_bytes(c)) return fail(c, TSLB_EINVAL, "workspace smaller than tslb_workspace_bytes");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(c, "cudaGetDevice", e);
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(c, "cudaDeviceGetAttribute", e);
    c->sm_count = sms > 0 ? sms : 148;
    c->ws = dev_ptr; c->ws_bytes = bytes;
    c->buf[0] = dev_ptr;
    c->buf[1] = (char *)dev_ptr + buffer_bytes(c);
    c->scratch = (double *)((char *)dev_ptr + 2 * buffer_bytes(c));
    c->beta_z = (char *)dev_ptr + 2 * buffer_bytes(c) + scratch_bytes(c);
    c->sponge_dirty = c->beta_z_host != nullptr;
    c->cur = 0; c->t = 0; c->have_state = 0; c->halo_valid = 0;
    c->nb_on[0] = c->nb_on[1] = 0;
    // padding cells are never written by the kernels: give them a defined (zero) value once
    e = cudaMemset(dev_ptr, 0, 2 * buffer_bytes(c));
    if (e != cudaSuccess) return cuda_fail(c, "cudaMemset(workspace)", e);
    // the memset runs on the legacy default stream; later calls enqueue on the caller's (possibly non-blocking) stream:
    // bind is one-off, so simply wait for it
    e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return cuda_fail(c, "cudaDeviceSynchronize(bind)", e);
    c->tmap_ok = 0;
    e = tslb_tile_prepare(c);            // TMA descriptors of the two buffers
    if (e != cudaSuccess) {              // not fatal: the gather kernel covers everything; TSLB_KERNEL_TILE then reports why
        (void)cudaGetLastError();
        c->tmap_ok = 0;
        snprintf(c->err, sizeof c->err, "TMA descriptor setup failed (%s): tile kernel disabled", cudaGetErrorString(e));
    }
    return TSLB_OK;
}

int tslb_set_moments(tslb_ctx *c, const void *dev_src, void *stream)
{
    int rc = check_ready(c, false);
    if (rc) return rc;
    if (!dev_src) return fail(c, TSLB_EINVAL, "dev_src == NULL");
    cudaError_t e = tslb_launch_import(c, dev_src, c->buf[0], (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(c, "import kernel", e);
    c->cur = 0; c->t = 0; c->have_state = 1; c->halo_valid = 0;
    c->nb_on[0] = c->nb_on[1] = 0;
    return TSLB_OK;
}

int tslb_set_moments_host(tslb_ctx *c, const void *host_src, void *stream)
{
    int rc = check_ready(c, false);
    if (rc) return rc;
    if (!host_src) return fail(c, TSLB_EINVAL, "host_src == NULL");
    cudaStream_t st = (cudaStream_t)stream;
    // buffer 1 is free while the state is being replaced: use it as the staging area
    cudaError_t e = cudaMemcpyAsync(c->buf[1], host_src, TSLB_NF * tslb_sites(c) * tslb_elem(c), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(c, "H2D copy", e);
    e = tslb_launch_import(c, c->buf[1], c->buf[0], st);
    if (e != cudaSuccess) return cuda_fail(c, "import kernel", e);
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(c, "cudaStreamSynchronize", e);
    c->cur = 0; c->t = 0; c->have_state = 1; c->halo_valid = 0;
    c->nb_on[0] = c->nb_on[1] = 0;
    return TSLB_OK;
}

int tslb_set_boundary(tslb_ctx *c, int face, int kind, const void *params)
{
    if (!c) return TSLB_EINVAL;
    if (kind == TSLB_BC_BODY_FORCE) {
        if (!params) return fail(c, TSLB_EINVAL, "BODY_FORCE needs params -> double g[3]");
        const double *g = (const double *)params;
        for (int a = 0; a < 3; ++a)
            if (!isfinite(g[a])) return fail(c, TSLB_EINVAL, "body force must be finite");
        for (int a = 0; a < 3; ++a) c->g[a] = g[a];
        return TSLB_OK;
    }
    if (face < 0 || face > 5) return fail(c, TSLB_EINVAL, "unknown face");
    if (kind < 0 || kind > TSLB_BC_EXCHANGE) return fail(c, TSLB_EINVAL, "unknown boundary kind");
    if (kind == TSLB_BC_EXCHANGE && face != TSLB_FACE_ZLO && face != TSLB_FACE_ZHI)
        return fail(c, TSLB_EINVAL, "EXCHANGE (slab ghost plane) exists on the z faces only");
    if (kind == TSLB_BC_OUTLET_PRESSURE) {
        if (!params) return fail(c, TSLB_EINVAL, "OUTLET_PRESSURE needs params -> double rho_out");
        const double rho = *(const double *)params;
        if (!isfinite(rho) || !(rho > 0)) return fail(c, TSLB_EINVAL, "rho_out must be finite and > 0");
        c->rho_out[face] = rho;
    }
    if (kind == TSLB_BC_VELOCITY_INLET) {
        if (!params) return fail(c, TSLB_EINVAL, "VELOCITY_INLET needs params -> tslb_inlet_params");
        const tslb_inlet_params *ip = (const tslb_inlet_params *)params;
        if (!ip->dev_u_plane) return fail(c, TSLB_EINVAL, "inlet dev_u_plane == NULL");
        if (!isfinite(ip->noise_amp)) return fail(c, TSLB_EINVAL, "inlet noise_amp must be finite");
        c->inlet[face].u_plane = ip->dev_u_plane;
        c->inlet[face].noise_amp = ip->noise_amp;
        c->inlet[face].seed = ip->seed;
        c->inlet[face].mask = ip->noise_component_mask;
    } else {
        memset(&c->inlet[face], 0, sizeof c->inlet[face]);
    }
    c->kind[face] = kind;
    c->halo_valid = 0;
    return TSLB_OK;
}

int tslb_set_order(tslb_ctx *c, int order)
{
    if (!c) return TSLB_EINVAL;
    if (order != 2 && order != 3) return fail(c, TSLB_EINVAL, "order must be 2 (Eq. 8) or 3 (Eq. 18)");
    c->order = order;
    return TSLB_OK;
}

int tslb_set_sponge(tslb_ctx *c, int z_start, double K, double p)
{
    if (!c) return TSLB_EINVAL;
    if (!isfinite(K) || !isfinite(p) || K < 0) return fail(c, TSLB_EINVAL, "sponge: K must be finite and >= 0, p finite");
    free(c->beta_z_host);
    c->beta_z_host = nullptr;
    c->sponge_dirty = 0;
    if (K == 0) return TSLB_OK;
    if (z_start < 0 || z_start >= c->nz) return fail(c, TSLB_EINVAL, "sponge: z_start outside [0, nz)");
    c->beta_z_host = malloc((size_t)c->nz * tslb_elem(c));
    if (!c->beta_z_host) return fail(c, TSLB_ENOMEM, "host allocation failed");
    // Eq. 26 in double; 1 - omega(z) rounded once to the context dtype, like the uniform beta (Eq. 5)
    const double nu = (c->tau - 0.5) / 3.0;
    for (int z = 0; z < c->nz; ++z) {
        double nuz = nu;
        if (z >= z_start) nuz = nu * (K * pow((double)(z - z_start) / (double)(c->nz - z_start), p) + 1.0);
        const double beta = 1.0 - 1.0 / (0.5 + 3.0 * nuz);
        if (c->dtype == TSLB_F64) ((double *)c->beta_z_host)[z] = beta;
        else ((float *)c->beta_z_host)[z] = (float)beta;
    }
    c->sponge_dirty = 1;
    return TSLB_OK;
}

int tslb_set_kernel(tslb_ctx *c, int kernel)
{
    if (!c) return TSLB_EINVAL;
    if (kernel < TSLB_KERNEL_AUTO || kernel > TSLB_KERNEL_TILE) return fail(c, TSLB_EINVAL, "unknown kernel id");
    c->kernel_req = kernel;
    return TSLB_OK;
}

int tslb_active_kernel(const tslb_ctx *c)
{
    if (!c) return -1;
    const char *why = "";
    return pick_kernel(c, &why);
}

int tslb_step(tslb_ctx *c, int n, void *stream)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (n < 0) return fail(c, TSLB_EINVAL, "n < 0");
    rc = check_boundary_set(c);
    if (rc) return rc;
    const char *why = "";
    const int k = pick_kernel(c, &why);
    if (k < 0) return fail(c, TSLB_EINVAL, "TSLB_KERNEL_TILE does not cover this configuration: %s", why);
    if (k != TSLB_KERNEL_TILE && (c->nb_on[0] || c->nb_on[1]))
        return fail(c, TSLB_EINVAL, "a neighbour is attached (tslb_set_neighbor) but the gather kernel would run: %s", why);
    cudaStream_t st = (cudaStream_t)stream;
    if (c->sponge_dirty) {               // per-plane relaxation table of the sponge layer
        cudaError_t e = cudaMemcpyAsync(c->beta_z, c->beta_z_host, (size_t)c->nz * tslb_elem(c), cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return cuda_fail(c, "sponge table upload", e);
        c->sponge_dirty = 0;
    }
    for (int s = 0; s < n; ++s) {
        cudaError_t e = refresh_boundary(c, k == TSLB_KERNEL_TILE, st);    // step 1: boundary nodes (+ ghost layers) at time t
        if (e != cudaSuccess) return cuda_fail(c, "fill/halo kernel", e);
        const bool timed = c->timing && c->ev_n < c->ev_cap;
        if (timed) cudaEventRecord(c->ev[2 * c->ev_n], st);
        e = (k == TSLB_KERNEL_TILE) ? tslb_launch_tile(c, st) : tslb_launch_gather(c, st);  // steps 2-4
        if (timed) cudaEventRecord(c->ev[2 * c->ev_n++ + 1], st);
        if (e != cudaSuccess) return cuda_fail(c, "sweep kernel", e);
        c->cur = 1 - c->cur;                                               // step 5: AB flip-flop
        c->t += 1;
        // 3: periodic ghost images written by the sweep, fill pending; 2: the sweep also wrote the open-face boundary nodes
        // of time t+1 (fused fill; x is not periodic there, so the ghost columns are not used)
        c->halo_valid = (k == TSLB_KERNEL_TILE) ? (c->last_fused ? 2 : 3) : 0;
    }
    return TSLB_OK;
}

int tslb_get_moments(tslb_ctx *c, void *dev_dst, void *stream)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (!dev_dst) return fail(c, TSLB_EINVAL, "dev_dst == NULL");
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = refresh_boundary(c, false, st);
    if (e != cudaSuccess) return cuda_fail(c, "fill kernel", e);
    e = tslb_launch_export(c, c->buf[c->cur], dev_dst, st);
    if (e != cudaSuccess) return cuda_fail(c, "export kernel", e);
    return TSLB_OK;
}

int tslb_get_moments_host(tslb_ctx *c, void *host_dst, void *stream)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (!host_dst) return fail(c, TSLB_EINVAL, "host_dst == NULL");
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = refresh_boundary(c, false, st);
    if (e != cudaSuccess) return cuda_fail(c, "fill kernel", e);
    // the other buffer holds only the stale time t-1 state: use it as the staging area
    e = tslb_launch_export(c, c->buf[c->cur], c->buf[1 - c->cur], st);
    if (e != cudaSuccess) return cuda_fail(c, "export kernel", e);
    e = cudaMemcpyAsync(host_dst, c->buf[1 - c->cur], TSLB_NF * tslb_sites(c) * tslb_elem(c), cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return cuda_fail(c, "D2H copy", e);
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(c, "cudaStreamSynchronize", e);
    return TSLB_OK;
}

int tslb_export_state(tslb_ctx *c, void *dev_dst, long long *step_count, void *stream)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (!dev_dst) return fail(c, TSLB_EINVAL, "dev_dst == NULL");
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = refresh_boundary(c, false, st);
    if (e != cudaSuccess) return cuda_fail(c, "fill kernel", e);
    e = tslb_launch_export_raw(c, c->buf[c->cur], dev_dst, st);
    if (e != cudaSuccess) return cuda_fail(c, "export kernel", e);
    if (step_count) *step_count = c->t;
    return TSLB_OK;
}

int tslb_import_state(tslb_ctx *c, const void *dev_src, long long step_count, void *stream)
{
    int rc = check_ready(c, false);
    if (rc) return rc;
    if (!dev_src) return fail(c, TSLB_EINVAL, "dev_src == NULL");
    if (step_count < 0) return fail(c, TSLB_EINVAL, "step_count < 0");
    cudaError_t e = tslb_launch_import_raw(c, dev_src, c->buf[0], (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(c, "import kernel", e);
    c->cur = 0; c->t = step_count; c->have_state = 1; c->halo_valid = 0;
    c->nb_on[0] = c->nb_on[1] = 0;
    return TSLB_OK;
}

size_t tslb_face_bytes(const tslb_ctx *c)
{
    return c ? (size_t)TSLB_NF * c->ny * c->nx * tslb_elem(c) : 0;
}

static int face_check(tslb_ctx *c, int face, const void *ptr)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (face != TSLB_FACE_ZLO && face != TSLB_FACE_ZHI) return fail(c, TSLB_EINVAL, "face must be TSLB_FACE_ZLO or TSLB_FACE_ZHI");
    if (c->kind[face] != TSLB_BC_EXCHANGE) return fail(c, TSLB_EINVAL, "face is not of kind TSLB_BC_EXCHANGE");
    if (!ptr) return fail(c, TSLB_EINVAL, "face array == NULL");
    return TSLB_OK;
}

int tslb_export_face(tslb_ctx *c, int face, void *dev_dst, void *stream)
{
    int rc = face_check(c, face, dev_dst);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = refresh_boundary(c, false, st);      // lateral open-face nodes of the owned plane, at the current time
    if (e != cudaSuccess) return cuda_fail(c, "fill kernel", e);
    e = tslb_launch_face(c, -1, face == TSLB_FACE_ZLO ? 1 : c->nz - 2, dev_dst, st);
    if (e != cudaSuccess) return cuda_fail(c, "face export kernel", e);
    return TSLB_OK;
}

int tslb_import_face(tslb_ctx *c, int face, const void *dev_src, void *stream)
{
    int rc = face_check(c, face, dev_src);
    if (rc) return rc;
    // the plane's ghost columns are written with it, so halo_valid keeps its value
    cudaError_t e = tslb_launch_face(c, +1, face == TSLB_FACE_ZLO ? 0 : c->nz - 1, (void *)dev_src, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(c, "face import kernel", e);
    return TSLB_OK;
}

int tslb_face_planes(tslb_ctx *c, int face, void **dev_owned, void **dev_ghost, size_t *plane_bytes,
                     size_t *field_stride_bytes, void *stream)
{
    int rc = face_check(c, face, dev_owned);
    if (rc) return rc;
    if (!dev_ghost || !plane_bytes || !field_stride_bytes) return fail(c, TSLB_EINVAL, "NULL output argument");
    const char *why = "";
    cudaError_t e = refresh_boundary(c, pick_kernel(c, &why) == TSLB_KERNEL_TILE, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(c, "fill/halo kernel", e);
    const size_t es = tslb_elem(c);
    char *base = (char *)c->buf[c->cur];
    const int zo = face == TSLB_FACE_ZLO ? 1 : c->nz - 2, zg = face == TSLB_FACE_ZLO ? 0 : c->nz - 1;
    *dev_owned = base + (size_t)zo * c->L.plane * es;
    *dev_ghost = base + (size_t)zg * c->L.plane * es;
    *plane_bytes = (size_t)c->L.plane * es;
    *field_stride_bytes = (size_t)c->L.field * es;
    return TSLB_OK;
}

int tslb_buffers(const tslb_ctx *c, void *dev_buf[2], int *cur)
{
    if (!c || !dev_buf || !cur) return TSLB_EINVAL;
    if (!c->ws) return TSLB_ESTATE;
    dev_buf[0] = c->buf[0]; dev_buf[1] = c->buf[1];
    *cur = c->cur;
    return TSLB_OK;
}

int tslb_set_neighbor(tslb_ctx *c, int face, void *const peer_buf[2], int peer_nz, int peer_cur)
{
    if (!c) return TSLB_EINVAL;
    if (face != TSLB_FACE_ZLO && face != TSLB_FACE_ZHI) return fail(c, TSLB_EINVAL, "face must be TSLB_FACE_ZLO or TSLB_FACE_ZHI");
    const int side = face == TSLB_FACE_ZLO ? 0 : 1;
    if (!peer_buf) { c->nb_on[side] = 0; return TSLB_OK; }
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (c->kind[face] != TSLB_BC_EXCHANGE) return fail(c, TSLB_EINVAL, "face is not of kind TSLB_BC_EXCHANGE");
    if (!peer_buf[0] || !peer_buf[1]) return fail(c, TSLB_EINVAL, "peer buffer == NULL");
    if (peer_nz < 3 || (peer_cur != 0 && peer_cur != 1)) return fail(c, TSLB_EINVAL, "peer_nz < 3 or peer_cur not 0 / 1");
    c->nb_buf[side][0] = peer_buf[0]; c->nb_buf[side][1] = peer_buf[1];
    c->nb_nz[side] = peer_nz; c->nb_cur0[side] = peer_cur; c->nb_t0[side] = c->t;
    cudaError_t e = tslb_tile_prepare_neighbor(c, side);
    if (e != cudaSuccess) return cuda_fail(c, "TMA descriptors of the neighbour", e);
    c->nb_on[side] = 1;
    return TSLB_OK;
}

int tslb_refresh(tslb_ctx *c, void *stream)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    const char *why = "";
    cudaError_t e = refresh_boundary(c, pick_kernel(c, &why) == TSLB_KERNEL_TILE, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(c, "fill/halo kernel", e);
    return TSLB_OK;
}

int tslb_diagnostics(tslb_ctx *c, double *dev_out5, void *stream)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (!dev_out5) return fail(c, TSLB_EINVAL, "dev_out5 == NULL");
    cudaError_t e = tslb_launch_diag(c, dev_out5, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(c, "diagnostics kernels", e);
    return TSLB_OK;
}

int tslb_plane_statistics(tslb_ctx *c, int axis, double *dev_sums, void *stream)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (axis < 0 || axis > 2) return fail(c, TSLB_EINVAL, "axis must be 0, 1 or 2");
    if (!dev_sums) return fail(c, TSLB_EINVAL, "dev_sums == NULL");
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = refresh_boundary(c, false, st);
    if (e != cudaSuccess) return cuda_fail(c, "fill kernel", e);
    e = tslb_launch_plane_stats(c, axis, dev_sums, st);
    if (e != cudaSuccess) return cuda_fail(c, "plane statistics kernels", e);
    return TSLB_OK;
}

int tslb_radial_statistics(tslb_ctx *c, double xc, double yc, double dr, int nr, double *dev_sums, void *stream)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (!dev_sums) return fail(c, TSLB_EINVAL, "dev_sums == NULL");
    if (!isfinite(xc) || !isfinite(yc) || !isfinite(dr) || !(dr > 0)) return fail(c, TSLB_EINVAL, "radial statistics: axis and dr must be finite, dr > 0");
    if (nr < 1 || nr > 512) return fail(c, TSLB_EINVAL, "radial statistics: nr must be in [1, 512]");
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = refresh_boundary(c, false, st);
    if (e != cudaSuccess) return cuda_fail(c, "fill kernel", e);
    e = tslb_launch_radial_stats(c, xc, yc, dr, nr, dev_sums, st);
    if (e != cudaSuccess) return cuda_fail(c, "radial statistics kernel", e);
    return TSLB_OK;
}

int tslb_plane_statistics_static(tslb_ctx *c, int axis, double *dev_sums, void *stream)
{
    int rc = check_ready(c, true);
    if (rc) return rc;
    if (axis < 0 || axis > 2) return fail(c, TSLB_EINVAL, "axis must be 0, 1 or 2");
    if (!dev_sums) return fail(c, TSLB_EINVAL, "dev_sums == NULL");
    const int na = axis == 0 ? c->nx : (axis == 1 ? c->ny : c->nz);
    if (na > TSLB_PLANE_STATISTICS_STATIC_MAX) {
        snprintf(c->err, sizeof c->err, "tslb_plane_statistics_static: axis %d has %d planes, the static scratch holds %d (use tslb_plane_statistics)",
                 axis, na, TSLB_PLANE_STATISTICS_STATIC_MAX);
        return TSLB_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = refresh_boundary(c, false, st);
    if (e != cudaSuccess) return cuda_fail(c, "fill kernel", e);
    e = tslb_launch_plane_stats_static(c, axis, dev_sums, st);
    if (e != cudaSuccess) return cuda_fail(c, "plane statistics kernels (static scratch)", e);
    return TSLB_OK;
}

long long tslb_step_count(const tslb_ctx *c) { return c && c->have_state ? c->t : -1; }
long long tslb_launch_count(const tslb_ctx *c) { return c ? c->launches : -1; }
const char *tslb_last_error(const tslb_ctx *c) { return c ? c->err : g_create_err; }
const char *tslb_version(void) { return "tslb-b200 0.3 (sm_100a)"; }

}  // extern "C"

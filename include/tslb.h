/*
 * tslb.h -- C ABI of libtslb.so: the fused per-timestep sweep of the high-order thread-safe
 * lattice Boltzmann (TSLB) method on the D3Q27 lattice, hand-written for NVIDIA B200 (sm_100a).
 *
 * "PAPER.md:N" = line N of the extracted text of arXiv 2401.17074; DESIGN.md lists how garbled or
 * silent passages are read ("reading A<n>").
 *
 * What the library computes (PAPER.md:68 Eq. 6, :154 Eq. 18, :45 / :126 Eq. 12, :157):
 *   state      10 hydrodynamic moments per lattice node (rho, u[3], Pi_neq[6]) in two ping-pong
 *              ("AB flip-flop") buffers; nothing else is stored.
 *   one step   for every node x and each of the 27 directions c_i, the post-collision population of
 *              the upstream node x - c_i is rebuilt from that node's moments with the third-order
 *              Hermite-regularised expansion  f*_i = f_i^eq + (1 - 1/tau) f_i^neq  (Eq. 14, 17, 18),
 *              pulled, and the new moments rho = sum f, rho u = sum c f, Pi = sum c c f - Pi_eq are
 *              accumulated and written at x only ("thread-safe").  Body force, halfway
 *              bounce-back walls, and the non-equilibrium-extrapolation velocity inlet / zero-gradient
 *              outlet (PAPER.md:181-202 Eq. 22-23, :258) are part of the same step.
 *
 * Conventions
 *   - Every call returns an int status (TSLB_OK = 0).  No exception or abort crosses this boundary;
 *     output arguments are written only on success.  tslb_last_error() gives a message.
 *   - Moment arrays exchanged with the caller are plain SoA  [10][nz][ny][nx], x fastest, of the
 *     context's dtype (float or double), field order
 *         rho, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz      (Pi = NON-equilibrium momentum flux).
 *   - "dev" pointers are CUDA device pointers, "host" pointers are ordinary host memory
 *     (pinned memory makes the copies asynchronous).  The library never allocates device memory:
 *     the caller binds one workspace (tslb_workspace_bytes) and keeps it alive until destroy/rebind.
 *   - `stream` is a borrowed cudaStream_t passed as void* (NULL = legacy default stream).  All
 *     device work is enqueued on it and the call returns without synchronising, except the
 *     *_host calls, which synchronise the stream before returning.
 *   - A context is not thread-safe; distinct contexts are independent.
 *   - There is no CPU fallback: without a CUDA device every call that needs one fails with TSLB_ECUDA.
 */
#ifndef TSLB_H_
#define TSLB_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tslb_ctx tslb_ctx; /* opaque, owned by the library */

enum { TSLB_F32 = 0, TSLB_F64 = 1 };
enum { TSLB_OK = 0, TSLB_EINVAL = 1, TSLB_ENOMEM = 2, TSLB_ECUDA = 3, TSLB_ESTATE = 4 };
enum { TSLB_FACE_XLO = 0, TSLB_FACE_XHI, TSLB_FACE_YLO, TSLB_FACE_YHI, TSLB_FACE_ZLO, TSLB_FACE_ZHI };
enum {
    TSLB_BC_PERIODIC = 0,             /* index wraps modulo n on that axis (both faces of the axis)   */
    TSLB_BC_BOUNCE_BACK = 1,          /* halfway bounce-back no-slip wall half a cell outside the face */
    TSLB_BC_VELOCITY_INLET = 2,       /* nodes ON the face: u imposed, rho and Pi_neq from x_F          */
    TSLB_BC_OUTLET_ZERO_GRADIENT = 3, /* nodes ON the face: all 10 moments copied from x_F              */
    TSLB_BC_BODY_FORCE = 4,           /* not a face kind: sets the body acceleration g (face ignored)   */
    TSLB_BC_OUTLET_PRESSURE = 5,      /* nodes ON the face: rho imposed, u and Pi_neq copied from x_F    */
    TSLB_BC_EXCHANGE = 6              /* z faces only: nodes ON the face are the ghost plane of a slab     */
                                      /* decomposition, supplied by tslb_import_face (below)               */
};
/* Bit 8 of tslb_inlet_params.noise_component_mask: Gaussian noise law instead of the uniform one (below). */
#define TSLB_NOISE_GAUSSIAN 0x100
/* Which sweep kernel tslb_step uses. AUTO picks the TMA-staged register-marching tile kernel when the
 * boundary set allows it and the per-direction gather kernel otherwise. */
enum { TSLB_KERNEL_AUTO = 0, TSLB_KERNEL_GATHER = 1, TSLB_KERNEL_TILE = 2 };

/* Parameters of TSLB_BC_VELOCITY_INLET (PAPER.md:181 Eq. 22, :270; readings A13, A14).
 * dev_u_plane: imposed velocity on the face, [3][n_b][n_a] of the context dtype, a = lower in-plane
 * axis (fastest), b = higher in-plane axis; caller-owned and must outlive the context's use of it.
 * Component k of node x_B at step t is  u_in,k * (1 + noise_amp * xi(seed, t, lin(x_B)))  when bit k of
 * noise_component_mask is set, else u_in,k;  xi in [-1,1) = 2 r24 / 2^24 - 1 with r24 the top 24 bits
 * of mix64(mix64(seed ^ (0x9E3779B97F4A7C15 * (t+1))) + lin), mix64 = SplitMix64's finaliser and
 * lin = (z*ny + y)*nx + x.  With TSLB_NOISE_GAUSSIAN set in the mask xi is instead the unit normal
 * sqrt(-2 ln u1) cos(2 pi u2), u1 = (r24 + 1)/2^24, u2 = r24'/2^24 with r24' the top 24 bits of mix64 applied once
 * more ("time-varying Gaussian noise"; evaluated in fp64).
 * A zero u_in with no noise is the thread-safe NEQ no-slip wall of PAPER.md:161-187 (wall nodes ON the face). */
typedef struct tslb_inlet_params {
    const void *dev_u_plane;
    double noise_amp;
    uint64_t seed;
    int32_t noise_component_mask;
} tslb_inlet_params;

/* Create a context for an nx x ny x nz lattice with BGK relaxation time tau (omega = 1/tau,
 * nu = (tau - 1/2)/3).  Pure host call (no CUDA).  Defaults: all faces PERIODIC, g = 0.
 * TSLB_EINVAL: out == NULL, a dimension < 3, the lattice exceeds 2^31-1 nodes or ny > 131070, tau not finite or
 * <= 0.5, unknown dtype.  TSLB_ENOMEM: host allocation failed. */
int tslb_create(int nx, int ny, int nz, double tau, int dtype, tslb_ctx **out);

/* Free the context (host memory only; the workspace and inlet planes stay the caller's). NULL is a no-op. */
void tslb_destroy(tslb_ctx *ctx);

/* Bytes of device memory the context needs: two moment buffers in the internal layout (10 fields, rows padded by the two
 * ghost columns to a multiple of 16 bytes) plus scratch for the diagnostics reduction.  0 if ctx == NULL. */
size_t tslb_workspace_bytes(const tslb_ctx *ctx);

/* Give the context its device memory (256-byte aligned, >= tslb_workspace_bytes, caller-owned).  First
 * call that touches CUDA: queries the current device, zeroes the workspace, builds the TMA descriptors.  Rebinding discards the state (set_moments again).
 * TSLB_EINVAL: NULL / misaligned / too small.  TSLB_ECUDA: no usable device. */
int tslb_bind_workspace(tslb_ctx *ctx, void *dev_ptr, size_t bytes);

/* Load the state at t = 0 from a device array [10][nz][ny][nx] of the context dtype (layout above);
 * resets the step counter.  Enqueued on `stream`.  TSLB_ESTATE: no workspace bound. */
int tslb_set_moments(tslb_ctx *ctx, const void *dev_src, void *stream);
/* Same from host memory (H2D copy through the workspace's staging area, then the same conversion);
 * synchronises `stream` before returning. */
int tslb_set_moments_host(tslb_ctx *ctx, const void *host_src, void *stream);

/* Set the kind of one face, or the body force.
 *   PERIODIC / BOUNCE_BACK / OUTLET_ZERO_GRADIENT / EXCHANGE (z faces only) : params == NULL.
 *   VELOCITY_INLET : params -> tslb_inlet_params.
 *   OUTLET_PRESSURE: params -> const double rho_out (> 0): density imposed on the face nodes, u and Pi_neq from x_F
 *                    (PAPER.md:187 "either momentum or density/pressure", :202).
 *   BODY_FORCE     : params -> const double g[3] (acceleration; adds w_i rho c_i.g / cs^2 to the
 *                    post-collision population of the SOURCE node, reading A11); face ignored.
 * TSLB_EINVAL: unknown face/kind, missing params, non-finite g or noise_amp.  Consistency of the whole
 * set (PERIODIC must be on both faces of an axis) is checked by tslb_step. */
int tslb_set_boundary(tslb_ctx *ctx, int face, int kind, const void *params);

/* Hermite order of the reconstruction: 3 (default) = the high-order TSLB of PAPER.md:154 (Eq. 18); 2 = the second-order
 * TSLB of PAPER.md:86-89 (Eq. 8: second-order equilibrium, Eq. 2, plus (1 - omega) times the projected non-equilibrium
 * part, Eq. 7).  Same stored state, same traffic; only the arithmetic changes.  TSLB_EINVAL for any other value. */
int tslb_set_order(tslb_ctx *ctx, int order);

/* Sponge layer towards the z = nz exit (Eq. 26): the kinematic viscosity of the nodes of plane z is
 *     nu(z) = nu ( K ((z - z_start) / (nz - z_start))^p + 1 )   for z >= z_start,     nu otherwise,
 * i.e. a relaxation time tau(z) = 1/2 + 3 nu(z) per plane; the post-collision population of a node is
 * relaxed with the tau of THAT (source) node (Eq. 6).  Reading A24: the printed denominator "N_z - z_end"
 * is the width of the layer and the printed exponent "-3" is +3; p is an argument (paper: K = 1000, z_start = nz - 50).
 * K == 0 removes the layer.  Host-side call, takes effect at the next tslb_step (the per-plane table lives in the
 * workspace and is uploaded on the stream of that step).  Both sweep kernels honour it.
 * TSLB_EINVAL: K < 0, non-finite K or p, z_start outside [0, nz). */
int tslb_set_sponge(tslb_ctx *ctx, int z_start, double K, double p);

/* Choose the sweep kernel (TSLB_KERNEL_*).  TSLB_EINVAL if TILE is forced on a configuration it does not
 * cover (reported by tslb_step). */
int tslb_set_kernel(tslb_ctx *ctx, int kernel);
/* The kernel the next tslb_step would launch (TSLB_KERNEL_GATHER or TSLB_KERNEL_TILE), or -1. */
int tslb_active_kernel(const tslb_ctx *ctx);

/* Advance n time steps (n >= 0): n x { boundary-node fill + ghost-column refresh at time t ; fused stream-collide
 * sweep A -> B ; swap }.  Asynchronous on `stream`; no host<->device traffic.  TSLB_ESTATE before bind/set_moments,
 * TSLB_EINVAL for n < 0 or an inconsistent boundary set, TSLB_ECUDA on a launch error. */
int tslb_step(tslb_ctx *ctx, int n, void *stream);

/* Write the current state (boundary nodes filled at the current t first) to a device array of the layout
 * above. */
int tslb_get_moments(tslb_ctx *ctx, void *dev_dst, void *stream);
/* Same to host memory; synchronises `stream` before returning. */
int tslb_get_moments_host(tslb_ctx *ctx, void *host_dst, void *stream);

/* Checkpoint / resume (the 10 moment arrays are the whole state).  tslb_export_state writes the state
 * bit for bit as it is held -- the layout of tslb_get_moments, except that field 0 is rho - 1, the shifted form the buffers
 * store (tslb_get_moments adds the 1 back, which rounds fp32 values once) -- and returns the
 * step counter, which the seeded inlet noise depends on.  tslb_import_state loads such an array and restores the counter:
 * run 2n  ==  run n, export, import, run n  bitwise, on the same kernel.  Device pointers, enqueued on `stream`.
 * TSLB_EINVAL: NULL array, step_count < 0; TSLB_ESTATE: no workspace / (export) no state. */
int tslb_export_state(tslb_ctx *ctx, void *dev_dst, long long *step_count, void *stream);
int tslb_import_state(tslb_ctx *ctx, const void *dev_src, long long step_count, void *stream);

/* Mass sum(rho), momentum sum(rho u)[3] and kinetic energy 1/2 sum(rho |u|^2) over the nodes that are not
 * on an open (inlet/outlet) face, accumulated in fp64 with warp-shuffle reductions and a fixed-order final
 * pass (bitwise reproducible).  dev_out5: 5 doubles in device memory. */
int tslb_diagnostics(tslb_ctx *ctx, double *dev_out5, void *stream);

/* Per-kernel timing of the sweep launches (bench.py's roofline figure).  tslb_set_timing(ctx, m) with m > 0 makes
 * tslb_step bracket each of its next m sweep-kernel launches with a CUDA event pair recorded on the launching stream
 * (m = 0 switches it off and frees the events).  tslb_get_timing waits for the recorded launches, returns how many
 * there were and the sum of their durations in milliseconds, and resets the count.  The events sit between launches
 * of the same stream, so they add no synchronisation; leave timing off inside a throughput measurement. */
int tslb_set_timing(tslb_ctx *ctx, int max_launches);
int tslb_get_timing(tslb_ctx *ctx, int *n_launches, double *total_ms);

/* Running plane statistics for the turbulence statistics of PAPER.md:236 (Eq. 24) and :242 (Eq. 25).  For every plane j
 * of constant coordinate along `axis` (0 = x, 1 = y, 2 = z) the sums over the nodes of the plane of
 *     1 | ux uy uz | ux ux, uy uy, uz uz, ux uy, ux uz, uy uz | ux^3 uy^3 uz^3
 * at the current time (open-face boundary nodes refilled first) are ADDED to dev_sums, 13 rows of n_axis doubles in
 * device memory ([13][n_axis], row order as listed).  The caller zeroes the array once and calls once per sample; means,
 * Reynolds stresses <u'_i u'_j> and skewness follow from the raw sums.  fp64 accumulation, warp-shuffle reduction,
 * fixed-order final pass (bitwise reproducible).  TSLB_EINVAL: bad axis or NULL; TSLB_ESTATE: no state. */
int tslb_plane_statistics(tslb_ctx *ctx, int axis, double *dev_sums, void *stream);

/* The same sums as tslb_plane_statistics, for callers that must not allocate or hand over scratch (CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the per-CTA partial sums live in a file-scope device array of the
 * library -- [13][TSLB_PLANE_STATISTICS_STATIC_MAX][8] doubles = 832 KiB, held by every GPU that loads the library until
 * exit -- instead of the workspace.  The call itself allocates nothing (no cudaMalloc / cudaFree, two kernel launches on
 * `stream`, preceded by the boundary-fill launch when boundary nodes are stale, as in tslb_plane_statistics).
 * dev_sums: [13][n_axis] doubles in device memory, caller-owned, sums are ADDED as above; same fixed summation order,
 * hence bitwise the same result as tslb_plane_statistics.
 * All calls on one device share the array: it keeps the last call's contents (every entry that is read is rewritten
 * first, so nothing needs clearing), and calls that overlap on the GPU -- different streams without ordering, also from
 * different contexts -- race on it.
 * TSLB_EINVAL: bad axis, NULL, or n_axis > TSLB_PLANE_STATISTICS_STATIC_MAX (use tslb_plane_statistics then);
 * TSLB_ESTATE: no state; TSLB_ECUDA: the array's device address could not be obtained, or a launch failed. */
#define TSLB_PLANE_STATISTICS_STATIC_MAX 1024
int tslb_plane_statistics_static(tslb_ctx *ctx, int axis, double *dev_sums, void *stream);

/* Running (r, z)-bin statistics of a round jet along z (Fig. 7-8: centre-line velocity and Eq. 27,
 * half-width, mean axial profile, axial / radial rms, Reynolds stress <u'_z u'_r> on sections z = const).  Reading A27
 * (DESIGN.md): with (xc, yc) the jet axis in node coordinates, dx = x - xc, dy = y - yc, r = sqrt(dx^2 + dy^2), a node
 * belongs to ring k = floor(r / dr) of its plane if k < nr; u_r = (u_x dx + u_y dy) / r, u_t = (u_y dx - u_x dy) / r
 * (both 0 on the axis).  For every plane z and ring k the sums of
 *     1 | u_z | u_r | u_t | u_z^2 | u_r^2 | u_t^2 | u_z u_r
 * at the current time (open-face boundary nodes refilled first) are ADDED to dev_sums, [8][nz][nr] doubles in device
 * memory.  The caller zeroes the array once and calls once per sample.  fp64 throughout; the ring index is decided in
 * fp64 without fused multiply-adds (identical on every IEEE machine); the additions use atomics, so repeated runs agree
 * to rounding, not bitwise.  TSLB_EINVAL: NULL, dr <= 0, non-finite arguments, nr outside [1, 512]; TSLB_ESTATE: no state. */
int tslb_radial_statistics(tslb_ctx *ctx, double xc, double yc, double dr, int nr, double *dev_sums, void *stream);

/* Slab decomposition along z (PAPER.md:318 names multi-GPU domain decomposition as the next step).
 * A rank owns planes [z_lo, z_hi) of the global lattice and holds them in a context of its own whose z axis is extended by
 * one GHOST plane per cut face: face kind TSLB_BC_EXCHANGE on TSLB_FACE_ZLO and/or TSLB_FACE_ZHI.  The nodes of a ghost plane
 * are never filled by the library (the tile kernel does not write them, what the gather kernel writes there is meaningless); their time-t moments are the caller's to
 * supply before every tslb_step (n = 1 per exchange): because a sweep reads only time-t nearest neighbours (Eq. 6, :157), the
 * owned planes then advance exactly -- bit for bit -- as they would in the undivided lattice.  Per step and cut face:
 *     tslb_export_face(face)  the 10 moments of the outermost OWNED plane (z = 1 for ZLO, z = nz - 2 for ZHI) at the current
 *                             time, as held internally ([10][ny][nx], x fastest, field 0 = rho - 1: no rounding), after the
 *                             open-face boundary nodes of that plane have been filled for the current time;
 *     (transport: the caller's -- NCCL send/recv over NVLink in paper_2401_17074_b200/slab.py, a device copy on one GPU)
 *     tslb_import_face(face)  such an array into the ghost plane (z = 0 for ZLO, z = nz - 1 for ZHI) of the current state,
 *                             ghost columns included.
 * Both are asynchronous on `stream`; face_bytes = 10 * ny * nx * sizeof(dtype) (tslb_face_bytes).  Ghost planes are left out
 * of tslb_diagnostics and tslb_plane_statistics(_static) (on axis 2 their rows stay as they were), so the sums of the ranks add up
 * to those of the undivided lattice; tslb_radial_statistics is per plane: drop the ghost planes' rows.  The seeded inlet noise is keyed
 * on the node's index in the context's own lattice: an inlet on the z = 0 face of the first slab draws the numbers of the
 * undivided run, inlets on faces the cuts cross do not.
 * TSLB_EINVAL: face is not ZLO / ZHI or not of kind EXCHANGE, NULL pointer; TSLB_ESTATE: no state. */
size_t tslb_face_bytes(const tslb_ctx *ctx);
int tslb_export_face(tslb_ctx *ctx, int face, void *dev_dst, void *stream);
int tslb_import_face(tslb_ctx *ctx, int face, const void *dev_src, void *stream);
/* Zero-copy form of the same exchange, for transports that can read and write the workspace in place (NCCL send / recv,
 * peer-to-peer or same-device copies): where the two planes of an EXCHANGE face live in the CURRENT moment buffer.
 * *dev_owned / *dev_ghost: field 0 of the outermost owned plane / of the ghost plane; field f of either starts
 * f * *field_stride_bytes further on and is one contiguous run of *plane_bytes bytes (the plane's rows with their padding and
 * ghost columns).  Two contexts with the same nx, ny and dtype have the same plane layout, so copying the
 * ten runs of a neighbour's owned plane onto this context's ghost plane is the whole exchange: no staging, ghost columns
 * included.  Before returning, the call enqueues on `stream` whatever completes the owned plane for the current time (fill
 * of lateral open-face nodes, ghost-column refresh).  The pointers are valid until the next tslb_step / set_moments /
 * import_state of this context (the buffers ping-pong): ask again after every step.  The ghost plane must be written
 * before the next tslb_step and after the sweep that precedes it has finished (stream order does that).
 * Same error codes as tslb_export_face. */
int tslb_face_planes(tslb_ctx *ctx, int face, void **dev_owned, void **dev_ghost, size_t *plane_bytes,
                     size_t *field_stride_bytes, void *stream);

/* Fused form of the exchange: no exchange at all.  After tslb_set_neighbor the tile kernel's TMA producer loads the source
 * plane ON the EXCHANGE face `face` -- this context's ghost plane -- straight from the neighbouring slab's current moment
 * buffer (its outermost owned plane), tile by tile while it sweeps: peer memory over NVLink when the neighbour lives on another
 * GPU (peer access enabled, or its buffers mapped through CUDA IPC), plain global memory when it lives on the same one.  The
 * ghost plane of this context is then never read and nothing has to be copied between steps.
 *   peer_buf   the neighbour's two moment buffers as tslb_buffers reports them (addresses valid on THIS device), or NULL to
 *              detach (back to tslb_import_face / tslb_face_planes);
 *   peer_nz    the neighbour context's nz (its own ghost planes included); nx, ny and dtype must equal this context's;
 *   peer_cur   which of the two buffers holds the neighbour's current time level now.
 * Contract: from here on both contexts take their steps in lockstep (tslb_step(n = 1) on each, then the next step), so
 * that the neighbour's current buffer alternates with this context's; the caller orders the work so that (a) the neighbour's
 * state of time t is complete (its sweep of the previous step has finished and tslb_refresh has run on it) before this
 * context's sweep of step t starts, and (b) that sweep has finished before the neighbour's sweep of step t+1 starts (it
 * overwrites the buffer being read): one stream, or one barrier per step between neighbours.  tslb_set_moments,
 * tslb_import_state and tslb_bind_workspace detach every neighbour.  Tile kernel only: tslb_step fails with TSLB_EINVAL if
 * the gather kernel would run while a neighbour is attached.
 * TSLB_EINVAL: face not ZLO / ZHI or not EXCHANGE, peer_nz < 3, peer_cur not 0 / 1, NULL buffer; TSLB_ESTATE: no state;
 * TSLB_ECUDA: the TMA descriptors could not be built. */
int tslb_buffers(const tslb_ctx *ctx, void *dev_buf[2], int *cur);
int tslb_set_neighbor(tslb_ctx *ctx, int face, void *const peer_buf[2], int peer_nz, int peer_cur);
/* Enqueue on `stream` whatever completes the current state (open-face boundary nodes of the current time, ghost columns):
 * what tslb_step does first.  For callers that let another context read this one's planes (tslb_set_neighbor). */
int tslb_refresh(tslb_ctx *ctx, void *stream);

/* Steps taken since the last set_moments, or -1. */
long long tslb_step_count(const tslb_ctx *ctx);
/* Number of kernels this context has launched so far (all kinds), for bench.py's gpu_launches. */
long long tslb_launch_count(const tslb_ctx *ctx);
/* Message of the last failing call on this context (ctx-owned, valid until the next call); for
 * ctx == NULL the message of the last failed tslb_create in this thread. */
const char *tslb_last_error(const tslb_ctx *ctx);
/* Library version string, e.g. "tslb-b200 0.1 (sm_100a)". */
const char *tslb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TSLB_H_ */

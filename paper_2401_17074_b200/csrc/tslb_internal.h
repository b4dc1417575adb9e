// tslb_internal.h -- host-side context and the parameter block handed to every kernel.
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/tslb.h"

#define TSLB_NF 10  // rho, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz

// Device-visible description of one lattice + its boundary set (passed by value).
template <typename T>
struct SweepParams {
    int nx, ny, nz;
    int kind[6];   // TSLB_BC_* per face
    T beta;        // 1 - omega = 1 - 1/tau, formed in double and rounded once (Eq. 5)
    T g[3];        // body acceleration
};

struct InletDev {
    const void *u_plane;  // [3][n_b][n_a], context dtype
    double noise_amp;
    uint64_t seed;
    int mask;
};

struct FillParams {
    int nx, ny, nz;
    int kind[6];
    InletDev inlet[6];
    long long t;  // step index the fill belongs to (noise counter)
};

struct tslb_ctx {
    int nx, ny, nz, dtype;
    double tau, omega;
    double g[3];
    int kind[6];
    InletDev inlet[6];
    // device memory (caller-owned workspace)
    void *ws;
    size_t ws_bytes;
    void *buf[2];     // moment buffers, internal form: field 0 holds rho - 1
    double *scratch;  // diagnostics partials
    int cur;          // buf[cur] holds time t
    long long t;
    int have_state;
    int kernel_req;   // TSLB_KERNEL_*
    int sm_count;
    long long launches;
    char err[256];
};

static inline size_t tslb_elem(const tslb_ctx *c) { return c->dtype == TSLB_F64 ? 8 : 4; }
static inline size_t tslb_sites(const tslb_ctx *c) { return (size_t)c->nx * c->ny * c->nz; }

#define TSLB_DIAG_BLOCKS 592  // 148 SMs x 4
#define TSLB_DIAG_THREADS 256

// launchers (defined in the .cu files; all asynchronous on `st`, return cudaGetLastError())
cudaError_t tslb_launch_gather(tslb_ctx *c, cudaStream_t st);
cudaError_t tslb_launch_march(tslb_ctx *c, cudaStream_t st);
bool tslb_march_supported(const tslb_ctx *c, const char **why);
cudaError_t tslb_launch_fill(tslb_ctx *c, void *buf, cudaStream_t st);
cudaError_t tslb_launch_import(tslb_ctx *c, const void *src, void *dst, cudaStream_t st);  // API -> internal
cudaError_t tslb_launch_export(tslb_ctx *c, const void *src, void *dst, cudaStream_t st);  // internal -> API
cudaError_t tslb_launch_diag(tslb_ctx *c, double *dev_out5, cudaStream_t st);

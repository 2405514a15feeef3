// wilson_ctx.cuh — the context record behind the opaque wd_ctx of include/wilson_cg.h and the small host helpers
// shared by the translation units that implement the C ABI (wilson_cg.cu, wilson_coo.cu).
#pragma once
#include "../../include/wilson_cg.h"
#include "wilson_launch.cuh"

#include <cstdarg>
#include <cstdio>

struct wd_ctx {
    int dims[4];
    int V;
    int precision;
    int bc_t;
    int recon;            // reals stored per link: 18 (default) or 12 (rows 0, 1; row 2 rebuilt in the kernels)
    cudaStream_t stream;
    int tile;       // tile index in use
    int tile_user;  // -1 = automatic
    int poll;       // 0 = automatic
    int waves;            // resident waves of the persistent stencil grid (0 -> 1)
    int cg_mode;          // 0 = automatic, 1 = three kernels per iteration, 2 = one cooperative launch
    int coop_ok;          // device supports cooperative launches
    int last_cg_mode;     // what the last cg_solve used
    int prefetch;         // L2 prefetch distance: -1 = automatic (one grid ahead), 0 = off, n > 0 = n tiles
    int zchunk_user;      // z layers per rasterisation chunk, 0 = automatic
    double l2_budget_mb;  // reuse-distance budget of the automatic choice
    int sm_count;
    // CG workspace (native layout), device
    void *r, *p, *q, *y;
    void *w5;             // fifth work vector (BiCGSTAB: t)
    wd::CgScalars *sc;
    double *partials;
    size_t partials_cap;
    unsigned int *counter;
    double *hist;
    int hist_cap;
    double *result_dev;
    // pinned host mirrors
    wd::CgScalars *sc_host;
    double *result_host;
    // staging of the *_host calls
    void *U_can, *U_nat, *s_can, *s_nat_in, *s_nat_out;
    int have_gauge;
    cudaEvent_t ev[4];
    // per-kernel-class timing (wd_set_profile): 4 events per iteration of one poll chunk
    int profile;
    cudaEvent_t *pev;
    int pev_cap;            // iterations the pool covers
    double prof_ms[3];      // accumulated device time of a2, a3, a4
    long prof_n;            // iterations accumulated
    cudaEvent_t bev[6];     // BiCGSTAB: events around the five kernels of the first iteration of every poll chunk
    double bprof_ms[5];
    long bprof_n;
    int last_iters;
    int launches;
    char err[512];
};

extern char g_create_err[512];

static inline int fail(wd_ctx *ctx, int code, const char *fmt, ...)
{
    char *dst = ctx ? ctx->err : g_create_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(ctx, expr)                                                                              \
    do {                                                                                                 \
        cudaError_t e_ = (expr);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? WD_ERR_ALLOC : WD_ERR_CUDA, "%s: %s", #expr, \
                        cudaGetErrorString(e_));                                                         \
    } while (0)

static inline size_t real_bytes(const wd_ctx *c) { return c->precision == 32 ? 4 : 8; }
static inline size_t vpad(const wd_ctx *c) { return ((size_t)c->V + wd::SB - 1) / wd::SB * wd::SB; }  // volume padded to whole site blocks
static inline int padded(const wd_ctx *c) { return vpad(c) != (size_t)c->V; }
static inline size_t spinor_bytes(const wd_ctx *c) { return (size_t)24 * vpad(c) * real_bytes(c); }       // native
static inline size_t gauge_bytes(const wd_ctx *c) { return (size_t)(c->recon == 12 ? 48 : 72) * vpad(c) * real_bytes(c); }        // native
static inline size_t spinor_can_bytes(const wd_ctx *c) { return (size_t)24 * c->V * real_bytes(c); }     // canonical
static inline size_t gauge_can_bytes(const wd_ctx *c) { return (size_t)72 * c->V * real_bytes(c); }      // canonical
static inline size_t spinor_vecs(const wd_ctx *c) { return (size_t)(c->precision == 32 ? 6 : 12) * vpad(c); }


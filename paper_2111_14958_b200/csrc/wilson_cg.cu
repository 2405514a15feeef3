// wilson_cg.cu — the C ABI of include/wilson_cg.h: context, launch logic, the device-resident CG loop.
// Every arithmetic step runs in the kernels of wilson_kernels.cuh; this file only sizes grids,
// enqueues launches on the caller's stream and polls the device stop flag.
#include "wilson_ctx.cuh"
#include "wilson_split.cuh"
#include "wilson_resident.cuh"
#include "wilson_ures.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>

using namespace wd;

// Largest volumes solved by the one-launch CG kernels in automatic mode (sites).  Measured on B200 (near-identity links,
// ms per solve, three kernels / one launch with the launch configuration small_tile_for picks): fp32 16^4 3.48 / 2.23,
// 20^4 7.50 / 6.4, 24^4 13.27 / 14.06; fp64 12^4 5.50 / 3.77, 16^4 9.08 / 8.4, 20^4 24.3 / 26.7.  The split kernel (hopping sum over four warps) wins in fp64 at 4^4 and 8^4 (0.65 / 2.58
// -> 0.49 / 1.76 ms) and loses from 12^4 on.
#ifndef WD_ONELAUNCH_MAX_SITES_F32
#define WD_ONELAUNCH_MAX_SITES_F32 200000
#endif
#ifndef WD_ONELAUNCH_MAX_SITES_F64
#define WD_ONELAUNCH_MAX_SITES_F64 65536
#endif
#ifndef WD_SPLIT_MAX_SITES_F64
#define WD_SPLIT_MAX_SITES_F64 8192
#endif

char g_create_err[512] = "";

/* Host self-test of the fast-division constants used by the tile decode: number of n in [0, n_max) for which
   (n * M) >> (32 + sh) differs from n / d (0 = correct).  No GPU needed. */
extern "C" long wd_selftest_fastdiv(unsigned int d, unsigned int n_max)
{
    if (d == 0) return -1;
    const FastDiv f = make_fastdiv(d);
    long bad = 0;
    for (unsigned int n = 0; n < n_max; ++n) {
        const unsigned int q = f.sh < 0 ? n : (unsigned int)(((unsigned long long)n * f.M) >> 32) >> f.sh;
        bad += (q != n / d);
    }
    return bad;
}

// ---------------------------------------------------------------- launches
template <int DAG, int MODE>
static cudaError_t launch_dslash(wd_ctx *c, const void *U, const void *in, void *out, double kappa, void *r, int it)
{
    const int srow = stage_row_for(c, MODE);
    if (srow >= 0) {   // links through the shared-memory pipeline (wilson_tma.cuh)
        TmaArgs t;
        t.g = make_geom_dims(c, kTmaRows[srow].b, c->zchunk_user);
        t.sm_count = c->sm_count;
        t.stream = c->stream;
        t.U = U; t.in = in; t.out = out; t.r = r; t.kappa = kappa;
        t.sc = MODE == MODE_PLAIN ? nullptr : c->sc;
        t.partials = c->partials; t.counter = c->counter; t.hist = hist_at(c, it); t.it = it;
        c->launches++;
        return c->precision == 32 ? launch_dslash_tma_f32(srow, DAG, MODE, t) : launch_dslash_tma_f64(srow, DAG, MODE, t);
    }
    DslashArgs a;
    a.g = make_geom(c, c->tile);
    a.sm_count = c->sm_count;
    a.stream = c->stream;
    a.U = U; a.Ub = U; a.in = in; a.cen = in; a.out = out; a.kappa = kappa; a.r = r;
    a.sc = MODE == MODE_PLAIN ? nullptr : c->sc;
    a.partials = c->partials; a.counter = c->counter; a.hist = hist_at(c, it); a.it = it;
    c->launches++;
    if (c->recon == 12)
        return c->precision == 32 ? launch_dslash12_f32(c->tile, DAG, MODE, a) : launch_dslash12_f64(c->tile, DAG, MODE, a);
    return c->precision == 32 ? launch_dslash_f32(c->tile, DAG, MODE, a) : launch_dslash_f64(c->tile, DAG, MODE, a);
}

static unsigned int vec_grid(const wd_ctx *c, size_t n)
{
    return wd_vec_grid(c, n, WD_VEC_PER_SM);
}

int wd_ensure_workspace(wd_ctx *c, int max_iter)
{
    const size_t sb = spinor_bytes(c);
    if (!c->r) {
        CUDA_TRY(c, cudaMalloc(&c->r, sb));
        CUDA_TRY(c, cudaMalloc(&c->p, sb));
        CUDA_TRY(c, cudaMalloc(&c->q, sb));
        CUDA_TRY(c, cudaMalloc(&c->y, sb));
        // pad lanes (V not a multiple of 16) are never written by the stencil: zero them once so that the
        // vector kernels can stream whole buffers
        for (void *b : {c->r, c->p, c->q, c->y}) CUDA_TRY(c, cudaMemsetAsync(b, 0, sb, c->stream));
    }
    if (hist_len(max_iter) > c->hist_cap) {
        if (c->hist) cudaFree(c->hist);
        c->hist = nullptr;
        c->hist_cap = 0;
        CUDA_TRY(c, cudaMalloc(&c->hist, sizeof(double) * (size_t)hist_len(max_iter)));
        c->hist_cap = hist_len(max_iter);
    }
    return WD_OK;
}

static int ensure_partials(wd_ctx *c)
{
    // enough for the largest grid any kernel of this ctx can use (smallest tile = 128 threads, no padding bound: use
    // the per-tile maximum) and the vector kernels
    size_t need = (size_t)c->sm_count * 32 * 3;   // one-launch CG: 3 buffers x (at most 32 resident CTAs per SM)
    for (int t = 0; t < WD_NUM_TILES; ++t) {
        const size_t nb = (size_t)tile_blocks(c, t);
        if (nb > need) need = nb;
    }
    need *= 3;                                    // up to three values per CTA (grid_sum_n)
    if (need > c->partials_cap) {
        if (c->partials) cudaFree(c->partials);
        c->partials = nullptr;
        c->partials_cap = 0;
        CUDA_TRY(c, cudaMalloc(&c->partials, need * sizeof(double)));
        c->partials_cap = need;
    }
    return WD_OK;
}

// ---------------------------------------------------------------- context
extern "C" int wd_create(wd_ctx **out, const int dims[4], int precision, int bc_t, void *cuda_stream)
{
    if (!out || !dims) return fail(nullptr, WD_ERR_ARG, "wd_create: NULL argument");
    *out = nullptr;
    if (precision != 32 && precision != 64) return fail(nullptr, WD_ERR_PRECISION, "wd_create: precision must be 32 or 64");
    if (bc_t != -1 && bc_t != 1) return fail(nullptr, WD_ERR_ARG, "wd_create: bc_t must be -1 or +1");
    double vol = 1.0;
    for (int d = 0; d < 4; ++d) {
        if (dims[d] < 4) return fail(nullptr, WD_ERR_DIMS, "wd_create: extent %d of direction %d is < 4", dims[d], d);
        vol *= dims[d];
    }
    if (vol * 36.0 >= 2147483647.0) return fail(nullptr, WD_ERR_DIMS, "wd_create: volume too large for 32-bit plane indexing");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, WD_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return fail(nullptr, WD_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
    wd_ctx *c = (wd_ctx *)calloc(1, sizeof(wd_ctx));
    if (!c) return fail(nullptr, WD_ERR_ALLOC, "wd_create: out of host memory");
    for (int d = 0; d < 4; ++d) c->dims[d] = dims[d];
    c->V = (int)vol;
    c->precision = precision;
    c->bc_t = bc_t;
    c->recon = 18;
    c->stream = (cudaStream_t)cuda_stream;
    c->sm_count = sms;
    cudaDeviceGetAttribute(&c->coop_ok, cudaDevAttrCooperativeLaunch, dev);
    c->tile_user = -1;
    c->tile = auto_tile(c);
    c->l2_budget_mb = 40.0;
    c->small_tile_user = -1;
    c->stage_row = -2;
    c->coo_fast = 1;
    bool ok = true;
    ok = ok && cudaMalloc(&c->sc, sizeof(CgScalars)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->counter, sizeof(unsigned int)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->result_dev, sizeof(double)) == cudaSuccess;
    ok = ok && cudaMallocHost(&c->sc_host, sizeof(CgScalars)) == cudaSuccess;
    ok = ok && cudaMallocHost(&c->result_host, sizeof(double)) == cudaSuccess;
    ok = ok && cudaMallocHost(&c->sc_poll, 2 * sizeof(CgScalars)) == cudaSuccess;
    for (int i = 0; i < 2 && ok; ++i) ok = cudaEventCreateWithFlags(&c->poll_ev[i], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaMemsetAsync(c->counter, 0, sizeof(unsigned int), c->stream) == cudaSuccess;
    ok = ok && cudaMemsetAsync(c->sc, 0, sizeof(CgScalars), c->stream) == cudaSuccess;
    for (int i = 0; i < 4 && ok; ++i) ok = cudaEventCreate(&c->ev[i]) == cudaSuccess;
    if (ok) ok = ensure_partials(c) == WD_OK;
    if (!ok) {
        fail(nullptr, WD_ERR_ALLOC, "wd_create: allocating the ctx state failed: %s", cudaGetErrorString(cudaGetLastError()));
        wd_destroy(c);
        return WD_ERR_ALLOC;
    }
    *out = c;
    return WD_OK;
}

extern "C" int wd_destroy(wd_ctx *c)
{
    if (!c) return WD_OK;
    cudaStreamSynchronize(c->stream);
    void *dev[] = {c->r, c->p, c->q, c->y, c->w5, c->w6, c->w7, c->eo_n2, c->m_ws[0], c->m_ws[1], c->m_ws[2], c->m_ws[3], c->m_sc,
                   c->m_counter, c->m_hist, c->sc, c->partials, c->counter, c->hist, c->result_dev,
                   c->U_can, c->U_nat, c->s_can, c->s_nat_in, c->s_nat_out, c->coo_bad};
    for (void *ptr : dev)
        if (ptr) cudaFree(ptr);
    if (c->sc_host) cudaFreeHost(c->sc_host);
    if (c->m_sc_host) cudaFreeHost(c->m_sc_host);
    if (c->result_host) cudaFreeHost(c->result_host);
    if (c->sc_poll) cudaFreeHost(c->sc_poll);
    for (int i = 0; i < 2; ++i)
        if (c->poll_ev[i]) cudaEventDestroy(c->poll_ev[i]);
    for (int i = 0; i < 4; ++i)
        if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    for (int i = 0; i < 4 * c->pev_cap; ++i) cudaEventDestroy(c->pev[i]);
    for (int i = 0; i < 8; ++i)
        if (c->bev[i]) cudaEventDestroy(c->bev[i]);
    for (int i = 0; i < WD_HOST_SLABS + 1; ++i)
        if (c->slab_ev[i]) cudaEventDestroy(c->slab_ev[i]);
    if (c->copy_stream) { cudaStreamSynchronize(c->copy_stream); cudaStreamDestroy(c->copy_stream); }
    if (c->pack_stream) { cudaStreamSynchronize(c->pack_stream); cudaStreamDestroy(c->pack_stream); cudaEventDestroy(c->pack_ev); }
    free(c->pev);
    free(c);
    return WD_OK;
}

extern "C" const char *wd_last_error(wd_ctx *c) { return c ? c->err : g_create_err; }
extern "C" size_t wd_gauge_native_bytes(wd_ctx *c) { return c ? gauge_bytes(c) : 0; }
extern "C" size_t wd_spinor_native_bytes(wd_ctx *c) { return c ? spinor_bytes(c) : 0; }
extern "C" const char *wd_version(void) { return "wilson_cg 0.1 sm_100a"; }

extern "C" int wd_num_tiles(void) { return WD_NUM_TILES; }
extern "C" int wd_tile_shape(int index, int shape[4])
{
    if (index < 0 || index >= WD_NUM_TILES || !shape) return WD_ERR_ARG;
    for (int d = 0; d < 4; ++d) shape[d] = kTiles[index].b[d];
    return WD_OK;
}
extern "C" int wd_tile_info(int index, int info[3])
{
    if (index < 0 || index >= WD_NUM_TILES || !info) return WD_ERR_ARG;
    info[0] = kTiles[index].minb; info[1] = kTiles[index].f32; info[2] = kTiles[index].f64;
    return WD_OK;
}
extern "C" int wd_set_tile(wd_ctx *c, int index)
{
    if (!c) return WD_ERR_ARG;
    if (index == -1) {
        c->tile_user = -1;
        c->tile = auto_tile(c);
        return WD_OK;
    }
    if (!tile_ok(c, index)) return fail(c, WD_ERR_ARG, "wd_set_tile: tile %d not available for precision %d", index, c->precision);
    c->tile_user = index;
    c->tile = index;
    return WD_OK;
}
extern "C" int wd_get_tile(wd_ctx *c) { return c ? c->tile : WD_ERR_ARG; }
static bool resident_plan(const wd_ctx *c, int *nc_out, int *spc_out);
static int ures_row_for(const wd_ctx *c);
extern "C" int wd_set_cg_mode(wd_ctx *c, int mode)
{
    if (!c || mode < 0 || (mode > 2 && mode != 6 && mode != 9 && mode != 10)) return WD_ERR_ARG;
    if (mode == 10) {
        const int keep = c->cg_mode;
        c->cg_mode = 10;
        const bool ok = c->recon == 18 && ures_row_for(c) >= 0;
        c->cg_mode = keep;
        if (!ok) return fail(c, WD_ERR_ARG, "wd_set_cg_mode(10): the lattice has more tiles than CTAs can be co-resident (or 12-real links)");
    }
    if (mode == 9) {
        int nc, spc;
        if (!resident_plan(c, &nc, &spc))
            return fail(c, WD_ERR_ARG, "wd_set_cg_mode(9): the lattice does not fit a cluster's shared memory (V / nc a power of two <= %d, nc <= 16, 18-real links)",
                        c->precision == 32 ? 256 : 128);
    }
    if (mode >= 2 && !c->coop_ok) return fail(c, WD_ERR_CUDA, "wd_set_cg_mode: the device does not support cooperative launches");
    if (mode >= 2 && c->recon != 18) return fail(c, WD_ERR_ARG, "wd_set_cg_mode: the one-launch kernels need 18-real links");
    c->cg_mode = mode;
    return WD_OK;
}
extern "C" int wd_set_gauge_recon(wd_ctx *c, int reals)
{
    if (!c) return WD_ERR_ARG;
    if (reals != 18 && reals != 12) return fail(c, WD_ERR_ARG, "wd_set_gauge_recon: %d reals per link (18 or 12)", reals);
    if (reals != c->recon) {
        // the staged gauge field of the *_host calls is in the old format
        if (c->U_nat) { cudaStreamSynchronize(c->stream); cudaFree(c->U_nat); c->U_nat = nullptr; }
        c->have_gauge = 0;
    }
    c->recon = reals;
    return WD_OK;
}
extern "C" int wd_get_gauge_recon(wd_ctx *c) { return c ? c->recon : WD_ERR_ARG; }
extern "C" int wd_set_zchunk(wd_ctx *c, int layers)
{
    if (!c || layers < 0) return WD_ERR_ARG;
    c->zchunk_user = layers;
    return WD_OK;
}
extern "C" int wd_set_small_tile(wd_ctx *c, int index)
{
    if (!c || index < -1 || index >= WD_NUM_SMALL_TILES) return WD_ERR_ARG;
    c->small_tile_user = index;
    return WD_OK;
}
extern "C" int wd_num_staging_rows(void) { return WD_NUM_TMA_ROWS; }
extern "C" int wd_staging_row_info(int row, int info[9])
{
    if (row < 0 || row >= WD_NUM_TMA_ROWS || !info) return WD_ERR_ARG;
    const TmaRowInfo &t = kTmaRows[row];
    for (int d = 0; d < 4; ++d) info[d] = t.b[d];
    info[4] = t.nstage; info[5] = t.ahead; info[6] = t.minb; info[7] = t.f32; info[8] = t.f64;
    return WD_OK;
}
extern "C" int wd_set_link_staging(wd_ctx *c, int row)
{
    if (!c) return WD_ERR_ARG;
    if (row == -1 || row == -2) { c->stage_row = row; return WD_OK; }
    if (!stage_row_ok(c, row))
        return fail(c, WD_ERR_ARG, "wd_set_link_staging: row %d does not cover this lattice / precision / link storage", row);
    c->stage_row = row;
    return WD_OK;
}
extern "C" int wd_get_link_staging(wd_ctx *c) { return c ? stage_row_for(c, MODE_QQ) : WD_ERR_ARG; }
extern "C" int wd_set_poll_interval(wd_ctx *c, int n)
{
    if (!c || n < 0) return WD_ERR_ARG;
    c->poll = n;
    return WD_OK;
}

extern "C" int wd_set_profile(wd_ctx *c, int on)
{
    if (!c) return WD_ERR_ARG;
    c->profile = on > 0 ? on : 0;   // n > 1: cg_solve times the kernels of every n-th iteration only
    c->prof_ms[0] = c->prof_ms[1] = c->prof_ms[2] = 0.0;
    c->prof_n = 0;
    for (int j = 0; j < 7; ++j) c->bprof_ms[j] = 0.0;
    c->bprof_n = 0;
    return WD_OK;
}
extern "C" int wd_get_profile(wd_ctx *c, double ms[3], long *iterations)
{
    if (!c || !ms || !iterations) return WD_ERR_ARG;
    for (int j = 0; j < 3; ++j) ms[j] = c->prof_ms[j];
    *iterations = c->prof_n;
    return WD_OK;
}

// ---------------------------------------------------------------- a0: pack / unpack
extern "C" int wd_pack_gauge(wd_ctx *c, const void *can, void *nat)
{
    if (!c) return WD_ERR_ARG;
    if (!can || !nat || can == nat) return fail(c, WD_ERR_ARG, "wd_pack_gauge: NULL or aliased argument");
    const int Vp = (int)vpad(c);
    const unsigned int grid = (Vp + VEC_NT - 1) / VEC_NT;
    if (c->precision == 32 && c->recon == 18)
        pack_gauge_kernel<float, 18><<<grid, VEC_NT, 0, c->stream>>>((const float2 *)can, (float2 *)nat, c->V, Vp);
    else if (c->precision == 32)
        pack_gauge_kernel<float, 12><<<grid, VEC_NT, 0, c->stream>>>((const float2 *)can, (float2 *)nat, c->V, Vp);
    else if (c->recon == 18)
        pack_gauge_kernel<double, 18><<<grid, VEC_NT, 0, c->stream>>>((const double2 *)can, (double2 *)nat, c->V, Vp);
    else
        pack_gauge_kernel<double, 12><<<grid, VEC_NT, 0, c->stream>>>((const double2 *)can, (double2 *)nat, c->V, Vp);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    return WD_OK;
}
extern "C" int wd_pack_spinor(wd_ctx *c, const void *can, void *nat)
{
    if (!c) return WD_ERR_ARG;
    if (!can || !nat || can == nat) return fail(c, WD_ERR_ARG, "wd_pack_spinor: NULL or aliased argument");
    const int Vp = (int)vpad(c);
    const unsigned int grid = (Vp + VEC_NT - 1) / VEC_NT;
    if (c->precision == 32)
        pack_spinor_kernel<float><<<grid, VEC_NT, 0, c->stream>>>((const float4 *)can, (float4 *)nat, c->V, Vp);
    else
        pack_spinor_kernel<double><<<grid, VEC_NT, 0, c->stream>>>((const double2 *)can, (double2 *)nat, c->V, Vp);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    return WD_OK;
}
extern "C" int wd_unpack_spinor(wd_ctx *c, const void *nat, void *can)
{
    if (!c) return WD_ERR_ARG;
    if (!can || !nat || can == nat) return fail(c, WD_ERR_ARG, "wd_unpack_spinor: NULL or aliased argument");
    const unsigned int grid = (c->V + VEC_NT - 1) / VEC_NT;
    if (c->precision == 32)
        unpack_spinor_kernel<float><<<grid, VEC_NT, 0, c->stream>>>((const float4 *)nat, (float4 *)can, c->V);
    else
        unpack_spinor_kernel<double><<<grid, VEC_NT, 0, c->stream>>>((const double2 *)nat, (double2 *)can, c->V);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    return WD_OK;
}

// ---------------------------------------------------------------- a7: wd_apply
extern "C" int wd_apply(wd_ctx *c, const void *U, const void *psi, void *out, double kappa, int dagger)
{
    if (!c) return WD_ERR_ARG;
    if (!U || !psi || !out || psi == out) return fail(c, WD_ERR_ARG, "wd_apply: NULL argument or out aliases psi");
    if (!std::isfinite(kappa)) return fail(c, WD_ERR_ARG, "wd_apply: kappa is not finite");
    cudaError_t e = dagger ? launch_dslash<1, MODE_PLAIN>(c, U, psi, out, kappa, nullptr, 0)
                           : launch_dslash<0, MODE_PLAIN>(c, U, psi, out, kappa, nullptr, 0);
    CUDA_TRY(c, e);
    return WD_OK;
}

/* `reps` back-to-back applications enqueued from C (no binding overhead between the launches), timed with CUDA events
   on the ctx stream: *ms_per_application = device time / reps.  Synchronous. */
extern "C" int wd_apply_repeat(wd_ctx *c, const void *U, const void *psi, void *out, double kappa, int dagger, int reps,
                               double *ms_per_application)
{
    if (!c) return WD_ERR_ARG;
    if (reps < 1 || !ms_per_application) return fail(c, WD_ERR_ARG, "wd_apply_repeat: reps < 1 or NULL result");
    int rc = wd_apply(c, U, psi, out, kappa, dagger);   // argument checks + warm-up
    if (rc != WD_OK) return rc;
    CUDA_TRY(c, cudaEventRecord(c->ev[0], c->stream));
    for (int i = 0; i < reps; ++i) {
        rc = wd_apply(c, U, psi, out, kappa, dagger);
        if (rc != WD_OK) return rc;
    }
    CUDA_TRY(c, cudaEventRecord(c->ev[1], c->stream));
    CUDA_TRY(c, cudaEventSynchronize(c->ev[1]));
    float ms = 0.f;
    CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]));
    *ms_per_application = (double)ms / reps;
    return WD_OK;
}

extern "C" int wd_norm2(wd_ctx *c, const void *a, double *result)
{
    if (!c) return WD_ERR_ARG;
    if (!a || !result) return fail(c, WD_ERR_ARG, "wd_norm2: NULL argument");
    const size_t n = spinor_vecs(c);
    const unsigned int grid = vec_grid(c, n);
    if (c->precision == 32)
        norm2_kernel<float><<<grid, VEC_NT, 0, c->stream>>>((const float4 *)a, n, c->V, padded(c), c->partials, c->counter, c->result_dev);
    else
        norm2_kernel<double><<<grid, VEC_NT, 0, c->stream>>>((const double2 *)a, n, c->V, padded(c), c->partials, c->counter, c->result_dev);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    CUDA_TRY(c, wd_fetch(c, c->result_host, c->result_dev, sizeof(double)));   // not the copy engine: see wd_fetch
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    *result = *c->result_host;
    return WD_OK;
}

// ---------------------------------------------------------------- a1-a6: cg_solve
static int auto_poll(const wd_ctx *c)
{
    // enqueue about 0.4 ms of modelled work (1536 B/site/iteration fp32 at ~6 TB/s) between two polls
    const double t_iter = (c->precision == 32 ? 1536.0 : 3072.0) * c->V / 6.0e12;
    int n = (int)std::ceil(4.0e-4 / (t_iter > 1e-9 ? t_iter : 1e-9));
    if (n < 4) n = 4;
    if (n > 32) n = 32;
    return n;
}

// Small-volume path: the whole solve in one cooperative launch.
static int small_tile_for(const wd_ctx *c)
{
    if (c->small_tile_user >= 0) return c->small_tile_user;
    // modelled time of a phase = rounds of tiles x cost of the row per round (x a mild penalty for threads hanging
    // over the lattice); rounds = ceil(tiles / co-resident CTAs), co-resident CTAs per SM = the row's register bound, or
    // what 255 registers allow (4 CTAs of 64 threads, 2 of 128).  E.g. 14^4: 16x2x2x2 needs 343 CTAs, 296 fit at 255
    // registers (two rounds), 444 at 168 registers (one round): the bounded row wins, 0.61 -> 0.51 ms per solve.
    int best = 0;
    double best_cost = 1e300;
    for (int t = 0; t < WD_NUM_SMALL_TILES; ++t) {
        double blocks = 1.0, threads = 1.0;
        for (int d = 0; d < 4; ++d) {
            blocks *= (c->dims[d] + kSmallTiles[t][d] - 1) / kSmallTiles[t][d];
            threads *= kSmallTiles[t][d];
        }
        const int occ = kSmallMinb[t] > 1 ? kSmallMinb[t] : (threads <= 64 ? 4 : 2);
        const double resident = (double)occ * c->sm_count;
        const double rounds = std::ceil(blocks / resident);
        const double waste = blocks * threads / (double)c->V;
        const double cost = rounds * kSmallCost[t] * (1.0 + 0.1 * (waste - 1.0));
        if (cost < best_cost - 1e-12) { best_cost = cost; best = t; }
    }
    return best;
}

static int split_tile_for(const wd_ctx *c)
{
    int best = 0;
    double best_waste = 1e300;
    for (int t = 0; t < WD_NUM_SPLIT_TILES; ++t) {
        double blocks = 1.0;
        for (int d = 0; d < 4; ++d) blocks *= (c->dims[d] + kSplitTiles[t][d] - 1) / kSplitTiles[t][d];
        const double waste = blocks * 32.0 / (double)c->V;
        if (waste < best_waste - 1e-12) { best_waste = waste; best = t; }
    }
    return best;
}

static bool use_onelaunch(const wd_ctx *c)
{
    if (!c->coop_ok || c->recon != 18) return false;   // the one-launch kernels are compiled for 18-real links only
    if (c->cg_mode == 1) return false;
    if (c->cg_mode >= 2 && c->cg_mode != 9 && c->cg_mode != 10) return true;
    // automatic: volumes whose CG iteration is shorter than three launches (measured crossovers above)
    return c->V <= (c->precision == 64 ? WD_ONELAUNCH_MAX_SITES_F64 : WD_ONELAUNCH_MAX_SITES_F32);
}

// Shared-memory-resident CG (wilson_resident.cuh): the lattice is cut into nc slabs of spc consecutive sites, one CTA of a
// thread-block cluster each.  spc must be a power of two (owner and local index of a neighbour are a shift and a mask), a
// multiple of 32, at most 256 sites in fp32 / 128 in fp64 (672 / 1344 B of shared memory per site), nc <= 16.
static bool resident_plan(const wd_ctx *c, int *nc_out, int *spc_out)
{
    if (c->recon != 18) return false;
    const int max_spc = c->precision == 32 ? 256 : 128;
    for (int nc = 1; nc <= 16; nc *= 2) {
        if (c->V % nc) continue;
        const int spc = c->V / nc;
        if (spc > max_spc || spc % 32 || (spc & (spc - 1))) continue;
        *nc_out = nc; *spc_out = spc;
        return true;
    }
    return false;
}

// Automatic wherever the lattice fits a cluster (measured, us per iteration, resident / best of the other one-launch kernels:
// fp32 4^4 5.1 / 8.6, 512 sites (2 CTAs) 6.6 / 9.5, 1024 sites (4) 7.5 / 9.4-9.8, 2048 sites (8, exports) 8.1-8.3 / 9.6-9.9, 8^4 and
// other 4096-site lattices (16, exports) 8.9-9.0 / 9.7-10.3; fp64 4^4 (2 CTAs) 7.6 / 10.5, 512 sites (4) 7.7 / 10.5, 1024 sites (8)
// 9.6-9.8 / 10.4-11.2, 2048 sites (16, exports) 10.1-10.2 / 10.5).  From eight CTAs on the remote neighbours are read as
// half-spinors exported by their owners (wilson_resident_ex.cuh): pulling whole spinors and links through distributed shared
// memory made the stencil phases of the 16-CTA cluster 4.1 us against 1.9 us without remote neighbours.
static bool use_resident(const wd_ctx *c)
{
    int nc, spc;
    if (c->cg_mode != 0 && c->cg_mode != 9) return false;
    if (!resident_plan(c, &nc, &spc)) return false;
    if (c->cg_mode == 9 || nc <= 4) return true;
    // eight and sixteen CTAs: only where the exported half-spinors fit the shared memory beside the slabs (otherwise the launcher
    // falls back to pulling whole spinors and links, which loses to the cooperative kernels: 10.5-11 against 9.7-10.3 us)
    const int nslots = resident_export_slots(c->dims, spc, nc);
    const size_t need = c->precision == 64 ? resident_ex_smem<double>(spc, nslots) : resident_ex_smem<float>(spc, nslots);
    return nslots < 65536 && need <= WD_RESIDENT_SMEM_MAX;
}

static bool use_split(const wd_ctx *c)
{
    return c->cg_mode == 6 || (c->cg_mode == 0 && c->precision == 64 && c->V <= WD_SPLIT_MAX_SITES_F64);
}

// One-launch CG with the gauge field resident in shared memory (wilson_ures.cuh): the row with the fewest padded threads among
// those compiled for the precision whose tiles all fit one co-resident wave (one tile per CTA for the whole solve); -1 = none.
static int ures_row_for(const wd_ctx *c)
{
    if (!c->coop_ok || c->recon != 18) return -1;
    int best = -1;
    double best_waste = 1e300;
    for (int r = 0; r < WD_NUM_URES_ROWS; ++r) {
        if (!(c->precision == 64 ? kUresRows[r].f64 : kUresRows[r].f32)) continue;
        double blocks = 1.0, threads = 1.0;
        for (int d = 0; d < 4; ++d) {
            blocks *= (c->dims[d] + kUresRows[r].b[d] - 1) / kUresRows[r].b[d];
            threads *= kUresRows[r].b[d];
        }
        const int occ = c->precision == 64 ? ures_occupancy_f64(r) : ures_occupancy_f32(r);
        if (occ < 1 || blocks > (double)occ * c->sm_count) continue;
        const double waste = blocks * threads / (double)c->V;
        if (waste < best_waste - 1e-12) { best_waste = waste; best = r; }
    }
    return best;
}

static bool use_ures(const wd_ctx *c)
{
    if (c->cg_mode != 0 && c->cg_mode != 10) return false;
    if (ures_row_for(c) < 0) return false;
    if (c->cg_mode == 10) return true;
    // automatic: wherever it fits, it beat the L2-resident one-launch kernel (8^4 ... 16^3 x 12, ms per solve, fp32: 0.812 / 0.823,
    // 10^4 0.934 / 0.987, 12^4 1.141 / 1.231, 14^4 1.653 / 1.836, 16^3x12 1.638 / 1.851; fp64: 10^4 2.485 / 2.833, 12^4 3.226 / 3.745,
    // 16^2x12^2 4.024 / 4.366) -- except in fp64 up to 4096 sites, where the four-warp split kernel is faster (8^4: 1.591 / 1.894)
    if (c->precision == 64 && c->V <= 4096) return false;
    return c->V <= (c->precision == 64 ? WD_ONELAUNCH_MAX_SITES_F64 : WD_ONELAUNCH_MAX_SITES_F32);
}

static int cg_onelaunch(wd_ctx *c, const void *U, const void *eta, void *psi, double kappa, double r_min, int max_iter)
{
    if (use_ures(c)) {
        const int row = ures_row_for(c);
        CgOneLaunchArgs a;
        a.g = make_geom_dims(c, kUresRows[row].b, 0);
        a.sm_count = c->sm_count;
        a.stream = c->stream;
        a.U = U; a.eta = eta; a.y = c->y; a.r = c->r; a.p = c->p; a.q = c->q; a.psi = psi;
        a.kappa = kappa; a.sc = c->sc; a.partials = c->partials; a.partials_cap = c->partials_cap; a.hist = hist_whole(c, max_iter);
        a.r_min = r_min; a.max_iter = max_iter;
        c->launches++;
        CUDA_TRY(c, c->precision == 32 ? launch_cg_ures_f32(row, a) : launch_cg_ures_f64(row, a));
        return WD_OK;
    }
    const bool split = use_split(c);
    const int st = split ? split_tile_for(c) : small_tile_for(c);
    CgOneLaunchArgs a;
    a.g = make_geom_dims(c, split ? kSplitTiles[st] : kSmallTiles[st], 0);
    a.sm_count = c->sm_count;
    a.stream = c->stream;
    a.U = U; a.eta = eta; a.y = c->y; a.r = c->r; a.p = c->p; a.q = c->q; a.psi = psi;
    a.kappa = kappa; a.sc = c->sc; a.partials = c->partials; a.partials_cap = c->partials_cap; a.hist = hist_whole(c, max_iter);
    a.r_min = r_min; a.max_iter = max_iter;
    c->launches++;
    if (split) CUDA_TRY(c, c->precision == 32 ? launch_cg_split_f32(st, a) : launch_cg_split_f64(st, a));
    else CUDA_TRY(c, c->precision == 32 ? launch_cg_onelaunch_f32(st, a) : launch_cg_onelaunch_f64(st, a));
    return WD_OK;
}

static int cg_device(wd_ctx *c, const void *U, const void *eta, void *psi, double kappa, double r_min, int max_iter,
                     wd_cg_info *info, bool record_events)
{
    int rc = wd_ensure_workspace(c, max_iter);
    if (rc != WD_OK) return rc;
    if (use_resident(c)) {
        // the paper's smallest volumes: the whole solve in one launch with every field resident in shared memory
        ResidentArgs a;
        for (int d = 0; d < 4; ++d) a.L[d] = c->dims[d];
        a.bc_t = c->bc_t;
        resident_plan(c, &a.nc, &a.spc);
        a.stream = c->stream;
        a.U = U; a.eta = eta; a.psi = psi; a.kappa = kappa; a.sc = c->sc; a.hist = hist_whole(c, max_iter);
        a.r_min = r_min; a.max_iter = max_iter;
        c->last_cg_mode = 9;
        if (record_events) CUDA_TRY(c, cudaEventRecord(c->ev[0], c->stream));
        c->launches++;
        CUDA_TRY(c, c->precision == 32 ? launch_cg_resident_f32(a) : launch_cg_resident_f64(a));
        if (record_events) CUDA_TRY(c, cudaEventRecord(c->ev[1], c->stream));
        CUDA_TRY(c, wd_fetch(c, c->sc_host, c->sc, sizeof(CgScalars)));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        const CgScalars &s1 = *c->sc_host;
        c->last_iters = s1.k;
        if (info) {
            info->iterations = s1.k;
            info->converged = s1.converged;
            info->rel_residual = s1.eta2 > 0.0 ? std::sqrt(s1.rr / s1.eta2) : 0.0;
            info->eta_norm2 = s1.eta2;
            float ms = 0.f;
            if (record_events) CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]));
            info->gpu_ms = ms;
            info->total_ms = ms;
            info->kernel_launches = c->launches;
            info->cg_mode = 9;
        }
        return s1.converged ? WD_OK : (s1.breakdown ? WD_BREAKDOWN : WD_NOT_CONVERGED);
    }
    if (use_ures(c) || use_onelaunch(c)) {
        c->last_cg_mode = use_ures(c) ? 10 : (use_split(c) ? 6 : 2);
        if (record_events) CUDA_TRY(c, cudaEventRecord(c->ev[0], c->stream));
        rc = cg_onelaunch(c, U, eta, psi, kappa, r_min, max_iter);
        if (rc != WD_OK) return rc;
        if (record_events) CUDA_TRY(c, cudaEventRecord(c->ev[1], c->stream));
        CUDA_TRY(c, wd_fetch(c, c->sc_host, c->sc, sizeof(CgScalars)));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        const CgScalars &s1 = *c->sc_host;
        c->last_iters = s1.k;
        if (info) {
            info->iterations = s1.k;
            info->converged = s1.converged;
            info->rel_residual = s1.eta2 > 0.0 ? std::sqrt(s1.rr / s1.eta2) : 0.0;
            info->eta_norm2 = s1.eta2;
            float ms = 0.f;
            if (record_events) CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]));
            info->gpu_ms = ms;
            info->total_ms = ms;
            info->kernel_launches = c->launches;
            info->cg_mode = c->last_cg_mode;
        }
        return s1.converged ? WD_OK : (s1.breakdown ? WD_BREAKDOWN : WD_NOT_CONVERGED);
    }
    c->last_cg_mode = 1;
    const size_t n = spinor_vecs(c);
    const unsigned int vgrid = vec_grid(c, n);
    if (record_events) CUDA_TRY(c, cudaEventRecord(c->ev[0], c->stream));
    if (c->precision == 32)
        cg_init_kernel<float><<<vgrid, VEC_NT, 0, c->stream>>>((const float4 *)eta, (float4 *)c->y, (float4 *)c->r,
                                                               (float4 *)c->p, n, c->V, padded(c), c->sc, c->partials,
                                                               c->counter, c->hist, r_min, max_iter);
    else
        cg_init_kernel<double><<<vgrid, VEC_NT, 0, c->stream>>>((const double2 *)eta, (double2 *)c->y, (double2 *)c->r,
                                                                (double2 *)c->p, n, c->V, padded(c), c->sc, c->partials,
                                                                c->counter, c->hist, r_min, max_iter);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());

    const unsigned int ugrid = wd_vec_grid(c, n, WD_UPD_PER_SM);
    const int poll = c->poll > 0 ? c->poll : auto_poll(c);
    if (c->profile && c->pev_cap < 2 * poll) {   // two chunks of `poll` iterations are in flight at a time
        cudaEvent_t *pe = (cudaEvent_t *)realloc(c->pev, sizeof(cudaEvent_t) * 4 * (size_t)(2 * poll));
        if (!pe) return fail(c, WD_ERR_ALLOC, "cg_solve: out of host memory");
        c->pev = pe;
        for (; c->pev_cap < 2 * poll; ++c->pev_cap)
            for (int j = 0; j < 4; ++j) CUDA_TRY(c, cudaEventCreate(&c->pev[4 * c->pev_cap + j]));
    }
    // One chunk of `poll` iterations is always enqueued AHEAD of the one whose stop flag the host waits for
    // (wd_poll_loop).  The per-kernel profiling events come from a pool of two chunks, indexed like the poll mirrors.
    auto enqueue_chunk = [&](int first, int chunk, int pslot) -> int {
        cudaEvent_t *pev = c->profile ? c->pev + 4 * (size_t)pslot * poll : nullptr;
        for (int i = 0; i < chunk; ++i) {
            const int it = first + i;
            const bool sample = c->profile && (it % c->profile == 0);
            if (sample) CUDA_TRY(c, cudaEventRecord(pev[4 * i + 0], c->stream));
            // a2: q = D-dagger p, qq, alpha
            CUDA_TRY(c, (launch_dslash<1, MODE_QQ>(c, U, c->p, c->q, kappa, nullptr, it)));
            if (sample) CUDA_TRY(c, cudaEventRecord(pev[4 * i + 1], c->stream));
            // a3: r -= alpha D q, rr', beta, loop condition
            CUDA_TRY(c, (launch_dslash<0, MODE_RUPD>(c, U, c->q, nullptr, kappa, c->r, it)));
            if (sample) CUDA_TRY(c, cudaEventRecord(pev[4 * i + 2], c->stream));
            // a4: y += alpha p ; p = r + beta p
            if (c->precision == 32)
                cg_update_kernel<float><<<ugrid, VEC_NT, 0, c->stream>>>((float4 *)c->y, (float4 *)c->p, (const float4 *)c->r, n, c->sc, it);
            else
                cg_update_kernel<double><<<ugrid, VEC_NT, 0, c->stream>>>((double2 *)c->y, (double2 *)c->p, (const double2 *)c->r, n, c->sc, it);
            c->launches++;
            CUDA_TRY(c, cudaGetLastError());
            if (sample) CUDA_TRY(c, cudaEventRecord(pev[4 * i + 3], c->stream));
        }
        return WD_OK;
    };
    auto polled = [&](int first, int chunk, int pslot) -> int {
        if (!c->profile) return WD_OK;
        // only iterations that really ran (it < k_stop) count; over-launched ones are no-ops
        const cudaEvent_t *pev = c->pev + 4 * (size_t)pslot * poll;
        for (int i = 0; i < chunk && first + i < c->sc_host->k_stop; ++i) {
            if ((first + i) % c->profile != 0) continue;   // not sampled
            for (int j = 0; j < 3; ++j) {
                float ms = 0.f;
                CUDA_TRY(c, cudaEventElapsedTime(&ms, pev[4 * i + j], pev[4 * i + j + 1]));
                c->prof_ms[j] += ms;
            }
            c->prof_n++;
        }
        return WD_OK;
    };
    // look ahead only where a chunk of real iterations is long against the chunk of no-op launches it can cost at the end
    // of the solve (3 x poll launches of ~2.5 us): measured at 32^4 40.6 -> 39.8 ms per solve, at 4^4..14^4 a loss
    const bool ahead = (c->precision == 32 ? 1536.0 : 3072.0) * c->V / 6.0e12 >= 150.0e-6;
    rc = wd_poll_loop(c, max_iter, poll, ahead, enqueue_chunk, polled);
    if (rc != WD_OK) return rc;
    // a6: psi = D-dagger y ("then we multiply the solution by D-dagger")
    CUDA_TRY(c, (launch_dslash<1, MODE_PLAIN>(c, U, c->y, psi, kappa, nullptr, 0)));
    if (record_events) CUDA_TRY(c, cudaEventRecord(c->ev[1], c->stream));
    CUDA_TRY(c, wd_fetch(c, c->sc_host, c->sc, sizeof(CgScalars)));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    const CgScalars &s = *c->sc_host;
    c->last_iters = s.k;
    if (info) {
        info->iterations = s.k;
        info->converged = s.converged;
        info->rel_residual = s.eta2 > 0.0 ? std::sqrt(s.rr / s.eta2) : 0.0;
        info->eta_norm2 = s.eta2;
        float ms = 0.f;
        if (record_events) CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]));
        info->gpu_ms = ms;
        info->total_ms = ms;
        info->kernel_launches = c->launches;
        info->cg_mode = 1;
    }
    return s.converged ? WD_OK : (s.breakdown ? WD_BREAKDOWN : WD_NOT_CONVERGED);
}

static int check_cg_args(wd_ctx *c, const void *a, const void *b, const void *out, double kappa, double r_min,
                         int max_iter, const char *who)
{
    if (!a && !c->have_gauge) return fail(c, WD_ERR_ARG, "%s: NULL gauge field", who);
    if (!b || !out || b == out) return fail(c, WD_ERR_ARG, "%s: NULL argument or output aliases eta", who);
    if (!std::isfinite(kappa)) return fail(c, WD_ERR_ARG, "%s: kappa is not finite", who);
    if (!(r_min > 0.0) || !std::isfinite(r_min)) return fail(c, WD_ERR_ARG, "%s: r_min must be > 0", who);
    if (max_iter < 0) return fail(c, WD_ERR_ARG, "%s: max_iter < 0", who);
    return WD_OK;
}

extern "C" int cg_solve(wd_ctx *c, const void *U, const void *eta, void *psi, double kappa, double r_min, int max_iter,
                        wd_cg_info *info)
{
    if (!c) return WD_ERR_ARG;
    if (!U) return fail(c, WD_ERR_ARG, "cg_solve: NULL gauge field");
    int rc = check_cg_args(c, U, eta, psi, kappa, r_min, max_iter, "cg_solve");
    if (rc != WD_OK) return rc;
    c->launches = 0;
    return cg_device(c, U, eta, psi, kappa, r_min, max_iter, info, true);
}

// ---------------------------------------------------------------- f4: BiCGSTAB on D (reading B1)
template <int MODE>
static cudaError_t launch_dslash_bi(wd_ctx *c, const void *U, const void *in, void *out, double kappa, void *rhat, int it)
{
    DslashArgs a;
    a.g = make_geom(c, c->tile);
    a.sm_count = c->sm_count;
    a.stream = c->stream;
    a.U = U; a.Ub = U; a.in = in; a.cen = in; a.out = out; a.kappa = kappa; a.r = rhat;
    a.sc = c->sc; a.partials = c->partials; a.counter = c->counter; a.hist = hist_at(c, it); a.it = it;
    c->launches++;
    return c->precision == 32 ? launch_dslash_bi_f32(c->tile, MODE, a) : launch_dslash_bi_f64(c->tile, MODE, a);
}

template <typename real>
static int bicgstab_loop(wd_ctx *c, const void *U, const void *eta_, void *psi_, double kappa, double r_min, int max_iter)
{
    using svec = typename Field<real>::svec;
    const svec *eta = (const svec *)eta_;
    svec *psi = (svec *)psi_, *r = (svec *)c->r, *p = (svec *)c->p, *v = (svec *)c->q, *s = (svec *)c->y, *t = (svec *)c->w5;
    const size_t n = spinor_vecs(c);
    const unsigned int vgrid = vec_grid(c, n);
    bi_init_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>(eta, psi, r, p, n, c->V, padded(c), c->sc, c->partials, c->counter,
                                                         c->hist, r_min, max_iter);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    const int poll = c->poll > 0 ? c->poll : auto_poll(c);
    auto enqueue = [&](int first, int chunk, int) -> int {
        for (int i = 0; i < chunk; ++i) {
            const int it = first + i;
            if (c->profile && i == 0) CUDA_TRY(c, cudaEventRecord(c->bev[0], c->stream));
            // v = D p, <rhat,v>, alpha
            CUDA_TRY(c, (launch_dslash_bi<MODE_RV>(c, U, p, v, kappa, (void *)eta, it)));
            if (c->profile && i == 0) CUDA_TRY(c, cudaEventRecord(c->bev[1], c->stream));
            // s = r - alpha v
            bi_s_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>(s, r, v, n, c->V, padded(c), c->sc, it);
            if (c->profile && i == 0) CUDA_TRY(c, cudaEventRecord(c->bev[2], c->stream));
            // t = D s, <t,s>, <t,t>, omega
            CUDA_TRY(c, (launch_dslash_bi<MODE_TS>(c, U, s, t, kappa, nullptr, it)));
            if (c->profile && i == 0) CUDA_TRY(c, cudaEventRecord(c->bev[3], c->stream));
            // psi += alpha p + omega s ; r = s - omega t ; rho', rr, beta, loop test
            bi_xr_kernel<real><<<wd_vec_grid(c, n, WD_UPD_PER_SM), VEC_NT, 0, c->stream>>>(psi, r, p, s, t, eta, n, c->V, padded(c), c->sc, c->partials, c->counter,
                                                               hist_at(c, it), it);
            if (c->profile && i == 0) CUDA_TRY(c, cudaEventRecord(c->bev[4], c->stream));
            // p = r + beta (p - omega v)
            bi_p_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>(p, r, v, n, c->V, padded(c), c->sc, it);
            if (c->profile && i == 0) CUDA_TRY(c, cudaEventRecord(c->bev[5], c->stream));
            c->launches += 3;
            CUDA_TRY(c, cudaGetLastError());
        }
        return WD_OK;
    };
    auto polled = [&](int first, int, int) -> int {
        if (c->profile && first < c->sc_host->k_stop) {   // the first iteration of the chunk really ran
            for (int j = 0; j < 5; ++j) {
                float ms = 0.f;
                CUDA_TRY(c, cudaEventElapsedTime(&ms, c->bev[j], c->bev[j + 1]));
                c->bprof_ms[j] += ms;
            }
            c->bprof_n++;
        }
        return WD_OK;
    };
    // one chunk at a time: looking ahead measured no gain here (five launches per iteration make the over-launched
    // chunk at the end as expensive as the poll gaps it removes)
    int rc = wd_poll_loop(c, max_iter, poll, false, enqueue, polled);
    if (rc != WD_OK) return rc;
    return WD_OK;
}

extern "C" int bicgstab_solve(wd_ctx *c, const void *U, const void *eta, void *psi, double kappa, double r_min,
                              int max_iter, wd_cg_info *info)
{
    if (!c) return WD_ERR_ARG;
    if (!U) return fail(c, WD_ERR_ARG, "bicgstab_solve: NULL gauge field");
    int rc = check_cg_args(c, U, eta, psi, kappa, r_min, max_iter, "bicgstab_solve");
    if (rc != WD_OK) return rc;
    if (c->recon != 18) return fail(c, WD_ERR_ARG, "bicgstab_solve: compiled for 18-real links only (wd_set_gauge_recon)");
    rc = wd_ensure_workspace(c, max_iter);
    if (rc != WD_OK) return rc;
    if (!c->w5) {
        CUDA_TRY(c, cudaMalloc(&c->w5, spinor_bytes(c)));
        CUDA_TRY(c, cudaMemsetAsync(c->w5, 0, spinor_bytes(c), c->stream));
    }
    if (c->profile && !c->bev[0])
        for (int j = 0; j < 8; ++j) CUDA_TRY(c, cudaEventCreate(&c->bev[j]));
    c->launches = 0;
    CUDA_TRY(c, cudaEventRecord(c->ev[0], c->stream));
    rc = c->precision == 32 ? bicgstab_loop<float>(c, U, eta, psi, kappa, r_min, max_iter)
                            : bicgstab_loop<double>(c, U, eta, psi, kappa, r_min, max_iter);
    if (rc != WD_OK) return rc;
    CUDA_TRY(c, cudaEventRecord(c->ev[1], c->stream));
    CUDA_TRY(c, wd_fetch(c, c->sc_host, c->sc, sizeof(CgScalars)));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    const CgScalars &s = *c->sc_host;
    c->last_iters = s.k;
    if (info) {
        info->iterations = s.k;
        info->converged = s.converged;
        info->rel_residual = s.eta2 > 0.0 ? std::sqrt(s.rr / s.eta2) : 0.0;
        info->eta_norm2 = s.eta2;
        float ms = 0.f;
        CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]));
        info->gpu_ms = ms;
        info->total_ms = ms;
        info->kernel_launches = c->launches;
        info->cg_mode = 3;
    }
    return s.converged ? WD_OK : (s.breakdown ? WD_BREAKDOWN : WD_NOT_CONVERGED);
}

extern "C" int wd_get_profile_bicgstab(wd_ctx *c, double ms[5], long *iterations)
{
    if (!c || !ms || !iterations) return WD_ERR_ARG;
    for (int j = 0; j < 5; ++j) ms[j] = c->bprof_ms[j];
    *iterations = c->bprof_n;
    return WD_OK;
}

extern "C" int wd_get_profile_eo_bicgstab(wd_ctx *c, double ms[7], long *iterations)
{
    if (!c || !ms || !iterations) return WD_ERR_ARG;
    for (int j = 0; j < 7; ++j) ms[j] = c->bprof_ms[j];
    *iterations = c->bprof_n;
    return WD_OK;
}

/* rr after 0..k iterations of the last cg_solve on this ctx (device history copied to the host). */
extern "C" int wd_cg_history(wd_ctx *c, double *out, int n)
{
    if (!c || !out || n < 0) return WD_ERR_ARG;
    if (n > c->last_iters + 1) n = c->last_iters + 1;
    if (n > c->hist_cap) n = c->hist_cap;
    if (n > 0) {
        CUDA_TRY(c, cudaMemcpyAsync(out, c->hist, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    }
    return n;
}

// ---------------------------------------------------------------- host-buffer forms
static int ensure_staging(wd_ctx *c)
{
    if (!c->U_can) CUDA_TRY(c, cudaMalloc(&c->U_can, gauge_can_bytes(c)));
    if (!c->U_nat) CUDA_TRY(c, cudaMalloc(&c->U_nat, gauge_bytes(c)));
    if (!c->s_can) CUDA_TRY(c, cudaMalloc(&c->s_can, spinor_can_bytes(c)));
    if (!c->s_nat_in) CUDA_TRY(c, cudaMalloc(&c->s_nat_in, spinor_bytes(c)));
    if (!c->s_nat_out) CUDA_TRY(c, cudaMalloc(&c->s_nat_out, spinor_bytes(c)));
    return WD_OK;
}

// The host-buffer calls move their fields in WD_HOST_SLABS slabs of whole 16-site blocks on a second stream (copy_stream)
// while a third stream (pack_stream) packs the slab that has just landed (the ctx stream unpacks on the way back): the permutation kernels (about 2 ms for the 4 GB of
// config 4) hide behind the PCIe transfer instead of following it.  The solve itself needs all of U and eta, so the
// transfers as such cannot overlap it: the host-buffer form stays PCIe-bound (bench.py reports the measured rate beside it).
static int ensure_copy_stream(wd_ctx *c)
{
    if (!c->copy_stream) {
        CUDA_TRY(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        // The pack kernels get a stream of the LOWEST priority: when a second ctx iterates on a stream of higher priority
        // (split-phase calls, bench.py e2e), their CTAs are placed only where that solve leaves room
        int least = 0, greatest = 0;
        CUDA_TRY(c, cudaDeviceGetStreamPriorityRange(&least, &greatest));
        CUDA_TRY(c, cudaStreamCreateWithPriority(&c->pack_stream, cudaStreamNonBlocking, least));
        CUDA_TRY(c, cudaEventCreateWithFlags(&c->pack_ev, cudaEventDisableTiming));
        for (int i = 0; i < WD_HOST_SLABS + 1; ++i) CUDA_TRY(c, cudaEventCreateWithFlags(&c->slab_ev[i], cudaEventDisableTiming));
    }
    return WD_OK;
}

// sites [s0, s1) of slab i of n (whole blocks; the last slab takes the padded tail)
static inline void slab_range(const wd_ctx *c, int i, int n, int *s0, int *s1, int *s1_pad)
{
    const long nblk = (long)(vpad(c) / SB);
    const long b0 = nblk * i / n, b1 = nblk * (i + 1) / n;
    *s0 = (int)(b0 * SB);
    *s1_pad = (int)(b1 * SB);
    *s1 = *s1_pad < c->V ? *s1_pad : c->V;
}

template <typename real>
static int stage_inputs_t(wd_ctx *c, const void *U_host, const void *s_host)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    // the copy stream starts after everything already enqueued on the ctx stream (the staging buffers may be in use)
    CUDA_TRY(c, cudaEventRecord(c->slab_ev[WD_HOST_SLABS], c->stream));
    CUDA_TRY(c, cudaStreamWaitEvent(c->copy_stream, c->slab_ev[WD_HOST_SLABS], 0));
    CUDA_TRY(c, cudaStreamWaitEvent(c->pack_stream, c->slab_ev[WD_HOST_SLABS], 0));
    for (int pass = 0; pass < 2; ++pass) {
        if (pass == 0 && !U_host) continue;
        const size_t site_bytes = (pass == 0 ? 72 : 24) * sizeof(real);
        const char *src = (const char *)(pass == 0 ? U_host : s_host);
        char *dst = (char *)(pass == 0 ? c->U_can : c->s_can);
        for (int i = 0; i < WD_HOST_SLABS; ++i) {
            int s0, s1, s1p;
            slab_range(c, i, WD_HOST_SLABS, &s0, &s1, &s1p);
            if (s1 > s0)
                CUDA_TRY(c, cudaMemcpyAsync(dst + (size_t)s0 * site_bytes, src + (size_t)s0 * site_bytes,
                                            (size_t)(s1 - s0) * site_bytes, cudaMemcpyHostToDevice, c->copy_stream));
            CUDA_TRY(c, cudaEventRecord(c->slab_ev[i], c->copy_stream));
            CUDA_TRY(c, cudaStreamWaitEvent(c->pack_stream, c->slab_ev[i], 0));
            if (s1p <= s0) continue;
            const unsigned int grid = (unsigned int)((s1p - s0 + VEC_NT - 1) / VEC_NT);
            // sites s0 .. s1p - 1: the kernels take the end of the slab as their padded-volume bound
            if (pass == 0) {
                if (c->recon == 18)
                    pack_gauge_kernel<real, 18><<<grid, VEC_NT, 0, c->pack_stream>>>((const gvec *)c->U_can, (gvec *)c->U_nat, c->V, s1p, s0);
                else
                    pack_gauge_kernel<real, 12><<<grid, VEC_NT, 0, c->pack_stream>>>((const gvec *)c->U_can, (gvec *)c->U_nat, c->V, s1p, s0);
            } else {
                pack_spinor_kernel<real><<<grid, VEC_NT, 0, c->pack_stream>>>((const svec *)c->s_can, (svec *)c->s_nat_in, c->V, s1p, s0);
            }
            c->launches++;
        }
        if (pass == 0) c->have_gauge = 1;
    }
    CUDA_TRY(c, cudaGetLastError());
    // the ctx stream goes on when the last slab has been packed
    CUDA_TRY(c, cudaEventRecord(c->pack_ev, c->pack_stream));
    CUDA_TRY(c, cudaStreamWaitEvent(c->stream, c->pack_ev, 0));
    return WD_OK;
}

static int stage_inputs(wd_ctx *c, const void *U_host, const void *s_host)
{
    int rc = ensure_staging(c);
    if (rc != WD_OK) return rc;
    if ((rc = ensure_copy_stream(c)) != WD_OK) return rc;
    return c->precision == 32 ? stage_inputs_t<float>(c, U_host, s_host) : stage_inputs_t<double>(c, U_host, s_host);
}

template <typename real>
static int return_output_t(wd_ctx *c, void *out_host, bool sync)
{
    using svec = typename Field<real>::svec;
    const size_t site_bytes = 24 * sizeof(real);
    for (int i = 0; i < WD_HOST_SLABS; ++i) {
        int s0, s1, s1p;
        slab_range(c, i, WD_HOST_SLABS, &s0, &s1, &s1p);
        if (s1 > s0) {
            const unsigned int grid = (unsigned int)((s1 - s0 + VEC_NT - 1) / VEC_NT);
            unpack_spinor_kernel<real><<<grid, VEC_NT, 0, c->stream>>>((const svec *)c->s_nat_out, (svec *)c->s_can, s1, s0);
            c->launches++;
        }
        CUDA_TRY(c, cudaEventRecord(c->slab_ev[i], c->stream));
        CUDA_TRY(c, cudaStreamWaitEvent(c->copy_stream, c->slab_ev[i], 0));
        if (s1 > s0)
            CUDA_TRY(c, cudaMemcpyAsync((char *)out_host + (size_t)s0 * site_bytes, (const char *)c->s_can + (size_t)s0 * site_bytes,
                                        (size_t)(s1 - s0) * site_bytes, cudaMemcpyDeviceToHost, c->copy_stream));
    }
    CUDA_TRY(c, cudaGetLastError());
    // the ctx stream ends where the last copy ends (ev[3] closes the total_ms interval of cg_solve_host)
    CUDA_TRY(c, cudaEventRecord(c->slab_ev[WD_HOST_SLABS], c->copy_stream));
    CUDA_TRY(c, cudaStreamWaitEvent(c->stream, c->slab_ev[WD_HOST_SLABS], 0));
    CUDA_TRY(c, cudaEventRecord(c->ev[3], c->stream));
    if (sync) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return WD_OK;
}

static int return_output(wd_ctx *c, void *out_host, bool sync = true)
{
    return c->precision == 32 ? return_output_t<float>(c, out_host, sync) : return_output_t<double>(c, out_host, sync);
}

extern "C" int wd_apply_host(wd_ctx *c, const void *U_host, const void *psi_host, void *out_host, double kappa, int dagger)
{
    if (!c) return WD_ERR_ARG;
    if (!U_host && !c->have_gauge) return fail(c, WD_ERR_ARG, "wd_apply_host: NULL gauge field and none cached");
    if (!psi_host || !out_host || psi_host == out_host) return fail(c, WD_ERR_ARG, "wd_apply_host: NULL or aliased argument");
    if (!std::isfinite(kappa)) return fail(c, WD_ERR_ARG, "wd_apply_host: kappa is not finite");
    c->launches = 0;
    int rc = stage_inputs(c, U_host, psi_host);
    if (rc != WD_OK) return rc;
    rc = wd_apply(c, c->U_nat, c->s_nat_in, c->s_nat_out, kappa, dagger);
    if (rc != WD_OK) return rc;
    return return_output(c, out_host);
}

extern "C" int cg_solve_host(wd_ctx *c, const void *U_host, const void *eta_host, void *psi_host, double kappa,
                             double r_min, int max_iter, wd_cg_info *info)
{
    if (!c) return WD_ERR_ARG;
    int rc = check_cg_args(c, U_host, eta_host, psi_host, kappa, r_min, max_iter, "cg_solve_host");
    if (rc != WD_OK) return rc;
    c->launches = 0;
    CUDA_TRY(c, cudaEventRecord(c->ev[2], c->stream));
    rc = stage_inputs(c, U_host, eta_host);
    if (rc != WD_OK) return rc;
    const int status = cg_device(c, c->U_nat, c->s_nat_in, c->s_nat_out, kappa, r_min, max_iter, info, true);
    if (status < 0) return status;
    rc = return_output(c, psi_host);
    if (rc != WD_OK) return rc;
    if (info) {
        float ms = 0.f;
        CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[2], c->ev[3]));
        info->total_ms = ms;
        info->kernel_launches = c->launches;
    }
    return status;
}

// Split-phase form of cg_solve_host (include/wilson_cg.h): begin = enqueue the uploads, run = the solve and the enqueue of the
// download, wait = the download has landed.  With two contexts a caller overlaps the transfers of one solve with the
// iterations of another; every piece is the code of cg_solve_host.
extern "C" int cg_solve_host_begin(wd_ctx *c, const void *U_host, const void *eta_host)
{
    if (!c) return WD_ERR_ARG;
    if (!U_host && !c->have_gauge) return fail(c, WD_ERR_ARG, "cg_solve_host_begin: NULL gauge field and none cached");
    if (!eta_host) return fail(c, WD_ERR_ARG, "cg_solve_host_begin: NULL source");
    if (c->host_staged) return fail(c, WD_ERR_ARG, "cg_solve_host_begin: inputs are already staged (call cg_solve_host_run)");
    c->launches = 0;
    // device-ordered behind a download that may still be in flight (same streams): no host wait here
    const int rc = stage_inputs(c, U_host, eta_host);
    if (rc != WD_OK) return rc;
    c->host_staged = 1;
    return WD_OK;
}

extern "C" int cg_solve_host_run(wd_ctx *c, void *psi_host, double kappa, double r_min, int max_iter, wd_cg_info *info)
{
    if (!c) return WD_ERR_ARG;
    if (!c->host_staged) return fail(c, WD_ERR_ARG, "cg_solve_host_run: no inputs staged (call cg_solve_host_begin)");
    if (!psi_host) return fail(c, WD_ERR_ARG, "cg_solve_host_run: NULL output");
    if (!std::isfinite(kappa)) return fail(c, WD_ERR_ARG, "cg_solve_host_run: kappa is not finite");
    if (!(r_min > 0.0) || !std::isfinite(r_min)) return fail(c, WD_ERR_ARG, "cg_solve_host_run: r_min must be > 0");
    if (max_iter < 0) return fail(c, WD_ERR_ARG, "cg_solve_host_run: max_iter < 0");
    const int status = cg_device(c, c->U_nat, c->s_nat_in, c->s_nat_out, kappa, r_min, max_iter, info, true);
    c->host_staged = 0;   // consumed, also by a failed solve: the caller starts again from begin
    if (status < 0) return status;
    const int rc = return_output(c, psi_host, false);
    if (rc != WD_OK) return rc;
    c->host_out_pending = 1;
    if (info) {
        info->total_ms = info->gpu_ms;   // the transfers of a split-phase solve overlap other work: no per-call total
        info->kernel_launches = c->launches;   // pack kernels of begin + the solve + the unpack kernels
    }
    return status;
}

extern "C" int cg_solve_host_wait(wd_ctx *c)
{
    if (!c) return WD_ERR_ARG;
    if (!c->host_out_pending) return WD_OK;
    c->host_out_pending = 0;
    CUDA_TRY(c, cudaEventSynchronize(c->ev[3]));
    return WD_OK;
}

// wilson_ctx.cuh — the context record behind the opaque wd_ctx of include/wilson_cg.h and the small host helpers
// shared by the translation units that implement the C ABI (wilson_cg.cu, wilson_coo.cu).
#pragma once
#include "../../include/wilson_cg.h"
#include "wilson_launch.cuh"
#include "wilson_tma.cuh"

#include <cstdarg>
#include <cstdio>
#include <cstdlib>

#ifndef WD_HOST_SLABS
#define WD_HOST_SLABS 8   // slabs the host-buffer calls move their fields in (wilson_cg.cu, stage_inputs)
#endif

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
    int cg_mode;          // 0 = automatic, 1 = three kernels per iteration, 2 = one cooperative launch
    int coop_ok;          // device supports cooperative launches
    int last_cg_mode;     // what the last cg_solve used
    int zchunk_user;      // z layers per rasterisation chunk, 0 = automatic
    int small_tile_user;  // launch configuration of the one-launch CG kernel: -1 = automatic
    int stage_row;        // row of the shared-memory link pipeline (wilson_tma.cuh) used by wd_apply / cg_solve: -1 = off,
                          // -2 = automatic (fp64: the D-dagger / plain passes, where it measured 9 % faster; fp32: off)
    double l2_budget_mb;  // reuse-distance budget of the automatic choice
    int sm_count;
    // CG workspace (native layout), device
    void *r, *p, *q, *y;
    void *w5;             // fifth work vector (BiCGSTAB: t; even-odd: the odd-parity intermediate)
    void *w6;             // even-odd: etahat (half length)
    void *w7;             // even-odd BiCGSTAB: t = Mhat s (half length)
    double *eo_n2;        // even-odd: <eta_e,eta_e>, <eta_o,eta_o> (device)
    // multi-right-hand-side CG: r, p, q, y for a group of up to 4 sources, per-source scalars, counters, histories
    void *m_ws[4];
    size_t m_bytes;
    wd::CgScalars *m_sc, *m_sc_host;
    unsigned int *m_counter;
    double *m_hist;
    int m_hist_cap;
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
    wd::CgScalars *sc_poll;   // two pinned mirrors of sc: the poll of chunk k is read while chunk k+1 is already enqueued
    cudaEvent_t poll_ev[2];
    // staging of the *_host calls
    void *U_can, *U_nat, *s_can, *s_nat_in, *s_nat_out;
    int have_gauge;
    int host_staged;        // cg_solve_host_begin has staged inputs that no run has consumed yet
    int host_out_pending;   // cg_solve_host_run has enqueued the copy of psi to the host; cg_solve_host_wait has not been called
    cudaStream_t copy_stream;   // the *_host calls: transfers run here, slab by slab, beside the pack / unpack kernels
    cudaStream_t pack_stream;   // the pack kernels of the uploads: lowest priority, so that they fill gaps of another ctx's solve
    cudaEvent_t pack_ev;
    cudaEvent_t slab_ev[WD_HOST_SLABS + 1];
    cudaEvent_t ev[4];
    // per-kernel-class timing (wd_set_profile): 4 events per iteration of one poll chunk
    int profile;
    cudaEvent_t *pev;
    int pev_cap;            // iterations the pool covers
    double prof_ms[3];      // accumulated device time of a2, a3, a4
    long prof_n;            // iterations accumulated
    cudaEvent_t bev[8];     // BiCGSTAB / even-odd solvers: events around the 5 (7: even-odd BiCGSTAB) kernels of the first
                            // iteration of every poll chunk
    double bprof_ms[7];
    long bprof_n;
    // the arrays of the last wd_coo_assemble (wd_coo_spmv's sorted-row fast path), its violation flag and call counter
    const void *coo_val, *coo_row, *coo_col;
    unsigned int *coo_bad;
    unsigned int coo_epoch;
    int coo_fast;
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


// Device scalars -> pinned host mirror WITHOUT the copy engine.  A D2H memcpy of a few bytes queues behind every large
// download that any stream has in flight on the same engine: beside a continuous 4 GB download a 48^3x96 solve took 1860 ms
// instead of 364 (each poll waited for a whole copy), and in the pipelined host-buffer solves (cg_solve_host_begin / _run /
// _wait) the first polls of a solve waited for the previous solve's psi.  A one-warp kernel writes the mirror instead
// (pinned host memory is device-accessible under UVA; the writes are visible to the host once an event recorded behind
// the kernel has completed).
static __global__ void wd_scalars_to_host_kernel(const unsigned int *__restrict__ src, unsigned int *dst, int nwords)
{
    for (int i = threadIdx.x; i < nwords; i += blockDim.x) dst[i] = src[i];
}
static inline cudaError_t wd_fetch(wd_ctx *c, void *host_dst, const void *dev_src, size_t bytes)
{
    wd_scalars_to_host_kernel<<<1, 64, 0, c->stream>>>((const unsigned int *)dev_src, (unsigned int *)host_dst, (int)(bytes / 4));
    c->launches++;
    return cudaGetLastError();
}

// Host side of the device-resident solver loops (reading R1).  Iterations are enqueued in chunks of
// `poll`; after each chunk the device scalars are written to a pinned mirror (wd_fetch) and the host waits for that write to learn
// whether the loop condition has failed (k_stop).  With `ahead`, the NEXT chunk is enqueued before the host waits, so the
// stream never drains at a poll; kernels of iterations >= k_stop return at once, which makes the over-launch harmless.
//   enqueue(first_iteration, n_iterations, slot) -> WD_OK / error      slot in {0,1}: which of two event pools to use
//   polled(first_iteration, n_iterations, slot)  -> WD_OK / error      called after the chunk's scalars are in c->sc_host
template <typename Enqueue, typename Polled>
static inline int wd_poll_loop(wd_ctx *c, int max_iter, int poll, bool ahead, Enqueue enqueue, Polled polled)
{
    int launched = 0;      // iterations whose stop flag has been read back
    int enqueued = 0;      // iterations enqueued
    int slot = 0;          // pinned mirror / event the next chunk reports into
    auto report = [&](int sl) -> int {
        CUDA_TRY(c, wd_fetch(c, &c->sc_poll[sl], c->sc, sizeof(wd::CgScalars)));
        CUDA_TRY(c, cudaEventRecord(c->poll_ev[sl], c->stream));
        return WD_OK;
    };
    while (launched < max_iter) {
        const int chunk = (max_iter - launched) < poll ? (max_iter - launched) : poll;
        int rc;
        if (enqueued == launched) {   // nothing in flight for this chunk yet
            if ((rc = enqueue(launched, chunk, slot)) != WD_OK) return rc;
            enqueued = launched + chunk;
            if ((rc = report(slot)) != WD_OK) return rc;
        }
        const int wait_slot = slot;
        slot ^= 1;
        if (ahead && enqueued < max_iter) {   // the next chunk, before this one's flag is known
            const int next = (max_iter - enqueued) < poll ? (max_iter - enqueued) : poll;
            if ((rc = enqueue(enqueued, next, slot)) != WD_OK) return rc;
            enqueued += next;
            if ((rc = report(slot)) != WD_OK) return rc;
        }
        CUDA_TRY(c, cudaEventSynchronize(c->poll_ev[wait_slot]));
        *c->sc_host = c->sc_poll[wait_slot];
        if ((rc = polled(launched, chunk, wait_slot)) != WD_OK) return rc;
        launched += chunk;
        if (c->sc_host->k_stop <= launched) break;  // the device loop condition failed (or eta = 0)
    }
    return WD_OK;
}

// Grid of a streaming vector kernel over n 128-bit vectors: enough CTAs of VEC_NT threads to cover n, at most `per_sm` per SM
// (the kernels grid-stride beyond), divided over `parts` grid rows.  How many CTAs per SM stream fastest depends on the number of
// streams of the kernel (measured on B200 at 48^3x96, round 2): the kernels with five or more streams do best with 1024
// threads per SM -- cg_update (3 reads, 2 writes) 861 -> 783 us = 6.5 TB/s at 4 instead of 16 CTAs per SM (982 us at 2, 839 at 3,
// 842 at 5), fp64 163.5 -> 153.3 us at 32^4, the even-odd axpy 428 -> 389 us, bi_xr (5 reads, 2 writes) 1136 -> 1087 us --
// while the two- and three-stream kernels (bi_s, bi_p, the init kernels, norm2) are already at 6.3-6.7 TB/s with 16 and lose 2-6 %
// with fewer.  Fewer concurrent streams per SM keep more of each DRAM page's accesses together.
constexpr int WD_VEC_PER_SM = 16;    // two- and three-stream kernels
constexpr int WD_UPD_PER_SM = 4;     // cg_update, bi_xr
static inline unsigned int wd_vec_grid(const wd_ctx *c, size_t n, int per_sm, int parts = 1)
{
    const size_t need = (n + wd::VEC_NT - 1) / wd::VEC_NT;
    size_t cap = (size_t)c->sm_count * per_sm / parts;
    if (cap < 1) cap = 1;
    return (unsigned int)(need < cap ? (need ? need : 1) : cap);
}

// CG workspace of the ctx (r, p, q, y at full length, zeroed once; history of min(max_iter, WD_HIST_MAX) + 1 doubles);
// wilson_cg.cu
int wd_ensure_workspace(wd_ctx *c, int max_iter);

// The residual history is a measurement aid, not part of the method: its length is capped so that max_iter = INT_MAX
// ("no limit") neither overflows max_iter + 1 nor asks for gigabytes.  Iterations beyond the cap are not recorded: the
// host passes a NULL history to their launches (hist_at) and to a one-launch solve that could outrun it (hist_whole).
constexpr int WD_HIST_MAX = 1 << 20;
static inline int hist_len(int max_iter) { return (max_iter < WD_HIST_MAX ? max_iter : WD_HIST_MAX) + 1; }
static inline double *hist_at(const wd_ctx *c, int it) { return (long)it + 1 < (long)c->hist_cap ? c->hist : nullptr; }
static inline double *hist_whole(const wd_ctx *c, int max_iter) { return (long)max_iter + 1 <= (long)c->hist_cap ? c->hist : nullptr; }

// ---------------------------------------------------------------- geometry helpers shared by the ABI translation units
static inline wd::FastDiv make_fastdiv(unsigned int d)
{
    wd::FastDiv f;
    f.d = d;
    if (d <= 1) { f.d = 1; f.M = 0; f.sh = -1; return f; }
    int s = 0;
    while ((1u << s) < d) ++s;                       // s = ceil(log2 d) >= 1
    const unsigned long long p2 = 1ull << (31 + s);
    f.M = (unsigned int)((p2 + d - 1) / d);          // in [2^31, 2^32)
    f.sh = s - 1;                                    // (n*M) >> (31+s) = umulhi(n,M) >> (s-1)
    return f;
}

// Launch geometry of a lattice of extents `dims` (the real lattice, or one parity of it with dims[0] = Lx/2) tiled
// by tb.  z chunk of the CTA rasterisation: the largest divisor of the z tile count whose t-reuse distance
// Lx*Ly*(zc*BZ)*BT sites * ~600 B (spinor in/out, gauge, halos) stays within the L2 budget.
static inline wd::Geom make_geom_lattice(const int dims[4], int bc_t, const int tb[4], int zchunk_user, double l2_budget_mb)
{
    wd::Geom g;
    long vol = 1;
    for (int d = 0; d < 4; ++d) {
        g.L[d] = dims[d];
        g.nt[d] = (dims[d] + tb[d] - 1) / tb[d];
        vol *= dims[d];
    }
    g.V = (int)vol;
    g.bc_t = bc_t;
    g.eo = 0;
    g.par = 0;
    const double layer = 600.0 * dims[0] * dims[1] * tb[3];   // bytes per z layer of one t-tile row
    const double budget = l2_budget_mb * 1.0e6;
    int zc = 1;
    if (zchunk_user > 0) {
        zc = (zchunk_user + tb[2] - 1) / tb[2];
        if (zc > g.nt[2]) zc = g.nt[2];
    } else {
        for (int d = 1; d <= g.nt[2]; ++d)
            if (g.nt[2] % d == 0 && layer * d * tb[2] <= budget) zc = d;
    }
    g.zc = zc;
    g.ntiles = g.nt[0] * g.nt[1] * g.nt[2] * g.nt[3];
    g.d_chunk = make_fastdiv((unsigned)(g.nt[0] * g.nt[1] * g.zc * g.nt[3]));
    g.d_nt0 = make_fastdiv((unsigned)g.nt[0]);
    g.d_nt1 = make_fastdiv((unsigned)g.nt[1]);
    g.d_zc = make_fastdiv((unsigned)g.zc);
    const int zlast = g.nt[2] % g.zc ? g.nt[2] % g.zc : g.zc;
    g.d_zlast = make_fastdiv((unsigned)zlast);
    return g;
}
static inline wd::Geom make_geom_dims(const wd_ctx *c, const int tb[4], int zchunk_user)
{
    return make_geom_lattice(c->dims, c->bc_t, tb, zchunk_user, c->l2_budget_mb);
}
static inline wd::Geom make_geom(const wd_ctx *c, int tile) { return make_geom_dims(c, wd::kTiles[tile].b, c->zchunk_user); }

static inline long tile_blocks_dims(const int dims[4], int tile)
{
    long n = 1;
    for (int d = 0; d < 4; ++d) n *= (dims[d] + wd::kTiles[tile].b[d] - 1) / wd::kTiles[tile].b[d];
    return n;
}
static inline long tile_blocks(const wd_ctx *c, int tile) { return tile_blocks_dims(c->dims, tile); }
static inline int tile_threads(int tile)
{
    return wd::kTiles[tile].b[0] * wd::kTiles[tile].b[1] * wd::kTiles[tile].b[2] * wd::kTiles[tile].b[3];
}
static inline bool tile_ok(const wd_ctx *c, int tile)
{
    if (tile < 0 || tile >= WD_NUM_TILES) return false;
    return c->precision == 64 ? wd::kTiles[tile].f64 != 0 : wd::kTiles[tile].f32 != 0;
}
// Automatic choice: the first row of the table (rows are in order of measured preference) among those compiled
// for this precision that waste the fewest threads on tiles overhanging the lattice `dims`.
static inline int auto_tile_dims(const wd_ctx *c, const int dims[4])
{
    int best = -1;
    double best_waste = 1e300, vol = 1.0;
    for (int d = 0; d < 4; ++d) vol *= dims[d];
    for (int t = 0; t < WD_NUM_TILES; ++t) {
        if (!tile_ok(c, t)) continue;
        const double waste = (double)tile_blocks_dims(dims, t) * tile_threads(t) / vol;
        if (waste < best_waste - 1e-12) { best_waste = waste; best = t; }
    }
    return best;
}
static inline int auto_tile(const wd_ctx *c) { return auto_tile_dims(c, c->dims); }

// The staged stencil (wilson_tma.cuh) covers: plain lattice, 18 reals per link, the row compiled for the precision, Lx a
// multiple of the 16-site block and every other extent a multiple of the row's tile edge (whole tiles only).
static inline bool stage_row_ok(const wd_ctx *c, int row)
{
    if (row < 0 || row >= WD_NUM_TMA_ROWS || c->recon != 18) return false;
    const wd::TmaRowInfo &t = wd::kTmaRows[row];
    if (!(c->precision == 64 ? t.f64 : t.f32)) return false;
    for (int d = 0; d < 4; ++d)
        if (c->dims[d] % t.b[d] != 0) return false;
    return true;
}
// row the pass of the given mode runs on, or -1 = links through L1
static inline int stage_row_for(const wd_ctx *c, int mode)
{
    if (c->stage_row >= 0) return stage_row_ok(c, c->stage_row) ? c->stage_row : -1;
    if (c->stage_row == -2 && c->precision == 64 && mode != wd::MODE_RUPD && stage_row_ok(c, WD_TMA_AUTO_ROW_F64))
        return WD_TMA_AUTO_ROW_F64;
    return -1;
}

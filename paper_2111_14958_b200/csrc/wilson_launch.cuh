// wilson_launch.cuh — the table of compiled stencil launch configurations and the per-precision launchers.
// A "tile" (the name of the C ABI, wd_set_tile) is one row: CTA tile BX x BY x BZ x BT (threads per CTA =
// product) and MINB = minimum resident CTAs per SM asked of ptxas (bounds registers per thread).  Every row runs the
// software-pipelined hop loop (two register buffers, diagonal term first where the pass allows it).  This is the CUDA
// analogue of the paper's workgroup-size knob.  F32 / F64 = 1 if the row is compiled for that precision.
// Rows measured and retired in round 1 (unpipelined, three buffers, cp.async-staged forward links, 64-thread and 4-site-run
// tiles that never won: DESIGN.md section 6) are no longer compiled.
#pragma once
#include "wilson_kernels.cuh"

// Rows are in order of preference (measured on B200, profiles/): the automatic choice takes the first row
// with the fewest padded threads for the lattice and precision at hand.
//   X(index, BX, BY, BZ, BT, MINB, F32, F64)
#define WD_TILE_TABLE(X) \
    X(0, 16, 2, 2, 2, 4, 1, 0) \
    X(1, 16, 4, 4, 2, 1, 1, 0) \
    X(2, 32, 2, 2, 1, 4, 1, 0) \
    X(3, 8, 4, 2, 2, 4, 1, 0) \
    X(4, 32, 2, 2, 1, 2, 0, 1) \
    X(5, 16, 2, 2, 1, 3, 0, 1) \
    X(6, 16, 2, 2, 2, 2, 0, 1) \
    X(7, 8, 4, 2, 1, 4, 0, 1) \
    X(8, 4, 4, 2, 2, 4, 1, 1)
#define WD_NUM_TILES 9

// Launch configurations of the one-launch CG kernel (small volumes): 64- and 128-thread tiles,
// no register bound (ptxas then hoists the loads of all 8 hops: one memory round trip per site instead of 8,
// which is what matters when the lattice lives in L2 and there are few warps per SM).
//   Y(index, BX, BY, BZ, BT, MINB, PIPE)
#define WD_SMALL_TABLE(Y)  \
    Y(0, 4, 4, 2, 2, 1, 0) \
    Y(1, 8, 4, 2, 1, 1, 0) \
    Y(2, 16, 2, 2, 1, 1, 0) \
    Y(3, 16, 2, 2, 2, 1, 0) \
    Y(4, 8, 4, 2, 2, 1, 0) \
    Y(5, 16, 2, 2, 1, 5, 0) \
    Y(6, 16, 2, 2, 2, 3, 0) \
    Y(7, 8, 4, 2, 1, 5, 0) \
    Y(8, 4, 4, 2, 2, 5, 0) \
    Y(9, 16, 2, 2, 1, 6, 1) \
    Y(10, 16, 2, 2, 2, 4, 1)
#define WD_NUM_SMALL_TILES 11

namespace wd {

struct TileInfo {
    int b[4];
    int minb, f32, f64;
};
static const TileInfo kTiles[WD_NUM_TILES] = {
#define X(i, a, b, c, d, m, f32, f64) {{a, b, c, d}, m, f32, f64},
    WD_TILE_TABLE(X)
#undef X
};

static const int kSmallTiles[WD_NUM_SMALL_TILES][4] = {
#define Y(i, a, b, c, d, m, p) {a, b, c, d},
    WD_SMALL_TABLE(Y)
#undef Y
};
// register bound (MINB) of each row, and its measured relative cost per round of tiles (B200, 4^4 ... 20^4, both
// precisions): 128-thread CTAs with x runs of 16 sites are the cheapest, 4-site x runs and the
// register-bounded / pipelined rows the dearest
static const int kSmallMinb[WD_NUM_SMALL_TILES] = {
#define Y(i, a, b, c, d, m, p) m,
    WD_SMALL_TABLE(Y)
#undef Y
};
static const double kSmallCost[WD_NUM_SMALL_TILES] = {1.10, 1.00, 1.00, 0.93, 1.02, 1.25, 1.19, 1.25, 1.40, 1.90, 1.93};

struct CgOneLaunchArgs {
    Geom g;            // nt / ntiles / fast-division constants for the chosen small tile
    int sm_count;
    cudaStream_t stream;
    const void *U;
    const void *eta;
    void *y, *r, *p, *q, *psi;
    double kappa;
    CgScalars *sc;
    double *partials;  // 3 * grid doubles
    size_t partials_cap;
    double *hist;
    double r_min;
    int max_iter;
};
cudaError_t launch_cg_onelaunch_f32(int small_tile, const CgOneLaunchArgs &a);
cudaError_t launch_cg_onelaunch_f64(int small_tile, const CgOneLaunchArgs &a);

struct DslashArgs {
    Geom g;
    int sm_count;
    cudaStream_t stream;
    const void *U;
    const void *Ub;   // links read by the backward hops: U itself on a plain lattice, the other parity's with even-odd
    const void *in;
    const void *cen;  // field of the diagonal term: `in` on a plain lattice; nullptr = none
    void *out;
    double kappa;     // out = cen - kappa * (hopping sum)
    void *r;
    CgScalars *sc;
    double *partials;
    unsigned int *counter;
    double *hist;
    int it;
};

// dagger in {0,1}; mode in {MODE_PLAIN, MODE_QQ (dagger = 1 only), MODE_RUPD (dagger = 0 only)}
cudaError_t launch_dslash_f32(int tile, int dagger, int mode, const DslashArgs &a);
cudaError_t launch_dslash_f64(int tile, int dagger, int mode, const DslashArgs &a);
// the same with 12-real link storage (wd_set_gauge_recon(ctx, 12))
cudaError_t launch_dslash12_f32(int tile, int dagger, int mode, const DslashArgs &a);
cudaError_t launch_dslash12_f64(int tile, int dagger, int mode, const DslashArgs &a);
// one parity of the lattice (even-odd preconditioning; a.g.eo = 1)
cudaError_t launch_dslash_eo_f32(int tile, int dagger, int mode, const DslashArgs &a);
cudaError_t launch_dslash_eo_f64(int tile, int dagger, int mode, const DslashArgs &a);
// one parity with 12-real links; mode in {MODE_PLAIN, MODE_QQ, MODE_RUPD, MODE_RV, MODE_TS}
cudaError_t launch_dslash12_eo_f32(int tile, int dagger, int mode, const DslashArgs &a);
cudaError_t launch_dslash12_eo_f64(int tile, int dagger, int mode, const DslashArgs &a);
// BiCGSTAB passes (D only): mode in {MODE_RV, MODE_TS}
cudaError_t launch_dslash_bi_f32(int tile, int mode, const DslashArgs &a);
cudaError_t launch_dslash_bi_f64(int tile, int mode, const DslashArgs &a);
// the same on one parity of the lattice (even-odd preconditioned BiCGSTAB)
cudaError_t launch_dslash_eo_bi_f32(int tile, int mode, const DslashArgs &a);
cudaError_t launch_dslash_eo_bi_f64(int tile, int mode, const DslashArgs &a);

template <typename real, int DAG, int MODE, int RECON = 18, int EO = 0>
static cudaError_t launch_dslash_tile(int tile, const DslashArgs &a)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    switch (tile) {
#define X(i, bx, by, bz, bt, m, f32, f64)                                                                      \
    case i:                                                                                                    \
        if constexpr (sizeof(real) == 4 ? f32 : f64) {                                                         \
            auto kern = dslash_kernel<real, DAG, MODE, bx, by, bz, bt, m, RECON, EO>;                          \
            static int occ_tab[WD_MAXDEV];                                                                     \
            int occ = 0;                                                                                       \
            cudaError_t e = cached_occupancy(occ_tab, kern, bx * by * bz * bt, 0, &occ);                       \
            if (e != cudaSuccess) return e;                                                                    \
            long grid = (long)occ * a.sm_count;                                                                \
            if (grid > a.g.ntiles) grid = a.g.ntiles;                                                          \
            kern<<<(unsigned)grid, bx * by * bz * bt, 0, a.stream>>>(                                          \
                a.g, (const gvec *)a.U, (const gvec *)a.Ub, (const svec *)a.in, (const svec *)a.cen, (svec *)a.out, \
                (real)a.kappa, (svec *)a.r, a.sc, a.partials, a.counter, a.hist, a.it);                        \
            return cudaGetLastError();                                                                         \
        }                                                                                                      \
        return cudaErrorInvalidValue;
        WD_TILE_TABLE(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

template <typename real>
static cudaError_t launch_cg_onelaunch_any(int small_tile, const CgOneLaunchArgs &a)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    switch (small_tile) {
#define Y(i, bx, by, bz, bt, mb_, pi_)                                                                           \
    case i: {                                                                                                  \
        auto kern = cg_onelaunch_kernel<real, bx, by, bz, bt, mb_, pi_>;                                      \
        static int occ_tab[WD_MAXDEV];                                                                         \
        int occ = 0;                                                                                           \
        {                                                                                                      \
            cudaError_t e = cached_occupancy(occ_tab, kern, bx * by * bz * bt, 0, &occ);                       \
            if (e != cudaSuccess) return e;                                                                    \
        }                                                                                                      \
        long grid = (long)occ * a.sm_count;            /* all CTAs must be co-resident (grid barrier) */       \
        if (grid > a.g.ntiles) grid = a.g.ntiles;                                                              \
        if ((size_t)(3 * grid) > a.partials_cap) return cudaErrorInvalidValue;                                 \
        Geom g = a.g;                                                                                          \
        const gvec *U = (const gvec *)a.U;                                                                     \
        const svec *eta = (const svec *)a.eta;                                                                 \
        svec *y = (svec *)a.y, *r = (svec *)a.r, *pp = (svec *)a.p, *q = (svec *)a.q, *psi = (svec *)a.psi;    \
        real kappa = (real)a.kappa;                                                                            \
        CgScalars *sc = a.sc;                                                                                  \
        double *partials = a.partials, *hist = a.hist;                                                         \
        double r_min = a.r_min;                                                                                \
        int max_iter = a.max_iter;                                                                             \
        void *args[] = {&g, &U, &eta, &y, &r, &pp, &q, &psi, &kappa, &sc, &partials, &hist, &r_min, &max_iter}; \
        return cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)grid), dim3(bx * by * bz * bt),  \
                                           args, 0, a.stream);                                                 \
    }
        WD_SMALL_TABLE(Y)
#undef Y
        default: return cudaErrorInvalidValue;
    }
}

template <typename real, int RECON = 18, int EO = 0>
static cudaError_t launch_dslash_any(int tile, int dagger, int mode, const DslashArgs &a)
{
    if (mode == MODE_PLAIN)
        return dagger ? launch_dslash_tile<real, 1, MODE_PLAIN, RECON, EO>(tile, a)
                      : launch_dslash_tile<real, 0, MODE_PLAIN, RECON, EO>(tile, a);
    if (mode == MODE_QQ && dagger) return launch_dslash_tile<real, 1, MODE_QQ, RECON, EO>(tile, a);
    if (mode == MODE_RUPD && !dagger) return launch_dslash_tile<real, 0, MODE_RUPD, RECON, EO>(tile, a);
    return cudaErrorInvalidValue;
}

}  // namespace wd

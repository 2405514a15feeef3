// wilson_mrhs.cuh — the stencil and CG kernels for several right-hand sides at once ("multi-right-
// hand-side dslash (amortises the 288 B/site gauge read)").
//
// One thread per (site, right-hand side): a CTA owns a BX x BY x BZ x BT tile of sites for NRHS sources, thread
// t = rhs * NS + site-in-tile, so a warp is uniform in rhs and the NRHS warps that own the same 32 sites issue the
// same link loads at about the same time: the first one misses, the others hit L1 (or merge with the miss in
// flight).  Links cross DRAM -> L2 -> L1 once per NRHS sources; the per-thread code is exactly that of the
// single-source kernel (hopping_sum).  The sources are independent CG problems: every right-hand side has its own
// alpha, beta, rr, loop test and stop iteration (CgScalars sc[NRHS]); a source whose loop has ended is skipped
// warp by warp while the others go on.
#pragma once
#include "wilson_kernels.cuh"

namespace wd {

// fields of the NRHS sources are NRHS native spinors at a constant stride (in 128-bit vectors)
template <typename real, int DAG, int MODE, int BX, int BY, int BZ, int BT, int NRHS, int MINB>
__global__ void __launch_bounds__(BX *BY *BZ *BT *NRHS, MINB)
dslash_mrhs_kernel(const Geom g, const typename Field<real>::gvec *__restrict__ U,
                   const typename Field<real>::svec *__restrict__ in, typename Field<real>::svec *out, size_t stride,
                   real kappa, typename Field<real>::svec *r, CgScalars *sc, double *partials, unsigned int *counter,
                   double *hist, int hist_stride, int it)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    constexpr int NS = BX * BY * BZ * BT;
    constexpr int NT = NS * NRHS;
    static_assert(NS % 32 == 0, "a warp must be uniform in the right-hand side");
    const int tid = threadIdx.x;
    const int rhs = tid / NS, st = tid - rhs * NS;
    const int lx = st % BX, ly = (st / BX) % BY, lz = (st / (BX * BY)) % BZ, lt = st / (BX * BY * BZ);
    // live: this source still iterates (always true for a plain pass)
    const bool live = (MODE == MODE_PLAIN) || (it < sc[rhs].k_stop);
    if (MODE != MODE_PLAIN) {
        bool any = false;
#pragma unroll
        for (int j = 0; j < NRHS; ++j) any = any || (it < sc[j].k_stop);
        if (!any) return;   // uniform over the grid
    }
    in += (size_t)rhs * stride;
    if (MODE != MODE_RUPD) out += (size_t)rhs * stride;
    if (MODE == MODE_RUPD) r += (size_t)rhs * stride;
    const real alpha = (MODE == MODE_RUPD) ? (real)sc[rhs].alpha : (real)0;
    double local = 0.0;
    // No barrier between tiles: keeping the warps of the different sources in step with a __syncthreads per tile was
    // measured slower (a2/a3 1048/1041 us per source against 966/975 at 48^3x96, 4 sources).
    for (int b = blockIdx.x; b < g.ntiles; b += gridDim.x) {
        int tx, ty, tz, tt;
        tile_of_block(g, b, tx, ty, tz, tt);
        const int x = tx * BX + lx, y = ty * BY + ly, z = tz * BZ + lz, t = tt * BT + lt;
        if (!live || x >= g.L[0] || y >= g.L[1] || z >= g.L[2] || t >= g.L[3]) continue;
        const int s = x + g.L[0] * (y + g.L[1] * (z + g.L[2] * t));
        real acc[24], c[24], rv[24];
        constexpr bool CF = MODE != MODE_RUPD;   // diagonal term first, as in dslash_kernel
        hopping_sum<DAG, 1, MODE == MODE_RUPD, true, real, svec, gvec, 18, 0, CF>(g, U, U, in, in, r, x, y, z, t, s,
                                                                               acc, c, rv, kappa);
#pragma unroll
        for (int i = 0; i < 24; ++i) c[i] = CF ? acc[i] : fma(-kappa, acc[i], c[i]);
        if (MODE == MODE_RUPD) {
            real n2 = 0;
#pragma unroll
            for (int i = 0; i < 24; ++i) {
                rv[i] = fma(-alpha, c[i], rv[i]);
                n2 = fma(rv[i], rv[i], n2);
            }
            store_spinor(r, s, rv);
            local += (double)n2;
        } else {
            store_spinor(out, s, c);
            if (MODE == MODE_QQ) {
                real n2 = 0;
#pragma unroll
                for (int i = 0; i < 24; ++i) n2 = fma(c[i], c[i], n2);
                local += (double)n2;
            }
        }
    }
    if (MODE != MODE_PLAIN) {
        double v[NRHS], tot[NRHS];
#pragma unroll
        for (int j = 0; j < NRHS; ++j) v[j] = (j == rhs) ? local : 0.0;
        if (grid_sum_n<NT, NRHS>(v, partials, counter, tot)) {
#pragma unroll
            for (int j = 0; j < NRHS; ++j)
                if (it < sc[j].k_stop) {
                    if (MODE == MODE_QQ) finish_qq(sc + j, tot[j]);
                    else finish_rr(sc + j, tot[j], it, hist ? hist + (size_t)j * hist_stride : nullptr);
                }
        }
    }
}

// a1 / a4 for NRHS sources: gridDim.y = NRHS, blockIdx.y selects the source (fields at `stride`, scalars sc[y],
// reduction scratch partials + y * gridDim.x and counter + y)
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
cg_init_mrhs_kernel(const typename Field<real>::svec *__restrict__ eta, typename Field<real>::svec *y,
                    typename Field<real>::svec *r, typename Field<real>::svec *p, size_t n, size_t stride, int V,
                    int padded, CgScalars *sc, double *partials, unsigned int *counter, double *hist, int hist_stride,
                    double r_min, int max_iter)
{
    using svec = typename Field<real>::svec;
    const size_t off = (size_t)blockIdx.y * stride;
    eta += off; y += off; r += off; p += off;
    sc += blockIdx.y;
    double local = 0.0;
    for (size_t i = (size_t)blockIdx.x * VEC_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * VEC_NT) {
        const svec e = real_site<Field<real>::NSP>(i, V, padded) ? __ldg(eta + i) : svec();
        y[i] = vzero(e);
        r[i] = e;
        p[i] = e;
        local += vnorm2<svec>(e);
    }
    double total;
    if (grid_sum<VEC_NT>(local, partials + (size_t)blockIdx.y * gridDim.x, counter + blockIdx.y, &total)) {
        sc->rr = total; sc->eta2 = total; sc->qq = 0.0; sc->alpha = 0.0; sc->beta = 0.0;
        sc->r_min = r_min; sc->k = 0; sc->max_iter = max_iter;
        loop_begin(sc, total, total, r_min, max_iter);
        if (hist) hist[(size_t)blockIdx.y * hist_stride] = total;
    }
}

template <typename real>
__global__ void __launch_bounds__(VEC_NT)
cg_update_mrhs_kernel(typename Field<real>::svec *y, typename Field<real>::svec *p,
                      const typename Field<real>::svec *__restrict__ r, size_t n, size_t stride, const CgScalars *sc,
                      int it)
{
    sc += blockIdx.y;
    if (it >= sc->k_stop) return;
    const size_t off = (size_t)blockIdx.y * stride;
    y += off; p += off; r += off;
    const real alpha = (real)sc->alpha, beta = (real)sc->beta;
    for (size_t i = (size_t)blockIdx.x * VEC_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * VEC_NT) {
        const typename Field<real>::svec pv = p[i];
        const typename Field<real>::svec rv = __ldg(r + i);
        y[i] = vaxpy(alpha, pv, y[i]);
        p[i] = vaxpy(beta, pv, rv);
    }
}

// launch configurations of the multi-source stencil: site tile x NRHS threads
//   M(index, BX, BY, BZ, BT)
#define WD_MRHS_TABLE(M) \
    M(0, 16, 2, 2, 2)    \
    M(1, 16, 2, 2, 1)    \
    M(2, 8, 4, 2, 2)     \
    M(3, 8, 4, 2, 1)
#define WD_NUM_MRHS_TILES 4
static const int kMrhsTiles[WD_NUM_MRHS_TILES][4] = {
#define M(i, a, b, c, d) {a, b, c, d},
    WD_MRHS_TABLE(M)
#undef M
};

struct MrhsArgs {
    Geom g;
    int sm_count;
    cudaStream_t stream;
    const void *U, *in;
    void *out, *r;
    size_t stride;     // in 128-bit vectors
    double kappa;
    CgScalars *sc;
    double *partials;
    unsigned int *counter;
    double *hist;
    int hist_stride;
    int it;
};
// nrhs in {2, 4}; dagger / mode as launch_dslash_*
cudaError_t launch_mrhs_f32(int tile, int nrhs, int dagger, int mode, const MrhsArgs &a);
cudaError_t launch_mrhs_f64(int tile, int nrhs, int dagger, int mode, const MrhsArgs &a);

template <typename real, int DAG, int MODE, int NRHS>
static cudaError_t launch_mrhs_tile(int tile, const MrhsArgs &a)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    switch (tile) {
#define M(i, bx, by, bz, bt)                                                                                       \
    case i: {                                                                                                      \
        constexpr int nt = bx * by * bz * bt * NRHS;                                                               \
        constexpr int per_sm = sizeof(real) == 4 ? 512 : 256;   /* threads per SM the register file allows */      \
        constexpr int minb = per_sm / nt > 0 ? per_sm / nt : 1;                                                    \
        if constexpr (nt <= per_sm) {                                                                              \
            auto kern = dslash_mrhs_kernel<real, DAG, MODE, bx, by, bz, bt, NRHS, minb>;                           \
            static int occ_tab[WD_MAXDEV];                                                                     \
            int occ = 0;                                                                                       \
            {                                                                                                  \
                cudaError_t e = cached_occupancy(occ_tab, kern, nt, 0, &occ);                                  \
                if (e != cudaSuccess) return e;                                                                \
            }                                                                                                  \
            long grid = (long)occ * a.sm_count;                                                                    \
            if (grid > a.g.ntiles) grid = a.g.ntiles;                                                              \
            kern<<<(unsigned)grid, nt, 0, a.stream>>>(a.g, (const gvec *)a.U, (const svec *)a.in, (svec *)a.out,   \
                                                      a.stride, (real)a.kappa, (svec *)a.r, a.sc, a.partials,      \
                                                      a.counter, a.hist, a.hist_stride, a.it);                     \
            return cudaGetLastError();                                                                             \
        }                                                                                                          \
        return cudaErrorInvalidValue;                                                                              \
    }
        WD_MRHS_TABLE(M)
#undef M
        default: return cudaErrorInvalidValue;
    }
}

template <typename real, int NRHS>
static cudaError_t launch_mrhs_modes(int tile, int dagger, int mode, const MrhsArgs &a)
{
    if (mode == MODE_PLAIN)
        return dagger ? launch_mrhs_tile<real, 1, MODE_PLAIN, NRHS>(tile, a) : launch_mrhs_tile<real, 0, MODE_PLAIN, NRHS>(tile, a);
    if (mode == MODE_QQ && dagger) return launch_mrhs_tile<real, 1, MODE_QQ, NRHS>(tile, a);
    if (mode == MODE_RUPD && !dagger) return launch_mrhs_tile<real, 0, MODE_RUPD, NRHS>(tile, a);
    return cudaErrorInvalidValue;
}
template <typename real>
static cudaError_t launch_mrhs_any(int tile, int nrhs, int dagger, int mode, const MrhsArgs &a)
{
    if (nrhs == 2) return launch_mrhs_modes<real, 2>(tile, dagger, mode, a);
    if (nrhs == 4) return launch_mrhs_modes<real, 4>(tile, dagger, mode, a);
    return cudaErrorInvalidValue;
}

}  // namespace wd

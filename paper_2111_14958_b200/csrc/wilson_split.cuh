// wilson_split.cuh — the one-launch CG of SURVEY.md 8(f1) with the hopping sum of a site SPLIT OVER FOUR WARPS.
//
// On the paper's own volumes (4^4 ... 14^4) there are 256 ... 38 416 sites for 148 SMs: with one thread per
// site (cg_onelaunch_kernel) an SM holds 2-8 warps, each of which walks the whole eight-hop chain (~1300 instructions,
// 94 loads) by itself, and the iteration time is that serial chain.  Here a CTA is 32 sites x 4
// directions: warp mu computes the two hops (forward and backward) of direction mu for the CTA's 32 sites, the four
// partial sums meet in shared memory, and the per-site tail of the phase (diagonal term, CG update, norm) is spread over
// the warps by spinor plane.  Four times the warps, a quarter of the chain per warp; the direction is uniform in a warp,
// so the compile-time projector tables of wilson_kernels.cuh are used unchanged.
//
// Same recurrence, same precision rules and the same fixed-order reductions as cg_onelaunch_kernel (PAPER.md:46-48,
// readings G1-G5, G17); the hopping sum is accumulated in the order (x+, x-) + (y+, y-) + (z+, z-) + (t+, t-) with the
// four direction pairs summed last, so results differ from the one-thread-per-site kernels by rounding only.
#pragma once
#include "wilson_launch.cuh"

namespace wd {

// site tiles of 32 sites (one warp wide)
#define WD_SPLIT_TABLE(Z) \
    Z(0, 4, 4, 2, 1)      \
    Z(1, 8, 4, 1, 1)      \
    Z(2, 16, 2, 1, 1)     \
    Z(3, 2, 2, 2, 4)
#define WD_NUM_SPLIT_TILES 4
static const int kSplitTiles[WD_NUM_SPLIT_TILES][4] = {
#define Z(i, a, b, c, d) {a, b, c, d},
    WD_SPLIT_TABLE(Z)
#undef Z
};

cudaError_t launch_cg_split_f32(int split_tile, const CgOneLaunchArgs &a);
cudaError_t launch_cg_split_f64(int split_tile, const CgOneLaunchArgs &a);

template <int D> struct DagTag { static constexpr int value = D; };

// reals per 128-bit spinor plane
template <typename real> struct PlaneW;
template <> struct PlaneW<float> { static constexpr int W = 4; };
template <> struct PlaneW<double> { static constexpr int W = 2; };

__device__ __forceinline__ void plane_get(const float4 &t, float v[4]) { v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w; }
__device__ __forceinline__ void plane_get(const double2 &t, double v[2]) { v[0] = t.x; v[1] = t.y; }
__device__ __forceinline__ float4 plane_make(const float v[4]) { return make_float4(v[0], v[1], v[2], v[3]); }
__device__ __forceinline__ double2 plane_make(const double v[2]) { return make_double2(v[0], v[1]); }

// the two hops of direction MU at site s: acc += sgf (1 -+ gamma) U(s) in(nf) + sgb (1 +- gamma) U(nb)^dagger in(nb)
template <int DAG, int MU, typename real, typename svec, typename gvec>
__device__ __forceinline__ void dir_hops(const gvec *__restrict__ U, const svec *in, int s, int nf, int nb, real sgf,
                                         real sgb, real acc[24])
{
    constexpr int SF = DAG ? +1 : -1;
    real va[24], ua[18], vb[24], ub[18];
    hop_load<MU, false, 18, real>(U, in, s, nf, va, ua);
    hop_load<MU, false, 18, real>(U, in, nb, nb, vb, ub);
    hop_compute<MU, SF, false, real>(va, ua, sgf, acc);
    hop_compute<MU, -SF, true, real>(vb, ub, sgb, acc);
}

template <typename real, int BX, int BY, int BZ, int BT>
__global__ void __launch_bounds__(128, 1)
cg_split_kernel(const Geom g, const typename Field<real>::gvec *__restrict__ U,
                const typename Field<real>::svec *__restrict__ eta, typename Field<real>::svec *y,
                typename Field<real>::svec *r, typename Field<real>::svec *p, typename Field<real>::svec *q,
                typename Field<real>::svec *psi, real kappa, CgScalars *sc, double *partials, double *hist,
                double r_min, int max_iter)
{
    namespace cg = cooperative_groups;
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    static_assert(BX * BY * BZ * BT == 32, "a site tile is one warp wide");
    constexpr int NT = 128;
    constexpr int NSP = Field<real>::NSP;
    constexpr int W = PlaneW<real>::W;
    cg::grid_group grid = cg::this_grid();
    __shared__ double sm[33];
    __shared__ real part[4][24][32];      // part[mu][component][site of the tile]
    const int G = gridDim.x;
    double *part0 = partials, *part1 = partials + G, *part2 = partials + 2 * G;
    const int tid = threadIdx.x;
    const int mu = tid >> 5, lane = tid & 31;
    const int lx = lane % BX, ly = (lane / BX) % BY, lz = (lane / (BX * BY)) % BZ, lt = lane / (BX * BY * BZ);

    // site of this lane in tile b (the same for the four warps); false: outside the lattice
    auto site_of = [&](int b, int &x, int &yy, int &z, int &t, int &s) -> bool {
        int tx, ty, tz, tt;
        tile_of_block(g, b, tx, ty, tz, tt);
        x = tx * BX + lx; yy = ty * BY + ly; z = tz * BZ + lz; t = tt * BT + lt;
        s = x + g.L[0] * (yy + g.L[1] * (z + g.L[2] * t));
        return x < g.L[0] && yy < g.L[1] && z < g.L[2] && t < g.L[3];
    };
    // hopping sum of `in` at the sites of tile b: warp mu -> part[mu]; all threads must call it (barrier inside)
    auto hops_to_shared = [&](auto dag_tag, const svec *in, bool active, int x, int yy, int z, int t, int s) {
        constexpr int DAG = decltype(dag_tag)::value;
        real acc[24];
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = 0;
        if (active) {
            const Hops n = neighbours<0>(g, x, yy, z, t, s);
            const real one = (real)1;
            if (mu == 0) dir_hops<DAG, 0, real>(U, in, s, n.f[0], n.b[0], one, one, acc);
            else if (mu == 1) dir_hops<DAG, 1, real>(U, in, s, n.f[1], n.b[1], one, one, acc);
            else if (mu == 2) dir_hops<DAG, 2, real>(U, in, s, n.f[2], n.b[2], one, one, acc);
            else {
                // boundary sign of reading C-1 on the hop that wraps the t boundary
                const real sgf = (t == g.L[3] - 1) ? (real)g.bc_t : one;
                const real sgb = (t == 0) ? (real)g.bc_t : one;
                dir_hops<DAG, 3, real>(U, in, s, n.f[3], n.b[3], sgf, sgb, acc);
            }
        }
        __syncthreads();                  // the previous tile's tail has read part[]
#pragma unroll
        for (int i = 0; i < 24; ++i) part[mu][i][lane] = acc[i];
        __syncthreads();
    };
    // components W j .. W j + W - 1 of the hopping sum at this lane's site
    auto hop_plane = [&](int j, real h[W]) {
#pragma unroll
        for (int k = 0; k < W; ++k)
            h[k] = (part[0][W * j + k][lane] + part[1][W * j + k][lane]) + (part[2][W * j + k][lane] + part[3][W * j + k][lane]);
    };
    using Dag0 = DagTag<0>;
    using Dag1 = DagTag<1>;

#define WD_FOR_EACH_TILE for (int b = blockIdx.x; b < g.ntiles; b += G)

    // a1: y <- 0, r <- eta, p <- eta, rr = <eta,eta>    (plane j of a site is handled by warp j mod 4)
    double local = 0.0;
    WD_FOR_EACH_TILE {
        int x, yy, z, t, s;
        if (!site_of(b, x, yy, z, t, s)) continue;
        const size_t base = spinor_index<svec, NSP>(s);
        for (int j = mu; j < NSP; j += 4) {
            const svec e = __ldg(eta + base + j * SB);
            y[base + j * SB] = vzero(e);
            r[base + j * SB] = e;
            p[base + j * SB] = e;
            local += vnorm2<svec>(e);
        }
    }
    {
        const double bsum = block_sum<NT>(local, sm);
        if (tid == 0) part0[blockIdx.x] = bsum;
    }
    grid.sync();
    const double eta2 = all_cta_sum<NT>(part0, G, sm);
    double rr = eta2, alpha = 0.0, beta = 0.0;
    int k = 0;
    bool go = isfinite(eta2) && eta2 > 0.0 && loop_test(rr, eta2, r_min).go;
    if (blockIdx.x == 0 && tid == 0 && hist) hist[0] = eta2;

    while (go && k < max_iter) {
        // a2: q = D-dagger p, qq
        local = 0.0;
        WD_FOR_EACH_TILE {
            int x, yy, z, t, s;
            const bool active = site_of(b, x, yy, z, t, s);
            hops_to_shared(Dag1{}, p, active, x, yy, z, t, s);
            if (!active) continue;
            const size_t base = spinor_index<svec, NSP>(s);
            for (int j = mu; j < NSP; j += 4) {
                real h[W], c[W];
                hop_plane(j, h);
                plane_get(p[base + j * SB], c);
                real n2 = 0;
#pragma unroll
                for (int i = 0; i < W; ++i) { c[i] = fma(-kappa, h[i], c[i]); n2 = fma(c[i], c[i], n2); }
                q[base + j * SB] = plane_make(c);
                local += (double)n2;
            }
        }
        {
            const double bsum = block_sum<NT>(local, sm);
            if (tid == 0) part1[blockIdx.x] = bsum;
        }
        grid.sync();
        const double qq = all_cta_sum<NT>(part1, G, sm);
        alpha = rr / qq;                                     // alpha <- |r|^2 / |D-dagger p|^2 (G1)
        const real al = (real)alpha;
        // a3: r <- r - alpha D q, rr'
        local = 0.0;
        WD_FOR_EACH_TILE {
            int x, yy, z, t, s;
            const bool active = site_of(b, x, yy, z, t, s);
            hops_to_shared(Dag0{}, q, active, x, yy, z, t, s);
            if (!active) continue;
            const size_t base = spinor_index<svec, NSP>(s);
            for (int j = mu; j < NSP; j += 4) {
                real h[W], c[W], rv[W];
                hop_plane(j, h);
                plane_get(q[base + j * SB], c);
                plane_get(r[base + j * SB], rv);
                real n2 = 0;
#pragma unroll
                for (int i = 0; i < W; ++i) {
                    c[i] = fma(-kappa, h[i], c[i]);
                    rv[i] = fma(-al, c[i], rv[i]);
                    n2 = fma(rv[i], rv[i], n2);
                }
                r[base + j * SB] = plane_make(rv);
                local += (double)n2;
            }
        }
        {
            const double bsum = block_sum<NT>(local, sm);
            if (tid == 0) part2[blockIdx.x] = bsum;
        }
        grid.sync();
        const double rr_new = all_cta_sum<NT>(part2, G, sm);
        beta = rr_new / rr;                                  // beta <- |r'|^2 / |r|^2
        const real be = (real)beta;
        // a4: y <- y + alpha p ; p <- r + beta p (own sites only)
        WD_FOR_EACH_TILE {
            int x, yy, z, t, s;
            if (!site_of(b, x, yy, z, t, s)) continue;
            const size_t base = spinor_index<svec, NSP>(s);
            for (int j = mu; j < NSP; j += 4) {
                const svec pv = p[base + j * SB];
                y[base + j * SB] = vaxpy(al, pv, y[base + j * SB]);
                p[base + j * SB] = vaxpy(be, pv, r[base + j * SB]);
            }
        }
        rr = rr_new;
        ++k;
        if (blockIdx.x == 0 && tid == 0 && hist) hist[k] = rr;
        go = sqrt(rr) >= r_min * sqrt(eta2);                 // while |r| >= r_min (G4)
        grid.sync();                                         // p complete before its neighbours are read
    }
    // a6: psi = D-dagger y
    WD_FOR_EACH_TILE {
        int x, yy, z, t, s;
        const bool active = site_of(b, x, yy, z, t, s);
        hops_to_shared(Dag1{}, y, active, x, yy, z, t, s);
        if (!active) continue;
        const size_t base = spinor_index<svec, NSP>(s);
        for (int j = mu; j < NSP; j += 4) {
            real h[W], c[W];
            hop_plane(j, h);
            plane_get(y[base + j * SB], c);
#pragma unroll
            for (int i = 0; i < W; ++i) c[i] = fma(-kappa, h[i], c[i]);
            psi[base + j * SB] = plane_make(c);
        }
    }
#undef WD_FOR_EACH_TILE
    if (blockIdx.x == 0 && tid == 0) {
        sc->rr = rr; sc->eta2 = eta2; sc->alpha = alpha; sc->beta = beta; sc->qq = 0.0; sc->r_min = r_min;
        sc->k = k; sc->k_stop = k; sc->max_iter = max_iter;
        sc->converged = (eta2 == 0.0 || loop_test(rr, eta2, r_min).converged) ? 1 : 0;
        sc->breakdown = (!go && !sc->converged) ? 1 : 0;
    }
}

template <typename real>
static cudaError_t launch_cg_split_any(int split_tile, const CgOneLaunchArgs &a)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    switch (split_tile) {
#define Z(i, bx, by, bz, bt)                                                                                   \
    case i: {                                                                                                  \
        auto kern = cg_split_kernel<real, bx, by, bz, bt>;                                                     \
        static int occ_tab[WD_MAXDEV];                                                                         \
        int occ = 0;                                                                                           \
        {                                                                                                      \
            cudaError_t e = cached_occupancy(occ_tab, kern, 128, 0, &occ);                                     \
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
        return cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)grid), dim3(128), args, 0, a.stream); \
    }
        WD_SPLIT_TABLE(Z)
#undef Z
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace wd

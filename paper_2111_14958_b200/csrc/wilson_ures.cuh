// wilson_ures.cuh — SURVEY.md 8(f1): the one-launch CG with the GAUGE FIELD RESIDENT IN SHARED MEMORY (round 2).
//
// cg_onelaunch_kernel keeps every field in L2; at the paper's volumes (Figs. 1-2 at 14^4) its iteration is a
// chain of L2 round trips: 94 loads per site and phase, 40 of them links, with two or three warps per scheduler.  The links
// never change during a solve and are 60 % of the bytes.  When the lattice has no more tiles than CTAs can be co-resident
// (V <= ~57 000 sites in fp32), every CTA owns ONE tile for the whole solve, so it can keep that tile's links in shared
// memory: the four forward links of its sites and, for the sites on a -mu face of the tile, the backward link U_mu(x - mu)
// that belongs to a neighbouring tile (51 KB per 128-site tile in fp32).  They are loaded once; after that a phase reads only
// spinors from L2, and with the link registers gone the spinors of THREE hops are kept in flight instead of one.
// Same recurrence, phases, barriers and fixed-order reductions as cg_onelaunch_kernel, same per-site arithmetic and hop order
// (the iterates differ from it only through the grouping of the reduction partials, which follows the tiles).
#pragma once
#include "wilson_launch.cuh"

namespace wd {

// A region of link slots: N entries, plane-major (fp32: four float4 planes and one float2 plane; fp64: nine double2 planes),
// so that consecutive entries are consecutive 128-bit words of a plane (conflict-free shared loads of a warp).
template <typename real> struct UresLink;
template <> struct UresLink<float> {
    static constexpr int BYTES = 72;   // per entry
    static __device__ __forceinline__ void load(const unsigned char *reg, int N, int idx, float u[18])
    {
        const float4 *p4 = reinterpret_cast<const float4 *>(reg);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float4 t = p4[q * N + idx];
            u[4 * q] = t.x; u[4 * q + 1] = t.y; u[4 * q + 2] = t.z; u[4 * q + 3] = t.w;
        }
        const float2 t2 = reinterpret_cast<const float2 *>(reg + (size_t)4 * N * 16)[idx];
        u[16] = t2.x; u[17] = t2.y;
    }
    static __device__ __forceinline__ void store(unsigned char *reg, int N, int idx, const float u[18])
    {
        float4 *p4 = reinterpret_cast<float4 *>(reg);
#pragma unroll
        for (int q = 0; q < 4; ++q) p4[q * N + idx] = make_float4(u[4 * q], u[4 * q + 1], u[4 * q + 2], u[4 * q + 3]);
        reinterpret_cast<float2 *>(reg + (size_t)4 * N * 16)[idx] = make_float2(u[16], u[17]);
    }
};
template <> struct UresLink<double> {
    static constexpr int BYTES = 144;
    static __device__ __forceinline__ void load(const unsigned char *reg, int N, int idx, double u[18])
    {
        const double2 *p = reinterpret_cast<const double2 *>(reg);
#pragma unroll
        for (int k = 0; k < 9; ++k) {
            const double2 t = p[k * N + idx];
            u[2 * k] = t.x; u[2 * k + 1] = t.y;
        }
    }
    static __device__ __forceinline__ void store(unsigned char *reg, int N, int idx, const double u[18])
    {
        double2 *p = reinterpret_cast<double2 *>(reg);
#pragma unroll
        for (int k = 0; k < 9; ++k) p[k * N + idx] = make_double2(u[2 * k], u[2 * k + 1]);
    }
};

template <int D> struct DagTagU { static constexpr int value = D; };

// shared memory of one CTA: forward links of the NT sites and the halo links of the four -mu faces
template <typename real, int BX, int BY, int BZ, int BT> struct UresShape {
    static constexpr int NT = BX * BY * BZ * BT;
    static constexpr int NH0 = NT / BX, NH1 = NT / BY, NH2 = NT / BZ, NH3 = NT / BT;
    static constexpr int LB = UresLink<real>::BYTES;
    static constexpr int FWD = 4 * NT * LB;
    static constexpr int H0 = FWD, H1 = H0 + NH0 * LB, H2 = H1 + NH1 * LB, H3 = H2 + NH2 * LB;
    static constexpr int SMEM = H3 + NH3 * LB;
};

template <typename real, int BX, int BY, int BZ, int BT, int MINB>
__global__ void __launch_bounds__(BX *BY *BZ *BT, MINB)
cg_ures_kernel(const Geom g, const typename Field<real>::gvec *__restrict__ U,
               const typename Field<real>::svec *__restrict__ eta, typename Field<real>::svec *y,
               typename Field<real>::svec *r, typename Field<real>::svec *p, typename Field<real>::svec *q,
               typename Field<real>::svec *psi, real kappa, CgScalars *sc, double *partials, double *hist,
               double r_min, int max_iter)
{
    namespace cg = cooperative_groups;
    using svec = typename Field<real>::svec;
    using S = UresShape<real, BX, BY, BZ, BT>;
    using UL = UresLink<real>;
    constexpr int NT = S::NT;
    cg::grid_group grid = cg::this_grid();
    __shared__ double sm[33];
    extern __shared__ __align__(16) unsigned char ures_smem[];
    const int G = gridDim.x;                      // == g.ntiles: CTA b owns tile b for the whole solve
    double *part0 = partials, *part1 = partials + G, *part2 = partials + 2 * G;
    const int tid = threadIdx.x;
    const int lx = tid % BX, ly = (tid / BX) % BY, lz = (tid / (BX * BY)) % BZ, lt = tid / (BX * BY * BZ);
    int tx, ty, tz, tt;
    tile_of_block(g, blockIdx.x, tx, ty, tz, tt);
    const int x = tx * BX + lx, yy = ty * BY + ly, z = tz * BZ + lz, t = tt * BT + lt;
    const bool active = x < g.L[0] && yy < g.L[1] && z < g.L[2] && t < g.L[3];
    const int s = active ? x + g.L[0] * (yy + g.L[1] * (z + g.L[2] * t)) : 0;
    Hops n;
    if (active) n = neighbours<0>(g, x, yy, z, t, s);
    else {
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) { n.f[mu] = 0; n.b[mu] = 0; }
    }
    const real one = (real)1;
    const real sgf = (t == g.L[3] - 1) ? (real)g.bc_t : one;
    const real sgb = (t == 0) ? (real)g.bc_t : one;

    // where U_mu(x - mu) of this thread's backward hop lives: the forward slot of another thread of the tile, or the tile's
    // -mu halo (entry = tid with the mu coordinate removed)
    int bidx[4];
    unsigned int inmask = 0;
    {
        const int c[4] = {x, yy, z, t}, l[4] = {lx, ly, lz, lt}, o[4] = {tx * BX, ty * BY, tz * BZ, tt * BT};
        const int B[4] = {BX, BY, BZ, BT}, st[4] = {1, BX, BX * BY, BX * BY * BZ};
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            const int cn = c[mu] == 0 ? g.L[mu] - 1 : c[mu] - 1;
            const int d = cn - o[mu];
            const bool in_tile = d >= 0 && d < B[mu];
            const int lo = tid % st[mu], hi = tid / (st[mu] * B[mu]);
            bidx[mu] = in_tile ? tid + (d - l[mu]) * st[mu] : lo + hi * st[mu];
            inmask |= in_tile ? (1u << mu) : 0u;
        }
    }
    // ---- stage the links once
    if (active) {
        real u[18];
        load_link<0>(U, s, u); UL::store(ures_smem + 0 * NT * S::LB, NT, tid, u);
        load_link<1>(U, s, u); UL::store(ures_smem + 1 * NT * S::LB, NT, tid, u);
        load_link<2>(U, s, u); UL::store(ures_smem + 2 * NT * S::LB, NT, tid, u);
        load_link<3>(U, s, u); UL::store(ures_smem + 3 * NT * S::LB, NT, tid, u);
        if (!(inmask & 1u)) { load_link<0>(U, n.b[0], u); UL::store(ures_smem + S::H0, S::NH0, bidx[0], u); }
        if (!(inmask & 2u)) { load_link<1>(U, n.b[1], u); UL::store(ures_smem + S::H1, S::NH1, bidx[1], u); }
        if (!(inmask & 4u)) { load_link<2>(U, n.b[2], u); UL::store(ures_smem + S::H2, S::NH2, bidx[2], u); }
        if (!(inmask & 8u)) { load_link<3>(U, n.b[3], u); UL::store(ures_smem + S::H3, S::NH3, bidx[3], u); }
    }
    __syncthreads();

#define WD_URES_FWD(MU, u) UL::load(ures_smem + (MU) * NT * S::LB, NT, tid, u)
#define WD_URES_BWD(MU, HOFF, NH, u)                                                                     \
    {                                                                                                    \
        const bool it_ = (inmask >> (MU)) & 1u;                                                          \
        UL::load(ures_smem + (it_ ? (MU) * NT * S::LB : (HOFF)), it_ ? NT : (NH), bidx[MU], u);          \
    }
    // hopping sum of `in` at this thread's site: links from shared memory, the spinors of three hops in flight; c = in(s)
    auto hops = [&](auto dag_tag, const svec *in, real acc[24], real c[24]) {
        constexpr int DAG = decltype(dag_tag)::value;
        constexpr int SF = DAG ? +1 : -1;
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = 0;
        real v0[24], v1[24], v2[24], u[18];
        load_spinor_rw(in, n.f[0], v0);
        load_spinor_rw(in, n.b[0], v1);
        load_spinor_rw(in, n.f[1], v2);
        WD_URES_FWD(0, u);                  hop_compute<0, SF, false, real>(v0, u, one, acc);  load_spinor_rw(in, n.b[1], v0);
        WD_URES_BWD(0, S::H0, S::NH0, u);   hop_compute<0, -SF, true, real>(v1, u, one, acc);  load_spinor_rw(in, n.f[2], v1);
        WD_URES_FWD(1, u);                  hop_compute<1, SF, false, real>(v2, u, one, acc);  load_spinor_rw(in, n.b[2], v2);
        WD_URES_BWD(1, S::H1, S::NH1, u);   hop_compute<1, -SF, true, real>(v0, u, one, acc);  load_spinor_rw(in, n.f[3], v0);
        WD_URES_FWD(2, u);                  hop_compute<2, SF, false, real>(v1, u, one, acc);  load_spinor_rw(in, n.b[3], v1);
        WD_URES_BWD(2, S::H2, S::NH2, u);   hop_compute<2, -SF, true, real>(v2, u, one, acc);  load_spinor_rw(in, s, c);
        WD_URES_FWD(3, u);                  hop_compute<3, SF, false, real>(v0, u, sgf, acc);
        WD_URES_BWD(3, S::H3, S::NH3, u);   hop_compute<3, -SF, true, real>(v1, u, sgb, acc);
    };
    using Dag0 = DagTagU<0>;
    using Dag1 = DagTagU<1>;

    // a1: y <- 0, r <- eta, p <- eta, rr = <eta,eta>
    double local = 0.0;
    if (active) {
        real e[24], zero[24];
        load_spinor(eta, s, e);
        real n2 = 0;
#pragma unroll
        for (int i = 0; i < 24; ++i) { zero[i] = 0; n2 = fma(e[i], e[i], n2); }
        store_spinor(y, s, zero); store_spinor(r, s, e); store_spinor(p, s, e);
        local = (double)n2;
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
        if (active) {
            real acc[24], c[24];
            hops(Dag1{}, p, acc, c);
            real n2 = 0;
#pragma unroll
            for (int i = 0; i < 24; ++i) { c[i] = fma(-kappa, acc[i], c[i]); n2 = fma(c[i], c[i], n2); }
            store_spinor(q, s, c);
            local = (double)n2;
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
        real rv[24];
        if (active) {
            real acc[24], c[24];
            hops(Dag0{}, q, acc, c);
            load_spinor_rw(r, s, rv);
            real n2 = 0;
#pragma unroll
            for (int i = 0; i < 24; ++i) {
                c[i] = fma(-kappa, acc[i], c[i]);
                rv[i] = fma(-al, c[i], rv[i]);
                n2 = fma(rv[i], rv[i], n2);
            }
            store_spinor(r, s, rv);
            local = (double)n2;
        }
        {
            const double bsum = block_sum<NT>(local, sm);
            if (tid == 0) part2[blockIdx.x] = bsum;
        }
        grid.sync();
        const double rr_new = all_cta_sum<NT>(part2, G, sm);
        beta = rr_new / rr;                                  // beta <- |r'|^2 / |r|^2
        const real be = (real)beta;
        // a4: y <- y + alpha p ; p <- r + beta p (own site; r is still in registers)
        if (active) {
            real yv[24], pv[24];
            load_spinor_rw(y, s, yv); load_spinor_rw(p, s, pv);
#pragma unroll
            for (int i = 0; i < 24; ++i) { yv[i] = fma(al, pv[i], yv[i]); pv[i] = fma(be, pv[i], rv[i]); }
            store_spinor(y, s, yv); store_spinor(p, s, pv);
        }
        rr = rr_new;
        ++k;
        if (blockIdx.x == 0 && tid == 0 && hist) hist[k] = rr;
        go = loop_test(rr, eta2, r_min).go;                  // while |r| >= r_min (G4)
        grid.sync();                                         // p complete before its neighbours are read
    }
    // a6: psi = D-dagger y
    if (active) {
        real acc[24], c[24];
        hops(Dag1{}, y, acc, c);
#pragma unroll
        for (int i = 0; i < 24; ++i) c[i] = fma(-kappa, acc[i], c[i]);
        store_spinor(psi, s, c);
    }
#undef WD_URES_FWD
#undef WD_URES_BWD
    if (blockIdx.x == 0 && tid == 0) {
        sc->rr = rr; sc->eta2 = eta2; sc->alpha = alpha; sc->beta = beta; sc->qq = 0.0; sc->r_min = r_min;
        sc->k = k; sc->k_stop = k; sc->max_iter = max_iter;
        sc->converged = (eta2 == 0.0 || loop_test(rr, eta2, r_min).converged) ? 1 : 0;
        sc->breakdown = (!go && !sc->converged) ? 1 : 0;
    }
}

// ---------------------------------------------------------------- launch configurations
//   R(index, BX, BY, BZ, BT, MINB, F32, F64)
#define WD_URES_TABLE(R)          \
    R(0, 16, 2, 2, 2, 3, 1, 0)    \
    R(1, 8, 4, 2, 2, 3, 1, 0)     \
    R(2, 16, 2, 2, 1, 4, 0, 1)    \
    R(3, 8, 4, 2, 1, 4, 0, 1)
#define WD_NUM_URES_ROWS 4
struct UresRowInfo {
    int b[4];
    int minb, f32, f64;
};
static const UresRowInfo kUresRows[WD_NUM_URES_ROWS] = {
#define R(i, a, b, c, d, m, f32, f64) {{a, b, c, d}, m, f32, f64},
    WD_URES_TABLE(R)
#undef R
};
// resident CTAs per SM of row `row` on the current device (0 if the row is not compiled for the precision), and the launch
int ures_occupancy_f32(int row);
int ures_occupancy_f64(int row);
cudaError_t launch_cg_ures_f32(int row, const CgOneLaunchArgs &a);
cudaError_t launch_cg_ures_f64(int row, const CgOneLaunchArgs &a);

template <typename real>
static cudaError_t ures_dispatch(int row, const CgOneLaunchArgs *a, int *occ_out)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    switch (row) {
#define R(i, bx, by, bz, bt, m, f32, f64)                                                                      \
    case i:                                                                                                    \
        if constexpr (sizeof(real) == 4 ? f32 : f64) {                                                         \
            using S = UresShape<real, bx, by, bz, bt>;                                                         \
            auto kern = cg_ures_kernel<real, bx, by, bz, bt, m>;                                               \
            static int occ_tab[WD_MAXDEV];                                                                     \
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM);  \
            if (e != cudaSuccess) return e;                                                                    \
            int occ = 0;                                                                                       \
            e = cached_occupancy(occ_tab, kern, S::NT, S::SMEM, &occ);                                         \
            if (e != cudaSuccess) return e;                                                                    \
            if (occ_out) *occ_out = occ;                                                                       \
            if (!a) return cudaSuccess;                                                                        \
            if ((long)a->g.ntiles > (long)occ * a->sm_count) return cudaErrorInvalidValue;                     \
            if ((size_t)(3 * a->g.ntiles) > a->partials_cap) return cudaErrorInvalidValue;                     \
            Geom g = a->g;                                                                                     \
            const gvec *U = (const gvec *)a->U;                                                                \
            const svec *eta = (const svec *)a->eta;                                                            \
            svec *y = (svec *)a->y, *r = (svec *)a->r, *pp = (svec *)a->p, *q = (svec *)a->q, *psi = (svec *)a->psi; \
            real kappa = (real)a->kappa;                                                                       \
            CgScalars *sc = a->sc;                                                                             \
            double *partials = a->partials, *hist = a->hist;                                                   \
            double r_min = a->r_min;                                                                           \
            int max_iter = a->max_iter;                                                                        \
            void *args[] = {&g, &U, &eta, &y, &r, &pp, &q, &psi, &kappa, &sc, &partials, &hist, &r_min, &max_iter}; \
            return cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)g.ntiles), dim3(S::NT), args, \
                                               S::SMEM, a->stream);                                            \
        }                                                                                                      \
        return cudaErrorInvalidValue;
        WD_URES_TABLE(R)
#undef R
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace wd

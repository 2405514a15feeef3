// wilson_eo_onelaunch.cuh — even-odd preconditioned BiCGSTAB (readings E1 + B1 = EB1 of DESIGN.md) in ONE cooperative
// launch, for the paper's own volumes (4^4 ... 14^4; SURVEY.md 8(f1) x 8(f3) x 8(f4)).
//
// bicgstab_solve_eo needs seven launches per iteration and an iteration moves a few MB there: the solve is a chain of
// launches.  This kernel runs the set-up (etahat = eta_e + kappa H_eo eta_o, norms), the whole loop and the final
// psi_o = eta_o + kappa H_oe psi_e with grid barriers where a launch boundary was: seven per iteration (after each of
// the two hops to the odd sites, after the three reductions, after s and after p are complete at every site).  Every
// CTA sums the per-CTA partials in the same fixed order, so the complex scalars alpha, omega, beta and the loop test are
// identical everywhere (no broadcast, deterministic).  Same recurrence, same precision rules (fp64 scalars and sums,
// reading G17) and the same breakdown rules as the seven-kernel path; one thread per site of one parity, the stencil
// code (hopping_sum with EO = 1) is that of wilson_kernels.cuh.
#pragma once
#include "wilson_launch.cuh"

namespace wd {

// CTA tiles on the half lattice (Lx/2, Ly, Lz, Lt)
#define WD_EO1_TABLE(Z) \
    Z(0, 8, 4, 2, 2)    \
    Z(1, 4, 4, 2, 2)    \
    Z(2, 8, 2, 2, 2)    \
    Z(3, 16, 2, 2, 2)   \
    Z(4, 2, 4, 4, 2)
#define WD_NUM_EO1_TILES 5
static const int kEo1Tiles[WD_NUM_EO1_TILES][4] = {
#define Z(i, a, b, c, d) {a, b, c, d},
    WD_EO1_TABLE(Z)
#undef Z
};

struct EoOneLaunchArgs {
    Geom g;                 // geometry of ONE PARITY (eo = 1), tiled by the chosen row; par is set inside the kernel
    int sm_count;
    cudaStream_t stream;
    const void *Ue, *Uo;    // links of the even / odd sites
    const void *eta_e, *eta_o;
    void *psi_e, *psi_o;
    void *r, *p, *v, *s, *t, *to, *etah;   // half-length work vectors
    double kappa;
    CgScalars *sc;
    double *partials;       // 8 * grid doubles
    size_t partials_cap;
    double *hist;
    double r_min;
    int max_iter;
};
cudaError_t launch_eo_bicgstab_onelaunch_f32(int tile, const EoOneLaunchArgs &a);
cudaError_t launch_eo_bicgstab_onelaunch_f64(int tile, const EoOneLaunchArgs &a);

// y[j] += (ar + i ai) x[j] on the 12 complex numbers of a site
template <typename real>
__device__ __forceinline__ void site_caxpy(real ar, real ai, const real x[24], real y[24])
{
#pragma unroll
    for (int j = 0; j < 12; ++j) {
        y[2 * j] = fma(-ai, x[2 * j + 1], fma(ar, x[2 * j], y[2 * j]));
        y[2 * j + 1] = fma(ai, x[2 * j], fma(ar, x[2 * j + 1], y[2 * j + 1]));
    }
}
// sum_j conj(a_j) b_j -> (re, im)
template <typename real>
__device__ __forceinline__ void site_cdot(const real a[24], const real b[24], real &re, real &im)
{
    re = 0; im = 0;
#pragma unroll
    for (int j = 0; j < 12; ++j) {
        re = fma(a[2 * j], b[2 * j], re); re = fma(a[2 * j + 1], b[2 * j + 1], re);
        im = fma(a[2 * j], b[2 * j + 1], im); im = fma(-a[2 * j + 1], b[2 * j], im);
    }
}
template <typename real>
__device__ __forceinline__ real site_norm2(const real a[24])
{
    real n2 = 0;
#pragma unroll
    for (int i = 0; i < 24; ++i) n2 = fma(a[i], a[i], n2);
    return n2;
}

template <typename real, int BX, int BY, int BZ, int BT>
__global__ void __launch_bounds__(BX *BY *BZ *BT, 1)
eo_bicgstab_onelaunch_kernel(const Geom g0, const typename Field<real>::gvec *__restrict__ Ue,
                             const typename Field<real>::gvec *__restrict__ Uo,
                             const typename Field<real>::svec *__restrict__ eta_e,
                             const typename Field<real>::svec *__restrict__ eta_o, typename Field<real>::svec *psi_e,
                             typename Field<real>::svec *psi_o, typename Field<real>::svec *r,
                             typename Field<real>::svec *p, typename Field<real>::svec *v, typename Field<real>::svec *s_,
                             typename Field<real>::svec *t_, typename Field<real>::svec *to,
                             typename Field<real>::svec *etah, real kappa, CgScalars *sc, double *partials, double *hist,
                             double r_min, int max_iter)
{
    namespace cg = cooperative_groups;
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    constexpr int NT = BX * BY * BZ * BT;
    cg::grid_group grid = cg::this_grid();
    __shared__ double sm[33];
    const int G = gridDim.x;
    const int tid = threadIdx.x;
    const int lx = tid % BX, ly = (tid / BX) % BY, lz = (tid / (BX * BY)) % BZ, lt = tid / (BX * BY * BZ);
    Geom gE = g0, gO = g0;       // launches on the even / on the odd sites
    gE.par = 0; gO.par = 1;
    const real k2 = kappa * kappa;

    // CTA partials of value j of a phase: j * G + blockIdx.x; every CTA then sums them in index order
    auto put = [&](int j, double val) {
        const double b = block_sum<NT>(val, sm);
        if (tid == 0) partials[(size_t)j * G + blockIdx.x] = b;
    };
    auto get = [&](int j) -> double { return all_cta_sum<NT>(partials + (size_t)j * G, G, sm); };

#define WD_EO_FOR_EACH_SITE(...)                                                                   \
    for (int b_ = blockIdx.x; b_ < g0.ntiles; b_ += G) {                                            \
        int tx_, ty_, tz_, tt_;                                                                     \
        tile_of_block(g0, b_, tx_, ty_, tz_, tt_);                                                  \
        const int x = tx_ * BX + lx, y = ty_ * BY + ly, z = tz_ * BZ + lz, t = tt_ * BT + lt;       \
        if (x < g0.L[0] && y < g0.L[1] && z < g0.L[2] && t < g0.L[3]) {                             \
            const int s = x + g0.L[0] * (y + g0.L[1] * (z + g0.L[2] * t));                          \
            __VA_ARGS__                                                                             \
        }                                                                                           \
    }
    // out(s) = hopping sum over the other parity's `in` at the sites of parity PAR (no diagonal term, no kappa)
#define WD_EO_HOPS(PAR, in, acc)                                                                               \
    real acc[24];                                                                                              \
    {                                                                                                          \
        real c_[24], rv_[24];                                                                                  \
        hopping_sum<0, 0, false, false, real, svec, gvec, 18, 1, false>(                                       \
            (PAR) ? gO : gE, (PAR) ? Uo : Ue, (PAR) ? Ue : Uo, in, (const svec *)nullptr, (const svec *)nullptr, x, y, z, t, s, \
            acc, c_, rv_);                                                                                     \
    }

    // ---- set-up: etahat = eta_e + kappa H_eo eta_o ; psi_e <- 0 ; r <- etahat ; p <- etahat ; norms
    double l0 = 0.0, l1 = 0.0;
    WD_EO_FOR_EACH_SITE({
        WD_EO_HOPS(0, eta_o, acc)
        real e[24], o[24], zero[24];
        load_spinor(eta_e, s, e);
        load_spinor(eta_o, s, o);
        l1 += (double)site_norm2(e) + (double)site_norm2(o);
#pragma unroll
        for (int i = 0; i < 24; ++i) { e[i] = fma(kappa, acc[i], e[i]); zero[i] = 0; }
        store_spinor(etah, s, e); store_spinor(r, s, e); store_spinor(p, s, e); store_spinor(psi_e, s, zero);
        l0 += (double)site_norm2(e);
    })
    put(0, l0); put(1, l1);
    grid.sync();
    double rr = get(0);
    const double eta2 = get(1);
    double rho[2] = {rr, 0.0}, alpha[2] = {0.0, 0.0}, omega[2] = {0.0, 0.0}, beta[2] = {0.0, 0.0};
    int k = 0, breakdown = 0;
    bool go = isfinite(eta2) && isfinite(rr) && eta2 > 0.0 && loop_test(rr, eta2, r_min).go;
    if (blockIdx.x == 0 && tid == 0 && hist) hist[0] = rr;

    while (go && k < max_iter) {
        // to = H_oe p
        WD_EO_FOR_EACH_SITE({
            WD_EO_HOPS(1, p, acc)
            store_spinor(to, s, acc);
        })
        grid.sync();
        // v = p - kappa^2 H_eo to ; <rhat, v>
        l0 = 0.0; l1 = 0.0;
        WD_EO_FOR_EACH_SITE({
            WD_EO_HOPS(0, to, acc)
            real pv[24], rh[24];
            load_spinor_rw(p, s, pv);
            load_spinor_rw(etah, s, rh);
#pragma unroll
            for (int i = 0; i < 24; ++i) pv[i] = fma(-k2, acc[i], pv[i]);
            store_spinor(v, s, pv);
            real dr, di;
            site_cdot(rh, pv, dr, di);
            l0 += (double)dr; l1 += (double)di;
        })
        put(2, l0); put(3, l1);
        grid.sync();
        {
            const double rv[2] = {get(2), get(3)};
            if (!cdiv(rho, rv, alpha) || (rho[0] == 0.0 && rho[1] == 0.0)) { breakdown = 1; break; }
        }
        // s = r - alpha v
        {
            const real ar = (real)(-alpha[0]), ai = (real)(-alpha[1]);
            WD_EO_FOR_EACH_SITE({
                real rv_[24], vv[24];
                load_spinor_rw(r, s, rv_);
                load_spinor_rw(v, s, vv);
                site_caxpy(ar, ai, vv, rv_);
                store_spinor(s_, s, rv_);
            })
        }
        grid.sync();
        // to = H_oe s
        WD_EO_FOR_EACH_SITE({
            WD_EO_HOPS(1, s_, acc)
            store_spinor(to, s, acc);
        })
        grid.sync();
        // t = s - kappa^2 H_eo to ; <t,s>, <t,t>
        l0 = 0.0; l1 = 0.0;
        double l2 = 0.0;
        WD_EO_FOR_EACH_SITE({
            WD_EO_HOPS(0, to, acc)
            real sv[24], tv[24];
            load_spinor_rw(s_, s, sv);
#pragma unroll
            for (int i = 0; i < 24; ++i) tv[i] = fma(-k2, acc[i], sv[i]);
            store_spinor(t_, s, tv);
            real dr, di;
            site_cdot(tv, sv, dr, di);
            l0 += (double)dr; l1 += (double)di; l2 += (double)site_norm2(tv);
        })
        put(4, l0); put(5, l1); put(6, l2);
        grid.sync();
        {
            const double ts0 = get(4), ts1 = get(5), tt = get(6);
            omega[0] = tt > 0.0 ? ts0 / tt : 0.0;
            omega[1] = tt > 0.0 ? ts1 / tt : 0.0;
        }
        // psi_e += alpha p + omega s ; r = s - omega t ; rho' = <rhat, r> ; rr = <r,r>
        l0 = 0.0; l1 = 0.0; l2 = 0.0;
        {
            const real ar = (real)alpha[0], ai = (real)alpha[1], wr = (real)omega[0], wi = (real)omega[1];
            WD_EO_FOR_EACH_SITE({
                real xs[24], pv[24], sv[24], tv[24], rh[24];
                load_spinor_rw(psi_e, s, xs);
                load_spinor_rw(p, s, pv);
                load_spinor_rw(s_, s, sv);
                site_caxpy(ar, ai, pv, xs);
                site_caxpy(wr, wi, sv, xs);
                store_spinor(psi_e, s, xs);
                load_spinor_rw(t_, s, tv);
                site_caxpy(-wr, -wi, tv, sv);       // sv = s - omega t = the new r
                store_spinor(r, s, sv);
                load_spinor_rw(etah, s, rh);
                real dr, di;
                site_cdot(rh, sv, dr, di);
                l0 += (double)dr; l1 += (double)di; l2 += (double)site_norm2(sv);
            })
        }
        put(2, l0); put(3, l1); put(7, l2);
        grid.sync();
        const double rho_new[2] = {get(2), get(3)};
        rr = get(7);
        ++k;
        if (blockIdx.x == 0 && tid == 0 && hist) hist[k] = rr;
        go = sqrt(rr) >= r_min * sqrt(eta2);                 // loop test of reading E1 (relative to the FULL source)
        if (!go) break;
        {
            double a[2], b[2];
            if (!(cdiv(rho_new, rho, a) && cdiv(alpha, omega, b))) { breakdown = 1; break; }
            beta[0] = a[0] * b[0] - a[1] * b[1];
            beta[1] = a[0] * b[1] + a[1] * b[0];
            rho[0] = rho_new[0]; rho[1] = rho_new[1];
        }
        // p = r + beta (p - omega v)
        {
            const real br = (real)beta[0], bi = (real)beta[1], wr = (real)(-omega[0]), wi = (real)(-omega[1]);
            WD_EO_FOR_EACH_SITE({
                real pv[24], vv[24], rv_[24];
                load_spinor_rw(p, s, pv);
                load_spinor_rw(v, s, vv);
                load_spinor_rw(r, s, rv_);
                site_caxpy(wr, wi, vv, pv);         // p - omega v
                site_caxpy(br, bi, pv, rv_);        // r + beta (...)
                store_spinor(p, s, rv_);
            })
        }
        grid.sync();
    }
    grid.sync();                                             // psi_e complete at every site (also after a break)
    // psi_o = eta_o + kappa H_oe psi_e
    WD_EO_FOR_EACH_SITE({
        WD_EO_HOPS(1, psi_e, acc)
        real o[24];
        load_spinor(eta_o, s, o);
#pragma unroll
        for (int i = 0; i < 24; ++i) o[i] = fma(kappa, acc[i], o[i]);
        store_spinor(psi_o, s, o);
    })
#undef WD_EO_HOPS
#undef WD_EO_FOR_EACH_SITE
    if (blockIdx.x == 0 && tid == 0) {
        sc->rr = rr; sc->eta2 = eta2; sc->alpha = 0.0; sc->beta = 0.0; sc->qq = 0.0; sc->r_min = r_min;
        sc->rho[0] = rho[0]; sc->rho[1] = rho[1]; sc->calpha[0] = alpha[0]; sc->calpha[1] = alpha[1];
        sc->omega[0] = omega[0]; sc->omega[1] = omega[1]; sc->cbeta[0] = beta[0]; sc->cbeta[1] = beta[1];
        sc->k = k; sc->k_stop = k; sc->max_iter = max_iter;
        sc->converged = (eta2 == 0.0 || loop_test(rr, eta2, r_min).converged) ? 1 : 0;
        sc->breakdown = (breakdown || (!go && !sc->converged)) ? 1 : 0;   // a stop that is not a convergence: NaN or vanishing denominator
    }
}

template <typename real>
static cudaError_t launch_eo_bicgstab_onelaunch_any(int tile, const EoOneLaunchArgs &a)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    switch (tile) {
#define Z(i, bx, by, bz, bt)                                                                                   \
    case i: {                                                                                                  \
        auto kern = eo_bicgstab_onelaunch_kernel<real, bx, by, bz, bt>;                                        \
        static int occ_tab[WD_MAXDEV];                                                                         \
        int occ = 0;                                                                                           \
        {                                                                                                      \
            cudaError_t e = cached_occupancy(occ_tab, kern, bx * by * bz * bt, 0, &occ);                       \
            if (e != cudaSuccess) return e;                                                                    \
        }                                                                                                      \
        long grid = (long)occ * a.sm_count;            /* all CTAs must be co-resident (grid barrier) */       \
        if (grid > a.g.ntiles) grid = a.g.ntiles;                                                              \
        if ((size_t)(8 * grid) > a.partials_cap) return cudaErrorInvalidValue;                                 \
        Geom g = a.g;                                                                                          \
        const gvec *Ue = (const gvec *)a.Ue, *Uo = (const gvec *)a.Uo;                                         \
        const svec *ee = (const svec *)a.eta_e, *eo = (const svec *)a.eta_o;                                   \
        svec *pe = (svec *)a.psi_e, *po = (svec *)a.psi_o, *r = (svec *)a.r, *pp = (svec *)a.p, *v = (svec *)a.v; \
        svec *s = (svec *)a.s, *t = (svec *)a.t, *to = (svec *)a.to, *etah = (svec *)a.etah;                    \
        real kappa = (real)a.kappa;                                                                            \
        CgScalars *sc = a.sc;                                                                                  \
        double *partials = a.partials, *hist = a.hist;                                                         \
        double r_min = a.r_min;                                                                                \
        int max_iter = a.max_iter;                                                                             \
        void *args[] = {&g, &Ue, &Uo, &ee, &eo, &pe, &po, &r, &pp, &v, &s, &t, &to, &etah, &kappa, &sc,        \
                        &partials, &hist, &r_min, &max_iter};                                                  \
        return cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)grid), dim3(bx * by * bz * bt),  \
                                           args, 0, a.stream);                                                 \
    }
        WD_EO1_TABLE(Z)
#undef Z
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace wd

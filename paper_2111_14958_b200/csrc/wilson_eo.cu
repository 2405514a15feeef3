// wilson_eo.cu — even-odd (Schur) preconditioned CG (reading E1 of DESIGN.md).
//
// Sites are coloured by the parity of x+y+z+t.  The hopping term connects opposite parities only, so with
// D = [[1, -kappa H_eo], [-kappa H_oe, 1]] the system D psi = eta becomes
//     Mhat psi_e = etahat,  Mhat = 1 - kappa^2 H_eo H_oe,  etahat = eta_e + kappa H_eo eta_o,  psi_o = eta_o + kappa H_oe psi_e
// and the paper's CG recurrence runs on Mhat Mhat-dagger over HALF-length vectors with a
// better-conditioned operator.  The stencil kernel is the one of the plain path (wilson_kernels.cuh) launched on a
// half lattice (Geom.eo = 1): same tiles, same fused epilogues; only the +-x neighbour rule and the fields the
// links / the diagonal term come from differ.  This file holds the checkerboard pack kernels and the host loop.
#include "wilson_ctx.cuh"
#include "wilson_eo_onelaunch.cuh"

#include <cmath>

using namespace wd;

namespace {

struct EoDims {
    int hd[4];          // extents of one parity: {Lx/2, Ly, Lz, Lt}
    int Vh;             // sites per parity
    size_t Vh_pad;      // padded to whole 16-site blocks
};
EoDims eo_dims(const wd_ctx *c)
{
    EoDims e;
    e.hd[0] = c->dims[0] / 2; e.hd[1] = c->dims[1]; e.hd[2] = c->dims[2]; e.hd[3] = c->dims[3];
    e.Vh = c->V / 2;
    e.Vh_pad = ((size_t)e.Vh + SB - 1) / SB * SB;
    return e;
}
size_t half_spinor_bytes(const wd_ctx *c) { return 24 * eo_dims(c).Vh_pad * real_bytes(c); }
size_t half_gauge_bytes(const wd_ctx *c) { return (size_t)(c->recon == 12 ? 48 : 72) * eo_dims(c).Vh_pad * real_bytes(c); }
size_t half_spinor_vecs(const wd_ctx *c) { return (size_t)(c->precision == 32 ? 6 : 12) * eo_dims(c).Vh_pad; }

int eo_check(wd_ctx *c, const char *who)
{
    for (int d = 0; d < 4; ++d)
        if (c->dims[d] & 1) return fail(c, WD_ERR_DIMS, "%s: extent %d of direction %d is odd (even-odd needs even extents)", who, c->dims[d], d);
    return WD_OK;
}

// parity and checkerboard index of lexicographic site s: the pair (2 xh, 2 xh + 1) of a row holds one site of
// each parity, so the index inside a parity is simply s / 2 (Lx even).
__device__ __forceinline__ int site_parity(int s, int L0, int L1, int L2)
{
    const int x = s % L0, y = (s / L0) % L1, z = (s / (L0 * L1)) % L2, t = s / (L0 * L1 * L2);
    return (x + y + z + t) & 1;
}

template <typename real>
__global__ void __launch_bounds__(VEC_NT)
eo_pack_spinor_kernel(const typename Field<real>::svec *__restrict__ can, typename Field<real>::svec *nat, int V, int L0,
                      int L1, int L2, size_t half_vecs)
{
    using svec = typename Field<real>::svec;
    constexpr int NSP = Field<real>::NSP;
    const int s = blockIdx.x * VEC_NT + threadIdx.x;
    if (s >= V) return;
    svec *p = nat + site_parity(s, L0, L1, L2) * half_vecs + spinor_index<svec, NSP>(s >> 1);
#pragma unroll
    for (int j = 0; j < NSP; ++j) p[j * SB] = __ldg(can + (size_t)s * NSP + j);
}
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
eo_unpack_spinor_kernel(const typename Field<real>::svec *__restrict__ nat, typename Field<real>::svec *can, int V, int L0,
                        int L1, int L2, size_t half_vecs)
{
    using svec = typename Field<real>::svec;
    constexpr int NSP = Field<real>::NSP;
    const int s = blockIdx.x * VEC_NT + threadIdx.x;
    if (s >= V) return;
    const svec *p = nat + site_parity(s, L0, L1, L2) * half_vecs + spinor_index<svec, NSP>(s >> 1);
#pragma unroll
    for (int j = 0; j < NSP; ++j) can[(size_t)s * NSP + j] = __ldg(p + j * SB);
}
template <typename real, int RECON>
__global__ void __launch_bounds__(VEC_NT)
eo_pack_gauge_kernel(const typename Field<real>::gvec *__restrict__ can, typename Field<real>::gvec *nat, int V, int L0,
                     int L1, int L2, size_t half_cplx)
{
    using gvec = typename Field<real>::gvec;
    const int s = blockIdx.x * VEC_NT + threadIdx.x;
    if (s >= V) return;
    gvec *half = nat + site_parity(s, L0, L1, L2) * half_cplx;
    for (int mu = 0; mu < 4; ++mu) {
        gvec k9[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) k9[k] = __ldg(can + (size_t)s * 36 + mu * 9 + k);
        if (RECON == 12) store_link12(half, s >> 1, mu, k9);
        else store_link(half, s >> 1, mu, k9);
    }
}

// after cg_init on etahat: the loop test is taken against the FULL source norm (reading E1)
__global__ void eo_set_eta2_kernel(CgScalars *sc, const double *n2, double r_min, int max_iter)
{
    const double eta2 = n2[0] + n2[1];
    sc->eta2 = eta2;
    loop_begin(sc, sc->rr, eta2, r_min, max_iter);
}

// one stencil pass on the sites of parity `par`:  out = cen - coef * (hopping sum over the other parity's `in`)
struct EoPass {
    int dagger, mode, par;
    const void *in, *cen;
    void *out, *r;
    double coef;
    int it;
    bool in_loop;   // plain passes inside the CG loop obey the device stop flag
};

cudaError_t eo_launch(wd_ctx *c, const void *U_eo, const EoPass &p)
{
    const EoDims e = eo_dims(c);
    const int tile = c->tile_user >= 0 ? c->tile_user : auto_tile_dims(c, e.hd);
    DslashArgs a;
    a.g = make_geom_lattice(e.hd, c->bc_t, kTiles[tile].b, c->zchunk_user, c->l2_budget_mb);
    a.g.eo = 1;
    a.g.par = p.par;
    a.sm_count = c->sm_count;
    a.stream = c->stream;
    const size_t hg = half_gauge_bytes(c);
    a.U = (const char *)U_eo + (size_t)p.par * hg;
    a.Ub = (const char *)U_eo + (size_t)(1 - p.par) * hg;
    a.in = p.in; a.cen = p.cen; a.out = p.out; a.kappa = p.coef; a.r = p.r;
    a.sc = (p.mode != MODE_PLAIN || p.in_loop) ? c->sc : nullptr;
    a.partials = c->partials; a.counter = c->counter; a.hist = hist_at(c, p.it); a.it = p.it;
    c->launches++;
    if (c->recon == 12)
        return c->precision == 32 ? launch_dslash12_eo_f32(tile, p.dagger, p.mode, a) : launch_dslash12_eo_f64(tile, p.dagger, p.mode, a);
    if (p.mode == MODE_RV || p.mode == MODE_TS)
        return c->precision == 32 ? launch_dslash_eo_bi_f32(tile, p.mode, a) : launch_dslash_eo_bi_f64(tile, p.mode, a);
    return c->precision == 32 ? launch_dslash_eo_f32(tile, p.dagger, p.mode, a) : launch_dslash_eo_f64(tile, p.dagger, p.mode, a);
}

}  // namespace

extern "C" size_t wd_eo_spinor_bytes(wd_ctx *c) { return c ? 2 * half_spinor_bytes(c) : 0; }
extern "C" size_t wd_eo_gauge_bytes(wd_ctx *c) { return c ? 2 * half_gauge_bytes(c) : 0; }

extern "C" int wd_eo_pack_spinor(wd_ctx *c, const void *can, void *nat)
{
    if (!c) return WD_ERR_ARG;
    if (!can || !nat || can == nat) return fail(c, WD_ERR_ARG, "wd_eo_pack_spinor: NULL or aliased argument");
    int rc = eo_check(c, "wd_eo_pack_spinor");
    if (rc != WD_OK) return rc;
    const EoDims e = eo_dims(c);
    if (e.Vh_pad != (size_t)e.Vh) CUDA_TRY(c, cudaMemsetAsync(nat, 0, 2 * half_spinor_bytes(c), c->stream));
    const unsigned int grid = (c->V + VEC_NT - 1) / VEC_NT;
    if (c->precision == 32)
        eo_pack_spinor_kernel<float><<<grid, VEC_NT, 0, c->stream>>>((const float4 *)can, (float4 *)nat, c->V, c->dims[0],
                                                                    c->dims[1], c->dims[2], half_spinor_vecs(c));
    else
        eo_pack_spinor_kernel<double><<<grid, VEC_NT, 0, c->stream>>>((const double2 *)can, (double2 *)nat, c->V, c->dims[0],
                                                                     c->dims[1], c->dims[2], half_spinor_vecs(c));
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    return WD_OK;
}

extern "C" int wd_eo_unpack_spinor(wd_ctx *c, const void *nat, void *can)
{
    if (!c) return WD_ERR_ARG;
    if (!can || !nat || can == nat) return fail(c, WD_ERR_ARG, "wd_eo_unpack_spinor: NULL or aliased argument");
    int rc = eo_check(c, "wd_eo_unpack_spinor");
    if (rc != WD_OK) return rc;
    const unsigned int grid = (c->V + VEC_NT - 1) / VEC_NT;
    if (c->precision == 32)
        eo_unpack_spinor_kernel<float><<<grid, VEC_NT, 0, c->stream>>>((const float4 *)nat, (float4 *)can, c->V, c->dims[0],
                                                                      c->dims[1], c->dims[2], half_spinor_vecs(c));
    else
        eo_unpack_spinor_kernel<double><<<grid, VEC_NT, 0, c->stream>>>((const double2 *)nat, (double2 *)can, c->V,
                                                                       c->dims[0], c->dims[1], c->dims[2], half_spinor_vecs(c));
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    return WD_OK;
}

extern "C" int wd_eo_pack_gauge(wd_ctx *c, const void *can, void *nat)
{
    if (!c) return WD_ERR_ARG;
    if (!can || !nat || can == nat) return fail(c, WD_ERR_ARG, "wd_eo_pack_gauge: NULL or aliased argument");
    int rc = eo_check(c, "wd_eo_pack_gauge");
    if (rc != WD_OK) return rc;
    const EoDims e = eo_dims(c);
    if (e.Vh_pad != (size_t)e.Vh) CUDA_TRY(c, cudaMemsetAsync(nat, 0, 2 * half_gauge_bytes(c), c->stream));
    const unsigned int grid = (c->V + VEC_NT - 1) / VEC_NT;
    const size_t half_cplx = (size_t)(c->recon == 12 ? 24 : 36) * e.Vh_pad;   // complex slots per parity
    const int d0 = c->dims[0], d1 = c->dims[1], d2 = c->dims[2];
    if (c->precision == 32 && c->recon == 18)
        eo_pack_gauge_kernel<float, 18><<<grid, VEC_NT, 0, c->stream>>>((const float2 *)can, (float2 *)nat, c->V, d0, d1, d2, half_cplx);
    else if (c->precision == 32)
        eo_pack_gauge_kernel<float, 12><<<grid, VEC_NT, 0, c->stream>>>((const float2 *)can, (float2 *)nat, c->V, d0, d1, d2, half_cplx);
    else if (c->recon == 18)
        eo_pack_gauge_kernel<double, 18><<<grid, VEC_NT, 0, c->stream>>>((const double2 *)can, (double2 *)nat, c->V, d0, d1, d2, half_cplx);
    else
        eo_pack_gauge_kernel<double, 12><<<grid, VEC_NT, 0, c->stream>>>((const double2 *)can, (double2 *)nat, c->V, d0, d1, d2, half_cplx);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    return WD_OK;
}

extern "C" int wd_eo_hop(wd_ctx *c, const void *U_eo, const void *in_eo, void *out_eo, int out_parity, int dagger)
{
    if (!c) return WD_ERR_ARG;
    if (!U_eo || !in_eo || !out_eo) return fail(c, WD_ERR_ARG, "wd_eo_hop: NULL argument");
    if (out_parity != 0 && out_parity != 1) return fail(c, WD_ERR_ARG, "wd_eo_hop: out_parity must be 0 or 1");
    int rc = eo_check(c, "wd_eo_hop");
    if (rc != WD_OK) return rc;
    const size_t hs = half_spinor_bytes(c);
    EoPass p{dagger ? 1 : 0, MODE_PLAIN, out_parity, (const char *)in_eo + (size_t)(1 - out_parity) * hs, nullptr,
             (char *)out_eo + (size_t)out_parity * hs, nullptr, -1.0, 0, false};
    CUDA_TRY(c, eo_launch(c, U_eo, p));
    return WD_OK;
}

template <typename real>
static int eo_loop(wd_ctx *c, const void *U_eo, const void *eta_eo, void *psi_eo, double kappa, double r_min, int max_iter)
{
    using svec = typename Field<real>::svec;
    const EoDims e = eo_dims(c);
    const size_t hs = half_spinor_bytes(c), n = half_spinor_vecs(c);
    const int pad = e.Vh_pad != (size_t)e.Vh;
    const char *eta_e = (const char *)eta_eo, *eta_o = eta_e + hs;
    char *psi_e = (char *)psi_eo, *psi_o = psi_e + hs;
    void *r = c->r, *p = c->p, *q = c->q, *y = c->y, *t = c->w5, *etah = c->w6;
    const double k2 = kappa * kappa;
    const unsigned int vgrid = wd_vec_grid(c, n, WD_VEC_PER_SM), ugrid = wd_vec_grid(c, n, WD_UPD_PER_SM);

    // <eta,eta> of the full source (two halves), etahat = eta_e + kappa H_eo eta_o
    norm2_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>((const svec *)eta_e, n, e.Vh, pad, c->partials, c->counter, c->eo_n2);
    norm2_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>((const svec *)eta_o, n, e.Vh, pad, c->partials, c->counter, c->eo_n2 + 1);
    c->launches += 2;
    CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_PLAIN, 0, eta_o, eta_e, etah, nullptr, -kappa, 0, false}));
    // a1 on the half lattice: y <- 0, r <- etahat, p <- etahat, rr = <etahat,etahat>
    cg_init_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>((const svec *)etah, (svec *)y, (svec *)r, (svec *)p, n, e.Vh, pad,
                                                         c->sc, c->partials, c->counter, c->hist, r_min, max_iter);
    eo_set_eta2_kernel<<<1, 1, 0, c->stream>>>(c->sc, c->eo_n2, r_min, max_iter);
    c->launches += 2;
    CUDA_TRY(c, cudaGetLastError());

    const int poll = c->poll > 0 ? c->poll : 8;
    auto enqueue = [&](int first, int chunk, int) -> int {
        for (int i = 0; i < chunk; ++i) {
            const int it = first + i;
            const bool ev = c->profile && i == 0;
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[0], c->stream));
            // t_o = H-dagger_oe p_e
            CUDA_TRY(c, eo_launch(c, U_eo, EoPass{1, MODE_PLAIN, 1, p, nullptr, t, nullptr, -1.0, it, true}));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[1], c->stream));
            // q_e = p_e - kappa^2 H-dagger_eo t_o = Mhat-dagger p ; qq ; alpha
            CUDA_TRY(c, eo_launch(c, U_eo, EoPass{1, MODE_QQ, 0, t, p, q, nullptr, k2, it, true}));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[2], c->stream));
            // t_o = H_oe q_e
            CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_PLAIN, 1, q, nullptr, t, nullptr, -1.0, it, true}));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[3], c->stream));
            // r_e <- r_e - alpha (q_e - kappa^2 H_eo t_o) = r - alpha Mhat Mhat-dagger p ; rr' ; beta ; loop test
            CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_RUPD, 0, t, q, nullptr, r, k2, it, true}));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[4], c->stream));
            // y += alpha p ; p = r + beta p
            cg_update_kernel<real><<<ugrid, VEC_NT, 0, c->stream>>>((svec *)y, (svec *)p, (const svec *)r, n, c->sc, it);
            c->launches++;
            CUDA_TRY(c, cudaGetLastError());
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[5], c->stream));
        }
        return WD_OK;
    };
    auto polled = [&](int first, int, int) -> int {
        if (c->profile && first < c->sc_host->k_stop) {
            for (int j = 0; j < 5; ++j) {
                float ms = 0.f;
                CUDA_TRY(c, cudaEventElapsedTime(&ms, c->bev[j], c->bev[j + 1]));
                c->bprof_ms[j] += ms;
            }
            c->bprof_n++;
        }
        return WD_OK;
    };
    int rc = wd_poll_loop(c, max_iter, poll, false, enqueue, polled);   // no look-ahead: measured no gain (wilson_cg.cu)
    if (rc != WD_OK) return rc;
    // psi_e = Mhat-dagger y ; psi_o = eta_o + kappa H_oe psi_e
    CUDA_TRY(c, eo_launch(c, U_eo, EoPass{1, MODE_PLAIN, 1, y, nullptr, t, nullptr, -1.0, 0, false}));
    CUDA_TRY(c, eo_launch(c, U_eo, EoPass{1, MODE_PLAIN, 0, t, y, psi_e, nullptr, k2, 0, false}));
    CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_PLAIN, 1, psi_e, eta_o, psi_o, nullptr, -kappa, 0, false}));
    return WD_OK;
}

extern "C" int cg_solve_eo(wd_ctx *c, const void *U_eo, const void *eta_eo, void *psi_eo, double kappa, double r_min,
                           int max_iter, wd_cg_info *info)
{
    if (!c) return WD_ERR_ARG;
    if (!U_eo || !eta_eo || !psi_eo || eta_eo == psi_eo) return fail(c, WD_ERR_ARG, "cg_solve_eo: NULL argument or output aliases eta");
    if (!std::isfinite(kappa)) return fail(c, WD_ERR_ARG, "cg_solve_eo: kappa is not finite");
    if (!(r_min > 0.0) || !std::isfinite(r_min)) return fail(c, WD_ERR_ARG, "cg_solve_eo: r_min must be > 0");
    if (max_iter < 0) return fail(c, WD_ERR_ARG, "cg_solve_eo: max_iter < 0");
    int rc = eo_check(c, "cg_solve_eo");
    if (rc != WD_OK) return rc;
    rc = wd_ensure_workspace(c, max_iter);
    if (rc != WD_OK) return rc;
    if (!c->w5) {
        CUDA_TRY(c, cudaMalloc(&c->w5, spinor_bytes(c)));
        CUDA_TRY(c, cudaMemsetAsync(c->w5, 0, spinor_bytes(c), c->stream));
    }
    if (!c->w6) {
        CUDA_TRY(c, cudaMalloc(&c->w6, half_spinor_bytes(c)));
        CUDA_TRY(c, cudaMemsetAsync(c->w6, 0, half_spinor_bytes(c), c->stream));   // pad lanes stay zero
    }
    if (!c->eo_n2) CUDA_TRY(c, cudaMalloc(&c->eo_n2, 2 * sizeof(double)));
    if (c->profile && !c->bev[0])
        for (int j = 0; j < 8; ++j) CUDA_TRY(c, cudaEventCreate(&c->bev[j]));
    c->launches = 0;
    CUDA_TRY(c, cudaEventRecord(c->ev[0], c->stream));
    rc = c->precision == 32 ? eo_loop<float>(c, U_eo, eta_eo, psi_eo, kappa, r_min, max_iter)
                            : eo_loop<double>(c, U_eo, eta_eo, psi_eo, kappa, r_min, max_iter);
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
        info->cg_mode = 4;
    }
    return s.converged ? WD_OK : (s.breakdown ? WD_BREAKDOWN : WD_NOT_CONVERGED);
}

// ---------------------------------------------------------------- even-odd preconditioned BiCGSTAB (readings E1 + B1)
// The BiCGSTAB recurrence of bicgstab_solve (wilson_cg.cu) on the Schur operator Mhat = 1 - kappa^2 H_eo H_oe over
// half-length vectors.  Every Mhat application is two launches of the one-parity stencil: a plain hop to the odd sites
// and the hop back fused with the diagonal term and the dot products of the BiCGSTAB pass (MODE_RV / MODE_TS, EO = 1).
template <typename real>
static int eo_bicgstab_loop(wd_ctx *c, const void *U_eo, const void *eta_eo, void *psi_eo, double kappa, double r_min,
                            int max_iter)
{
    using svec = typename Field<real>::svec;
    const EoDims e = eo_dims(c);
    const size_t hs = half_spinor_bytes(c), n = half_spinor_vecs(c);
    const int pad = e.Vh_pad != (size_t)e.Vh;
    const char *eta_e = (const char *)eta_eo, *eta_o = eta_e + hs;
    char *psi_e = (char *)psi_eo, *psi_o = psi_e + hs;
    svec *r = (svec *)c->r, *p = (svec *)c->p, *v = (svec *)c->q, *s = (svec *)c->y;
    void *to = c->w5;                                 // odd-parity intermediate H_oe (.)
    svec *t = (svec *)c->w7;                          // t = Mhat s
    const svec *etah = (const svec *)c->w6;           // etahat = shadow residual rhat
    const double k2 = kappa * kappa;
    const unsigned int vgrid = wd_vec_grid(c, n, WD_VEC_PER_SM), ugrid = wd_vec_grid(c, n, WD_UPD_PER_SM);

    norm2_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>((const svec *)eta_e, n, e.Vh, pad, c->partials, c->counter, c->eo_n2);
    norm2_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>((const svec *)eta_o, n, e.Vh, pad, c->partials, c->counter, c->eo_n2 + 1);
    c->launches += 2;
    CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_PLAIN, 0, eta_o, eta_e, c->w6, nullptr, -kappa, 0, false}));
    // psi_e <- 0, r <- etahat, p <- etahat, rho = rr = <etahat,etahat>; then the loop test against the FULL source norm
    bi_init_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>(etah, (svec *)psi_e, r, p, n, e.Vh, pad, c->sc, c->partials,
                                                         c->counter, c->hist, r_min, max_iter);
    eo_set_eta2_kernel<<<1, 1, 0, c->stream>>>(c->sc, c->eo_n2, r_min, max_iter);
    c->launches += 2;
    CUDA_TRY(c, cudaGetLastError());

    const int poll = c->poll > 0 ? c->poll : 4;
    auto enqueue = [&](int first, int chunk, int) -> int {
        for (int i = 0; i < chunk; ++i) {
            const int it = first + i;
            const bool ev = c->profile && i == 0;
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[0], c->stream));
            // to = H_oe p
            CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_PLAIN, 1, p, nullptr, to, nullptr, -1.0, it, true}));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[1], c->stream));
            // v = p - kappa^2 H_eo to = Mhat p ; <rhat,v> ; alpha
            CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_RV, 0, to, p, v, (void *)etah, k2, it, true}));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[2], c->stream));
            // s = r - alpha v
            bi_s_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>(s, r, v, n, e.Vh, pad, c->sc, it);
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[3], c->stream));
            // to = H_oe s
            CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_PLAIN, 1, s, nullptr, to, nullptr, -1.0, it, true}));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[4], c->stream));
            // t = s - kappa^2 H_eo to = Mhat s ; <t,s>, <t,t> ; omega
            CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_TS, 0, to, s, t, nullptr, k2, it, true}));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[5], c->stream));
            // psi_e += alpha p + omega s ; r = s - omega t ; rho', rr, beta, loop test
            bi_xr_kernel<real><<<ugrid, VEC_NT, 0, c->stream>>>((svec *)psi_e, r, p, s, t, etah, n, e.Vh, pad, c->sc, c->partials,
                                                               c->counter, hist_at(c, it), it);
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[6], c->stream));
            // p = r + beta (p - omega v)
            bi_p_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>(p, r, v, n, e.Vh, pad, c->sc, it);
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[7], c->stream));
            c->launches += 3;
            CUDA_TRY(c, cudaGetLastError());
        }
        return WD_OK;
    };
    auto polled = [&](int first, int, int) -> int {
        if (c->profile && first < c->sc_host->k_stop) {
            for (int j = 0; j < 7; ++j) {
                float ms = 0.f;
                CUDA_TRY(c, cudaEventElapsedTime(&ms, c->bev[j], c->bev[j + 1]));
                c->bprof_ms[j] += ms;
            }
            c->bprof_n++;
        }
        return WD_OK;
    };
    int rc = wd_poll_loop(c, max_iter, poll, false, enqueue, polled);   // no look-ahead: measured no gain (wilson_cg.cu)
    if (rc != WD_OK) return rc;
    // psi_o = eta_o + kappa H_oe psi_e
    CUDA_TRY(c, eo_launch(c, U_eo, EoPass{0, MODE_PLAIN, 1, psi_e, eta_o, psi_o, nullptr, -kappa, 0, false}));
    return WD_OK;
}

// Largest volume (sites of the FULL lattice) that bicgstab_solve_eo solves in one cooperative launch in automatic mode.
// Measured on B200, ms per solve, seven kernels per iteration / one launch: fp32 4^4 0.39 / 0.16, 14^4 0.40 / 0.26, 16^4
// 1.14 / 0.78, 20^4 1.79 / 2.14; fp64 4^4 0.54 / 0.33, 14^4 0.77 / 0.64, 16^4 2.67 / 2.38, 20^4 5.63 / 8.99.
#ifndef WD_EO_ONELAUNCH_MAX_SITES
#define WD_EO_ONELAUNCH_MAX_SITES 65536
#endif

static bool eo_use_onelaunch(const wd_ctx *c)
{
    if (!c->coop_ok || c->recon != 18) return false;
    if (c->cg_mode == 1) return false;
    if (c->cg_mode == 2) return true;
    return c->V <= WD_EO_ONELAUNCH_MAX_SITES;
}

static int eo_bicgstab_onelaunch(wd_ctx *c, const void *U_eo, const void *eta_eo, void *psi_eo, double kappa, double r_min,
                                 int max_iter)
{
    const EoDims e = eo_dims(c);
    int best = 0;
    double best_waste = 1e300;
    for (int t = 0; t < WD_NUM_EO1_TILES; ++t) {
        double blocks = 1.0, threads = 1.0;
        for (int d = 0; d < 4; ++d) {
            blocks *= (e.hd[d] + kEo1Tiles[t][d] - 1) / kEo1Tiles[t][d];
            threads *= kEo1Tiles[t][d];
        }
        const double waste = blocks * threads / (double)e.Vh;
        if (waste < best_waste - 1e-12) { best_waste = waste; best = t; }
    }
    const size_t hs = half_spinor_bytes(c), hg = half_gauge_bytes(c);
    EoOneLaunchArgs a;
    a.g = make_geom_lattice(e.hd, c->bc_t, kEo1Tiles[best], 0, c->l2_budget_mb);
    a.g.eo = 1;
    a.sm_count = c->sm_count;
    a.stream = c->stream;
    a.Ue = U_eo; a.Uo = (const char *)U_eo + hg;
    a.eta_e = eta_eo; a.eta_o = (const char *)eta_eo + hs;
    a.psi_e = psi_eo; a.psi_o = (char *)psi_eo + hs;
    a.r = c->r; a.p = c->p; a.v = c->q; a.s = c->y; a.t = c->w7; a.to = c->w5; a.etah = c->w6;
    a.kappa = kappa; a.sc = c->sc; a.partials = c->partials; a.partials_cap = c->partials_cap; a.hist = hist_whole(c, max_iter);
    a.r_min = r_min; a.max_iter = max_iter;
    c->launches++;
    CUDA_TRY(c, c->precision == 32 ? launch_eo_bicgstab_onelaunch_f32(best, a) : launch_eo_bicgstab_onelaunch_f64(best, a));
    return WD_OK;
}

extern "C" int bicgstab_solve_eo(wd_ctx *c, const void *U_eo, const void *eta_eo, void *psi_eo, double kappa, double r_min,
                                 int max_iter, wd_cg_info *info)
{
    if (!c) return WD_ERR_ARG;
    if (!U_eo || !eta_eo || !psi_eo || eta_eo == psi_eo) return fail(c, WD_ERR_ARG, "bicgstab_solve_eo: NULL argument or output aliases eta");
    if (!std::isfinite(kappa)) return fail(c, WD_ERR_ARG, "bicgstab_solve_eo: kappa is not finite");
    if (!(r_min > 0.0) || !std::isfinite(r_min)) return fail(c, WD_ERR_ARG, "bicgstab_solve_eo: r_min must be > 0");
    if (max_iter < 0) return fail(c, WD_ERR_ARG, "bicgstab_solve_eo: max_iter < 0");
    int rc = eo_check(c, "bicgstab_solve_eo");
    if (rc != WD_OK) return rc;
    rc = wd_ensure_workspace(c, max_iter);
    if (rc != WD_OK) return rc;
    if (!c->w5) {
        CUDA_TRY(c, cudaMalloc(&c->w5, spinor_bytes(c)));
        CUDA_TRY(c, cudaMemsetAsync(c->w5, 0, spinor_bytes(c), c->stream));
    }
    if (!c->w6) {
        CUDA_TRY(c, cudaMalloc(&c->w6, half_spinor_bytes(c)));
        CUDA_TRY(c, cudaMemsetAsync(c->w6, 0, half_spinor_bytes(c), c->stream));   // pad lanes stay zero
    }
    if (!c->w7) {
        CUDA_TRY(c, cudaMalloc(&c->w7, half_spinor_bytes(c)));
        CUDA_TRY(c, cudaMemsetAsync(c->w7, 0, half_spinor_bytes(c), c->stream));   // pad lanes stay zero
    }
    if (!c->eo_n2) CUDA_TRY(c, cudaMalloc(&c->eo_n2, 2 * sizeof(double)));
    if (c->profile && !c->bev[0])
        for (int j = 0; j < 8; ++j) CUDA_TRY(c, cudaEventCreate(&c->bev[j]));
    c->launches = 0;
    CUDA_TRY(c, cudaEventRecord(c->ev[0], c->stream));
    const bool one = eo_use_onelaunch(c);
    if (one) rc = eo_bicgstab_onelaunch(c, U_eo, eta_eo, psi_eo, kappa, r_min, max_iter);
    else rc = c->precision == 32 ? eo_bicgstab_loop<float>(c, U_eo, eta_eo, psi_eo, kappa, r_min, max_iter)
                                 : eo_bicgstab_loop<double>(c, U_eo, eta_eo, psi_eo, kappa, r_min, max_iter);
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
        info->cg_mode = one ? 8 : 7;
    }
    return s.converged ? WD_OK : (s.breakdown ? WD_BREAKDOWN : WD_NOT_CONVERGED);
}

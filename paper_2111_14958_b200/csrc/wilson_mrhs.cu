// wilson_mrhs.cu — C ABI of the multi-right-hand-side calls: wd_apply_multi, cg_solve_multi.
// The sources are independent problems D psi_j = eta_j sharing one gauge field; they are processed in groups of 4
// (then 2, then singly through the plain path) so that every link is loaded once per group.
#include "wilson_ctx.cuh"
#include "wilson_mrhs.cuh"

#include <cmath>
#include <cstdlib>

using namespace wd;

namespace {

int mrhs_tile_for(const wd_ctx *c, int nrhs)
{
    const int per_sm = c->precision == 32 ? 512 : 256;
    int best = -1;
    double best_waste = 1e300;
    for (int t = 0; t < WD_NUM_MRHS_TILES; ++t) {
        double blocks = 1.0, sites = 1.0;
        for (int d = 0; d < 4; ++d) {
            blocks *= (c->dims[d] + kMrhsTiles[t][d] - 1) / kMrhsTiles[t][d];
            sites *= kMrhsTiles[t][d];
        }
        if (sites * nrhs > per_sm) continue;
        const double waste = blocks * sites / (double)c->V;
        if (waste < best_waste - 1e-12) { best_waste = waste; best = t; }
    }
    return best;
}

cudaError_t mrhs_launch(wd_ctx *c, int nrhs, int dagger, int mode, const void *U, const void *in, void *out, void *r,
                        double kappa, CgScalars *sc, double *hist, int hist_stride, int it)
{
    const int tile = mrhs_tile_for(c, nrhs);
    if (tile < 0) return cudaErrorInvalidValue;
    MrhsArgs a;
    a.g = make_geom_lattice(c->dims, c->bc_t, kMrhsTiles[tile], c->zchunk_user, c->l2_budget_mb / nrhs * 2);
    a.sm_count = c->sm_count;
    a.stream = c->stream;
    a.U = U; a.in = in; a.out = out; a.r = r;
    a.stride = spinor_vecs(c);
    a.kappa = kappa;
    a.sc = sc; a.partials = c->partials; a.counter = c->counter; a.hist = hist; a.hist_stride = hist_stride; a.it = it;
    c->launches++;
    return c->precision == 32 ? launch_mrhs_f32(tile, nrhs, dagger, mode, a) : launch_mrhs_f64(tile, nrhs, dagger, mode, a);
}

int ensure_multi(wd_ctx *c, int max_iter)
{
    const size_t need = 4 * spinor_bytes(c);   // a group holds at most 4 sources
    if (c->m_bytes < need) {
        for (int j = 0; j < 4; ++j) {
            if (c->m_ws[j]) cudaFree(c->m_ws[j]);
            c->m_ws[j] = nullptr;
        }
        c->m_bytes = 0;
        for (int j = 0; j < 4; ++j) {
            CUDA_TRY(c, cudaMalloc(&c->m_ws[j], need));
            CUDA_TRY(c, cudaMemsetAsync(c->m_ws[j], 0, need, c->stream));
        }
        c->m_bytes = need;
    }
    if (!c->m_sc) {
        CUDA_TRY(c, cudaMalloc(&c->m_sc, 4 * sizeof(CgScalars)));
        CUDA_TRY(c, cudaMallocHost(&c->m_sc_host, 4 * sizeof(CgScalars)));
        CUDA_TRY(c, cudaMalloc(&c->m_counter, 4 * sizeof(unsigned int)));
        CUDA_TRY(c, cudaMemsetAsync(c->m_counter, 0, 4 * sizeof(unsigned int), c->stream));
    }
    if (c->m_hist_cap < hist_len(max_iter)) {
        if (c->m_hist) cudaFree(c->m_hist);
        c->m_hist = nullptr;
        c->m_hist_cap = 0;
        CUDA_TRY(c, cudaMalloc(&c->m_hist, 4 * sizeof(double) * (size_t)hist_len(max_iter)));
        c->m_hist_cap = hist_len(max_iter);
    }
    return WD_OK;
}

// one group of g in {2, 4} sources
template <typename real>
int cg_group(wd_ctx *c, int g, const void *U, const void *eta, void *psi, double kappa, double r_min, int max_iter,
             wd_cg_info *infos)
{
    using svec = typename Field<real>::svec;
    const size_t n = spinor_vecs(c), stride = n;
    svec *r = (svec *)c->m_ws[0], *p = (svec *)c->m_ws[1], *q = (svec *)c->m_ws[2], *y = (svec *)c->m_ws[3];
    const dim3 vgrid(wd_vec_grid(c, n, WD_VEC_PER_SM, g), g), ugrid(wd_vec_grid(c, n, WD_UPD_PER_SM, g), g);
    const int hs = c->m_hist_cap;
    CUDA_TRY(c, cudaEventRecord(c->ev[0], c->stream));
    cg_init_mrhs_kernel<real><<<vgrid, VEC_NT, 0, c->stream>>>((const svec *)eta, y, r, p, n, stride, c->V, padded(c), c->m_sc,
                                                              c->partials, c->m_counter, c->m_hist, hs, r_min, max_iter);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    const int poll = c->poll > 0 ? c->poll : 8;
    int launched = 0;
    while (launched < max_iter) {
        const int chunk = (max_iter - launched) < poll ? (max_iter - launched) : poll;
        for (int i = 0; i < chunk; ++i) {
            const int it = launched + i;
            const bool ev = c->profile && i == 0;
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[0], c->stream));
            CUDA_TRY(c, mrhs_launch(c, g, 1, MODE_QQ, U, p, q, nullptr, kappa, c->m_sc, c->m_hist, hs, it));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[1], c->stream));
            CUDA_TRY(c, mrhs_launch(c, g, 0, MODE_RUPD, U, q, nullptr, r, kappa, c->m_sc, (long)it + 1 < (long)hs ? c->m_hist : nullptr, hs, it));
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[2], c->stream));
            cg_update_mrhs_kernel<real><<<ugrid, VEC_NT, 0, c->stream>>>(y, p, r, n, stride, c->m_sc, it);
            c->launches++;
            CUDA_TRY(c, cudaGetLastError());
            if (ev) CUDA_TRY(c, cudaEventRecord(c->bev[3], c->stream));
        }
        CUDA_TRY(c, wd_fetch(c, c->m_sc_host, c->m_sc, g * sizeof(CgScalars)));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        int k_stop_max = 0;
        for (int j = 0; j < g; ++j)
            if (c->m_sc_host[j].k_stop > k_stop_max) k_stop_max = c->m_sc_host[j].k_stop;
        if (c->profile && launched < k_stop_max) {
            for (int j = 0; j < 3; ++j) {
                float ms = 0.f;
                CUDA_TRY(c, cudaEventElapsedTime(&ms, c->bev[j], c->bev[j + 1]));
                c->bprof_ms[j] += ms;
            }
            c->bprof_n++;
        }
        launched += chunk;
        if (k_stop_max <= launched) break;
    }
    CUDA_TRY(c, mrhs_launch(c, g, 1, MODE_PLAIN, U, y, psi, nullptr, kappa, c->m_sc, nullptr, 0, 0));
    CUDA_TRY(c, cudaEventRecord(c->ev[1], c->stream));
    CUDA_TRY(c, wd_fetch(c, c->m_sc_host, c->m_sc, g * sizeof(CgScalars)));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    float ms = 0.f;
    CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]));
    int status = WD_OK;
    for (int j = 0; j < g; ++j) {
        const CgScalars &s = c->m_sc_host[j];
        if (!s.converged && status != WD_BREAKDOWN) status = s.breakdown ? WD_BREAKDOWN : WD_NOT_CONVERGED;
        if (infos) {
            infos[j].iterations = s.k;
            infos[j].converged = s.converged;
            infos[j].rel_residual = s.eta2 > 0.0 ? std::sqrt(s.rr / s.eta2) : 0.0;
            infos[j].eta_norm2 = s.eta2;
            infos[j].gpu_ms = ms;      // device time of the whole group
            infos[j].total_ms = ms;
            infos[j].kernel_launches = c->launches;
            infos[j].cg_mode = 5;
        }
    }
    return status;
}

}  // namespace

extern "C" int wd_apply_multi(wd_ctx *c, const void *U, const void *in, void *out, int nrhs, double kappa, int dagger)
{
    if (!c) return WD_ERR_ARG;
    if (!U || !in || !out || in == out || nrhs < 1) return fail(c, WD_ERR_ARG, "wd_apply_multi: NULL or aliased argument, or nrhs < 1");
    if (!std::isfinite(kappa)) return fail(c, WD_ERR_ARG, "wd_apply_multi: kappa is not finite");
    if (c->recon != 18) return fail(c, WD_ERR_ARG, "wd_apply_multi: 18-real links only (wd_set_gauge_recon)");
    const size_t sb = spinor_bytes(c);
    int done = 0;
    while (done < nrhs) {
        const int left = nrhs - done, g = left >= 4 ? 4 : (left >= 2 ? 2 : 1);
        const char *gi = (const char *)in + (size_t)done * sb;
        char *go = (char *)out + (size_t)done * sb;
        if (g == 1 || mrhs_tile_for(c, g) < 0) {
            for (int j = 0; j < g; ++j) {
                int rc = wd_apply(c, U, gi + (size_t)j * sb, go + (size_t)j * sb, kappa, dagger);
                if (rc != WD_OK) return rc;
            }
        } else {
            CUDA_TRY(c, mrhs_launch(c, g, dagger ? 1 : 0, MODE_PLAIN, U, gi, go, nullptr, kappa, nullptr, nullptr, 0, 0));
        }
        done += g;
    }
    return WD_OK;
}

extern "C" int cg_solve_multi(wd_ctx *c, const void *U, const void *eta, void *psi, int nrhs, double kappa, double r_min,
                              int max_iter, wd_cg_info *infos)
{
    if (!c) return WD_ERR_ARG;
    if (!U || !eta || !psi || eta == psi || nrhs < 1) return fail(c, WD_ERR_ARG, "cg_solve_multi: NULL or aliased argument, or nrhs < 1");
    if (!std::isfinite(kappa)) return fail(c, WD_ERR_ARG, "cg_solve_multi: kappa is not finite");
    if (!(r_min > 0.0) || !std::isfinite(r_min)) return fail(c, WD_ERR_ARG, "cg_solve_multi: r_min must be > 0");
    if (max_iter < 0) return fail(c, WD_ERR_ARG, "cg_solve_multi: max_iter < 0");
    if (c->recon != 18) return fail(c, WD_ERR_ARG, "cg_solve_multi: 18-real links only (wd_set_gauge_recon)");
    if (c->profile && !c->bev[0])
        for (int j = 0; j < 8; ++j) CUDA_TRY(c, cudaEventCreate(&c->bev[j]));
    const size_t sb = spinor_bytes(c);
    int status = WD_OK, done = 0;
    c->launches = 0;
    while (done < nrhs) {
        const int left = nrhs - done, g = left >= 4 ? 4 : (left >= 2 ? 2 : 1);
        const char *ge = (const char *)eta + (size_t)done * sb;
        char *gp = (char *)psi + (size_t)done * sb;
        wd_cg_info *gi = infos ? infos + done : nullptr;
        if (g == 1 || mrhs_tile_for(c, g) < 0) {
            for (int j = 0; j < g; ++j) {
                const int rc = cg_solve(c, U, ge + (size_t)j * sb, gp + (size_t)j * sb, kappa, r_min, max_iter, gi ? gi + j : nullptr);
                if (rc < 0) return rc;
                if (rc != WD_OK) status = rc;
            }
        } else {
            int rc = ensure_multi(c, max_iter);
            if (rc != WD_OK) return rc;
            rc = c->precision == 32 ? cg_group<float>(c, g, U, ge, gp, kappa, r_min, max_iter, gi)
                                    : cg_group<double>(c, g, U, ge, gp, kappa, r_min, max_iter, gi);
            if (rc < 0) return rc;
            if (rc != WD_OK) status = rc;
        }
        done += g;
    }
    return status;
}

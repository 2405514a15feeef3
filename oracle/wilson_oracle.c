/*
 * wilson_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU fp64 implementation of what the hot path computes:
 * the 4D Wilson-Dirac operator D / D-dagger and the paper's conjugate-gradient solve of
 * D psi = eta through D D-dagger.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code, header, table or
 * helper with the CUDA path under paper_2111_14958_b200/csrc and includes nothing of it.
 *
 * Sources (the paper is /root/reference/PAPER.md; SURVEY.md section 8(c) fixes the readings
 * where the paper is silent — each is listed in DESIGN.md "Readings"):
 *   - linear system D psi = eta, colour A,B in 0..2, spin alpha,beta in 0..3: PAPER.md:27-32 (Eq. 1)
 *   - gamma5-hermiticity, "solve for D D-dagger, then multiply the solution by D-dagger": PAPER.md:44 (section 2)
 *   - CG listing: PAPER.md:46-48
 *   - the operator itself is only cited (Ref. [5]); reading C-1:
 *       (D psi)(x) = psi(x) - kappa sum_mu [ s+ (1 - gamma_mu) U_mu(x)        psi(x+mu)
 *                                          + s- (1 + gamma_mu) U_mu(x-mu)^dag  psi(x-mu) ]
 *       D-dagger: gamma_mu -> -gamma_mu.  s+- = -1 on the hop that wraps an antiperiodic t boundary.
 *   - gamma basis: reading C-2 (chiral basis, gamma5 = diag(1,1,-1,-1)).
 *
 * No blocking, fusion or reordering: one loop over sites, inside it one loop over the four
 * directions, the full 4x4 matrices (1 -+ gamma_mu), plain summation.  OpenMP is used only
 * to spread the site loop over cores.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): dense 12V x 12V matrix on 2^4 and 4x3x2x4 built
 * from Kronecker blocks (P1), gamma5-hermiticity (P2), free-field plane-wave eigenvalue (P3),
 * gauge covariance (P4), per-direction unitarity (P5), CG vs dense LU solve + monotone error
 * (P6), finite termination in the free field (P7), closed-form inverse incl. point source by
 * FFT (P8), residual identity (P10), COO route with N_NZ = 588 V (P11).
 * Iteration counts of the five BASELINE configs: parity unpinned by the paper (it prints none).
 *
 * Canonical layouts (x fastest): site s = x + Lx (y + Ly (z + Lz t));
 *   U[s][mu][a][b] complex (U_mu(x) sits on the link x -> x+mu), psi[s][alpha][a] complex.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex cplx;

/* Reading C-2: rows of gamma_x, gamma_y, gamma_z, gamma_t. */
static const cplx GAMMA[4][4][4] = {
    {{0, 0, 0, I}, {0, 0, I, 0}, {0, -I, 0, 0}, {-I, 0, 0, 0}},
    {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    {{0, 0, I, 0}, {0, 0, 0, -I}, {-I, 0, 0, 0}, {0, I, 0, 0}},
    {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}},
};

static long site_of(const int L[4], const int x[4])
{
    return x[0] + (long)L[0] * (x[1] + (long)L[1] * (x[2] + (long)L[2] * x[3]));
}

/* out[12] = (D psi)(s) or (D-dagger psi)(s), reading C-1, full 4x4 projectors. */
static void wd_site(const int L[4], int bc_t, const cplx *U, const cplx *psi, double kappa,
                    int dagger, long s, cplx out[12])
{
    int x[4];
    long rem = s;
    for (int d = 0; d < 4; ++d) {
        x[d] = (int)(rem % L[d]);
        rem /= L[d];
    }
    const double g = dagger ? -1.0 : 1.0; /* D-dagger: gamma_mu -> -gamma_mu */
    cplx acc[4][3];
    memset(acc, 0, sizeof acc);

    for (int mu = 0; mu < 4; ++mu) {
        cplx w[4][3];
        int y[4];

        /* forward hop: sigma+ (1 - g gamma_mu) (x) U_mu(x) psi(x+mu) */
        memcpy(y, x, sizeof y);
        y[mu] = (x[mu] + 1) % L[mu];
        double sig = (mu == 3 && bc_t == -1 && x[3] == L[3] - 1) ? -1.0 : 1.0;
        const cplx *Uf = U + (s * 4 + mu) * 9;
        const cplx *pf = psi + site_of(L, y) * 12;
        for (int b = 0; b < 4; ++b)
            for (int a = 0; a < 3; ++a) {
                cplx t = 0;
                for (int c = 0; c < 3; ++c) t += Uf[a * 3 + c] * pf[b * 3 + c];
                w[b][a] = t;
            }
        for (int al = 0; al < 4; ++al)
            for (int a = 0; a < 3; ++a) {
                cplx t = 0;
                for (int b = 0; b < 4; ++b) t += ((al == b ? 1.0 : 0.0) - g * GAMMA[mu][al][b]) * w[b][a];
                acc[al][a] += sig * t;
            }

        /* backward hop: sigma- (1 + g gamma_mu) (x) U_mu(x-mu)^dagger psi(x-mu) */
        memcpy(y, x, sizeof y);
        y[mu] = (x[mu] - 1 + L[mu]) % L[mu];
        sig = (mu == 3 && bc_t == -1 && x[3] == 0) ? -1.0 : 1.0;
        long sb = site_of(L, y);
        const cplx *Ub = U + (sb * 4 + mu) * 9;
        const cplx *pb = psi + sb * 12;
        for (int b = 0; b < 4; ++b)
            for (int a = 0; a < 3; ++a) {
                cplx t = 0;
                for (int c = 0; c < 3; ++c) t += conj(Ub[c * 3 + a]) * pb[b * 3 + c];
                w[b][a] = t;
            }
        for (int al = 0; al < 4; ++al)
            for (int a = 0; a < 3; ++a) {
                cplx t = 0;
                for (int b = 0; b < 4; ++b) t += ((al == b ? 1.0 : 0.0) + g * GAMMA[mu][al][b]) * w[b][a];
                acc[al][a] += sig * t;
            }
    }
    for (int al = 0; al < 4; ++al)
        for (int a = 0; a < 3; ++a) out[al * 3 + a] = psi[s * 12 + al * 3 + a] - kappa * acc[al][a];
}

static long volume_of(const int L[4]) { return (long)L[0] * L[1] * L[2] * L[3]; }

/* out = D psi (dagger = 0) or D-dagger psi (dagger = 1) on the whole lattice. out must not alias psi. */
int oracle_wd_apply(const int L[4], int bc_t, const double *U, const double *psi, double *out,
                    double kappa, int dagger)
{
    if (!L || !U || !psi || !out || psi == out) return -1;
    for (int d = 0; d < 4; ++d)
        if (L[d] < 2) return -2;
    const long V = volume_of(L);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s)
        wd_site(L, bc_t, (const cplx *)U, (const cplx *)psi, kappa, dagger, s, (cplx *)out + s * 12);
    return 0;
}

/* Same operator evaluated only at the listed sites: out[i][12] = (D psi)(sites[i]). */
int oracle_wd_apply_sites(const int L[4], int bc_t, const double *U, const double *psi, double *out,
                          double kappa, int dagger, const long *sites, long n_sites)
{
    if (!L || !U || !psi || !out || !sites) return -1;
    const long V = volume_of(L);
    for (long i = 0; i < n_sites; ++i)
        if (sites[i] < 0 || sites[i] >= V) return -3;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n_sites; ++i)
        wd_site(L, bc_t, (const cplx *)U, (const cplx *)psi, kappa, dagger, sites[i], (cplx *)out + i * 12);
    return 0;
}

/* <a,a> = sum over all 12V components of |a|^2, plain summation (per-thread partial sums under OpenMP). */
static double norm2(const cplx *a, long n)
{
    double acc = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : acc)
    for (long i = 0; i < n; ++i) acc += creal(a[i]) * creal(a[i]) + cimag(a[i]) * cimag(a[i]);
    return acc;
}

double oracle_norm2(const double *a, long n_complex) { return norm2((const cplx *)a, n_complex); }

typedef struct {
    int iterations;        /* k: completed loop bodies */
    int converged;         /* sqrt(rr) < r_min sqrt(eta2) at exit */
    double rel_residual;   /* sqrt(rr/eta2), rr the recursed residual */
    double eta_norm2;      /* <eta,eta> */
    double seconds;        /* wall time of the loop + final D-dagger */
} oracle_cg_info;

/*
 * CG listing of PAPER.md:46-48 with readings G1-G5:
 *   y <- 0; r <- eta; p <- r; rr <- <r,r>
 *   while sqrt(rr) >= r_min sqrt(<eta,eta>) and k < max_iter:
 *       q <- D-dagger p; alpha <- rr / <q,q>
 *       y <- y + alpha p
 *       r <- r - alpha D q; rr' <- <r,r>
 *       beta <- rr'/rr; p <- r + beta p; rr <- rr'; k <- k+1
 *   psi <- D-dagger y
 * rr_history (optional, length >= max_iter+1) receives rr after 0,1,...,k iterations.
 * Returns 0 converged, 1 max_iter reached, <0 bad argument / out of memory.
 */
int oracle_cg_solve(const int L[4], int bc_t, const double *U, const double *eta, double *psi_out,
                    double kappa, double r_min, int max_iter, oracle_cg_info *info, double *rr_history)
{
    if (!L || !U || !eta || !psi_out || max_iter < 0 || !(r_min > 0.0)) return -1;
    for (int d = 0; d < 4; ++d)
        if (L[d] < 2) return -2;
    const long n = volume_of(L) * 12;
    const cplx *b = (const cplx *)eta;
    cplx *y = calloc((size_t)n, sizeof(cplx));
    cplx *r = malloc((size_t)n * sizeof(cplx));
    cplx *p = malloc((size_t)n * sizeof(cplx));
    cplx *q = malloc((size_t)n * sizeof(cplx));
    cplx *s = malloc((size_t)n * sizeof(cplx));
    if (!y || !r || !p || !q || !s) {
        free(y); free(r); free(p); free(q); free(s);
        return -4;
    }
#ifdef _OPENMP
    double t0 = omp_get_wtime();
#endif
    memcpy(r, b, (size_t)n * sizeof(cplx));
    memcpy(p, b, (size_t)n * sizeof(cplx));
    double rr = norm2(r, n);
    const double eta2 = rr;
    int k = 0;
    if (rr_history) rr_history[0] = rr;

    if (eta2 > 0.0) {
        while (sqrt(rr) >= r_min * sqrt(eta2) && k < max_iter) {
            oracle_wd_apply(L, bc_t, U, (const double *)p, (double *)q, kappa, 1); /* q = D-dagger p */
            const double qq = norm2(q, n);
            const double alpha = rr / qq;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) y[i] += alpha * p[i];
            oracle_wd_apply(L, bc_t, U, (const double *)q, (double *)s, kappa, 0); /* s = D q = D D-dagger p */
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) r[i] -= alpha * s[i];
            const double rr_new = norm2(r, n);
            const double beta = rr_new / rr;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
            rr = rr_new;
            ++k;
            if (rr_history) rr_history[k] = rr;
        }
    }
    oracle_wd_apply(L, bc_t, U, (const double *)y, psi_out, kappa, 1); /* psi = D-dagger y */
    const int converged = (eta2 == 0.0) || (sqrt(rr) < r_min * sqrt(eta2));
    if (info) {
        info->iterations = k;
        info->converged = converged;
        info->rel_residual = eta2 > 0.0 ? sqrt(rr / eta2) : 0.0;
        info->eta_norm2 = eta2;
#ifdef _OPENMP
        info->seconds = omp_get_wtime() - t0;
#else
        info->seconds = 0.0;
#endif
    }
    free(y); free(r); free(p); free(q); free(s);
    return converged ? 0 : 1;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

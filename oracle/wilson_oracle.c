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
 * FFT (P8), residual identity (P10), COO route with N_NZ = 588 V (P11); BiCGSTAB (B-P1..4), even-odd CG (E-P1..4),
 * even-odd BiCGSTAB (EB-P1..3): dense solves and dense-matrix retyping of the first iterates on 2^4.
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

/* <a,b> = sum conj(a_i) b_i, plain summation. */
static cplx cdot(const cplx *a, const cplx *b, long n)
{
    double re = 0.0, im = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : re, im)
    for (long i = 0; i < n; ++i) {
        const cplx t = conj(a[i]) * b[i];
        re += creal(t);
        im += cimag(t);
    }
    return re + im * I;
}

/*
 * BiCGSTAB on D directly.  The paper only NAMES the method ("the
 * biconjugate gradient stabilized method (BiCGSTAB)", general reference [8]) and prints no listing;
 * reading B1 of DESIGN.md: the standard unpreconditioned listing with shadow residual rhat = r0,
 * psi0 = 0, complex inner products <a,b> = sum conj(a) b, and the same relative stopping test as
 * the CG (reading G4), evaluated at the top of the loop:
 *   psi <- 0; r <- eta; rhat <- r; p <- r; rho <- <rhat,r>
 *   while sqrt(<r,r>) >= r_min sqrt(<eta,eta>) and k < max_iter:
 *       v <- D p;           alpha <- rho / <rhat,v>
 *       s <- r - alpha v
 *       t <- D s;           omega <- <t,s> / <t,t>
 *       psi <- psi + alpha p + omega s
 *       r <- s - omega t;   rho' <- <rhat,r>
 *       beta <- (rho'/rho)(alpha/omega);  p <- r + beta (p - omega v);  rho <- rho';  k <- k+1
 * A breakdown (rho, <rhat,v>, <t,t> or omega exactly 0 or not finite) leaves the loop: returns 2.
 * Pins (tests/test_oracle_pins.py): dense LU solve on 2^4 (B-P1), first iterate from the dense matrix
 * (B-P2), termination in <= 2 iterations on a free-field plane wave whose 4x4 symbol has two distinct
 * eigenvalues and in 1 iteration at kappa = 0 (B-P3), closed-form plane-wave-sum inverse (B-P4).
 * Returns 0 converged, 1 max_iter reached, 2 breakdown, <0 bad argument / out of memory.
 */
int oracle_bicgstab_solve(const int L[4], int bc_t, const double *U, const double *eta, double *psi_out,
                          double kappa, double r_min, int max_iter, oracle_cg_info *info, double *rr_history)
{
    if (!L || !U || !eta || !psi_out || max_iter < 0 || !(r_min > 0.0)) return -1;
    for (int d = 0; d < 4; ++d)
        if (L[d] < 2) return -2;
    const long n = volume_of(L) * 12;
    const cplx *b = (const cplx *)eta;
    cplx *x = (cplx *)psi_out;
    cplx *r = malloc((size_t)n * sizeof(cplx));
    cplx *p = malloc((size_t)n * sizeof(cplx));
    cplx *v = malloc((size_t)n * sizeof(cplx));
    cplx *s = malloc((size_t)n * sizeof(cplx));
    cplx *t = malloc((size_t)n * sizeof(cplx));
    if (!r || !p || !v || !s || !t) {
        free(r); free(p); free(v); free(s); free(t);
        return -4;
    }
#ifdef _OPENMP
    double t0 = omp_get_wtime();
#endif
    memset(x, 0, (size_t)n * sizeof(cplx));
    memcpy(r, b, (size_t)n * sizeof(cplx));
    memcpy(p, b, (size_t)n * sizeof(cplx));
    const cplx *rhat = b; /* rhat = r0 = eta */
    double rr = norm2(r, n);
    const double eta2 = rr;
    cplx rho = rr; /* <rhat,r0> = <eta,eta> */
    int k = 0, breakdown = 0;
    if (rr_history) rr_history[0] = rr;

    if (eta2 > 0.0) {
        while (sqrt(rr) >= r_min * sqrt(eta2) && k < max_iter) {
            oracle_wd_apply(L, bc_t, U, (const double *)p, (double *)v, kappa, 0); /* v = D p */
            const cplx rv = cdot(rhat, v, n);
            if (rv == 0.0 || rho == 0.0) { breakdown = 1; break; }
            const cplx alpha = rho / rv;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) s[i] = r[i] - alpha * v[i];
            oracle_wd_apply(L, bc_t, U, (const double *)s, (double *)t, kappa, 0); /* t = D s */
            const double tt = norm2(t, n);
            if (tt == 0.0) { /* s = 0: psi + alpha p is exact */
#pragma omp parallel for schedule(static)
                for (long i = 0; i < n; ++i) x[i] += alpha * p[i];
                memset(r, 0, (size_t)n * sizeof(cplx));
                rr = 0.0;
                ++k;
                if (rr_history) rr_history[k] = rr;
                break;
            }
            const cplx omega = cdot(t, s, n) / tt;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) x[i] += alpha * p[i] + omega * s[i];
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) r[i] = s[i] - omega * t[i];
            const cplx rho_new = cdot(rhat, r, n);
            rr = norm2(r, n);
            ++k;
            if (rr_history) rr_history[k] = rr;
            if (omega == 0.0 || !isfinite(creal(omega)) || !isfinite(cimag(omega))) { breakdown = 1; break; }
            const cplx beta = (rho_new / rho) * (alpha / omega);
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) p[i] = r[i] + beta * (p[i] - omega * v[i]);
            rho = rho_new;
        }
    }
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
    free(r); free(p); free(v); free(s); free(t);
    return converged ? 0 : (breakdown ? 2 : 1);
}

/*
 * Even-odd (Schur) preconditioned CG (the paper: "the solver performance is often improved by
 * preconditioning", and "can be further improved designing algorithms more suitable for the Dirac
 * operator").  Reading E1 of DESIGN.md.  Sites are coloured by the parity of x+y+z+t (all extents even).
 * The hopping term only connects opposite parities, D = [[1, -kappa H_eo], [-kappa H_oe, 1]], so D psi = eta is
 *     Mhat psi_e = etahat,   Mhat = 1 - kappa^2 H_eo H_oe,   etahat = eta_e + kappa H_eo eta_o,
 *     psi_o = eta_o + kappa H_oe psi_e.
 * Mhat is solved with the paper's CG recurrence (readings G1-G5) applied to Mhat Mhat-dagger
 * (Mhat-dagger = 1 - kappa^2 H-dagger_eo H-dagger_oe, H-dagger = gamma_mu -> -gamma_mu), then psi_e = Mhat-dagger y.
 * Stopping test: sqrt(<r,r>) < r_min sqrt(<eta,eta>) with eta the FULL source; because the odd rows of
 * eta - D psi vanish identically, <r,r> is the squared true residual of the full system, so r_min means what it
 * means in oracle_cg_solve.
 * Written on full-lattice arrays: a field "on the even sites" is a full field that is zero on the odd sites, and
 * H_oe v is simply (H v) for such a v (H maps even-supported fields to odd-supported ones).  No parity indexing.
 * Pins: the Schur operator against the dense blocks D_ee - D_eo D_oe of the Kronecker-built matrix (E-P1), the
 * solution against the dense LU solve and the unpreconditioned oracle (E-P2), fewer iterations than the plain CG
 * and finite termination counted from the dense spectrum (E-P3).
 */
static int parity_of(const int L[4], long s)
{
    int par = 0;
    for (int d = 0; d < 4; ++d) { par += (int)(s % L[d]); s /= L[d]; }
    return par & 1;
}

/* out = H in (dagger = 0) or H-dagger in: the hopping sum of reading C-1 without the diagonal and without kappa,
 * i.e. D = 1 - kappa H.  Obtained from the one-site routine as (in - D in) at kappa = 1. */
static void hop_apply(const int L[4], int bc_t, const cplx *U, const cplx *in, cplx *out, int dagger)
{
    const long V = volume_of(L);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s) {
        cplx d[12];
        wd_site(L, bc_t, U, in, 1.0, dagger, s, d);
        for (int i = 0; i < 12; ++i) out[s * 12 + i] = in[s * 12 + i] - d[i];
    }
}

/* out = Mhat v (dagger = 0) or Mhat-dagger v for an even-supported v: v - kappa^2 H (H v).  tmp: scratch field. */
static void schur_apply(const int L[4], int bc_t, const cplx *U, const cplx *v, cplx *out, cplx *tmp, double kappa,
                        int dagger)
{
    const long n = volume_of(L) * 12;
    hop_apply(L, bc_t, U, v, tmp, dagger);   /* odd-supported */
    hop_apply(L, bc_t, U, tmp, out, dagger); /* even-supported */
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) out[i] = v[i] - kappa * kappa * out[i];
}

/* Mhat (or Mhat-dagger) applied to the even part of `in`; the odd sites of out are zero.  For the pins. */
int oracle_schur_apply(const int L[4], int bc_t, const double *U, const double *in, double *out, double kappa,
                       int dagger)
{
    if (!L || !U || !in || !out || in == out) return -1;
    for (int d = 0; d < 4; ++d)
        if (L[d] < 2 || (L[d] & 1)) return -2;
    const long V = volume_of(L);
    cplx *v = calloc((size_t)V * 12, sizeof(cplx)), *tmp = malloc((size_t)V * 12 * sizeof(cplx));
    if (!v || !tmp) { free(v); free(tmp); return -4; }
    for (long s = 0; s < V; ++s)
        if (parity_of(L, s) == 0) memcpy(v + s * 12, (const cplx *)in + s * 12, 12 * sizeof(cplx));
    schur_apply(L, bc_t, (const cplx *)U, v, (cplx *)out, tmp, kappa, dagger);
    free(v); free(tmp);
    return 0;
}

int oracle_cg_solve_eo(const int L[4], int bc_t, const double *U_, const double *eta_, double *psi_out,
                       double kappa, double r_min, int max_iter, oracle_cg_info *info, double *rr_history)
{
    if (!L || !U_ || !eta_ || !psi_out || max_iter < 0 || !(r_min > 0.0)) return -1;
    for (int d = 0; d < 4; ++d)
        if (L[d] < 2 || (L[d] & 1)) return -2;
    const long V = volume_of(L), n = V * 12;
    const cplx *U = (const cplx *)U_, *eta = (const cplx *)eta_;
    cplx *psi = (cplx *)psi_out;
    cplx *eo = calloc((size_t)n, sizeof(cplx)); /* eta_o, odd-supported */
    cplx *y = calloc((size_t)n, sizeof(cplx));
    cplx *r = calloc((size_t)n, sizeof(cplx));
    cplx *p = malloc((size_t)n * sizeof(cplx));
    cplx *q = malloc((size_t)n * sizeof(cplx));
    cplx *w = malloc((size_t)n * sizeof(cplx));
    cplx *tmp = malloc((size_t)n * sizeof(cplx));
    if (!eo || !y || !r || !p || !q || !w || !tmp) {
        free(eo); free(y); free(r); free(p); free(q); free(w); free(tmp);
        return -4;
    }
#ifdef _OPENMP
    double t0 = omp_get_wtime();
#endif
    const double eta2 = norm2(eta, n);
    /* etahat = eta_e + kappa H_eo eta_o  (stored in r: r <- etahat, psi0 = 0) */
    for (long s = 0; s < V; ++s)
        if (parity_of(L, s) == 1) memcpy(eo + s * 12, eta + s * 12, 12 * sizeof(cplx));
    hop_apply(L, bc_t, U, eo, tmp, 0); /* even-supported */
    for (long s = 0; s < V; ++s)
        if (parity_of(L, s) == 0)
            for (int i = 0; i < 12; ++i) r[s * 12 + i] = eta[s * 12 + i] + kappa * tmp[s * 12 + i];
    memcpy(p, r, (size_t)n * sizeof(cplx));
    double rr = norm2(r, n);
    int k = 0;
    if (rr_history) rr_history[0] = rr;
    if (eta2 > 0.0) {
        while (sqrt(rr) >= r_min * sqrt(eta2) && k < max_iter) {
            schur_apply(L, bc_t, U, p, q, tmp, kappa, 1); /* q = Mhat-dagger p */
            const double qq = norm2(q, n);
            const double alpha = rr / qq;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) y[i] += alpha * p[i];
            schur_apply(L, bc_t, U, q, w, tmp, kappa, 0); /* w = Mhat q */
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) r[i] -= alpha * w[i];
            const double rr_new = norm2(r, n);
            const double beta = rr_new / rr;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
            rr = rr_new;
            ++k;
            if (rr_history) rr_history[k] = rr;
        }
    }
    schur_apply(L, bc_t, U, y, q, tmp, kappa, 1); /* psi_e = Mhat-dagger y */
    hop_apply(L, bc_t, U, q, tmp, 0);             /* H_oe psi_e, odd-supported */
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) psi[i] = q[i] + eo[i] + kappa * tmp[i]; /* psi_e on even, eta_o + kappa H_oe psi_e on odd */
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
    free(eo); free(y); free(r); free(p); free(q); free(w); free(tmp);
    return converged ? 0 : 1;
}

/*
 * Even-odd preconditioned BiCGSTAB: the two SURVEY.md 8(f) rows composed (reading EB1 of DESIGN.md).  The Schur system
 * Mhat psi_e = etahat of reading E1 (above) is solved with the BiCGSTAB listing of reading B1 (oracle_bicgstab_solve)
 * applied to Mhat itself, shadow residual rhat = r0 = etahat, psi_e0 = 0; then psi_o = eta_o + kappa H_oe psi_e.
 * Stopping test as in oracle_cg_solve_eo: sqrt(<r,r>) < r_min sqrt(<eta,eta>) with the FULL source, r = etahat - Mhat psi_e
 * (the even rows of eta - D psi; the odd rows vanish identically), tested at the top of the loop.
 * Full-lattice arrays, even-supported fields, as in oracle_cg_solve_eo.
 * Pins (tests/test_oracle_pins.py): dense LU solve of the full system (EB-P1), first iterates retyped with the dense
 * Schur complement (EB-P2), kappa = 0 and agreement with the three other oracle solvers on the BASELINE configs (EB-P3).
 * Returns 0 converged, 1 max_iter reached, 2 breakdown, <0 bad argument / out of memory.
 */
int oracle_bicgstab_solve_eo(const int L[4], int bc_t, const double *U_, const double *eta_, double *psi_out,
                             double kappa, double r_min, int max_iter, oracle_cg_info *info, double *rr_history)
{
    if (!L || !U_ || !eta_ || !psi_out || max_iter < 0 || !(r_min > 0.0)) return -1;
    for (int d = 0; d < 4; ++d)
        if (L[d] < 2 || (L[d] & 1)) return -2;
    const long V = volume_of(L), n = V * 12;
    const cplx *U = (const cplx *)U_, *eta = (const cplx *)eta_;
    cplx *psi = (cplx *)psi_out;
    cplx *eo = calloc((size_t)n, sizeof(cplx));   /* eta_o, odd-supported */
    cplx *x = calloc((size_t)n, sizeof(cplx));    /* psi_e */
    cplx *rhat = calloc((size_t)n, sizeof(cplx)); /* etahat */
    cplx *r = malloc((size_t)n * sizeof(cplx));
    cplx *p = malloc((size_t)n * sizeof(cplx));
    cplx *v = malloc((size_t)n * sizeof(cplx));
    cplx *s = malloc((size_t)n * sizeof(cplx));
    cplx *t = malloc((size_t)n * sizeof(cplx));
    cplx *tmp = malloc((size_t)n * sizeof(cplx));
    if (!eo || !x || !rhat || !r || !p || !v || !s || !t || !tmp) {
        free(eo); free(x); free(rhat); free(r); free(p); free(v); free(s); free(t); free(tmp);
        return -4;
    }
#ifdef _OPENMP
    double t0 = omp_get_wtime();
#endif
    const double eta2 = norm2(eta, n);
    /* etahat = eta_e + kappa H_eo eta_o */
    for (long i = 0; i < V; ++i)
        if (parity_of(L, i) == 1) memcpy(eo + i * 12, eta + i * 12, 12 * sizeof(cplx));
    hop_apply(L, bc_t, U, eo, tmp, 0);
    for (long i = 0; i < V; ++i)
        if (parity_of(L, i) == 0)
            for (int j = 0; j < 12; ++j) rhat[i * 12 + j] = eta[i * 12 + j] + kappa * tmp[i * 12 + j];
    memcpy(r, rhat, (size_t)n * sizeof(cplx));
    memcpy(p, rhat, (size_t)n * sizeof(cplx));
    double rr = norm2(r, n);
    cplx rho = rr;
    int k = 0, breakdown = 0;
    if (rr_history) rr_history[0] = rr;
    if (eta2 > 0.0) {
        while (sqrt(rr) >= r_min * sqrt(eta2) && k < max_iter) {
            schur_apply(L, bc_t, U, p, v, tmp, kappa, 0); /* v = Mhat p */
            const cplx rv = cdot(rhat, v, n);
            if (rv == 0.0 || rho == 0.0) { breakdown = 1; break; }
            const cplx alpha = rho / rv;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) s[i] = r[i] - alpha * v[i];
            schur_apply(L, bc_t, U, s, t, tmp, kappa, 0); /* t = Mhat s */
            const double tt = norm2(t, n);
            if (tt == 0.0) { /* s = 0: psi_e + alpha p is exact */
#pragma omp parallel for schedule(static)
                for (long i = 0; i < n; ++i) x[i] += alpha * p[i];
                rr = 0.0;
                ++k;
                if (rr_history) rr_history[k] = rr;
                break;
            }
            const cplx omega = cdot(t, s, n) / tt;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) x[i] += alpha * p[i] + omega * s[i];
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) r[i] = s[i] - omega * t[i];
            const cplx rho_new = cdot(rhat, r, n);
            rr = norm2(r, n);
            ++k;
            if (rr_history) rr_history[k] = rr;
            if (omega == 0.0 || !isfinite(creal(omega)) || !isfinite(cimag(omega))) { breakdown = 1; break; }
            const cplx beta = (rho_new / rho) * (alpha / omega);
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) p[i] = r[i] + beta * (p[i] - omega * v[i]);
            rho = rho_new;
        }
    }
    hop_apply(L, bc_t, U, x, tmp, 0); /* H_oe psi_e, odd-supported */
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) psi[i] = x[i] + eo[i] + kappa * tmp[i];
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
    free(eo); free(x); free(rhat); free(r); free(p); free(v); free(s); free(t); free(tmp);
    return converged ? 0 : (breakdown ? 2 : 1);
}

/*
 * The paper's own data structure: D (dagger = 0) or D-dagger (dagger = 1) in
 * coordinate format, assembled entry by entry from reading C-1.  Vector index i = (s*4 + alpha)*3 + a.
 * Every row holds 1 + 8*2*3 = 49 entries (N_NZ = 588 V); entry k = row*49 + j with
 *   j = 0                         the diagonal, Val = 1
 *   j = 1 + (mu*2 + dir)*6 + n*3 + b,  dir 0 = forward hop, 1 = backward hop; n = 0,1 counts the two spin columns
 *       beta (ascending) in which row alpha of (1 -+ gamma_mu) is non-zero; b = colour column:
 *       forward : Val = -kappa sigma+ (1 - g gamma_mu)[alpha][beta] U_mu(x)[a][b],             Col = (x+mu, beta, b)
 *       backward: Val = -kappa sigma- (1 + g gamma_mu)[alpha][beta] conj(U_mu(x-mu)[b][a]),    Col = (x-mu, beta, b)
 *   (g = +1 for D, -1 for D-dagger).  val: 2*nnz doubles (re, im), row/col: nnz ints.
 */
long oracle_coo_nnz(const int L[4]) { return volume_of(L) * 588; }

int oracle_coo_assemble(const int L[4], int bc_t, const double *U_, double kappa, int dagger, double *val_,
                        int *row, int *col)
{
    if (!L || !U_ || !val_ || !row || !col) return -1;
    const cplx *U = (const cplx *)U_;
    cplx *val = (cplx *)val_;
    const long V = volume_of(L);
    if (V * 12 > 2147483647L) return -2;
    const double g = dagger ? -1.0 : 1.0;
    for (long s = 0; s < V; ++s) {
        int x[4];
        long rem = s;
        for (int d = 0; d < 4; ++d) { x[d] = (int)(rem % L[d]); rem /= L[d]; }
        for (int al = 0; al < 4; ++al)
            for (int a = 0; a < 3; ++a) {
                const long r = (s * 4 + al) * 3 + a;
                long k = r * 49;
                val[k] = 1.0; row[k] = (int)r; col[k] = (int)r; ++k;
                for (int mu = 0; mu < 4; ++mu)
                    for (int dir = 0; dir < 2; ++dir) {
                        int y[4];
                        memcpy(y, x, sizeof y);
                        y[mu] = dir == 0 ? (x[mu] + 1) % L[mu] : (x[mu] - 1 + L[mu]) % L[mu];
                        const long sn = site_of(L, y);
                        const int wraps = dir == 0 ? (x[3] == L[3] - 1) : (x[3] == 0);
                        const double sig = (mu == 3 && bc_t == -1 && wraps) ? -1.0 : 1.0;
                        const double sgn = dir == 0 ? -g : g; /* (1 - g gamma) forward, (1 + g gamma) backward */
                        int n = 0;
                        for (int be = 0; be < 4; ++be) {
                            const cplx pr = (al == be ? 1.0 : 0.0) + sgn * GAMMA[mu][al][be];
                            if (pr == 0.0) continue;
                            for (int b = 0; b < 3; ++b) {
                                const cplx u = dir == 0 ? U[(s * 4 + mu) * 9 + a * 3 + b]
                                                        : conj(U[(sn * 4 + mu) * 9 + b * 3 + a]);
                                val[k] = -kappa * sig * pr * u;
                                row[k] = (int)r;
                                col[k] = (int)((sn * 4 + be) * 3 + b);
                                ++k;
                            }
                            ++n;
                        }
                        if (n != 2) return -5; /* every row of (1 -+ gamma_mu) has exactly two non-zeros */
                    }
                if (k != (r + 1) * 49) return -5;
            }
    }
    return 0;
}

/* Alg. COO of PAPER.md:52-54, verbatim: for k = 1..N_NZ: out[Row[k]] = out[Row[k]] + Val[k]*in[Col[k]]. */
int oracle_coo_spmv(long nnz, const double *val_, const int *row, const int *col, const double *in_, double *out_,
                    long n_out)
{
    if (!val_ || !row || !col || !in_ || !out_) return -1;
    const cplx *val = (const cplx *)val_, *in = (const cplx *)in_;
    cplx *out = (cplx *)out_;
    for (long i = 0; i < n_out; ++i) out[i] = 0.0;
    for (long k = 0; k < nnz; ++k) out[row[k]] = out[row[k]] + val[k] * in[col[k]];
    return 0;
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

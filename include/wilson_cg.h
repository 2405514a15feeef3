/*
 * wilson_cg.h — C ABI of the B200-native Wilson-Dirac / CG library (libwilson_cg.so).
 *
 * The library is the hot path of arXiv:2111.14958 ("Implementation of the conjugate gradient
 * algorithm for heterogeneous systems"): the 4D Wilson-Dirac operator D / D-dagger as a
 * matrix-free stencil and the paper's conjugate gradient on D D-dagger, all of it hand-written
 * CUDA for sm_100a.  Citations are lines of the paper text and, where the paper is
 * silent, the readings listed in DESIGN.md ("Readings", G1..G18, C-1, C-2).
 *
 * Conventions common to every call
 * --------------------------------
 *  * Return value: 0 = WD_OK; < 0 = error (see WD_ERR_*); cg_solve* may also return
 *    +1 = WD_NOT_CONVERGED (max_iter reached; the current psi = D-dagger y has been written).
 *    No C++ exception crosses this boundary.  wd_last_error(ctx) gives a ctx-owned,
 *    NUL-terminated description of the last failure (valid until the next call on that ctx).
 *  * A "device pointer" is a CUDA device address in the current device's primary context
 *    (e.g. torch.Tensor.data_ptr()); a "host pointer" is ordinary host memory (pinned memory
 *    makes the copies faster but is not required).  Every buffer passed in is owned by the
 *    caller and is never freed, resized or (for inputs) written by the library.
 *  * The ctx owns its CG workspace (r, p, q, y, device scalars, reduction partials, staging
 *    buffers of the *_host calls), allocated lazily with cudaMalloc and freed by wd_destroy.
 *  * All device work is enqueued on the ctx stream given to wd_create.  wd_pack_*, wd_unpack_*,
 *    wd_apply are asynchronous on that stream; cg_solve, wd_norm2 and the *_host calls return
 *    after their result is available on the host.
 *  * A ctx is not thread-safe; use one ctx per host thread / stream.
 *
 * Canonical (caller-visible) layouts — x fastest, interleaved (re, im), element type float
 * (precision 32) or double (precision 64):
 *    site   s = x + Lx*(y + Ly*(z + Lz*t)),  dims = {Lx, Ly, Lz, Lt},  V = Lx*Ly*Lz*Lt
 *    spinor psi[s][alpha 0..3][a 0..2][2]            24 reals per site   (Eq. 1, PAPER.md:27-32:
 *                                                    alpha = spin index, a = colour index)
 *    gauge  U[s][mu 0..3][a 0..2][b 0..2][2]         72 reals per site;  mu = 0:x 1:y 2:z 3:t;
 *                                                    U_mu(x) sits on the link x -> x+mu, row a, col b.
 *
 * Native (internal, site-planar SoA) layouts — produced by wd_pack_*, consumed by wd_apply /
 * cg_solve; opaque to the caller except for their size (wd_*_native_bytes):
 *    sites are grouped in blocks of 16 consecutive site indices (the volume is padded up to a
 *    multiple of 16; pad lanes hold zeros); inside a block the data is planar:
 *    precision 32: spinor block = 6 planes x 16 sites of float4 (plane j holds complex components
 *                  2j, 2j+1 of the 12 = alpha*3+a), 1.5 KB;  gauge block = 4 links x 1152 B, 4.5 KB; a link is 4 planes
 *                  x 16 sites of float4 (reals 4q..4q+3 of the 18 = (a*3+b)*2+ri) followed by one plane x 16
 *                  sites of float2 (reals 16, 17).
 *    precision 64: spinor block = 12 planes of double2, gauge block = 36 planes of double2.
 *    Every per-thread access is one 128-bit (spinor) or 64/128-bit (gauge) load at a compile-time
 *    offset from the site's base address; 16 consecutive lanes read 256 contiguous bytes of a plane.
 *
 * The operator (reading C-1; the paper only cites Wilson, and states
 * gamma5 D gamma5 = D-dagger):
 *    (D psi)(x) = psi(x) - kappa sum_mu [ s+ (1 - gamma_mu) U_mu(x)          psi(x+mu)
 *                                       + s- (1 + gamma_mu) U_mu(x-mu)^dagger psi(x-mu) ]
 *    D-dagger: gamma_mu -> -gamma_mu.   x +- mu is taken modulo L_mu (periodic); in t the hop that
 *    wraps the boundary carries the factor bc_t (-1 antiperiodic, +1 periodic), applied in-kernel.
 *    gamma matrices: chiral basis of reading C-2 (gamma5 = diag(1,1,-1,-1)).
 */
#ifndef WILSON_CG_H
#define WILSON_CG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WD_OK 0
#define WD_NOT_CONVERGED 1
#define WD_BREAKDOWN 2       /* the loop stopped without converging and without reaching max_iter: a denominator of the
                                BiCGSTAB recurrence vanished, or (every solver) the residual norm is not a number because U,
                                eta or a step length is not finite; info->converged = 0, psi holds the last iterate */
#define WD_ERR_ARG (-1)     /* NULL pointer, aliasing out == in, non-finite kappa, r_min <= 0, max_iter < 0 */
#define WD_ERR_DIMS (-2)    /* an extent < 4 (forward and backward neighbours must be distinct sites) or volume too large */
#define WD_ERR_CUDA (-3)    /* a CUDA runtime call or kernel launch failed; wd_last_error() has the CUDA string */
#define WD_ERR_ALLOC (-4)   /* cudaMalloc / host allocation failed */
#define WD_ERR_PRECISION (-5) /* precision not 32 or 64 */

typedef struct wd_ctx wd_ctx; /* opaque */

/* Result record of cg_solve / cg_solve_host (host memory, written before the call returns). */
typedef struct wd_cg_info {
    int iterations;        /* k = number of completed CG loop bodies */
    int converged;         /* 1 iff sqrt(rr) < r_min*sqrt(<eta,eta>) at exit (reading G4) */
    double rel_residual;   /* sqrt(rr/<eta,eta>), rr the recursed residual norm^2 */
    double eta_norm2;      /* <eta,eta> */
    double gpu_ms;         /* device time of init + loop + final D-dagger (CUDA events on the ctx stream) */
    double total_ms;       /* *_host calls: device time including H2D copies, pack, solve, unpack, D2H; else = gpu_ms */
    int kernel_launches;   /* number of this library's kernels launched by the call (including the one-warp kernels that write
                              the device scalars to the pinned host mirror at every poll) */
    int cg_mode;           /* 1 = three kernels per iteration, 2 = whole solve in one cooperative launch (one thread per site),
                              3 = BiCGSTAB, 4 = even-odd CG, 5 = multi-source CG, 6 = one cooperative launch with the hopping sum of
                              a site split over four warps, 7 = even-odd BiCGSTAB (seven kernels per iteration), 8 = even-odd BiCGSTAB in one
                              cooperative launch */
} wd_cg_info;

/*
 * wd_create — make a context for one lattice geometry and precision.
 *   out          receives the ctx (host pointer to a pointer).
 *   dims         {Lx, Ly, Lz, Lt}, each >= 4 (any integer, e.g. 14); V*36 must fit in 31 bits.
 *   precision    32 (float) or 64 (double): the arithmetic type of fields and stencil.  Dot products
 *                are always accumulated, and alpha/beta formed, in fp64 (reading G17).
 *   bc_t         -1 antiperiodic in t (all BASELINE configs), +1 periodic.  x, y, z are periodic.
 *   cuda_stream  a cudaStream_t (as void*) owned by the caller, or NULL for the legacy default stream.
 * Errors: WD_ERR_ARG, WD_ERR_DIMS, WD_ERR_PRECISION, WD_ERR_CUDA (no usable device), WD_ERR_ALLOC.
 */
int wd_create(wd_ctx **out, const int dims[4], int precision, int bc_t, void *cuda_stream);

/* wd_destroy — free the ctx and everything it owns (synchronises the ctx stream first). NULL is OK. */
int wd_destroy(wd_ctx *ctx);

/* Last error text of this ctx ("" if none).  ctx == NULL returns the text of the last failed wd_create. */
const char *wd_last_error(wd_ctx *ctx);

/* Sizes in bytes of the native buffers the caller must allocate (device memory). */
size_t wd_gauge_native_bytes(wd_ctx *ctx);   /* 72 (48 with 12-real links) * Vpad * sizeof(real), Vpad = V rounded up to 16 */
size_t wd_spinor_native_bytes(wd_ctx *ctx);  /* 24 * Vpad * sizeof(real) */

/*
 * wd_set_gauge_recon — number of reals stored per link in the NATIVE gauge layout (byte reduction):
 *   18 (default): all nine complex entries;
 *   12: rows 0 and 1 only (fp32: 3 planes of float4 per link and 16-site block, fp64: 6 planes of double2); the stencil
 *       kernels rebuild row 2 = conj(row0 x row1) in registers, exact for special-unitary links.  The gauge traffic of a
 *       stencil pass drops from 288 to 192 B/site in fp32 (wd_apply 480 -> 384, CG iteration 1536 -> 1344).
 *       The caller's links must be SU(3) to the accuracy wanted: the rebuilt row differs from the stored one by the
 *       unitarity defect of rows 0, 1.
 * Call it BEFORE wd_gauge_native_bytes / wd_pack_gauge: native gauge buffers of the two formats are not interchangeable,
 * and a gauge field staged by an earlier *_host call is dropped.  With 12, cg_solve always uses the three-kernel loop,
 * and bicgstab_solve / wd_coo_assemble return WD_ERR_ARG (compiled for 18-real links only).
 * wd_get_gauge_recon returns 18 or 12.
 */
int wd_set_gauge_recon(wd_ctx *ctx, int reals_per_link);
int wd_get_gauge_recon(wd_ctx *ctx);

/*
 * wd_pack_gauge / wd_pack_spinor / wd_unpack_spinor — pure permutations between the canonical
 * and the native layout.  Device pointers; in and out must not overlap.
 * The antiperiodic sign is NOT folded into the links.  Asynchronous on the ctx stream.
 */
int wd_pack_gauge(wd_ctx *ctx, const void *U_canonical_dev, void *U_native_dev);
int wd_pack_spinor(wd_ctx *ctx, const void *psi_canonical_dev, void *psi_native_dev);
int wd_unpack_spinor(wd_ctx *ctx, const void *psi_native_dev, void *psi_canonical_dev);

/*
 * wd_apply — out = D psi (dagger = 0) or D-dagger psi (dagger != 0); the paper's "sparse-matrix
 * vector multiplication" done matrix-free: for each of the 8 neighbours, spin
 * projection to a half-spinor, one SU(3) (or SU(3)-dagger) multiply, boundary sign, reconstruction
 * (reading C-1/C-2; row a7 of SURVEY.md 8(a)).
 *   U_native, psi_native, out_native: device pointers, native layout; out must not alias psi.
 *   kappa: hopping parameter (finite).  Asynchronous on the ctx stream.
 */
int wd_apply(wd_ctx *ctx, const void *U_native, const void *psi_native, void *out_native,
             double kappa, int dagger);

/*
 * wd_apply_repeat — measurement aid for "standalone wd_apply timing over 100 applications" (BASELINE.json configs[2]):
 * one warm-up application, then `reps` applications of the same input enqueued back to back from C (at 4^4..14^4 an
 * application is shorter than the call overhead of a scripting-language binding), bracketed by CUDA events on the ctx
 * stream.  *ms_per_application (host pointer) = device time / reps.  Arguments as wd_apply; reps >= 1.  Synchronous.
 */
int wd_apply_repeat(wd_ctx *ctx, const void *U_native, const void *psi_native, void *out_native, double kappa,
                    int dagger, int reps, double *ms_per_application);

/*
 * cg_solve — solve D psi = eta (Eq. 1) by the paper's CG on D D-dagger followed
 * by one multiplication with D-dagger (readings G1-G5):
 *     y <- 0; r <- eta; p <- r; rr <- <r,r>
 *     while sqrt(rr) >= r_min*sqrt(<eta,eta>) and k < max_iter:
 *         q <- D-dagger p ; alpha <- rr / <q,q>        (one kernel: stencil + fused |q|^2)
 *         r <- r - alpha D q ; rr' <- <r,r>            (one kernel: stencil + fused update + |r|^2)
 *         y <- y + alpha p ; beta <- rr'/rr ; p <- r + beta p ; rr <- rr' ; k <- k+1   (one kernel)
 *     psi <- D-dagger y
 * alpha, beta, rr, k and the loop condition live in device memory; the host only polls.
 *   U_native, eta_native: device inputs (native layout); psi_native_out: device output, must not alias eta.
 *   r_min: relative tolerance (> 0); max_iter >= 0 (INT_MAX = no limit; the residual history then keeps its first
 *   2^20 entries).  eta == 0 gives psi = 0, 0 iterations, WD_OK.
 *   info: host pointer, may be NULL.  info->converged = 1 iff sqrt(rr) < r_min*sqrt(<eta,eta>) held (a true comparison:
 *   a NaN or infinite residual stops the loop but is reported as WD_BREAKDOWN, never as converged).
 * Returns WD_OK, WD_NOT_CONVERGED, WD_BREAKDOWN or an error.  Synchronous (returns after info is filled).
 */
int cg_solve(wd_ctx *ctx, const void *U_native, const void *eta_native, void *psi_native_out,
             double kappa, double r_min, int max_iter, wd_cg_info *info);

/*
 * bicgstab_solve — solve D psi = eta with BiCGSTAB applied to D directly.  The paper names the
 * method among the Krylov solvers of lattice QCD but prints no listing; reading B1 is the
 * standard unpreconditioned recurrence with shadow residual rhat = r0 = eta, psi0 = 0, <a,b> = sum conj(a) b:
 *     psi <- 0; r <- eta; p <- r; rho <- <rhat,r>
 *     while sqrt(<r,r>) >= r_min*sqrt(<eta,eta>) and k < max_iter:
 *         v <- D p ; alpha <- rho / <rhat,v>                                   (stencil + fused complex dot)
 *         s <- r - alpha v                                                     (vector kernel)
 *         t <- D s ; omega <- <t,s> / <t,t>                                    (stencil + fused dots)
 *         psi <- psi + alpha p + omega s ; r <- s - omega t ; rho' <- <rhat,r> ; rr <- <r,r>   (one kernel)
 *         beta <- (rho'/rho)(alpha/omega) ; p <- r + beta (p - omega v) ; rho <- rho' ; k <- k+1
 * Complex alpha, omega, beta, rho live in device memory in fp64; loop control as in cg_solve.
 * Arguments and ownership as cg_solve (device pointers, native layout; psi must not alias eta).
 * Returns WD_OK, WD_NOT_CONVERGED, WD_BREAKDOWN (rho, <rhat,v> or omega vanished) or an error.  Synchronous.
 * info->cg_mode = 3.  wd_cg_history works as after cg_solve.
 */
int bicgstab_solve(wd_ctx *ctx, const void *U_native, const void *eta_native, void *psi_native_out,
                   double kappa, double r_min, int max_iter, wd_cg_info *info);

/*
 * Even-odd (Schur) preconditioned CG ("the solver performance is often improved by preconditioning",
 * PAPER.md:32).  Reading E1: sites are coloured by the parity of x+y+z+t (all four extents must be even);
 * the hopping term H of D = 1 - kappa H connects opposite parities only, so D psi = eta is equivalent to
 *     Mhat psi_e = etahat,   Mhat = 1 - kappa^2 H_eo H_oe,   etahat = eta_e + kappa H_eo eta_o,
 *     psi_o = eta_o + kappa H_oe psi_e.
 * cg_solve_eo runs the paper's CG recurrence (readings G1-G5) on Mhat Mhat-dagger over half-length
 * vectors, then psi_e = Mhat-dagger y.  The loop test is sqrt(<r,r>) < r_min*sqrt(<eta,eta>) with the FULL source eta:
 * <r,r> is the squared true residual of the full system, because the odd rows of eta - D psi vanish identically.
 * Per iteration: two plain half-lattice hop passes, two with the fused CG epilogues of cg_solve (|q|^2; r update +
 * |r|^2), one fused axpy-xpay.
 *
 * Checkerboard ("eo") native layouts: two halves, even parity first; inside a half the site index is (lexicographic
 * index)/2 and the data is blocked exactly like the plain native layout.  With wd_set_gauge_recon(ctx, 12) selected
 * BEFORE wd_eo_gauge_bytes / wd_eo_pack_gauge the links are stored as 12 reals and every even-odd call below uses them.
 *   wd_eo_spinor_bytes / wd_eo_gauge_bytes   sizes of the device buffers the caller allocates.
 *   wd_eo_pack_spinor / wd_eo_unpack_spinor / wd_eo_pack_gauge   permutations canonical <-> eo native (device pointers).
 *   wd_eo_hop(ctx, U_eo, in_eo, out_eo, out_parity, dagger)   out(x) = sum over the 8 hops (H in)(x) (H-dagger for
 *       dagger != 0) on the sites of parity out_parity, read from the other half of in_eo; the other half of out_eo is
 *       not touched.  No kappa, no diagonal term.  Asynchronous.
 *   cg_solve_eo   arguments as cg_solve with eo-native buffers; info->cg_mode = 4.  Synchronous.
 *   bicgstab_solve_eo   the BiCGSTAB recurrence of bicgstab_solve (reading B1) applied to Mhat itself (readings E1 + B1
 *       composed; the two SURVEY.md 8(f) rows together): shadow residual rhat = etahat, psi_e0 = 0, the same loop test as
 *       cg_solve_eo, then psi_o = eta_o + kappa H_oe psi_e.  Per iteration: two plain half-lattice hops to the odd sites,
 *       the two hops back fused with the diagonal term and the dot products of the BiCGSTAB passes (<rhat,v>; <t,s>,
 *       <t,t>), three half-length vector kernels.  Arguments as cg_solve_eo; returns WD_OK, WD_NOT_CONVERGED,
 *       WD_BREAKDOWN or an error; info->cg_mode = 7.  Synchronous.  Up to 65536 sites (the paper's 4^4..14^4 range and
 *       16^4) the whole solve runs in ONE cooperative launch instead (grid barriers where the launch boundaries were, the
 *       same recurrence, precision and breakdown rules; info->cg_mode = 8); wd_set_cg_mode(ctx, 1) forces the seven-kernel
 *       loop, 2 the one-launch kernel (18-real links only).
 * Errors: WD_ERR_DIMS for an odd extent, WD_ERR_ARG (NULL, aliasing), WD_ERR_CUDA, WD_ERR_ALLOC.
 */
size_t wd_eo_spinor_bytes(wd_ctx *ctx);
size_t wd_eo_gauge_bytes(wd_ctx *ctx);
int wd_eo_pack_spinor(wd_ctx *ctx, const void *psi_canonical_dev, void *psi_eo_dev);
int wd_eo_unpack_spinor(wd_ctx *ctx, const void *psi_eo_dev, void *psi_canonical_dev);
int wd_eo_pack_gauge(wd_ctx *ctx, const void *U_canonical_dev, void *U_eo_dev);
int wd_eo_hop(wd_ctx *ctx, const void *U_eo, const void *in_eo, void *out_eo, int out_parity, int dagger);
int cg_solve_eo(wd_ctx *ctx, const void *U_eo, const void *eta_eo, void *psi_eo_out,
                double kappa, double r_min, int max_iter, wd_cg_info *info);
int bicgstab_solve_eo(wd_ctx *ctx, const void *U_eo, const void *eta_eo, void *psi_eo_out,
                      double kappa, double r_min, int max_iter, wd_cg_info *info);

/*
 * Several right-hand sides at once (the gauge field is 60 % of the bytes of a stencil pass and is the
 * same for every source).  The nrhs sources are INDEPENDENT problems D psi_j = eta_j on one gauge field: each has its own
 * alpha, beta, residual, loop test and iteration count, exactly as nrhs calls of cg_solve would (the oracle of these calls
 * is nrhs oracle solves).  Fields: nrhs native spinors one after the other (source j at byte offset
 * j * wd_spinor_native_bytes(ctx)).  Sources are processed in groups of 4 (then 2; a last single one through the plain
 * path); inside a group one CTA handles a tile of sites for all sources of the group, so every link is fetched from
 * DRAM / L2 once per group instead of once per source.  18-real links only.
 *   wd_apply_multi   out_j = D in_j (or D-dagger in_j), j < nrhs.  Asynchronous on the ctx stream.
 *   cg_solve_multi   psi_j = solution of D psi_j = eta_j by the CG of cg_solve; infos: host array of nrhs records
 *                    (may be NULL; gpu_ms is the device time of the source's whole group, cg_mode = 5).  Returns WD_OK,
 *                    WD_NOT_CONVERGED if any source hit max_iter, or an error.  Synchronous.
 */
int wd_apply_multi(wd_ctx *ctx, const void *U_native, const void *in_multi, void *out_multi, int nrhs,
                   double kappa, int dagger);
int cg_solve_multi(wd_ctx *ctx, const void *U_native, const void *eta_multi, void *psi_multi_out, int nrhs,
                   double kappa, double r_min, int max_iter, wd_cg_info *infos);

/*
 * The paper's own route: "we store the sparse matrix D in the so-called coordinate format, i.e. D is
 * stored using three arrays: one array contains the value of the non-zero elements and the other two arrays the
 * corresponding row and column indices", and the SpMV loop
 *     for k = 1..N_NZ: out[Row[k]] = out[Row[k]] + Val[k]*in[Col[k]].
 * Vectors are in the CANONICAL layout: component index i = (s*4 + alpha)*3 + a, complex interleaved, 12 V entries.
 *
 * wd_coo_nnz       N_NZ = 588 V (49 entries in each of the 12 V rows: the diagonal and 8 hops x 2 spin x 3 colour).
 * wd_coo_assemble  writes D (dagger = 0) or D-dagger (dagger != 0) for the gauge field U_native (device, native layout):
 *                  val_dev: N_NZ complex numbers of the ctx precision, row_dev / col_dev: N_NZ 32-bit ints (device,
 *                  caller-owned).  Entry k = row*49 + j; j = 0 is the diagonal (Val = 1); j = 1 + (mu*2 + dir)*6 + n*3 + b
 *                  with dir 0 = forward hop, 1 = backward hop, n = 0, 1 the two spin columns beta (ascending) in which
 *                  row alpha of (1 -+ gamma_mu) is non-zero, b the colour column:
 *                    forward : Val = -kappa s+ (1 - gamma_mu)[alpha][beta] U_mu(x)[a][b],            Col = (x+mu, beta, b)
 *                    backward: Val = -kappa s- (1 + gamma_mu)[alpha][beta] conj(U_mu(x-mu)[b][a]),   Col = (x-mu, beta, b)
 *                  (gamma_mu -> -gamma_mu for D-dagger; s+- = bc_t on the hop that wraps in t).  Needs 12 V < 2^31.
 * wd_coo_spmv      the loop above for ANY coordinate-format matrix with 12 V rows (entries in any order, duplicates are
 *                  summed).  General path: out = 0, then parallel over k, equal rows of adjacent entries combined inside a
 *                  warp before one atomic add per run (the sum order of a row is not fixed: results agree to rounding, not
 *                  bitwise).  Fast path, taken in fp32 when val/row/col are the arrays the last wd_coo_assemble of this ctx wrote
 *                  (N_NZ = 588 V): one warp per site, 12 row accumulators, plain stores, fixed summation order; Row is still
 *                  read and checked entry by entry, and if it is not the assembled structure any more (the caller edited the
 *                  arrays) the general path recomputes the product inside the same call.  wd_set_coo_fast(ctx, 0) forces
 *                  the general path.  in_dev, out_dev: canonical vectors on the device, must not alias.
 * All three are asynchronous on the ctx stream.  Errors: WD_ERR_ARG, WD_ERR_DIMS, WD_ERR_CUDA.
 */
size_t wd_coo_nnz(wd_ctx *ctx);
int wd_coo_assemble(wd_ctx *ctx, const void *U_native, double kappa, int dagger, void *val_dev, int *row_dev,
                    int *col_dev);
int wd_coo_spmv(wd_ctx *ctx, size_t nnz, const void *val_dev, const int *row_dev, const int *col_dev,
                const void *in_dev, void *out_dev);
int wd_set_coo_fast(wd_ctx *ctx, int on);

/*
 * Host-buffer forms: the same operations with HOST pointers in the CANONICAL layout.  Each call
 * copies its inputs to the device, packs, runs the device path above, unpacks and copies the result
 * back, on the ctx stream, and returns when the host output is complete.  U_host may be NULL in
 * cg_solve_host / wd_apply_host to reuse the gauge field of the previous *_host call on this ctx.
 */
int wd_apply_host(wd_ctx *ctx, const void *U_host, const void *psi_host, void *out_host,
                  double kappa, int dagger);
int cg_solve_host(wd_ctx *ctx, const void *U_host, const void *eta_host, void *psi_host_out,
                  double kappa, double r_min, int max_iter, wd_cg_info *info);

/*
 * Split-phase form of cg_solve_host, for callers with a queue of systems to solve (PAPER.md:44-48 is one solve; a
 * production run is thousands of them).  A solve needs all of U and eta before its first iteration, so inside ONE solve
 * the PCIe transfers cannot hide; with TWO contexts (two streams) the uploads of solve i+1 and the download of solve i-1
 * run while the GPU iterates on solve i:
 *
 *     cg_solve_host_begin(ctx[0], U_0, eta_0);
 *     for i = 0 .. n-1:   if (i+1 < n) cg_solve_host_begin(ctx[(i+1)%2], U_{i+1}, eta_{i+1});   // enqueues, returns
 *                         cg_solve_host_run(ctx[i%2], psi_i, kappa, r_min, max_iter, &info);   // the solve (host polls)
 *                         if (i > 0) cg_solve_host_wait(ctx[(i-1)%2]);                          // psi_{i-1} is complete
 *     cg_solve_host_wait(ctx[(n-1)%2]);
 *
 *   cg_solve_host_begin   enqueues the copies of U_host (NULL = the gauge field of the previous *_host call on this ctx) and
 *                         eta_host to the device and the pack kernels, slab by slab, and returns without waiting.  The host
 *                         buffers must be pinned for the copies to overlap anything, and must stay untouched until
 *                         cg_solve_host_run on the same ctx has returned.  Device-ordered behind a download of this ctx that is
 *                         still in flight.  WD_ERR_ARG if inputs are already staged.
 *   cg_solve_host_run     cg_solve on the staged fields (same recurrence, same result as cg_solve_host, bit for bit), then
 *                         enqueues the unpack kernels and the copy to psi_host_out and returns WITHOUT waiting for that copy.
 *                         Return value and *info as cg_solve (info->total_ms = info->gpu_ms: there is no per-call total when
 *                         transfers overlap other solves; kernel_launches counts begin + run).  WD_ERR_ARG if nothing is staged.
 *   cg_solve_host_wait    returns when psi_host_out of the last run on this ctx is complete (no-op if nothing is pending).
 * cg_solve_host(ctx, ...) is begin + run + wait on one ctx.  A ctx is still single-threaded: one host thread drives both.
 * The pack kernels of the uploads run on a library stream of the LOWEST priority; give the contexts streams of a higher
 * priority (cudaStreamCreateWithPriority) and those kernels take only the room the other context's solve leaves.
 */
int cg_solve_host_begin(wd_ctx *ctx, const void *U_host, const void *eta_host);
int cg_solve_host_run(wd_ctx *ctx, void *psi_host_out, double kappa, double r_min, int max_iter, wd_cg_info *info);
int cg_solve_host_wait(wd_ctx *ctx);

/*
 * wd_cg_history — rr = <r,r> after 0, 1, ..., k iterations of the last cg_solve / cg_solve_host on this
 * ctx (the device-side record of the recursed residual; used to compare convergence with the oracle).
 *   out: host pointer to n doubles.  Returns the number of values written (<= k+1), or < 0 on error.
 */
int wd_cg_history(wd_ctx *ctx, double *out, int n);

/*
 * wd_norm2 — <a,a> = sum over all 12V complex components of |a|^2 (the paper's dot-product kernel,
 * PAPER.md:60), fp64 accumulation, deterministic single-pass grid reduction.
 *   a_native: device pointer; result: host pointer.  Synchronous.
 */
int wd_norm2(wd_ctx *ctx, const void *a_native, double *result);

/*
 * wd_norm2_noalloc — the same <a,a> for callers that cannot call cudaMalloc: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid allocation.  Needs NO context and allocates nothing, on the host
 * or on the device: the scratch of the grid reduction (one fp64 partial per 4096 128-bit vectors of the field, and the
 * ticket counter) lives in a file-scope __device__ array of 128.25 KB that every GPU loading the library holds until
 * the process exits.  The call enqueues a 256-byte memset (the ticket counter must start at zero) and one kernel on
 * `cuda_stream` and returns; it does not synchronise.
 *   precision     32 or 64.
 *   n_sites       V, the number of lattice sites of the field (native layout: Vpad = V rounded up to 16).
 *   a_native      DEVICE pointer, native spinor layout, 24 * Vpad reals; read only.
 *   result_dev    DEVICE pointer to one double, owned by the caller; written by the kernel in stream order.
 *   cuda_stream   a cudaStream_t (as void*) of the CURRENT device, or NULL for the legacy default stream.  The current
 *                 device must be the one that owns the stream and the buffers.
 * Limit: n_sites <= wd_noalloc_max_sites(precision) = 11 184 800 (fp32) / 5 592 400 (fp64) — 16384 partials; 48^3x96
 * in fp32 and 32^4 in both precisions fit.  Larger fields are rejected with WD_ERR_DIMS (use wd_norm2).
 * Result: fp64 accumulation in an order fixed by n_sites alone (bit-identical from call to call and from GPU to GPU);
 * it differs from wd_norm2's, whose grouping follows the SM count, by fp64 rounding only.
 * SHARED STATE: every call on a device uses the one static array.  Calls that overlap on the GPU (two streams, or two
 * host threads without ordering between their streams) race on it and give wrong sums: serialise them per device.
 * Errors: WD_ERR_PRECISION, WD_ERR_ARG (NULL pointer), WD_ERR_DIMS (n_sites 0 or beyond the limit), WD_ERR_CUDA;
 * wd_noalloc_last_error() returns the message of the calling thread's last failed call ("" after a success).
 * wd_noalloc_prepare() does the one-time set-up for the current device (cudaGetSymbolAddress of the static array) so
 * that a caller can have it done before a stream capture begins; wd_norm2_noalloc does it itself if it was not.
 */
int wd_norm2_noalloc(int precision, size_t n_sites, const void *a_native, double *result_dev, void *cuda_stream);
size_t wd_noalloc_max_sites(int precision);   /* 0 for a precision other than 32 / 64; needs no GPU */
int wd_noalloc_prepare(void);
const char *wd_noalloc_last_error(void);

/*
 * Tuning knobs (the paper's workgroup-size tuning):
 *   wd_num_tiles()            number of compiled stencil launch configurations ("tiles").
 *   wd_tile_shape(i, shape)   writes {BX,BY,BZ,BT} of tile i (threads per CTA = product); returns 0 or WD_ERR_ARG.
 *   wd_tile_info(i, info)     writes {min resident CTAs per SM asked of the compiler, 1 if compiled for precision 32,
 *                             1 if compiled for precision 64}.
 *   wd_set_tile(ctx, i)       select tile i for the stencil kernels of this ctx; i = -1 restores the automatic choice.
 *   wd_get_tile(ctx)          index in use.
 *   wd_set_cg_mode(ctx, m)        0 = automatic (mode 9 wherever the lattice fits a cluster of it: V / nc a power of two <= 256 (fp32) / 128 (fp64) for some nc <= 16, i.e. up to 4096 / 2048 sites, else one cooperative launch for the whole solve when V <= 200000 sites in fp32 /
 *                             65536 in fp64 — this covers the paper's own 4^4..14^4 range — else three kernels per iteration),
 *                             1 = always three kernels, 2 = always one launch, one thread per site (grid barriers between the
 *                             phases; same recurrence and precision), 6 = always one launch with a CTA of 32 sites x 4
 *                             directions: warp mu computes the two hops of direction mu, the partial sums meet in shared
 *                             memory (the automatic choice in fp64 up to 8192 sites),
 *                             9 = one launch with the whole lattice RESIDENT IN SHARED MEMORY (csrc/wilson_resident.cuh): a
 *                             thread-block cluster of nc <= 16 CTAs, V / nc sites each (a power of two, <= 256 in fp32, <= 128
 *                             in fp64), neighbours in other CTAs read through distributed shared memory (from eight CTAs on as
 *                             half-spinors that their owner has already projected: csrc/wilson_resident_ex.cuh), barrier.cluster
 *                             between the phases; covers 4^4 (one CTA in fp32) and 8^4 in fp32 (16 CTAs); WD_ERR_ARG if the
 *                             lattice does not fit;
 *                             10 = one cooperative launch with the GAUGE FIELD resident in shared memory (csrc/wilson_ures.cuh): every
 *                             CTA owns one tile for the whole solve and keeps its links (and the backward links of its faces) in
 *                             shared memory, the spinors stay in L2 with three hops in flight; needs no more tiles than co-resident
 *                             CTAs (up to ~57 000 sites in fp32, ~37 000 in fp64), automatic there; per-site arithmetic and hop order of mode 2.
 *                             Mode 9 is automatic where nc <= 2 (larger clusters are bound by the distributed-shared-
 *                             memory bandwidth and measured slower than mode 2).
 *   wd_set_zchunk(ctx, layers)    z extent (in sites) of one chunk of the CTA rasterisation x,y,z-in-chunk,t,z-chunk that
 *                             keeps the +-t neighbours of a tile in L2; 0 = automatic (fits a 40 MB reuse distance).
 *   wd_set_small_tile(ctx, i)     launch configuration (CTA tile, register bound) of the one-launch CG kernel of mode 2:
 *                             -1 = automatic (default), 0 <= i < number of compiled configurations.
 *   wd_set_link_staging(ctx, row) the stencil passes of wd_apply and of the three-kernel cg_solve fetch the gauge field through the
 *                             shared-memory link pipeline of csrc/wilson_tma.cuh (bulk copies global -> shared of the contiguous
 *                             16-site link blocks, mbarrier ring, both uses of every link served from shared memory; BASELINE.json
 *                             north_star (2)); row selects a compiled configuration {16,BY,BZ,BT, stages, copies ahead, min CTAs/SM},
 *                             -1 = off: links through L1 with the register pipeline, -2 = automatic (default): the row that measured
 *                             faster, which today means the D-dagger / plain passes in fp64 (a2 9 % faster at 32^4) and nothing in
 *                             fp32 (profiles/r2_ncu_link_staging.md).  Results are bit-identical either way.  A row covers
 *                             a lattice only if Lx % 16 == 0 and Ly, Lz, Lt are multiples of BY, BZ, BT, 18 reals per link; otherwise
 *                             WD_ERR_ARG.  wd_get_link_staging(ctx) = row the D-dagger passes run on (-1 = none).  wd_num_staging_rows() / wd_staging_row_info(row, info[9]) list the rows
 *                             (info = {16, BY, BZ, BT, stages, ahead, min CTAs per SM, compiled for fp32, for fp64}).
 *   wd_set_poll_interval(ctx, n)  CG iterations enqueued between two host polls of the device stop flag (n >= 1; 0 = automatic).
 */
int wd_num_tiles(void);
int wd_tile_shape(int index, int shape[4]);
int wd_tile_info(int index, int info[3]);
int wd_set_tile(wd_ctx *ctx, int index);
int wd_get_tile(wd_ctx *ctx);
int wd_set_cg_mode(wd_ctx *ctx, int mode);
int wd_set_zchunk(wd_ctx *ctx, int layers);
int wd_set_small_tile(wd_ctx *ctx, int index);
int wd_num_staging_rows(void);
int wd_staging_row_info(int row, int info[9]);
int wd_set_link_staging(wd_ctx *ctx, int row);
int wd_get_link_staging(wd_ctx *ctx);
int wd_set_poll_interval(wd_ctx *ctx, int n);

/*
 * Per-kernel timing of the CG loop (measurement aid).  With profiling on, cg_solve records
 * CUDA events on the ctx stream around the three kernels of every iteration (a2: D-dagger pass + |q|^2,
 * a3: D pass + r update + |r|^2, a4: axpy-xpay) and accumulates their device times.
 *   wd_set_profile(ctx, n)             n = 0 off, 1 every iteration, n > 1 every n-th iteration (the events cost about
 *                                      1.5 us each on the stream, which shows at 32^4); clears the accumulators.
 *   wd_get_profile(ctx, ms, iters)     ms[0..2] = accumulated milliseconds of a2, a3, a4 over the *iters timed iterations.
 */
int wd_set_profile(wd_ctx *ctx, int on);
int wd_get_profile(wd_ctx *ctx, double ms[3], long *iterations);
/* The same for bicgstab_solve: ms[0..4] = accumulated milliseconds of its five kernels (D p + <rhat,v>; s update;
 * D s + dots; psi/r update + dots; p update) over *iters sampled iterations (the first of every poll chunk).
 * After cg_solve_eo the same call returns its five kernels (H-dagger_oe p; Mhat-dagger tail + |q|^2; H_oe q; Mhat tail
 * + r update + |r|^2; axpy-xpay). */
int wd_get_profile_bicgstab(wd_ctx *ctx, double ms[5], long *iterations);
/* After bicgstab_solve_eo: ms[0..6] = its seven kernels (H_oe p; Mhat tail + <rhat,v>; s update; H_oe s; Mhat tail +
 * <t,s>, <t,t>; psi/r update + dots; p update) over *iters sampled iterations. */
int wd_get_profile_eo_bicgstab(wd_ctx *ctx, double ms[7], long *iterations);

/* Host-only self-test of the fast-division constants of the CTA tile decode: returns the number of n in
 * [0, n_max) with a wrong quotient n / d (0 = correct), or -1 for d = 0.  Needs no GPU. */
long wd_selftest_fastdiv(unsigned int d, unsigned int n_max);

/* Library version string, e.g. "wilson_cg 0.1 sm_100a". */
const char *wd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WILSON_CG_H */

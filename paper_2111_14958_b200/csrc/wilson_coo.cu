// wilson_coo.cu — the paper's own data structure on the B200: the Wilson-Dirac matrix in
// coordinate format (Val, Row, Col) and its SpMV loop out[Row[k]] += Val[k]*in[Col[k]]
// (PAPER.md:52-54).  Kept as a reproduction of the paper's route and as a third way to the same D psi;
// the product path is the matrix-free stencil (the paper itself calls the format "not optimal").
#include "wilson_ctx.cuh"

#include <algorithm>
#include <cmath>

using namespace wd;

namespace {

constexpr int COO_NT = 256;
constexpr int ROW_NNZ = 49;   // 1 + 8 hops * 2 spin columns * 3 colour columns

// Row alpha of gamma_mu (reading C-2) has one non-zero: column PARTNER[mu][alpha] with value GRE + i GIM.
__constant__ int c_partner[4][4] = {{3, 2, 1, 0}, {3, 2, 1, 0}, {2, 3, 0, 1}, {2, 3, 0, 1}};
__constant__ float c_gre[4][4] = {{0, 0, 0, 0}, {-1, 1, 1, -1}, {0, 0, 0, 0}, {1, 1, 1, 1}};
__constant__ float c_gim[4][4] = {{1, 1, -1, -1}, {0, 0, 0, 0}, {1, -1, -1, 1}, {0, 0, 0, 0}};

// element (a, b) of link mu at site s of the native gauge layout
__device__ __forceinline__ float2 link_elem(const float2 *U, int s, int mu, int a, int b)
{
    const float2 *blk = U + (size_t)(s >> SB_SHIFT) * (36 * SB) + mu * 9 * SB;
    const int lane = s & (SB - 1), idx = a * 3 + b;
    if (idx == 8) return blk[8 * SB + lane];
    return blk[((idx >> 1) * SB + lane) * 2 + (idx & 1)];   // float4 plane idx/2, low or high half
}
__device__ __forceinline__ double2 link_elem(const double2 *U, int s, int mu, int a, int b)
{
    return U[(size_t)(s >> SB_SHIFT) * (36 * SB) + (mu * 9 + a * 3 + b) * SB + (s & (SB - 1))];
}

// One thread per entry k = row*49 + j (entry order of include/wilson_cg.h, "wd_coo_assemble").
template <typename real, typename cvec>
__global__ void __launch_bounds__(COO_NT)
coo_assemble_kernel(const Geom g, const cvec *__restrict__ U, real kappa, int dagger, cvec *val, int *row, int *col,
                    long nnz)
{
    const long k = (long)blockIdx.x * COO_NT + threadIdx.x;
    if (k >= nnz) return;
    const int r = (int)(k / ROW_NNZ), j = (int)(k - (long)r * ROW_NNZ);
    const int s = r / 12, al = (r / 3) & 3, a = r % 3;
    row[k] = r;
    if (j == 0) {
        col[k] = r;
        val[k].x = 1; val[k].y = 0;
        return;
    }
    const int m = j - 1, hop = m / 6, mu = hop >> 1, dir = hop & 1, n = (m % 6) / 3, b = m % 3;
    int x[4], rem = s;
    x[0] = rem % g.L[0]; rem /= g.L[0];
    x[1] = rem % g.L[1]; rem /= g.L[1];
    x[2] = rem % g.L[2]; rem /= g.L[2];
    x[3] = rem;
    int y[4] = {x[0], x[1], x[2], x[3]};
    y[mu] = dir == 0 ? (x[mu] + 1 == g.L[mu] ? 0 : x[mu] + 1) : (x[mu] == 0 ? g.L[mu] - 1 : x[mu] - 1);
    const int sn = y[0] + g.L[0] * (y[1] + g.L[1] * (y[2] + g.L[2] * y[3]));
    const bool wraps = mu == 3 && (dir == 0 ? x[3] == g.L[3] - 1 : x[3] == 0);
    const real sig = wraps ? (real)g.bc_t : (real)1;
    // projector (1 + sgn gamma_mu): forward hop of D carries (1 - gamma), backward (1 + gamma); D-dagger swaps them
    const real sgn = ((dir == 0) != (dagger != 0)) ? (real)-1 : (real)1;
    const int pb = c_partner[mu][al];
    const int be = (n == 0) ? min(al, pb) : max(al, pb);
    const real pr = be == al ? (real)1 : sgn * (real)c_gre[mu][al];
    const real pi = be == al ? (real)0 : sgn * (real)c_gim[mu][al];
    cvec u;
    if (dir == 0) u = link_elem(U, s, mu, a, b);
    else { u = link_elem(U, sn, mu, b, a); u.y = -u.y; }
    const real f = -kappa * sig;
    cvec v;
    v.x = f * (pr * u.x - pi * u.y);
    v.y = f * (pr * u.y + pi * u.x);
    val[k] = v;
    col[k] = (sn * 4 + be) * 3 + b;
}

__device__ __forceinline__ void atomic_add_c(float2 *p, float2 v)
{
    atomicAdd(&p->x, v.x);
    atomicAdd(&p->y, v.y);
}
__device__ __forceinline__ void atomic_add_c(double2 *p, double2 v)
{
    atomicAdd(&p->x, v.x);
    atomicAdd(&p->y, v.y);
}

// The paper's loop, parallel over k.  A warp takes 32 consecutive entries per step, multiplies, then adds up runs
// of equal Row inside the warp with shuffles (a segmented scan: rows sorted as wd_coo_assemble writes them give at
// most two runs per step) and only the last lane of each run issues the atomic add.  Any entry order is correct.
// only_if != nullptr: run only if *only_if == epoch (the fall-back behind the sorted-row fast path below)
template <typename cvec>
__global__ void __launch_bounds__(COO_NT)
coo_spmv_kernel(long nnz, const cvec *__restrict__ val, const int *__restrict__ row, const int *__restrict__ col,
                const cvec *__restrict__ in, cvec *out, const unsigned int *only_if, unsigned int epoch)
{
    if (only_if && *only_if != epoch) return;
    constexpr int UNROLL = 4;   // independent 32-entry groups per trip: the Col -> in[Col] dependent loads overlap
    const int lane = threadIdx.x & 31;
    const long warp = ((long)blockIdx.x * COO_NT + threadIdx.x) >> 5;
    const long nwarps = ((long)gridDim.x * COO_NT) >> 5;
    for (long base = warp * (32 * UNROLL); base < nnz; base += nwarps * (32 * UNROLL)) {
        int r[UNROLL];
        cvec p[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const long k = base + u * 32 + lane;
            r[u] = -1;
            p[u].x = 0; p[u].y = 0;
            if (k < nnz) {
                r[u] = __ldg(row + k);
                const cvec v = __ldg(val + k), x = __ldg(in + __ldg(col + k));
                p[u].x = v.x * x.x - v.y * x.y;
                p[u].y = v.x * x.y + v.y * x.x;
            }
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            // runs of equal Row among ADJACENT lanes: head flags -> lane of my run's head -> segmented inclusive scan
            const int rprev = __shfl_up_sync(0xffffffffu, r[u], 1);
            const unsigned int heads = __ballot_sync(0xffffffffu, lane == 0 || rprev != r[u]);
            const int head = 31 - __clz(heads & (0xffffffffu >> (31 - lane)));
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const auto px = __shfl_up_sync(0xffffffffu, p[u].x, o);
                const auto py = __shfl_up_sync(0xffffffffu, p[u].y, o);
                if (lane - o >= head) { p[u].x += px; p[u].y += py; }
            }
            const int rnext = __shfl_down_sync(0xffffffffu, r[u], 1);
            if (r[u] >= 0 && (lane == 31 || rnext != r[u])) atomic_add_c(out + r[u], p[u]);
        }
    }
}

template <typename cvec>
__global__ void __launch_bounds__(COO_NT)
coo_zero_if_kernel(cvec *out, size_t n, const unsigned int *only_if, unsigned int epoch)
{
    if (*only_if != epoch) return;
    for (size_t i = (size_t)blockIdx.x * COO_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * COO_NT) { out[i].x = 0; out[i].y = 0; }
}

// Sorted-row fast path: the matrix as wd_coo_assemble writes it has its entries grouped by row, 49 per row, i.e. 588
// consecutive entries per site.  One warp takes one site at a time: 19 coalesced groups of 32 entries (Val, Row, Col read
// exactly once, as in the paper's loop), the product of every entry added to one of 12 per-lane row accumulators -- which
// row a lane's entry of group i belongs to is a compile-time function of (i, lane), because the rows are 49 long -- then
// one butterfly reduction per row and 12 plain stores: no atomics, no zero-fill pass, and a fixed summation order (the
// result is bitwise reproducible).  The Row array is still READ and CHECKED entry by entry: the first entry that is not
// where the structure says raises *bad = epoch, and the caller's fall-back (zero-fill + the any-order kernel above, both
// conditional on that flag) recomputes the product, so the call is correct for any coordinate-format input.
template <typename cvec>
__global__ void __launch_bounds__(COO_NT)
coo_spmv_rows49_kernel(int nsites, const cvec *__restrict__ val, const int *__restrict__ row, const int *__restrict__ col,
                       const cvec *__restrict__ in, cvec *out, unsigned int *bad, unsigned int epoch)
{
    constexpr int SITE_NNZ = 12 * ROW_NNZ;            // 588
    constexpr int NG = (SITE_NNZ + 31) / 32;           // 19 groups of 32 entries
    const int lane = threadIdx.x & 31;
    const int warp = (int)(((long)blockIdx.x * COO_NT + threadIdx.x) >> 5);
    const int nwarps = (int)(((long)gridDim.x * COO_NT) >> 5);
    bool viol = false;
    for (int site = warp; site < nsites; site += nwarps) {
        const long base = (long)site * SITE_NNZ;
        cvec acc[12];
#pragma unroll
        for (int r = 0; r < 12; ++r) { acc[r].x = 0; acc[r].y = 0; }
        // groups in batches of GB: all Val / Row / Col loads of a batch are issued before the first dependent in[Col] gather.
        // (Measured and not kept: prefetching the next batch's three streams before the gathers of this one, on a grid of
        // exactly one resident wave -- 32^4 fp32 1710 -> 1900 us: the extra registers cost more warps than the overlap gains.)
        constexpr int GB = 5;
#pragma unroll
        for (int i0 = 0; i0 < NG; i0 += GB) {
            cvec v[GB];
            int rw[GB], cl[GB];
#pragma unroll
            for (int u = 0; u < GB; ++u) {
                const int e = 32 * (i0 + u) + lane;
                v[u].x = 0; v[u].y = 0; rw[u] = -1; cl[u] = 0;
                if (i0 + u < NG && e < SITE_NNZ) {
                    v[u] = __ldg(val + base + e);
                    rw[u] = __ldg(row + base + e);
                    cl[u] = __ldg(col + base + e);
                }
            }
            cvec x[GB];
#pragma unroll
            for (int u = 0; u < GB; ++u) {
                x[u].x = 0; x[u].y = 0;
                if (rw[u] >= 0) x[u] = __ldg(in + cl[u]);
            }
#pragma unroll
            for (int u = 0; u < GB; ++u) {
                const int i = i0 + u;
                if (i < NG) {
                    const int r0 = (32 * i) / ROW_NNZ;                       // compile-time after unrolling
                    const int bnd = ROW_NNZ * (r0 + 1) - 32 * i;             // lanes >= bnd belong to row r0 + 1
                    const int r1 = r0 + 1 < 12 ? r0 + 1 : 11;                // (group 18: lanes >= bnd are past the site)
                    const bool in_a = lane < bnd;
                    const bool valid = 32 * i + lane < SITE_NNZ;
                    viol = viol || (valid && rw[u] != site * 12 + (in_a ? r0 : r0 + 1));
                    cvec p;
                    p.x = v[u].x * x[u].x - v[u].y * x[u].y;
                    p.y = v[u].x * x[u].y + v[u].y * x[u].x;
                    if (in_a) { acc[r0].x += p.x; acc[r0].y += p.y; }
                    else { acc[r1].x += p.x; acc[r1].y += p.y; }
                }
            }
        }
        cvec mine;
        mine.x = 0; mine.y = 0;
#pragma unroll
        for (int r = 0; r < 12; ++r) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                acc[r].x += __shfl_xor_sync(0xffffffffu, acc[r].x, o);
                acc[r].y += __shfl_xor_sync(0xffffffffu, acc[r].y, o);
            }
            if (lane == r) mine = acc[r];
        }
        if (lane < 12) out[(size_t)site * 12 + lane] = mine;
    }
    if (__any_sync(0xffffffffu, viol) && lane == 0) atomicExch(bad, epoch);
}

}  // namespace

extern "C" size_t wd_coo_nnz(wd_ctx *c) { return c ? (size_t)c->V * 588 : 0; }

extern "C" int wd_coo_assemble(wd_ctx *c, const void *U_native, double kappa, int dagger, void *val, int *row, int *col)
{
    if (!c) return WD_ERR_ARG;
    if (!U_native || !val || !row || !col) return fail(c, WD_ERR_ARG, "wd_coo_assemble: NULL argument");
    if (!std::isfinite(kappa)) return fail(c, WD_ERR_ARG, "wd_coo_assemble: kappa is not finite");
    if (c->recon != 18) return fail(c, WD_ERR_ARG, "wd_coo_assemble: needs 18-real links (wd_set_gauge_recon)");
    if ((double)c->V * 12.0 >= 2147483647.0) return fail(c, WD_ERR_DIMS, "wd_coo_assemble: 12 V does not fit a 32-bit index");
    Geom g;
    for (int d = 0; d < 4; ++d) g.L[d] = c->dims[d];
    g.V = c->V;
    g.bc_t = c->bc_t;
    const long nnz = (long)c->V * 588;
    const unsigned int grid = (unsigned int)((nnz + COO_NT - 1) / COO_NT);
    if (c->precision == 32)
        coo_assemble_kernel<float, float2><<<grid, COO_NT, 0, c->stream>>>(g, (const float2 *)U_native, (float)kappa,
                                                                          dagger, (float2 *)val, row, col, nnz);
    else
        coo_assemble_kernel<double, double2><<<grid, COO_NT, 0, c->stream>>>(g, (const double2 *)U_native, kappa, dagger,
                                                                            (double2 *)val, row, col, nnz);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    // wd_coo_spmv takes its sorted-row fast path for exactly these arrays (and checks the structure as it reads them)
    c->coo_val = val; c->coo_row = row; c->coo_col = col;
    return WD_OK;
}

extern "C" int wd_coo_spmv(wd_ctx *c, size_t nnz, const void *val, const int *row, const int *col, const void *in,
                           void *out)
{
    if (!c) return WD_ERR_ARG;
    if (!in || !out || in == out || (nnz > 0 && (!val || !row || !col)))
        return fail(c, WD_ERR_ARG, "wd_coo_spmv: NULL or aliased argument");
    const size_t out_bytes = (size_t)c->V * 12 * 2 * (c->precision == 32 ? 4 : 8);
    size_t need = (nnz + 4 * COO_NT - 1) / (4 * COO_NT);   // 4 groups of 32 entries per warp and trip
    const size_t cap = (size_t)c->sm_count * 8 * 4;   // 8 CTAs per SM resident, 4 waves: warps stride over the entries
    const unsigned int grid = (unsigned int)(need < cap ? (need ? need : 1) : cap);
    // fp32 only: in fp64 the 12 complex accumulators per lane cost too many warps (measured 14^4 / 32^4: 174 / 4009 us
    // against 133 / 3656 us for the any-order kernel), so fp64 keeps the atomic path
    const bool assembled = c->coo_fast && c->precision == 32 && nnz == (size_t)c->V * 588 && val == c->coo_val &&
                           row == c->coo_row && col == c->coo_col;
    if (assembled) {
        // the arrays wd_coo_assemble wrote: sorted-row kernel (plain stores, structure checked on the fly), and behind it the
        // any-order path as a fall-back that runs only if the check failed (the caller changed the arrays since)
        if (!c->coo_bad) {
            CUDA_TRY(c, cudaMalloc(&c->coo_bad, sizeof(unsigned int)));
            CUDA_TRY(c, cudaMemsetAsync(c->coo_bad, 0, sizeof(unsigned int), c->stream));
        }
        const unsigned int epoch = ++c->coo_epoch ? c->coo_epoch : ++c->coo_epoch;   // never 0
        const size_t wneed = ((size_t)c->V * 32 + COO_NT - 1) / COO_NT;             // one warp per site at a time ...
        const size_t wcap = (size_t)c->sm_count * 8;                                // ... 8 CTAs per SM, warps stride over the sites
        const unsigned int fgrid = (unsigned int)(wneed < wcap ? wneed : wcap);
        const size_t nout = (size_t)c->V * 12;
        const unsigned int zgrid = (unsigned int)std::min<size_t>((nout + COO_NT - 1) / COO_NT, (size_t)c->sm_count * 8);
        coo_spmv_rows49_kernel<float2><<<fgrid, COO_NT, 0, c->stream>>>(c->V, (const float2 *)val, row, col, (const float2 *)in,
                                                                      (float2 *)out, c->coo_bad, epoch);
        coo_zero_if_kernel<float2><<<zgrid, COO_NT, 0, c->stream>>>((float2 *)out, nout, c->coo_bad, epoch);
        coo_spmv_kernel<float2><<<grid, COO_NT, 0, c->stream>>>((long)nnz, (const float2 *)val, row, col, (const float2 *)in,
                                                               (float2 *)out, c->coo_bad, epoch);
        c->launches += 3;
        CUDA_TRY(c, cudaGetLastError());
        return WD_OK;
    }
    CUDA_TRY(c, cudaMemsetAsync(out, 0, out_bytes, c->stream));
    if (nnz == 0) return WD_OK;
    if (c->precision == 32)
        coo_spmv_kernel<float2><<<grid, COO_NT, 0, c->stream>>>((long)nnz, (const float2 *)val, row, col,
                                                               (const float2 *)in, (float2 *)out, nullptr, 0u);
    else
        coo_spmv_kernel<double2><<<grid, COO_NT, 0, c->stream>>>((long)nnz, (const double2 *)val, row, col,
                                                                (const double2 *)in, (double2 *)out, nullptr, 0u);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    return WD_OK;
}

/* 1 (default): wd_coo_spmv takes the sorted-row kernel for the arrays the last wd_coo_assemble of this ctx wrote; 0: always
   the any-order atomic kernel (the comparison row of the measurement tables). */
extern "C" int wd_set_coo_fast(wd_ctx *c, int on)
{
    if (!c || on < 0 || on > 1) return WD_ERR_ARG;
    c->coo_fast = on;
    return WD_OK;
}

// wilson_coo.cu — the paper's own data structure on the B200: the Wilson-Dirac matrix in
// coordinate format (Val, Row, Col) and its SpMV loop out[Row[k]] += Val[k]*in[Col[k]]
// (PAPER.md:52-54).  Kept as a reproduction of the paper's route and as a third way to the same D psi;
// the product path is the matrix-free stencil (the paper itself calls the format "not optimal").
#include "wilson_ctx.cuh"

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
template <typename cvec>
__global__ void __launch_bounds__(COO_NT)
coo_spmv_kernel(long nnz, const cvec *__restrict__ val, const int *__restrict__ row, const int *__restrict__ col,
                const cvec *__restrict__ in, cvec *out)
{
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
    return WD_OK;
}

extern "C" int wd_coo_spmv(wd_ctx *c, size_t nnz, const void *val, const int *row, const int *col, const void *in,
                           void *out)
{
    if (!c) return WD_ERR_ARG;
    if (!in || !out || in == out || (nnz > 0 && (!val || !row || !col)))
        return fail(c, WD_ERR_ARG, "wd_coo_spmv: NULL or aliased argument");
    const size_t out_bytes = (size_t)c->V * 12 * 2 * (c->precision == 32 ? 4 : 8);
    CUDA_TRY(c, cudaMemsetAsync(out, 0, out_bytes, c->stream));
    if (nnz == 0) return WD_OK;
    size_t need = (nnz + 4 * COO_NT - 1) / (4 * COO_NT);   // 4 groups of 32 entries per warp and trip
    const size_t cap = (size_t)c->sm_count * 8 * 4;   // 8 CTAs per SM resident, 4 waves: warps stride over the entries
    const unsigned int grid = (unsigned int)(need < cap ? need : cap);
    if (c->precision == 32)
        coo_spmv_kernel<float2><<<grid, COO_NT, 0, c->stream>>>((long)nnz, (const float2 *)val, row, col,
                                                               (const float2 *)in, (float2 *)out);
    else
        coo_spmv_kernel<double2><<<grid, COO_NT, 0, c->stream>>>((long)nnz, (const double2 *)val, row, col,
                                                                (const double2 *)in, (double2 *)out);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    return WD_OK;
}

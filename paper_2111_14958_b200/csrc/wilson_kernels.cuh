// wilson_kernels.cuh — device code of the Wilson-Dirac stencil and the fused CG kernels (sm_100a).
//
// What is computed (citations: PAPER.md = the paper text; C-1/C-2/Gnn = readings in DESIGN.md):
//   * D / D-dagger of reading C-1 as a matrix-free 9-point stencil: per site and direction, spin
//     projection to a half-spinor BEFORE the SU(3) multiply, U (forward) or U^dagger (backward, by
//     index transposition + conjugation of the neighbour's link), boundary sign on the t-wrap hop,
//     reconstruction into the 4-spinor accumulator.  This replaces the paper's COO SpMV
//     (PAPER.md:50-56), which it calls "not optimal".
//   * the CG recurrence of PAPER.md:46-48 (readings G1-G5) with its dot products and vector updates
//     fused into the stencil passes: MODE_QQ produces |D-dagger p|^2 and alpha, MODE_RUPD applies
//     r <- r - alpha D q and produces |r|^2, beta and the loop condition, all in device memory.
//
// Data layout (include/wilson_cg.h "Native layouts"): site-blocked SoA.  Blocks of 16 lexicographic sites;
// inside a block a spinor is NSP planes of 128-bit vectors (float4 = two complex components, double2 = one)
// and each of the 4 links occupies 9 complex slots per site (fp32: four float4 planes and one float2 plane; 12-real
// storage: 6 slots).  One thread owns one site; a CTA owns a
// BX x BY x BZ x BT tile so that the 8 neighbours of most sites are fetched by the same CTA (L1 reuse) and
// all loads of a warp are contiguous runs of BX sites.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace wd {

// Division by a run-time constant d >= 1 of n < 2^31: q = (n * M) >> (32 + sh), M = ceil(2^(31+ceil(log2 d)) / d)
// (two instructions instead of the ~20 of an emulated integer division; the tile decode does five per tile).
struct FastDiv {
    unsigned int d, M;
    int sh;   // -1 encodes d == 1
};
__device__ __forceinline__ int fdiv(int n, const FastDiv &f)
{
    return f.sh < 0 ? n : (int)(__umulhi((unsigned int)n, f.M) >> f.sh);
}

struct Geom {
    int L[4];    // Lx, Ly, Lz, Lt
    int V;       // volume = plane stride
    int nt[4];   // tiles per direction (ceil)
    int bc_t;    // -1 antiperiodic, +1 periodic
    int zc;      // z tiles per chunk of the CTA rasterisation (see tile_of_block)
    int ntiles;  // nt[0]*nt[1]*nt[2]*nt[3]
    int eo;      // 1: the lattice of this launch is ONE PARITY of the real lattice (even-odd preconditioning, SURVEY.md
                 //    8(f3)): L[0] = Lx/2, site (xh,y,z,t) stands for x = 2 xh + ((y+z+t+par) & 1); 0: plain lattice
    int par;     // eo = 1: parity (x+y+z+t) & 1 of the sites this launch WRITES; its neighbours have parity 1 - par
    FastDiv d_chunk, d_nt0, d_nt1, d_zc, d_zlast;   // per_chunk, nt[0], nt[1], zc, size of the last z chunk
};

// CTA rasterisation.  Tiles are visited x, y, z-within-chunk fastest, then t, then z-chunk: the sites a CTA
// shares with its +-t neighbours (2 spinor layers and one layer of U_t per tile) are then touched again
// after Lx*Ly*(zc*BZ)*BT sites instead of after a whole t-slice, which keeps them in L2 on lattices whose
// t-slice (spinor + gauge) is larger than L2 (48^3x96: 42 MB per slice).  Only the chunk faces in z are
// read twice from DRAM.  zc = nt[2] is the plain lexicographic order.
__device__ __forceinline__ void tile_of_block(const Geom &g, int b, int &tx, int &ty, int &tz, int &tt)
{
    const int c = fdiv(b, g.d_chunk);
    int rem = b - c * (int)g.d_chunk.d;
    const int z0 = c * g.zc;
    const bool last = z0 + g.zc > g.nt[2];              // the last chunk may be shorter
    int q = fdiv(rem, g.d_nt0);
    tx = rem - q * g.nt[0]; rem = q;
    q = fdiv(rem, g.d_nt1);
    ty = rem - q * g.nt[1]; rem = q;
    const FastDiv &dz = last ? g.d_zlast : g.d_zc;
    q = fdiv(rem, dz);
    tz = z0 + rem - q * (int)dz.d;
    tt = q;
}

// Device-resident CG state.  All fp64 (reading G17).
struct CgScalars {
    double rr;        // <r,r> (recursed)
    double qq;        // <q,q>, q = D-dagger p
    double alpha;     // rr / qq
    double beta;      // rr' / rr
    double eta2;      // <eta,eta>
    double r_min;     // relative tolerance
    int k;            // completed loop bodies
    int k_stop;       // kernels of iteration `it` run iff it < k_stop (initially max_iter)
    int max_iter;
    int converged;
    // BiCGSTAB only (reading B1): complex scalars as (re, im)
    double rho[2];    // <rhat, r>
    double calpha[2]; // rho / <rhat, v>
    double omega[2];  // <t,s> / <t,t>
    double cbeta[2];  // (rho'/rho)(alpha/omega)
    int breakdown;    // a denominator was 0 or not finite: the loop stopped without converging
};

template <typename real> struct Field;
template <> struct Field<float> {
    using svec = float4;
    using gvec = float2;
    static constexpr int NSP = 6;  // spinor planes
};
template <> struct Field<double> {
    using svec = double2;
    using gvec = double2;
    static constexpr int NSP = 12;
};

// ---------------------------------------------------------------- site-blocked SoA addressing
// Sites are grouped in blocks of SB = 16 consecutive lexicographic sites (x fastest).  Inside a block the
// data is planar: spinor block = NSP planes x 16 sites x 128-bit vector (1.5 KB fp32), gauge block =
// 36 planes (mu*9 + a*3+b) x 16 sites x one complex (4.5 KB fp32).  A half-warp reading one plane of one
// block reads 256 (128) contiguous, aligned bytes, a whole block is ONE contiguous chunk (so the next
// tile can be pulled into L2 with one bulk prefetch per block), and every plane of a site is at a
// COMPILE-TIME offset from the
// site's base address, so the 15 loads of a hop share one address register and use immediate offsets
// (the site-planar layout with stride V cost ~30 % of all issued instructions in address arithmetic).
// The volume is padded up to a multiple of 16 sites; pad lanes are never read as sites and are skipped
// by the vector kernels.
constexpr int SB = 16;
constexpr int SB_SHIFT = 4;

template <typename svec, int NSP>
__device__ __forceinline__ size_t spinor_index(int s)
{
    return (size_t)(s >> SB_SHIFT) * (NSP * SB) + (s & (SB - 1));
}
__device__ __forceinline__ size_t gauge_index(int s) { return (size_t)(s >> SB_SHIFT) * (36 * SB) + (s & (SB - 1)); }

// ---------------------------------------------------------------- loads / stores
__device__ __forceinline__ void load_spinor(const float4 *__restrict__ base, int s, float v[24])
{
    const float4 *p = base + spinor_index<float4, 6>(s);
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const float4 t = __ldg(p + j * SB);
        v[4 * j + 0] = t.x; v[4 * j + 1] = t.y; v[4 * j + 2] = t.z; v[4 * j + 3] = t.w;
    }
}
__device__ __forceinline__ void load_spinor(const double2 *__restrict__ base, int s, double v[24])
{
    const double2 *p = base + spinor_index<double2, 12>(s);
#pragma unroll
    for (int j = 0; j < 12; ++j) {
        const double2 t = __ldg(p + j * SB);
        v[2 * j + 0] = t.x; v[2 * j + 1] = t.y;
    }
}
// Read-write fields (r in MODE_RUPD): coherent load, not the read-only path.
__device__ __forceinline__ void load_spinor_rw(const float4 *base, int s, float v[24])
{
    const float4 *p = base + spinor_index<float4, 6>(s);
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const float4 t = p[j * SB];
        v[4 * j + 0] = t.x; v[4 * j + 1] = t.y; v[4 * j + 2] = t.z; v[4 * j + 3] = t.w;
    }
}
__device__ __forceinline__ void load_spinor_rw(const double2 *base, int s, double v[24])
{
    const double2 *p = base + spinor_index<double2, 12>(s);
#pragma unroll
    for (int j = 0; j < 12; ++j) {
        const double2 t = p[j * SB];
        v[2 * j + 0] = t.x; v[2 * j + 1] = t.y;
    }
}
__device__ __forceinline__ void store_spinor(float4 *base, int s, const float v[24])
{
    float4 *p = base + spinor_index<float4, 6>(s);
#pragma unroll
    for (int j = 0; j < 6; ++j) p[j * SB] = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
}
__device__ __forceinline__ void store_spinor(double2 *base, int s, const double v[24])
{
    double2 *p = base + spinor_index<double2, 12>(s);
#pragma unroll
    for (int j = 0; j < 12; ++j) p[j * SB] = make_double2(v[2 * j], v[2 * j + 1]);
}
// Link U_mu(s): 18 reals u[(a*3+b)*2 + ri].  Inside the site block the link mu occupies 9*SB complex slots
// (1152 B fp32): fp64 = 9 planes of double2 (one complex each); fp32 = 4 planes of float4 (reals 4q..4q+3,
// i.e. two complex entries) followed by one plane of float2 (reals 16, 17), so that a link is 4 x 128-bit +
// 1 x 64-bit loads instead of 9 x 64-bit.
template <int MU>
__device__ __forceinline__ void load_link(const double2 *__restrict__ U, int s, double u[18])
{
    const double2 *p = U + gauge_index(s) + MU * 9 * SB;
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const double2 t = __ldg(p + k * SB);
        u[2 * k] = t.x; u[2 * k + 1] = t.y;
    }
}
template <int MU>
__device__ __forceinline__ void load_link(const float2 *__restrict__ U, int s, float u[18])
{
    const float2 *blk = U + (size_t)(s >> SB_SHIFT) * (36 * SB) + MU * 9 * SB;
    const int lane = s & (SB - 1);
    const float4 *p4 = reinterpret_cast<const float4 *>(blk) + lane;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float4 t = __ldg(p4 + q * SB);
        u[4 * q] = t.x; u[4 * q + 1] = t.y; u[4 * q + 2] = t.z; u[4 * q + 3] = t.w;
    }
    const float2 t2 = __ldg(blk + 8 * SB + lane);
    u[16] = t2.x; u[17] = t2.y;
}
// 12-real storage: only rows 0 and 1 of the SU(3) matrix are kept (fp32: 3 planes of float4 per
// link, 768 B per link and 16-site block; fp64: 6 planes of double2); the third row is rebuilt in registers as
// conj(row0 x row1), which is exact for a special-unitary matrix (and accurate to the unitarity defect of the
// stored rows otherwise).  Gauge traffic drops from 288 to 192 B/site in fp32.
template <typename real>
__device__ __forceinline__ void rebuild_row2(real u[18])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        const real ar = u[c1 * 2], ai = u[c1 * 2 + 1], br = u[(3 + c2) * 2], bi = u[(3 + c2) * 2 + 1];
        const real cr = u[c2 * 2], ci = u[c2 * 2 + 1], dr = u[(3 + c1) * 2], di = u[(3 + c1) * 2 + 1];
        // conj(a b - c d)
        u[(6 + c) * 2] = fma(ar, br, -ai * bi) - fma(cr, dr, -ci * di);
        u[(6 + c) * 2 + 1] = -(fma(ar, bi, ai * br) - fma(cr, di, ci * dr));
    }
}
template <int MU>
__device__ __forceinline__ void load_link12(const double2 *__restrict__ U, int s, double u[18])
{
    const double2 *p = U + (size_t)(s >> SB_SHIFT) * (24 * SB) + MU * 6 * SB + (s & (SB - 1));
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const double2 t = __ldg(p + k * SB);
        u[2 * k] = t.x; u[2 * k + 1] = t.y;
    }
    rebuild_row2(u);
}
template <int MU>
__device__ __forceinline__ void load_link12(const float2 *__restrict__ U, int s, float u[18])
{
    const float2 *blk = U + (size_t)(s >> SB_SHIFT) * (24 * SB) + MU * 6 * SB;
    const float4 *p4 = reinterpret_cast<const float4 *>(blk) + (s & (SB - 1));
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const float4 t = __ldg(p4 + q * SB);
        u[4 * q] = t.x; u[4 * q + 1] = t.y; u[4 * q + 2] = t.z; u[4 * q + 3] = t.w;
    }
    rebuild_row2(u);
}
__device__ __forceinline__ void store_link12(double2 *U, int s, int mu, const double2 k9[9])
{
    double2 *p = U + (size_t)(s >> SB_SHIFT) * (24 * SB) + mu * 6 * SB + (s & (SB - 1));
#pragma unroll
    for (int k = 0; k < 6; ++k) p[k * SB] = k9[k];
}
__device__ __forceinline__ void store_link12(float2 *U, int s, int mu, const float2 k9[9])
{
    float2 *blk = U + (size_t)(s >> SB_SHIFT) * (24 * SB) + mu * 6 * SB;
    float4 *p4 = reinterpret_cast<float4 *>(blk) + (s & (SB - 1));
#pragma unroll
    for (int q = 0; q < 3; ++q) p4[q * SB] = make_float4(k9[2 * q].x, k9[2 * q].y, k9[2 * q + 1].x, k9[2 * q + 1].y);
}
// the same slots, written by the pack kernel
__device__ __forceinline__ void store_link(double2 *U, int s, int mu, const double2 k9[9])
{
    double2 *p = U + gauge_index(s) + mu * 9 * SB;
#pragma unroll
    for (int k = 0; k < 9; ++k) p[k * SB] = k9[k];
}
__device__ __forceinline__ void store_link(float2 *U, int s, int mu, const float2 k9[9])
{
    float2 *blk = U + (size_t)(s >> SB_SHIFT) * (36 * SB) + mu * 9 * SB;
    const int lane = s & (SB - 1);
    float4 *p4 = reinterpret_cast<float4 *>(blk) + lane;
#pragma unroll
    for (int q = 0; q < 4; ++q) p4[q * SB] = make_float4(k9[2 * q].x, k9[2 * q].y, k9[2 * q + 1].x, k9[2 * q + 1].y);
    blk[8 * SB + lane] = k9[8];
}

// ---------------------------------------------------------------- spin projection (reading C-2)
// v[(alpha*3+c)*2+ri] -> h[(sp*3+c)*2+ri], the upper two rows of (1 + S gamma_MU) v, S = +-1.
template <int MU, int S, typename real>
__device__ __forceinline__ void project(const real v[24], real h[12])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const real p0r = v[(0 + c) * 2], p0i = v[(0 + c) * 2 + 1];
        const real p1r = v[(3 + c) * 2], p1i = v[(3 + c) * 2 + 1];
        const real p2r = v[(6 + c) * 2], p2i = v[(6 + c) * 2 + 1];
        const real p3r = v[(9 + c) * 2], p3i = v[(9 + c) * 2 + 1];
        real h0r, h0i, h1r, h1i;
        if (MU == 0) {        // h0 = p0 + S i p3 ; h1 = p1 + S i p2
            h0r = p0r - S * p3i; h0i = p0i + S * p3r;
            h1r = p1r - S * p2i; h1i = p1i + S * p2r;
        } else if (MU == 1) { // h0 = p0 - S p3 ; h1 = p1 + S p2
            h0r = p0r - S * p3r; h0i = p0i - S * p3i;
            h1r = p1r + S * p2r; h1i = p1i + S * p2i;
        } else if (MU == 2) { // h0 = p0 + S i p2 ; h1 = p1 - S i p3
            h0r = p0r - S * p2i; h0i = p0i + S * p2r;
            h1r = p1r + S * p3i; h1i = p1i - S * p3r;
        } else {              // h0 = p0 + S p2 ; h1 = p1 + S p3
            h0r = p0r + S * p2r; h0i = p0i + S * p2i;
            h1r = p1r + S * p3r; h1i = p1i + S * p3i;
        }
        h[(0 + c) * 2] = h0r; h[(0 + c) * 2 + 1] = h0i;
        h[(3 + c) * 2] = h1r; h[(3 + c) * 2 + 1] = h1i;
    }
}

// g = U h (ADJ = false) or U^dagger h (ADJ = true) on both spin components of the half-spinor.
template <bool ADJ, typename real>
__device__ __forceinline__ void mul_su3(const real u[18], const real h[12], real g[12])
{
#pragma unroll
    for (int sp = 0; sp < 2; ++sp)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            real gr = 0, gi = 0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const real ur = ADJ ? u[(c * 3 + a) * 2] : u[(a * 3 + c) * 2];
                const real ui = ADJ ? -u[(c * 3 + a) * 2 + 1] : u[(a * 3 + c) * 2 + 1];
                const real hr = h[(sp * 3 + c) * 2], hi = h[(sp * 3 + c) * 2 + 1];
                gr = fma(ur, hr, gr); gr = fma(-ui, hi, gr);
                gi = fma(ur, hi, gi); gi = fma(ui, hr, gi);
            }
            g[(sp * 3 + a) * 2] = gr; g[(sp * 3 + a) * 2 + 1] = gi;
        }
}

// acc += sg * reconstruct_{MU,S}(g): rows 0,1 get g, rows 2,3 the table of reading C-2.
template <int MU, int S, typename real>
__device__ __forceinline__ void reconstruct(const real g[12], real sg, real acc[24])
{
    const real c = sg * S;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const real g0r = g[(0 + a) * 2], g0i = g[(0 + a) * 2 + 1];
        const real g1r = g[(3 + a) * 2], g1i = g[(3 + a) * 2 + 1];
        acc[(0 + a) * 2] = fma(sg, g0r, acc[(0 + a) * 2]);
        acc[(0 + a) * 2 + 1] = fma(sg, g0i, acc[(0 + a) * 2 + 1]);
        acc[(3 + a) * 2] = fma(sg, g1r, acc[(3 + a) * 2]);
        acc[(3 + a) * 2 + 1] = fma(sg, g1i, acc[(3 + a) * 2 + 1]);
        if (MU == 0) {        // row2 += -S i g1 ; row3 += -S i g0
            acc[(6 + a) * 2] = fma(c, g1i, acc[(6 + a) * 2]);
            acc[(6 + a) * 2 + 1] = fma(-c, g1r, acc[(6 + a) * 2 + 1]);
            acc[(9 + a) * 2] = fma(c, g0i, acc[(9 + a) * 2]);
            acc[(9 + a) * 2 + 1] = fma(-c, g0r, acc[(9 + a) * 2 + 1]);
        } else if (MU == 1) { // row2 += S g1 ; row3 += -S g0
            acc[(6 + a) * 2] = fma(c, g1r, acc[(6 + a) * 2]);
            acc[(6 + a) * 2 + 1] = fma(c, g1i, acc[(6 + a) * 2 + 1]);
            acc[(9 + a) * 2] = fma(-c, g0r, acc[(9 + a) * 2]);
            acc[(9 + a) * 2 + 1] = fma(-c, g0i, acc[(9 + a) * 2 + 1]);
        } else if (MU == 2) { // row2 += -S i g0 ; row3 += S i g1
            acc[(6 + a) * 2] = fma(c, g0i, acc[(6 + a) * 2]);
            acc[(6 + a) * 2 + 1] = fma(-c, g0r, acc[(6 + a) * 2 + 1]);
            acc[(9 + a) * 2] = fma(-c, g1i, acc[(9 + a) * 2]);
            acc[(9 + a) * 2 + 1] = fma(c, g1r, acc[(9 + a) * 2 + 1]);
        } else {              // row2 += S g0 ; row3 += S g1
            acc[(6 + a) * 2] = fma(c, g0r, acc[(6 + a) * 2]);
            acc[(6 + a) * 2 + 1] = fma(c, g0i, acc[(6 + a) * 2 + 1]);
            acc[(9 + a) * 2] = fma(c, g1r, acc[(9 + a) * 2]);
            acc[(9 + a) * 2 + 1] = fma(c, g1i, acc[(9 + a) * 2 + 1]);
        }
    }
}

// ---------------------------------------------------------------- the fp32 hop on packed arithmetic (FFMA2 / FADD2)
// sm_100 executes fma.rn.f32x2 / add.rn.f32x2: two IEEE fp32 operations on a 64-bit register pair per instruction,
// with a scalar-broadcast, a swapped-halves and per-half sign form of the operands.  A complex number (re, im) of the
// spinor layout already IS such a pair (two adjacent 32-bit registers of a 128-bit load), so the complex arithmetic of a
// hop maps onto it without any data movement:
//     u h           = u_re (h_re, h_im) + u_im (-h_im, h_re)         u_re, u_im broadcast, the second pair is i h
//     conj(u) h     = u_re (h_re, h_im) - u_im (i h)
//     h = p + S i q = (p_re, p_im) + S (-q_im, q_re)                  one FADD2 with a swapped, half-negated operand
// Per hop: projection 12 FADD2 (h and i h), SU(3) multiply 36 FFMA2, reconstruction 12 FFMA2 -- 60 instructions for the
// 108 scalar ones, every lane performing exactly the scalar code's operations in the scalar code's order (bit-identical).
// MEASURED SLOWER and therefore compiled out (WD_F32X2 = 0; -DWD_F32X2=1 builds it, the whole -m gpu suite passed with
// it): ptxas folds every pack, swap and sign into operand modifiers (FP instructions of the fp32 stencil unit 48 452 ->
// 28 328, MOVs unchanged), yet at 48^3x96 a2 goes 1.027 -> 1.190 ms and a3 1.084 -> 1.178 ms on the same box, same
// session, although the SM clock under the power cap rises 1440 -> 1533 MHz.  DESIGN.md section 6.
#ifndef WD_F32X2
#define WD_F32X2 0
#endif
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(f32x2 p, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
// h[sp*3+c] = (re, im) of the half-spinor, ih = i h (the operand of the u_im products)
template <int MU, int S>
__device__ __forceinline__ void project_x2(const float v[24], f32x2 h[6], f32x2 ih[6])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float p0r = v[(0 + c) * 2], p0i = v[(0 + c) * 2 + 1];
        const float p1r = v[(3 + c) * 2], p1i = v[(3 + c) * 2 + 1];
        const float p2r = v[(6 + c) * 2], p2i = v[(6 + c) * 2 + 1];
        const float p3r = v[(9 + c) * 2], p3i = v[(9 + c) * 2 + 1];
        const f32x2 P0 = pk2(p0r, p0i), P1 = pk2(p1r, p1i), iP0 = pk2(-p0i, p0r), iP1 = pk2(-p1i, p1r);
        if (MU == 0) {        // h0 = p0 + S i p3 ; h1 = p1 + S i p2
            h[c] = add2(P0, pk2(-S * p3i, S * p3r));      ih[c] = add2(iP0, pk2(-S * p3r, -S * p3i));
            h[3 + c] = add2(P1, pk2(-S * p2i, S * p2r));  ih[3 + c] = add2(iP1, pk2(-S * p2r, -S * p2i));
        } else if (MU == 1) { // h0 = p0 - S p3 ; h1 = p1 + S p2
            h[c] = add2(P0, pk2(-S * p3r, -S * p3i));     ih[c] = add2(iP0, pk2(S * p3i, -S * p3r));
            h[3 + c] = add2(P1, pk2(S * p2r, S * p2i));   ih[3 + c] = add2(iP1, pk2(-S * p2i, S * p2r));
        } else if (MU == 2) { // h0 = p0 + S i p2 ; h1 = p1 - S i p3
            h[c] = add2(P0, pk2(-S * p2i, S * p2r));      ih[c] = add2(iP0, pk2(-S * p2r, -S * p2i));
            h[3 + c] = add2(P1, pk2(S * p3i, -S * p3r));  ih[3 + c] = add2(iP1, pk2(S * p3r, S * p3i));
        } else {              // h0 = p0 + S p2 ; h1 = p1 + S p3
            h[c] = add2(P0, pk2(S * p2r, S * p2i));       ih[c] = add2(iP0, pk2(-S * p2i, S * p2r));
            h[3 + c] = add2(P1, pk2(S * p3r, S * p3i));   ih[3 + c] = add2(iP1, pk2(-S * p3i, S * p3r));
        }
    }
}
template <bool ADJ>
__device__ __forceinline__ void mul_su3_x2(const float u[18], const f32x2 h[6], const f32x2 ih[6], f32x2 g[6])
{
#pragma unroll
    for (int sp = 0; sp < 2; ++sp)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            f32x2 acc = pk2(0.f, 0.f);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float ur = ADJ ? u[(c * 3 + a) * 2] : u[(a * 3 + c) * 2];
                const float ui = ADJ ? -u[(c * 3 + a) * 2 + 1] : u[(a * 3 + c) * 2 + 1];
                acc = fma2(pk2(ur, ur), h[sp * 3 + c], acc);
                acc = fma2(pk2(ui, ui), ih[sp * 3 + c], acc);
            }
            g[sp * 3 + a] = acc;
        }
}
template <int MU, int S>
__device__ __forceinline__ void reconstruct_x2(const f32x2 g[6], float sg, float acc[24])
{
    const float c = sg * S;
    const f32x2 sg2 = pk2(sg, sg), cpp = pk2(c, c), cpn = pk2(c, -c), cnp = pk2(-c, c), cnn = pk2(-c, -c);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float g0r, g0i, g1r, g1i;
        upk2(g[a], g0r, g0i);
        upk2(g[3 + a], g1r, g1i);
        const f32x2 G0 = g[a], G1 = g[3 + a], G0s = pk2(g0i, g0r), G1s = pk2(g1i, g1r);
        f32x2 A0 = pk2(acc[(0 + a) * 2], acc[(0 + a) * 2 + 1]), A1 = pk2(acc[(3 + a) * 2], acc[(3 + a) * 2 + 1]);
        f32x2 A2 = pk2(acc[(6 + a) * 2], acc[(6 + a) * 2 + 1]), A3 = pk2(acc[(9 + a) * 2], acc[(9 + a) * 2 + 1]);
        A0 = fma2(sg2, G0, A0);
        A1 = fma2(sg2, G1, A1);
        if (MU == 0) {        // row2 += -S i g1 ; row3 += -S i g0
            A2 = fma2(cpn, G1s, A2);  A3 = fma2(cpn, G0s, A3);
        } else if (MU == 1) { // row2 += S g1 ; row3 += -S g0
            A2 = fma2(cpp, G1, A2);   A3 = fma2(cnn, G0, A3);
        } else if (MU == 2) { // row2 += -S i g0 ; row3 += S i g1
            A2 = fma2(cpn, G0s, A2);  A3 = fma2(cnp, G1s, A3);
        } else {              // row2 += S g0 ; row3 += S g1
            A2 = fma2(cpp, G0, A2);   A3 = fma2(cpp, G1, A3);
        }
        upk2(A0, acc[(0 + a) * 2], acc[(0 + a) * 2 + 1]);
        upk2(A1, acc[(3 + a) * 2], acc[(3 + a) * 2 + 1]);
        upk2(A2, acc[(6 + a) * 2], acc[(6 + a) * 2 + 1]);
        upk2(A3, acc[(9 + a) * 2], acc[(9 + a) * 2 + 1]);
    }
}

// One hop, split into its loads and its arithmetic so that the loads of the next hop can be in flight
// while this one is computed:  acc += sg (1 + S gamma_MU) (x) [U or U^dagger](link_site) in(spinor_site).
// RO = true: `in` is not written while the kernel runs -> read-only (non-coherent) path; false: coherent loads
// (the one-launch CG kernel reads fields other CTAs wrote before the last grid barrier).
template <bool RO, typename svec, typename real>
__device__ __forceinline__ void load_spinor_sel(const svec *in, int s, real v[24])
{
    if (RO) load_spinor(in, s, v);
    else load_spinor_rw(in, s, v);
}
// MAYBE_NULL = false (plain lattice): cen is the input field itself, no test (a run-time test here costs the plain
// kernels a spill and ~4 % because the centre loads can no longer be scheduled freely around the last hop)
template <bool RO, bool MAYBE_NULL, typename svec, typename real>
__device__ __forceinline__ void load_centre(const svec *cen, int s, real c[24])
{
    if (!MAYBE_NULL || cen) load_spinor_sel<RO>(cen, s, c);
    else {
#pragma unroll
        for (int i = 0; i < 24; ++i) c[i] = 0;
    }
}
// RECON = 18: all nine complex entries are stored; 12: rows 0, 1 stored, row 2 rebuilt.  With RECON = 12 the rebuild
// happens at load time, i.e. inside the software pipeline one hop ahead of its use.
template <int MU, bool RO, int RECON, typename real, typename svec, typename gvec>
__device__ __forceinline__ void hop_load(const gvec *__restrict__ U, const svec *in,
                                         int link_site, int spinor_site, real v[24], real u[18])
{
    load_spinor_sel<RO>(in, spinor_site, v);
    if (RECON == 12) load_link12<MU>(U, link_site, u);
    else load_link<MU>(U, link_site, u);
}
template <int MU, int S, bool ADJ, typename real>
__device__ __forceinline__ void hop_compute(const real v[24], const real u[18], real sg, real acc[24])
{
    if constexpr (WD_F32X2 && sizeof(real) == 4) {
        f32x2 h[6], ih[6], g[6];
        project_x2<MU, S>(v, h, ih);
        mul_su3_x2<ADJ>(u, h, ih, g);
        reconstruct_x2<MU, S>(g, sg, acc);
    } else {
        real h[12], g[12];
        project<MU, S, real>(v, h);
        mul_su3<ADJ, real>(u, h, g);
        reconstruct<MU, S, real>(g, sg, acc);
    }
}

// Neighbour sites and boundary signs of site s = (x,y,z,t).
struct Hops {
    int f[4], b[4];
};
template <int EO = 0>
__device__ __forceinline__ Hops neighbours(const Geom &g, int x, int y, int z, int t, int s)
{
    const int L0 = g.L[0], L1 = g.L[1], L2 = g.L[2], L3 = g.L[3];
    const int s1 = L0, s2 = L0 * L1, s3 = L0 * L1 * L2;
    Hops h;
    h.f[0] = s + (x == L0 - 1 ? 1 - L0 : 1);
    h.b[0] = s + (x == 0 ? L0 - 1 : -1);
    if (EO) {
        // checkerboard: the +-x neighbours live in the other parity's field; a site with odd real x (rp = 1) has its
        // +x neighbour in the NEXT pair and its -x neighbour in its own pair, a site with even x the other way round
        const int rp = (y + z + t + g.par) & 1;
        if (rp) h.b[0] = s;
        else h.f[0] = s;
    }
    h.f[1] = s + (y == L1 - 1 ? (1 - L1) * s1 : s1);
    h.b[1] = s + (y == 0 ? (L1 - 1) * s1 : -s1);
    h.f[2] = s + (z == L2 - 1 ? (1 - L2) * s2 : s2);
    h.b[2] = s + (z == 0 ? (L2 - 1) * s2 : -s2);
    h.f[3] = s + (t == L3 - 1 ? (1 - L3) * s3 : s3);
    h.b[3] = s + (t == 0 ? (L3 - 1) * s3 : -s3);
    return h;
}

// acc = sum over the 8 hops at site s; then c = centre spinor in(s) (loaded last so that its latency
// overlaps the last hop).  DAG = 0: D (forward projector 1 - gamma), 1: D-dagger.
// PIPE = 0: hop after hop (load, compute).  PIPE = 1: software pipeline, two register buffers: the loads of
// hop k+1 are issued before hop k is computed, so every thread keeps one hop (168 B fp32) in flight while
// it computes (memory-level parallelism without more threads).
// LOADR: also fetch r(s) into rv together with the centre spinor (MODE_RUPD), so that it too overlaps the last hop.
// U: links of the sites being written (forward hops); UB: links of the neighbours' field (backward hops; == U on a
// plain lattice, the other parity's links with even-odd); cen: the field of the diagonal term (== in on a plain
// lattice; nullptr = no diagonal term, c = 0).
// CFIRST (PIPE = 1 only): the diagonal term goes FIRST.  acc starts as in(s), fetched together with the +-x hops (the
// same cache lines), and every hop is accumulated with the factor -kappa folded into its boundary sign, so that on
// return acc = in(s) - kappa * hops = (D in)(s) and c is not touched: no centre fetch at the end of the tile's life
// (when its lines have left the L1), one dependent load step and 24 live registers fewer in the epilogue.
template <int DAG, int PIPE, bool LOADR, bool RO, typename real, typename svec, typename gvec, int RECON = 18,
          int EO = 0, bool CFIRST = false>
__device__ __forceinline__ void hopping_sum(const Geom &g, const gvec *__restrict__ U, const gvec *__restrict__ UB,
                                            const svec *in, const svec *cen, const svec *r, int x, int y, int z, int t,
                                            int s, real acc[24], real c[24], real rv[24], real kappa = 0)
{
    static_assert(!CFIRST || PIPE == 1, "centre-first is implemented for the two-buffer pipeline");
    constexpr int SF = DAG ? +1 : -1;
    const Hops n = neighbours<EO>(g, x, y, z, t, s);
    // boundary sign sigma+- of reading C-1: only the hop that wraps the t boundary carries bc_t
    const real one = CFIRST ? -kappa : (real)1;
    const real sgf = (t == g.L[3] - 1) ? (real)g.bc_t * one : one;
    const real sgb = (t == 0) ? (real)g.bc_t * one : one;
    if (CFIRST) {
        load_centre<RO, EO != 0>(cen, s, acc);
    } else {
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = 0;
    }
    if (PIPE == 0) {
        real v[24], u[18];
        hop_load<0, RO, RECON, real>(U, in, s, n.f[0], v, u);       hop_compute<0, SF, false, real>(v, u, one, acc);
        hop_load<0, RO, RECON, real>(UB, in, n.b[0], n.b[0], v, u);  hop_compute<0, -SF, true, real>(v, u, one, acc);
        hop_load<1, RO, RECON, real>(U, in, s, n.f[1], v, u);       hop_compute<1, SF, false, real>(v, u, one, acc);
        hop_load<1, RO, RECON, real>(UB, in, n.b[1], n.b[1], v, u);  hop_compute<1, -SF, true, real>(v, u, one, acc);
        hop_load<2, RO, RECON, real>(U, in, s, n.f[2], v, u);       hop_compute<2, SF, false, real>(v, u, one, acc);
        hop_load<2, RO, RECON, real>(UB, in, n.b[2], n.b[2], v, u);  hop_compute<2, -SF, true, real>(v, u, one, acc);
        hop_load<3, RO, RECON, real>(U, in, s, n.f[3], v, u);       hop_compute<3, SF, false, real>(v, u, sgf, acc);
        hop_load<3, RO, RECON, real>(UB, in, n.b[3], n.b[3], v, u);  hop_compute<3, -SF, true, real>(v, u, sgb, acc);
        load_centre<RO, EO != 0>(cen, s, c);
        if (LOADR) load_spinor_rw(r, s, rv);
    } else if (PIPE == 1) {
        real va[24], ua[18], vb[24], ub[18];
        hop_load<0, RO, RECON, real>(U, in, s, n.f[0], va, ua);
        hop_load<0, RO, RECON, real>(UB, in, n.b[0], n.b[0], vb, ub);  hop_compute<0, SF, false, real>(va, ua, one, acc);
        hop_load<1, RO, RECON, real>(U, in, s, n.f[1], va, ua);       hop_compute<0, -SF, true, real>(vb, ub, one, acc);
        hop_load<1, RO, RECON, real>(UB, in, n.b[1], n.b[1], vb, ub);  hop_compute<1, SF, false, real>(va, ua, one, acc);
        hop_load<2, RO, RECON, real>(U, in, s, n.f[2], va, ua);       hop_compute<1, -SF, true, real>(vb, ub, one, acc);
        hop_load<2, RO, RECON, real>(UB, in, n.b[2], n.b[2], vb, ub);  hop_compute<2, SF, false, real>(va, ua, one, acc);
        hop_load<3, RO, RECON, real>(U, in, s, n.f[3], va, ua);       hop_compute<2, -SF, true, real>(vb, ub, one, acc);
        hop_load<3, RO, RECON, real>(UB, in, n.b[3], n.b[3], vb, ub);  hop_compute<3, SF, false, real>(va, ua, sgf, acc);
        if (!CFIRST) load_centre<RO, EO != 0>(cen, s, c);
        hop_compute<3, -SF, true, real>(vb, ub, sgb, acc);
        if (LOADR) load_spinor_rw(r, s, rv);   // after the last hop: an earlier fetch costs registers (spills at 128)
    }
}

// ---------------------------------------------------------------- deterministic reductions
// Fixed-shape tree: warp shuffle -> one slot per warp -> warp 0.  Result valid on thread 0.
template <int NT>
__device__ __forceinline__ double block_sum(double v, double *sm /* >= 32 doubles */)
{
    constexpr int NW = (NT + 31) / 32;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) sm[w] = v;
    __syncthreads();
    double t = 0.0;
    if (w == 0) {
        t = lane < NW ? sm[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    __syncthreads();
    return t;
}

// Single-pass grid reduction: every CTA stores its partial; the CTA that draws the last ticket sums
// the partials in index order (same order every run -> run-to-run identical alpha, beta).
// Returns true on thread 0 of that last CTA only, with the grid total in *total.
template <int NT>
__device__ __forceinline__ bool grid_sum(double v, double *partials, unsigned int *counter, double *total)
{
    __shared__ double sm[32];
    __shared__ int is_last;
    const double b = block_sum<NT>(v, sm);
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = b;
        __threadfence();
        const unsigned int ticket = atomicAdd(counter, 1u);
        is_last = (ticket == gridDim.x - 1);
        __threadfence();
    }
    __syncthreads();
    if (!is_last) return false;
    double a = 0.0;
    for (unsigned int i = threadIdx.x; i < gridDim.x; i += NT) a += __ldcg(partials + i);
    const double tot = block_sum<NT>(a, sm);
    if (threadIdx.x == 0) {
        *counter = 0u;  // ready for the next launch on this stream
        *total = tot;
        return true;
    }
    return false;
}

// The same single-pass reduction for N values at once (BiCGSTAB needs a complex and a real dot product per pass).
// partials holds N * gridDim.x doubles, value j of CTA b at j * gridDim.x + b.
template <int NT, int N>
__device__ __forceinline__ bool grid_sum_n(const double v[N], double *partials, unsigned int *counter, double total[N])
{
    __shared__ double sm[32];
    __shared__ int is_last;
    double b[N];
#pragma unroll
    for (int j = 0; j < N; ++j) b[j] = block_sum<NT>(v[j], sm);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int j = 0; j < N; ++j) partials[(size_t)j * gridDim.x + blockIdx.x] = b[j];
        __threadfence();
        const unsigned int ticket = atomicAdd(counter, 1u);
        is_last = (ticket == gridDim.x - 1);
        __threadfence();
    }
    __syncthreads();
    if (!is_last) return false;
    double tot[N];
#pragma unroll
    for (int j = 0; j < N; ++j) {
        double a = 0.0;
        for (unsigned int i = threadIdx.x; i < gridDim.x; i += NT) a += __ldcg(partials + (size_t)j * gridDim.x + i);
        tot[j] = block_sum<NT>(a, sm);
    }
    if (threadIdx.x == 0) {
        *counter = 0u;
#pragma unroll
        for (int j = 0; j < N; ++j) total[j] = tot[j];
        return true;
    }
    return false;
}

// The while-test of PAPER.md:47 read as relative 2-norm (G4): the loop goes on while sqrt(rr) >= r_min sqrt(eta2).  It
// STOPS as soon as that comparison fails -- also when rr is NaN or infinite (a non-finite link or source, qq = 0) --
// but `converged` is set only by the true comparison sqrt(rr) < r_min sqrt(eta2); a stop that is not a convergence
// raises `breakdown` and the solver returns WD_BREAKDOWN, never WD_OK with a NaN field.
struct LoopTest {
    bool go, converged;
};
__device__ __forceinline__ LoopTest loop_test(double rr, double eta2, double r_min)
{
    LoopTest t;
    const double rn = sqrt(rr), thr = r_min * sqrt(eta2);
    t.go = rn >= thr;
    t.converged = rn < thr;
    return t;
}
// state before the first iteration, rr = <r0,r0> (r0 = eta: rr = eta2, or the Schur source with eta2 the full norm):
// eta2 = 0 means psi = 0 is the solution (converged, no iteration); a non-finite norm is a breakdown
__device__ __forceinline__ void loop_begin(CgScalars *sc, double rr, double eta2, double r_min, int max_iter)
{
    const LoopTest t = loop_test(rr, eta2, r_min);
    const bool finite = isfinite(rr) && isfinite(eta2);
    const bool go = finite && eta2 > 0.0 && t.go;
    sc->k_stop = go ? max_iter : 0;
    sc->converged = (finite && !go) ? 1 : 0;
    sc->breakdown = finite ? 0 : 1;
}

// Scalar epilogues, run by one thread of the last CTA.
__device__ __forceinline__ void finish_qq(CgScalars *sc, double qq)
{
    sc->qq = qq;
    sc->alpha = sc->rr / qq;                       // alpha <- |r|^2 / |D-dagger p|^2 (G1)
}
__device__ __forceinline__ void finish_rr(CgScalars *sc, double rr_new, int it, double *hist)
{
    sc->beta = rr_new / sc->rr;                    // beta <- |r'|^2 / |r|^2 (G1)
    sc->rr = rr_new;
    sc->k = it + 1;
    if (hist) hist[it + 1] = rr_new;
    // while |r| >= r_min read as relative 2-norm (G4): stop as soon as it fails
    const LoopTest t = loop_test(rr_new, sc->eta2, sc->r_min);
    if (!t.go) {
        sc->k_stop = it + 1;
        if (t.converged) sc->converged = 1;
        else sc->breakdown = 1;              // rr is not a number: alpha or the fields are not finite
    }
}

// BiCGSTAB scalar epilogues (reading B1).  Complex division in fp64; a zero or non-finite denominator stops the
// loop (k_stop) and raises `breakdown`.
__device__ __forceinline__ bool cdiv(const double a[2], const double b[2], double q[2])
{
    const double d = b[0] * b[0] + b[1] * b[1];
    q[0] = (a[0] * b[0] + a[1] * b[1]) / d;
    q[1] = (a[1] * b[0] - a[0] * b[1]) / d;
    return d > 0.0 && isfinite(q[0]) && isfinite(q[1]);
}
__device__ __forceinline__ void bi_stop(CgScalars *sc, int it)
{
    sc->k_stop = it;   // kernels of iteration `it` launched after this one are no-ops
    sc->breakdown = 1;
}
// after v = D p: alpha <- rho / <rhat, v>
__device__ __forceinline__ void finish_rv(CgScalars *sc, const double rv[2], int it)
{
    if (!cdiv(sc->rho, rv, sc->calpha) || (sc->rho[0] == 0.0 && sc->rho[1] == 0.0)) bi_stop(sc, it);
}
// after t = D s: omega <- <t,s> / <t,t>   (tt = 0 means s = 0: omega = 0 and the x/r update finishes the solve)
__device__ __forceinline__ void finish_ts(CgScalars *sc, const double ts[2], double tt)
{
    sc->omega[0] = tt > 0.0 ? ts[0] / tt : 0.0;
    sc->omega[1] = tt > 0.0 ? ts[1] / tt : 0.0;
}
// after r <- s - omega t: rho' = <rhat, r>, rr = <r,r>; beta <- (rho'/rho)(alpha/omega); k <- k+1; loop test
__device__ __forceinline__ void finish_bi(CgScalars *sc, const double rho_new[2], double rr_new, int it, double *hist)
{
    sc->rr = rr_new;
    sc->k = it + 1;
    if (hist) hist[it + 1] = rr_new;
    const LoopTest lt = loop_test(rr_new, sc->eta2, sc->r_min);
    if (!lt.go) {
        sc->k_stop = it + 1;
        if (lt.converged) sc->converged = 1;
        else sc->breakdown = 1;
        return;
    }
    double a[2], b[2];
    const bool ok = cdiv(rho_new, sc->rho, a) && cdiv(sc->calpha, sc->omega, b);
    if (!ok) {
        sc->k_stop = it + 1;
        sc->breakdown = 1;
        return;
    }
    sc->cbeta[0] = a[0] * b[0] - a[1] * b[1];
    sc->cbeta[1] = a[0] * b[1] + a[1] * b[0];
    sc->rho[0] = rho_new[0];
    sc->rho[1] = rho_new[1];
}

// ---------------------------------------------------------------- the stencil kernel
enum { MODE_PLAIN = 0, MODE_QQ = 1, MODE_RUPD = 2, MODE_RV = 3, MODE_TS = 4 };

// MODE_PLAIN : out = D in / D-dagger in                                  (wd_apply, a6, a7)
// MODE_QQ    : out = q = D-dagger p, qq = |q|^2, alpha = rr/qq           (a2)
// MODE_RUPD  : s = D q (not stored), r <- r - alpha s, rr' = |r|^2, beta, loop condition   (a3)
// MODE_RV    : out = v = D p, <rhat, v> (rhat passed as `r`, read only), alpha = rho/<rhat,v>   (BiCGSTAB)
// MODE_TS    : out = t = D s, <t,s> and <t,t>, omega = <t,s>/<t,t>                              (BiCGSTAB)
// EO = 0: plain lattice (UB and cen are ignored: the backward links come from U, the diagonal term from `in`);
// EO = 1: the launch covers one parity of the lattice (even-odd preconditioning, Geom.eo / Geom.par).
template <typename real, int DAG, int MODE, int BX, int BY, int BZ, int BT, int MINB, int RECON = 18, int EO = 0>
__global__ void __launch_bounds__(BX *BY *BZ *BT, MINB)
dslash_kernel(const Geom g, const typename Field<real>::gvec *__restrict__ U,
              const typename Field<real>::gvec *__restrict__ UB, const typename Field<real>::svec *__restrict__ in,
              const typename Field<real>::svec *__restrict__ cen, typename Field<real>::svec *out, real kappa,
              typename Field<real>::svec *r, CgScalars *sc, double *partials, unsigned int *counter,
              double *hist, int it)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    constexpr int NT = BX * BY * BZ * BT;
    // The two-buffer pipeline with the diagonal term FIRST (hopping_sum CFIRST) wherever the pass has no second
    // per-site stream: measured at 48^3x96 fp32, a2 999 -> 920-934 us, wd_apply 990 -> 940 us.  MODE_RUPD keeps
    // the centre and r last: centre-first made a3 slower (1017 -> 1086 us), and so did folding r into the
    // accumulator as well (acc = r - alpha in, hops scaled by alpha kappa: 1056 us).  MODE_TS needs s(x) beside t(x).
    constexpr bool RU = MODE == MODE_RUPD;
    constexpr bool CF = MODE != MODE_TS && !RU;
    if (MODE != MODE_PLAIN) {
        if (it >= sc->k_stop) return;  // uniform over the grid: over-launched iterations are no-ops
    } else if (sc) {
        if (it >= sc->k_stop) return;  // a plain pass inside a solver loop (even-odd: the inner hop of Mhat)
    }
    const int tid = threadIdx.x;
    const int lx = tid % BX, ly = (tid / BX) % BY, lz = (tid / (BX * BY)) % BZ, lt = tid / (BX * BY * BZ);
    const real alpha = RU ? (real)sc->alpha : (real)0;
    double local = 0.0, local1 = 0.0, local2 = 0.0;
    // Persistent CTAs: the grid is one resident wave; CTA i takes tiles i, i + gridDim.x, ... so that at any
    // moment the chip works on gridDim.x consecutive tiles of the rasterisation (L2 locality) and the
    // reduction epilogue (barriers, fence, ticket) is paid once per CTA, not once per tile.
    for (int b = blockIdx.x; b < g.ntiles; b += gridDim.x) {
        int tx, ty, tz, tt;
        tile_of_block(g, b, tx, ty, tz, tt);
        const int x = tx * BX + lx, y = ty * BY + ly, z = tz * BZ + lz, t = tt * BT + lt;
        const bool active = (x < g.L[0]) && (y < g.L[1]) && (z < g.L[2]) && (t < g.L[3]);
        if (!active) continue;
        const int s = x + g.L[0] * (y + g.L[1] * (z + g.L[2] * t));
        real acc[24], c[24], rv[24];
        hopping_sum<DAG, 1, RU || MODE == MODE_RV, true, real, svec, gvec, RECON, EO, CF>(
            g, U, EO ? UB : U, in, EO ? cen : in, r, x, y, z, t, s, acc, c, rv, kappa);
        if constexpr (MODE == MODE_TS) {
            // c holds s(x); t(x) = s(x) - kappa * hops replaces it component by component
            real tsr = 0, tsi = 0, tt = 0;
#pragma unroll
            for (int j = 0; j < 12; ++j) {
                const real sr = c[2 * j], si = c[2 * j + 1];
                const real tr = fma(-kappa, acc[2 * j], sr), ti = fma(-kappa, acc[2 * j + 1], si);
                tsr = fma(tr, sr, tsr); tsr = fma(ti, si, tsr);      // conj(t) s
                tsi = fma(tr, si, tsi); tsi = fma(-ti, sr, tsi);
                tt = fma(tr, tr, tt); tt = fma(ti, ti, tt);
                c[2 * j] = tr; c[2 * j + 1] = ti;
            }
            store_spinor(out, s, c);
            local += (double)tsr; local1 += (double)tsi; local2 += (double)tt;
        } else {
#pragma unroll
        for (int i = 0; i < 24; ++i) c[i] = CF ? acc[i] : fma(-kappa, acc[i], c[i]);  // (D in)(x) = in(x) - kappa * hops
        if (MODE == MODE_RV) {
            real dr = 0, di = 0;
#pragma unroll
            for (int j = 0; j < 12; ++j) {                              // conj(rhat) v
                dr = fma(rv[2 * j], c[2 * j], dr); dr = fma(rv[2 * j + 1], c[2 * j + 1], dr);
                di = fma(rv[2 * j], c[2 * j + 1], di); di = fma(-rv[2 * j + 1], c[2 * j], di);
            }
            store_spinor(out, s, c);
            local += (double)dr; local1 += (double)di;
        } else if (RU) {
            real n2 = 0;
#pragma unroll
            for (int i = 0; i < 24; ++i) {
                rv[i] = fma(-alpha, c[i], rv[i]);                      // r <- r - alpha D D-dagger p
                n2 = fma(rv[i], rv[i], n2);
            }
            store_spinor(r, s, rv);
            local += (double)n2;
        } else {
            store_spinor(out, s, c);
            if (MODE == MODE_QQ) {
                real n2 = 0;
#pragma unroll
                for (int i = 0; i < 24; ++i) n2 = fma(c[i], c[i], n2);
                local += (double)n2;
            }
        }
        }  // MODE != MODE_TS
    }
    if (MODE == MODE_QQ || RU) {
        double total;
        if (grid_sum<NT>(local, partials, counter, &total)) {
            if (MODE == MODE_QQ) finish_qq(sc, total);
            else finish_rr(sc, total, it, hist);
        }
    } else if (MODE == MODE_RV) {
        const double v2[2] = {local, local1};
        double tot[2];
        if (grid_sum_n<NT, 2>(v2, partials, counter, tot)) finish_rv(sc, tot, it);
    } else if (MODE == MODE_TS) {
        const double v3[3] = {local, local1, local2};
        double tot[3];
        if (grid_sum_n<NT, 3>(v3, partials, counter, tot)) finish_ts(sc, tot, tot[2]);
    }
}

// ---------------------------------------------------------------- the whole CG in ONE launch (small volumes)
// SURVEY.md 8(f1).  On the paper's own volumes (4^4 ... 14^4) one CG iteration moves 0.4-59 MB, all of
// it L2-resident: 0.05-9 us of memory time, far below three kernel launches.  This kernel runs init, the loop
// and the final D-dagger in a single cooperative launch; the three phases of an iteration are separated by
// grid barriers instead of kernel boundaries.  Every CTA sums the per-CTA partials in the same fixed order, so
// alpha, beta and the loop test are identical everywhere (no broadcast, deterministic).  The recurrence and the
// precision rules are exactly those of the three-kernel path.
template <int NT>
__device__ __forceinline__ double all_cta_sum(const double *partials, int n, double *sm)
{
    double a = 0.0;
    for (int i = threadIdx.x; i < n; i += NT) a += __ldcg(partials + i);
    const double t = block_sum<NT>(a, sm);
    if (threadIdx.x == 0) sm[32] = t;
    __syncthreads();
    const double out = sm[32];
    __syncthreads();
    return out;
}

template <typename real, int BX, int BY, int BZ, int BT, int MINB, int PIPE>
__global__ void __launch_bounds__(BX *BY *BZ *BT, MINB)
cg_onelaunch_kernel(const Geom g, const typename Field<real>::gvec *__restrict__ U,
                    const typename Field<real>::svec *__restrict__ eta, typename Field<real>::svec *y,
                    typename Field<real>::svec *r, typename Field<real>::svec *p, typename Field<real>::svec *q,
                    typename Field<real>::svec *psi, real kappa, CgScalars *sc, double *partials, double *hist,
                    double r_min, int max_iter)
{
    namespace cg = cooperative_groups;
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    constexpr int NT = BX * BY * BZ * BT;
    cg::grid_group grid = cg::this_grid();
    __shared__ double sm[33];
    const int G = gridDim.x;
    double *part0 = partials, *part1 = partials + G, *part2 = partials + 2 * G;
    const int tid = threadIdx.x;
    const int lx = tid % BX, ly = (tid / BX) % BY, lz = (tid / (BX * BY)) % BZ, lt = tid / (BX * BY * BZ);

#define WD_FOR_EACH_SITE(...)                                                                     \
    for (int b_ = blockIdx.x; b_ < g.ntiles; b_ += G) {                                             \
        int tx_, ty_, tz_, tt_;                                                                     \
        tile_of_block(g, b_, tx_, ty_, tz_, tt_);                                                   \
        const int x = tx_ * BX + lx, y_ = ty_ * BY + ly, z = tz_ * BZ + lz, t = tt_ * BT + lt;      \
        if (x < g.L[0] && y_ < g.L[1] && z < g.L[2] && t < g.L[3]) {                                \
            const int s = x + g.L[0] * (y_ + g.L[1] * (z + g.L[2] * t));                            \
            __VA_ARGS__                                                                             \
        }                                                                                           \
    }

    // a1: y <- 0, r <- eta, p <- eta, rr = <eta,eta>
    double local = 0.0;
    WD_FOR_EACH_SITE({
        real e[24], zero[24];
        load_spinor(eta, s, e);
        real n2 = 0;
#pragma unroll
        for (int i = 0; i < 24; ++i) { zero[i] = 0; n2 = fma(e[i], e[i], n2); }
        store_spinor(y, s, zero); store_spinor(r, s, e); store_spinor(p, s, e);
        local += (double)n2;
    })
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
        WD_FOR_EACH_SITE({
            real acc[24], c[24], dummy[24];
            hopping_sum<1, PIPE, false, false, real, svec, gvec>(g, U, U, p, p, nullptr, x, y_, z, t, s, acc, c, dummy);
            real n2 = 0;
#pragma unroll
            for (int i = 0; i < 24; ++i) { c[i] = fma(-kappa, acc[i], c[i]); n2 = fma(c[i], c[i], n2); }
            store_spinor(q, s, c);
            local += (double)n2;
        })
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
        WD_FOR_EACH_SITE({
            real acc[24], c[24], rv[24];
            hopping_sum<0, PIPE, true, false, real, svec, gvec>(g, U, U, q, q, r, x, y_, z, t, s, acc, c, rv);
            real n2 = 0;
#pragma unroll
            for (int i = 0; i < 24; ++i) {
                c[i] = fma(-kappa, acc[i], c[i]);
                rv[i] = fma(-al, c[i], rv[i]);
                n2 = fma(rv[i], rv[i], n2);
            }
            store_spinor(r, s, rv);
            local += (double)n2;
        })
        {
            const double bsum = block_sum<NT>(local, sm);
            if (tid == 0) part2[blockIdx.x] = bsum;
        }
        grid.sync();
        const double rr_new = all_cta_sum<NT>(part2, G, sm);
        beta = rr_new / rr;                                  // beta <- |r'|^2 / |r|^2
        const real be = (real)beta;
        // a4: y <- y + alpha p ; p <- r + beta p (own sites only)
        WD_FOR_EACH_SITE({
            real yv[24], pv[24], rv[24];
            load_spinor_rw(y, s, yv); load_spinor_rw(p, s, pv); load_spinor_rw(r, s, rv);
#pragma unroll
            for (int i = 0; i < 24; ++i) { yv[i] = fma(al, pv[i], yv[i]); pv[i] = fma(be, pv[i], rv[i]); }
            store_spinor(y, s, yv); store_spinor(p, s, pv);
        })
        rr = rr_new;
        ++k;
        if (blockIdx.x == 0 && tid == 0 && hist) hist[k] = rr;
        go = loop_test(rr, eta2, r_min).go;                  // while |r| >= r_min (G4)
        grid.sync();                                         // p complete before its neighbours are read
    }
    // a6: psi = D-dagger y
    WD_FOR_EACH_SITE({
        real acc[24], c[24], dummy[24];
        hopping_sum<1, PIPE, false, false, real, svec, gvec>(g, U, U, y, y, nullptr, x, y_, z, t, s, acc, c, dummy);
#pragma unroll
        for (int i = 0; i < 24; ++i) c[i] = fma(-kappa, acc[i], c[i]);
        store_spinor(psi, s, c);
    })
#undef WD_FOR_EACH_SITE
    if (blockIdx.x == 0 && tid == 0) {
        sc->rr = rr; sc->eta2 = eta2; sc->alpha = alpha; sc->beta = beta; sc->qq = 0.0; sc->r_min = r_min;
        sc->k = k; sc->k_stop = k; sc->max_iter = max_iter;
        // converged: psi = 0 for eta = 0, or the true comparison; a loop that stopped otherwise met a NaN (loop_test)
        sc->converged = (eta2 == 0.0 || loop_test(rr, eta2, r_min).converged) ? 1 : 0;
        sc->breakdown = (!go && !sc->converged) ? 1 : 0;
    }
}

// ---------------------------------------------------------------- streaming vector kernels
constexpr int VEC_NT = 256;

template <typename vec> __device__ __forceinline__ double vnorm2(const vec &a);
template <> __device__ __forceinline__ double vnorm2<float4>(const float4 &a)
{
    return (double)(a.x * a.x + a.y * a.y + a.z * a.z + a.w * a.w);
}
template <> __device__ __forceinline__ double vnorm2<double2>(const double2 &a) { return a.x * a.x + a.y * a.y; }

__device__ __forceinline__ float4 vzero(float4) { return make_float4(0.f, 0.f, 0.f, 0.f); }
__device__ __forceinline__ double2 vzero(double2) { return make_double2(0.0, 0.0); }
__device__ __forceinline__ float4 vaxpy(float a, const float4 &x, const float4 &y)
{
    return make_float4(fmaf(a, x.x, y.x), fmaf(a, x.y, y.y), fmaf(a, x.z, y.z), fmaf(a, x.w, y.w));
}
__device__ __forceinline__ double2 vaxpy(double a, const double2 &x, const double2 &y)
{
    return make_double2(fma(a, x.x, y.x), fma(a, x.y, y.y));
}

// Element i of a native spinor buffer (i counts 128-bit vectors) belongs to site (i / (NSP*SB))*SB + i % SB.
// `V` is the number of real sites; when the volume is not a multiple of SB the pad lanes of the last block
// are skipped (padded == 0 -> no test at all).
template <int NSP>
__device__ __forceinline__ bool real_site(size_t i, int V, int padded)
{
    if (!padded) return true;
    const size_t blk = i / (NSP * SB);
    return (int)(blk * SB + (i & (SB - 1))) < V;
}

// a1: y <- 0, r <- eta, p <- eta, rr = eta2 = <eta,eta>, k = 0 ("psi <- psi0; r <- eta - D psi; p <- r", psi0 = 0)
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
cg_init_kernel(const typename Field<real>::svec *__restrict__ eta, typename Field<real>::svec *y,
               typename Field<real>::svec *r, typename Field<real>::svec *p, size_t n, int V, int padded,
               CgScalars *sc, double *partials, unsigned int *counter, double *hist, double r_min, int max_iter)
{
    using svec = typename Field<real>::svec;
    double local = 0.0;
    for (size_t i = (size_t)blockIdx.x * VEC_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * VEC_NT) {
        const svec e = real_site<Field<real>::NSP>(i, V, padded) ? __ldg(eta + i) : svec();
        y[i] = vzero(e);
        r[i] = e;
        p[i] = e;
        local += vnorm2<svec>(e);
    }
    double total;
    if (grid_sum<VEC_NT>(local, partials, counter, &total)) {
        sc->rr = total; sc->eta2 = total; sc->qq = 0.0; sc->alpha = 0.0; sc->beta = 0.0;
        sc->r_min = r_min; sc->k = 0; sc->max_iter = max_iter;
        loop_begin(sc, total, total, r_min, max_iter);
        if (hist) hist[0] = total;
    }
}

// a4: y <- y + alpha p ; p <- r + beta p   ("psi <- psi + alpha p", "p <- r + beta p"; G3: y, not psi)
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
cg_update_kernel(typename Field<real>::svec *y, typename Field<real>::svec *p,
                 const typename Field<real>::svec *__restrict__ r, size_t n, const CgScalars *sc, int it)
{
    using svec = typename Field<real>::svec;
    if (it >= sc->k_stop) return;
    const real alpha = (real)sc->alpha, beta = (real)sc->beta;
    for (size_t i = (size_t)blockIdx.x * VEC_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * VEC_NT) {
        const svec pv = p[i];
        const svec rv = __ldg(r + i);
        y[i] = vaxpy(alpha, pv, y[i]);
        p[i] = vaxpy(beta, pv, rv);
    }
}

// ---------------------------------------------------------------- BiCGSTAB vector kernels (reading B1)
// complex a (ar + i ai) times x plus y on one 128-bit vector (fp32: two complex numbers, fp64: one)
__device__ __forceinline__ float4 vcaxpy(float ar, float ai, const float4 &x, const float4 &y)
{
    return make_float4(fmaf(-ai, x.y, fmaf(ar, x.x, y.x)), fmaf(ai, x.x, fmaf(ar, x.y, y.y)),
                       fmaf(-ai, x.w, fmaf(ar, x.z, y.z)), fmaf(ai, x.z, fmaf(ar, x.w, y.w)));
}
__device__ __forceinline__ double2 vcaxpy(double ar, double ai, const double2 &x, const double2 &y)
{
    return make_double2(fma(-ai, x.y, fma(ar, x.x, y.x)), fma(ai, x.x, fma(ar, x.y, y.y)));
}
// conj(a) b summed over the complex numbers of one vector: (re, im)
__device__ __forceinline__ void vcdot(const float4 &a, const float4 &b, double &re, double &im)
{
    re += (double)(a.x * b.x + a.y * b.y + a.z * b.z + a.w * b.w);
    im += (double)(a.x * b.y - a.y * b.x + a.z * b.w - a.w * b.z);
}
__device__ __forceinline__ void vcdot(const double2 &a, const double2 &b, double &re, double &im)
{
    re += a.x * b.x + a.y * b.y;
    im += a.x * b.y - a.y * b.x;
}

// psi <- 0; r <- eta; p <- eta; rho = rr = eta2 = <eta,eta>; k = 0   (rhat = eta itself, never copied)
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
bi_init_kernel(const typename Field<real>::svec *__restrict__ eta, typename Field<real>::svec *psi,
               typename Field<real>::svec *r, typename Field<real>::svec *p, size_t n, int V, int padded,
               CgScalars *sc, double *partials, unsigned int *counter, double *hist, double r_min, int max_iter)
{
    using svec = typename Field<real>::svec;
    double local = 0.0;
    for (size_t i = (size_t)blockIdx.x * VEC_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * VEC_NT) {
        const svec e = real_site<Field<real>::NSP>(i, V, padded) ? __ldg(eta + i) : svec();
        psi[i] = vzero(e);
        r[i] = e;
        p[i] = e;
        local += vnorm2<svec>(e);
    }
    double total;
    if (grid_sum<VEC_NT>(local, partials, counter, &total)) {
        sc->rr = total; sc->eta2 = total; sc->qq = 0.0; sc->alpha = 0.0; sc->beta = 0.0;
        sc->rho[0] = total; sc->rho[1] = 0.0;
        sc->calpha[0] = sc->calpha[1] = sc->omega[0] = sc->omega[1] = sc->cbeta[0] = sc->cbeta[1] = 0.0;
        sc->r_min = r_min; sc->k = 0; sc->max_iter = max_iter;
        loop_begin(sc, total, total, r_min, max_iter);
        if (hist) hist[0] = total;
    }
}

// The BiCGSTAB vector kernels never trust the pad lanes of their inputs (volume not a multiple of the 16-site block):
// v and t are written by the stencil, which skips pad lanes, and the even-odd solvers run on half-length views of
// work vectors that earlier full-lattice solves have filled; rhat = eta belongs to the caller.  Pad lanes of every
// output are written as zero and contribute nothing to the dot products.
// s <- r - alpha v
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
bi_s_kernel(typename Field<real>::svec *s, const typename Field<real>::svec *__restrict__ r,
            const typename Field<real>::svec *__restrict__ v, size_t n, int V, int padded, const CgScalars *sc, int it)
{
    using svec = typename Field<real>::svec;
    if (it >= sc->k_stop) return;
    const real ar = (real)(-sc->calpha[0]), ai = (real)(-sc->calpha[1]);
    for (size_t i = (size_t)blockIdx.x * VEC_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * VEC_NT)
        s[i] = real_site<Field<real>::NSP>(i, V, padded) ? vcaxpy(ar, ai, __ldg(v + i), __ldg(r + i)) : vzero(svec());
}

// psi <- psi + alpha p + omega s ; r <- s - omega t ; rho' = <rhat,r> ; rr = <r,r> ; beta ; k ; loop test
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
bi_xr_kernel(typename Field<real>::svec *psi, typename Field<real>::svec *r,
             const typename Field<real>::svec *__restrict__ p, const typename Field<real>::svec *__restrict__ s,
             const typename Field<real>::svec *__restrict__ t, const typename Field<real>::svec *__restrict__ rhat,
             size_t n, int V, int padded, CgScalars *sc, double *partials, unsigned int *counter, double *hist, int it)
{
    using svec = typename Field<real>::svec;
    if (it >= sc->k_stop) return;
    const real ar = (real)sc->calpha[0], ai = (real)sc->calpha[1];
    const real wr = (real)sc->omega[0], wi = (real)sc->omega[1];
    double v3[3] = {0.0, 0.0, 0.0};
    for (size_t i = (size_t)blockIdx.x * VEC_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * VEC_NT) {
        if (!real_site<Field<real>::NSP>(i, V, padded)) {
            psi[i] = vzero(svec());
            r[i] = vzero(svec());
            continue;
        }
        const svec sv = __ldg(s + i);
        psi[i] = vcaxpy(wr, wi, sv, vcaxpy(ar, ai, __ldg(p + i), psi[i]));
        const svec rn = vcaxpy(-wr, -wi, __ldg(t + i), sv);
        r[i] = rn;
        vcdot(__ldg(rhat + i), rn, v3[0], v3[1]);
        v3[2] += vnorm2<svec>(rn);
    }
    double tot[3];
    if (grid_sum_n<VEC_NT, 3>(v3, partials, counter, tot)) finish_bi(sc, tot, tot[2], it, hist);
}

// p <- r + beta (p - omega v)
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
bi_p_kernel(typename Field<real>::svec *p, const typename Field<real>::svec *__restrict__ r,
            const typename Field<real>::svec *__restrict__ v, size_t n, int V, int padded, const CgScalars *sc, int it)
{
    using svec = typename Field<real>::svec;
    if (it >= sc->k_stop) return;
    const real br = (real)sc->cbeta[0], bi = (real)sc->cbeta[1];
    const real wr = (real)(-sc->omega[0]), wi = (real)(-sc->omega[1]);
    for (size_t i = (size_t)blockIdx.x * VEC_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * VEC_NT)
        p[i] = real_site<Field<real>::NSP>(i, V, padded)
                   ? vcaxpy(br, bi, vcaxpy(wr, wi, __ldg(v + i), p[i]), __ldg(r + i)) : vzero(svec());
}

// the paper's dot-product kernel on its own: <a,a>
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
norm2_kernel(const typename Field<real>::svec *__restrict__ a, size_t n, int V, int padded, double *partials,
             unsigned int *counter, double *result)
{
    using svec = typename Field<real>::svec;
    double local = 0.0;
    for (size_t i = (size_t)blockIdx.x * VEC_NT + threadIdx.x; i < n; i += (size_t)gridDim.x * VEC_NT)
        if (real_site<Field<real>::NSP>(i, V, padded)) local += vnorm2<svec>(__ldg(a + i));
    double total;
    if (grid_sum<VEC_NT>(local, partials, counter, &total)) *result = total;
}

// ---------------------------------------------------------------- a0: canonical <-> native permutations
// One thread per (padded) site.  canonical gauge U[s][mu][a][b] (36 complex, contiguous) -> plane mu*9+a*3+b of
// the site's block; canonical spinor psi[s][alpha][a] (NSP vectors, contiguous) -> plane j.  Pad lanes get zeros.
template <typename real, int RECON = 18>
__global__ void __launch_bounds__(VEC_NT)
pack_gauge_kernel(const typename Field<real>::gvec *__restrict__ can, typename Field<real>::gvec *nat, int V, int Vpad,
                  int s0 = 0)
{
    // sites s0 .. Vpad - 1 (the host-buffer calls pack slab by slab as the copies land; the grid bounds the slab)
    using gvec = typename Field<real>::gvec;
    const int s = s0 + blockIdx.x * VEC_NT + threadIdx.x;
    if (s >= Vpad) return;
    for (int mu = 0; mu < 4; ++mu) {
        gvec k9[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) k9[k] = s < V ? __ldg(can + (size_t)s * 36 + mu * 9 + k) : gvec();
        if (RECON == 12) store_link12(nat, s, mu, k9);
        else store_link(nat, s, mu, k9);
    }
}
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
pack_spinor_kernel(const typename Field<real>::svec *__restrict__ can, typename Field<real>::svec *nat, int V, int Vpad,
                   int s0 = 0)
{
    using svec = typename Field<real>::svec;
    constexpr int NSP = Field<real>::NSP;
    const int s = s0 + blockIdx.x * VEC_NT + threadIdx.x;
    if (s >= Vpad) return;
    svec *p = nat + spinor_index<svec, NSP>(s);
#pragma unroll
    for (int j = 0; j < NSP; ++j) p[j * SB] = s < V ? __ldg(can + (size_t)s * NSP + j) : svec();
}
template <typename real>
__global__ void __launch_bounds__(VEC_NT)
unpack_spinor_kernel(const typename Field<real>::svec *__restrict__ nat, typename Field<real>::svec *can, int V, int s0 = 0)
{
    using svec = typename Field<real>::svec;
    constexpr int NSP = Field<real>::NSP;
    const int s = s0 + blockIdx.x * VEC_NT + threadIdx.x;
    if (s >= V) return;
    const svec *p = nat + spinor_index<svec, NSP>(s);
#pragma unroll
    for (int j = 0; j < NSP; ++j) can[(size_t)s * NSP + j] = __ldg(p + j * SB);
}

// ---------------------------------------------------------------- host helper shared by all launchers
// Resident CTAs per SM of a kernel on the CURRENT device, cached per device in `table` (WD_MAXDEV ints, zero-initialised,
// one table per kernel instantiation: declare it `static` next to the launch).  A process may drive several GPUs (one ctx
// per device) and the persistent / cooperative grids are sized from this number, so one process-wide value is not enough.
constexpr int WD_MAXDEV = 64;
template <typename Kern>
static cudaError_t cached_occupancy(int *table, Kern kern, int threads, size_t dyn_smem, int *out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= WD_MAXDEV) dev = WD_MAXDEV - 1;
    int v = __atomic_load_n(&table[dev], __ATOMIC_RELAXED);
    if (!v) {
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, kern, threads, dyn_smem);
        if (e != cudaSuccess) return e;
        if (v < 1) return cudaErrorLaunchOutOfResources;
        __atomic_store_n(&table[dev], v, __ATOMIC_RELAXED);
    }
    *out = v;
    return cudaSuccess;
}

}  // namespace wd

// wilson_tma.cuh — the Wilson-Dirac stencil with a COMPLETE shared-memory link pipeline (BASELINE.json north_star (2):
// "stages neighbour spinors and links through shared memory or TMA tiles"; the matrix-vector product is
// the most demanding, memory-bound part).
//
// Same arithmetic, same hop order and same fused epilogues as dslash_kernel (wilson_kernels.cuh): results are bit-identical.
// What changes is how the gauge field -- 60 % of the bytes of a pass -- reaches the arithmetic:
//
//   * the links never pass through L1 or through registers held in flight.  The site-blocked layout keeps the link U_mu
//     of 16 consecutive sites in ONE contiguous chunk (1152 B fp32, 2304 B fp64), so a CTA tile of 16 x BY x BZ x BT
//     sites needs, per direction mu, NR = BY*BZ*BT bulk copies for its own rows plus the rows of its -mu face (the
//     links U_mu(x - mu) of the backward hop of the sites on that face).  They are fetched by the bulk-copy engine
//     (cp.async.bulk.shared.global = TMA without a tensor map, SASS UBLKCP) into a ring of two shared-memory stages,
//     one stage per (tile, mu), each guarded by a `full` mbarrier (expect_tx / complete_tx) and an `empty` mbarrier
//     (one arrival per consumer warp);
//   * BOTH uses of a link are served from that copy: the forward hop of the owner reads its own slot, the backward hop
//     of the +mu neighbour reads the slot of the site behind it (same row one lane to the left for mu = x, another row or
//     a halo row otherwise).  Only the x-halo (lane 15 of the previous 16-site block, one site per row) is read straight
//     from global memory by the one lane that needs it;
//   * the copies run one stage (one direction) in front of the arithmetic and across tile boundaries (the ring does not
//     drain when the persistent CTA moves to its next tile), with no register and no L1 line held while they are in flight;
//   * warp 0 is the issuer (its 32 lanes issue the row copies of a stage in parallel after waiting for the stage to be
//     empty); there is no dedicated producer warp, because an idle warp would cost every CTA 32 x 128 registers;
//   * the L1 keeps the neighbour spinors only (they still come through the read-only path with the two-buffer register
//     pipeline of hopping_sum: a tile plus its eight halo faces of spinors does not fit shared memory twice).
//
// Preconditions (checked by the launcher, which otherwise falls back to dslash_kernel): plain lattice (no even-odd),
// 18 reals per link, Lx a multiple of 16 and the other extents multiples of BY, BZ, BT.
#pragma once
#include "wilson_kernels.cuh"

namespace wd {

// ---------------------------------------------------------------- mbarrier / bulk-copy primitives (PTX ISA 8.0+, sm_90+)
__device__ __forceinline__ unsigned int smem_u32(const void *p) { return (unsigned int)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// makes the initialised barriers visible to the async proxy (the bulk-copy engine completes transactions on them)
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *bar, unsigned int bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// blocks until the phase with the given parity has completed (try_wait suspends the thread in hardware, it is not a spin)
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned int parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// contiguous global -> shared copy by the bulk-copy engine; completes `bytes` on the mbarrier.  16-byte aligned, size % 16 == 0.
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned int bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---------------------------------------------------------------- link reads from a stage row
// A stage row is the link-mu section of one 16-site gauge block, byte for byte as in global memory.  Addresses are 32-bit
// shared-window addresses (one register per row base instead of a 64-bit generic pointer); `a16` = row base + 16 * lane.
// The loads are volatile asm so that they stay behind the mbarrier wait that guards the stage.
__device__ __forceinline__ float4 lds_f4(unsigned int a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ float2 lds_f2(unsigned int a)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ double2 lds_d2(unsigned int a)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
// fp32: four float4 planes (lane stride 16 B) and one float2 plane (lane stride 8 B: a16 + 1024 - 8 * lane)
__device__ __forceinline__ void load_link_row(unsigned int a16, int lane8, float u[18])
{
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float4 t = lds_f4(a16 + q * SB * 16);
        u[4 * q] = t.x; u[4 * q + 1] = t.y; u[4 * q + 2] = t.z; u[4 * q + 3] = t.w;
    }
    const float2 t2 = lds_f2(a16 + 4 * SB * 16 - lane8);
    u[16] = t2.x; u[17] = t2.y;
}
__device__ __forceinline__ void load_link_row(unsigned int a16, int, double u[18])
{
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const double2 t = lds_d2(a16 + k * SB * 16);
        u[2 * k] = t.x; u[2 * k + 1] = t.y;
    }
}

constexpr int tma_max3(int a, int b, int c) { return a > b ? (a > c ? a : c) : (b > c ? b : c); }
// The ring has TWO stages and a CTA walks stage j = 4 * (tile number) + mu: slot = j & 1 = mu & 1 and the phase parity of
// the slot's barriers, (j >> 1) & 1 = mu >> 1, are COMPILE-TIME constants of the direction (a deeper ring costs modulo
// arithmetic in every direction of every tile and shared memory the L1 needs for the neighbour spinors; measured).
constexpr int TMA_NSTAGE = 2;
template <typename real, int BY, int BZ, int BT> struct TmaShape {
    static constexpr int NR = BY * BZ * BT;                                   // rows (16-site blocks) of the tile
    static constexpr int NH = tma_max3(BZ * BT, BY * BT, BY * BZ);            // rows of the largest -mu face
    static constexpr int LB = 9 * SB * 2 * (int)sizeof(real);                 // bytes of one link direction of one block
    static constexpr int STAGE = (NR + NH) * LB;
    static constexpr int HEADER = 128;                                        // 2 x 2 mbarriers, padded
    static constexpr int SMEM = HEADER + TMA_NSTAGE * STAGE;
    static constexpr int NT = SB * NR;
};

// Warp 0, all lanes: enqueue the copies of direction MU of the tile at (x0, y0, z0, t0) into slot MU & 1, after every warp
// has released the slot's previous tenant.  Lane c copies row c: rows 0 .. NR-1 are the tile's own 16-site blocks, rows
// NR .. NR+nh-1 the blocks of its -MU face (U_mu(x - mu) of the backward hop), with the lattice wrap.
template <typename real, int MU, int BY, int BZ, int BT>
__device__ __forceinline__ void tma_issue(const Geom &g, const unsigned char *Ubytes, unsigned char *ring,
                                          unsigned long long *full, unsigned long long *empty, int lane, int x0, int y0,
                                          int z0, int t0)
{
    using S = TmaShape<real, BY, BZ, BT>;
    constexpr int NR = S::NR, LB = S::LB, SLOT = MU & 1;
    constexpr int NH = MU == 0 ? 0 : (MU == 1 ? BZ * BT : (MU == 2 ? BY * BT : BY * BZ));
    constexpr size_t BLOCK_BYTES = (size_t)36 * SB * 2 * sizeof(real);
    static_assert(NR + NH <= 64, "two copies per lane at most");
    // stage jf = 4 k + MU is tenant number n = jf >> 1 of its slot: tenant n - 1 must have been released, i.e. phase
    // n - 1 of `empty` completed; its parity ((n - 1) & 1) is 1 for MU in {0, 1} and 0 for MU in {2, 3} (a fresh barrier
    // reports the phase of parity 1 as complete, so the first two stages pass at once)
    mbar_wait(empty + SLOT, MU < 2 ? 1u : 0u);
    if (lane == 0) mbar_arrive_expect_tx(full + SLOT, (unsigned int)((NR + NH) * LB));
    __syncwarp();
    unsigned char *dst0 = ring + (size_t)SLOT * S::STAGE;
#pragma unroll
    for (int c0 = 0; c0 < NR + NH; c0 += 32) {
        const int c = c0 + lane;
        if (c < NR + NH) {
            int y, z, t;
            if (c < NR) {
                y = y0 + c % BY; z = z0 + (c / BY) % BZ; t = t0 + c / (BY * BZ);
            } else {
                const int h = c - NR;
                if (MU == 1) {
                    y = y0 == 0 ? g.L[1] - 1 : y0 - 1; z = z0 + h % BZ; t = t0 + h / BZ;
                } else if (MU == 2) {
                    y = y0 + h % BY; z = z0 == 0 ? g.L[2] - 1 : z0 - 1; t = t0 + h / BY;
                } else {
                    y = y0 + h % BY; z = z0 + h / BY; t = t0 == 0 ? g.L[3] - 1 : t0 - 1;
                }
            }
            const int s0 = x0 + g.L[0] * (y + g.L[1] * (z + g.L[2] * t));
            bulk_g2s(dst0 + (size_t)c * LB, Ubytes + (size_t)(s0 >> SB_SHIFT) * BLOCK_BYTES + (size_t)MU * LB, LB, full + SLOT);
        }
    }
}

// MODE_PLAIN / MODE_QQ / MODE_RUPD as in dslash_kernel.
template <typename real, int DAG, int MODE, int BY, int BZ, int BT, int MINB, int UB2>
__global__ void __launch_bounds__(SB *BY *BZ *BT, MINB)
dslash_tma_kernel(const Geom g, const typename Field<real>::gvec *__restrict__ U,
                  const typename Field<real>::svec *__restrict__ in, typename Field<real>::svec *out, real kappa,
                  typename Field<real>::svec *r, CgScalars *sc, double *partials, unsigned int *counter, double *hist, int it)
{
    using svec = typename Field<real>::svec;
    using S = TmaShape<real, BY, BZ, BT>;
    constexpr int NR = S::NR, NT = S::NT, NW = NT / 32, LB = S::LB;
    static_assert(NT % 32 == 0, "whole warps");
    static_assert(MODE == MODE_PLAIN || MODE == MODE_QQ || MODE == MODE_RUPD, "CG modes only");
    constexpr bool RU = MODE == MODE_RUPD;
    constexpr bool CF = !RU;                                   // diagonal term first, as in dslash_kernel
    constexpr int SF = DAG ? +1 : -1;
    if (MODE != MODE_PLAIN) {
        if (it >= sc->k_stop) return;   // uniform over the grid: over-launched iterations are no-ops
    } else if (sc) {
        if (it >= sc->k_stop) return;
    }
    extern __shared__ __align__(128) unsigned char tma_smem[];
    unsigned long long *full = reinterpret_cast<unsigned long long *>(tma_smem);
    unsigned long long *empty = full + TMA_NSTAGE;
    unsigned char *ring = tma_smem + S::HEADER;

    const int tid = threadIdx.x, lane = tid & 31;
    const bool issuer = tid < 32;                              // warp 0
    const int lx = tid % SB, row = tid / SB;
    const int ly = row % BY, lz = (row / BY) % BZ, lt = row / (BY * BZ);
    // this thread's slots in a stage: its own link, and U_mu(x - mu): same row one lane to the left, another row of the
    // tile, or a halo row behind the NR own rows
    const unsigned int ring32 = smem_u32(ring) + 16u * lx;
    const int lx8 = 8 * lx;
    const unsigned int own = ring32 + row * LB;
    const unsigned int rb1 = ring32 + (ly > 0 ? row - 1 : NR + lz + BZ * lt) * LB;
    const unsigned int rb2 = ring32 + (lz > 0 ? row - BY : NR + ly + BY * lt) * LB;
    const unsigned int rb3 = ring32 + (lt > 0 ? row - BY * BZ : NR + ly + BY * lz) * LB;
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < TMA_NSTAGE; ++i) {
            mbar_init(full + i, 1);      // the issuer's arrive.expect_tx; the copies complete the transaction bytes
            mbar_init(empty + i, NW);    // one arrival per consumer warp
        }
        mbar_fence_init();
    }
    __syncthreads();
    if ((int)blockIdx.x >= g.ntiles) return;
    const unsigned char *Ubytes = reinterpret_cast<const unsigned char *>(U);
    int tx, ty, tz, tt;
    tile_of_block(g, blockIdx.x, tx, ty, tz, tt);
    if (issuer) tma_issue<real, 0, BY, BZ, BT>(g, Ubytes, ring, full, empty, lane, tx * SB, ty * BY, tz * BZ, tt * BT);

    const real alpha = RU ? (real)sc->alpha : (real)0;
    double local = 0.0;
    for (int b = blockIdx.x; b < g.ntiles; b += gridDim.x) {
        const int x0 = tx * SB, y0 = ty * BY, z0 = tz * BZ, t0 = tt * BT;
        const int x = x0 + lx, y = y0 + ly, z = z0 + lz, t = t0 + lt;
        const int s = x + g.L[0] * (y + g.L[1] * (z + g.L[2] * t));
        const Hops n = neighbours<0>(g, x, y, z, t, s);
        const real one = CF ? -kappa : (real)1;
        const real sgf = (t == g.L[3] - 1) ? (real)g.bc_t * one : one;
        const real sgb = (t == 0) ? (real)g.bc_t * one : one;
        real acc[24], c[24], rv[24];
        real va[24], vb[24], u[18];
        [[maybe_unused]] real u2[18];   // UB2: the backward link is read before the forward hop is computed
        if (CF) {
            load_spinor(in, s, acc);
        } else {
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[i] = 0;
        }
        load_spinor(in, n.f[0], va);
        load_spinor(in, n.b[0], vb);

        // One direction: the stage of slot MU & 1 holds U_mu of the tile (+ its -mu face).  Warp 0 first enqueues the NEXT
        // stage (direction MU + 1 of this tile, or direction 0 of the CTA's next tile) into the other slot; then forward hop
        // with the thread's own slot, backward hop with the slot of the site behind it; the spinors of the next direction
        // are requested before the arithmetic of this one.
#define WD_TMA_DIRECTION(MU, ISSUE, BROW, BLANE8, NEXTF, NEXTB, SGF, SGB, XHALO)                               \
        {                                                                                                      \
            if (issuer) { ISSUE; }                                                                             \
            constexpr unsigned int so = ((MU) & 1) * S::STAGE;                                                 \
            mbar_wait(full + ((MU) & 1), (unsigned int)((MU) >> 1));                                           \
            load_link_row(own + so, lx8, u);                                                                   \
            if (UB2) {                                                                                         \
                if (XHALO) load_link<0>(U, n.b[0], u2);                                                        \
                else load_link_row((BROW) + so, BLANE8, u2);                                                   \
                __syncwarp();                                                                                  \
                if (lane == 0) mbar_arrive(empty + ((MU) & 1));                                                \
            }                                                                                                  \
            hop_compute<MU, SF, false, real>(va, u, SGF, acc);                                                 \
            if (NEXTF >= 0) load_spinor(in, NEXTF, va);                                                        \
            if (!UB2) {                                                                                        \
                if (XHALO) load_link<0>(U, n.b[0], u);                                                         \
                else load_link_row((BROW) + so, BLANE8, u);                                                    \
                __syncwarp();                                                                                  \
                if (lane == 0) mbar_arrive(empty + ((MU) & 1));                                                \
            }                                                                                                  \
            hop_compute<MU, -SF, true, real>(vb, UB2 ? u2 : u, SGB, acc);                                      \
            if (NEXTB >= 0) load_spinor(in, NEXTB, vb);                                                        \
        }
#define WD_TMA_ISSUE_SAME(MU) tma_issue<real, MU, BY, BZ, BT>(g, Ubytes, ring, full, empty, lane, x0, y0, z0, t0)
        WD_TMA_DIRECTION(0, WD_TMA_ISSUE_SAME(1), own - 16u, lx8 - 8, n.f[1], n.b[1], one, one, lx == 0)
        WD_TMA_DIRECTION(1, WD_TMA_ISSUE_SAME(2), rb1, lx8, n.f[2], n.b[2], one, one, false)
        WD_TMA_DIRECTION(2, WD_TMA_ISSUE_SAME(3), rb2, lx8, n.f[3], n.b[3], one, one, false)
        if (!CF) load_spinor(in, s, c);
        // the CTA's next tile: decoded here, once per tile, for the issuer now and for every thread in the next iteration
        const bool more = b + (int)gridDim.x < g.ntiles;
        if (more) tile_of_block(g, b + gridDim.x, tx, ty, tz, tt);
#define WD_TMA_ISSUE_NEXT_TILE \
        if (more) tma_issue<real, 0, BY, BZ, BT>(g, Ubytes, ring, full, empty, lane, tx * SB, ty * BY, tz * BZ, tt * BT)
        WD_TMA_DIRECTION(3, WD_TMA_ISSUE_NEXT_TILE, rb3, lx8, -1, -1, sgf, sgb, false)
#undef WD_TMA_ISSUE_NEXT_TILE
#undef WD_TMA_ISSUE_SAME
#undef WD_TMA_DIRECTION
        if (RU) load_spinor_rw(r, s, rv);
#pragma unroll
        for (int i = 0; i < 24; ++i) c[i] = CF ? acc[i] : fma(-kappa, acc[i], c[i]);  // (D in)(x) = in(x) - kappa * hops
        if (RU) {
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
    }
    if (MODE == MODE_QQ || RU) {
        double total;
        if (grid_sum<NT>(local, partials, counter, &total)) {
            if (MODE == MODE_QQ) finish_qq(sc, total);
            else finish_rr(sc, total, it, hist);
        }
    }
}

// ---------------------------------------------------------------- launch configurations of the staged kernel
//   T(index, BY, BZ, BT, MINB, UB2, F32, F64)        CTA tile = 16 x BY x BZ x BT, two stages; UB2 = two link buffers
// Measured on B200 (profiles/r2_ncu_link_staging.md; a2 / a3 per CG iteration inside the solve, links through L1 = 1.00):
//   row 0  fp32 16x2x2x2, 4 CTAs/SM, 128 registers              48^3x96: 1.18 / 1.35     32^4: 1.08 / 1.17
//   row 1  fp32 16x2x2x2, 3 CTAs/SM, 168 registers, 2 buffers   48^3x96: 1.07 / 1.12     32^4: 1.08 / 1.14
//   row 2  fp64 16x2x2x1, 4 CTAs/SM, 255 registers              32^4:    0.91 / 1.00     (the automatic choice for a2 in fp64)
// Retired after measurement: three-stage rings (modulo arithmetic per direction, 200 KB carve-out: 1.4-1.6), 16x4x2x2 and
// 16x4x4x2 tiles (1.2-1.7), 64-thread fp32 CTAs (1.08 / 1.24), two link buffers at 128 registers (spills: 1.6).
#define WD_TMA_TABLE(T)         \
    T(0, 2, 2, 2, 4, 0, 1, 0)   \
    T(1, 2, 2, 2, 3, 1, 1, 0)   \
    T(2, 2, 2, 1, 4, 0, 0, 1)
#define WD_NUM_TMA_ROWS 3
#define WD_TMA_AUTO_ROW_F64 2

struct TmaRowInfo {
    int b[4];
    int nstage, ahead, minb, f32, f64;
};
static const TmaRowInfo kTmaRows[WD_NUM_TMA_ROWS] = {
#define T(i, by, bz, bt, m, ub2, f32, f64) {{SB, by, bz, bt}, TMA_NSTAGE, 1 + ub2, m, f32, f64},
    WD_TMA_TABLE(T)
#undef T
};

struct TmaArgs {
    Geom g;            // tiled with {16, BY, BZ, BT} of the row
    int sm_count;
    cudaStream_t stream;
    const void *U, *in;
    void *out, *r;
    double kappa;
    CgScalars *sc;
    double *partials;
    unsigned int *counter;
    double *hist;
    int it;
};
cudaError_t launch_dslash_tma_f32(int row, int dagger, int mode, const TmaArgs &a);
cudaError_t launch_dslash_tma_f64(int row, int dagger, int mode, const TmaArgs &a);

template <typename real, int DAG, int MODE>
static cudaError_t launch_dslash_tma_row(int row, const TmaArgs &a)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    switch (row) {
#define T(i, by, bz, bt, m, ub2, f32, f64)                                                                     \
    case i:                                                                                                    \
        if constexpr (sizeof(real) == 4 ? f32 : f64) {                                                         \
            using S = TmaShape<real, by, bz, bt>;                                                              \
            auto kern = dslash_tma_kernel<real, DAG, MODE, by, bz, bt, m, ub2>;                                \
            static int occ_tab[WD_MAXDEV];                                                                     \
            static int attr_set[WD_MAXDEV];                                                                    \
            int dev = 0;                                                                                       \
            cudaError_t e = cudaGetDevice(&dev);                                                               \
            if (e != cudaSuccess) return e;                                                                    \
            if (dev < 0 || dev >= WD_MAXDEV) dev = WD_MAXDEV - 1;                                              \
            if (!attr_set[dev]) {                                                                              \
                e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM);          \
                if (e != cudaSuccess) return e;                                                                \
                /* shared-memory carve-out: what m resident CTAs need (+1 KB each), the rest stays L1 */       \
                int pct = (int)((m * (S::SMEM + 1024) * 100 + 228 * 1024 - 1) / (228 * 1024));                 \
                if (pct > 100) pct = 100;                                                                      \
                e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, pct);           \
                if (e != cudaSuccess) return e;                                                                \
                attr_set[dev] = 1;                                                                             \
            }                                                                                                  \
            int occ = 0;                                                                                       \
            e = cached_occupancy(occ_tab, kern, S::NT, S::SMEM, &occ);                                         \
            if (e != cudaSuccess) return e;                                                                    \
            long grid = (long)occ * a.sm_count;                                                                \
            if (grid > a.g.ntiles) grid = a.g.ntiles;                                                          \
            kern<<<(unsigned)grid, S::NT, S::SMEM, a.stream>>>(a.g, (const gvec *)a.U, (const svec *)a.in, (svec *)a.out, \
                                                              (real)a.kappa, (svec *)a.r, a.sc, a.partials, a.counter, \
                                                              a.hist, a.it);                                   \
            return cudaGetLastError();                                                                         \
        }                                                                                                      \
        return cudaErrorInvalidValue;
        WD_TMA_TABLE(T)
#undef T
        default: return cudaErrorInvalidValue;
    }
}
template <typename real>
static cudaError_t launch_dslash_tma_any(int row, int dagger, int mode, const TmaArgs &a)
{
    if (mode == MODE_PLAIN)
        return dagger ? launch_dslash_tma_row<real, 1, MODE_PLAIN>(row, a) : launch_dslash_tma_row<real, 0, MODE_PLAIN>(row, a);
    if (mode == MODE_QQ && dagger) return launch_dslash_tma_row<real, 1, MODE_QQ>(row, a);
    if (mode == MODE_RUPD && !dagger) return launch_dslash_tma_row<real, 0, MODE_RUPD>(row, a);
    return cudaErrorInvalidValue;
}

}  // namespace wd

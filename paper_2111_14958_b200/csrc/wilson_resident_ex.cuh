// wilson_resident_ex.cuh — the shared-memory-resident CG (wilson_resident.cuh) for the LARGER clusters: remote neighbours are
// read as HALF-SPINORS that their owner has already projected (and, for the backward hop, already multiplied by its link).
//
// In cg_resident_kernel a hop to a site of another CTA pulls the whole neighbour spinor (24 reals) and, for the backward hop,
// the neighbour's link (18 reals) through distributed shared memory: 96 + 168 B per direction.  At 8^4 (16 CTAs of 256 sites)
// that is 84 KB per CTA and stencil pass at the ~17 B per clock a CTA gets from its peers: the stencil phases take 4.1 us against
// 1.9 us for the same 256 sites per CTA with no remote neighbour (timestamps inside the kernel).  Here the OWNER
// of a site does the part of a remote hop that needs only its own data, right after it has produced the field, and leaves the
// 12-real result in an export buffer of its shared memory:
//     forward hop of a remote site x - mu:   h = (1 -+ gamma_mu) psi(x)                (the reader multiplies by its own U_mu(x - mu))
//     backward hop of a remote site x + mu:  g = U_mu(x)^dagger (1 +- gamma_mu) psi(x)  (the reader only reconstructs)
// The reader pulls 48 B per remote hop (fp32) instead of 96 / 168 B, and no link ever crosses CTAs.  The export buffers are
// PLANE-MAJOR (plane j of all slots, 16 B per slot): the threads of a warp, whose slots are consecutive, read whole 128-byte
// lines of the owner's shared memory (a slot-major buffer moved three times the useful bytes and gained nothing).  The
// arithmetic of a hop is the same project -> SU(3) multiply -> reconstruct in the same order, split between two threads:
// bit-identical results.  Which slot a reader has to pull is settled once, at start: every owner numbers its exports per
// direction (a block-wide scan) and writes the slot number into the reader's table through distributed shared memory.
// y lives in registers in fp32 and in the caller's psi buffer in fp64 (its slab makes room for the two export buffers).
#pragma once

namespace wd {

// a half-spinor (12 reals) in a plane-major export buffer of `nslots` slots: plane j of slot i at (j * nslots + i) * 16 bytes
template <typename real> struct RsHalf;
template <> struct RsHalf<float> {
    static constexpr int BYTES = 48;
    static __device__ __forceinline__ void load_remote(unsigned int base, unsigned int rank, int nslots, int slot, float h[12])
    {
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const float4 t = rs_ld4<true>(rs_map<true>(base + (unsigned int)(j * nslots + slot) * 16u, rank));
            h[4 * j] = t.x; h[4 * j + 1] = t.y; h[4 * j + 2] = t.z; h[4 * j + 3] = t.w;
        }
    }
    static __device__ __forceinline__ void store(unsigned char *base, int nslots, int slot, const float h[12])
    {
        float4 *q = reinterpret_cast<float4 *>(base);
#pragma unroll
        for (int j = 0; j < 3; ++j) q[j * nslots + slot] = make_float4(h[4 * j], h[4 * j + 1], h[4 * j + 2], h[4 * j + 3]);
    }
};
template <> struct RsHalf<double> {
    static constexpr int BYTES = 96;
    static __device__ __forceinline__ void load_remote(unsigned int base, unsigned int rank, int nslots, int slot, double h[12])
    {
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            const double2 t = rs_ldd<true>(rs_map<true>(base + (unsigned int)(j * nslots + slot) * 16u, rank));
            h[2 * j] = t.x; h[2 * j + 1] = t.y;
        }
    }
    static __device__ __forceinline__ void store(unsigned char *base, int nslots, int slot, const double h[12])
    {
        double2 *q = reinterpret_cast<double2 *>(base);
#pragma unroll
        for (int j = 0; j < 6; ++j) q[j * nslots + slot] = make_double2(h[2 * j], h[2 * j + 1]);
    }
};

__device__ __forceinline__ void rs_st_remote_u16(unsigned int a, unsigned short v)
{
    asm volatile("st.shared::cluster.u16 [%0], %1;" ::"r"(a), "h"(v) : "memory");
}

// dynamic shared memory: scratch, U, r, p, q, the two slot tables, the two export buffers
template <typename real> constexpr size_t resident_ex_smem(int spc, int nslots)
{
    return 1024 + (size_t)spc * (RsLayout<real>::SITE - 24 * sizeof(real)) + 2 * (size_t)8 * spc * 2 +
           2 * (size_t)nslots * RsHalf<real>::BYTES;
}

template <typename real>
__global__ void __launch_bounds__(256, 1)
cg_resident_ex_kernel(int L0, int L1, int L2, int L3, int bc_t, int spc_shift, int nslots,
                      const typename Field<real>::gvec *__restrict__ U, const typename Field<real>::svec *__restrict__ eta,
                      typename Field<real>::svec *psi, real kappa, CgScalars *sc, double *hist, double r_min, int max_iter)
{
    using LY = RsLayout<real>;
    using HB = RsHalf<real>;
    constexpr bool YREG = sizeof(real) == 4;      // fp32: y in registers; fp64: y in the psi buffer (own site only)
    extern __shared__ __align__(128) unsigned char rs_smem[];
    const int spc = 1 << spc_shift;
    const unsigned int mask = (unsigned int)spc - 1u;
    const int tid = threadIdx.x;                 // local site
    unsigned int rank, nc;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(nc));
    double *scratch = reinterpret_cast<double *>(rs_smem);          // [0..2] partials; [8..40] block_sum; [48..] scan counters
    unsigned char *Us = rs_smem + 1024;
    unsigned char *rsl = Us + (size_t)(spc >> SB_SHIFT) * LY::GPB;
    unsigned char *ps = rsl + (size_t)(spc >> SB_SHIFT) * LY::SPB;
    unsigned char *qs = ps + (size_t)(spc >> SB_SHIFT) * LY::SPB;
    unsigned short *rtab = reinterpret_cast<unsigned short *>(qs + (size_t)(spc >> SB_SHIFT) * LY::SPB);   // [hop][site]: slot to READ
    unsigned short *wtab = rtab + 8 * spc;                                                                  // [export][site]: slot to WRITE
    unsigned char *exA = reinterpret_cast<unsigned char *>(wtab + 8 * spc);
    unsigned char *exB = exA + (size_t)nslots * HB::BYTES;
    const unsigned int U32 = smem_u32_rs(Us), r32 = smem_u32_rs(rsl), p32 = smem_u32_rs(ps), q32 = smem_u32_rs(qs),
                       sc32 = smem_u32_rs(scratch), rtab32 = smem_u32_rs(rtab), exA32 = smem_u32_rs(exA), exB32 = smem_u32_rs(exB);

    const int s = (int)rank * spc + tid;         // global site
    int x, y, z, t;
    {
        int rem = s;
        x = rem % L0; rem /= L0;
        y = rem % L1; rem /= L1;
        z = rem % L2; t = rem / L2;
    }
    Geom g;
    g.L[0] = L0; g.L[1] = L1; g.L[2] = L2; g.L[3] = L3; g.par = 0;
    const Hops n = neighbours<0>(g, x, y, z, t, s);
    const real one = (real)1;
    const real sgf = (t == L3 - 1) ? (real)bc_t : one;
    const real sgb = (t == 0) ? (real)bc_t : one;
    // hop h = 2 mu (forward) / 2 mu + 1 (backward) of this site reaches another CTA
    unsigned int remote = 0;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        if ((unsigned int)(n.f[mu] >> spc_shift) != rank) remote |= 1u << (2 * mu);
        if ((unsigned int)(n.b[mu] >> spc_shift) != rank) remote |= 1u << (2 * mu + 1);
    }

    // ---- load the U slab
    {
        const uint4 *src = reinterpret_cast<const uint4 *>(reinterpret_cast<const unsigned char *>(U) + (size_t)((s - tid) >> SB_SHIFT) * LY::GPB);
        uint4 *dst = reinterpret_cast<uint4 *>(Us);
        const int nvec = (spc >> SB_SHIFT) * LY::GPB / 16;
        for (int i = tid; i < nvec; i += spc) dst[i] = __ldg(src + i);
    }
    for (int i = tid; i < 120; i += spc) scratch[i] = 0.0;
    __syncthreads();
    rs_sync<true>();                              // every CTA of the cluster is running before anyone writes into a peer

    // ---- export slots.  This site is read by the forward hop mu of x - mu (if that is another CTA's: the same condition as
    // "my backward hop is remote") and by the backward hop mu of x + mu ("my forward hop is remote").  Export e = 2 mu serves
    // the reader's forward hop, e = 2 mu + 1 its backward hop; slots are numbered per export class by a block-wide scan.
    {
        int *cnt = reinterpret_cast<int *>(scratch + 48);            // [8 classes][8 warps]
        const int lane = tid & 31, w = tid >> 5;
        unsigned int flags = 0;                                      // bit e: export e exists
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            if (remote & (1u << (2 * mu + 1))) flags |= 1u << (2 * mu);
            if (remote & (1u << (2 * mu))) flags |= 1u << (2 * mu + 1);
        }
        int wrank[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const unsigned int b = __ballot_sync(0xffffffffu, (flags >> e) & 1u);
            wrank[e] = __popc(b & ((1u << lane) - 1u));
            if (lane == 0) cnt[e * 8 + w] = __popc(b);
        }
        __syncthreads();
        int base = 0;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            int before = 0, total = 0;
            for (int ww = 0; ww < 8; ++ww) {
                const int c = cnt[e * 8 + ww];
                if (ww < w) before += c;
                total += c;
            }
            const int slot = base + before + wrank[e];
            base += total;
            wtab[e * spc + tid] = (unsigned short)slot;
            if ((flags >> e) & 1u) {
                const int mu = e >> 1;
                const int reader = (e & 1) ? n.f[mu] : n.b[mu];      // backward-hop reader sits at x + mu, forward-hop reader at x - mu
                rs_st_remote_u16(rs_map<true>(rtab32 + 2u * (unsigned int)(e * spc + (reader & (int)mask)),
                                              (unsigned int)(reader >> spc_shift)), (unsigned short)slot);
            }
        }
        if (base > nslots) __trap();                                  // the launcher sizes the buffers from the same geometry
    }

    // the exports of this site's spinor v for the pass with dagger flag DAG that will READ them, into buffer `ex`
    auto export_site = [&](auto dag_tag, const real v[24], unsigned char *ex) {
        constexpr int DAG = decltype(dag_tag)::value;
        constexpr int SF = DAG ? +1 : -1;
#define WD_RS_EXPORT(MU)                                                                                             \
        if (remote & (1u << (2 * MU + 1))) {          /* x - mu is remote: its forward hop needs (1 + SF gamma) psi(x) */ \
            real h[12];                                                                                              \
            project<MU, SF, real>(v, h);                                                                             \
            HB::store(ex, nslots, (int)wtab[(2 * MU) * spc + tid], h);                                               \
        }                                                                                                            \
        if (remote & (1u << (2 * MU))) {              /* x + mu is remote: its backward hop needs U^dagger (1 - SF gamma) psi(x) */ \
            real h[12], gg[12], u[18];                                                                               \
            project<MU, -SF, real>(v, h);                                                                            \
            rs_load_link<false, MU>(U32, tid, u);                                                                    \
            mul_su3<true, real>(u, h, gg);                                                                           \
            HB::store(ex, nslots, (int)wtab[(2 * MU + 1) * spc + tid], gg);                                          \
        }
        WD_RS_EXPORT(0)
        WD_RS_EXPORT(1)
        WD_RS_EXPORT(2)
        WD_RS_EXPORT(3)
#undef WD_RS_EXPORT
    };
    // the hopping sum of the field in slab `f32` (this CTA's copy) at this thread's site; remote neighbours from the owners' `ex32`
    auto hops = [&](auto dag_tag, unsigned int f32, unsigned int ex32, real acc[24]) {
        constexpr int DAG = decltype(dag_tag)::value;
        constexpr int SF = DAG ? +1 : -1;
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = 0;
#define WD_RS_HOP(MU, SGF, SGB)                                                                                      \
        {                                                                                                            \
            real v[24], u[18], h[12], gg[12];                                                                        \
            const int nf = n.f[MU], nb = n.b[MU];                                                                    \
            rs_load_link<false, MU>(U32, tid, u);                                                                    \
            if (remote & (1u << (2 * MU))) {                                                                         \
                HB::load_remote(ex32, (unsigned int)(nf >> spc_shift), nslots, (int)rtab[(2 * MU) * spc + tid], h);  \
            } else {                                                                                                 \
                rs_load_spinor<false>(f32 + rs_soff((real)0, nf & (int)mask), v);                                    \
                project<MU, SF, real>(v, h);                                                                         \
            }                                                                                                        \
            mul_su3<false, real>(u, h, gg);                                                                          \
            reconstruct<MU, SF, real>(gg, SGF, acc);                                                                 \
            if (remote & (1u << (2 * MU + 1))) {                                                                     \
                HB::load_remote(ex32, (unsigned int)(nb >> spc_shift), nslots, (int)rtab[(2 * MU + 1) * spc + tid], gg); \
            } else {                                                                                                 \
                rs_load_spinor<false>(f32 + rs_soff((real)0, nb & (int)mask), v);                                    \
                rs_load_link<false, MU>(U32, nb & (int)mask, u);                                                     \
                project<MU, -SF, real>(v, h);                                                                        \
                mul_su3<true, real>(u, h, gg);                                                                       \
            }                                                                                                        \
            reconstruct<MU, -SF, real>(gg, SGB, acc);                                                                \
        }
        WD_RS_HOP(0, one, one)
        WD_RS_HOP(1, one, one)
        WD_RS_HOP(2, one, one)
        WD_RS_HOP(3, sgf, sgb)
#undef WD_RS_HOP
    };
    using Dag0 = DagTag<0>;
    using Dag1 = DagTag<1>;
    auto cta_partial = [&](double v, int slot) {
        const double b = block_sum<256>(v, scratch + 8);
        if (tid == 0) scratch[slot] = b;
    };
    auto cluster_total = [&](int slot) -> double {
        const int lane = tid & 31;
        double v = 0.0;
        if (lane < (int)nc) v = rs_ld1d<true>(rs_map<true>(sc32 + 8 * slot, (unsigned int)lane));
        double tot = 0.0;
        for (int c = 0; c < (int)nc; ++c) tot += __shfl_sync(0xffffffffu, v, c);   // rank order, as in cg_resident_kernel
        return tot;
    };

    // ---- a1: y <- 0, r <- eta, p <- eta, rr = <eta,eta>; the exports of p for the first D-dagger pass
    real yv[YREG ? 24 : 1];
    double local = 0.0;
    {
        real e[24];
        load_spinor(eta, s, e);
        real n2 = 0;
#pragma unroll
        for (int i = 0; i < 24; ++i) n2 = fma(e[i], e[i], n2);
        rs_store_spinor(rsl, tid, e); rs_store_spinor(ps, tid, e);
        if constexpr (YREG) {
#pragma unroll
            for (int i = 0; i < 24; ++i) yv[i] = 0;
        } else {
            real zero[24];
#pragma unroll
            for (int i = 0; i < 24; ++i) zero[i] = 0;
            store_spinor(psi, s, zero);
        }
        export_site(Dag1{}, e, exA);
        local = (double)n2;
    }
    cta_partial(local, 0);
    rs_sync<true>();                              // also: every slot table is complete
    const double eta2 = cluster_total(0);
    double rr = eta2, alpha = 0.0, beta = 0.0;
    int k = 0;
    bool go = isfinite(eta2) && eta2 > 0.0 && loop_test(rr, eta2, r_min).go;
    if (rank == 0 && tid == 0 && hist) hist[0] = eta2;

    while (go && k < max_iter) {
        // a2: q = D-dagger p, qq; the exports of q for the D pass
        {
            real acc[24], c[24];
            hops(Dag1{}, p32, exA32, acc);
            rs_load_spinor<false>(p32 + rs_soff((real)0, tid), c);
            real n2 = 0;
#pragma unroll
            for (int i = 0; i < 24; ++i) { c[i] = fma(-kappa, acc[i], c[i]); n2 = fma(c[i], c[i], n2); }
            rs_store_spinor(qs, tid, c);
            export_site(Dag0{}, c, exB);
            cta_partial((double)n2, 1);
        }
        rs_sync<true>();
        const double qq = cluster_total(1);
        alpha = rr / qq;                                     // alpha <- |r|^2 / |D-dagger p|^2 (G1)
        const real al = (real)alpha;
        // a3: r <- r - alpha D q, rr'
        {
            real acc[24], c[24], rv[24];
            hops(Dag0{}, q32, exB32, acc);
            rs_load_spinor<false>(q32 + rs_soff((real)0, tid), c);
            rs_load_spinor<false>(r32 + rs_soff((real)0, tid), rv);
            real n2 = 0;
#pragma unroll
            for (int i = 0; i < 24; ++i) {
                c[i] = fma(-kappa, acc[i], c[i]);
                rv[i] = fma(-al, c[i], rv[i]);
                n2 = fma(rv[i], rv[i], n2);
            }
            rs_store_spinor(rsl, tid, rv);
            cta_partial((double)n2, 2);
        }
        rs_sync<true>();
        const double rr_new = cluster_total(2);
        beta = rr_new / rr;                                  // beta <- |r'|^2 / |r|^2
        const real be = (real)beta;
        // a4: y <- y + alpha p ; p <- r + beta p (own site); the exports of the new p
        {
            real pv[24], rv[24];
            rs_load_spinor<false>(p32 + rs_soff((real)0, tid), pv);
            rs_load_spinor<false>(r32 + rs_soff((real)0, tid), rv);
            if constexpr (YREG) {
#pragma unroll
                for (int i = 0; i < 24; ++i) yv[i] = fma(al, pv[i], yv[i]);
            } else {
                real yg[24];
                load_spinor_rw(psi, s, yg);
#pragma unroll
                for (int i = 0; i < 24; ++i) yg[i] = fma(al, pv[i], yg[i]);
                store_spinor(psi, s, yg);
            }
#pragma unroll
            for (int i = 0; i < 24; ++i) pv[i] = fma(be, pv[i], rv[i]);
            rs_store_spinor(ps, tid, pv);
            export_site(Dag1{}, pv, exA);
        }
        rr = rr_new;
        ++k;
        if (rank == 0 && tid == 0 && hist) hist[k] = rr;
        go = loop_test(rr, eta2, r_min).go;                  // while |r| >= r_min (G4)
        rs_sync<true>();                                     // p and its exports complete before they are read
    }
    // a6: psi = D-dagger y.  y goes into the r slab (r is dead) with its exports in buffer A (p is dead)
    {
        real c[24];
        if constexpr (YREG) {
#pragma unroll
            for (int i = 0; i < 24; ++i) c[i] = yv[i];
        } else {
            load_spinor_rw(psi, s, c);
        }
        rs_store_spinor(rsl, tid, c);
        export_site(Dag1{}, c, exA);
        rs_sync<true>();
        real acc[24];
        hops(Dag1{}, r32, exA32, acc);
#pragma unroll
        for (int i = 0; i < 24; ++i) c[i] = fma(-kappa, acc[i], c[i]);
        store_spinor(psi, s, c);
    }
    if (rank == 0 && tid == 0) {
        sc->rr = rr; sc->eta2 = eta2; sc->alpha = alpha; sc->beta = beta; sc->qq = 0.0; sc->r_min = r_min;
        sc->k = k; sc->k_stop = k; sc->max_iter = max_iter;
        sc->converged = (eta2 == 0.0 || loop_test(rr, eta2, r_min).converged) ? 1 : 0;
        sc->breakdown = (!go && !sc->converged) ? 1 : 0;
    }
    rs_sync<true>();                                         // no CTA leaves while its shared memory may still be read
}

}  // namespace wd

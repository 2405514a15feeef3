// wilson_resident.cuh — SURVEY.md 8(f1), second generation: the whole CG with the lattice RESIDENT IN SHARED MEMORY.
//
// The paper's experiments run at 4^4 ... 14^4 (Figs. 1-2 at 14^4).  At 4^4 the complete working
// set of the solve in fp32 -- U (73.7 KB) and the four CG vectors y, r, p, q (4 x 24.6 KB) -- is 172 KB: it fits the shared
// memory of ONE SM.  At 8^4 (3.1 MB) it fits the shared memory of a 16-CTA thread-block cluster, 256 sites per CTA.  The
// one-launch kernels of round 1 (cg_onelaunch_kernel, cg_split_kernel) keep the fields in L2 and separate the phases of an
// iteration by grid barriers: every operand is an L2 round trip away and every phase boundary costs a grid-wide barrier with
// its fences (10.7 / 10.0 us per iteration at 4^4 / 8^4).  Here
//   * a cluster of NC CTAs (NC = 1: a plain CTA) owns the lattice, CTA c the sites [c spc, (c+1) spc), one thread per site;
//   * U and y, r, p, q of those sites live in the CTA's shared memory for the whole solve, in the same site-blocked layout
//     as in global memory (16-site blocks, 128-bit planes: conflict-free 128-bit shared loads);
//   * a neighbour that belongs to another CTA is read from THAT CTA's shared memory (distributed shared memory: mapa +
//     ld.shared::cluster); nothing but eta (once), psi (once) and the final scalars touches global memory;
//   * the phases are separated by barrier.cluster (NC = 1: __syncthreads), and the per-CTA partial sums of the two
//     reductions are read by every warp of every CTA from the owners' shared memory and summed in rank order: alpha, beta and
//     the loop test are identical everywhere and run-to-run reproducible.
// Same recurrence, same precision rules as everywhere else (readings G1-G5, G17).
#pragma once
#include "wilson_split.cuh"   // DagTag

namespace wd {

__device__ __forceinline__ unsigned int smem_u32_rs(const void *p) { return (unsigned int)__cvta_generic_to_shared(p); }

template <bool CL> __device__ __forceinline__ unsigned int rs_map(unsigned int a, unsigned int rank)
{
    if (!CL) return a;
    unsigned int r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
// 128-bit / 64-bit loads from the shared window (CL: any CTA of the cluster, address from rs_map)
template <bool CL> __device__ __forceinline__ float4 rs_ld4(unsigned int a)
{
    float4 v;
    if (CL) asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a) : "memory");
    else asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a) : "memory");
    return v;
}
template <bool CL> __device__ __forceinline__ float2 rs_ld2(unsigned int a)
{
    float2 v;
    if (CL) asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a) : "memory");
    else asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a) : "memory");
    return v;
}
template <bool CL> __device__ __forceinline__ double2 rs_ldd(unsigned int a)
{
    double2 v;
    if (CL) asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a) : "memory");
    else asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a) : "memory");
    return v;
}
template <bool CL> __device__ __forceinline__ double rs_ld1d(unsigned int a)
{
    double v;
    if (CL) asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
    else asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
    return v;
}
template <bool CL> __device__ __forceinline__ void rs_sync()
{
    if (CL) {
        asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    } else {
        __syncthreads();
    }
}

// byte offsets inside a CTA's slab of a field (site-blocked layout of wilson_kernels.cuh, local site l)
template <typename real> struct RsLayout;
template <> struct RsLayout<float> {
    static constexpr int SPB = 6 * SB * 16;     // spinor block bytes (1536)
    static constexpr int GPB = 36 * SB * 8;     // gauge block bytes (4608)
    static constexpr int LB = 9 * SB * 8;       // one link direction of a block (1152)
    static constexpr int SITE = 72 * 4 + 4 * 24 * 4;   // U + y, r, p, q per site (672)
};
template <> struct RsLayout<double> {
    static constexpr int SPB = 12 * SB * 16;    // 3072
    static constexpr int GPB = 36 * SB * 16;    // 9216
    static constexpr int LB = 9 * SB * 16;      // 2304
    static constexpr int SITE = 72 * 8 + 4 * 24 * 8;   // 1344
};
__device__ __forceinline__ unsigned int rs_soff(float, int l) { return (unsigned int)((l >> SB_SHIFT) * RsLayout<float>::SPB + (l & (SB - 1)) * 16); }
__device__ __forceinline__ unsigned int rs_soff(double, int l) { return (unsigned int)((l >> SB_SHIFT) * RsLayout<double>::SPB + (l & (SB - 1)) * 16); }

template <bool CL> __device__ __forceinline__ void rs_load_spinor(unsigned int a, float v[24])
{
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const float4 t = rs_ld4<CL>(a + j * SB * 16);
        v[4 * j] = t.x; v[4 * j + 1] = t.y; v[4 * j + 2] = t.z; v[4 * j + 3] = t.w;
    }
}
template <bool CL> __device__ __forceinline__ void rs_load_spinor(unsigned int a, double v[24])
{
#pragma unroll
    for (int j = 0; j < 12; ++j) {
        const double2 t = rs_ldd<CL>(a + j * SB * 16);
        v[2 * j] = t.x; v[2 * j + 1] = t.y;
    }
}
__device__ __forceinline__ void rs_store_spinor(unsigned char *slab, int l, const float v[24])
{
    float4 *p = reinterpret_cast<float4 *>(slab + rs_soff(0.f, l));
#pragma unroll
    for (int j = 0; j < 6; ++j) p[j * SB] = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
}
__device__ __forceinline__ void rs_store_spinor(unsigned char *slab, int l, const double v[24])
{
    double2 *p = reinterpret_cast<double2 *>(slab + rs_soff(0.0, l));
#pragma unroll
    for (int j = 0; j < 12; ++j) p[j * SB] = make_double2(v[2 * j], v[2 * j + 1]);
}
// link mu of local site l of the slab whose (mapped) base address is ub
template <bool CL, int MU> __device__ __forceinline__ void rs_load_link(unsigned int ub, int l, float u[18])
{
    const unsigned int a = ub + (l >> SB_SHIFT) * RsLayout<float>::GPB + MU * RsLayout<float>::LB;
    const int lane = l & (SB - 1);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float4 t = rs_ld4<CL>(a + q * SB * 16 + lane * 16);
        u[4 * q] = t.x; u[4 * q + 1] = t.y; u[4 * q + 2] = t.z; u[4 * q + 3] = t.w;
    }
    const float2 t2 = rs_ld2<CL>(a + 4 * SB * 16 + lane * 8);
    u[16] = t2.x; u[17] = t2.y;
}
template <bool CL, int MU> __device__ __forceinline__ void rs_load_link(unsigned int ub, int l, double u[18])
{
    const unsigned int a = ub + (l >> SB_SHIFT) * RsLayout<double>::GPB + MU * RsLayout<double>::LB + (l & (SB - 1)) * 16;
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const double2 t = rs_ldd<CL>(a + k * SB * 16);
        u[2 * k] = t.x; u[2 * k + 1] = t.y;
    }
}

struct ResidentArgs {
    int L[4];
    int bc_t;
    int spc;           // sites per CTA (power of two, multiple of 32, <= 256)
    int nc;            // CTAs in the cluster (1, 2, 4, 8 or 16)
    cudaStream_t stream;
    const void *U, *eta;
    void *psi;
    double kappa;
    CgScalars *sc;
    double *hist;
    double r_min;
    int max_iter;
};
cudaError_t launch_cg_resident_f32(const ResidentArgs &a);
cudaError_t launch_cg_resident_f64(const ResidentArgs &a);
// dynamic shared memory of one CTA: the slabs, NC-independent scratch
template <typename real> constexpr size_t resident_smem(int spc) { return (size_t)spc * RsLayout<real>::SITE + 1024; }

template <typename real, bool CL>
__global__ void __launch_bounds__(256, 1)
cg_resident_kernel(int L0, int L1, int L2, int L3, int bc_t, int spc_shift, const typename Field<real>::gvec *__restrict__ U,
                   const typename Field<real>::svec *__restrict__ eta, typename Field<real>::svec *psi, real kappa,
                   CgScalars *sc, double *hist, double r_min, int max_iter)
{
    using LY = RsLayout<real>;
    extern __shared__ __align__(128) unsigned char rs_smem[];
    const int spc = 1 << spc_shift;
    const int tid = threadIdx.x;                 // local site
    unsigned int rank = 0, nc = 1;
    if (CL) {
        asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
        asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(nc));
    }
    // slabs: scratch (1 KB: 3 partial sums + the block-sum slots), U, y, r, p, q
    double *scratch = reinterpret_cast<double *>(rs_smem);          // [0..2]: this CTA's partials of eta2, qq, rr; [8..40]: block_sum
    unsigned char *Us = rs_smem + 1024;
    unsigned char *ys = Us + (size_t)(spc >> SB_SHIFT) * LY::GPB;
    unsigned char *rsl = ys + (size_t)(spc >> SB_SHIFT) * LY::SPB;
    unsigned char *ps = rsl + (size_t)(spc >> SB_SHIFT) * LY::SPB;
    unsigned char *qs = ps + (size_t)(spc >> SB_SHIFT) * LY::SPB;
    const unsigned int U32 = smem_u32_rs(Us), p32 = smem_u32_rs(ps), q32 = smem_u32_rs(qs), y32 = smem_u32_rs(ys),
                       sc32 = smem_u32_rs(scratch);

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

    // ---- load: U slab (the CTA's 16-site blocks are contiguous in the native layout), r = p = eta, y = 0
    {
        const uint4 *src = reinterpret_cast<const uint4 *>(reinterpret_cast<const unsigned char *>(U) + (size_t)((s - tid) >> SB_SHIFT) * LY::GPB);
        uint4 *dst = reinterpret_cast<uint4 *>(Us);
        const int nvec = (spc >> SB_SHIFT) * LY::GPB / 16;
        for (int i = tid; i < nvec; i += spc) dst[i] = __ldg(src + i);
    }
    if (tid < 48) scratch[tid] = 0.0;            // (block_sum reads one slot per possible warp; the CTA may have fewer)
    __syncthreads();
    double local = 0.0;
    {
        real e[24], zero[24];
        load_spinor(eta, s, e);
        real n2 = 0;
#pragma unroll
        for (int i = 0; i < 24; ++i) { zero[i] = 0; n2 = fma(e[i], e[i], n2); }
        rs_store_spinor(rsl, tid, e); rs_store_spinor(ps, tid, e); rs_store_spinor(ys, tid, zero);
        local = (double)n2;
    }
    // block sum in a fixed tree (threads = spc <= 256), result to scratch[slot]; every warp then sums the NC partials of the
    // cluster in rank order (lane c reads CTA c's slot through distributed shared memory)
    auto cta_partial = [&](double v, int slot) {
        const double b = block_sum<256>(v, scratch + 8);     // (block_sum only uses the warps that exist)
        if (tid == 0) scratch[slot] = b;
    };
    auto cluster_total = [&](int slot) -> double {
        const int lane = tid & 31;
        double v = 0.0;
        if (lane < (int)nc) v = rs_ld1d<CL>(rs_map<CL>(sc32 + 8 * slot, (unsigned int)lane));
        // rank order: serial sum over the lanes that hold a partial (nc <= 16)
        double tot = 0.0;
        for (int c = 0; c < (int)nc; ++c) tot += __shfl_sync(0xffffffffu, v, c);
        return tot;
    };
    cta_partial(local, 0);
    rs_sync<CL>();
    const double eta2 = cluster_total(0);
    double rr = eta2, alpha = 0.0, beta = 0.0;
    int k = 0;
    bool go = isfinite(eta2) && eta2 > 0.0 && loop_test(rr, eta2, r_min).go;
    if (rank == 0 && tid == 0 && hist) hist[0] = eta2;

    // the hopping sum of the field in slab `f32` (shared address of the slab in THIS CTA) at this thread's site
    auto hops = [&](auto dag_tag, unsigned int f32, real acc[24]) {
        constexpr int DAG = decltype(dag_tag)::value;
        constexpr int SF = DAG ? +1 : -1;
        const unsigned int mask = (unsigned int)spc - 1u;
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = 0;
        real v[24], u[18];
#define WD_RS_HOP(MU, SGF, SGB)                                                                                     \
        {                                                                                                            \
            const int nf = n.f[MU], nb = n.b[MU];                                                                    \
            rs_load_spinor<CL>(rs_map<CL>(f32 + rs_soff((real)0, nf & mask), (unsigned int)(nf >> spc_shift)), v);   \
            rs_load_link<false, MU>(U32, tid, u);                                                                    \
            hop_compute<MU, SF, false, real>(v, u, SGF, acc);                                                        \
            rs_load_spinor<CL>(rs_map<CL>(f32 + rs_soff((real)0, nb & mask), (unsigned int)(nb >> spc_shift)), v);   \
            rs_load_link<CL, MU>(rs_map<CL>(U32, (unsigned int)(nb >> spc_shift)), nb & mask, u);                    \
            hop_compute<MU, -SF, true, real>(v, u, SGB, acc);                                                        \
        }
        WD_RS_HOP(0, one, one)
        WD_RS_HOP(1, one, one)
        WD_RS_HOP(2, one, one)
        WD_RS_HOP(3, sgf, sgb)
#undef WD_RS_HOP
    };
    using Dag0 = DagTag<0>;
    using Dag1 = DagTag<1>;

    while (go && k < max_iter) {
        // a2: q = D-dagger p, qq
        {
            real acc[24], c[24];
            hops(Dag1{}, p32, acc);
            rs_load_spinor<false>(p32 + rs_soff((real)0, tid), c);
            real n2 = 0;
#pragma unroll
            for (int i = 0; i < 24; ++i) { c[i] = fma(-kappa, acc[i], c[i]); n2 = fma(c[i], c[i], n2); }
            rs_store_spinor(qs, tid, c);
            cta_partial((double)n2, 1);
        }
        rs_sync<CL>();
        const double qq = cluster_total(1);
        alpha = rr / qq;                                     // alpha <- |r|^2 / |D-dagger p|^2 (G1)
        const real al = (real)alpha;
        // a3: r <- r - alpha D q, rr'
        {
            real acc[24], c[24], rv[24];
            hops(Dag0{}, q32, acc);
            rs_load_spinor<false>(q32 + rs_soff((real)0, tid), c);
            rs_load_spinor<false>(smem_u32_rs(rsl) + rs_soff((real)0, tid), rv);
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
        rs_sync<CL>();
        const double rr_new = cluster_total(2);
        beta = rr_new / rr;                                  // beta <- |r'|^2 / |r|^2
        const real be = (real)beta;
        // a4: y <- y + alpha p ; p <- r + beta p (own site)
        {
            real yv[24], pv[24], rv[24];
            rs_load_spinor<false>(y32 + rs_soff((real)0, tid), yv);
            rs_load_spinor<false>(p32 + rs_soff((real)0, tid), pv);
            rs_load_spinor<false>(smem_u32_rs(rsl) + rs_soff((real)0, tid), rv);
#pragma unroll
            for (int i = 0; i < 24; ++i) { yv[i] = fma(al, pv[i], yv[i]); pv[i] = fma(be, pv[i], rv[i]); }
            rs_store_spinor(ys, tid, yv); rs_store_spinor(ps, tid, pv);
        }
        rr = rr_new;
        ++k;
        if (rank == 0 && tid == 0 && hist) hist[k] = rr;
        go = loop_test(rr, eta2, r_min).go;                  // while |r| >= r_min (G4)
        rs_sync<CL>();                                       // p (and y) complete before their neighbours are read
    }
    // a6: psi = D-dagger y, straight to global memory
    {
        real acc[24], c[24];
        hops(Dag1{}, y32, acc);
        rs_load_spinor<false>(y32 + rs_soff((real)0, tid), c);
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
    rs_sync<CL>();                                           // no CTA leaves while its shared memory may still be read
}

}  // namespace wd
#include "wilson_resident_ex.cuh"
namespace wd {

// Largest number of half-spinors a CTA has to export: over the sites of a slab, the hops that leave the slab (host, once per
// geometry: the slabs are ranges of consecutive sites).
static int resident_export_slots(const int L[4], int spc, int nc)
{
    thread_local int key[6] = {0, 0, 0, 0, 0, 0}, val = 0;
    if (key[0] == L[0] && key[1] == L[1] && key[2] == L[2] && key[3] == L[3] && key[4] == spc && key[5] == nc) return val;
    int worst = 0;
    const int stride[4] = {1, L[0], L[0] * L[1], L[0] * L[1] * L[2]};
    for (int r = 0; r < nc; ++r) {
        int count = 0;
        for (int l = 0; l < spc; ++l) {
            const int s = r * spc + l;
            int c[4], rem = s;
            for (int d = 0; d < 4; ++d) { c[d] = rem % L[d]; rem /= L[d]; }
            for (int d = 0; d < 4; ++d) {
                const int f = s + (c[d] == L[d] - 1 ? -(L[d] - 1) : 1) * stride[d];
                const int b = s + (c[d] == 0 ? (L[d] - 1) : -1) * stride[d];
                count += (f / spc != r) + (b / spc != r);
            }
        }
        if (count > worst) worst = count;
    }
    for (int d = 0; d < 4; ++d) key[d] = L[d];
    key[4] = spc; key[5] = nc; val = worst;
    return val;
}
constexpr size_t WD_RESIDENT_SMEM_MAX = 232448;   // 227 KB opt-in limit per CTA on sm_100

template <typename real>
static cudaError_t launch_cg_resident_any(const ResidentArgs &a)
{
    using svec = typename Field<real>::svec;
    using gvec = typename Field<real>::gvec;
    int shift = 0;
    while ((1 << shift) < a.spc) ++shift;
    if ((1 << shift) != a.spc || a.spc % 32 || a.spc > 256) return cudaErrorInvalidValue;
    const size_t smem = resident_smem<real>(a.spc);
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)a.nc);
    lc.blockDim = dim3((unsigned)a.spc);
    lc.dynamicSmemBytes = smem;
    lc.stream = a.stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)a.nc; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.attrs = at;
    const gvec *U = (const gvec *)a.U;
    const svec *eta = (const svec *)a.eta;
    svec *psi = (svec *)a.psi;
    const real kappa = (real)a.kappa;
    cudaError_t e;
    // Clusters of eight and sixteen CTAs: remote neighbours as half-spinors exported by their owners (wilson_resident_ex.cuh).
    // Measured, us per iteration, pulling whole spinors and links / exports: fp32 2048 sites (8 CTAs) 9.6-10.3 / 8.1-8.3, 4096
    // sites (16) 10.5-11.0 / 8.9-9.0; fp64 1024 sites (8) 9.9 / 9.8, 2048 sites (16) 11.5-12.4 / 10.1-10.2; smaller clusters have
    // too few remote hops to pay for the exports (4 CTAs 7.2 / 7.3, 2 CTAs 6.8 / 7.4; fp64 2 and 4 CTAs 7.6 / 8.8).
    {
        constexpr int min_nc = 8;
        const int nslots = a.nc >= min_nc ? resident_export_slots(a.L, a.spc, a.nc) : 0;
        const size_t ex_smem = resident_ex_smem<real>(a.spc, nslots);
        if (a.nc >= min_nc && nslots < 65536 && ex_smem <= WD_RESIDENT_SMEM_MAX) {
            auto kern = cg_resident_ex_kernel<real>;
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ex_smem);
            if (e != cudaSuccess) return e;
            if (a.nc > 8) {
                e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
                if (e != cudaSuccess) return e;
            }
            lc.dynamicSmemBytes = ex_smem;
            lc.numAttrs = 1;
            return cudaLaunchKernelEx(&lc, kern, a.L[0], a.L[1], a.L[2], a.L[3], a.bc_t, shift, nslots, U, eta, psi, kappa, a.sc,
                                      a.hist, a.r_min, a.max_iter);
        }
    }
    if (a.nc > 1) {
        auto kern = cg_resident_kernel<real, true>;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (a.nc > 8) {
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (e != cudaSuccess) return e;
        }
        lc.numAttrs = 1;
        return cudaLaunchKernelEx(&lc, kern, a.L[0], a.L[1], a.L[2], a.L[3], a.bc_t, shift, U, eta, psi, kappa, a.sc, a.hist,
                                  a.r_min, a.max_iter);
    }
    auto kern = cg_resident_kernel<real, false>;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    lc.numAttrs = 0;
    return cudaLaunchKernelEx(&lc, kern, a.L[0], a.L[1], a.L[2], a.L[3], a.bc_t, shift, U, eta, psi, kappa, a.sc, a.hist,
                              a.r_min, a.max_iter);
}

}  // namespace wd

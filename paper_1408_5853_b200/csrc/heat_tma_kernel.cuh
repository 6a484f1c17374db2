// heat_tma_kernel.cuh -- second-generation fused time-step kernel for sm_100a
// (same arithmetic contract as heat_line_kernel.cuh).
//
// What differs from heat_line_kernel.cuh (and from the paper's one-work-item-per-line kernel,
// P:L233):
//   * A z-line is viewed as a 2-D tensor [nr/16 rows][16 doubles]; thread t of the line owns
//     row t (nodes 16t .. 16t+15).  The three lines j-1, j, j+1 of the current level are
//     brought into shared memory by TMA (cp.async.bulk.tensor, SWIZZLE_128B), so HBM/L2 see
//     only fully coalesced 128-byte rows and each thread reads its own row with conflict-free
//     16-byte shared loads.
//   * The sweep coefficients (alpha, beta, gamma) of eq. (12) P:L133-136 are written IN PLACE
//     over the (T_{j-1}, T_j, T_{j+1}) slots they were computed from, so a CTA of 128 threads
//     needs 48 KB of shared memory and four CTAs are resident per SM, out of phase: while one
//     waits for its TMA loads or its cluster barrier the others keep the FP64 pipe busy.
//   * Lines longer than 2048 nodes are split over a thread-block cluster (2 or 4 CTAs); the
//     only cross-CTA step is one DSMEM exchange of 12 doubles per warp before the separator
//     solve.  Lines shorter than 2048 nodes are packed several per CTA.
//   * Chunks (16 nodes) that are regular nodes of one layer whose laws belong to a small set
//     of kinds run class-templated code with the geometry generated on the fly (uniform r
//     grid, rows scaled by i = r_i/h); every other chunk (r boundaries, interface nodes (18),
//     non-uniform grids, other laws, face_mode 1) runs a table-driven generic loop.
//   * The new level goes back with a TMA store; probes are read from the solved tile.
// "P:Lnnn" cites a line of the paper text; readings G1..G22 are listed in DESIGN.md.
#pragma once
#include <cuda.h>

#include "heat_line_kernel.cuh"

namespace heat {

// chunk classes (per 16-node chunk, host-built): 0 = generic, else (k kind, rho*c kind)
enum : uint32_t { CC_GENERIC = 0, CC_K0_C0 = 1, CC_K1_C3 = 2, CC_K2_C3 = 3, CC_K1_C2 = 4, CC_K15_C3 = 5 };

struct TParams {
    CUtensorMap tm_ld; // current level, box {16 doubles, 128 rows}
    CUtensorMap tm_st; // next level,    box {16 doubles, min(threads per line, 128) rows}
    KParams k;         // tables of the generic path (nrp == nr), scalars of this step
    const uint32_t *cdesc; // [batch][nr/16]: bits 0-7 chunk class, bits 8-15 layer
    double g0;         // 1/h^2 of the uniform r grid (fast classes only)
    int rpl;           // tensor rows per line = nr/16
    int slabs_per_member, total_slabs;
};

// ---------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap *tm, int c0, int c1, uint32_t src)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(tm), "r"(c0), "r"(c1), "r"(src) : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_all0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ uint32_t map_to_rank(uint32_t local, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_f64(uint32_t addr, double v)
{
    asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}

__device__ __forceinline__ double2 lds128(uint32_t a)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts128(uint32_t a, double x, double y)
{
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(x), "d"(y) : "memory");
}
__device__ __forceinline__ double lds64(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts64(uint32_t a, double x)
{
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(x) : "memory");
}

// byte offset of element e (0..15) of tensor row r inside a SWIZZLE_128B tile (1024-aligned)
__device__ __forceinline__ uint32_t sw_off(int r, int e)
{
    return (uint32_t)(r * 128 + ((((e >> 1) ^ (r & 7)) << 4) | ((e & 1) << 3)));
}

// ---------------------------------------------------------------- class-templated row math
// Law kinds of the fast classes: 0 = CONST, 1 = T^1, 2 = T^2, 3 = T^3, 15 = T^1.5.
// lambda at a half node is lambda_m((Ta+Tb)/2) = ckh * (Ta+Tb)^p (reading G3).

// reciprocal: MUFU.RCP64H seed + one cubic step (error e -> e^3) + one Newton step
__device__ __forceinline__ double rcp_fast(double x) { return rcp_nr(x); }

template <int KK>
__device__ __forceinline__ double face_coef(double kcf, double s)
{
    if (KK == 0) return kcf;
    if (KK == 1) return kcf * s;
    if (KK == 2) return kcf * (s * s);
    return kcf * (s * sqrt(s)); // KK == 15
}

template <int CK>
__device__ __forceinline__ double cap_coef(double ctf, double T, double T2)
{
    if (CK == 0) return ctf;
    if (CK == 2) return ctf * T2;
    return (ctf * T2) * T; // CK == 3
}

// fi * [Lambda_j[T] (11) P:L125 + X] without the fi: ezp*lam_{j+1/2}(Tu-T) - ezm*lam_{j-1/2}(T-Td) + qs,
// kzp = ezp*ckh, kzm = ezm*ckh.  For lambda ~ T the face product is ckh*(Tu^2 - T^2).
template <int KK>
__device__ __forceinline__ double zflux_src(double T, double T2, double Tu, double Td, double kzp, double kzm, double qs)
{
    double fU, fD;
    if (KK == 0) {
        fU = Tu - T; fD = T - Td;
    } else if (KK == 1) {
        fU = fma(Tu, Tu, -T2); fD = fma(-Td, Td, T2);
    } else if (KK == 2) {
        const double sU = T + Tu, sD = T + Td;
        fU = (sU * sU) * (Tu - T); fD = (sD * sD) * (T - Td);
    } else {
        const double sU = T + Tu, sD = T + Td;
        fU = (sU * sqrt(sU)) * (Tu - T); fD = (sD * sqrt(sD)) * (T - Td);
    }
    double r = fma(kzp, fU, qs);
    return fma(-kzm, fD, r);
}

struct SweepOut {
    double al, be, gm; // last row of the chunk: x_last = al*x_next + be + gm*u
    double P, Q, S;    // x_first = P*x_last + Q + S*u
};

// One regular row (13) P:L140-145 of a uniform r grid, scaled by i = r_i/h, pushed through
// the sweep (12) in its all-positive form: den = W + cfR + cfL*(1 - alpha_{i-1}).
#define HEAT_FAST_ROW(Tc_, Tr_, Td_, Tu_, AL_, BE_, GM_)                                          \
    {                                                                                             \
        const double kcf_ = fma(kc, fi, kch);                                                     \
        const double cfR_ = face_coef<KK>(kcf_, (Tc_) + (Tr_));                                   \
        const double T2_ = (Tc_) * (Tc_);                                                         \
        const double Wt_ = cap_coef<CK>(ct * fi, (Tc_), T2_);                                     \
        const double Lz_ = zflux_src<KK>((Tc_), T2_, (Tu_), (Td_), kzp, kzm, qs);                 \
        const double Ft_ = fma(Wt_, (Tc_), fi * Lz_);                                             \
        const double g_ = fma(cfL, om, Wt_);                                                      \
        const double inv_ = rcp_fast(g_ + cfR_);                                                  \
        const double tA_ = cfL * inv_;                                                            \
        AL_ = cfR_ * inv_;                                                                        \
        om = g_ * inv_;                                                                           \
        be = fma(tA_, be, Ft_ * inv_);                                                            \
        gm = tA_ * gm;                                                                            \
        BE_ = be;                                                                                 \
        GM_ = gm;                                                                                 \
        cfL = cfR_;                                                                               \
        fi += 1.0;                                                                                \
    }

// a0 = shared address of the thread's row in tile 0; tiles 1, 2 follow at +TILE bytes.
// On entry the tiles hold T_{j-1}, T_j, T_{j+1}; on exit alpha, beta, gamma of every row.
template <int KK, int CK, int TILE>
__device__ __forceinline__ SweepOut fast_chunk(uint32_t a0, int sw, const DLayer &L, double f0, double g0,
                                               double hl, double hr, double ezm, double ezp, double qa,
                                               double inv_tau)
{
    const double kc = ((KK == 0) ? L.k.ck : L.k.ckh) * g0;
    const double kch = 0.5 * kc;
    const double kz = (KK == 0) ? L.k.ck : L.k.ckh;
    const double kzp = ezp * kz, kzm = ezm * kz;
    const double ct = L.rc.ck * inv_tau;
    const double qs = L.heater ? qa * L.src.ck : 0.0;
    double om = 1.0, be = 0.0, gm = 1.0, P = 1.0, Q = 0.0, S = 0.0, al1 = 0.0;
    double fi = f0;
    double2 tl = lds128(a0 + TILE + ((0 ^ sw) << 4));
    double cfL = face_coef<KK>(fma(kc, f0, -kch), hl + tl.x); // face i0 - 1/2
#pragma unroll 2
    for (int c = 0; c < 8; ++c) {
        const uint32_t off = (uint32_t)((c ^ sw) << 4);
        double2 tn;
        if (c < 7) tn = lds128(a0 + TILE + (uint32_t)(((c + 1) ^ sw) << 4));
        else tn = make_double2(hr, hr);
        const double2 td = lds128(a0 + off);
        const double2 tu = lds128(a0 + 2 * TILE + off);
        double al0, be0, gm0, be1, gm1;
        HEAT_FAST_ROW(tl.x, tl.y, td.x, tu.x, al0, be0, gm0)
        Q = fma(P, be0, Q); S = fma(P, gm0, S); P = P * al0;
        HEAT_FAST_ROW(tl.y, tn.x, td.y, tu.y, al1, be1, gm1)
        if (c < 7) { Q = fma(P, be1, Q); S = fma(P, gm1, S); P = P * al1; }
        sts128(a0 + off, al0, al1);
        sts128(a0 + TILE + off, be0, be1);
        sts128(a0 + 2 * TILE + off, gm0, gm1);
        tl = tn;
    }
    SweepOut o;
    o.al = al1; o.be = be; o.gm = gm; o.P = P; o.Q = Q; o.S = S;
    return o;
}

// Table-driven chunk: any row kind (13)/(15)/(18), any law, non-uniform grid, face_mode 0/1.
// Same row arithmetic as heat_line_kernel.cuh (unscaled rows).
template <int TILE>
__device__ __noinline__ SweepOut generic_chunk(uint32_t a0, int row, const KParams &p, const DLayer *lay, int b,
                                               int i0, double hl, double hr, double ezm, double ezp, double qa)
{
    const double *ga = p.ga + (size_t)b * p.nrp + i0;
    const double *gc = p.gc + (size_t)b * p.nrp + i0;
    const uint32_t *info = p.info + (size_t)b * p.nrp + i0;
    const int fm = p.face_mode;
    const double inv_tau = p.inv_tau;
    double al = 0.0, be = 0.0, gm = 1.0, P = 1.0, Q = 0.0, S = 0.0;
    double Tprev = hl, T = lds64(a0 - row * 128 + TILE + sw_off(row, 0));
#pragma unroll 1
    for (int k = 0; k < 16; ++k) {
        const uint32_t o = a0 - row * 128 + sw_off(row, k);
        const double Tnext = (k < 15) ? lds64(a0 - row * 128 + TILE + sw_off(row, k + 1)) : hr;
        const double Tdn = lds64(o), Tup = lds64(o + 2 * TILE);
        const uint32_t nf = __ldg(info + k);
        const double gak = __ldg(ga + k), gck = __ldg(gc + k);
        const uint32_t kind = nf & 3u;
        double A, B, C, F;
        if (kind == NK_FIXED) {
            A = gak; B = 1.0; C = gck; F = p.fixF[(nf >> 2) & 3u];
        } else {
            const DLayer &mL = lay[(nf >> 8) & 0xffu];
            const DLayer &mR = lay[(nf >> 16) & 0xffu];
            const bool reg = (kind == NK_REG);
            const double lamL = law_face(mL.k, T, reg ? Tprev : T, fm);
            const double lamR = law_face(mR.k, T, reg ? Tnext : T, fm);
            A = -gak * lamL;
            C = -gck * lamR;
            if (reg) {
                const double W = law_at(mL.rc, T) * inv_tau;
                const double lamU = law_face(mL.k, T, Tup, fm);
                const double lamD = law_face(mL.k, T, Tdn, fm);
                double Lj = ezp * (lamU * (Tup - T));
                Lj = fma(-ezm, lamD * (T - Tdn), Lj);
                F = fma(W, T, Lj);
                if (mL.heater && qa != 0.0) F = fma(qa, law_at(mL.src, T), F);
                B = W - A - C;
            } else {
                B = -A - C; // (18) P:L178-181 at the new level (reading G7)
                F = 0.0;
            }
        }
        const double inv = rcp_nr(fma(A, al, B));
        const double tA = A * inv;
        al = -C * inv;
        be = fma(-tA, be, F * inv);
        gm = -tA * gm;
        sts64(o, al);
        sts64(o + TILE, be);
        sts64(o + 2 * TILE, gm);
        if (k < 15) { Q = fma(P, be, Q); S = fma(P, gm, S); P = P * al; }
        Tprev = T; T = Tnext;
    }
    SweepOut out;
    out.al = al; out.be = be; out.gm = gm; out.P = P; out.Q = Q; out.S = S;
    return out;
}

// ---------------------------------------------------------------- the kernel
// G  = threads of this CTA that work on one line (8..128); a CTA has 128 threads = 128 tensor
//      rows = LPB = 128/G consecutive lines ("slab") when CL == 1.
// CL = cluster size; CL > 1 needs G == 128 and the line has 128*CL threads, rank c owning
//      nodes [2048c, 2048c + 2048).
template <int G, int CL>
struct TmaCfg {
    static constexpr int NT = 128;
    static constexpr int LPB = NT / G;
    static constexpr int GL = G * CL;                      // threads per line
    static constexpr bool MULTI = (GL > 32);
    static constexpr int SEG = MULTI ? 32 : GL;            // shuffle segment width
    static constexpr int WG = MULTI ? GL / 32 : 1;         // warps (= separators) per line
    static constexpr int NSEP = MULTI ? (NT / 32) * CL : 1; // separators a CTA sees
    static constexpr int TILE = NT * 128;                  // bytes of one staged tile
    static constexpr int PUB = 12;                         // doubles published per warp
    static constexpr size_t smem_bytes(int nlayers)
    {
        return 1024 /* alignment slack */ + 3 * (size_t)TILE + sizeof(double) * (size_t)(2 * NSEP * PUB + NSEP + 2) +
               sizeof(DLayer) * (size_t)nlayers;
    }
};

template <int G, int CL>
__global__ void __launch_bounds__(128, 4) heat_tma_kernel(const __grid_constant__ TParams p)
{
    using Cfg = TmaCfg<G, CL>;
    constexpr int TILE = Cfg::TILE;
    constexpr int LPB = Cfg::LPB;
    constexpr int WG = Cfg::WG;
    constexpr int NSEP = Cfg::NSEP;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char *gbase = smem_raw + (sbase - smem_u32(smem_raw));
    double *pub = reinterpret_cast<double *>(gbase + 3 * TILE); // [2][NSEP][PUB]
    double *ysep = pub + 2 * NSEP * Cfg::PUB;                   // [NSEP]
    uint64_t *mbar = reinterpret_cast<uint64_t *>(ysep + NSEP);
    DLayer *lay = reinterpret_cast<DLayer *>(mbar + 2);
    const uint32_t mbar_a = smem_u32(mbar);
    const uint32_t pub_a = smem_u32(pub);

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const int crank = (CL > 1) ? (int)cluster_ctarank() : 0;
    const int lsl = tid / G;            // line within the slab
    const int t = crank * G + tid % G;  // thread within the line
    const int i0 = t * 16;
    const int wig = t >> 5;             // warp within the line
    const int gs = Cfg::MULTI ? ((CL > 1) ? wig : warp) : 0; // this warp's separator slot
    const int sw = tid & 7;
    const uint32_t a0 = sbase + (uint32_t)tid * 128u;

    for (int q = tid; q < p.k.nlayers * (int)(sizeof(DLayer) / sizeof(int)); q += Cfg::NT)
        reinterpret_cast<int *>(lay)[q] = reinterpret_cast<const int *>(p.k.layers)[q];
    if (tid == 0) {
        mbar_init(mbar_a, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (CL > 1) { cluster_arrive(); cluster_wait(); }

    const int nr = p.k.nr, nz = p.k.nz;
    const int cluster_id = blockIdx.x / CL, nclusters = gridDim.x / CL;
    uint32_t it = 0;
    for (int slab = cluster_id; slab < p.total_slabs; slab += nclusters, ++it) {
        const int b = slab / p.slabs_per_member;
        const int j0 = 1 + (slab - b * p.slabs_per_member) * LPB;
        const int j = j0 + lsl;
        const bool live = (j <= nz - 2);
        const int R0 = (b * nz + j0) * p.rpl + crank * ((CL > 1) ? G : 0); // tensor row of the slab
        // ---- stage lines j-1, j, j+1 (TMA, swizzled), one elected thread
        if (tid == 0) {
            tma_wait_read0(); // the previous store has finished reading the tiles
            mbar_expect_tx(mbar_a, 3u * (uint32_t)TILE);
            tma_load_2d(sbase, &p.tm_ld, 0, R0 - p.rpl, mbar_a);
            tma_load_2d(sbase + TILE, &p.tm_ld, 0, R0, mbar_a);
            tma_load_2d(sbase + 2 * TILE, &p.tm_ld, 0, R0 + p.rpl, mbar_a);
        }
        const uint32_t cd = __ldg(p.cdesc + (size_t)b * p.rpl + t);
        const double ezm = __ldg(p.k.ezm + (live ? j : 1)), ezp = __ldg(p.k.ezp + (live ? j : 1));
        const double qa = __ldg(p.k.Q0 + b) * p.k.amp; // Q0 nu(t_k) p^2(t_k), (2)-(4),(22)
        const size_t line = ((size_t)b * nz + (live ? j : 1)) * (size_t)nr;
        // halo across CTA / line ends comes from global memory (L2)
        double hl = 0.0, hr = 0.0;
        if (tid % G == 0 && t > 0) hl = __ldg(p.k.Told + line + i0 - 1);
        if (tid % G == G - 1 && t < Cfg::GL - 1) hr = __ldg(p.k.Told + line + i0 + 16);
        while (!mbar_try_wait(mbar_a, it & 1u)) {}
        if (tid % G != 0) hl = lds64(sbase + TILE + sw_off(tid - 1, 15));
        if (tid % G != G - 1) hr = lds64(sbase + TILE + sw_off(tid + 1, 0));
        __syncthreads(); // halos are read before anyone overwrites a T slot

        // ---- level 1: assemble (13)/(15)/(18) and sweep (12) the thread's 16 rows
        SweepOut o;
        const DLayer &L = lay[(cd >> 8) & 0xffu];
        const double f0 = (double)i0;
        switch (cd & 0xffu) {
        case CC_K0_C0: o = fast_chunk<0, 0, TILE>(a0, sw, L, f0, p.g0, hl, hr, ezm, ezp, qa, p.k.inv_tau); break;
        case CC_K1_C3: o = fast_chunk<1, 3, TILE>(a0, sw, L, f0, p.g0, hl, hr, ezm, ezp, qa, p.k.inv_tau); break;
        case CC_K2_C3: o = fast_chunk<2, 3, TILE>(a0, sw, L, f0, p.g0, hl, hr, ezm, ezp, qa, p.k.inv_tau); break;
        case CC_K1_C2: o = fast_chunk<1, 2, TILE>(a0, sw, L, f0, p.g0, hl, hr, ezm, ezp, qa, p.k.inv_tau); break;
        case CC_K15_C3: o = fast_chunk<15, 3, TILE>(a0, sw, L, f0, p.g0, hl, hr, ezm, ezp, qa, p.k.inv_tau); break;
        default: o = generic_chunk<TILE>(a0, tid, p.k, lay, b, i0, hl, hr, ezm, ezp, qa); break;
        }

        // ---- reduced row of this thread: a*y_{t-1} + y_t + c*y_{t+1} = d  (y = x of the last row)
        double Pn = __shfl_down_sync(0xffffffffu, o.P, 1, Cfg::SEG);
        double Qn = __shfl_down_sync(0xffffffffu, o.Q, 1, Cfg::SEG);
        double Sn = __shfl_down_sync(0xffffffffu, o.S, 1, Cfg::SEG);
        const bool seg_last = Cfg::MULTI ? (lane == 31) : (t == Cfg::GL - 1);
        if (seg_last) { Pn = 0.0; Qn = 0.0; Sn = 0.0; }
        Row3 row;
        {
            const double r = rcp_nr(fma(-o.al, Sn, 1.0));
            row.a = -o.gm * r;
            row.c = -o.al * Pn * r;
            row.d = fma(o.al, Qn, o.be) * r;
        }
        double y, u;
        if (!Cfg::MULTI) {
            row = pcr_segment<Cfg::SEG>(row, t, 0, Cfg::GL - 1);
            y = row.d;
            u = __shfl_up_sync(0xffffffffu, y, 1, Cfg::SEG);
            if (t == 0) u = 0.0;
        } else {
            // ---- level 2: PCR over lanes 0..30; lane 31 is the warp's separator
            const Row3 rp = pcr_segment<32>(row, lane, 0, 30);
            Row3 r30;
            r30.a = __shfl_sync(0xffffffffu, rp.a, 30);
            r30.c = __shfl_sync(0xffffffffu, rp.c, 30);
            r30.d = __shfl_sync(0xffffffffu, rp.d, 30);
            // publish what any CTA of the cluster needs to build this warp's separator row
            const uint32_t slot = pub_a + (uint32_t)(((it & 1u) * NSEP + gs) * Cfg::PUB) * 8u;
            if (lane == 0 || lane == 31) {
                const uint32_t s6 = slot + (lane == 31 ? 48u : 0u);
                const double v0 = lane == 31 ? o.al : o.P, v1 = lane == 31 ? o.be : o.Q, v2 = lane == 31 ? o.gm : o.S;
                const double v3 = lane == 31 ? r30.a : rp.a, v4 = lane == 31 ? r30.c : rp.c, v5 = lane == 31 ? r30.d : rp.d;
                if (CL > 1) {
#pragma unroll
                    for (int rk = 0; rk < CL; ++rk) {
                        const uint32_t ra = map_to_rank(s6, (uint32_t)rk);
                        st_cluster_f64(ra, v0); st_cluster_f64(ra + 8, v1); st_cluster_f64(ra + 16, v2);
                        st_cluster_f64(ra + 24, v3); st_cluster_f64(ra + 32, v4); st_cluster_f64(ra + 40, v5);
                    }
                } else {
                    sts64(s6, v0); sts64(s6 + 8, v1); sts64(s6 + 16, v2);
                    sts64(s6 + 24, v3); sts64(s6 + 32, v4); sts64(s6 + 40, v5);
                }
            }
            if (CL > 1) { cluster_arrive(); cluster_wait(); } else __syncthreads();
            // ---- level 3: warp 0 builds every separator row and solves them (PCR per line)
            if (warp == 0) {
                const bool in3 = lane < NSEP;
                const int s = in3 ? lane : 0;
                const double *D = pub + ((it & 1u) * NSEP + s) * Cfg::PUB;
                const bool has_next = ((s % WG) + 1 < WG);
                const double *Dn = D + (has_next ? Cfg::PUB : 0);
                const double al = D[6], be = D[7], gm = D[8];
                Row3 l30; l30.a = D[9]; l30.c = D[10]; l30.d = D[11];
                Row3 nx; nx.a = nx.c = nx.d = 0.0;
                double Pw = 0.0, Qw = 0.0, Sw = 0.0;
                if (has_next) { Pw = Dn[0]; Qw = Dn[1]; Sw = Dn[2]; nx.a = Dn[3]; nx.c = Dn[4]; nx.d = Dn[5]; }
                Row3 me;
                const double r = rcp_nr(fma(-al, Sw, 1.0));
                me.a = -gm * r;
                me.c = -al * Pw * r;
                me.d = fma(al, Qw, be) * r;
                Row3 s3 = pcr_combine(me, l30, true, nx, has_next);
                s3 = pcr_segment<(WG > 1 ? WG : 2)>(s3, s % WG, 0, WG - 1);
                if (in3) ysep[s] = s3.d;
            }
            __syncthreads();
            const double Vs = ysep[gs];
            const double U = (wig > 0) ? ysep[gs - 1] : 0.0;
            y = (lane == 31) ? Vs : fma(-rp.c, Vs, fma(-rp.a, U, rp.d));
            u = __shfl_up_sync(0xffffffffu, y, 1);
            if (lane == 0) u = U;
        }

        // ---- back substitution (14) P:L150; the new level replaces tile 0 in place
        {
            double xn = y;
#pragma unroll 2
            for (int c = 7; c >= 0; --c) {
                const uint32_t off = (uint32_t)((c ^ sw) << 4);
                const double2 va = lds128(a0 + off);
                const double2 vb = lds128(a0 + TILE + off);
                const double2 vg = lds128(a0 + 2 * TILE + off);
                const double x1 = (c == 7) ? y : fma(va.y, xn, fma(vg.y, u, vb.y));
                const double x0 = fma(va.x, x1, fma(vg.x, u, vb.x));
                sts128(a0 + off, x0, x1);
                xn = x0;
            }
        }
        // ---- probes: T of the new level at (i_p, j_p)
        if (p.k.probe_out != nullptr && live) {
            for (int q = 0; q < p.k.nprobes; ++q) {
                const ProbeSrc ps = p.k.probes[q];
                if (ps.i < i0 || ps.i >= i0 + 16) continue;
                if (ps.is_static) {
                    if (j == 1) p.k.probe_out[b * p.k.nprobes + q] = p.k.Told[((size_t)b * nz + ps.j_store) * nr + ps.i];
                } else if (ps.j_src == j) {
                    p.k.probe_out[b * p.k.nprobes + q] = lds64(sbase + sw_off(tid, ps.i - i0));
                }
            }
        }
        fence_proxy_async();
        __syncthreads();
        // ---- store T^ (and the Neumann z lines, which copy their neighbour; reading G16)
        if (tid == 0) {
#pragma unroll
            for (int l = 0; l < LPB; ++l) {
                const int jl = j0 + l;
                if (jl > nz - 2) break;
                const int Rl = R0 + l * p.rpl;
                const uint32_t src = sbase + (uint32_t)(l * G) * 128u;
                tma_store_2d(&p.tm_st, 0, Rl, src);
                if (jl == 1 && p.k.z_lo_neumann) tma_store_2d(&p.tm_st, 0, Rl - p.rpl, src);
                if (jl == nz - 2 && p.k.z_hi_neumann) tma_store_2d(&p.tm_st, 0, Rl + p.rpl, src);
            }
            tma_commit();
        }
    }
    if (tid == 0) tma_wait_all0();
    if (CL > 1) { cluster_arrive(); cluster_wait(); }
}

} // namespace heat

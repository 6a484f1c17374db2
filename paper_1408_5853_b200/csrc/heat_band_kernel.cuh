// heat_band_kernel.cuh -- third-generation fused time-step kernel for sm_100a ("band kernel")
// (same arithmetic contract as heat_line_kernel.cuh).
//
// What differs from heat_tma_kernel.cuh (v2) and from the paper's one-work-item-per-line
// kernel:
//   * A CTA group owns a BAND of consecutive z-lines and walks it line by line.  Each line of the
//     current level is brought into shared memory exactly once (TMA, SWIZZLE_128B, prefetched two
//     lines ahead through a ring of four slots), so L2 -> SM traffic is 8 B per cell instead of 24.
//   * The explicit axial face flux lambda_{i,j+1/2} (T_{i,j+1} - T_{i,j}) of eq. (11) P:L125 is
//     computed once per face: line j computes its upper flux, keeps it in a thread-private shared
//     slot, and line j+1 reuses it (with the opposite sign) as its lower flux.
//   * A thread owns 8 consecutive nodes; the sweep coefficients (alpha, beta, gamma) of eq. (12)
//     P:L133-136 stay in REGISTERS between the forward sweep and the back substitution (14).
//   * The row arithmetic is branch free across materials: every property law is a polynomial
//     (optionally times a square root) whose coefficients live in per-thread registers, loaded
//     once per band, so warps that span two layers do not serialise.  r-boundary rows (15) are
//     selects at fixed positions; only the thread that holds an interface node (18) takes a short
//     fix-up branch.
//   * The reduced system (one row per thread) is solved as in v2: shuffle PCR inside a warp,
//     one separator row per warp, separators exchanged through (distributed) shared memory and
//     solved by PCR in one warp.  Lines longer than 2048 nodes span a cluster of 2 or 4 CTAs.
// The kernel covers uniform r grids starting at r = 0 with nr in {512,1024,2048,4096,8192},
// laws CONST / POWER(p in {0,.5,1,1.5,2,3}) / POLY, lambda at the mean temperature (face_mode 0)
// and a temperature-independent source shape; heat_create picks v2 / v1 for everything else.
// "P:Lnnn" cites a line of the paper text; readings G1..G22 are listed in DESIGN.md.
#pragma once
#include <cuda.h>

#include "heat_band_params.cuh"
#include "heat_tma_kernel.cuh"

namespace heat {

__device__ __forceinline__ void bulk_load_16(uint32_t dst, const void *src, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 16, [%2];"
                 ::"r"(dst), "l"(src), "r"(bar) : "memory");
}
__device__ __forceinline__ double2 ld_cluster_v2(uint32_t a)
{
    double2 v;
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
// 16-byte store into the shared memory of a CTA of the cluster, completing on that CTA's mbarrier
__device__ __forceinline__ void st_async_v2(uint32_t remote_addr, double x, double y, uint32_t remote_bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];"
                 ::"r"(remote_addr), "d"(x), "d"(y), "r"(remote_bar) : "memory");
}
__device__ __forceinline__ void tma_wait_read1() { asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory"); }

// square root for lambda ~ T^(p+1/2): MUFU.RSQ64H seed y (>= 20 bits) + one cubic step on
// sqrt s = s y (1 - h)^(-1/2), h = 1 - s y^2:  g = t + t h (1/2 + 3/8 h), t = s y; the truncation
// error is 5/16 h^3 < 2^-61, so the result is within rounding of the exact root; s > 0 here
__device__ __forceinline__ double sqrt_pos(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    const double t = s * y;
    const double h = fma(-t, y, 1.0);
    const double q = h * fma(0.375, h, 0.5);
    return fma(t, q, t);
}

template <int DEGK>
struct BCoef {
    double K[DEGK + 1];
    double C[4]; // times 1/tau
    double qs;   // Q0 nu p^2 s  (2)-(4),(22); 0 outside the heater
    bool sq;
};

template <int DEGK>
__device__ __forceinline__ BCoef<DEGK> load_coef(const PLayer &L, double inv_tau, double qa)
{
    BCoef<DEGK> c;
#pragma unroll
    for (int n = 0; n <= DEGK; ++n) c.K[n] = L.K[n];
#pragma unroll
    for (int n = 0; n < 4; ++n) c.C[n] = L.C[n] * inv_tau;
    c.qs = L.heater ? qa * L.src : 0.0;
    c.sq = (L.sqrtk != 0);
    return c;
}

// lambda at a face from s = Ta + Tb; anysq is warp-uniform
template <int DEGK>
__device__ __forceinline__ double lam_eval(const BCoef<DEGK> &c, bool anysq, double s)
{
    double v = c.K[DEGK];
#pragma unroll
    for (int n = DEGK - 1; n >= 0; --n) v = fma(v, s, c.K[n]);
    if (anysq) {
        const double r = sqrt_pos(s);
        v = c.sq ? v * r : v;
    }
    return v;
}

template <int DEGK>
__device__ __forceinline__ double cap_eval(const BCoef<DEGK> &c, double T)
{
    double v = c.C[3];
    v = fma(v, T, c.C[2]);
    v = fma(v, T, c.C[1]);
    v = fma(v, T, c.C[0]);
    return v;
}

// One row pushed through the sweep (12) P:L133-136 in its all-positive form.  The row is
//   -a x_{i-1} + (a + c + w) x_i - c x_{i+1} = f,      a, c, w >= 0,
// a = cfL, c = cfR, and with om = 1 - alpha_{i-1}:  den = w + c + a om,  alpha_i = c / den,
// 1 - alpha_i = (w + a om) / den,  beta_i = (f + a beta_{i-1}) / den,  gamma_i = a gamma_{i-1} / den.
struct SweepState {
    double cfL, om, be, gm;
};

__device__ __forceinline__ void sweep_row(SweepState &s, double cfR, double w, double f, double &al)
{
    const double g = fma(s.cfL, s.om, w);
    const double inv = rcp_cubic(g + cfR);
    const double tA = s.cfL * inv;
    al = cfR * inv;
    s.om = g * inv;
    s.be = fma(tA, s.be, f * inv);
    s.gm = tA * s.gm;
    s.cfL = cfR;
}

// A regular row (13) P:L140-145 of the uniform r grid, scaled by i = r_i / h:
//   cfR = (i + 1/2) g0 lambda_{i+1/2,j},  w = i rho c / tau,  f = w T + i (Lambda_j[T] + X),
// Lambda_j[T] (11) P:L125 = ezp fU - ezm fD with the face fluxes fU, fD = lambda (T' - T).
template <int DEGK>
__device__ __forceinline__ void regular_row(const BCoef<DEGK> &c, bool anysq, double T, double Tr, double Tu, double fD,
                                            double fi, double g0, double ezp, double ezm, double &cfR, double &w,
                                            double &f, double &fU)
{
    cfR = lam_eval<DEGK>(c, anysq, T + Tr) * fma(g0, fi, 0.5 * g0);
    w = cap_eval<DEGK>(c, T) * fi;
    fU = lam_eval<DEGK>(c, anysq, T + Tu) * (Tu - T);
    double lz = fma(ezp, fU, c.qs);
    lz = fma(-ezm, fD, lz);
    f = fma(w, T, fi * lz);
}

// Arguments of the 8-row sweep of one thread (all in registers after inlining).
template <int DEGK>
struct SweepArgs {
    uint32_t sc, su, fr, fw; // shared addresses: line j, line j+1, lower flux (read), upper flux (write)
    double hl, hr;           // r neighbours of the chunk at line j
    double fi0, g0, ezp, ezm, inv_tau, qa;
    uint32_t cd;
    int ks;
    bool first, last;
    double rin_om, rin_be, rout_a, rout_w, rout_f;
    const PLayer *lay;
};

// Level 1 for one thread: rows (13) P:L140-145 assembled and pushed through the sweep (12); with
// SP also the interface row (18)-(20) P:L176-192 at row ks (the chunk's laws switch to layer B
// there) and the r-boundary rows (15)-(17) P:L158-174 at rows 0 / 7 of the first / last chunk.
template <int DEGK, bool SQ, bool SP>
__device__ __forceinline__ void sweep8(const SweepArgs<DEGK> &A, const uint32_t (&co)[4], BCoef<DEGK> &cA,
                                       double (&al)[8], double (&be)[8], double (&gm)[8])
{
    if (SP && A.ks >= 0) cA = load_coef<DEGK>(A.lay[A.cd & 0xffu], A.inv_tau, A.qa);
    SweepState st;
    st.om = 1.0; st.be = 0.0; st.gm = 1.0;
    double2 tl = lds128(A.sc + co[0]);
    st.cfL = lam_eval<DEGK>(cA, SQ, A.hl + tl.x) * fma(A.g0, A.fi0, -0.5 * A.g0); // face i0 - 1/2
#pragma unroll
    for (int qq = 0; qq < 4; ++qq) {
        double2 tn;
        if (qq < 3) tn = lds128(A.sc + co[qq < 3 ? qq + 1 : 3]);
        else tn = make_double2(A.hr, A.hr);
        const double2 tu = lds128(A.su + co[qq]);
        const double2 fd = lds128(A.fr + co[qq]);
        double fu[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int k = 2 * qq + e;
            const double T = e ? tl.y : tl.x;
            // interface node: lam*_A, lam*_B at T_{i*,j}; from here on the chunk is layer B
            const bool isif = SP && (k == A.ks);
            double lamA = 0.0;
            if (SP && isif) {
                lamA = lam_eval<DEGK>(cA, true, T + T);
                cA = load_coef<DEGK>(A.lay[(A.cd >> 8) & 0xffu], A.inv_tau, A.qa);
            }
            double cfR, w, f;
            regular_row<DEGK>(cA, SQ, T, e ? tn.x : tl.y, e ? tu.y : tu.x, e ? fd.y : fd.x,
                              A.fi0 + (double)k, A.g0, A.ezp, A.ezm, cfR, w, f, fu[e]);
            const double cfNext = cfR; // face i + 1/2 as the next regular row sees it
            if (SP && isif) {
                // (18) times h: -lam_A x_{i-1} + (lam_A + lam_B) x_i - lam_B x_{i+1} = 0 (new level, G7)
                st.cfL = lamA;
                cfR = lam_eval<DEGK>(cA, true, T + T);
                w = 0.0; f = 0.0;
            }
            if (SP && k == 7) { // r_out boundary row (15),(17) P:L158-174
                st.cfL = A.last ? A.rout_a : st.cfL;
                cfR = A.last ? 0.0 : cfR;
                w = A.last ? A.rout_w : w;
                f = A.last ? A.rout_f : f;
            }
            sweep_row(st, cfR, w, f, al[k]);
            if (SP && isif) st.cfL = cfNext;
            if (SP && k == 0) { // r_in boundary row (15),(16) P:L158-169
                al[0] = A.first ? 1.0 - A.rin_om : al[0];
                st.om = A.first ? A.rin_om : st.om;
                st.be = A.first ? A.rin_be : st.be;
                st.gm = A.first ? 0.0 : st.gm;
            }
            be[k] = st.be; gm[k] = st.gm;
        }
        sts128(A.fw + co[qq], fu[0], fu[1]);
        tl = tn;
    }
}

// PCR over lanes 0..30 of a warp; lane 31 (the separator) runs along and produces values nobody
// reads.  On exit row i reads a_i*U + x_i + c_i*V = d_i (U left of lane 0, V = lane 31's unknown).
__device__ __forceinline__ Row3 pcr_lanes_0_30(Row3 row, int lane)
{
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
        Row3 L, R;
        L.a = __shfl_up_sync(0xffffffffu, row.a, s);
        L.c = __shfl_up_sync(0xffffffffu, row.c, s);
        L.d = __shfl_up_sync(0xffffffffu, row.d, s);
        R.a = __shfl_down_sync(0xffffffffu, row.a, s);
        R.c = __shfl_down_sync(0xffffffffu, row.c, s);
        R.d = __shfl_down_sync(0xffffffffu, row.d, s);
        row = pcr_combine(row, L, lane >= s, R, lane + s <= 30);
    }
    return row;
}

// NT = threads per CTA (128 or 256).  G = threads of this CTA that work on one line (64 .. NT).
// CL = cluster size; CL > 1 needs G == NT: the line has NT*CL threads, rank c owns nodes
//      [8 NT c, 8 NT (c + 1)).
// DEGK = degree of the lambda polynomials.
template <int G, int CL, int DEGK, int NT>
__global__ void __launch_bounds__(NT, 512 / NT) heat_band_kernel(const __grid_constant__ BParams p)
{
    using Cfg = BandCfg<G, CL, NT>;
    constexpr int SLOT = Cfg::SLOT;
    constexpr uint32_t NSLOT = Cfg::NSLOT;
    constexpr int LPB = Cfg::LPB;
    constexpr int WG = Cfg::WG;
    constexpr int NSEP = Cfg::NSEP;
    constexpr uint32_t FULL = 0xffffffffu;
    static_assert(CL == 1 || G == NT, "a cluster line needs whole CTAs");
    constexpr int NW = NT / 32;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char *gbase = smem_raw + (sbase - smem_u32(smem_raw));
    double *pub = reinterpret_cast<double *>(gbase + Cfg::OFF_PUB);   // [2][NSEP][PUB]
    double *ysep = reinterpret_cast<double *>(gbase + Cfg::OFF_YSEP); // [NSEP]
    PLayer *lay = reinterpret_cast<PLayer *>(gbase + Cfg::OFF_LAY);
    const uint32_t mbar_a = sbase + Cfg::OFF_MBAR;
    const uint32_t pub_a = sbase + Cfg::OFF_PUB;
    const uint32_t halo_a = sbase + Cfg::OFF_HALO;

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    // rank of this CTA within the line: the hardware rank, rotated by p.rank_rot in odd clusters so
    // that CTAs sharing an SM need not hold the same (possibly most expensive) part of the radius
    const int crank = (CL > 1) ? (int)((cluster_ctarank() + (uint32_t)(((blockIdx.x / CL) & 1) ? p.rank_rot : 0)) % (uint32_t)CL) : 0;
    const int grp = tid / G;            // group (line) within the CTA
    const int tg = tid % G;             // thread within the CTA's part of the line
    const int t = crank * G + tg;       // thread within the line
    const int i0 = t * 8;
    const int wig = t >> 5;             // warp within the line
    const int gs = crank * NW + warp;    // this warp's separator slot
    const int trow = tid >> 1, half = tid & 1, sw = trow & 7;
    // byte offsets inside a slot: own 16-byte chunks q = 0..3, and the two r neighbours
    const uint32_t rowo = (uint32_t)trow * 128u;
    uint32_t co[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) co[q] = rowo + (uint32_t)((((half << 2) | q) ^ sw) << 4);
    const uint32_t hlo = half ? (rowo + (uint32_t)((3 ^ sw) << 4) + 8u)
                              : (rowo - 128u + (uint32_t)((7 ^ ((trow - 1) & 7)) << 4) + 8u);
    const uint32_t hro = half ? (rowo + 128u + (uint32_t)((0 ^ ((trow + 1) & 7)) << 4))
                              : (rowo + (uint32_t)((4 ^ sw) << 4));
    const bool edgeL = (tg == 0), edgeR = (tg == G - 1);

    for (int q = tid; q < p.nlayers * (int)(sizeof(PLayer) / sizeof(int)); q += Cfg::NT)
        reinterpret_cast<int *>(lay)[q] = reinterpret_cast<const int *>(p.players)[q];
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < Cfg::NSLOT + 2; ++s) mbar_init(mbar_a + 8u * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (CL > 1) { cluster_arrive(); cluster_wait(); }
    // Programmatic dependent launch: everything above (shared-memory carve-up, barrier init, law
    // table) overlaps the tail of the previous time step; the field is touched only from here on.
    // The next step's CTAs may be scheduled as soon as this grid leaves room for them.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    const int nr = p.nr, nz = p.nz, BL = p.BL, bpm = p.bands_per_member;
    const int cluster_id = blockIdx.x / CL, nclusters = gridDim.x / CL;
    const double g0 = p.g0;
    double fi0 = (double)i0;
    uint32_t qbase = 0;   // load sequence number of line offset -1 of this round
    uint32_t pubpar = 0;  // parity of the separator exchange buffer
    uint32_t lcount = 0;  // lines done (phase of the exchange barriers)

    // line offset L (-1 .. BL) of this CTA's bands -> TMA loads into slot (qbase+L+1)&3
    auto issue_loads = [&](int round, int L) {
        const uint32_t q = qbase + (uint32_t)(L + 1);
        const uint32_t sl = q % NSLOT;
        const uint32_t slot = sbase + sl * (uint32_t)SLOT;
        const uint32_t bar = mbar_a + 8u * sl;
        uint32_t bytes = 0;
        int R[LPB];
#pragma unroll
        for (int g = 0; g < LPB; ++g) {
            const int band = (round * nclusters + cluster_id) * LPB + g;
            R[g] = -1;
            if (band < p.total_bands) {
                const int b = band / bpm, j0 = 1 + (band - b * bpm) * BL;
                const int j1 = min(j0 + BL, nz - 1);
                const int j = j0 + L;
                if (j <= j1) {
                    R[g] = (b * nz + j) * p.rpl + crank * (G / 2);
                    bytes += (uint32_t)(G * 64);
                }
            }
        }
        if (CL > 1 && R[0] >= 0) bytes += (crank > 0 ? 16u : 0u) + (crank < CL - 1 ? 16u : 0u);
        mbar_expect_tx(bar, bytes);
#pragma unroll
        for (int g = 0; g < LPB; ++g)
            if (R[g] >= 0) tma_load_2d(slot + (uint32_t)(g * G * 64), &p.tm_ld, 0, R[g], bar);
        if (CL > 1 && R[0] >= 0) {
            const double *row0 = p.Told + (size_t)R[0] * 16;
            if (crank > 0) bulk_load_16(halo_a + sl * 32u, row0 - 2, bar);
            if (crank < CL - 1) bulk_load_16(halo_a + sl * 32u + 16u, row0 + (size_t)(G / 2) * 16, bar);
        }
    };
    auto wait_slot = [&](int L) {
        const uint32_t q = qbase + (uint32_t)(L + 1);
        while (!mbar_try_wait(mbar_a + 8u * (q % NSLOT), (q / NSLOT) & 1u)) {}
    };
    // line offset L of this CTA's bands -> TMA stores of the new level from its slot
    auto issue_stores = [&](int round, int L) {
        const uint32_t q = qbase + (uint32_t)(L + 1);
        const uint32_t slot = sbase + (q % NSLOT) * (uint32_t)SLOT;
#pragma unroll
        for (int g = 0; g < LPB; ++g) {
            const int band = (round * nclusters + cluster_id) * LPB + g;
            if (band >= p.total_bands) continue;
            const int b = band / bpm, j0 = 1 + (band - b * bpm) * BL;
            const int j1 = min(j0 + BL, nz - 1);
            const int j = j0 + L;
            if (j >= j1) continue;
            const int Rg = (b * nz + j) * p.rpl + crank * (G / 2);
            const uint32_t src = slot + (uint32_t)(g * G * 64);
            tma_store_2d(&p.tm_st, 0, Rg, src);
            // Neumann z lines copy their neighbour (reading G16)
            if (j == 1 && p.z_lo_neumann) tma_store_2d(&p.tm_st, 0, Rg - p.rpl, src);
            if (j == nz - 2 && p.z_hi_neumann) tma_store_2d(&p.tm_st, 0, Rg + p.rpl, src);
        }
        tma_commit();
    };

    for (int round = 0; (round * nclusters) * LPB < p.total_bands; ++round) {
        const int band = (round * nclusters + cluster_id) * LPB + grp;
        const bool live = band < p.total_bands;
        const int bandc = live ? band : p.total_bands - 1;
        const int b = bandc / bpm;
        const int j0 = 1 + (bandc - b * bpm) * BL;
        const int j1 = min(j0 + BL, nz - 1);

        // ---- per-thread constants of this band: laws of the chunk's layer, row flags
        const uint32_t cd = __ldg(p.cdesc + (size_t)b * (nr / 8) + t);
        const double qa = __ldg(p.Q0 + b) * p.amp; // Q0 nu(t_k) p^2(t_k), (2)-(4),(22)
        BCoef<DEGK> cA = load_coef<DEGK>(lay[cd & 0xffu], p.inv_tau, qa);
        const int ks = (int)((cd >> 16) & 0xfu) - 1;
        const bool first = (cd & BD_FIRST) != 0, last = (cd & BD_LAST) != 0;
        // a chunk with an interface node switches to the laws of layer B behind it (warp-uniform flag)
        const bool anysp = __any_sync(FULL, ks >= 0 || first || last);
        const bool anysq = __any_sync(FULL, cA.sq || (ks >= 0 && lay[(cd >> 8) & 0xffu].sqrtk != 0));

        if (tid == 32) { // thread 32 issues every TMA load and store (bulk groups are per thread)
            for (int Lp = -1; Lp <= min(2, BL); ++Lp) issue_loads(round, Lp);
        }
        wait_slot(-1);
        wait_slot(0);

        // ---- prologue: the flux through the faces between lines j0-1 and j0
        {
            const uint32_t sd = sbase + ((qbase + 0u) % NSLOT) * (uint32_t)SLOT;
            const uint32_t sc = sbase + ((qbase + 1u) % NSLOT) * (uint32_t)SLOT;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const double2 td = lds128(sd + co[q]);
                const double2 tc = lds128(sc + co[q]);
                double fl[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int k = 2 * q + e;
                    if (anysp && k == ks) cA = load_coef<DEGK>(lay[(cd >> 8) & 0xffu], p.inv_tau, qa);
                    const double a_ = e ? tc.y : tc.x, d_ = e ? td.y : td.x;
                    fl[e] = lam_eval<DEGK>(cA, anysq, a_ + d_) * (a_ - d_);
                }
                sts128(sbase + Cfg::OFF_FLUX + co[q], fl[0], fl[1]);
            }
        }

        for (int L = 0; L < BL; ++L) {
            const uint32_t q = qbase + (uint32_t)(L + 1);
            const uint32_t qs = q % NSLOT, qu = (q + 1u) % NSLOT;
            const uint32_t sc = sbase + qs * (uint32_t)SLOT; // line j   (centre)
            const uint32_t su = sbase + qu * (uint32_t)SLOT; // line j+1 (up)
            const uint32_t fr = sbase + Cfg::OFF_FLUX;       // lower flux fD, replaced in place by fU
            const uint32_t fw = fr;
            const int j = j0 + L;
            const bool line_live = live && (j < j1);
            const int jc = min(j, nz - 2);
            const double ezm = __ldg(p.ezm + jc), ezp = __ldg(p.ezp + jc);
            asm volatile("" : "+d"(fi0)); // keep the per-row geometry out of registers across lines
            wait_slot(L + 1);

            // ---- line j of the current level: the two r neighbours of the thread's 8 nodes
            double hl, hr;
            {
                const double2 v0 = lds128(sc + co[0]);
                const double2 v3 = lds128(sc + co[3]);
                hl = v0.x; hr = v3.y;
            }
            if (!edgeL) hl = lds64(sc + hlo);
            else if (CL > 1 && crank > 0) hl = lds64(halo_a + qs * 32u + 8u);
            if (!edgeR) hr = lds64(sc + hro);
            else if (CL > 1 && crank < CL - 1) hr = lds64(halo_a + qs * 32u + 16u);

            // ---- level 1: assemble (13)/(15)/(18) and sweep (12) the thread's 8 rows; the code path
            //      is chosen per warp: SQ = some lane has a square-root law, SP = some lane holds an
            //      interface node or an r-boundary row
            double al[8], be[8], gm[8];
            {
                SweepArgs<DEGK> A;
                A.sc = sc; A.su = su; A.fr = fr; A.fw = fw; A.hl = hl; A.hr = hr; A.fi0 = fi0; A.g0 = g0;
                A.ezp = ezp; A.ezm = ezm; A.inv_tau = p.inv_tau; A.qa = qa; A.cd = cd; A.ks = ks;
                A.first = first; A.last = last; A.rin_om = p.rin_om; A.rin_be = p.rin_be;
                A.rout_a = p.rout_a; A.rout_w = p.rout_w; A.rout_f = p.rout_f; A.lay = lay;
                if (!anysq) {
                    if (!anysp) sweep8<DEGK, false, false>(A, co, cA, al, be, gm);
                    else sweep8<DEGK, false, true>(A, co, cA, al, be, gm);
                } else {
                    if (!anysp) sweep8<DEGK, true, false>(A, co, cA, al, be, gm);
                    else sweep8<DEGK, true, true>(A, co, cA, al, be, gm);
                }
            }

            // ---- x_first = P x_last + Q + S u from the stored sweep coefficients
            double P = al[6], Q = be[6], S = gm[6];
#pragma unroll
            for (int k = 5; k >= 0; --k) {
                Q = fma(al[k], Q, be[k]);
                S = fma(al[k], S, gm[k]);
                P = P * al[k];
            }

            // ---- reduced row of this thread: a*y_{t-1} + y_t + c*y_{t+1} = d  (y = x of the last row)
            double Pn = __shfl_down_sync(FULL, P, 1);
            double Qn = __shfl_down_sync(FULL, Q, 1);
            double Sn = __shfl_down_sync(FULL, S, 1);
            if (lane == 31) { Pn = 0.0; Qn = 0.0; Sn = 0.0; }
            Row3 row;
            {
                const double r = rcp_cubic(fma(-al[7], Sn, 1.0));
                row.a = -gm[7] * r;
                row.c = -al[7] * Pn * r;
                row.d = fma(al[7], Qn, be[7]) * r;
            }
            // ---- level 2: PCR over lanes 0..30; lane 31 is the warp's separator
            const Row3 rp = pcr_lanes_0_30(row, lane);
            Row3 r30;
            r30.a = __shfl_sync(FULL, rp.a, 30);
            r30.c = __shfl_sync(FULL, rp.c, 30);
            r30.d = __shfl_sync(FULL, rp.d, 30);
            // publish what the separator solve needs from this warp (12 doubles) to every CTA of the
            // cluster: asynchronous DSMEM stores that complete on the receiver's mbarrier, so no
            // cluster-wide barrier and no release fence are needed
            const uint32_t pbar = sbase + Cfg::OFF_XBAR + 8u * pubpar;
            if (lane == 0 || lane == 31) {
                const uint32_t s6 = pub_a + (uint32_t)((pubpar * NSEP + gs) * Cfg::PUB) * 8u + (lane == 31 ? 48u : 0u);
                const double v0 = lane == 31 ? al[7] : P, v1 = lane == 31 ? be[7] : Q, v2 = lane == 31 ? gm[7] : S;
                const double v3 = lane == 31 ? r30.a : rp.a, v4 = lane == 31 ? r30.c : rp.c, v5 = lane == 31 ? r30.d : rp.d;
                if (CL > 1) {
#pragma unroll
                    for (int rk = 0; rk < CL; ++rk) {
                        const uint32_t ra = map_to_rank(s6, (uint32_t)rk), rb = map_to_rank(pbar, (uint32_t)rk);
                        st_async_v2(ra, v0, v1, rb);
                        st_async_v2(ra + 16, v2, v3, rb);
                        st_async_v2(ra + 32, v4, v5, rb);
                    }
                } else {
                    sts128(s6, v0, v1); sts128(s6 + 16, v2, v3); sts128(s6 + 32, v4, v5);
                }
            }
            if (CL == 1) __syncthreads();
            // ---- level 3: warp 0 builds every separator row and solves them (PCR per line)
            if (warp == 0) {
                if (CL > 1) {
                    if (lane == 0) mbar_expect_tx(pbar, (uint32_t)(NSEP * Cfg::PUB * 8));
                    while (!mbar_try_wait(pbar, (lcount >> 1) & 1u)) {}
                }
                const bool in3 = lane < NSEP;
                const int s = in3 ? lane : 0;
                const bool has_next = ((s % WG) + 1 < WG);
                const int sn = has_next ? s + 1 : s;
                const uint32_t Da = pub_a + (uint32_t)((pubpar * NSEP + s) * Cfg::PUB) * 8u;
                const uint32_t Dn = pub_a + (uint32_t)((pubpar * NSEP + sn) * Cfg::PUB) * 8u;
                const double2 d3 = lds128(Da + 48), d4 = lds128(Da + 64), d5 = lds128(Da + 80);
                const double2 n0 = lds128(Dn), n1 = lds128(Dn + 16), n2 = lds128(Dn + 32);
                const double sal = d3.x, sbe = d3.y, sgm = d4.x;
                Row3 l30; l30.a = d4.y; l30.c = d5.x; l30.d = d5.y;
                Row3 nx; nx.a = nx.c = nx.d = 0.0;
                double Pw = 0.0, Qw = 0.0, Sw = 0.0;
                if (has_next) { Pw = n0.x; Qw = n0.y; Sw = n1.x; nx.a = n1.y; nx.c = n2.x; nx.d = n2.y; }
                Row3 me;
                const double r = rcp_cubic(fma(-sal, Sw, 1.0));
                me.a = -sgm * r;
                me.c = -sal * Pw * r;
                me.d = fma(sal, Qw, sbe) * r;
                Row3 s3 = pcr_combine(me, l30, true, nx, has_next);
                s3 = pcr_segment<WG>(s3, s % WG, 0, WG - 1);
                if (in3) ysep[s] = s3.d;
            }
            __syncthreads();
            if (tid == 32) {
                // every thread wrote line L-1 before this barrier: store it, then refill the slot of
                // line L-2 (its store has read it) with line L+3
                if (L > 0) issue_stores(round, L - 1);
                if (L + 3 <= BL) { tma_wait_read1(); issue_loads(round, L + 3); }
            }
            pubpar ^= 1u;
            ++lcount;
            double y, u;
            {
                const double Vs = ysep[gs];
                const double U = (wig > 0) ? ysep[gs - 1] : 0.0;
                y = (lane == 31) ? Vs : fma(-rp.c, Vs, fma(-rp.a, U, rp.d));
                u = __shfl_up_sync(FULL, y, 1);
                if (lane == 0) u = U;
            }

            // ---- back substitution (14) P:L150; the new level replaces line j in its slot
            double x[8];
            x[7] = y;
#pragma unroll
            for (int k = 6; k >= 0; --k) x[k] = fma(al[k], x[k + 1], fma(gm[k], u, be[k]));
#pragma unroll
            for (int qq = 0; qq < 4; ++qq) sts128(sc + co[qq], x[2 * qq], x[2 * qq + 1]);
            fence_proxy_async();

            // ---- probes: T of the new level at (i_p, j_p)
            if (p.probe_out != nullptr && line_live) {
                for (int pq = 0; pq < p.nprobes; ++pq) {
                    const ProbeSrc ps = p.probes[pq];
                    if (ps.i < i0 || ps.i >= i0 + 8) continue;
                    if (ps.is_static) {
                        if (j == 1) p.probe_out[b * p.nprobes + pq] = p.Told[((size_t)b * nz + ps.j_store) * nr + ps.i];
                    } else if (ps.j_src == j) {
                        double v = 0.0;
#pragma unroll
                        for (int k = 0; k < 8; ++k)
                            if (i0 + k == ps.i) v = x[k];
                        p.probe_out[b * p.nprobes + pq] = v;
                    }
                }
            }
        }
        __syncthreads();
        if (tid == 32) issue_stores(round, BL - 1);
        qbase += (uint32_t)(BL + 2);
        if (tid == 32) tma_wait_read0(); // the next round's loads reuse the slots
        __syncthreads();
    }
    if (tid == 32) tma_wait_all0();
    if (CL > 1) { cluster_arrive(); cluster_wait(); }
}

} // namespace heat

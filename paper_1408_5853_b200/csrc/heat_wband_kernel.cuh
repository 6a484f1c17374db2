// heat_wband_kernel.cuh -- fourth-generation fused time-step kernel for sm_100a: the
// "warp-autonomous band kernel" (same arithmetic contract as
// heat_band_kernel.cuh, whose row formulas, sweep and PCR helpers it reuses).
//
// What the phase clocks of the band kernel showed on 8192 x 8192:
// the 8-row sweep of a warp is already bound by the FP64 pipe, but a line takes ~8300 cycles
// because (i) warps that hold an interface node or an r boundary run branchy code at half speed
// and every warp of the 4-SM cluster waits for them, (ii) the reduced system (PCR over the
// lanes, publication, a serial 32-row separator solve in one warp, __syncthreads) is pure latency
// paid once per 8 rows, (iii) every line ends in CTA-wide barriers.  Hence:
//   * a thread owns 16 consecutive nodes = one 128-byte tensor row, so the reduced system is
//     paid once per 16 rows and a line has half as many separators;
//   * every WARP runs its own TMA pipeline (its 4 KB part of each line, own ring of slots, own
//     mbarriers, own TMA stores): there is no __syncthreads in the line loop, the only coupling
//     between warps is the separator exchange itself (st.async + mbarrier transaction count
//     through (distributed) shared memory), after which every warp solves the <= 16 separator
//     rows itself (16 lanes, 4 PCR steps) instead of waiting for an elected warp and a barrier;
//   * rows (18) (interface) and (15) (r boundaries) need no code path of their own (see
//     wsweep16): every warp runs the same branch-free row loop, so there are two sweep bodies
//     (with / without the square root) instead of four and the hot code fits the 32 KB
//     instruction cache; the PCR loops are rolled for the same reason.
// Coverage: uniform r grid from r = 0, nr in {512, 1024, 2048, 4096, 8192}, laws CONST /
// POWER(p in {0,.5,1,1.5,2,3}) / POLY, lambda at the mean temperature (face_mode 0), temperature
// independent source shape, at most one interface node per 16-node chunk.
// "P:Lnnn" cites a line of the paper text; readings G1..G22 are listed in DESIGN.md.
#pragma once
#include <cuda.h>

#include "heat_band_kernel.cuh"
#include "heat_wband_params.cuh"

namespace heat {

template <int DEGK>
struct WCoef {
    double K[DEGK + 1];
    double Ct[4];
    double qs;
    bool sq;
};

template <int DEGK>
__device__ __forceinline__ WCoef<DEGK> wload_coef(const WLayer &L, double q0b)
{
    WCoef<DEGK> c;
#pragma unroll
    for (int n = 0; n <= DEGK; ++n) c.K[n] = L.K[n];
#pragma unroll
    for (int n = 0; n < 4; ++n) c.Ct[n] = L.Ct[n];
    c.qs = L.qsrc * q0b;
    c.sq = (L.sq != 0);
    return c;
}

// lambda at a face from s = Ta + Tb (G3); K may live in registers or in shared memory
template <int DEGK, bool SQ>
__device__ __forceinline__ double wlam(const double *K, bool sq, double s)
{
    double v = K[DEGK];
#pragma unroll
    for (int n = DEGK - 1; n >= 0; --n) v = fma(v, s, K[n]);
    if (SQ) {
        const double r = sqrt_pos(s);
        v = sq ? v * r : v;
    }
    return v;
}

// A regular row (13) P:L140-145 of the uniform r grid, scaled by i = r_i / h (see regular_row in
// heat_band_kernel.cuh): cfR = (i + 1/2) g0 lambda_{i+1/2,j}, w = i rho c / tau,
// f = w T + i (Lambda_j[T] + X), Lambda_j (11) P:L125 = ezp fU - ezm fD.
template <int DEGK, bool SQ>
__device__ __forceinline__ void wrow(const double *K, const double *Ct, double qs, bool sq, double T, double Tr,
                                     double Tu, double fD, double fi, double g0, double ezp, double ezm,
                                     double &cfR, double &w, double &f, double &fU)
{
    cfR = wlam<DEGK, SQ>(K, sq, T + Tr) * fma(g0, fi, 0.5 * g0);
    double c = Ct[3];
    c = fma(c, T, Ct[2]);
    c = fma(c, T, Ct[1]);
    c = fma(c, T, Ct[0]);
    w = c * fi;
    fU = wlam<DEGK, SQ>(K, sq, T + Tu) * (Tu - T);
    double lz = fma(ezp, fU, qs);
    lz = fma(-ezm, fD, lz);
    f = fma(w, T, fi * lz);
}

// The same row with separate factors for the r-face geometry (fi) and for the capacity / right-hand
// side (fie): fie = 0 turns the row into w = 0, f = 0, which is what the interface row (18) and the
// Neumann r_out row (15) need.
template <int DEGK, bool SQ>
__device__ __forceinline__ void wrow2(const double *K, const double *Ct, double qs, bool sq, double T, double Tr,
                                      double Tu, double fD, double fi, double fie, double g0, double ezp, double ezm,
                                      double &cfR, double &w, double &f, double &fU)
{
    cfR = wlam<DEGK, SQ>(K, sq, T + Tr) * fma(g0, fi, 0.5 * g0);
    double c = Ct[3];
    c = fma(c, T, Ct[2]);
    c = fma(c, T, Ct[1]);
    c = fma(c, T, Ct[0]);
    w = c * fie;
    fU = wlam<DEGK, SQ>(K, sq, T + Tu) * (Tu - T);
    double lz = fma(ezp, fU, qs);
    lz = fma(-ezm, fD, lz);
    f = fma(w, T, fie * lz);
}

// predicated reload of the law coefficients from a WLayer in shared memory (one predicate, paired
// loads): the registers keep their values where the predicate is false
template <int DEGK>
__device__ __forceinline__ void wcoef_reload_if(bool p, uint32_t a, WCoef<DEGK> &c)
{
    if (DEGK == 2) {
        asm("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %8, 0;\n\t"
            "@q ld.shared.v2.f64 {%0, %1}, [%7];\n\t"
            "@q ld.shared.f64 %2, [%7+16];\n\t"
            "@q ld.shared.v2.f64 {%3, %4}, [%7+48];\n\t"
            "@q ld.shared.v2.f64 {%5, %6}, [%7+64];\n\t}"
            : "+d"(c.K[0]), "+d"(c.K[1]), "+d"(c.K[2]), "+d"(c.Ct[0]), "+d"(c.Ct[1]), "+d"(c.Ct[2]), "+d"(c.Ct[3])
            : "r"(a), "r"((uint32_t)p));
    } else {
        asm("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %10, 0;\n\t"
            "@q ld.shared.v2.f64 {%0, %1}, [%9];\n\t"
            "@q ld.shared.v2.f64 {%2, %3}, [%9+16];\n\t"
            "@q ld.shared.f64 %4, [%9+32];\n\t"
            "@q ld.shared.v2.f64 {%5, %6}, [%9+48];\n\t"
            "@q ld.shared.v2.f64 {%7, %8}, [%9+64];\n\t}"
            : "+d"(c.K[0]), "+d"(c.K[1]), "+d"(c.K[2]), "+d"(c.K[3]), "+d"(c.K[DEGK]), "+d"(c.Ct[0]), "+d"(c.Ct[1]),
              "+d"(c.Ct[2]), "+d"(c.Ct[3])
            : "r"(a), "r"((uint32_t)p));
    }
}

struct WSweepArgs {
    uint32_t sc, su, fx;     // shared addresses: line j, line j+1, face fluxes (read fD, write fU in place)
    uint32_t rowo, sw;       // byte offset of the thread's tensor row in a slot, its swizzle phase
    uint32_t layA, layB;     // shared addresses of the WLayer before / from the interface row on
    double hl, hr;           // r neighbours of the chunk at line j
    double fi0, g0, ezp, ezm;
    double gl0;              // geometric factor of the face i0 - 1/2 (0 in the chunk that starts with a Neumann r_in row)
    double fie15;            // capacity / rhs factor of row 15 (0 in the chunk that ends with a Neumann r_out row)
    double qsB;              // source term of layer B
    int ks;                  // interface row (18) of this chunk, < 0: none
    bool sqB;
    bool din, dout;          // the chunk starts / ends with a Dirichlet r-boundary row
    bool nin, last;          // the chunk starts with the Neumann r_in row / ends with the r_out row
    double rin_be, rout_f;
};

// Level 1 for one thread: rows (13) P:L140-145 assembled and pushed through the sweep (12)
// P:L133-136, sixteen rows, no branch inside the row loop and ONE code path for every warp:
//   * interface row (18)-(20) P:L176-192 at row ks: the two face coefficients are replaced by
//     lam*_A, lam*_B (selects), capacity and right-hand side vanish (fie = 0), and the thread's law
//     coefficients switch to layer B by predicated loads from the shared table;
//   * Neumann r rows (15)-(17) P:L158-174 are ordinary rows with data chosen per band: the row
//     T^_0 = T^_1 is the regular row with a zero left face (gl0 = 0; its i = 0 already gives
//     w = f = 0), the row T^_N = T^_{N-1} is the regular row with fie = 0 and a zero right face;
//   * Dirichlet r rows are selects at rows 0 / 15.
template <int DEGK, bool SQ>
__device__ __forceinline__ void wsweep16(const WSweepArgs &A, const uint32_t (&co)[8], WCoef<DEGK> c,
                                         double (&al)[16], double (&be)[16], double (&gm)[16])
{
    SweepState st;
    st.om = 1.0; st.be = 0.0; st.gm = 1.0;
    // interface node: lam*_A, lam*_B at T_{i*,j} of the old level
    double lamA_if = 0.0, lamB_if = 0.0;
    if (A.ks >= 0) {
        const double Tk = lds64(A.sc + A.rowo + ((((uint32_t)A.ks >> 1) ^ A.sw) << 4) + (((uint32_t)A.ks & 1u) << 3));
        double KB[DEGK + 1];
#pragma unroll
        for (int n = 0; n <= DEGK; ++n) KB[n] = lds64(A.layB + 8u * n);
        lamA_if = wlam<DEGK, true>(c.K, c.sq, Tk + Tk);
        lamB_if = wlam<DEGK, true>(KB, A.sqB, Tk + Tk);
    }
    double2 tl = lds128(A.sc + co[0]);
    st.cfL = wlam<DEGK, SQ>(c.K, c.sq, A.hl + tl.x) * A.gl0; // face i0 - 1/2
#pragma unroll
    for (int qq = 0; qq < 8; ++qq) {
        double2 tn;
        if (qq < 7) tn = lds128(A.sc + co[qq < 7 ? qq + 1 : 7]);
        else tn = make_double2(A.hr, A.hr);
        const double2 tu = lds128(A.su + co[qq]);
        const double2 fd = lds128(A.fx + co[qq]);
        double fu[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int k = 2 * qq + e;
            const double T = e ? tl.y : tl.x;
            const bool isif = (k == A.ks);
            // from the interface row on the chunk is layer B (the face i* + 1/2 belongs to it, G14)
            wcoef_reload_if<DEGK>(isif, A.layB, c);
            c.qs = isif ? A.qsB : c.qs;
            c.sq = isif ? A.sqB : c.sq;
            const double fi = A.fi0 + (double)k;
            double fie = (k == 15) ? A.fie15 : fi;
            fie = isif ? 0.0 : fie;
            double cfR, w, f;
            wrow2<DEGK, SQ>(c.K, c.Ct, c.qs, c.sq, T, e ? tn.x : tl.y, e ? tu.y : tu.x, e ? fd.y : fd.x,
                            fi, fie, A.g0, A.ezp, A.ezm, cfR, w, f, fu[e]);
            // (18) times h: -lam_A x_{i-1} + (lam_A + lam_B) x_i - lam_B x_{i+1} = 0 (new level, G7)
            double cfL_use = isif ? lamA_if : st.cfL;
            double cfR_use = isif ? lamB_if : cfR;
            if (k == 15) { // r_out row (15),(17): x_N = x_{N-1} (fie15 = 0, no right face) or x_N = value
                cfR_use = A.last ? 0.0 : cfR_use;
                cfL_use = A.dout ? 0.0 : cfL_use;
                w = A.dout ? 1.0 : w;
                f = A.dout ? A.rout_f : f;
            }
            st.cfL = cfL_use;
            sweep_row(st, cfR_use, w, f, al[k]);
            st.cfL = cfR; // face i + 1/2 as the next regular row sees it
            if (k == 0) { // r_in row (15),(16): alpha_0 = 1 exactly (T^_0 = T^_1 bitwise); Dirichlet: x_0 = value
                al[0] = A.nin ? 1.0 : al[0];
                al[0] = A.din ? 0.0 : al[0];
                st.om = A.din ? 1.0 : st.om;
                st.be = A.din ? A.rin_be : st.be;
                st.gm = A.din ? 0.0 : st.gm;
            }
            be[k] = st.be; gm[k] = st.gm;
        }
        sts128(A.fx + co[qq], fu[0], fu[1]);
        tl = tn;
    }
}

// rolled PCR loops (code size: the instruction cache holds 32 KB)
__device__ __forceinline__ Row3 pcr_lanes_0_30_rolled(Row3 row, int lane)
{
#pragma unroll 1
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
template <int WIDTH>
__device__ __forceinline__ Row3 pcr_segment_rolled(Row3 row, int lane, int lo, int hi)
{
#pragma unroll 1
    for (int s = 1; s < WIDTH; s <<= 1) {
        Row3 L, R;
        L.a = __shfl_up_sync(0xffffffffu, row.a, s, WIDTH);
        L.c = __shfl_up_sync(0xffffffffu, row.c, s, WIDTH);
        L.d = __shfl_up_sync(0xffffffffu, row.d, s, WIDTH);
        R.a = __shfl_down_sync(0xffffffffu, row.a, s, WIDTH);
        R.c = __shfl_down_sync(0xffffffffu, row.c, s, WIDTH);
        R.d = __shfl_down_sync(0xffffffffu, row.d, s, WIDTH);
        const bool in = (lane >= lo) && (lane <= hi);
        const Row3 n = pcr_combine(row, L, in && (lane - s >= lo), R, in && (lane + s <= hi));
        if (in) row = n;
    }
    return row;
}

// WL = warps per line (nr = 512 WL), NW = warps per CTA, DEGK = degree of the lambda polynomials.
template <int WL, int NW, int DEGK>
__global__ void __launch_bounds__(32 * NW, 8 / NW) heat_wband_kernel(const __grid_constant__ WParams p)
{
    using Cfg = WBandCfg<WL, NW>;
    constexpr int CL = Cfg::CL, LPB = Cfg::LPB, WPL = Cfg::WPL, NS = Cfg::NS, SLOT = Cfg::SLOT;
    constexpr uint32_t FULL = 0xffffffffu;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char *gbase = smem_raw + (sbase - smem_u32(smem_raw));
    WLayer *lay = reinterpret_cast<WLayer *>(gbase + Cfg::OFF_LAY);

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = __shfl_sync(FULL, tid >> 5, 0); // provably warp-uniform: TMA operands stay in uniform registers
    const int grp = warp / WPL; // line (band) within the CTA
    const int wl = warp % WPL;  // warp within the CTA's part of the line
    const int cluster_id = blockIdx.x / CL, nclusters = gridDim.x / CL;
    // rank of this CTA within the line: the hardware rank, rotated by CL/2 in odd clusters so that
    // the CTAs sharing an SM do not hold the same (possibly most expensive) part of the radius
    const int crank = (CL > 1) ? (int)((cluster_ctarank() + (uint32_t)((cluster_id & 1) ? CL / 2 : 0)) % (uint32_t)CL) : 0;
    const int wig = crank * WPL + wl; // warp within the line = separator index
    const int t = wig * 32 + lane;    // thread within the line = tensor row within the line
    const int i0 = t * 16;
    const uint32_t wbase = sbase + (uint32_t)warp * (uint32_t)Cfg::WARP_BYTES;
    const uint32_t fx = wbase + (uint32_t)(NS * SLOT);
    const uint32_t halo_a = sbase + Cfg::OFF_HALO + (uint32_t)(warp * NS) * 32u;
    const uint32_t fbar_a = sbase + Cfg::OFF_FBAR + (uint32_t)(warp * NS) * 8u;
    const uint32_t xbar_a = sbase + Cfg::OFF_XBAR + (uint32_t)grp * 16u;
    const uint32_t pub_a = sbase + Cfg::OFF_PUB;
    // byte offsets of the thread's eight 16-byte chunks inside a SWIZZLE_128B slot, and of its two
    // r neighbours (last node of the row above, first node of the row below)
    uint32_t co[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) co[q] = (uint32_t)lane * 128u + (uint32_t)((q ^ (lane & 7)) << 4);
    const uint32_t hlo = (uint32_t)(lane - 1) * 128u + (uint32_t)((7 ^ ((lane - 1) & 7)) << 4) + 8u;
    const uint32_t hro = (uint32_t)(lane + 1) * 128u + (uint32_t)(((lane + 1) & 7) << 4);
    const bool has_l = (wig > 0), has_r = (wig < WL - 1); // the warp has a left / right neighbour warp

    // ---- law table scaled for this launch, barriers
    if (tid < p.nlayers) {
        const PLayer &P = p.players[tid];
        WLayer W;
#pragma unroll
        for (int n = 0; n < 5; ++n) W.K[n] = P.K[n];
        W.K[5] = 0.0;
#pragma unroll
        for (int n = 0; n < 4; ++n) W.Ct[n] = P.C[n] * p.inv_tau;
        W.qsrc = P.heater ? p.amp * P.src : 0.0;
        W.sq = P.sqrtk;
        W.pad_ = 0;
        lay[tid] = W;
    }
    if (tid == 0) {
#pragma unroll 1
        for (int s = 0; s < NW * NS; ++s) mbar_init(sbase + Cfg::OFF_FBAR + 8u * s, 1);
#pragma unroll 1
        for (int s = 0; s < LPB * 2; ++s) mbar_init(sbase + Cfg::OFF_XBAR + 8u * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (CL > 1) { cluster_arrive(); cluster_wait(); }
    // programmatic dependent launch: the set-up above overlaps the tail of the previous step
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    const int nz = p.nz, rpl = p.rpl, BL = p.BL, bpm = p.bands_per_member;
    const double g0 = p.g0;
    double fi0 = (double)i0;
    uint32_t qbase = 0;  // load sequence number of line offset -1 of this band
    uint32_t lcount = 0; // lines done (phase of the exchange barriers)

    for (int round = 0;; ++round) {
        const int band = (round * nclusters + cluster_id) * LPB + grp;
        if (band >= p.total_bands) break; // uniform over the warps of a line
        const int b = band / bpm;
        const int j0 = 1 + (band - b * bpm) * BL;
        const int j1 = min(j0 + BL, nz - 1);
        const int nl = j1 - j0;
        const int row0 = (b * nz + j0 - 1) * rpl + wig * 32; // tensor row of this warp's part of line j0 - 1

        // load sequence s (line j0 - 1 + s) -> slot s % NS; lane 0 issues every TMA operation of the warp
        auto issue_load = [&](uint32_t s) {
            const uint32_t q = qbase + s, sl = q % (uint32_t)NS;
            const uint32_t bar = fbar_a + 8u * sl;
            const int R = row0 + (int)s * rpl;
            mbar_expect_tx(bar, (uint32_t)SLOT + (has_l ? 16u : 0u) + (has_r ? 16u : 0u));
            tma_load_2d(wbase + sl * (uint32_t)SLOT, &p.tm_ld, 0, R, bar);
            const double *g = p.Told + (size_t)R * 16;
            if (has_l) bulk_load_16(halo_a + sl * 32u, g - 2, bar);
            if (has_r) bulk_load_16(halo_a + sl * 32u + 16u, g + 512, bar);
        };
        auto wait_seq = [&](uint32_t s) {
            const uint32_t q = qbase + s;
            while (!mbar_try_wait(fbar_a + 8u * (q % (uint32_t)NS), (q / (uint32_t)NS) & 1u)) {}
        };

        // ---- per-thread constants of this band
        const uint32_t cd = __ldg(p.wdesc + (size_t)b * rpl + t);
        const int la = (int)(cd & 0xffu), lb = (int)((cd >> 8) & 0xffu);
        const int ks = (int)((cd >> 16) & 0x1fu) - 1;
        const bool first = (cd & WD_FIRST) != 0, last = (cd & WD_LAST) != 0;
        const double q0b = __ldg(p.Q0 + b); // X = Q0 nu(t_k) p^2(t_k) s, (2)-(4),(22)
        const WCoef<DEGK> cA = wload_coef<DEGK>(lay[la], q0b);
        const bool anysq = __any_sync(FULL, cA.sq || (ks >= 0 && lay[lb].sq != 0));
        const bool rin_neu = (p.rin_om == 0.0), rout_neu = (p.rout_w == 0.0);
        WSweepArgs A;
        A.fx = fx; A.rowo = (uint32_t)lane * 128u; A.sw = (uint32_t)lane & 7u;
        A.layA = smem_u32(&lay[la]); A.layB = smem_u32(&lay[lb]);
        A.g0 = g0;
        A.gl0 = (first && rin_neu) ? 0.0 : fma(g0, (double)i0, -0.5 * g0);
        A.fie15 = (last && rout_neu) ? 0.0 : (double)(i0 + 15);
        A.qsB = lay[lb].qsrc * q0b; A.sqB = (lay[lb].sq != 0);
        A.ks = ks; A.din = first && !rin_neu; A.dout = last && !rout_neu; A.nin = first && rin_neu; A.last = last;
        A.rin_be = p.rin_be; A.rout_f = p.rout_f;

        if (lane == 0) {
            const uint32_t npre = (uint32_t)min(NS, nl + 2);
            for (uint32_t s = 0; s < npre; ++s) issue_load(s);
        }
        wait_seq(0);
        wait_seq(1);

        // ---- prologue: the flux through the faces between lines j0 - 1 and j0
        {
            const uint32_t sd = wbase + ((qbase + 0u) % (uint32_t)NS) * (uint32_t)SLOT;
            const uint32_t s1 = wbase + ((qbase + 1u) % (uint32_t)NS) * (uint32_t)SLOT;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const double2 td = lds128(sd + co[q]);
                const double2 tc = lds128(s1 + co[q]);
                double fl[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int k = 2 * q + e;
                    const WLayer &Lk = lay[(ks >= 0 && k >= ks) ? lb : la];
                    const double a_ = e ? tc.y : tc.x, d_ = e ? td.y : td.x;
                    fl[e] = wlam<DEGK, true>(Lk.K, Lk.sq != 0, a_ + d_) * (a_ - d_);
                }
                sts128(fx + co[q], fl[0], fl[1]);
            }
        }
        __syncwarp();
        if (lane == 0 && NS <= nl + 1) issue_load((uint32_t)NS); // the slot of line j0 - 1 is free again

        for (int L = 0; L < nl; ++L) {
            const uint32_t q = qbase + (uint32_t)(L + 1);
            const uint32_t qs = q % (uint32_t)NS, qu = (q + 1u) % (uint32_t)NS;
            const uint32_t sc = wbase + qs * (uint32_t)SLOT; // line j   (centre)
            const uint32_t su = wbase + qu * (uint32_t)SLOT; // line j+1 (up)
            const int j = j0 + L;
            const double ezm = __ldg(p.ezm + j), ezp = __ldg(p.ezp + j);
            asm volatile("" : "+d"(fi0)); // keep the per-row geometry out of registers across lines
            wait_seq((uint32_t)(L + 2));

            // ---- the two r neighbours of the thread's 16 nodes at line j
            double hl, hr;
            {
                const double2 v0 = lds128(sc + co[0]);
                const double2 v7 = lds128(sc + co[7]);
                hl = v0.x; hr = v7.y;
            }
            if (lane > 0) hl = lds64(sc + hlo);
            else if (has_l) hl = lds64(halo_a + qs * 32u + 8u);
            if (lane < 31) hr = lds64(sc + hro);
            else if (has_r) hr = lds64(halo_a + qs * 32u + 16u);

            // ---- level 1: assemble (13)/(15)/(18) and sweep (12) the thread's 16 rows; the code path
            //      is chosen per warp: SQ = some lane has a square-root law, SP = some lane holds an
            //      interface node or an r-boundary row
            double al[16], be[16], gm[16];
            A.sc = sc; A.su = su; A.hl = hl; A.hr = hr; A.fi0 = fi0; A.ezp = ezp; A.ezm = ezm;
            if (!anysq) wsweep16<DEGK, false>(A, co, cA, al, be, gm);
            else wsweep16<DEGK, true>(A, co, cA, al, be, gm);

            // ---- x_first = P x_last + Q + S u from the stored sweep coefficients
            double P = al[14], Q = be[14], S = gm[14];
#pragma unroll
            for (int k = 13; k >= 0; --k) {
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
                const double r = rcp_cubic(fma(-al[15], Sn, 1.0));
                row.a = -gm[15] * r;
                row.c = -al[15] * Pn * r;
                row.d = fma(al[15], Qn, be[15]) * r;
            }
            double y, u;
            if constexpr (WL == 1) {
                // the whole line is this warp: PCR over all 32 reduced rows
                row = pcr_segment_rolled<32>(row, lane, 0, 31);
                y = row.d;
                u = __shfl_up_sync(FULL, y, 1);
                if (lane == 0) u = 0.0;
            } else {
                // ---- level 2: PCR over lanes 0..30; lane 31 is the warp's separator
                const Row3 rp = pcr_lanes_0_30_rolled(row, lane);
                Row3 r30;
                r30.a = __shfl_sync(FULL, rp.a, 30);
                r30.c = __shfl_sync(FULL, rp.c, 30);
                r30.d = __shfl_sync(FULL, rp.d, 30);
                // publish what the separator solve needs from this warp (12 doubles) to every CTA of the
                // line: asynchronous (distributed) shared-memory stores that complete on the receiver's
                // mbarrier, so neither a barrier nor a release fence is needed
                const uint32_t pubpar = lcount & 1u;
                const uint32_t pbar = xbar_a + 8u * pubpar;
                const uint32_t pub0 = pub_a + (uint32_t)((pubpar * LPB + grp) * WL * Cfg::PUB) * 8u;
                if (wl == 0 && lane == 1) mbar_expect_tx(pbar, (uint32_t)(WL * Cfg::PUB * 8));
                if (lane == 0 || lane == 31) {
                    const uint32_t s6 = pub0 + (uint32_t)(wig * Cfg::PUB) * 8u + (lane == 31 ? 48u : 0u);
                    const double v0 = lane == 31 ? al[15] : P, v1 = lane == 31 ? be[15] : Q, v2 = lane == 31 ? gm[15] : S;
                    const double v3 = lane == 31 ? r30.a : rp.a, v4 = lane == 31 ? r30.c : rp.c, v5 = lane == 31 ? r30.d : rp.d;
#pragma unroll
                    for (int rk = 0; rk < CL; ++rk) {
                        const uint32_t ra = map_to_rank(s6, (uint32_t)rk), rb = map_to_rank(pbar, (uint32_t)rk);
                        st_async_v2(ra, v0, v1, rb);
                        st_async_v2(ra + 16, v2, v3, rb);
                        st_async_v2(ra + 32, v4, v5, rb);
                    }
                }
                while (!mbar_try_wait(pbar, (lcount >> 1) & 1u)) {}
                // ---- level 3: every warp builds the WL separator rows and solves them (PCR, 16 lanes)
                double ys;
                {
                    const bool in3 = lane < WL;
                    const int s = in3 ? lane : 0;
                    const bool has_next = (s + 1 < WL);
                    const int sn = has_next ? s + 1 : s;
                    const uint32_t Da = pub0 + (uint32_t)(s * Cfg::PUB) * 8u;
                    const uint32_t Dn = pub0 + (uint32_t)(sn * Cfg::PUB) * 8u;
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
                    s3 = pcr_segment_rolled<WL>(s3, s, 0, WL - 1);
                    ys = s3.d;
                }
                const double Vs = __shfl_sync(FULL, ys, wig);
                double U = __shfl_sync(FULL, ys, (wig + WL - 1) % WL);
                if (wig == 0) U = 0.0;
                y = (lane == 31) ? Vs : fma(-rp.c, Vs, fma(-rp.a, U, rp.d));
                u = __shfl_up_sync(FULL, y, 1);
                if (lane == 0) u = U;
            }
            ++lcount;

            // ---- back substitution (14) P:L150; the new level replaces line j in its slot
            double x[16];
            x[15] = y;
#pragma unroll
            for (int k = 14; k >= 0; --k) x[k] = fma(al[k], x[k + 1], fma(gm[k], u, be[k]));
#pragma unroll
            for (int qq = 0; qq < 8; ++qq) sts128(sc + co[qq], x[2 * qq], x[2 * qq + 1]);
            fence_proxy_async();
            __syncwarp();

            // ---- the warp's own TMA store of its 4 KB of the new level; Neumann z lines copy their
            //      neighbour (reading G16); then refill the slot of line j - 1 (its store has been read)
            if (lane == 0) {
                const int Rg = (b * nz + j) * rpl + wig * 32;
                tma_store_2d(&p.tm_st, 0, Rg, sc);
                if (j == 1 && p.z_lo_neumann) tma_store_2d(&p.tm_st, 0, Rg - rpl, sc);
                if (j == nz - 2 && p.z_hi_neumann) tma_store_2d(&p.tm_st, 0, Rg + rpl, sc);
                tma_commit();
                if (L >= 1 && L + NS <= nl + 1) { tma_wait_read1(); issue_load((uint32_t)(L + NS)); }
            }

            // ---- probes: T of the new level at (i_p, j_p)
            if (p.probe_out != nullptr) {
                for (int pq = 0; pq < p.nprobes; ++pq) {
                    const ProbeSrc ps = p.probes[pq];
                    if (ps.i < i0 || ps.i >= i0 + 16) continue;
                    if (ps.is_static) {
                        if (j == 1) p.probe_out[b * p.nprobes + pq] = p.Told[((size_t)b * nz + ps.j_store) * p.nr + ps.i];
                    } else if (ps.j_src == j) {
                        double v = 0.0;
#pragma unroll
                        for (int k = 0; k < 16; ++k)
                            if (i0 + k == ps.i) v = x[k];
                        p.probe_out[b * p.nprobes + pq] = v;
                    }
                }
            }
        }
        if (lane == 0) tma_wait_read0(); // the next band's loads reuse the slots
        __syncwarp();
        qbase += (uint32_t)(nl + 2);
    }
    if (lane == 0) tma_wait_all0();
    if (CL > 1) { cluster_arrive(); cluster_wait(); }
}

} // namespace heat

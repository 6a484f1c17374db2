// heat_tband_kernel.cuh -- fifth-generation fused time-step kernel for sm_100a: the warp-autonomous
// band kernel (heat_wband_kernel.cuh) with the sweep coefficients parked in TENSOR MEMORY.
//
// Why: heat_wband_kernel is purely latency-bound -- its throughput on 8192 x 8192 is proportional
// to the warps per SM (4 warps: 60, 6: 88, 8: 113 GCUPS, profiles/r02_tband_summary.md) -- and the
// 96 registers that hold (alpha, beta, gamma) of a thread's 16 rows between the forward sweep (12)
// and the back substitution (14) cap it at 8 warps per SM.  Blackwell's tensor memory gives every
// thread of a warp a private 512-byte strip (its lane x 128 columns of 32 bits): exactly 16 rows x
// (alpha, beta, gamma, face flux).  With those parked there (tcgen05.st during the sweep,
// tcgen05.ld during the back substitution) the kernel needs <= 128 registers and three 4 KB line
// slots per warp, so 16 warps = 8192 nodes x 16 B of state are in flight per SM: a whole line of
// the large grid.
// Further differences from heat_wband_kernel.cuh: the row loop is rolled over groups of four rows
// with a plain and a general body chosen per warp and group (tgroup), one duty warp per CTA solves
// the separator rows (and skips their PCR when it cannot change the result), a whole line sits in
// one CTA where it fits (nr = 8192: 16 warps, no cluster).  Per-warp TMA pipelines and the
// separator exchange by st.async + mbarrier are as there; same coverage, same arithmetic.
// "P:Lnnn" cites a line of the paper text; readings G1..G22 are listed in DESIGN.md.
#pragma once
#include <cuda.h>

#include "heat_wband_kernel.cuh"

namespace heat {

// WL = warps per line (nr = 512 WL), NW = warps per CTA (4, 8 or 16: every lane quarter of the
// tensor memory is used).  16 / NW CTAs per SM.
template <int WL, int NW>
struct TBandCfg {
    static constexpr int M = 16;
    static constexpr int NT = 32 * NW;
    static constexpr int CL = (WL > NW) ? WL / NW : 1;
    static constexpr int LPB = (WL < NW) ? NW / WL : 1;
    static constexpr int WPL = (WL < NW) ? WL : NW;
    static constexpr int NS = 3;                      // ring of staged line parts per warp: j, j+1, j+2
    static constexpr int SLOT = 4096;                 // 32 threads x 16 doubles
    static constexpr int PUB = 12;
    static constexpr int TCOLS = 128 * (NW / 4);      // tensor-memory columns of the CTA
    static constexpr int WARP_BYTES = NS * SLOT;
    static constexpr int OFF_HALO = NW * WARP_BYTES;                  // [NW][NS][4 doubles]
    static constexpr int OFF_PUB = OFF_HALO + NW * NS * 32;           // [2][LPB][WL][PUB]
    static constexpr int OFF_FBAR = OFF_PUB + 2 * LPB * WL * PUB * 8; // [NW][NS] load barriers
    static constexpr int OFF_XBAR = OFF_FBAR + NW * NS * 8;           // [LPB][2] exchange barriers
    static constexpr int OFF_YBAR = OFF_XBAR + LPB * 2 * 8;           // [LPB][2] separator-solution barriers
    static constexpr int OFF_YSEP = OFF_YBAR + LPB * 2 * 8;           // [2][LPB][WL] separator values
    static constexpr int OFF_TMEM = OFF_YSEP + 2 * LPB * WL * 8;      // tensor-memory base address
    static constexpr int OFF_LAY = OFF_TMEM + 16;
    static constexpr size_t smem_bytes(int nlayers) { return 1024 + (size_t)OFF_LAY + sizeof(WLayer) * (size_t)nlayers; }
};

// ---------------------------------------------------------------- tensor memory as a register file
// A warp addresses its own lane quarter; lane i of the warp owns tensor-memory lane (quarter*32 + i),
// `x8` moves eight consecutive 32-bit columns = four doubles per thread.
__device__ __forceinline__ void tmem_st4(uint32_t taddr, double a, double b, double c, double d)
{
    asm volatile("{\n\t.reg .b32 r<8>;\n\t"
                 "mov.b64 {r0, r1}, %1;\n\tmov.b64 {r2, r3}, %2;\n\tmov.b64 {r4, r5}, %3;\n\tmov.b64 {r6, r7}, %4;\n\t"
                 "tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {r0, r1, r2, r3, r4, r5, r6, r7};\n\t}"
                 ::"r"(taddr), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}
// one double per store: a double already sits in an aligned register pair, while the .x8 form wants eight
// consecutive registers and costs ~25 register moves per four-row group (measured: +0.7 % on 8192 x 8192)
__device__ __forceinline__ void tmem_st1(uint32_t taddr, double a)
{
    asm volatile("{\n\t.reg .b32 r<2>;\n\tmov.b64 {r0, r1}, %1;\n\t"
                 "tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {r0, r1};\n\t}"
                 ::"r"(taddr), "d"(a) : "memory");
}
struct TRaw8 {
    uint32_t r[8];
};
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, TRaw8 &v)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v.r[0]), "=r"(v.r[1]), "=r"(v.r[2]), "=r"(v.r[3]), "=r"(v.r[4]), "=r"(v.r[5]), "=r"(v.r[6]), "=r"(v.r[7])
                 : "r"(taddr) : "memory");
}
// the loaded registers are valid only after the wait: they pass through it as operands so that no
// use can be scheduled ahead of it
__device__ __forceinline__ void tmem_wait_ld(TRaw8 &v)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(v.r[0]), "+r"(v.r[1]), "+r"(v.r[2]), "+r"(v.r[3]), "+r"(v.r[4]), "+r"(v.r[5]), "+r"(v.r[6]), "+r"(v.r[7])
                 :: "memory");
}
__device__ __forceinline__ void tmem_wait_ld3(TRaw8 &a, TRaw8 &b, TRaw8 &c)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(a.r[0]), "+r"(a.r[1]), "+r"(a.r[2]), "+r"(a.r[3]), "+r"(a.r[4]), "+r"(a.r[5]), "+r"(a.r[6]), "+r"(a.r[7]),
                   "+r"(b.r[0]), "+r"(b.r[1]), "+r"(b.r[2]), "+r"(b.r[3]), "+r"(b.r[4]), "+r"(b.r[5]), "+r"(b.r[6]), "+r"(b.r[7]),
                   "+r"(c.r[0]), "+r"(c.r[1]), "+r"(c.r[2]), "+r"(c.r[3]), "+r"(c.r[4]), "+r"(c.r[5]), "+r"(c.r[6]), "+r"(c.r[7])
                 :: "memory");
}
struct TRaw16 {
    uint32_t r[16];
};
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, TRaw16 &v)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(v.r[0]), "=r"(v.r[1]), "=r"(v.r[2]), "=r"(v.r[3]), "=r"(v.r[4]), "=r"(v.r[5]), "=r"(v.r[6]), "=r"(v.r[7]),
                   "=r"(v.r[8]), "=r"(v.r[9]), "=r"(v.r[10]), "=r"(v.r[11]), "=r"(v.r[12]), "=r"(v.r[13]), "=r"(v.r[14]), "=r"(v.r[15])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld16(TRaw16 &a, TRaw16 &b, TRaw16 &c)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(a.r[0]), "+r"(a.r[1]), "+r"(a.r[2]), "+r"(a.r[3]), "+r"(a.r[4]), "+r"(a.r[5]), "+r"(a.r[6]), "+r"(a.r[7]),
                   "+r"(a.r[8]), "+r"(a.r[9]), "+r"(a.r[10]), "+r"(a.r[11]), "+r"(a.r[12]), "+r"(a.r[13]), "+r"(a.r[14]), "+r"(a.r[15]),
                   "+r"(b.r[0]), "+r"(b.r[1]), "+r"(b.r[2]), "+r"(b.r[3]), "+r"(b.r[4]), "+r"(b.r[5]), "+r"(b.r[6]), "+r"(b.r[7]),
                   "+r"(b.r[8]), "+r"(b.r[9]), "+r"(b.r[10]), "+r"(b.r[11]), "+r"(b.r[12]), "+r"(b.r[13]), "+r"(b.r[14]), "+r"(b.r[15]),
                   "+r"(c.r[0]), "+r"(c.r[1]), "+r"(c.r[2]), "+r"(c.r[3]), "+r"(c.r[4]), "+r"(c.r[5]), "+r"(c.r[6]), "+r"(c.r[7]),
                   "+r"(c.r[8]), "+r"(c.r[9]), "+r"(c.r[10]), "+r"(c.r[11]), "+r"(c.r[12]), "+r"(c.r[13]), "+r"(c.r[14]), "+r"(c.r[15])
                 :: "memory");
}
__device__ __forceinline__ double traw16(const TRaw16 &v, int n) { return __hiloint2double((int)v.r[2 * n + 1], (int)v.r[2 * n]); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ double traw(const TRaw8 &v, int n) { return __hiloint2double((int)v.r[2 * n + 1], (int)v.r[2 * n]); }

// columns of a thread's strip: rows in groups of four, group g: 24 columns of (alpha, beta, gamma) x 4
// at 24 g, the four face fluxes at 96 + 8 g
__device__ __forceinline__ constexpr uint32_t tcol_coef(int g, int part) { return (uint32_t)(24 * g + 8 * part); }
__device__ __forceinline__ constexpr uint32_t tcol_flux(int g) { return (uint32_t)(96 + 8 * g); }

// PCR elimination as pcr_combine (heat_line_kernel.cuh), with the boundary handled by masking the ONE
// coefficient that does the elimination (a where there is no left row, c where there is no right row)
// instead of the two values it would multiply: four selects fewer per step, same bits for finite rows
// (-0 * x = -0, and 1 + -0 = 1, d + -0 = d exactly).
__device__ __forceinline__ Row3 tpcr_combine(const Row3 &me, const Row3 &L, bool vl, const Row3 &R, bool vr)
{
    const double ae = vl ? me.a : 0.0, ce = vr ? me.c : 0.0;
    // (the minus sign on the shuffled operand: it is an operand modifier there, whereas negating the
    // selected ae / ce would cost an instruction on the FP64 pipe; the products are the same bits)
    double den = fma(ae, -L.c, 1.0);
    den = fma(ce, -R.a, den);
    const double r = rcp_cubic(den);
    double d = fma(ae, -L.d, me.d);
    d = fma(ce, -R.d, d);
    Row3 o;
    o.d = d * r;
    const double ar_ = me.a * r, cr_ = me.c * r;
    o.a = vl ? -ar_ * L.a : ar_; // an external reference keeps its coefficient
    o.c = vr ? -cr_ * R.c : cr_;
    return o;
}
// HI = 30: PCR over lanes 0..30 (lane 31, the warp's separator, runs along and produces values nobody reads);
// HI = 31: over the whole warp (a line of one warp).
template <bool UNROLL, int HI>
__device__ __forceinline__ Row3 tpcr_lanes(Row3 row, int lane)
{
#pragma unroll (UNROLL ? 5 : 1)
    for (int s = 1; s < 32; s <<= 1) {
        Row3 L, R;
        L.a = __shfl_up_sync(0xffffffffu, row.a, s);
        L.c = __shfl_up_sync(0xffffffffu, row.c, s);
        L.d = __shfl_up_sync(0xffffffffu, row.d, s);
        R.a = __shfl_down_sync(0xffffffffu, row.a, s);
        R.c = __shfl_down_sync(0xffffffffu, row.c, s);
        R.d = __shfl_down_sync(0xffffffffu, row.d, s);
        row = tpcr_combine(row, L, lane >= s, R, lane + s <= HI);
    }
    return row;
}

struct TSweepArgs {
    uint32_t sc, su;         // shared addresses: line j, line j+1
    uint32_t tm;             // tensor-memory address of the warp's strip (column 0)
    uint32_t rowo, sw;       // byte offset of the thread's tensor row in a slot, its swizzle phase
    uint32_t layA, layB;     // shared addresses of the WLayer before / from the interface row on
    double hl;               // left r neighbour of the chunk at line j
    uint32_t hra;            // shared address of a 16-byte pair whose first double is the right r neighbour
    int i0v;                 // index of the thread's first node (made opaque per line, see the kernel)
    double g0, ezp, ezm;
    double gl0;              // geometric factor of the face i0 - 1/2 (0 in the chunk that starts with a Neumann r_in row)
    double fie15;            // capacity / rhs factor of row 15 (0 in the chunk that ends with a Neumann r_out row)
    double qsA, qsB;         // source term X (2)-(4),(22) of the two layers
    int ks;                  // interface row (18) of this chunk, < 0: none
    bool sqA, sqB;
    bool din, dout;          // the chunk starts / ends with a Dirichlet r-boundary row
    bool nin, last;          // the chunk starts with the Neumann r_in row / ends with the r_out row
    double rin_be, rout_f;
};

// what the reduced system needs from a thread's sweep
struct TSweepOut {
    double P, Q, S;          // x_first = P x_last + Q + S u
    double al, be, gm;       // last row: x_last = al x_next + be + gm u
};

// law coefficients of one row, read from the shared table (layer A before the interface row, layer B
// from it on: the face i* + 1/2 belongs to layer B, G14).  All lanes but the one that holds an
// interface node read the same address, so these are broadcast loads; fetching them per row keeps
// them out of the long-lived registers and needs no branch.
template <int DEGK>
struct TRowCoef {
    double K[DEGK + 1];
    double Ct[4];
};
template <int DEGK>
__device__ __forceinline__ TRowCoef<DEGK> trow_coef(uint32_t a)
{
    TRowCoef<DEGK> c;
    const double2 k01 = lds128(a);
    c.K[0] = k01.x; c.K[1] = k01.y;
    if (DEGK == 2) {
        c.K[2] = lds64(a + 16);
    } else {
        const double2 k23 = lds128(a + 16);
        c.K[2] = k23.x; c.K[3] = k23.y;
        c.K[DEGK] = lds64(a + 32);
    }
    const double2 c01 = lds128(a + 48), c23 = lds128(a + 64);
    c.Ct[0] = c01.x; c.Ct[1] = c01.y; c.Ct[2] = c23.x; c.Ct[3] = c23.y;
    return c;
}

// Four consecutive rows (13) P:L140-145 of one thread, assembled and pushed through the sweep (12)
// P:L133-136.  g = group (rows 4g .. 4g+3), runtime.
// GEN = false: regular rows of the layer whose coefficients sit in registers (c): the plain, fast body.
// GEN = true : the group may hold an interface row (18)-(20) P:L176-192 (row ks: the two face
//              coefficients become lam*_A, lam*_B, capacity and right-hand side vanish, and from it on
//              the rows are layer B's, G14) or an r-boundary row (15)-(17) P:L158-174 (a Neumann row
//              is an ordinary row with a zero face and zero capacity, a Dirichlet row is a select);
//              coefficients are read row by row from the shared table.  Still no branch per row.
// The caller picks the body per warp and group (warp-uniform), so the common case runs the plain body
// and the instruction cache holds four rows of each kind instead of sixteen.
// LASTG: 0 / 1 = this is not / is the group with row 15 (known at compile time: the one-line-per-CTA kernel
// peels the last group, so that the other three carry no selects for it), 2 = decided by g at run time (the
// smaller CTAs, where several CTAs per SM sit at different places of the code and its size matters more)
template <int DEGK, bool SQ, bool GEN, int LASTG>
__device__ __forceinline__ void tgroup(const TSweepArgs &A, int g, WCoef<DEGK> &c, SweepState &st, TSweepOut &o,
                                       double2 &tl, double lamA_if, double lamB_if, uint32_t spmask)
{
    TRaw8 fraw;
    tmem_ld8(A.tm + 96u + 8u * (uint32_t)g, fraw); // the four lower face fluxes of the group
    const uint32_t q0 = 2u * (uint32_t)g;
    const uint32_t o0 = A.rowo + (((q0) ^ A.sw) << 4), o1 = A.rowo + (((q0 + 1u) ^ A.sw) << 4);
    const uint32_t o2 = A.rowo + (((q0 + 2u) & 7u) ^ A.sw) * 16u;
    const double2 t1 = lds128(A.sc + o1);
    // rows 4g+4, 4g+5 (the next group's first pair); beyond the chunk: the right neighbour's pair (one select
    // on the address instead of four on the data); the line's last thread has none and mirrors its own node
    const bool lastg = (LASTG == 2) ? (g == 3) : (LASTG == 1);
    double2 t2 = lds128(lastg ? A.hra : A.sc + o2);
    if (GEN && lastg && A.last) t2.x = t1.y;
    const double2 u0 = lds128(A.su + o0), u1 = lds128(A.su + o1);
    const int ig = A.i0v + 4 * g; // node index of the group's first row; i -> double on the conversion unit, not the FP64 pipe
    const uint32_t ksw = (GEN && A.ks >= 0) ? (uint32_t)A.ks : 99u;
    tmem_wait_ld(fraw);
    double fD[4], cf[12], fu[4];
#pragma unroll
    for (int n = 0; n < 4; ++n) fD[n] = traw(fraw, n);
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const double T = (r == 0) ? tl.x : (r == 1) ? tl.y : (r == 2) ? t1.x : t1.y;
        const double Tr = (r == 0) ? tl.y : (r == 1) ? t1.x : (r == 2) ? t1.y : t2.x;
        const double Tu = (r == 0) ? u0.x : (r == 1) ? u0.y : (r == 2) ? u1.x : u1.y;
        const uint32_t k = 4u * (uint32_t)g + (uint32_t)r;
        const double fi = (double)(ig + r);
        double cfR, w, f, alk;
        // GEN: only the rows that are special in SOME lane of the warp (warp-uniform bit of spmask) take
        // the general code; the thread that holds the interface row switches its coefficients to layer B
        // there (the face i* + 1/2 already belongs to layer B, G14) and keeps them for the rest of the line
        if (!GEN || !((spmask >> k) & 1u)) {
            wrow2<DEGK, SQ>(c.K, c.Ct, c.qs, c.sq, T, Tr, Tu, fD[r], fi, fi, A.g0, A.ezp, A.ezm, cfR, w, f, fu[r]);
            sweep_row(st, cfR, w, f, alk);
        } else {
            const bool isif = (k == ksw);
            if (isif) {
                const TRowCoef<DEGK> cb = trow_coef<DEGK>(A.layB);
#pragma unroll
                for (int n = 0; n <= DEGK; ++n) c.K[n] = cb.K[n];
#pragma unroll
                for (int n = 0; n < 4; ++n) c.Ct[n] = cb.Ct[n];
                c.qs = A.qsB; c.sq = A.sqB;
            }
            double fie = fi;
            if (r == 3) fie = lastg ? A.fie15 : fie;
            fie = isif ? 0.0 : fie;
            wrow2<DEGK, SQ>(c.K, c.Ct, c.qs, c.sq, T, Tr, Tu, fD[r], fi, fie, A.g0, A.ezp, A.ezm, cfR, w, f, fu[r]);
            // (18) times h: -lam_A x_{i-1} + (lam_A + lam_B) x_i - lam_B x_{i+1} = 0 (new level, G7)
            double cfL_use = isif ? lamA_if : st.cfL;
            double cfR_use = isif ? lamB_if : cfR;
            if (r == 3) { // row 15: r_out row (15),(17): x_N = x_{N-1} (fie15 = 0, no right face) or x_N = value
                cfR_use = (lastg && A.last) ? 0.0 : cfR_use;
                cfL_use = (lastg && A.dout) ? 0.0 : cfL_use;
                w = (lastg && A.dout) ? 1.0 : w;
                f = (lastg && A.dout) ? A.rout_f : f;
            }
            st.cfL = cfL_use;
            sweep_row(st, cfR_use, w, f, alk);
            st.cfL = cfR; // face i + 1/2 as the next regular row sees it
            if (r == 0) { // row 0: r_in row (15),(16): alpha_0 = 1 exactly (T^_0 = T^_1 bitwise); Dirichlet: x_0 = value
                const bool g0_ = (g == 0);
                alk = (g0_ && A.nin) ? 1.0 : alk;
                alk = (g0_ && A.din) ? 0.0 : alk;
                st.om = (g0_ && A.din) ? 1.0 : st.om;
                st.be = (g0_ && A.din) ? A.rin_be : st.be;
                st.gm = (g0_ && A.din) ? 0.0 : st.gm;
            }
        }
        cf[3 * r] = alk; cf[3 * r + 1] = st.be; cf[3 * r + 2] = st.gm;
        // x_0 = P x_{k+1} + Q + S u (rows 0 .. 14)
        if (r < 3 || LASTG != 1) {
            const double Qn = fma(o.P, st.be, o.Q), Sn = fma(o.P, st.gm, o.S), Pn = o.P * alk;
            if (r < 3 || LASTG == 0) { o.Q = Qn; o.S = Sn; o.P = Pn; }
            else { o.Q = lastg ? o.Q : Qn; o.S = lastg ? o.S : Sn; o.P = lastg ? o.P : Pn; }
        }
    }
    tl = t2;
    const uint32_t tc = A.tm + 24u * (uint32_t)g;
#pragma unroll
    for (int n = 0; n < 12; ++n) tmem_st1(tc + 2u * (uint32_t)n, cf[n]);
#pragma unroll
    for (int n = 0; n < 4; ++n) tmem_st1(A.tm + 96u + 8u * (uint32_t)g + 2u * (uint32_t)n, fu[n]);
    o.al = cf[9]; o.be = cf[10]; o.gm = cf[11];
}

// Level 1 for one thread: the sixteen rows in four groups of four (a rolled loop); (alpha, beta,
// gamma) and the new face fluxes of a group go to tensor memory, the prefix products for the reduced
// row are carried along.  genmask: bit g set = group g of this warp needs the general body.
template <int DEGK, bool SQ, bool PEEL>
__device__ __forceinline__ TSweepOut tsweep16(const TSweepArgs &A, WCoef<DEGK> &c, uint32_t genmask, uint32_t spmask)
{
    SweepState st;
    st.om = 1.0; st.be = 0.0; st.gm = 1.0;
    TSweepOut o;
    o.P = 1.0; o.Q = 0.0; o.S = 0.0;
    // interface node: lam*_A, lam*_B at T_{i*,j} of the old level; the thread that holds one
    // starts every line with layer A's coefficients
    double lamA_if = 0.0, lamB_if = 0.0;
    if (A.ks >= 0) {
        const double Tk = lds64(A.sc + A.rowo + ((((uint32_t)A.ks >> 1) ^ A.sw) << 4) + (((uint32_t)A.ks & 1u) << 3));
        const TRowCoef<DEGK> ca = trow_coef<DEGK>(A.layA), cb = trow_coef<DEGK>(A.layB);
        lamA_if = wlam<DEGK, true>(ca.K, A.sqA, Tk + Tk);
        lamB_if = wlam<DEGK, true>(cb.K, A.sqB, Tk + Tk);
#pragma unroll
        for (int n = 0; n <= DEGK; ++n) c.K[n] = ca.K[n];
#pragma unroll
        for (int n = 0; n < 4; ++n) c.Ct[n] = ca.Ct[n];
        c.qs = A.qsA; c.sq = A.sqA;
    }
    double2 tl = lds128(A.sc + A.rowo + (A.sw << 4));
    st.cfL = wlam<DEGK, SQ>(c.K, c.sq, A.hl + tl.x) * A.gl0; // face i0 - 1/2
    if (PEEL) {
#pragma unroll 1
        for (int g = 0; g < 3; ++g) {
            if (!((genmask >> g) & 1u)) tgroup<DEGK, SQ, false, 0>(A, g, c, st, o, tl, lamA_if, lamB_if, 0u);
            else tgroup<DEGK, SQ, true, 0>(A, g, c, st, o, tl, lamA_if, lamB_if, spmask);
        }
        if (!((genmask >> 3) & 1u)) tgroup<DEGK, SQ, false, 1>(A, 3, c, st, o, tl, lamA_if, lamB_if, 0u);
        else tgroup<DEGK, SQ, true, 1>(A, 3, c, st, o, tl, lamA_if, lamB_if, spmask);
    } else {
#pragma unroll 1
        for (int g = 0; g < 4; ++g) {
            if (!((genmask >> g) & 1u)) tgroup<DEGK, SQ, false, 2>(A, g, c, st, o, tl, lamA_if, lamB_if, 0u);
            else tgroup<DEGK, SQ, true, 2>(A, g, c, st, o, tl, lamA_if, lamB_if, spmask);
        }
    }
    return o;
}

template <int WL, int NW, int DEGK>
__global__ void __launch_bounds__(32 * NW, 16 / NW) heat_tband_kernel(const __grid_constant__ WParams p)
{
    using Cfg = TBandCfg<WL, NW>;
    constexpr int CL = Cfg::CL, LPB = Cfg::LPB, WPL = Cfg::WPL, NS = Cfg::NS, SLOT = Cfg::SLOT;
    constexpr uint32_t FULL = 0xffffffffu;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char *gbase = smem_raw + (sbase - smem_u32(smem_raw));
    WLayer *lay = reinterpret_cast<WLayer *>(gbase + Cfg::OFF_LAY);
    volatile uint32_t *tmem_slot = reinterpret_cast<volatile uint32_t *>(gbase + Cfg::OFF_TMEM);

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
    const uint32_t halo_a = sbase + Cfg::OFF_HALO + (uint32_t)(warp * NS) * 32u;
    const uint32_t fbar_a = sbase + Cfg::OFF_FBAR + (uint32_t)(warp * NS) * 8u;
    const uint32_t xbar_a = sbase + Cfg::OFF_XBAR + (uint32_t)grp * 16u;
    const uint32_t ybar_a = sbase + Cfg::OFF_YBAR + (uint32_t)grp * 16u;
    const uint32_t ysep_a = sbase + Cfg::OFF_YSEP;
    const uint32_t pub_a = sbase + Cfg::OFF_PUB;
    // byte offsets of the thread's eight 16-byte chunks inside a SWIZZLE_128B slot, and of its two
    // r neighbours (last node of the row above, first node of the row below)
    uint32_t co[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) co[q] = (uint32_t)lane * 128u + (uint32_t)((q ^ (lane & 7)) << 4);
    const uint32_t hlo = (uint32_t)(lane - 1) * 128u + (uint32_t)((7 ^ ((lane - 1) & 7)) << 4) + 8u;
    const uint32_t hro = (uint32_t)(lane + 1) * 128u + (uint32_t)(((lane + 1) & 7) << 4);
    const bool has_l = (wig > 0), has_r = (wig < WL - 1); // the warp has a left / right neighbour warp

    // ---- law table scaled for this launch, barriers, tensor memory
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
#pragma unroll 1
        for (int s = 0; s < LPB * 2; ++s) mbar_init(sbase + Cfg::OFF_YBAR + 8u * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     ::"r"(sbase + (uint32_t)Cfg::OFF_TMEM), "n"(Cfg::TCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;
    // the warp's strip: lane quarter warp % 4, 128 columns per group of four warps
    const uint32_t tm = tmem_base + ((uint32_t)(warp & 3) << 21) + (uint32_t)(warp >> 2) * 128u;
    if (CL > 1) { cluster_arrive(); cluster_wait(); }
    // programmatic dependent launch: the set-up above overlaps the tail of the previous step
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    const int nz = p.nz, rpl = p.rpl, BL = p.BL, bpm = p.bands_per_member;
    const double g0 = p.g0;
    int i0v = i0;
    uint32_t qbase = 0;  // load sequence number of line offset -1 of this band
    uint32_t lcount = 0; // lines done (phase of the exchange barriers)

    // CTAs that share an SM work on different lines; start them out of phase so that one sweeps (FP64
    // pipe) while the other sits in its reduced system (latency)
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
        const bool rin_neu = (p.rin_om == 0.0), rout_neu = (p.rout_w == 0.0);
        TSweepArgs A;
        A.tm = tm; A.rowo = (uint32_t)lane * 128u; A.sw = (uint32_t)lane & 7u;
        A.layA = smem_u32(&lay[la]); A.layB = smem_u32(&lay[lb]);
        A.g0 = g0;
        A.gl0 = (first && rin_neu) ? 0.0 : fma(g0, (double)i0, -0.5 * g0);
        A.fie15 = (last && rout_neu) ? 0.0 : (double)(i0 + 15);
        A.qsA = lay[la].qsrc * q0b; A.qsB = lay[lb].qsrc * q0b;
        A.sqA = (lay[la].sq != 0); A.sqB = (lay[lb].sq != 0);
        A.ks = ks; A.din = first && !rin_neu; A.dout = last && !rout_neu; A.nin = first && rin_neu; A.last = last;
        A.rin_be = p.rin_be; A.rout_f = p.rout_f;
        const bool anysq = __any_sync(FULL, A.sqA || (ks >= 0 && A.sqB));
        WCoef<DEGK> c = wload_coef<DEGK>(lay[la], q0b); // the thread's current layer (A at the start of a line)
        // groups of four rows that need the general body: the one with the interface row, the first
        // group of the first chunk and the last group of the last chunk of the line
        const uint32_t genmask = __reduce_or_sync(FULL, (ks >= 0 ? (1u << (ks >> 2)) : 0u) | (first ? 1u : 0u) | (last ? 8u : 0u));
        // rows (0 .. 15) that are an interface row or an r-boundary row in some lane of this warp
        const uint32_t spmask = __reduce_or_sync(FULL, (ks >= 0 ? (1u << ks) : 0u) | (first ? 1u : 0u) | (last ? (1u << 15) : 0u));

        if (lane == 0) {
            const uint32_t npre = (uint32_t)min(NS, nl + 2);
            for (uint32_t s = 0; s < npre; ++s) issue_load(s);
        }
        wait_seq(0);
        wait_seq(1);

        // ---- prologue: the flux through the faces between lines j0 - 1 and j0, into tensor memory
        {
            const uint32_t sd = wbase + ((qbase + 0u) % (uint32_t)NS) * (uint32_t)SLOT;
            const uint32_t s1 = wbase + ((qbase + 1u) % (uint32_t)NS) * (uint32_t)SLOT;
#pragma unroll 1
            for (int g = 0; g < 4; ++g) {
                double fl[4];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int q = 2 * g + h;
                    const uint32_t oq = A.rowo + ((((uint32_t)q) ^ A.sw) << 4);
                    const double2 td = lds128(sd + oq);
                    const double2 tc = lds128(s1 + oq);
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int k = 2 * q + e;
                        const bool isB = (ks >= 0 && k >= ks);
                        const TRowCoef<DEGK> c = trow_coef<DEGK>(isB ? A.layB : A.layA);
                        const double a_ = e ? tc.y : tc.x, d_ = e ? td.y : td.x;
                        fl[2 * h + e] = wlam<DEGK, true>(c.K, isB ? A.sqB : A.sqA, a_ + d_) * (a_ - d_);
                    }
                }
                tmem_st4(tm + 96u + 8u * (uint32_t)g, fl[0], fl[1], fl[2], fl[3]);
            }
            tmem_wait_st();
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
            asm volatile("" : "+r"(i0v)); // keep the per-row geometry out of registers across lines
            wait_seq((uint32_t)(L + 2));

            // ---- the two r neighbours of the thread's 16 nodes at line j
            // (one load through a selected address: three branches would diverge between lane 0 and the rest)
            const double hl = lds64((lane > 0) ? sc + hlo : has_l ? halo_a + qs * 32u + 8u : sc + co[0]);
            A.hra = (lane < 31) ? sc + hro : has_r ? halo_a + qs * 32u + 16u : sc + co[7];

            // ---- level 1: assemble (13)/(15)/(18) and sweep (12) the thread's 16 rows
            A.sc = sc; A.su = su; A.hl = hl; A.i0v = i0v; A.ezp = ezp; A.ezm = ezm;
            constexpr bool PEEL = (NW == 16);
            const TSweepOut o = anysq ? tsweep16<DEGK, true, PEEL>(A, c, genmask, spmask) : tsweep16<DEGK, false, PEEL>(A, c, genmask, spmask);
            tmem_wait_st();
            // the slot of line j - 1 has been stored (its TMA store was issued a whole sweep ago): refill it
            if (lane == 0 && L >= 1 && L + NS <= nl + 1) { tma_wait_read0(); issue_load((uint32_t)(L + NS)); }

            // ---- reduced row of this thread: a*y_{t-1} + y_t + c*y_{t+1} = d  (y = x of the last row)
            double Pn = __shfl_down_sync(FULL, o.P, 1);
            double Qn = __shfl_down_sync(FULL, o.Q, 1);
            double Sn = __shfl_down_sync(FULL, o.S, 1);
            if (lane == 31) { Pn = 0.0; Qn = 0.0; Sn = 0.0; }
            Row3 row;
            {
                const double r = rcp_cubic(fma(-o.al, Sn, 1.0));
                row.a = -o.gm * r;
                row.c = -o.al * Pn * r;
                row.d = fma(o.al, Qn, o.be) * r;
            }
            double y, u;
            if constexpr (WL == 1) {
                // the whole line is this warp: PCR over all 32 reduced rows
                row = tpcr_lanes<false, 31>(row, lane);
                y = row.d;
                u = __shfl_up_sync(FULL, y, 1);
                if (lane == 0) u = 0.0;
            } else {
                // ---- level 2: PCR over lanes 0..30; lane 31 is the warp's separator
                const Row3 rp = tpcr_lanes<NW == 16, 30>(row, lane);
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
                // one warp of the CTA (in turn) solves the separator rows for all the others
                const bool duty = ((uint32_t)wl == lcount % (uint32_t)WPL);
                const uint32_t ysl = ysep_a + (uint32_t)((pubpar * LPB + grp) * WL) * 8u;
                if (duty && lane == 1) mbar_expect_tx(pbar, (uint32_t)(WL * Cfg::PUB * 8));
                if (lane == 0 || lane == 31) {
                    const uint32_t s6 = pub0 + (uint32_t)(wig * Cfg::PUB) * 8u + (lane == 31 ? 48u : 0u);
                    const double v0 = lane == 31 ? o.al : o.P, v1 = lane == 31 ? o.be : o.Q, v2 = lane == 31 ? o.gm : o.S;
                    const double v3 = lane == 31 ? r30.a : rp.a, v4 = lane == 31 ? r30.c : rp.c, v5 = lane == 31 ? r30.d : rp.d;
#pragma unroll
                    for (int rk = 0; rk < CL; ++rk) {
                        const uint32_t ra = map_to_rank(s6, (uint32_t)rk), rb = map_to_rank(pbar, (uint32_t)rk);
                        st_async_v2(ra, v0, v1, rb);
                        st_async_v2(ra + 16, v2, v3, rb);
                        st_async_v2(ra + 32, v4, v5, rb);
                    }
                }
                double Vs, U;
                if (duty) {
                    while (!mbar_try_wait(pbar, (lcount >> 1) & 1u)) {}
                    // ---- level 3: build the WL separator rows and solve them (PCR over WL lanes)
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
                    // the separators are 512 rows apart: on diagonally dominant lines their mutual couplings
                    // have decayed far below rounding (|a|, |c| < 2^-80 means a dropped term is below
                    // 1e-24 |y|, i.e. < 1e-9 ulp), and then x = d already; otherwise PCR over WL lanes
                    if (__any_sync(FULL, in3 && (fabs(s3.a) > 8.271806125530277e-25 || fabs(s3.c) > 8.271806125530277e-25)))
                        s3 = pcr_segment_rolled<WL>(s3, s, 0, WL - 1);
                    if (in3) sts64(ysl + 8u * (uint32_t)lane, s3.d);
                    __syncwarp();
                    if (lane == 0) asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(ybar_a + 8u * pubpar) : "memory");
                    Vs = __shfl_sync(FULL, s3.d, wig);
                    U = __shfl_sync(FULL, s3.d, (wig + WL - 1) % WL);
                } else {
                    while (!mbar_try_wait(ybar_a + 8u * pubpar, (lcount >> 1) & 1u)) {}
                    Vs = lds64(ysl + 8u * (uint32_t)wig);
                    U = lds64(ysl + 8u * (uint32_t)((wig + WL - 1) % WL));
                }
                if (wig == 0) U = 0.0;
                y = (lane == 31) ? Vs : fma(-rp.c, Vs, fma(-rp.a, U, rp.d));
                u = __shfl_up_sync(FULL, y, 1);
                if (lane == 0) u = U;
            }
            ++lcount;

            // ---- back substitution (14) P:L150 with (alpha, beta, gamma) read back from tensor memory,
            //      eight rows per wait; the new level replaces line j in its slot
            double xn = y; // x_{k+1}
#pragma unroll
            for (int hh = 1; hh >= 0; --hh) {
                TRaw16 cr[3];
#pragma unroll
                for (int n = 0; n < 3; ++n) tmem_ld16(tm + (uint32_t)(48 * hh + 16 * n), cr[n]);
                tmem_wait_ld16(cr[0], cr[1], cr[2]);
                double xs[8];
#pragma unroll
                for (int r = 7; r >= 0; --r) {
                    // row k = 8 hh + r: its (al, be, gm) are doubles 3r, 3r+1, 3r+2 of the 24 loaded
                    const int k = 8 * hh + r;
                    const double a_ = traw16(cr[(3 * r) >> 3], (3 * r) & 7);
                    const double b_ = traw16(cr[(3 * r + 1) >> 3], (3 * r + 1) & 7);
                    const double g_ = traw16(cr[(3 * r + 2) >> 3], (3 * r + 2) & 7);
                    xs[r] = (k == 15) ? y : fma(a_, xn, fma(g_, u, b_));
                    xn = xs[r];
                }
#pragma unroll
                for (int q2 = 0; q2 < 4; ++q2) sts128(sc + co[4 * hh + q2], xs[2 * q2], xs[2 * q2 + 1]);
            }
            fence_proxy_async();
            __syncwarp();

            // ---- the warp's own TMA store of its 4 KB of the new level; Neumann z lines copy their
            //      neighbour (reading G16)
            if (lane == 0) {
                const int Rg = (b * nz + j) * rpl + wig * 32;
                tma_store_2d(&p.tm_st, 0, Rg, sc);
                if (j == 1 || j == nz - 2) { // the edge lines of the grid
                    if (j == 1 && p.z_lo_neumann) tma_store_2d(&p.tm_st, 0, Rg - rpl, sc);
                    if (j == nz - 2 && p.z_hi_neumann) tma_store_2d(&p.tm_st, 0, Rg + rpl, sc);
                    // z-slab run: the neighbour slabs' halo lines get this slab's edge lines over NVLink / peer memory
                    if (j == 1 && p.peer_lo_row >= 0) tma_store_2d(&p.tm_peer_lo, 0, p.peer_lo_row + b * p.peer_lo_rpm + wig * 32, sc);
                    if (j == nz - 2 && p.peer_hi_row >= 0) tma_store_2d(&p.tm_peer_hi, 0, p.peer_hi_row + b * p.peer_hi_rpm + wig * 32, sc);
                }
                tma_commit();
            }

            // ---- probes: T of the new level at (i_p, j_p)
            if (p.probe_out != nullptr) {
                for (int pq = 0; pq < p.nprobes; ++pq) {
                    const ProbeSrc ps = p.probes[pq];
                    if (ps.i < i0 || ps.i >= i0 + 16) continue;
                    if (ps.is_static) {
                        if (j == 1) p.probe_out[b * p.nprobes + pq] = p.Told[((size_t)b * nz + ps.j_store) * p.nr + ps.i];
                    } else if (ps.j_src == j) {
                        const uint32_t kk = (uint32_t)(ps.i - i0); // the value just written into the slot
                        p.probe_out[b * p.nprobes + pq] = lds64(sc + (uint32_t)lane * 128u + ((((kk >> 1) ^ ((uint32_t)lane & 7u))) << 4) + ((kk & 1u) << 3));
                    }
                }
            }
        }
        if (lane == 0) tma_wait_read0(); // the next band's loads reuse the slots
        __syncwarp();
        qbase += (uint32_t)(nl + 2);
    }
    if (lane == 0) tma_wait_all0();
    // every warp is done with its strip before warp 0 gives the tensor memory back
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(Cfg::TCOLS) : "memory");
    if (CL > 1) { cluster_arrive(); cluster_wait(); }
}

} // namespace heat

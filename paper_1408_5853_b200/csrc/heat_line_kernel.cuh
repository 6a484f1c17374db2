// heat_line_kernel.cuh -- the fused time-step kernel (property evaluation + explicit axial
// flux + source + row assembly + batched tridiagonal line solve), SURVEY 8(a) rows a1-a5.
//
// Decomposition (differs from the paper's one-work-item-per-line OpenCL kernel):
// a z-line of nr nodes is owned by a GROUP of G threads, M consecutive nodes per thread.
//   level 1 (thread) : Thomas forward sweep (12) on the thread's M rows, carrying the
//                      dependence on the unknown left neighbour u = x_{i0-1} as a third
//                      sweep coefficient:  x_k = alpha_k x_{k+1} + beta_k + gamma_k u.
//                      The same pass accumulates x_first = P y + Q + S u (y = x_last), so
//                      each thread contributes ONE row to a reduced tridiagonal system in y.
//   level 2 (warp)   : parallel cyclic reduction over the 32 reduced rows with shuffles;
//                      in a multi-warp group lane 31 is a separator that stays out of it.
//   level 3 (group)  : the <= 32 separator rows go through shared memory and one warp
//                      solves them with PCR.
//   back substitution: (14) x_k = alpha_k x_{k+1} + (beta_k + gamma_k u); T^ written once.
// The sweep coefficients never leave the SM (shared memory), so HBM sees 8 B read + 8 B
// written per cell-update.
#pragma once
#include <cooperative_groups.h>
#include "heat_device.cuh"

namespace heat {

struct Row3 {
    double a, c, d; // a*x_left + x + c*x_right = d
};

// One PCR elimination of `me` against its left / right neighbour rows (all normalised).
__device__ __forceinline__ Row3 pcr_combine(const Row3 &me, const Row3 &L, bool vl, const Row3 &R, bool vr)
{
    const double cl = vl ? L.c : 0.0, dl = vl ? L.d : 0.0;
    const double ar = vr ? R.a : 0.0, dr = vr ? R.d : 0.0;
    double den = fma(-me.a, cl, 1.0);
    den = fma(-me.c, ar, den);
    const double r = rcp_cubic(den);
    double d = fma(-me.a, dl, me.d);
    d = fma(-me.c, dr, d);
    Row3 o;
    o.d = d * r;
    const double ar_ = me.a * r, cr_ = me.c * r;
    o.a = vl ? -ar_ * L.a : ar_; // an external reference keeps its coefficient
    o.c = vr ? -cr_ * R.c : cr_;
    return o;
}

// PCR over lanes lo..hi (lane indices relative to a WIDTH-lane segment).  Rows outside keep
// their value.  On exit row i reads a_i*U + x_i + c_i*V = d_i where U / V are the unknowns
// left of lane lo / right of lane hi (coefficients exactly 0 if there are none).
template <int WIDTH>
__device__ __forceinline__ Row3 pcr_segment(Row3 row, int lane, int lo, int hi)
{
#pragma unroll
    for (int s = 1; s < WIDTH; s <<= 1) {
        Row3 L, R;
        L.a = __shfl_up_sync(0xffffffffu, row.a, s, WIDTH);
        L.c = __shfl_up_sync(0xffffffffu, row.c, s, WIDTH);
        L.d = __shfl_up_sync(0xffffffffu, row.d, s, WIDTH);
        R.a = __shfl_down_sync(0xffffffffu, row.a, s, WIDTH);
        R.c = __shfl_down_sync(0xffffffffu, row.c, s, WIDTH);
        R.d = __shfl_down_sync(0xffffffffu, row.d, s, WIDTH);
        const bool in = (lane >= lo) && (lane <= hi);
        const bool vl = in && (lane - s >= lo);
        const bool vr = in && (lane + s <= hi);
        const Row3 n = pcr_combine(row, L, vl, R, vr);
        if (in) row = n;
    }
    return row;
}

template <int M, int G, int TPBMIN = 256>
struct LineCfg {
    static constexpr int TPB = (G > TPBMIN) ? G : TPBMIN;
    static constexpr int LPB = TPB / G;               // lines in flight per block
    static constexpr int WG = (G >= 32) ? G / 32 : 1; // warps per group
    static constexpr bool MULTI = (G > 32);
    static constexpr int SEG = (G >= 32) ? 32 : G;    // shuffle segment width
    static constexpr int NW = TPB / 32;
    // shared: sweep state 3*M*TPB doubles, exchange 10*NW doubles, layer table
    static constexpr size_t smem_bytes(int nlayers)
    {
        return sizeof(double) * (size_t)(3 * M * TPB + 10 * NW) + sizeof(DLayer) * (size_t)nlayers;
    }
};

// field loads: read-only path for a one-step launch; for the persistent multi-step kernel the level
// read in step k was written in step k-1 of the same launch, so it must come from L2 (ld.global.cg)
// COH = 2: the field lives in shared memory (single-CTA kernel): plain loads through generic pointers
template <int COH, typename T>
__device__ __forceinline__ T ldT(const T *ptr)
{
    if (COH == 0) return __ldg(ptr);
    if (COH == 1) return __ldcg(ptr);
    return *ptr;
}

// One solver step of the lines this CTA owns (grid-stride over groups of LPB lines).
// IT = true: the iterated variant (heat_step_picard, reading G23): lambda, c_V and X are
// evaluated at the field Tcf (the previous iterate of the new level) instead of the current level,
// which stays where (8) has it: rho c_V (T^ - T)/tau and Lambda_j[T].
template <int M, int G, int COH, int TPBMIN = 256, bool IT = false>
__device__ __forceinline__ void line_step(const KParams &p, const double *Told, double *Tnew, double inv_tau_k, double amp_k,
                                          double *probe_out, double *st, double *xch, const DLayer *lay,
                                          const double *Tcf = nullptr)
{
    using Cfg = LineCfg<M, G, TPBMIN>;
    constexpr int TPB = Cfg::TPB;
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const int grp = tid / G;   // group within the block
    const int t = tid % G;     // thread within the group
    const int i0 = t * M;      // first node of this thread
    const int wig = t >> 5;    // warp within the group
    const int gw0 = (grp * G) >> 5; // first warp of the group (MULTI only)
    const int nr = p.nr, nz = p.nz;
    const bool stepped = (p.j_step > 0);
    const bool vec_ok = ((nr & 1) == 0) && !stepped; // the step may fall between the two nodes of a pair
    const int interior = nz - 2;

    for (int base = blockIdx.x * Cfg::LPB; base < p.total_lines; base += gridDim.x * Cfg::LPB) {
        int Lidx = base + grp;
        const bool live = Lidx < p.total_lines;
        if (!live) Lidx = p.total_lines - 1; // duplicate work keeps shuffles / barriers uniform
        const int b = Lidx / interior;
        const int j = 1 + (Lidx - b * interior);
        const size_t line = ((size_t)b * nz + j) * (size_t)nr;
        const double *Tl = Told + line;
        const double *Tm = Tl - nr;
        const double *Tp = Tl + nr;
        const bool upper = stepped && j > p.j_step; // a line above the step: N_j = i_step
        const double *ga = (upper ? p.ga2 : p.ga) + (size_t)b * p.nrp + i0;
        const double *gc = (upper ? p.gc2 : p.gc) + (size_t)b * p.nrp + i0;
        const uint32_t *info = (upper ? p.info2 : p.info) + (size_t)b * p.nrp + i0;

        // ---- load line j (current level) for the thread's nodes, plus the halo
        double Tc[M + 2];
        if (vec_ok) {
#pragma unroll
            for (int k = 0; k < M; k += 2) {
                double2 v = make_double2(1.0, 1.0);
                if (i0 + k < nr) v = ldT<COH>(reinterpret_cast<const double2 *>(Tl + i0 + k));
                Tc[k + 1] = v.x; Tc[k + 2] = v.y;
            }
        } else {
#pragma unroll
            for (int k = 0; k < M; ++k) Tc[k + 1] = (i0 + k < nr) ? ldT<COH>(Tl + i0 + k) : 1.0;
        }
        Tc[0] = (i0 > 0 && i0 - 1 < nr) ? ldT<COH>(Tl + i0 - 1) : 1.0;
        Tc[M + 1] = (i0 + M < nr) ? ldT<COH>(Tl + i0 + M) : 1.0;

        // ---- the same nodes of the field the laws are evaluated at (iterated variant only)
        double Sc[IT ? M + 2 : 1];
        const double *Sl = IT ? Tcf + line : Tl;
        if (IT) {
#pragma unroll
            for (int k = 0; k < M; ++k) Sc[k + 1] = (i0 + k < nr) ? ldT<COH>(Sl + i0 + k) : 1.0;
            Sc[0] = (i0 > 0 && i0 - 1 < nr) ? ldT<COH>(Sl + i0 - 1) : 1.0;
            Sc[IT ? M + 1 : 0] = (i0 + M < nr) ? ldT<COH>(Sl + i0 + M) : 1.0;
        }

        const double ezm = __ldg(p.ezm + j), ezp = __ldg(p.ezp + j);
        const double qa = __ldg(p.Q0 + b) * amp_k; // Q0 nu(t_k) p^2(t_k), (2)-(4),(22)
        const double inv_tau = inv_tau_k;
        const int fm = p.face_mode;

        // ---- level 1: assemble each row (13)/(15)/(18) and sweep it (12) at once
        double al = 0.0, be = 0.0, gm = 1.0; // alpha_{k-1}, beta_{k-1}, gamma_{k-1}
        double P = 0.0, Q = 0.0, S = 0.0;
        double2 Tdn2 = make_double2(1.0, 1.0), Tup2 = Tdn2;
#pragma unroll
        for (int k = 0; k < M; ++k) {
            // lines j-1 and j+1 at this node (pairwise 16-byte loads where alignment allows)
            if (vec_ok) {
                if ((k & 1) == 0) {
                    double2 vm = make_double2(1.0, 1.0), vp = vm;
                    if (i0 + k < nr) {
                        vm = ldT<COH>(reinterpret_cast<const double2 *>(Tm + i0 + k));
                        vp = ldT<COH>(reinterpret_cast<const double2 *>(Tp + i0 + k));
                    }
                    Tdn2 = vm; Tup2 = vp;
                }
            } else {
                const bool ok = i0 + k < nr;
                const double vm = ok ? ldT<COH>(Tm + i0 + k) : 1.0, vp = ok ? ldT<COH>(Tp + i0 + k) : 1.0;
                if ((k & 1) == 0) { Tdn2.x = vm; Tup2.x = vp; } else { Tdn2.y = vm; Tup2.y = vp; }
            }
            const double Tdn_k = (k & 1) ? Tdn2.y : Tdn2.x;
            const double Tup_k = (k & 1) ? Tup2.y : Tup2.x;
            double Sdn_k = Tdn_k, Sup_k = Tup_k;
            if (IT) {
                const bool ok = i0 + k < nr;
                Sdn_k = ok ? ldT<COH>(Sl - nr + i0 + k) : 1.0;
                Sup_k = ok ? ldT<COH>(Sl + nr + i0 + k) : 1.0;
            }
            const uint32_t nf = __ldg(info + k);
            const double gak = __ldg(ga + k), gck = __ldg(gc + k);
            const uint32_t kind = nf & 3u;
            double A, B, C, F;
            if (kind == NK_FIXED) {
                A = gak; B = 1.0; C = gck; F = p.fixF[(nf >> 2) & 3u];
            } else if (kind == NK_KEEP) {
                A = 0.0; B = 1.0; C = 0.0; F = Tc[k + 1]; // outside Omega: the node keeps its value
            } else {
                const DLayer &mL = lay[(nf >> 8) & 0xffu];
                const DLayer &mR = lay[(nf >> 16) & 0xffu];
                const double T = Tc[k + 1];
                const double Ts = IT ? Sc[IT ? k + 1 : 0] : T;         // where the laws are evaluated
                const double TsL = IT ? Sc[IT ? k : 0] : Tc[k], TsR = IT ? Sc[IT ? k + 2 : 0] : Tc[k + 2];
                const bool reg = (kind == NK_REG);
                // lambda_{i-1/2,j}, lambda_{i+1/2,j} P:L127; at an interface node
                // lambda*_m = lambda_m(T_{i*,j}), lambda*_{m+1} = lambda_{m+1}(T_{i*,j}) P:L183
                const double lamL = law_face(mL.k, Ts, reg ? TsL : Ts, fm);
                const double lamR = law_face(mR.k, Ts, reg ? TsR : Ts, fm);
                A = -gak * lamL;
                C = -gck * lamR;
                if (reg) {
                    const double W = law_at(mL.rc, Ts) * inv_tau;      // rho c_V / tau
                    const double lamU = law_face(mL.k, Ts, Sup_k, fm); // lambda_{i,j+1/2}
                    const double lamD = law_face(mL.k, Ts, Sdn_k, fm); // lambda_{i,j-1/2}
                    // Lambda_j[T] (11) P:L125
                    double Lj = ezp * (lamU * (Tup_k - T));
                    Lj = fma(-ezm, lamD * (T - Tdn_k), Lj);
                    F = fma(W, T, Lj);
                    if (mL.heater && qa != 0.0) F = fma(qa, law_at(mL.src, Ts), F);
                    B = W - A - C;
                } else {
                    B = -A - C; // (18) P:L178-181 at the new level (reading G7), scaled by h_i h_{i+1}
                    F = 0.0;
                }
            }
            // sweep (12) P:L133-136, with the left-neighbour dependence gamma
            const double den = fma(A, al, B);
            const double inv = rcp_nr(den);
            const double tA = A * inv;
            al = -C * inv;
            be = fma(-tA, be, F * inv);
            gm = -tA * gm;
            st[(0 * M + k) * TPB + tid] = al;
            st[(1 * M + k) * TPB + tid] = be;
            st[(2 * M + k) * TPB + tid] = gm;
            if (k == 0) {
                P = al; Q = be; S = gm;
            } else if (k < M - 1) {
                Q = fma(P, be, Q);
                S = fma(P, gm, S);
                P = P * al;
            }
        }

        // ---- reduced row of this thread:  -gm*y_{t-1} + (1 - al*S')*y_t - al*P'*y_{t+1} = be + al*Q'
        double Pn = __shfl_down_sync(0xffffffffu, P, 1, Cfg::SEG);
        double Qn = __shfl_down_sync(0xffffffffu, Q, 1, Cfg::SEG);
        double Sn = __shfl_down_sync(0xffffffffu, S, 1, Cfg::SEG);
        if (Cfg::MULTI) {
            if (lane == 0) { xch[0 * Cfg::NW + warp] = P; xch[1 * Cfg::NW + warp] = Q; xch[2 * Cfg::NW + warp] = S; }
        }
        const bool last_t = (t == G - 1);
        const bool seg_last = Cfg::MULTI ? (lane == 31) : last_t;
        if (seg_last) { Pn = 0.0; Qn = 0.0; Sn = 0.0; } // lane 31 of a multi-warp group is fixed up below
        Row3 row;
        {
            const double r = rcp_nr(fma(-al, Sn, 1.0));
            row.a = -gm * r;
            row.c = -al * Pn * r;
            row.d = fma(al, Qn, be) * r;
        }

        double y, u;
        if (!Cfg::MULTI) {
            // ---- level 2 only: the whole line sits in one shuffle segment
            const int sl = t; // lane within the segment
            row = pcr_segment<Cfg::SEG>(row, sl, 0, G - 1);
            y = row.d;
            u = __shfl_up_sync(0xffffffffu, y, 1, Cfg::SEG);
            if (t == 0) u = 0.0;
        } else {
            // ---- level 2: PCR over lanes 0..30, lane 31 is the warp's separator
            Row3 rp = pcr_segment<32>(row, lane, 0, 30);
            if (lane == 0) { xch[3 * Cfg::NW + warp] = rp.a; xch[4 * Cfg::NW + warp] = rp.c; xch[5 * Cfg::NW + warp] = rp.d; }
            Row3 r30;
            r30.a = __shfl_sync(0xffffffffu, rp.a, 30);
            r30.c = __shfl_sync(0xffffffffu, rp.c, 30);
            r30.d = __shfl_sync(0xffffffffu, rp.d, 30);
            __syncthreads();
            if (lane == 31) {
                const bool has_next = (wig + 1 < Cfg::WG);
                Row3 nx;
                nx.a = nx.c = nx.d = 0.0;
                double Pw = 0.0, Qw = 0.0, Sw = 0.0;
                if (has_next) {
                    Pw = xch[0 * Cfg::NW + warp + 1]; Qw = xch[1 * Cfg::NW + warp + 1]; Sw = xch[2 * Cfg::NW + warp + 1];
                    nx.a = xch[3 * Cfg::NW + warp + 1]; nx.c = xch[4 * Cfg::NW + warp + 1]; nx.d = xch[5 * Cfg::NW + warp + 1];
                }
                Row3 me;
                const double r = rcp_nr(fma(-al, Sw, 1.0));
                me.a = -gm * r;
                me.c = -al * Pw * r;
                me.d = fma(al, Qw, be) * r;
                // separator row: eliminate lane 30 (own warp) and lane 0 of the next warp
                const Row3 sep = pcr_combine(me, r30, true, nx, has_next);
                xch[6 * Cfg::NW + warp] = sep.a; xch[7 * Cfg::NW + warp] = sep.c; xch[8 * Cfg::NW + warp] = sep.d;
            }
            __syncthreads();
            // ---- level 3: the group's first warp solves the WG separator rows
            if (wig == 0) {
                Row3 s3;
                const bool in3 = lane < Cfg::WG;
                s3.a = in3 ? xch[6 * Cfg::NW + gw0 + lane] : 0.0;
                s3.c = in3 ? xch[7 * Cfg::NW + gw0 + lane] : 0.0;
                s3.d = in3 ? xch[8 * Cfg::NW + gw0 + lane] : 0.0;
                s3 = pcr_segment<(Cfg::WG > 1 ? Cfg::WG : 2)>(s3, lane & (Cfg::WG - 1), 0, Cfg::WG - 1);
                if (in3) xch[9 * Cfg::NW + gw0 + lane] = s3.d;
            }
            __syncthreads();
            const double Vs = xch[9 * Cfg::NW + warp];
            const double U = (wig > 0) ? xch[9 * Cfg::NW + warp - 1] : 0.0;
            y = (lane == 31) ? Vs : fma(-rp.c, Vs, fma(-rp.a, U, rp.d));
            u = __shfl_up_sync(0xffffffffu, y, 1);
            if (lane == 0) u = U;
        }

        // ---- back substitution (14) P:L150
        double x[M];
        x[M - 1] = y;
#pragma unroll
        for (int k = M - 2; k >= 0; --k) {
            const double a_ = st[(0 * M + k) * TPB + tid];
            const double b_ = st[(1 * M + k) * TPB + tid];
            const double g_ = st[(2 * M + k) * TPB + tid];
            x[k] = fma(a_, x[k + 1], fma(g_, u, b_));
        }

        // ---- store T^ (and the Neumann z lines, which copy their neighbour; reading G16)
        if (live) {
            double *out = Tnew + line;
            const bool lo = (j == 1) && p.z_lo_neumann;
            const bool hi = (j == nz - 2) && p.z_hi_neumann;
            if (vec_ok) {
#pragma unroll
                for (int k = 0; k < M; k += 2) {
                    if (i0 + k < nr) {
                        const double2 v = make_double2(x[k], x[k + 1]);
                        *reinterpret_cast<double2 *>(out + i0 + k) = v;
                        if (lo) *reinterpret_cast<double2 *>(out - nr + i0 + k) = v;
                        if (hi) *reinterpret_cast<double2 *>(out + nr + i0 + k) = v;
                    }
                }
            } else {
#pragma unroll
                for (int k = 0; k < M; ++k) {
                    if (i0 + k < nr) {
                        // stepped domain: the nodes above the step face mirror line j_step (no flux through
                        // the face, as a Neumann z line G16); line j_step + 1 itself leaves them alone
                        const bool beyond = stepped && (i0 + k > p.i_step);
                        if (!(beyond && j == p.j_step + 1)) out[i0 + k] = x[k];
                        if (beyond && j == p.j_step) out[i0 + k + nr] = x[k];
                        if (lo) out[i0 + k - nr] = x[k];
                        if (hi) out[i0 + k + nr] = x[k];
                    }
                }
            }
            // ---- z-slab run: the neighbour slabs' halo lines get this slab's edge lines (peer stores)
            if ((j == 1 && p.peer_lo != nullptr) || (j == nz - 2 && p.peer_hi != nullptr)) {
#pragma unroll
                for (int k = 0; k < M; ++k) {
                    if (i0 + k < nr) {
                        if (j == 1 && p.peer_lo != nullptr) p.peer_lo[(long long)b * p.peer_lo_stride + i0 + k] = x[k];
                        if (j == nz - 2 && p.peer_hi != nullptr) p.peer_hi[(long long)b * p.peer_hi_stride + i0 + k] = x[k];
                    }
                }
            }
            // ---- probes: T of the new level at (i_p, j_p)
            if (probe_out != nullptr) {
                for (int q = 0; q < p.nprobes; ++q) {
                    const ProbeSrc ps = p.probes[q];
                    if (ps.i < i0 || ps.i >= i0 + M) continue;
                    if (ps.is_static) {
                        if (j == 1) probe_out[b * p.nprobes + q] = Told[((size_t)b * nz + ps.j_store) * nr + ps.i];
                    } else if (ps.j_src == j) {
                        double v = 0.0;
#pragma unroll
                        for (int k = 0; k < M; ++k)
                            if (i0 + k == ps.i) v = x[k];
                        probe_out[b * p.nprobes + q] = v;
                    }
                }
            }
        }
        if (Cfg::MULTI) __syncthreads(); // xch is reused by the next line
    }
}

template <int M, int G>
__global__ void __launch_bounds__(LineCfg<M, G>::TPB) heat_line_kernel(const __grid_constant__ KParams p)
{
    using Cfg = LineCfg<M, G>;
    constexpr int TPB = Cfg::TPB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *st = reinterpret_cast<double *>(smem_raw); // [3][M][TPB]
    double *xch = st + 3 * M * TPB;                    // [10][NW]
    DLayer *lay = reinterpret_cast<DLayer *>(xch + 10 * Cfg::NW);
    for (int q = threadIdx.x; q < p.nlayers * (int)(sizeof(DLayer) / sizeof(int)); q += TPB)
        reinterpret_cast<int *>(lay)[q] = reinterpret_cast<const int *>(p.layers)[q];
    __syncthreads();
    line_step<M, G, 0>(p, p.Told, p.Tnew, p.inv_tau, p.amp, p.probe_out, st, xch, lay);
}

// (tau_k, amplitude_k) of solver step s from integer counters only: (4) P:L79 and (22) + procedure
// P:L212-217 (readings G8, G9, G18); the device twin of heat_schedule in heat_api.cu.
__device__ __forceinline__ void dev_schedule(const DSched &d, long long s, double &inv_tau, double &amp)
{
    if (d.P <= 0 || d.S <= 0) { inv_tau = d.inv_dt; amp = 0.0; return; }
    if (d.nsub > 0) {
        const long long len = (long long)d.nsub + d.P - 1; // solver steps per period
        const long long q = s % len;
        if (q < d.nsub) { inv_tau = d.inv_dt_sub; amp = d.amp_sub[q]; }
        else { const long long g = q - d.nsub + 1; inv_tau = d.inv_dt; amp = (g < d.S) ? 1.0 : 0.0; }
    } else {
        inv_tau = d.inv_dt; amp = ((s % d.P) < d.S) ? 1.0 : 0.0;
    }
}

// One iteration of the iterated variant (heat_step_picard): as heat_line_kernel with the laws at p.Tcoef.
template <int M, int G>
__global__ void __launch_bounds__(LineCfg<M, G>::TPB) heat_line_iter_kernel(const __grid_constant__ KParams p)
{
    using Cfg = LineCfg<M, G>;
    constexpr int TPB = Cfg::TPB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *st = reinterpret_cast<double *>(smem_raw); // [3][M][TPB]
    double *xch = st + 3 * M * TPB;                    // [10][NW]
    DLayer *lay = reinterpret_cast<DLayer *>(xch + 10 * Cfg::NW);
    for (int q = threadIdx.x; q < p.nlayers * (int)(sizeof(DLayer) / sizeof(int)); q += TPB)
        reinterpret_cast<int *>(lay)[q] = reinterpret_cast<const int *>(p.layers)[q];
    __syncthreads();
    line_step<M, G, 0, 256, true>(p, p.Told, p.Tnew, p.inv_tau, p.amp, p.probe_out, st, xch, lay, p.Tcoef);
}

// Persistent multi-step version for grids whose CTAs are all resident (cooperative launch): the
// schedule runs on the device, the two levels swap roles every step, a grid-wide barrier separates the
// steps.  One launch advances p.nsteps solver steps; this is what removes the launch latency that
// dominates small grids (the paper's own Table 4 shows the same flat per-step cost).
template <int M, int G>
__global__ void __launch_bounds__(LineCfg<M, G>::TPB) heat_line_persist_kernel(const __grid_constant__ KParams p)
{
    using Cfg = LineCfg<M, G>;
    constexpr int TPB = Cfg::TPB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *st = reinterpret_cast<double *>(smem_raw);
    double *xch = st + 3 * M * TPB;
    DLayer *lay = reinterpret_cast<DLayer *>(xch + 10 * Cfg::NW);
    for (int q = threadIdx.x; q < p.nlayers * (int)(sizeof(DLayer) / sizeof(int)); q += TPB)
        reinterpret_cast<int *>(lay)[q] = reinterpret_cast<const int *>(p.layers)[q];
    __syncthreads();
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const size_t rec = (size_t)p.batch * (size_t)p.nprobes;
    for (int k = 0; k < p.nsteps; ++k) {
        const long long s = p.step0 + k;
        double inv_tau, amp;
        dev_schedule(p.sched, s, inv_tau, amp);
        const double *Told = (k & 1) ? p.Tnew : p.Told;
        double *Tnew = (k & 1) ? const_cast<double *>(p.Told) : p.Tnew;
        // probe record of this step: records are appended while the ring has room (the host mirrors
        // this arithmetic to count written and dropped records)
        double *probe_out = nullptr;
        if (p.nprobes > 0 && (s + 1) % p.probe_every == 0) {
            const long long r = p.rec0 + ((s + 1) / p.probe_every - p.step0 / p.probe_every - 1);
            if ((size_t)(r + 1) * rec <= p.probe_cap) probe_out = p.probe_base + (size_t)r * rec;
        }
        line_step<M, G, 1>(p, Told, Tnew, inv_tau, amp, probe_out, st, xch, lay);
        grid.sync();
    }
}

// ---------------------------------------------------------------- fp64 FMA peak probe
static __global__ void fp64_peak_kernel(double *out, long long iters, double a, double b)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (long long it = 0; it < iters; ++it) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

} // namespace heat

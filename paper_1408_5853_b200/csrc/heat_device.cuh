// heat_device.cuh -- device-side data structures and arithmetic shared by the sm_100a kernels.
//
// One time step of the explicit-implicit scheme (8) P:L108-113 of arXiv 1408.5853.  Every
// node of a z-line is one tridiagonal row  A_i x_{i-1} + B_i x_i + C_i x_{i+1} = F_i :
//   regular node  : coefficients (13) P:L140-145,
//   interface node: flux continuity (18) P:L178-181 (scaled by h_i h_{i+1}),
//   r boundaries  : (15) P:L158-161 (or a Dirichlet row),
// so that the paper's sweep (12),(14),(16),(17),(20) is the Thomas algorithm on these rows.
// "P:Lnnn" cites a line of the paper text; readings G1..G22 are listed in DESIGN.md.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace heat {

// ---------------------------------------------------------------- property laws
// Device form of heat_law with the constants folded at create time (host, long double):
//   POWn : f(T) = ck * T^p, ck = c0 / T_ref^p ; ckh = ck * 0.5^p so that
//          f((Ta+Tb)/2) = ckh * (Ta+Tb)^p        (lambda at a half node, reading G3)
//   POLY : f(T) = sum c[k] T^k (23),(24) P:L245-248
// The heat-capacity law carries rho_m folded in (rho_m c_Vm(T) is what (13) uses).
enum LawKind : int {
    LK_CONST = 0, LK_POW1 = 1, LK_POW2 = 2, LK_POW3 = 3, LK_POW1_5 = 4, LK_POW0_5 = 5,
    LK_POWM0_5 = 6, LK_POWG = 7, LK_POLY = 8
};

struct DLaw {
    int kind;
    int pad_;
    double ck;   // CONST: value
    double ckh;
    double p;    // exponent (POWG)
    double c[5]; // POLY
};

struct DLayer {
    DLaw k;   // lambda_m(T)
    DLaw rc;  // rho_m * c_Vm(T)
    DLaw src; // s(T)
    int heater;
    int pad_;
};

// node kinds in the per-node info word: bits 0-1 kind, bits 2-3 fixed-row slot,
// bits 8-15 layer of the segment left of the node, bits 16-23 layer right of it
enum : uint32_t { NK_REG = 0, NK_IFACE = 1, NK_FIXED = 2, NK_KEEP = 3 }; // NK_KEEP: outside Omega (stepped domain), x = T

__device__ __forceinline__ double rcp_nr(double x)
{
    // MUFU.RCP64H seed (>= 20 good bits) + two Newton steps: relative error ~1 ulp.
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    return y;
}

// reciprocal: MUFU.RCP64H seed (>= 20 bits) + one cubic step e -> e^3: ~2^-60 before rounding
__device__ __forceinline__ double rcp_cubic(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
}

__device__ __forceinline__ double law_at(const DLaw &L, double T)
{
    switch (L.kind) {
    case LK_CONST: return L.ck;
    case LK_POW1: return L.ck * T;
    case LK_POW2: return L.ck * (T * T);
    case LK_POW3: return L.ck * (T * T * T);
    case LK_POW1_5: return L.ck * (T * sqrt(T));
    case LK_POW0_5: return L.ck * sqrt(T);
    case LK_POWM0_5: return L.ck * rsqrt(T);
    case LK_POWG: return L.ck * pow(T, L.p);
    default: { // LK_POLY, Horner
        double s = L.c[4];
        s = fma(s, T, L.c[3]);
        s = fma(s, T, L.c[2]);
        s = fma(s, T, L.c[1]);
        s = fma(s, T, L.c[0]);
        return s;
    }
    }
}

// lambda at the half node between temperatures Ta and Tb.
// face_mode 0: lambda((Ta+Tb)/2) (reading G3); face_mode 1: (lambda(Ta)+lambda(Tb))/2.
__device__ __forceinline__ double law_face(const DLaw &L, double Ta, double Tb, int face_mode)
{
    if (face_mode != 0) return 0.5 * (law_at(L, Ta) + law_at(L, Tb));
    const double s = Ta + Tb;
    switch (L.kind) {
    case LK_CONST: return L.ck;
    case LK_POW1: return L.ckh * s;
    case LK_POW2: return L.ckh * (s * s);
    case LK_POW3: return L.ckh * (s * s * s);
    case LK_POW1_5: return L.ckh * (s * sqrt(s));
    case LK_POW0_5: return L.ckh * sqrt(s);
    case LK_POWM0_5: return L.ckh * rsqrt(s);
    case LK_POWG: return L.ck * pow(0.5 * s, L.p);
    default: return law_at(L, 0.5 * s);
    }
}

// ---------------------------------------------------------------- kernel parameters
struct ProbeSrc {
    int i;       // radial node
    int j_src;   // line whose freshly solved value is recorded (1 / nz-2 for a Neumann z line)
    int j_store; // the probe's own line (source of a static value on a Dirichlet z line)
    int is_static;
};

// the step schedule on the device (persistent multi-step kernels): integer state -> (1/tau_k, amp_k)
struct DSched {
    long long P, S;      // steps per period / steps with the source on, in units of tau; 0 = no source
    int nsub;            // transient sub-steps replacing the first tau of a period; 0 = Heaviside
    int pad_;
    double inv_dt, inv_dt_sub;
    const double *amp_sub; // [nsub]: 1 - exp(-q / k), (22) P:L212 (reading G8)
};

struct KParams {
    const double *Told; // current level  [batch][nz][nr]
    double *Tnew;       // next level
    const double *ga;   // [batch][nrp]  regular: r_{i-1/2}/(r_i hbar_i h_i); interface: h_{i+1}; fixed: A
    const double *gc;   // [batch][nrp]  regular: r_{i+1/2}/(r_i hbar_i h_{i+1}); interface: h_i; fixed: C
    const uint32_t *info; // [batch][nrp]
    const double *ezm;  // [nz] 1/(etabar_j eta_j)      (11) P:L125, reading G2
    const double *ezp;  // [nz] 1/(etabar_j eta_{j+1})
    const DLayer *layers;
    const double *Q0;   // [batch]
    const ProbeSrc *probes;
    double *probe_out;  // record of this step ([batch][nprobes]) or nullptr
    double inv_tau;     // 1/tau_k
    double amp;         // nu(t_k) p^2(t_k)   (4) P:L79, (22) P:L212
    double fixF[4];     // right-hand sides of the fixed rows: r_in, r_out, padding
    int nr, nz, batch, nrp, nlayers, nprobes;
    int face_mode;
    int z_lo_neumann, z_hi_neumann;
    int total_lines;    // batch * (nz-2)
    // persistent multi-step launch (heat_line_persist_kernel)
    int nsteps, probe_every;
    long long step0, rec0;
    size_t probe_cap;
    double *probe_base;
    DSched sched;
    // iterated variant (heat_line_iter_kernel): the field the laws are evaluated at
    const double *Tcoef;
    // stepped domain (reading G24): the lines j > j_step use the second set of row tables, in which node
    // i_step is the (15) boundary row and the nodes beyond it are NK_KEEP; j_step = 0: rectangle
    const double *ga2, *gc2;
    const uint32_t *info2;
    int i_step, j_step;
    // z-slab run with direct peer stores (heat_set_halo_peer): where the first / last interior line of
    // the new level goes in the lower / upper neighbour slab's next level (batch member 0; nullptr: none)
    double *peer_lo, *peer_hi;
    long long peer_lo_stride, peer_hi_stride; // doubles per batch member there
};

} // namespace heat

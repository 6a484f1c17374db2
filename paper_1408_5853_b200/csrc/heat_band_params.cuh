// heat_band_params.cuh -- parameter block, per-layer law table and shared-memory layout of the
// band kernel (heat_band_kernel.cuh); included by the host code, which does not need the kernel.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda.h>

#include "heat_device.cuh"

namespace heat {

// per-layer laws in polynomial form (host-built, long double):
//   lambda_m((Ta+Tb)/2) = (sum_n K[n] s^n) * (sqrtk ? sqrt(s) : 1),  s = Ta + Tb   (G3)
//   rho_m c_Vm(T)       = sum_n C[n] T^n
struct PLayer {
    double K[5];
    double C[4];
    double src;   // s(T) == const
    int sqrtk;
    int heater;
};

// chunk descriptor (one per 8 nodes): bits 0-7 layer A, 8-15 layer B, 16-19 ks+1 (0 = no
// interface node in the chunk; else rows < ks are layer A, row ks is the interface node, rows
// > ks are layer B), bit 20 = chunk starts with the r_in boundary row, bit 21 = chunk ends with
// the r_out boundary row
enum : uint32_t { BD_FIRST = 1u << 20, BD_LAST = 1u << 21 };

struct BParams {
    CUtensorMap tm_ld; // current level, box {16 doubles, G/2 rows}
    CUtensorMap tm_st; // next level, same box
    const double *Told;
    const uint32_t *cdesc; // [batch][nr/8]
    const PLayer *players;
    const double *ezm, *ezp, *Q0;
    const ProbeSrc *probes;
    double *probe_out;
    double inv_tau, amp, g0;
    double rin_om, rin_be;         // state after the r_in row: om = 1 - alpha_0, beta_0   (15),(16)
    double rout_a, rout_w, rout_f; // the r_out row as (a, w, f): -a x_{N-1} + (a + w) x_N = f   (15),(17)
    int nr, nz, batch, nlayers, nprobes;
    int z_lo_neumann, z_hi_neumann;
    int rpl;  // tensor rows (16 doubles) per line
    int BL;   // lines per band
    int bands_per_member, total_bands;
    int rank_rot; // see heat_band_kernel: rotation of the cluster rank -> radius part map in odd clusters
};

template <int G, int CL, int NT_>
struct BandCfg {
    static constexpr int NT = NT_;
    static constexpr int M = 8;
    static constexpr int LPB = NT / G;       // lines (bands) a CTA works on side by side
    static constexpr int GL = G * CL;        // threads per line
    static constexpr int WG = GL / 32;       // warps (= separators) per line
    static constexpr int NSEP = (NT / 32) * CL;
    static constexpr int SLOT = NT * 64;     // bytes of one staged line tile
    static constexpr int PUB = 12;
    static constexpr int NSLOT = 5;           // ring of staged lines: j-1 (store draining), j, j+1, j+2, j+3
    static constexpr int OFF_FLUX = NSLOT * SLOT;
    static constexpr int OFF_HALO = 6 * SLOT;
    static constexpr int OFF_PUB = OFF_HALO + 256;
    static constexpr int OFF_YSEP = OFF_PUB + 2 * NSEP * PUB * 8;
    static constexpr int OFF_MBAR = OFF_YSEP + NSEP * 8;
    static constexpr int OFF_XBAR = OFF_MBAR + NSLOT * 8; // separator-exchange barriers
    static constexpr int OFF_LAY = OFF_XBAR + 2 * 8;
    static constexpr size_t smem_bytes(int nlayers) { return 1024 + (size_t)OFF_LAY + sizeof(PLayer) * (size_t)nlayers; }
};

} // namespace heat

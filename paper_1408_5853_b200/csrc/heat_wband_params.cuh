// heat_wband_params.cuh -- parameter block, law table and shared-memory layout of the
// warp-autonomous band kernel (heat_wband_kernel.cuh); included by the host code.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda.h>

#include "heat_band_params.cuh"

namespace heat {

// chunk descriptor of the wband kernel (one per 16 nodes = one thread): bits 0-7 layer A,
// 8-15 layer B, 16-20 ks+1 (0 = no interface node in the chunk; else rows < ks are layer A, row
// ks is the interface node (18), rows > ks are layer B), bit 24 = chunk starts with the r_in
// boundary row, bit 25 = chunk ends with the r_out boundary row (15)
enum : uint32_t { WD_FIRST = 1u << 24, WD_LAST = 1u << 25 };

// per-layer laws as the kernel keeps them in shared memory, scaled for this launch:
//   lambda_m((Ta+Tb)/2) = (sum_n K[n] s^n) * (sq ? sqrt(s) : 1),  s = Ta + Tb   (G3)
//   rho_m c_Vm(T) / tau = sum_n Ct[n] T^n
//   X_m / Q0            = qsrc = nu(t_k) p^2(t_k) s_m for the heater layer, else 0  (2)-(4),(22)
struct alignas(16) WLayer {
    double K[6];  // K[5] unused: keeps Ct 16-byte aligned for the paired reloads
    double Ct[4];
    double qsrc;
    int sq;
    int pad_;
};

struct WParams {
    CUtensorMap tm_ld; // current level as [rows][16 doubles], box {16, 32}, SWIZZLE_128B
    CUtensorMap tm_st; // next level, same box
    const double *Told;
    const uint32_t *wdesc; // [batch][nr/16]
    const PLayer *players;
    const double *ezm, *ezp, *Q0;
    const ProbeSrc *probes;
    double *probe_out;
    double inv_tau, amp, g0;
    double rin_om, rin_be;         // state after the r_in row: om = 1 - alpha_0, beta_0   (15),(16)
    double rout_a, rout_w, rout_f; // the r_out row as (a, w, f): -a x_{N-1} + (a + w) x_N = f   (15),(17)
    int nr, nz, batch, nlayers, nprobes;
    int z_lo_neumann, z_hi_neumann;
    int rpl;  // tensor rows (16 doubles) per line = threads per line
    int BL;   // lines per band
    int bands_per_member, total_bands;
    // z-slab run with direct peer stores (heat_set_halo_peer): the first / last interior line of the new
    // level is also stored into the halo line of the lower / upper neighbour slab's NEXT level
    CUtensorMap tm_peer_lo, tm_peer_hi;
    int peer_lo_row, peer_hi_row;   // tensor row of batch member 0's halo line there, < 0: no such neighbour
    int peer_lo_rpm, peer_hi_rpm;   // tensor rows per batch member there
};

// WL = warps per line (nr = 512 WL), NW = warps per CTA.  A line wider than a CTA spans a cluster
// of CL = WL / NW CTAs; a narrower one shares its CTA with LPB - 1 other lines (other bands).
template <int WL, int NW>
struct WBandCfg {
    static constexpr int M = 16;
    static constexpr int NT = 32 * NW;
    static constexpr int CL = (WL > NW) ? WL / NW : 1;
    static constexpr int LPB = (WL < NW) ? NW / WL : 1;
    static constexpr int WPL = (WL < NW) ? WL : NW; // warps of this CTA that work on one line
    static constexpr int NS = 5;                     // ring of staged line parts per warp
    static constexpr int SLOT = 4096;                // 32 threads x 16 doubles
    static constexpr int PUB = 12;                   // doubles a warp publishes for the separator solve
    static constexpr int WARP_BYTES = (NS + 1) * SLOT; // ring + the face fluxes
    static constexpr int OFF_HALO = NW * WARP_BYTES;                 // [NW][NS][4 doubles]
    static constexpr int OFF_PUB = OFF_HALO + NW * NS * 32;          // [2][LPB][WL][PUB]
    static constexpr int OFF_FBAR = OFF_PUB + 2 * LPB * WL * PUB * 8; // [NW][NS] load barriers
    static constexpr int OFF_XBAR = OFF_FBAR + NW * NS * 8;          // [LPB][2] exchange barriers
    static constexpr int OFF_LAY = OFF_XBAR + LPB * 2 * 8;
    static constexpr size_t smem_bytes(int nlayers) { return 1024 + (size_t)OFF_LAY + sizeof(WLayer) * (size_t)nlayers; }
};

} // namespace heat

// hydro_launch.cuh -- host-side launch descriptors shared by the C ABI (hydro_api.cu) and the
// per-variant instantiation units.  No device code here.
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include "hydro_math.cuh"

namespace hydro {

// uniform-grid mode of the fused CTU kernel (hydro_solve_grid_*): planes are fetched from / written to [5][Nz][Ny][Nx]
// grids directly, ghost zones by periodic wrap (bc 0) or zero-gradient clamp (bc 1); gin == nullptr: batch mode
template <class R> struct GridIO { const R* gin; R* gout; int Gx, Gy, Gz, bc; };

template <class R> struct SolveArgs {
  const R* in;          // [Ng][5][S^3], S = 16 + 2 g
  R* out;               // [Ng][5][16^3]
  R* face_flux;         // [Ng][9][5][16*16] or nullptr
  int Ng, g;
  Par<R> par;
  const R* max_speed;   // device scalar or nullptr: nu = cfl / *max_speed formed on the device
  R cfl;
  long long* status;    // device, [3] or nullptr
  void* workspace;      // staged path only
  size_t workspace_bytes;
  cudaStream_t stream;
  GridIO<R> grid;
};

template <class R> using LaunchFn = cudaError_t (*)(const SolveArgs<R>&);

// ghost width needed by (scheme, recon): S1 of DESIGN.md
inline int min_ghost(int scheme, int recon) { return (scheme == SCHEME_VL ? 3 : 2) + (recon == RECON_PPM ? 1 : 0); }

// staged path: per-CTA scratch = 50 SoA arrays over the (16 + 2 g_min)^3 work box
inline size_t staged_slot_bytes(int scheme, int recon, size_t elem) {
  const size_t s = PS + 2 * min_ghost(scheme, recon);
  return 50 * s * s * s * elem;
}
constexpr int STAGED_MAX_SLOTS = 148 * 4;

constexpr size_t SMEM_MAX_OPTIN = 227 * 1024;
constexpr int FUSED_COLS = (PS + 2) * (PS + 2);     // 18 x 18 columns: interior + one-cell ring

// ---- lean fused CTU kernel (hydro_lean_ctu.cuh): column-per-thread z-march, phase-crossing state in shared memory,
// two co-resident CTAs per SM where the tiles allow ------------------------------------------------------------
constexpr int LEAN_NT = 320;                        // 10 warps: 288 columns of the rows j = 0..15, 32 of the rows j = -1, 16
constexpr int LEAN_COLS = FUSED_COLS;
// PPM tiles are trimmed (one raw landing plane; the oldest z-pencil plane carried in registers) so that two fp32 CTAs fit
constexpr int LEAN_NRAW(int recon) { return recon == RECON_PPM ? 1 : 2; }
constexpr int LEAN_RING_CARRY(int recon) { return recon == RECON_PPM ? 1 : 0; }
// mbarriers | W ring | private z states [2][2][5][NT] | LOX UPX LOY UPY FX FY [6][5][324] | raw planes [NRAW][5][S*S]
constexpr size_t lean_smem_bytes(size_t elem, int recon, int g) {
  const size_t S = PS + 2 * g, SWP = PS + 2 * (2 + recon), NWS = 2 * (1 + recon) + 1 - LEAN_RING_CARRY(recon);
  return 64 + elem * (LEAN_NRAW(recon) * 5 * S * S + NWS * 5 * SWP * SWP + (size_t)20 * LEAN_NT + (size_t)30 * LEAN_COLS);
}
// fused MHM kernel (hydro_lean_mhm.cuh): mbarriers | raw planes | W ring | LOX UPX LOY UPY FX FY
constexpr size_t mhm_smem_bytes(size_t elem, int recon, int g) {
  const size_t S = PS + 2 * g, SWP = PS + 2 * (2 + recon), NW = 2 * (1 + recon) + 1;
  return 64 + elem * (2 * 5 * S * S + NW * 5 * SWP * SWP + (size_t)30 * LEAN_COLS);
}
// fused VL kernel (hydro_lean_vl.cuh): plus cells within E = recon + 2 of the interior + one warp of boundary faces
constexpr int VL_NT(int recon) { return 320 + 64 * (recon + 1) + 32; }
// merged schedule (two CTA barriers per plane instead of four; its first-pass fluxes need two fields of their own): fp32 only.
// Measured per 4096 groups: fp32 VL+PLM+Roe 1.87 -> 1.81 ms; fp64 5.08 -> 5.21 ms (and fp64 + PPM has no room for the fields)
constexpr bool vl_merged(size_t elem, int recon) { return (void)recon, elem == 4; }
// stages on warps of their own (hydro_lean_vl.cuh SPLIT): 23 warps leave 80 registers per thread, which the HLLE / HLLC solvers
// fit in and Roe / exact do not.  Measured per 4096 groups, fp32 PLM: HLLC 1.67 -> 1.53 ms; Roe 1.79 -> 2.01 ms (100 bytes of
// spills); PPM (25 warps, 72 registers) is slower with every solver.
#ifndef VL_SPLIT
#define VL_SPLIT 1
#endif
constexpr bool vl_split(size_t elem, int recon, int rs) {
  return VL_SPLIT && elem == 4 && recon == RECON_PLM && (rs == RS_HLLC || rs == RS_HLLE);
}
// mbarriers | one primitive plane | W-half ring | LOX UPX LOY UPY FX FY | (merged: F1_x F1_y) | one raw plane
constexpr size_t vl_smem_bytes(size_t elem, int recon, int g) {
  const size_t S = PS + 2 * g, SW = PS + 2 * (recon + 3), SH = PS + 2 * (recon + 2), NW = 2 * (1 + recon) + 1;
  const size_t SF = PS + 2 * (recon + 2) + 1, FPL = (SF * SF + 3) / 4 * 4;
  return 64 + elem * (5 * S * S + 5 * SW * SW + NW * 5 * SH * SH + (size_t)30 * LEAN_COLS + (vl_merged(elem, recon) ? 2 * 5 * FPL : 0));
}
constexpr bool lean_available(int precision_bytes, int scheme, int recon) {
  (void)precision_bytes; (void)recon;
  return scheme == SCHEME_CTU || scheme == SCHEME_MHM || scheme == SCHEME_VL;
}
constexpr bool lean_fits(int precision_bytes, int scheme, int recon, int g) {
  return lean_available(precision_bytes, scheme, recon) &&
         (scheme == SCHEME_MHM ? mhm_smem_bytes((size_t)precision_bytes, recon, g)
          : scheme == SCHEME_VL ? vl_smem_bytes((size_t)precision_bytes, recon, g)
                                : lean_smem_bytes((size_t)precision_bytes, recon, g)) <= SMEM_MAX_OPTIN;
}

template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_lean(const SolveArgs<R>& a);
template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_staged(const SolveArgs<R>& a);

}  // namespace hydro

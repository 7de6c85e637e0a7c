// hydro_launch.cuh -- host-side launch descriptors shared by the C ABI (hydro_api.cu) and the
// per-variant instantiation units.  No device code here.
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include "hydro_math.cuh"

namespace hydro {

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

// which (precision, scheme, recon) have a fused z-marching kernel (all four Riemann solvers each)
constexpr bool fused_available(int precision_bytes, int scheme, int recon) {
  (void)precision_bytes; (void)recon;
  return scheme == SCHEME_CTU;
}

// ---- shared-memory footprint of the fused CTU kernel (one formula for the kernel and the host) ----
constexpr int FUSED_NT = 352;                       // threads per CTA
constexpr int FUSED_COLS = (PS + 2) * (PS + 2);     // 18 x 18 columns
enum : int { SM_Z = 1, SM_F1Z = 2, SM_CARRY = 4, SM_XY = 8 };  // per-thread state kept in shared memory
constexpr int CTU_SM_F64 = SM_Z | SM_F1Z;
constexpr int ctu_sm_mask(size_t elem) { return elem == 8 ? CTU_SM_F64 : 0; }
constexpr int ctu_nslots(int mask) {
  return ((mask & SM_Z) ? 4 : 0) + ((mask & SM_F1Z) ? 2 : 0) + ((mask & SM_CARRY) ? 3 : 0) + ((mask & SM_XY) ? 5 : 0);
}
constexpr size_t ctu_smem_bytes(size_t elem, int recon, int g, int mask) {
  const size_t S = PS + 2 * g, SWP = PS + 2 * (2 + recon), NW = 2 * (1 + recon) + 1;
  return 16 + elem * (2 * 5 * S * S + NW * 5 * SWP * SWP + 4 * 5 * FUSED_COLS + (size_t)ctu_nslots(mask) * 5 * FUSED_NT);
}
constexpr size_t SMEM_MAX_OPTIN = 227 * 1024;
// does the fused kernel of (precision, scheme, recon) run with ghost width g ?
constexpr bool fused_fits(int precision_bytes, int scheme, int recon, int g) {
  return fused_available(precision_bytes, scheme, recon) &&
         ctu_smem_bytes((size_t)precision_bytes, recon, g, ctu_sm_mask((size_t)precision_bytes)) <= SMEM_MAX_OPTIN;
}

// ---- warp-specialised fused CTU kernel (hydro_ws_ctu.cuh): predictor group + corrector group -------
constexpr int WS_NT1 = 352;                         // group P: one thread per column (+ idle lanes of warp 10)
constexpr int WS_NT2 = 288;                         // group C: one thread per face, compacted
constexpr int WS_NT = WS_NT1 + WS_NT2;
constexpr int WS_COLS = FUSED_COLS;
constexpr bool ws_available(int precision_bytes, int scheme, int recon) {
  (void)recon;
  return precision_bytes == 4 && scheme == SCHEME_CTU;
}
// mbarriers | raw planes [2][5][S*S] | W ring | hand-off [2][9][5][324] | F* exchange [2][5][324] | F buffers [2][2][5][324]
constexpr size_t ws_smem_bytes(size_t elem, int recon, int g) {
  const size_t S = PS + 2 * g, SWP = PS + 2 * (2 + recon), NW = 2 * (1 + recon) + 1;
  return 64 + elem * (2 * 5 * S * S + NW * 5 * SWP * SWP + (size_t)(2 * 9 + 2 + 4) * 5 * WS_COLS);
}
constexpr bool ws_fits(int precision_bytes, int scheme, int recon, int g) {
  return ws_available(precision_bytes, scheme, recon) && ws_smem_bytes((size_t)precision_bytes, recon, g) <= SMEM_MAX_OPTIN;
}

// ---- lean fused CTU kernel (hydro_lean_ctu.cuh): column-per-thread z-march, phase-crossing state in shared memory,
// two co-resident CTAs per SM where the tiles allow ------------------------------------------------------------
constexpr int LEAN_NT = 320;                        // 10 warps: 288 columns of the rows j = 0..15, 32 of the rows j = -1, 16
constexpr int LEAN_COLS = FUSED_COLS;
// mbarriers | raw planes [2][5][S*S] | W ring | private z states [2][2][5][NT] | LOX UPX LOY UPY FX FY [6][5][324]
constexpr size_t lean_smem_bytes(size_t elem, int recon, int g) {
  const size_t S = PS + 2 * g, SWP = PS + 2 * (2 + recon), NW = 2 * (1 + recon) + 1;
  return 64 + elem * (2 * 5 * S * S + NW * 5 * SWP * SWP + (size_t)20 * LEAN_NT + (size_t)30 * LEAN_COLS);
}
constexpr bool lean_available(int precision_bytes, int scheme, int recon) {
  (void)precision_bytes; (void)recon;
  return scheme == SCHEME_CTU;
}
constexpr bool lean_fits(int precision_bytes, int scheme, int recon, int g) {
  return lean_available(precision_bytes, scheme, recon) && lean_smem_bytes((size_t)precision_bytes, recon, g) <= SMEM_MAX_OPTIN;
}

template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_lean(const SolveArgs<R>& a);
template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_ws(const SolveArgs<R>& a);
template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_staged(const SolveArgs<R>& a);
template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_fused(const SolveArgs<R>& a);

}  // namespace hydro

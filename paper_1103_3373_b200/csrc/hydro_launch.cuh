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
  (void)precision_bytes; (void)scheme; (void)recon;
  return false;
}

template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_staged(const SolveArgs<R>& a);
template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_fused(const SolveArgs<R>& a);

}  // namespace hydro

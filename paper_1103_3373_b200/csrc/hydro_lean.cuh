// hydro_lean.cuh -- dispatch of the fused z-marching kernels (CTU, MHM, VL); lean_fits() gates it in the C ABI.
#pragma once
#include "hydro_launch.cuh"
#include "hydro_lean_ctu.cuh"
#include "hydro_lean_mhm.cuh"
#include "hydro_lean_vl.cuh"

namespace hydro {

// co-resident CTAs per SM the register budget is set for: two where the tiles of two groups fit (fp32)
template <class R, int RECON> struct LeanTune { static constexpr int MINB = sizeof(R) == 4 ? 2 : 1; };

template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_lean(const SolveArgs<R>& a) {
  if constexpr (SCHEME == SCHEME_CTU) {
    // compile-time specialisation of the default options: van Leer limiter on primitive variables, no floors
    const bool fast = a.par.limiter == LIM_VANLEER && !a.par.char_limit && !(a.par.min_dens > R(0)) && !(a.par.min_pres > R(0));
    if (a.grid.gin) {  // uniform-grid mode (hydro_solve_grid_*)
      if (fast) return launch_ctu_lean<R, RECON, RS, 1, LeanTune<R, RECON>::MINB, 1>(a);
      return launch_ctu_lean<R, RECON, RS, 0, LeanTune<R, RECON>::MINB, 1>(a);
    }
    if (fast) return launch_ctu_lean<R, RECON, RS, 1, LeanTune<R, RECON>::MINB>(a);
    return launch_ctu_lean<R, RECON, RS, 0, LeanTune<R, RECON>::MINB>(a);
  } else if constexpr (SCHEME == SCHEME_MHM) {
    const bool fast = a.par.limiter == LIM_VANLEER && !a.par.char_limit && !(a.par.min_dens > R(0)) && !(a.par.min_pres > R(0));
    constexpr int MINB = sizeof(R) == 4 ? 2 : 1;
    if (a.grid.gin) {
      if (fast) return launch_mhm_lean<R, RECON, RS, 1, MINB, 1>(a);
      return launch_mhm_lean<R, RECON, RS, 0, MINB, 1>(a);
    }
    if (fast) return launch_mhm_lean<R, RECON, RS, 1, MINB>(a);
    return launch_mhm_lean<R, RECON, RS, 0, MINB>(a);
  } else {
    const bool fast = a.par.limiter == LIM_VANLEER && !a.par.char_limit && !(a.par.min_dens > R(0)) && !(a.par.min_pres > R(0));
    if (a.grid.gin) {
      if (a.par.min_dens > R(0) || a.par.min_pres > R(0)) return cudaErrorNotSupported;  // hydro_api.cu grid_mode_ok()
      if (fast) return launch_vl_lean<R, RECON, RS, 1, 1>(a);
      return launch_vl_lean<R, RECON, RS, 0, 1>(a);
    }
    if (fast) return launch_vl_lean<R, RECON, RS, 1>(a);
    return launch_vl_lean<R, RECON, RS, 0>(a);
  }
}

}  // namespace hydro

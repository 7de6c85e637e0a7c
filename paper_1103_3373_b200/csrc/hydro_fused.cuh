// hydro_fused.cuh -- dispatch of the fused z-marching kernels (one CTA per patch group, all
// intermediates on chip).  Variants without a fused kernel return cudaErrorNotSupported; the C ABI
// never reaches them because fused_available() gates the dispatch.
#pragma once
#include "hydro_fused_ctu.cuh"
#include "hydro_launch.cuh"

namespace hydro {

// per-precision tuning of the CTU kernel: which per-thread state lives in shared memory, CTAs per SM
template <class R, int RECON> struct CtuTune;
template <int RECON> struct CtuTune<float, RECON> { static constexpr int SM = 0, MINB = 1; };
template <int RECON> struct CtuTune<double, RECON> { static constexpr int SM = CTU_SM_F64, MINB = 1; };

template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_fused(const SolveArgs<R>& a) {
  if constexpr (SCHEME == SCHEME_CTU) {
    return launch_ctu_fused<R, RECON, RS, CtuTune<R, RECON>::SM, CtuTune<R, RECON>::MINB>(a);
  } else {
    (void)a;
    return cudaErrorNotSupported;
  }
}

}  // namespace hydro

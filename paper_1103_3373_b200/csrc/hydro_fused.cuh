// hydro_fused.cuh -- fused z-marching kernels (one CTA per patch group, intermediates on chip).
#pragma once
#include "hydro_launch.cuh"

namespace hydro {

template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_fused(const SolveArgs<R>& a) {
  (void)a;
  return cudaErrorNotSupported;  // unreachable through the C ABI: fused_available() gates the dispatch
}

}  // namespace hydro

// hydro_ws.cuh -- dispatch of the warp-specialised fused kernels.  Variants without one return
// cudaErrorNotSupported; the C ABI never reaches them because ws_available() gates the dispatch.
#pragma once
#include "hydro_launch.cuh"
#include "hydro_ws_ctu.cuh"

namespace hydro {

template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_ws(const SolveArgs<R>& a) {
  if constexpr (ws_available((int)sizeof(R), SCHEME, RECON)) {
    return launch_ctu_ws<R, RECON, RS>(a);
  } else {
    (void)a;
    return cudaErrorNotSupported;
  }
}

}  // namespace hydro

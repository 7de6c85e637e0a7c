// explicit instantiations of the lean fused CTU kernel: float, RECON_PPM, four Riemann solvers (x fast / generic options)
#include "hydro_lean.cuh"
namespace hydro {
#define INST(RS) template cudaError_t launch_lean<float, SCHEME_CTU, RECON_PPM, RS>(const SolveArgs<float>&);
INST(RS_EXACT) INST(RS_HLLE) INST(RS_HLLC) INST(RS_ROE)
#undef INST
}  // namespace hydro

// explicit instantiations of the warp-specialised fused CTU kernel: float, PLM / PPM x four Riemann solvers
#include "hydro_ws.cuh"
namespace hydro {
#define INST(RECON, RS) template cudaError_t launch_ws<float, SCHEME_CTU, RECON, RS>(const SolveArgs<float>&);
INST(RECON_PLM, RS_EXACT) INST(RECON_PLM, RS_HLLE) INST(RECON_PLM, RS_HLLC) INST(RECON_PLM, RS_ROE)
INST(RECON_PPM, RS_EXACT) INST(RECON_PPM, RS_HLLE) INST(RECON_PPM, RS_HLLC) INST(RECON_PPM, RS_ROE)
#undef INST
}  // namespace hydro

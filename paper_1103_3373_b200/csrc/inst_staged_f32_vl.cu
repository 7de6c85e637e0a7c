// explicit instantiations of the staged solver: float, SCHEME_VL, all reconstructions x Riemann solvers
#include "hydro_staged.cuh"
namespace hydro {
#define INST(RECON, RS) template cudaError_t launch_staged<float, SCHEME_VL, RECON, RS>(const SolveArgs<float>&);
INST(RECON_PLM, RS_EXACT) INST(RECON_PLM, RS_HLLE) INST(RECON_PLM, RS_HLLC) INST(RECON_PLM, RS_ROE)
INST(RECON_PPM, RS_EXACT) INST(RECON_PPM, RS_HLLE) INST(RECON_PPM, RS_HLLC) INST(RECON_PPM, RS_ROE)
#undef INST
}  // namespace hydro

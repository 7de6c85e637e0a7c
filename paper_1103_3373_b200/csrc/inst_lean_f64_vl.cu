// explicit instantiations of the fused VL kernel: double, PLM / PPM x four Riemann solvers (x fast / generic options)
#include "hydro_lean.cuh"
namespace hydro {
#define INST(RC, RS) template cudaError_t launch_lean<double, SCHEME_VL, RC, RS>(const SolveArgs<double>&);
INST(RECON_PLM, RS_EXACT) INST(RECON_PLM, RS_HLLE) INST(RECON_PLM, RS_HLLC) INST(RECON_PLM, RS_ROE)
INST(RECON_PPM, RS_EXACT) INST(RECON_PPM, RS_HLLE) INST(RECON_PPM, RS_HLLC) INST(RECON_PPM, RS_ROE)
#undef INST
}  // namespace hydro

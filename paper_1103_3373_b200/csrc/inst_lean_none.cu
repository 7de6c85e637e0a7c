// scheme without a fused kernel yet (VL): launchers that only fill the dispatch table
#include "hydro_lean.cuh"
namespace hydro {
#define INST(R, S, RC, RS) template cudaError_t launch_lean<R, S, RC, RS>(const SolveArgs<R>&);
#define FOR_RS(M, R, S, RC) M(R, S, RC, RS_EXACT) M(R, S, RC, RS_HLLE) M(R, S, RC, RS_HLLC) M(R, S, RC, RS_ROE)
#define FOR_RC(M, R, S) FOR_RS(M, R, S, RECON_PLM) FOR_RS(M, R, S, RECON_PPM)
FOR_RC(INST, float, SCHEME_VL)
FOR_RC(INST, double, SCHEME_VL)
}  // namespace hydro

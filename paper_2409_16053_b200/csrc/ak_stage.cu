// ak_stage.cu -- ak_hydro_stage kernels: fused c2p + reconstruction + HLLC in x1/x2/x3 +
// flux divergence + RK2 weighted update.  FMA contraction is allowed here (parity is to 1e-12, not
// bit-exact).
#include "ak_pack.h"
#include "ak_physics.cuh"
#include "ak_stage_simple.cuh"
#include "ak_stage_tiled.cuh"
#include "ak_stage_tma.cuh"

namespace ak {

cudaError_t launch_stage(const ak_pack& p, const double* Uin, const double* U0, double* Uout, const StageCoef& sc) {
  if (p.variant == 1) return launch_stage_simple(p, Uin, U0, Uout, sc);
  // TMA box origins must be 16-byte aligned in the innermost dimension: (ng - R) even.  The unusual case of
  // an odd surplus of ghost layers (ng = 4 with PPM4, ng = 3 with PLM) takes the LDG-staged tiled kernel.
  const int R = (p.recon == 0) ? 2 : 3;
  if (p.variant == 2 || ((p.d.ng - R) & 1)) return launch_stage_tiled(p, Uin, U0, Uout, sc);
  return launch_stage_tma(p, Uin, U0, Uout, sc);
}

int stage_launches_per_call(const ak_pack&) { return 1; }

}  // namespace ak

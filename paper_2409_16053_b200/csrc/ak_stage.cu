// ak_stage.cu -- ak_hydro_stage kernels: fused c2p + reconstruction + HLLC in x1/x2/x3 +
// flux divergence + RK2 weighted update.  Compiled with -fmad=false: every fused multiply-add of the
// production kernel is written out, so the same face solved by two tiles gives the same bits
// (DESIGN.md section 6.2).
#include "ak_pack.h"
#include "ak_physics.cuh"
#include "ak_stage_simple.cuh"
#include "ak_stage_tiled.cuh"
#include "ak_stage_v3.cuh"
#include "ak_fluxcorr.cuh"
#include "ak_fofc.cuh"

#include <cstdlib>

namespace ak {

// tile shape of the v3 kernel (workers + one edge warp): the one that wastes the fewest lanes on the ragged
// last tile row and on the edge warp.  0 = 16x10 (6 warps), 1 = 16x8 (5 warps)
static int pick_tile_v3(const ak_pack& p) {
  if (p.tile >= 0) return p.tile;
  const int n = p.d.nx[1];
  const double e10 = (double)n / (((n + 9) / 10) * 10) * (160.0 / 192.0);
  const double e8 = (double)n / (((n + 7) / 8) * 8) * (128.0 / 160.0);
  return e10 >= e8 ? 0 : 1;
}

template <int RECON, int RS>
static cudaError_t launch_stage_v3(const ak_pack& p, const double* Uin, const double* U0, double* Uout,
                                   const StageCoef& sc) {
  const bool stage2 = (Uin != U0);
  int tile = pick_tile_v3(p);
  if constexpr (RS != 0) { if (tile > 1) tile = 0; }   // LLF / HLLE: only the two 2-CTA/SM tiles are instantiated
  switch (tile) {
    case 1:  return launch_v3<RECON, RS, 16, 8, (RECON == 0 ? 3 : 2)>(p, Uin, U0, Uout, sc, stage2);   // PLM: 3 CTAs/SM fit
    case 2:  if constexpr (RS == 0) return launch_v3<RECON, RS, 16, 22, 1>(p, Uin, U0, Uout, sc, stage2);
    case 3:  if constexpr (RS == 0) return launch_v3<RECON, RS, 32, 11, 1>(p, Uin, U0, Uout, sc, stage2);
    default: return launch_v3<RECON, RS, 16, 10, 2>(p, Uin, U0, Uout, sc, stage2);
  }
}

template <int RECON>
static cudaError_t launch_stage_v3_rs(const ak_pack& p, const double* Uin, const double* U0, double* Uout,
                                      const StageCoef& sc) {
  switch (p.rsolver) {
    case 1:  return launch_stage_v3<RECON, 1>(p, Uin, U0, Uout, sc);
    case 2:  return launch_stage_v3<RECON, 2>(p, Uin, U0, Uout, sc);
    case 3:  return launch_stage_v3<RECON, 3>(p, Uin, U0, Uout, sc);
    default: return launch_stage_v3<RECON, 0>(p, Uin, U0, Uout, sc);
  }
}

cudaError_t launch_stage(const ak_pack& p, const double* Uin, const double* U0, double* Uout, const StageCoef& sc) {
  if (p.variant == 1) return launch_stage_simple(p, Uin, U0, Uout, sc);
  // TMA box origins must be 16-byte aligned in the innermost dimension: (ng - R) even.  The unusual case of
  // an odd surplus of ghost layers (ng = 4 with PPM4, ng = 3 with PLM) takes the LDG-staged tiled kernel.
  const int R = (p.recon == 0) ? 2 : 3;
  if (p.variant == 2 || ((p.d.ng - R) & 1)) return launch_stage_tiled(p, Uin, U0, Uout, sc);
  // PPMX / WENOZ: HLLC only, the two 2-CTA/SM tile shapes
  if (p.recon >= 2) {
    const bool stage2 = (Uin != U0);
    const int tile = pick_tile_v3(p) == 1 ? 1 : 0;
    if (p.recon == 2) return tile ? launch_v3<2, 0, 16, 8, 2>(p, Uin, U0, Uout, sc, stage2) : launch_v3<2, 0, 16, 10, 2>(p, Uin, U0, Uout, sc, stage2);
    return tile ? launch_v3<3, 0, 16, 8, 2>(p, Uin, U0, Uout, sc, stage2) : launch_v3<3, 0, 16, 10, 2>(p, Uin, U0, Uout, sc, stage2);
  }
  return p.recon == 0 ? launch_stage_v3_rs<0>(p, Uin, U0, Uout, sc) : launch_stage_v3_rs<1>(p, Uin, U0, Uout, sc);
}

cudaError_t launch_flux_correction(const ak_pack& p, const double* Uin, double* Uout, const StageCoef& sc) {
  if (p.recon == 2) return launch_flux_correction_t<2, 0>(p, Uin, Uout, sc);
  if (p.recon == 3) return launch_flux_correction_t<3, 0>(p, Uin, Uout, sc);
  switch (p.rsolver) {
    case 1:  return p.recon == 0 ? launch_flux_correction_t<0, 1>(p, Uin, Uout, sc) : launch_flux_correction_t<1, 1>(p, Uin, Uout, sc);
    case 2:  return p.recon == 0 ? launch_flux_correction_t<0, 2>(p, Uin, Uout, sc) : launch_flux_correction_t<1, 2>(p, Uin, Uout, sc);
    case 3:  return p.recon == 0 ? launch_flux_correction_t<0, 3>(p, Uin, Uout, sc) : launch_flux_correction_t<1, 3>(p, Uin, Uout, sc);
    default: return p.recon == 0 ? launch_flux_correction_t<0, 0>(p, Uin, Uout, sc) : launch_flux_correction_t<1, 0>(p, Uin, Uout, sc);
  }
}

cudaError_t launch_fofc(const ak_pack& p, const double* Uin, const double* U0, double* Uout, const StageCoef& sc) {
  if (p.recon == 2) return launch_fofc_t<2, 0>(p, Uin, U0, Uout, sc);
  if (p.recon == 3) return launch_fofc_t<3, 0>(p, Uin, U0, Uout, sc);
  switch (p.rsolver) {
    case 1:  return p.recon == 0 ? launch_fofc_t<0, 1>(p, Uin, U0, Uout, sc) : launch_fofc_t<1, 1>(p, Uin, U0, Uout, sc);
    case 2:  return p.recon == 0 ? launch_fofc_t<0, 2>(p, Uin, U0, Uout, sc) : launch_fofc_t<1, 2>(p, Uin, U0, Uout, sc);
    case 3:  return p.recon == 0 ? launch_fofc_t<0, 3>(p, Uin, U0, Uout, sc) : launch_fofc_t<1, 3>(p, Uin, U0, Uout, sc);
    default: return p.recon == 0 ? launch_fofc_t<0, 0>(p, Uin, U0, Uout, sc) : launch_fofc_t<1, 0>(p, Uin, U0, Uout, sc);
  }
}

int stage_launches_per_call(const ak_pack&) { return 1; }

}  // namespace ak

// ak_stage_simple.cuh -- cross-check implementation of one RK stage: one thread per active cell,
// stencil read straight from global memory, both faces of every direction recomputed by each cell.
// Roughly 2x the arithmetic of the tiled kernel; kept as variant 1 (ak_pack_set_variant) so the
// tiled kernel can be compared against an independent launch configuration on the device.
#pragma once
#include "ak_pack.h"
#include "ak_physics.cuh"

namespace ak {

template <int RECON>
__global__ void __launch_bounds__(128) stage_simple_kernel(PackDev P, const double* __restrict__ Uin,
                                                           const double* U0,
                                                           double* Uout, StageCoef sc) {
  constexpr int R = (RECON == 0) ? 2 : 3;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.nx[0]) return;
  const int j = blockIdx.y % P.nx[1], k = blockIdx.y / P.nx[1], m = blockIdx.z;
  GasConst g;
  g.gamma = P.gamma; g.gm1 = P.gamma - 1.0;
  g.ug_floor = P_FLOOR / (P.gamma - 1.0);
  const long long nc = P.ncell;
  const long long base = (long long)m * 5 * nc + ((long long)(k + P.ng) * P.nt[1] + (j + P.ng)) * P.nt[0] + (i + P.ng);
  const int lev = P.blk[m].x;
  const long long stride[3] = {1, P.nt[0], (long long)P.nt[0] * P.nt[1]};

  double acc[5];
#pragma unroll
  for (int n = 0; n < 5; n++) acc[n] = sc.g0 * Uin[base + n * nc] + sc.g1 * U0[base + n * nc];

  int nfl = 0;
#pragma unroll
  for (int d = 0; d < 3; d++) {
    const int iu = 1 + d, iv = 1 + (d + 1) % 3, iw = 1 + (d + 2) % 3;
    double W[2 * R + 1][5];                    // rotated primitives of cells c-R .. c+R along d
#pragma unroll
    for (int s = -R; s <= R; s++) {
      double u[5], w[5];
#pragma unroll
      for (int n = 0; n < 5; n++) u[n] = Uin[base + s * stride[d] + n * nc];
      int f = c2p(u, w, g.ug_floor);
      if (s == 0 && d == 0) nfl += f;
      W[s + R][0] = w[0]; W[s + R][1] = w[iu]; W[s + R][2] = w[iv]; W[s + R][3] = w[iw]; W[s + R][4] = w[4];
    }
    double WLlo[5], WRlo[5], WLhi[5], WRhi[5];
#pragma unroll
    for (int n = 0; n < 5; n++) {
      if constexpr (RECON == 0) {
        double hm = plm_halfslope(W[R - 2][n], W[R - 1][n], W[R][n]);
        double h0 = plm_halfslope(W[R - 1][n], W[R][n], W[R + 1][n]);
        double hp = plm_halfslope(W[R][n], W[R + 1][n], W[R + 2][n]);
        WLlo[n] = W[R - 1][n] + hm; WRlo[n] = W[R][n] - h0;
        WLhi[n] = W[R][n] + h0;     WRhi[n] = W[R + 1][n] - hp;
      } else {
        double fa = ppm4_iface(W[R - 3][n], W[R - 2][n], W[R - 1][n], W[R][n]);       // face -3/2
        double fb = ppm4_iface(W[R - 2][n], W[R - 1][n], W[R][n], W[R + 1][n]);       // face -1/2
        double fc = ppm4_iface(W[R - 1][n], W[R][n], W[R + 1][n], W[R + 2][n]);       // face +1/2
        double fd = ppm4_iface(W[R][n], W[R + 1][n], W[R + 2][n], W[R + 3][n]);  // face +3/2
        double aL = fa, aR = fb; ppm4_limit(W[R - 1][n], aL, aR); WLlo[n] = aR;
        aL = fb; aR = fc;        ppm4_limit(W[R][n], aL, aR);     WRlo[n] = aL; WLhi[n] = aR;
        aL = fc; aR = fd;        ppm4_limit(W[R + 1][n], aL, aR); WRhi[n] = aL;
      }
    }
    double Flo[5], Fhi[5];
    hllc(g, WLlo, WRlo, Flo);
    hllc(g, WLhi, WRhi, Fhi);
    const double cd = sc.c[lev][d];
    acc[0]  = acc[0]  - cd * (Fhi[0] - Flo[0]);
    acc[iu] = acc[iu] - cd * (Fhi[1] - Flo[1]);
    acc[iv] = acc[iv] - cd * (Fhi[2] - Flo[2]);
    acc[iw] = acc[iw] - cd * (Fhi[3] - Flo[3]);
    acc[4]  = acc[4]  - cd * (Fhi[4] - Flo[4]);
  }
#pragma unroll
  for (int n = 0; n < 5; n++) Uout[base + n * nc] = acc[n];
  if (nfl) atomicAdd(P.floor_cnt, (unsigned long long)nfl);
}

inline cudaError_t launch_stage_simple(const ak_pack& p, const double* Uin, const double* U0, double* Uout,
                                       const StageCoef& sc) {
  const PackDev& P = p.d;
  dim3 grid((P.nx[0] + 127) / 128, P.nx[1] * P.nx[2], P.nmb);
  if (p.recon == 0) stage_simple_kernel<0><<<grid, 128, 0, p.stream>>>(P, Uin, U0, Uout, sc);
  else              stage_simple_kernel<1><<<grid, 128, 0, p.stream>>>(P, Uin, U0, Uout, sc);
  return cudaGetLastError();
}

}  // namespace ak

// ak_fluxcorr.cuh -- flux correction at coarse-fine faces (paper P:57; optional, off by
// default because north_star's stage list omits it).  Runs after the stage kernel on refined meshes:
// for every face cell of a level-0 block whose neighbour across that face is refined, one thread
//   * recomputes the coarse flux F_c the stage kernel used at that face (same functions, same inputs: U_in of
//     the coarse block with its restricted ghosts),
//   * computes the four fine fluxes through the same area at the boundary face of the fine neighbour (U_in of
//     the fine block with its prolonged ghosts -- again exactly what the fine block's own update used),
//   * and replaces F_c by their mean in the coarse cell's update:  U_out -= +-c_d (mean(F_f) - F_c).
// Only the ~nx^2 face cells per coarse-fine block face do any work, so the face fluxes are recomputed from
// U_in instead of being written out by the stage kernel: no extra HBM traffic on the hot path, and the stage
// kernel stays as it is.  One launch per direction d (a cell can sit on level boundaries in two directions;
// launches in sequence keep its corrections in a fixed order, no atomics).
#pragma once
#include "ak_pack.h"
#include "ak_lean.cuh"          // recon2<>, flux3<>

namespace ak {

// flux of direction D at the lower D-face of cell `c` (index of variable 0 inside one block's U, stride st along D)
template <int RECON, int RS, int D>
__device__ __forceinline__ void face_flux_from_u(const GasConst& g, const double* __restrict__ Ub, long long nc, long long c,
                                                 long long st, double F[5]) {
  constexpr int R = (RECON == 0) ? 2 : 3;
  double w[5][2 * R];                       // primitives of cells c-R .. c+R-1 along D
#pragma unroll
  for (int a = 0; a < 2 * R; a++) {
    double u[5], ww[5];
#pragma unroll
    for (int n = 0; n < 5; n++) u[n] = Ub[n * nc + c + (a - R) * st];
    c2p_lean(u, ww, g.ug_floor);
#pragma unroll
    for (int n = 0; n < 5; n++) w[n][a] = ww[n];
  }
  double L[5], Rr[5];
#pragma unroll
  for (int n = 0; n < 5; n++) {
    double qm, qp;
    recon2<RECON>(&w[n][R - 1], 1, qm, qp); L[n] = qp;      // q+ of the cell on the - side
    recon2<RECON>(&w[n][R], 1, qm, qp);     Rr[n] = qm;     // q- of the cell on the + side
  }
  flux3<RS, D>(g, L, Rr, F);
}

template <int RECON, int RS, int D>
__global__ void __launch_bounds__(128) flux_correct_kernel(PackDev P, const double* __restrict__ Uin, double* __restrict__ Uout,
                                                           double cd) {
  constexpr int T1 = (D == 0) ? 1 : 0, T2 = (D == 2) ? 1 : 2;       // tangential directions, T1 faster
  const int m = blockIdx.z, side = blockIdx.y;
  const int4 b = P.blk[m];
  if (b.x != 0) return;
  int dd[3] = {0, 0, 0};
  dd[D] = side ? 1 : -1;
  if (P.nbr[27 * m + (dd[2] + 1) * 9 + (dd[1] + 1) * 3 + (dd[0] + 1)] >= 0) return;     // same-level neighbour
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= P.nx[T1] * P.nx[T2]) return;
  const int ng = P.ng;
  int cc[3];                                                         // coarse cell on the + side of the face
  cc[T2] = t / P.nx[T1] + ng; cc[T1] = t % P.nx[T1] + ng; cc[D] = side ? P.nx[D] + ng : ng;
  const long long nc = P.ncell;
  const long long str[3] = {1, P.nt[0], (long long)P.nt[0] * P.nt[1]};
  GasConst g;
  g.gamma = P.gamma; g.gm1 = P.gamma - 1.0;
  g.ug_floor = P_FLOOR / (P.gamma - 1.0);

  const long long c = cc[2] * str[2] + cc[1] * str[1] + cc[0];
  double Fc[5];
  face_flux_from_u<RECON, RS, D>(g, Uin + (long long)m * 5 * nc, nc, c, str[D], Fc);

  const int lxm[3] = {b.y, b.z, b.w};
  long long Gc[3];
  for (int e = 0; e < 3; e++) Gc[e] = (long long)lxm[e] * P.nx[e] + (cc[e] - ng);
  double Fm[5];
  {
    double f[2][2][5];
#pragma unroll
    for (int s2 = 0; s2 < 2; s2++)
#pragma unroll
      for (int s1 = 0; s1 < 2; s1++) {
        long long Gf[3];
        Gf[D] = 2 * Gc[D] - (side ? 0 : 1);                          // an active cell of the fine neighbour
        Gf[T1] = 2 * Gc[T1] + s1; Gf[T2] = 2 * Gc[T2] + s2;
        int cf[3], bf[3];
        for (int e = 0; e < 3; e++) {
          const long long N = (long long)(2 * P.nrb[e]) * P.nx[e];
          long long G = Gf[e] < 0 ? Gf[e] + N : (Gf[e] >= N ? Gf[e] - N : Gf[e]);
          bf[e] = (int)(G / P.nx[e]);
          cf[e] = (int)(G - (long long)bf[e] * P.nx[e]) + ng;
        }
        const int mf = P.leaf1[((long long)bf[2] * (2 * P.nrb[1]) + bf[1]) * (2 * P.nrb[0]) + bf[0]];
        if (!side) cf[D] += 1;                                       // the fine block's upper boundary face
        const long long cfi = cf[2] * str[2] + cf[1] * str[1] + cf[0];
        face_flux_from_u<RECON, RS, D>(g, Uin + (long long)mf * 5 * nc, nc, cfi, str[D], f[s2][s1]);
      }
#pragma unroll
    for (int n = 0; n < 5; n++) Fm[n] = 0.25 * ((f[0][0][n] + f[0][1][n]) + (f[1][0][n] + f[1][1][n]));
  }
  // the coarse cell that owns the face: the last active cell (upper face) or the first one (lower face)
  const long long cell = (long long)m * 5 * nc + (side ? c - str[D] : c);
  const double sgn = side ? -cd : cd;                               // U -= c_d (F_up - F_lo)
#pragma unroll
  for (int n = 0; n < 5; n++) Uout[cell + n * nc] = fma(sgn, Fm[n] - Fc[n], Uout[cell + n * nc]);
}

template <int RECON, int RS>
cudaError_t launch_flux_correction_t(const ak_pack& p, const double* Uin, double* Uout, const StageCoef& sc) {
  const PackDev& P = p.d;
  {
    dim3 grid((unsigned)((P.nx[1] * P.nx[2] + 127) / 128), 2, (unsigned)P.nmb);
    flux_correct_kernel<RECON, RS, 0><<<grid, 128, 0, p.stream>>>(P, Uin, Uout, sc.c[0][0]);
  }
  {
    dim3 grid((unsigned)((P.nx[0] * P.nx[2] + 127) / 128), 2, (unsigned)P.nmb);
    flux_correct_kernel<RECON, RS, 1><<<grid, 128, 0, p.stream>>>(P, Uin, Uout, sc.c[0][1]);
  }
  {
    dim3 grid((unsigned)((P.nx[0] * P.nx[1] + 127) / 128), 2, (unsigned)P.nmb);
    flux_correct_kernel<RECON, RS, 2><<<grid, 128, 0, p.stream>>>(P, Uin, Uout, sc.c[0][2]);
  }
  return cudaGetLastError();
}

}  // namespace ak

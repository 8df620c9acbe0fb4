// ak_fofc.cuh -- first-order flux correction (paper P:118; reading DESIGN.md Q31), optional.
// "If the density or pressure in any cell were to go negative, the fluxes on all faces of that cell are recalculated
// using first-order (piecewise constant) reconstruction and a diffusive LLF Riemann solver."
// The stage kernel is untouched: it writes its (tentative) result as always.  Then
//   fofc_flag_kernel    one thread per cell: flag = tentative rho <= 0 or E - |m|^2 / (2 rho) <= 0 (NaN included) for
//                       active cells, 0 for ghost cells; flagged cells are counted
//   fofc_ghost_kernel   the flags of the ghost cells, copied like the state (same-level neighbour or boundary image),
//                       so that both blocks sharing a face see the same pair of flags
//   fofc_fix_kernel     one thread per active cell with a flagged cell among itself and its six face neighbours: the cell
//                       is updated again from U_in and U0, every face with a flagged cell on either side with the LLF flux
//                       of the two cell-centred states, the others with the high-order flux recomputed from U_in by the
//                       same device functions the stage kernel used
// The last two return at once when the stage flagged nothing (the counter is read on the device: no host round trip).
// Single-level meshes; the production kernel's reconstruction / solver (template parameters RECON, RS).
#pragma once
#include "ak_pack.h"
#include "ak_lean.cuh"
#include "ak_fluxcorr.cuh"     // face_flux_from_u<>

namespace ak {

__global__ void __launch_bounds__(256) fofc_flag_kernel(PackDev P, const double* __restrict__ U, unsigned char* __restrict__ flags,
                                                        unsigned long long* __restrict__ cnt) {
  const int m = blockIdx.y;
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= P.ncell) return;
  const int n1 = P.nt[0], n2 = P.nt[1], ng = P.ng;
  const int i = (int)(c % n1), j = (int)((c / n1) % n2), k = (int)(c / ((long long)n1 * n2));
  unsigned char f = 0;
  if (i >= ng && i < P.nx[0] + ng && j >= ng && j < P.nx[1] + ng && k >= ng && k < P.nx[2] + ng) {
    const double* q = U + (long long)m * 5 * P.ncell + c;
    const double rho = q[0], m1 = q[P.ncell], m2 = q[2 * P.ncell], m3 = q[3 * P.ncell];
    const double eint = q[4 * P.ncell] - 0.5 * (m1 * m1 + (m2 * m2 + m3 * m3)) / rho;
    f = (!(rho > 0.0) || !(eint > 0.0)) ? 1 : 0;
    if (f) { atomicAdd(cnt, 1ull); atomicAdd(cnt + 1, 1ull); }      // this stage / since bind
  }
  flags[(long long)m * P.ncell + c] = f;
}

// image of ghost cell (i, j, k) of block m: source block and cell (same mapping as the state's copy-only ghost fill)
__device__ __forceinline__ long long ghost_image(const PackDev& P, int m, int i, int j, int k) {
  const int ng = P.ng, n1 = P.nt[0], n2 = P.nt[1];
  const int d1 = (i < ng) ? -1 : (i >= P.nx[0] + ng ? 1 : 0);
  const int d2 = (j < ng) ? -1 : (j >= P.nx[1] + ng ? 1 : 0);
  const int d3 = (k < ng) ? -1 : (k >= P.nx[2] + ng ? 1 : 0);
  const int dir = (d3 + 1) * 9 + (d2 + 1) * 3 + (d1 + 1);
  const int src = P.nbr[27 * m + dir];
  const int code = P.nbc[27 * m + dir];
  int si = i - d1 * P.nx[0], sj = j - d2 * P.nx[1], sk = k - d3 * P.nx[2];
  const int c1 = code & 3, c2 = (code >> 2) & 3, c3 = (code >> 4) & 3;
  if (c1) si = (c1 == 1) ? (d1 < 0 ? ng : P.nx[0] + ng - 1) : (d1 < 0 ? 2 * ng - 1 - i : 2 * (P.nx[0] + ng) - 1 - i);
  if (c2) sj = (c2 == 1) ? (d2 < 0 ? ng : P.nx[1] + ng - 1) : (d2 < 0 ? 2 * ng - 1 - j : 2 * (P.nx[1] + ng) - 1 - j);
  if (c3) sk = (c3 == 1) ? (d3 < 0 ? ng : P.nx[2] + ng - 1) : (d3 < 0 ? 2 * ng - 1 - k : 2 * (P.nx[2] + ng) - 1 - k);
  return (long long)src * P.ncell + ((long long)sk * n2 + sj) * n1 + si;
}

__global__ void __launch_bounds__(256) fofc_ghost_kernel(PackDev P, unsigned char* __restrict__ flags,
                                                         const unsigned long long* __restrict__ cnt) {
  if (*cnt == 0) return;
  const int m = blockIdx.y;
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= P.ncell) return;
  const int n1 = P.nt[0], n2 = P.nt[1], ng = P.ng;
  const int i = (int)(c % n1), j = (int)((c / n1) % n2), k = (int)(c / ((long long)n1 * n2));
  if (i >= ng && i < P.nx[0] + ng && j >= ng && j < P.nx[1] + ng && k >= ng && k < P.nx[2] + ng) return;
  flags[(long long)m * P.ncell + c] = flags[ghost_image(P, m, i, j, k)];
}

// flux at the lower D-face of cell c: LLF of the two cell-centred states where a flagged cell touches the face, else the
// high-order flux recomputed from U_in
template <int RECON, int RS, int D>
__device__ __forceinline__ void fofc_face(const GasConst& g, const double* __restrict__ Ub, long long nc, long long c,
                                          long long st, bool first_order, double F[5]) {
  if (first_order) {
    double uL[5], uR[5], wL[5], wR[5];
#pragma unroll
    for (int n = 0; n < 5; n++) { uL[n] = Ub[n * nc + c - st]; uR[n] = Ub[n * nc + c]; }
    c2p_lean(uL, wL, g.ug_floor);
    c2p_lean(uR, wR, g.ug_floor);
    flux3<1, D>(g, wL, wR, F);                                 // RS = 1: LLF
  } else {
    face_flux_from_u<RECON, RS, D>(g, Ub, nc, c, st, F);
  }
}

// A cell with a flagged cell among itself and its six face neighbours is updated again FROM SCRATCH (its tentative value
// may be NaN): U = g0 U_in + g1 U0 - sum_d c_d (F_hi - F_lo), evaluated left to right like the stage update.  U_out is
// never U0 here: with FOFC the last stage of a step writes a spare buffer instead of buffer A (ak_api.cu).
template <int RECON, int RS>
__global__ void __launch_bounds__(128) fofc_fix_kernel(PackDev P, const double* __restrict__ Uin, const double* __restrict__ U0,
                                                       double* __restrict__ Uout, const unsigned char* __restrict__ flags,
                                                       const unsigned long long* __restrict__ cnt, double g0, double g1,
                                                       double c1, double c2, double c3) {
  if (*cnt == 0) return;
  const int m = blockIdx.y;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long nact = (long long)P.nx[0] * P.nx[1] * P.nx[2];
  if (t >= nact) return;
  const int ng = P.ng;
  const int i = (int)(t % P.nx[0]) + ng, j = (int)((t / P.nx[0]) % P.nx[1]) + ng, k = (int)(t / ((long long)P.nx[0] * P.nx[1])) + ng;
  const long long nc = P.ncell;
  const long long str[3] = {1, P.nt[0], (long long)P.nt[0] * P.nt[1]};
  const long long c = k * str[2] + j * str[1] + i;
  const unsigned char* fb = flags + (long long)m * nc;
  const bool f0 = fb[c];
  const bool lo[3] = {f0 || fb[c - str[0]], f0 || fb[c - str[1]], f0 || fb[c - str[2]]};
  const bool hi[3] = {f0 || fb[c + str[0]], f0 || fb[c + str[1]], f0 || fb[c + str[2]]};
  if (!(lo[0] || lo[1] || lo[2] || hi[0] || hi[1] || hi[2])) return;
  GasConst g;
  g.gamma = P.gamma; g.gm1 = P.gamma - 1.0;
  g.ug_floor = P_FLOOR / (P.gamma - 1.0);
  const double* Ub = Uin + (long long)m * 5 * nc;
  const double* U0b = U0 + (long long)m * 5 * nc;
  double v[5], Fl[5], Fh[5];
#pragma unroll
  for (int n = 0; n < 5; n++) v[n] = fma(g0, Ub[n * nc + c], g1 * U0b[n * nc + c]);
  fofc_face<RECON, RS, 0>(g, Ub, nc, c, str[0], lo[0], Fl); fofc_face<RECON, RS, 0>(g, Ub, nc, c + str[0], str[0], hi[0], Fh);
#pragma unroll
  for (int n = 0; n < 5; n++) v[n] = fma(-c1, Fh[n] - Fl[n], v[n]);
  fofc_face<RECON, RS, 1>(g, Ub, nc, c, str[1], lo[1], Fl); fofc_face<RECON, RS, 1>(g, Ub, nc, c + str[1], str[1], hi[1], Fh);
#pragma unroll
  for (int n = 0; n < 5; n++) v[n] = fma(-c2, Fh[n] - Fl[n], v[n]);
  fofc_face<RECON, RS, 2>(g, Ub, nc, c, str[2], lo[2], Fl); fofc_face<RECON, RS, 2>(g, Ub, nc, c + str[2], str[2], hi[2], Fh);
#pragma unroll
  for (int n = 0; n < 5; n++) v[n] = fma(-c3, Fh[n] - Fl[n], v[n]);
  double* o = Uout + (long long)m * 5 * nc + c;
#pragma unroll
  for (int n = 0; n < 5; n++) o[n * nc] = v[n];
}

template <int RECON, int RS>
cudaError_t launch_fofc_t(const ak_pack& p, const double* Uin, const double* U0, double* Uout, const StageCoef& sc) {
  const PackDev& P = p.d;
  unsigned char* flags = p.fofc_flags;
  unsigned long long* cnt = p.fofc_cnt;
  cudaError_t e = cudaMemsetAsync(cnt, 0, 8, p.stream);
  if (e != cudaSuccess) return e;
  dim3 gall((unsigned)((P.ncell + 255) / 256), (unsigned)P.nmb);
  fofc_flag_kernel<<<gall, 256, 0, p.stream>>>(P, Uout, flags, cnt);
  fofc_ghost_kernel<<<gall, 256, 0, p.stream>>>(P, flags, cnt);
  const long long nact = (long long)P.nx[0] * P.nx[1] * P.nx[2];
  dim3 gact((unsigned)((nact + 127) / 128), (unsigned)P.nmb);
  fofc_fix_kernel<RECON, RS><<<gact, 128, 0, p.stream>>>(P, Uin, U0, Uout, flags, cnt, sc.g0, sc.g1, sc.c[0][0], sc.c[0][1], sc.c[0][2]);
  return cudaGetLastError();
}

}  // namespace ak

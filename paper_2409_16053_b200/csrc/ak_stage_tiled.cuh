// ak_stage_tiled.cuh -- the production ak_hydro_stage kernel: 2.5-D plane marching.
//
// A CTA owns a TI x TJ tile of (i,j) columns of one MeshBlock and marches along k over a chunk of
// planes; one thread per column.  Per plane:
//   L  load U of the plane (tile + cross-shaped halo of R cells), conserved->primitive, W -> shared memory
//   B  every thread reconstructs its own cell in x1 and x2 (q-, q+); q+ goes to shared memory for the
//      neighbour, q- stays in registers; the first wI+wJ threads also reconstruct the halo cells
//   C  every thread solves the HLLC problem at its lower x1 and x2 face and, from registers, at the
//      lower x3 face of the previous plane; the first wI+wJ threads solve the tile's upper-edge faces;
//      fluxes -> shared memory
//   D  flux divergence + RK weights; a plane is written once its upper x3 flux is known
// Each face flux is computed exactly once per tile (tile-edge faces twice, by the two tiles sharing them,
// with identical instruction sequences, so conservation holds to round-off) and never reaches HBM.
// The x3 direction lives in registers: own-column primitives of the last 2 (PLM) / 3 (PPM4) planes,
// the pending q+ and flux, and the partial updates t of the planes still waiting for their x3 flux.
#pragma once
#include "ak_pack.h"
#include "ak_physics.cuh"

namespace ak {

// rotate primitives so that component 1 is the face-normal velocity of direction D (cyclic transverse pair)
template <int D>
__device__ __forceinline__ void rot(const double w[5], double r[5]) {
  r[0] = w[0]; r[1] = w[1 + D]; r[2] = w[1 + (D + 1) % 3]; r[3] = w[1 + (D + 2) % 3]; r[4] = w[4];
}
template <int D>
__device__ __forceinline__ void flux_dir(const GasConst& g, const double L[5], const double Rr[5], double F[5]) {
  double l[5], r[5], f[5];
  rot<D>(L, l); rot<D>(Rr, r);
  hllc(g, l, r, f);
  F[0] = f[0]; F[1 + D] = f[1]; F[1 + (D + 1) % 3] = f[2]; F[1 + (D + 2) % 3] = f[3]; F[4] = f[4];
}

// reconstruct one cell along a line of primitives with stride `st` in shared memory: q- and q+ of the cell at p
template <int RECON>
__device__ __forceinline__ void recon_line(const double* p, int st, double& qm, double& qp) {
  if constexpr (RECON == 0) {
    double c = p[0];
    double h = plm_halfslope(p[-st], c, p[st]);
    qm = c - h; qp = c + h;
  } else {
    double a = p[0], m1 = p[-st], p1 = p[st];
    double lo = ppm4_iface(p[-2 * st], m1, a, p1);
    double hi = ppm4_iface(m1, a, p1, p[2 * st]);
    ppm4_limit(a, lo, hi);
    qm = lo; qp = hi;
  }
}

template <int RECON, int TI, int TJ>
struct TileSmem {
  static constexpr int R = (RECON == 0) ? 2 : 3;
  static constexpr int WI = TI + 2 * R, WJ = TJ + 2 * R;
  static constexpr int nW = 5 * WJ * WI, nQP1 = 5 * TJ * (TI + 1), nQP2 = 5 * (TJ + 1) * TI;
  static constexpr int total = nW + 2 * nQP1 + 2 * nQP2;     // + F1s, F2s of the same shapes
  static constexpr size_t bytes = sizeof(double) * total;
};

template <int RECON, int TI, int TJ>
__global__ void __launch_bounds__(TI * TJ, 2)
stage_tiled_kernel(PackDev P, const double* __restrict__ Uin, const double* U0, double* Uout, StageCoef sc,
                   int KC, int ntile_i) {
  using S = TileSmem<RECON, TI, TJ>;
  constexpr int R = S::R, WI = S::WI, WJ = S::WJ, NT = TI * TJ;
  constexpr int NP = R;                 // planes of partial updates waiting for their upper x3 flux
  extern __shared__ double smem[];
  double* Ws = smem;                    // [5][WJ][WI]      primitives of the current plane, halo included
  double* QP1 = Ws + S::nW;             // [5][TJ][TI+1]    q+ along x1 of cells i = -1 .. TI-1
  double* QP2 = QP1 + S::nQP1;          // [5][TJ+1][TI]    q+ along x2 of cells j = -1 .. TJ-1
  double* F1s = QP2 + S::nQP2;          // [5][TJ][TI+1]    x1 flux at faces i = 0 .. TI
  double* F2s = F1s + S::nQP1;          // [5][TJ+1][TI]    x2 flux at faces j = 0 .. TJ

  const int tid = threadIdx.x, ti = tid % TI, tj = tid / TI;
  const int tile_i = blockIdx.x % ntile_i, tile_j = blockIdx.x / ntile_i;
  const int i0 = tile_i * TI, j0 = tile_j * TJ, m = blockIdx.z;
  const int k0 = blockIdx.y * KC, k1 = min(k0 + KC, P.nx[2]);          // active planes [k0, k1)
  const int wI = min(TI, P.nx[0] - i0), wJ = min(TJ, P.nx[1] - j0);
  const bool valid = (ti < wI) && (tj < wJ);
  const int ng = P.ng, n1 = P.nt[0], n2 = P.nt[1];
  const long long nc = P.ncell;
  const long long plane = (long long)n1 * n2;
  const long long blk0 = (long long)m * 5 * nc;
  const long long col = blk0 + (long long)(j0 + tj + ng) * n1 + (i0 + ti + ng);   // own column, plane 0
  const int lev = P.blk[m].x;
  const double c1 = sc.c[lev][0], c2 = sc.c[lev][1], c3 = sc.c[lev][2];

  GasConst g;
  g.gamma = P.gamma; g.gm1 = P.gamma - 1.0;
  g.ug_floor = P_FLOOR / (P.gamma - 1.0);

  const int nextra = wI + wJ;           // threads that also handle halo cells / upper-edge faces
  const bool extra = tid < nextra;
  const bool ex1 = tid < wJ;            // extra for x1 (row tid) else for x2 (column tid - wJ)
  const int nhalo = 2 * R * (wI + wJ);

  // x3 pipeline state (registers)
  double wk[R][5];                      // own-column W of the previous R planes, wk[R-1] = newest
  double qlow[5];                       // PPM4: interface value at the lower face of the cell being limited
  double qp3[5];                        // q+ along x3 of the last reconstructed plane
  double G[5];                          // x3 flux at the lower face of the oldest pending plane
  double t[NP][5];                      // partial updates, t[0] = oldest pending plane
  int nfl = 0;
#pragma unroll
  for (int a = 0; a < R; a++)
#pragma unroll
    for (int n = 0; n < 5; n++) wk[a][n] = 1.0;
#pragma unroll
  for (int n = 0; n < 5; n++) { qlow[n] = 1.0; qp3[n] = 1.0; G[n] = 0.0; }
#pragma unroll
  for (int a = 0; a < NP; a++)
#pragma unroll
    for (int n = 0; n < 5; n++) t[a][n] = 0.0;

  for (int s = k0 - R; s < k1 + R; s++) {
    const bool inplane = (s >= k0) && (s < k1);
    const long long pl = (long long)(s + ng) * plane;
    // ---- L: load, c2p ---------------------------------------------------------------------------
    double wp[5] = {1.0, 0.0, 0.0, 0.0, 1.0};
    double tn[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (valid) {
      double u[5];
#pragma unroll
      for (int n = 0; n < 5; n++) u[n] = Uin[col + pl + n * nc];
      int f = c2p(u, wp, g.ug_floor);
      if (inplane) {
        nfl += f;
#pragma unroll
        for (int n = 0; n < 5; n++) {
          Ws[(n * WJ + tj + R) * WI + ti + R] = wp[n];
          tn[n] = sc.g0 * u[n] + sc.g1 * U0[col + pl + n * nc];
        }
      }
    }
    if (inplane) {
      for (int h = tid; h < nhalo; h += NT) {
        int ii, jj;
        if (h < 2 * R * wJ) { jj = h / (2 * R); int c = h - jj * (2 * R); ii = c < R ? c - R : wI + c - R; }
        else { int hh = h - 2 * R * wJ; int r = hh / wI; ii = hh - r * wI; jj = r < R ? r - R : wJ + r - R; }
        const long long a = blk0 + pl + (long long)(j0 + jj + ng) * n1 + (i0 + ii + ng);
        double u[5], w[5];
#pragma unroll
        for (int n = 0; n < 5; n++) u[n] = Uin[a + n * nc];
        c2p(u, w, g.ug_floor);
#pragma unroll
        for (int n = 0; n < 5; n++) Ws[(n * WJ + jj + R) * WI + ii + R] = w[n];
      }
      __syncthreads();
    }
    // ---- B: in-plane reconstruction -------------------------------------------------------------
    double qm1[5], qm2[5], qmE[5];
    if (inplane) {
      if (valid) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          const double* p = &Ws[(n * WJ + tj + R) * WI + ti + R];
          double qp;
          recon_line<RECON>(p, 1, qm1[n], qp);
          QP1[(n * TJ + tj) * (TI + 1) + ti + 1] = qp;
          recon_line<RECON>(p, WI, qm2[n], qp);
          QP2[(n * (TJ + 1) + tj + 1) * TI + ti] = qp;
        }
      }
      if (extra) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          double qm, qp;
          if (ex1) {
            const double* p = &Ws[(n * WJ + tid + R) * WI + R];          // row tid, cell i = 0
            recon_line<RECON>(p - 1, 1, qm, qp);  QP1[(n * TJ + tid) * (TI + 1)] = qp;      // cell i = -1
            recon_line<RECON>(p + wI, 1, qm, qp); qmE[n] = qm;                              // cell i = wI
          } else {
            const int c = tid - wJ;
            const double* p = &Ws[(n * WJ + R) * WI + c + R];            // column c, cell j = 0
            recon_line<RECON>(p - WI, WI, qm, qp);     QP2[(n * (TJ + 1)) * TI + c] = qp;   // cell j = -1
            recon_line<RECON>(p + wJ * WI, WI, qm, qp); qmE[n] = qm;                        // cell j = wJ
          }
        }
      }
      __syncthreads();
    }
    // ---- C: Riemann problems --------------------------------------------------------------------
    double F1lo[5], F2lo[5];
    if (inplane) {
      if (valid) {
        double L[5];
#pragma unroll
        for (int n = 0; n < 5; n++) L[n] = QP1[(n * TJ + tj) * (TI + 1) + ti];
        flux_dir<0>(g, L, qm1, F1lo);
#pragma unroll
        for (int n = 0; n < 5; n++) F1s[(n * TJ + tj) * (TI + 1) + ti] = F1lo[n];
#pragma unroll
        for (int n = 0; n < 5; n++) L[n] = QP2[(n * (TJ + 1) + tj) * TI + ti];
        flux_dir<1>(g, L, qm2, F2lo);
#pragma unroll
        for (int n = 0; n < 5; n++) F2s[(n * (TJ + 1) + tj) * TI + ti] = F2lo[n];
      }
      if (extra) {
        double L[5], F[5];
        if (ex1) {
#pragma unroll
          for (int n = 0; n < 5; n++) L[n] = QP1[(n * TJ + tid) * (TI + 1) + wI];
          flux_dir<0>(g, L, qmE, F);
#pragma unroll
          for (int n = 0; n < 5; n++) F1s[(n * TJ + tid) * (TI + 1) + wI] = F[n];
        } else {
          const int c = tid - wJ;
#pragma unroll
          for (int n = 0; n < 5; n++) L[n] = QP2[(n * (TJ + 1) + wJ) * TI + c];
          flux_dir<1>(g, L, qmE, F);
#pragma unroll
          for (int n = 0; n < 5; n++) F2s[(n * (TJ + 1) + wJ) * TI + c] = F[n];
        }
      }
    }
    // x3 (registers).  Let c = the plane whose cell can be reconstructed now that plane s has arrived:
    //   PLM: c = s-1 (needs s-2, s-1, s);  PPM4: c = s-2 (interface (c+1/2) needs s-3 .. s).
    // Then the flux at the LOWER face of c follows from q+ of plane c-1 (kept) and q- of c, and plane
    // c-1 is complete.
    if (valid) {
      const int c = s - (R - 1);
      double qm3[5], qpn[5];
#pragma unroll
      for (int n = 0; n < 5; n++) {
        if constexpr (RECON == 0) {
          double h = plm_halfslope(wk[0][n], wk[1][n], wp[n]);
          qm3[n] = wk[1][n] - h; qpn[n] = wk[1][n] + h;
        } else {
          double hi = ppm4_iface(wk[0][n], wk[1][n], wk[2][n], wp[n]);     // face between s-2 and s-1
          double lo = qlow[n];
          qlow[n] = hi;
          ppm4_limit(wk[1][n], lo, hi);
          qm3[n] = lo; qpn[n] = hi;
        }
      }
      if (c >= k0 && c <= k1) {                    // lower face of plane c is needed (uniform over the CTA)
        double Gn[5];
        flux_dir<2>(g, qp3, qm3, Gn);
        if (c > k0) {                              // plane c-1 complete: t[0] holds its in-plane part
#pragma unroll
          for (int n = 0; n < 5; n++)
            Uout[col + (long long)(c - 1 + ng) * plane + n * nc] = t[0][n] - c3 * (Gn[n] - G[n]);
        }
#pragma unroll
        for (int n = 0; n < 5; n++) G[n] = Gn[n];
      }
#pragma unroll
      for (int n = 0; n < 5; n++) qp3[n] = qpn[n];
    }
    // ---- D: in-plane flux divergence ------------------------------------------------------------
    if (inplane) {
      __syncthreads();
      if (valid) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          double v = tn[n];
          v = v - c1 * (F1s[(n * TJ + tj) * (TI + 1) + ti + 1] - F1lo[n]);
          v = v - c2 * (F2s[(n * (TJ + 1) + tj + 1) * TI + ti] - F2lo[n]);
          tn[n] = v;
        }
      }
    }
    // rotate the pipelines
#pragma unroll
    for (int a = 0; a + 1 < NP; a++)
#pragma unroll
      for (int n = 0; n < 5; n++) t[a][n] = t[a + 1][n];
#pragma unroll
    for (int n = 0; n < 5; n++) t[NP - 1][n] = tn[n];
#pragma unroll
    for (int a = 0; a + 1 < R; a++)
#pragma unroll
      for (int n = 0; n < 5; n++) wk[a][n] = wk[a + 1][n];
#pragma unroll
    for (int n = 0; n < 5; n++) wk[R - 1][n] = wp[n];
  }
  if (nfl) atomicAdd(P.floor_cnt, (unsigned long long)nfl);
}

template <int RECON, int TI, int TJ>
cudaError_t launch_tiled(const ak_pack& p, const double* Uin, const double* U0, double* Uout, const StageCoef& sc) {
  using S = TileSmem<RECON, TI, TJ>;
  const PackDev& P = p.d;
  auto kern = stage_tiled_kernel<RECON, TI, TJ>;
  static bool attr_set_dev[64] = {};   // the opt-in to > 48 KB of dynamic shared memory is per device
  bool& attr_set = attr_set_dev[p.device & 63];
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::bytes);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const int nti = (P.nx[0] + TI - 1) / TI, ntj = (P.nx[1] + TJ - 1) / TJ;
  const long long ntiles = (long long)nti * ntj * P.nmb;
  const long long target = (long long)p.sm_count * 2 * 8;        // >= 8 waves of 2 CTAs per SM
  int nchunk = (int)((target + ntiles - 1) / ntiles);
  int maxchunk = P.nx[2] / 8 > 0 ? P.nx[2] / 8 : 1;
  if (nchunk > maxchunk) nchunk = maxchunk;
  if (nchunk < 1) nchunk = 1;
  const int KC = (P.nx[2] + nchunk - 1) / nchunk;
  nchunk = (P.nx[2] + KC - 1) / KC;
  dim3 grid(nti * ntj, nchunk, P.nmb);
  kern<<<grid, TI * TJ, S::bytes, p.stream>>>(P, Uin, U0, Uout, sc, KC, nti);
  return cudaGetLastError();
}

inline cudaError_t launch_stage_tiled(const ak_pack& p, const double* Uin, const double* U0, double* Uout,
                                      const StageCoef& sc) {
  const bool narrow = p.d.nx[0] <= 16;
  if (p.recon == 0) return narrow ? launch_tiled<0, 16, 16>(p, Uin, U0, Uout, sc) : launch_tiled<0, 32, 8>(p, Uin, U0, Uout, sc);
  return narrow ? launch_tiled<1, 16, 16>(p, Uin, U0, Uout, sc) : launch_tiled<1, 32, 8>(p, Uin, U0, Uout, sc);
}

}  // namespace ak

// ak_stage_tma.cuh -- the production ak_hydro_stage kernel: TMA-staged 2.5-D plane marching.
//
// A CTA owns a TI x TJ tile of (i,j) columns of one MeshBlock and marches along k; one thread per column.
// Each k-plane of the tile WITH its R ghost/halo layers in i and j (all 5 variables) is fetched by ONE
// 5-D bulk-tensor copy (TMA, cp.async.bulk.tensor.5d) into a two-deep shared-memory ring, armed on an
// mbarrier one full plane ahead of its use, so no thread issues a global load for the stencil data and
// the DRAM/L2 latency is hidden behind a whole plane of arithmetic.  Per plane:
//   L  wait for the plane; conserved->primitive IN PLACE in shared memory (tile + cross-shaped halo)
//   B  every thread reconstructs its cell in x1 and x2; q+ -> shared memory, q- stays in registers;
//      x3 is reconstructed from the thread's own register pipeline of the last R planes
//   C  HLLC at the thread's lower x1, x2 faces (and, from registers, at the lower x3 face of the plane
//      that just became reconstructible); fluxes overwrite the q+ slots they consumed
//   D  in-plane flux divergence + RK weights -> a ring of partial updates in shared memory; a plane is
//      written to global memory once its upper x3 flux is known (R planes later)
// Face fluxes never reach device memory.  Tile-edge faces are solved by both tiles sharing them with the
// same instruction sequence, so conservation holds to round-off.
#pragma once
#include "ak_pack.h"
#include "ak_physics.cuh"
#include "ak_tma.cuh"

namespace ak {

template <int D>
__device__ __forceinline__ void flux_lean(const GasConst& g, const double L[5], const double Rr[5], double F[5]) {
  double l[5] = {L[0], L[1 + D], L[1 + (D + 1) % 3], L[1 + (D + 2) % 3], L[4]};
  double r[5] = {Rr[0], Rr[1 + D], Rr[1 + (D + 1) % 3], Rr[1 + (D + 2) % 3], Rr[4]};
  double f[5];
  hllc_lean(g, l, r, f);
  F[0] = f[0]; F[1 + D] = f[1]; F[1 + (D + 1) % 3] = f[2]; F[1 + (D + 2) % 3] = f[3]; F[4] = f[4];
}

template <int RECON>
__device__ __forceinline__ void recon_cell(const double* p, int st, double& qm, double& qp) {
  if constexpr (RECON == 0) {
    double c = p[0];
    double dL = c - p[-st], dR = p[st] - c, prod = dL * dR;
    double h = (prod > 0.0) ? div_lean(prod, dL + dR) : 0.0;
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
struct TmaTile {
  static constexpr int R = (RECON == 0) ? 2 : 3;
  static constexpr int WI = TI + 2 * R, WJ = TJ + 2 * R, NT = TI * TJ;
  static constexpr int nU = 5 * WJ * WI;                              // doubles per staged plane
  static constexpr int nUpad = (nU + 15) & ~15;                       // keep every buffer 128-B aligned
  static constexpr int nQ1 = 5 * TJ * (TI + 1), nQ2 = 5 * (TJ + 1) * TI;
  static constexpr int nT = R * 5 * NT;
  static constexpr int total = 2 * nUpad + ((nQ1 + nQ2 + 15) & ~15) + nT;
  static constexpr size_t bytes = sizeof(double) * total + 64 + 128;  // + mbarriers + alignment slack
  static constexpr unsigned tx_bytes = nU * 8;
};

template <int RECON, int TI, int TJ, bool STAGE2>
__global__ void __launch_bounds__(TI * TJ, 2)
stage_tma_kernel(const __grid_constant__ CUtensorMap tmU, PackDev P, const double* __restrict__ U0,
                 double* __restrict__ Uout, StageCoef sc, int KC, int ntile_i) {
  using S = TmaTile<RECON, TI, TJ>;
  constexpr int R = S::R, WI = S::WI, WJ = S::WJ, NT = S::NT;
  extern __shared__ unsigned char smem_raw[];
  double* smem = reinterpret_cast<double*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~(uintptr_t)127);
  double* Ub = smem;                            // [2][5][WJ][WI]  staged U plane, converted to W in place
  double* Q1 = Ub + 2 * S::nUpad;               // [5][TJ][TI+1]   q+ along x1 of cells -1..TI-1, then F1 at faces 0..TI
  double* Q2 = Q1 + S::nQ1;                     // [5][TJ+1][TI]   q+ along x2 of cells -1..TJ-1, then F2 at faces 0..TJ
  double* Tr = Q1 + ((S::nQ1 + S::nQ2 + 15) & ~15);   // [R][5][NT] partial updates waiting for their upper x3 flux
  uint64_t* bars = reinterpret_cast<uint64_t*>(Tr + S::nT);

  const int tid = threadIdx.x, ti = tid % TI, tj = tid / TI;
  const int tile_i = blockIdx.x % ntile_i, tile_j = blockIdx.x / ntile_i;
  const int i0 = tile_i * TI, j0 = tile_j * TJ, m = blockIdx.z;
  const int k0 = blockIdx.y * KC, k1 = min(k0 + KC, P.nx[2]);
  const int wI = min(TI, P.nx[0] - i0), wJ = min(TJ, P.nx[1] - j0);
  const bool valid = (ti < wI) && (tj < wJ);
  const int ng = P.ng;
  const long long nc = P.ncell;
  const long long plane = (long long)P.nt[0] * P.nt[1];
  const long long col = (long long)m * 5 * nc + (long long)(j0 + tj + ng) * P.nt[0] + (i0 + ti + ng);
  const int lev = P.blk[m].x;
  const double c1 = sc.c[lev][0], c2 = sc.c[lev][1], c3 = sc.c[lev][2];
  const int ci = i0 + ng - R, cj = j0 + ng - R;         // box origin in the (i, j) plane

  GasConst g;
  g.gamma = P.gamma; g.gm1 = P.gamma - 1.0; g.gq = (P.gamma + 1.0) / (2.0 * P.gamma);
  g.ug_floor = P_FLOOR / (P.gamma - 1.0);

  if (tid == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbar_init();
    mbar_expect_tx(&bars[0], S::tx_bytes);
    tma_load_5d(Ub, &tmU, &bars[0], ci, cj, k0 - R + ng, 0, m);
  }
  __syncthreads();

  const int nextra = wI + wJ;
  const bool extra = tid < nextra;
  const bool ex1 = tid < wJ;
  const int nhalo = 2 * R * (wI + wJ);

  double wk[R][5], qlow[5], qp3[5], G[5];
  int nfl = 0;
#pragma unroll
  for (int a = 0; a < R; a++)
#pragma unroll
    for (int n = 0; n < 5; n++) wk[a][n] = 1.0;
#pragma unroll
  for (int n = 0; n < 5; n++) { qlow[n] = 1.0; qp3[n] = 1.0; G[n] = 0.0; }

  int it = 0;
  for (int s = k0 - R; s < k1 + R; s++, it++) {
    const int b = it & 1;
    const bool inplane = (s >= k0) && (s < k1);
    const int slot = (s - k0 + R) % R;
    double* Ws = Ub + b * S::nUpad;
    // ---- L ----------------------------------------------------------------------------------------
    double u0[5];
    if constexpr (STAGE2) {
      if (inplane && valid) {
#pragma unroll
        for (int n = 0; n < 5; n++) u0[n] = __ldg(&U0[col + (long long)(s + ng) * plane + n * nc]);
      }
    }
    mbar_wait(&bars[b], (it >> 1) & 1);
    double wp[5] = {1.0, 0.0, 0.0, 0.0, 1.0};
    double tn[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (valid) {
      double u[5];
#pragma unroll
      for (int n = 0; n < 5; n++) u[n] = Ws[(n * WJ + tj + R) * WI + ti + R];
      int f = c2p(u, wp, g.ug_floor);
      if (inplane) {
        nfl += f;
#pragma unroll
        for (int n = 0; n < 5; n++) {
          Ws[(n * WJ + tj + R) * WI + ti + R] = wp[n];
          if constexpr (STAGE2) tn[n] = sc.g0 * u[n] + sc.g1 * u0[n];
          else tn[n] = u[n];                     // 0*U + 1*U of the stage-1 weights, exactly
        }
      }
    }
    if (inplane) {
      for (int h = tid; h < nhalo; h += NT) {
        int ii, jj;
        if (h < 2 * R * wJ) { jj = h / (2 * R); int c = h - jj * (2 * R); ii = c < R ? c - R : wI + c - R; }
        else { int hh = h - 2 * R * wJ; int r = hh / wI; ii = hh - r * wI; jj = r < R ? r - R : wJ + r - R; }
        double u[5], w[5];
#pragma unroll
        for (int n = 0; n < 5; n++) u[n] = Ws[(n * WJ + jj + R) * WI + ii + R];
        c2p(u, w, g.ug_floor);
#pragma unroll
        for (int n = 0; n < 5; n++) Ws[(n * WJ + jj + R) * WI + ii + R] = w[n];
      }
    }
    __syncthreads();
    // the other ring slot was last read before this barrier: refill it with the next plane
    if (tid == 0 && s + 1 < k1 + R) {
      fence_proxy_async();
      mbar_expect_tx(&bars[b ^ 1], S::tx_bytes);
      tma_load_5d(Ub + (b ^ 1) * S::nUpad, &tmU, &bars[b ^ 1], ci, cj, s + 1 + ng, 0, m);
    }
    // ---- B ----------------------------------------------------------------------------------------
    double qm1[5], qm2[5], qmE[5];
    if (inplane) {
      if (valid) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          const double* p = &Ws[(n * WJ + tj + R) * WI + ti + R];
          double qp;
          recon_cell<RECON>(p, 1, qm1[n], qp);
          Q1[(n * TJ + tj) * (TI + 1) + ti + 1] = qp;
          recon_cell<RECON>(p, WI, qm2[n], qp);
          Q2[(n * (TJ + 1) + tj + 1) * TI + ti] = qp;
        }
      }
      if (extra) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          double qm, qp;
          if (ex1) {
            const double* p = &Ws[(n * WJ + tid + R) * WI + R];
            recon_cell<RECON>(p - 1, 1, qm, qp);  Q1[(n * TJ + tid) * (TI + 1)] = qp;
            recon_cell<RECON>(p + wI, 1, qm, qp); qmE[n] = qm;
          } else {
            const int c = tid - wJ;
            const double* p = &Ws[(n * WJ + R) * WI + c + R];
            recon_cell<RECON>(p - WI, WI, qm, qp);      Q2[(n * (TJ + 1)) * TI + c] = qp;
            recon_cell<RECON>(p + wJ * WI, WI, qm, qp); qmE[n] = qm;
          }
        }
      }
    }
    // x3 reconstruction of plane c = s-(R-1) from the register pipeline (no shared memory involved)
    double qm3[5], qpn[5];
    if (valid) {
#pragma unroll
      for (int n = 0; n < 5; n++) {
        if constexpr (RECON == 0) {
          double a = wk[1][n];
          double dL = a - wk[0][n], dR = wp[n] - a, prod = dL * dR;
          double h = (prod > 0.0) ? div_lean(prod, dL + dR) : 0.0;
          qm3[n] = a - h; qpn[n] = a + h;
        } else {
          double hi = ppm4_iface(wk[0][n], wk[1][n], wk[2][n], wp[n]);
          double lo = qlow[n];
          qlow[n] = hi;
          ppm4_limit(wk[1][n], lo, hi);
          qm3[n] = lo; qpn[n] = hi;
        }
      }
    }
    __syncthreads();
    // ---- C ----------------------------------------------------------------------------------------
    double F1lo[5], F2lo[5];
    if (inplane) {
      if (valid) {
        double L[5];
#pragma unroll
        for (int n = 0; n < 5; n++) L[n] = Q1[(n * TJ + tj) * (TI + 1) + ti];
        flux_lean<0>(g, L, qm1, F1lo);
#pragma unroll
        for (int n = 0; n < 5; n++) Q1[(n * TJ + tj) * (TI + 1) + ti] = F1lo[n];
#pragma unroll
        for (int n = 0; n < 5; n++) L[n] = Q2[(n * (TJ + 1) + tj) * TI + ti];
        flux_lean<1>(g, L, qm2, F2lo);
#pragma unroll
        for (int n = 0; n < 5; n++) Q2[(n * (TJ + 1) + tj) * TI + ti] = F2lo[n];
      }
      if (extra) {
        double L[5], F[5];
        if (ex1) {
#pragma unroll
          for (int n = 0; n < 5; n++) L[n] = Q1[(n * TJ + tid) * (TI + 1) + wI];
          flux_lean<0>(g, L, qmE, F);
#pragma unroll
          for (int n = 0; n < 5; n++) Q1[(n * TJ + tid) * (TI + 1) + wI] = F[n];
        } else {
          const int c = tid - wJ;
#pragma unroll
          for (int n = 0; n < 5; n++) L[n] = Q2[(n * (TJ + 1) + wJ) * TI + c];
          flux_lean<1>(g, L, qmE, F);
#pragma unroll
          for (int n = 0; n < 5; n++) Q2[(n * (TJ + 1) + wJ) * TI + c] = F[n];
        }
      }
    }
    if (valid) {
      const int c = s - (R - 1);
      if (c >= k0 && c <= k1) {                    // lower x3 face of plane c (uniform over the CTA)
        double Gn[5];
        flux_lean<2>(g, qp3, qm3, Gn);
        if (c > k0) {                              // plane c-1 complete
#pragma unroll
          for (int n = 0; n < 5; n++)
            Uout[col + (long long)(c - 1 + ng) * plane + n * nc] = Tr[(slot * 5 + n) * NT + tid] - c3 * (Gn[n] - G[n]);
        }
#pragma unroll
        for (int n = 0; n < 5; n++) G[n] = Gn[n];
      }
#pragma unroll
      for (int n = 0; n < 5; n++) qp3[n] = qpn[n];
    }
    // ---- D ----------------------------------------------------------------------------------------
    if (inplane) {
      __syncthreads();
      if (valid) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          double v = tn[n];
          v = v - c1 * (Q1[(n * TJ + tj) * (TI + 1) + ti + 1] - F1lo[n]);
          v = v - c2 * (Q2[(n * (TJ + 1) + tj + 1) * TI + ti] - F2lo[n]);
          Tr[(slot * 5 + n) * NT + tid] = v;
        }
      }
    }
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
cudaError_t launch_tma(const ak_pack& p, const double* Uin, const double* U0, double* Uout, const StageCoef& sc,
                       bool stage2) {
  using S = TmaTile<RECON, TI, TJ>;
  const PackDev& P = p.d;
  if (p.tmap_box[0] != S::WI || p.tmap_box[1] != S::WJ) {
    for (int b = 0; b < 2; b++)
      if (!make_state_tmap(&p.tmap[b], p.u[b], P.nmb, P.nt, S::WI, S::WJ)) return cudaErrorNotSupported;
    p.tmap_box[0] = S::WI; p.tmap_box[1] = S::WJ;
  }
  const CUtensorMap& tm = (Uin == p.u[0]) ? p.tmap[0] : p.tmap[1];
  auto k1 = stage_tma_kernel<RECON, TI, TJ, false>;
  auto k2 = stage_tma_kernel<RECON, TI, TJ, true>;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::bytes);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const int nti = (P.nx[0] + TI - 1) / TI, ntj = (P.nx[1] + TJ - 1) / TJ;
  const long long ntiles = (long long)nti * ntj * P.nmb;
  const long long target = (long long)p.sm_count * 2 * 8;        // >= 8 waves of 2 CTAs per SM
  int nchunk = (int)((target + ntiles - 1) / ntiles);
  int maxchunk = P.nx[2] / 16 > 0 ? P.nx[2] / 16 : 1;
  if (nchunk > maxchunk) nchunk = maxchunk;
  if (nchunk < 1) nchunk = 1;
  const int KC = (P.nx[2] + nchunk - 1) / nchunk;
  nchunk = (P.nx[2] + KC - 1) / KC;
  dim3 grid(nti * ntj, nchunk, P.nmb);
  if (stage2) k2<<<grid, TI * TJ, S::bytes, p.stream>>>(tm, P, U0, Uout, sc, KC, nti);
  else        k1<<<grid, TI * TJ, S::bytes, p.stream>>>(tm, P, U0, Uout, sc, KC, nti);
  return cudaGetLastError();
}

inline cudaError_t launch_stage_tma(const ak_pack& p, const double* Uin, const double* U0, double* Uout,
                                    const StageCoef& sc) {
  const bool narrow = p.d.nx[0] <= 16;
  const bool stage2 = (Uin != U0);
  if (p.recon == 0) return narrow ? launch_tma<0, 16, 16>(p, Uin, U0, Uout, sc, stage2) : launch_tma<0, 32, 8>(p, Uin, U0, Uout, sc, stage2);
  return narrow ? launch_tma<1, 16, 16>(p, Uin, U0, Uout, sc, stage2) : launch_tma<1, 32, 8>(p, Uin, U0, Uout, sc, stage2);
}

}  // namespace ak

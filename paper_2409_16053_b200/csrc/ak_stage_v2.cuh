// ak_stage_v2.cuh -- production ak_hydro_stage kernel: TMA-staged 2.5-D plane marching,
// second generation.  Written against the ncu evidence of profiles/r01_v1_stage_cfg3.md: the path is bound
// by the FP64 pipe, and v1 lost 4x to register spills (128-register cap), to ~2 200 non-FP64 instructions
// per cell (moves/selects from fmin/fmax, generic-address shared loads, divergent limiter branches) and to
// three CTA-wide barriers per plane at 16 warps per SM.
//
// A CTA owns a TI x TJ tile of (i,j) columns of one MeshBlock and marches along k, one thread per column:
//   * each k-plane of the tile WITH its R halo layers in i and j, all 5 variables, arrives by ONE 5-D
//     cp.async.bulk.tensor (TMA) into a two-slot shared-memory ring, armed on an mbarrier a plane ahead;
//   * launch bounds give every thread 168 registers (2 CTAs of 192 threads per SM), enough to keep the x3
//     pipeline (the column's last R primitive planes, pending interface value, q+ and flux) in registers
//     without spilling;
//   * TWO barriers per plane.  Per iteration s (plane s already converted to primitives in slot b):
//       B(s)    reconstruct own cell in x1, x2: q+ -> Q[b] (the L state of the upper face), q- in registers
//       ---- barrier 1 ----   TMA for plane s+2 is issued into slot b
//       C(s)    HLLC at the lower x1 / x2 faces; fluxes overwrite the q+ they consumed in Q[b]
//       L(s+1)  wait for plane s+1 (slot b^1), conserved->primitive in place (+ cross-shaped halo), RK-weighted
//               old state -> T ring; x3 reconstruction + HLLC from registers; the plane whose upper x3 flux
//               just became known is written to global memory
//       ---- barrier 2 ----
//       D(s)    in-plane flux divergence into the T ring (thread-private slots)
//     Q is double-buffered by plane parity so that D(s) and B(s+1) need no barrier between them.
//   * all shared-memory traffic uses shared-space addresses (LDS/STS), all limiter / wave-speed logic is
//     straight-line (ak_lean.cuh), and the tile-edge faces (x1 and x2) run through one instruction stream.
// Face fluxes never reach device memory.  Tile-edge faces are solved by both tiles sharing them with the
// same arithmetic on the same inputs (the translation unit is compiled with -fmad=false and every fused
// multiply-add is written out), so results do not depend on the tiling or on the block decomposition.
#pragma once
#include "ak_pack.h"
#include "ak_lean.cuh"
#include "ak_tma.cuh"

namespace ak {

template <int RECON>
__device__ __forceinline__ void recon2(const double* p, int st, double& qm, double& qp) {
  if constexpr (RECON == 0) {
    plm_lean(p[-st], p[0], p[st], qm, qp);
  } else {
    const double m2 = p[-2 * st], m1 = p[-st], a = p[0], p1 = p[st], p2 = p[2 * st];
    double lo = iface_lean(m2, m1, a, p1);
    double hi = iface_lean(m1, a, p1, p2);
    limit_lean(a, lo, hi);
    qm = lo; qp = hi;
  }
}

template <int RECON, int TI, int TJ>
struct V2Tile {
  static constexpr int R = (RECON == 0) ? 2 : 3;
  static constexpr int WI = TI + 2 * R, WJ = TJ + 2 * R, NT = TI * TJ;
  static constexpr int nU = 5 * WJ * WI;                              // doubles per staged plane
  static constexpr int nUpad = (nU + 15) & ~15;                       // keep every slot 128-B aligned
  static constexpr int nQ1 = 5 * TJ * (TI + 1), nQ2 = 5 * (TJ + 1) * TI;
  static constexpr int nQ = (nQ1 + nQ2 + 15) & ~15;
  static constexpr int NS = R + 1;                                    // T-ring slots
  static constexpr int nT = NS * 5 * NT;
  static constexpr int oQ = 2 * nUpad, oT = oQ + 2 * nQ, oBar = oT + nT;
  static constexpr size_t bytes = sizeof(double) * oBar + 64;
  static constexpr unsigned tx_bytes = nU * 8;
  static constexpr int NH = (2 * R * (TI + TJ) + NT - 1) / NT;        // halo cells per thread (1 or 2)
  static_assert(TI + TJ <= NT, "one tile-edge face per thread");
};

template <int RECON, int TI, int TJ, int MINB, bool STAGE2>
__global__ void __launch_bounds__(TI * TJ, MINB)
stage_v2_kernel(const __grid_constant__ CUtensorMap tmU, PackDev P, const double* __restrict__ U0,
                double* __restrict__ Uout, StageCoef sc, int KC, int ntile_i) {
  using S = V2Tile<RECON, TI, TJ>;
  constexpr int R = S::R, WI = S::WI, WJ = S::WJ, NT = S::NT, NS = S::NS, NH = S::NH;
  extern __shared__ __align__(1024) double sm[];
  // sm[0 .. 2 nUpad)        staged U plane ring, converted to W in place      [2][5][WJ][WI]
  // sm[oQ .. oQ + 2 nQ)     per plane parity: Q1 [5][TJ][TI+1] (q+ along x1 of cells -1..TI-1, then F1 at
  //                         faces 0..TI) and Q2 [5][TJ+1][TI]
  // sm[oT .. oT + nT)       T ring [NS][5][NT]: partial updates waiting for their upper x3 flux
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + S::oBar);

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
  const int send = k1 + R;                              // planes k0-R .. send-1 are staged

  GasConst g;
  g.gamma = P.gamma; g.gm1 = P.gamma - 1.0; g.gq = (P.gamma + 1.0) / (2.0 * P.gamma);
  g.ug_floor = P_FLOOR / (P.gamma - 1.0);

  if (tid == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbar_init();
    mbar_expect_tx(&bars[0], S::tx_bytes);
    tma_load_5d(sm, &tmU, &bars[0], ci, cj, k0 - R + ng, 0, m);
    mbar_expect_tx(&bars[1], S::tx_bytes);
    tma_load_5d(sm + S::nUpad, &tmU, &bars[1], ci, cj, k0 - R + 1 + ng, 0, m);
  }
  __syncthreads();

  // per-thread constant offsets
  const int oW = (tj + R) * WI + ti + R;                // own cell inside a staged plane (variable stride WJ*WI)
  const int oQ1 = tj * (TI + 1) + ti;                   // lower x1 face of the own cell   (variable stride TJ*(TI+1))
  const int oQ2 = tj * TI + ti;                         // lower x2 face of the own cell   (variable stride (TJ+1)*TI)
  // cross-shaped halo: NH cells per thread, offsets fixed for the whole march
  int oH[NH];
  {
    const int nh1 = 2 * R * wJ, nhalo = nh1 + 2 * R * wI;
#pragma unroll
    for (int q = 0; q < NH; q++) {
      const int h = tid + q * NT;
      oH[q] = -1;
      if (h < nhalo) {
        int ii, jj;
        if (h < nh1) { jj = h / (2 * R); const int c = h - jj * (2 * R); ii = c < R ? c - R : wI + c - R; }
        else { const int hh = h - nh1; const int r = hh / wI; ii = hh - r * wI; jj = r < R ? r - R : wJ + r - R; }
        oH[q] = (jj + R) * WI + ii + R;
      }
    }
  }
  // tile-edge faces: thread e < wJ solves the upper x1 face of row e, thread wJ <= e < wJ+wI the upper x2 face
  // of column e-wJ; both kinds share one instruction stream (stride / offsets differ)
  const bool extra = tid < wI + wJ;
  const bool ex2 = tid >= wJ;
  int eA = 0, eB = 0, eSt = 1, eQlo = 0, eQhi = 0, eQn = 0;
  if (extra) {
    if (!ex2) {             // row tid: cells -1 and wI along x1
      eSt = 1; eA = (tid + R) * WI + R - 1; eB = (tid + R) * WI + R + wI;
      eQlo = tid * (TI + 1); eQhi = tid * (TI + 1) + wI; eQn = TJ * (TI + 1);
    } else {                // column c: cells -1 and wJ along x2
      const int c = tid - wJ;
      eSt = WI; eA = (R - 1) * WI + c + R; eB = (R + wJ) * WI + c + R;
      eQlo = S::nQ1 + c; eQhi = S::nQ1 + wJ * TI + c; eQn = (TJ + 1) * TI;
    }
  }

  double wk[R][5], qlow[5], qp3[5], G[5];
  int nfl = 0;
#pragma unroll
  for (int a = 0; a < R; a++)
#pragma unroll
    for (int n = 0; n < 5; n++) wk[a][n] = 1.0;
#pragma unroll
  for (int n = 0; n < 5; n++) { qlow[n] = 1.0; qp3[n] = 1.0; G[n] = 0.0; }

  // L(s): conserved -> primitive of plane s in ring slot `slot_u`, T-ring bookkeeping, x3 pipeline
  int tslot = 0;                                        // T-ring slot of the plane being converted
  auto phaseL = [&](int s, int it) {
    const bool inplane = (s >= k0) && (s < k1);
    double* Ws = sm + (it & 1) * S::nUpad;
    double u0[5];
    if constexpr (STAGE2) {
      if (inplane && valid) {
#pragma unroll
        for (int n = 0; n < 5; n++) u0[n] = __ldg(&U0[col + (long long)(s + ng) * plane + n * nc]);
      }
    }
    mbar_wait(&bars[it & 1], (it >> 1) & 1);
    double wp[5] = {1.0, 0.0, 0.0, 0.0, 1.0};
    if (valid) {
      double u[5];
#pragma unroll
      for (int n = 0; n < 5; n++) u[n] = Ws[n * (WJ * WI) + oW];
      const int f = c2p_lean(u, wp, g.ug_floor);
      if (inplane) {
        nfl += f;
        double* Tn = sm + S::oT + tslot * (5 * NT) + tid;
#pragma unroll
        for (int n = 0; n < 5; n++) {
          Ws[n * (WJ * WI) + oW] = wp[n];
          if constexpr (STAGE2) Tn[n * NT] = fma(sc.g0, u[n], sc.g1 * u0[n]);
          else Tn[n * NT] = u[n];                  // 0*U + 1*U of the stage-1 weights, exactly
        }
      }
    }
    if (inplane) {
#pragma unroll
      for (int q = 0; q < NH; q++) {
        if (oH[q] >= 0) {
          double u[5], w[5];
#pragma unroll
          for (int n = 0; n < 5; n++) u[n] = Ws[n * (WJ * WI) + oH[q]];
          c2p_lean(u, w, g.ug_floor);
#pragma unroll
          for (int n = 0; n < 5; n++) Ws[n * (WJ * WI) + oH[q]] = w[n];
        }
      }
    }
    // x3: plane c = s-(R-1) becomes reconstructible; its lower face flux completes plane c-1
    if (valid) {
      double qm3[5], qpn[5];
#pragma unroll
      for (int n = 0; n < 5; n++) {
        if constexpr (RECON == 0) {
          plm_lean(wk[0][n], wk[1][n], wp[n], qm3[n], qpn[n]);
        } else {
          double hi = iface_lean(wk[0][n], wk[1][n], wk[2][n], wp[n]);
          double lo = qlow[n];
          qlow[n] = hi;
          limit_lean(wk[1][n], lo, hi);
          qm3[n] = lo; qpn[n] = hi;
        }
      }
      const int c = s - (R - 1);
      if (c >= k0 && c <= k1) {                    // uniform over the CTA
        double Gn[5];
        flux2<2>(g, qp3, qm3, Gn);
        if (c > k0) {                              // plane c-1 complete: its slot is the one after tslot
          const int ts = (tslot + 1 == NS) ? 0 : tslot + 1;
          const double* Tc = sm + S::oT + ts * (5 * NT) + tid;
          double* o = Uout + col + (long long)(c - 1 + ng) * plane;
#pragma unroll
          for (int n = 0; n < 5; n++) o[n * nc] = fma(-c3, Gn[n] - G[n], Tc[n * NT]);
        }
#pragma unroll
        for (int n = 0; n < 5; n++) G[n] = Gn[n];
      }
#pragma unroll
      for (int n = 0; n < 5; n++) qp3[n] = qpn[n];
    }
#pragma unroll
    for (int a = 0; a + 1 < R; a++)
#pragma unroll
      for (int n = 0; n < 5; n++) wk[a][n] = wk[a + 1][n];
#pragma unroll
    for (int n = 0; n < 5; n++) wk[R - 1][n] = wp[n];
  };

  int it = 0;
  phaseL(k0 - R, 0);
  int dslot = 0;                                        // T-ring slot of plane s (the one D(s) updates)
  for (int s = k0 - R; s < send; s++, it++) {
    const int b = it & 1;
    const bool inplane = (s >= k0) && (s < k1);
    const double* Ws = sm + b * S::nUpad;
    double* Q = sm + S::oQ + b * S::nQ;
    double* Q1 = Q;
    double* Q2 = Q + S::nQ1;
    // ---- B(s)  (W(s) was completed before barrier 2 of the previous iteration; the prologue plane is never
    //            in-plane, so the first pass through B does nothing) --------------------------------------------------------------------------------------
    double qm1[5], qm2[5], qmE[5];
    if (inplane) {
      if (valid) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          const double* p = Ws + n * (WJ * WI) + oW;
          double qp;
          recon2<RECON>(p, 1, qm1[n], qp);
          Q1[n * (TJ * (TI + 1)) + oQ1 + 1] = qp;
          recon2<RECON>(p, WI, qm2[n], qp);
          Q2[n * ((TJ + 1) * TI) + oQ2 + TI] = qp;
        }
      }
      if (extra) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          double qm, qp;
          recon2<RECON>(Ws + n * (WJ * WI) + eA, eSt, qm, qp);
          Q[n * eQn + eQlo] = qp;
          recon2<RECON>(Ws + n * (WJ * WI) + eB, eSt, qmE[n], qp);
        }
      }
    }
    __syncthreads();                                    // q+ visible; every read of W(s) is done
    if (tid == 0 && s + 2 < send) {                     // refill slot b with plane s+2
      fence_proxy_async();
      mbar_expect_tx(&bars[b], S::tx_bytes);
      tma_load_5d(sm + b * S::nUpad, &tmU, &bars[b], ci, cj, s + 2 + ng, 0, m);
    }
    // ---- C(s) --------------------------------------------------------------------------------------
    if (inplane) {
      if (valid) {
        double L[5], F[5];
#pragma unroll
        for (int n = 0; n < 5; n++) L[n] = Q1[n * (TJ * (TI + 1)) + oQ1];
        flux2<0>(g, L, qm1, F);
#pragma unroll
        for (int n = 0; n < 5; n++) Q1[n * (TJ * (TI + 1)) + oQ1] = F[n];
#pragma unroll
        for (int n = 0; n < 5; n++) L[n] = Q2[n * ((TJ + 1) * TI) + oQ2];
        flux2<1>(g, L, qm2, F);
#pragma unroll
        for (int n = 0; n < 5; n++) Q2[n * ((TJ + 1) * TI) + oQ2] = F[n];
      }
      if (extra) {
        double L[5], F[5];
#pragma unroll
        for (int n = 0; n < 5; n++) L[n] = Q[n * eQn + eQhi];
        flux2_12(g, ex2, L, qmE, F);
#pragma unroll
        for (int n = 0; n < 5; n++) Q[n * eQn + eQhi] = F[n];
      }
    }
    // ---- L(s+1) ------------------------------------------------------------------------------------
    if (s + 1 < send) {
      tslot = (dslot + 1 == NS) ? 0 : dslot + 1;
      phaseL(s + 1, it + 1);
    }
    __syncthreads();                                    // fluxes of plane s visible
    // ---- D(s) --------------------------------------------------------------------------------------
    if (inplane && valid) {
      double* Td = sm + S::oT + dslot * (5 * NT) + tid;
#pragma unroll
      for (int n = 0; n < 5; n++) {
        const double* q1 = Q1 + n * (TJ * (TI + 1)) + oQ1;
        const double* q2 = Q2 + n * ((TJ + 1) * TI) + oQ2;
        double v = Td[n * NT];
        v = fma(-c1, q1[1] - q1[0], v);
        v = fma(-c2, q2[TI] - q2[0], v);
        Td[n * NT] = v;
      }
    }
    dslot = (dslot + 1 == NS) ? 0 : dslot + 1;
  }
  if (nfl) atomicAdd(P.floor_cnt, (unsigned long long)nfl);
}

template <int RECON, int TI, int TJ, int MINB>
cudaError_t launch_v2(const ak_pack& p, const double* Uin, const double* U0, double* Uout, const StageCoef& sc,
                      bool stage2) {
  using S = V2Tile<RECON, TI, TJ>;
  const PackDev& P = p.d;
  if (p.tmap_box[0] != S::WI || p.tmap_box[1] != S::WJ) {
    for (int b = 0; b < 2; b++)
      if (!make_state_tmap(&p.tmap[b], p.u[b], P.nmb, P.nt, S::WI, S::WJ)) return cudaErrorNotSupported;
    p.tmap_box[0] = S::WI; p.tmap_box[1] = S::WJ;
  }
  const CUtensorMap& tm = (Uin == p.u[0]) ? p.tmap[0] : p.tmap[1];
  auto k1 = stage_v2_kernel<RECON, TI, TJ, MINB, false>;
  auto k2 = stage_v2_kernel<RECON, TI, TJ, MINB, true>;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::bytes);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const int nti = (P.nx[0] + TI - 1) / TI, ntj = (P.nx[1] + TJ - 1) / TJ;
  const long long ntiles = (long long)nti * ntj * P.nmb;
  // split k only when the tiles alone cannot fill the machine a few times over
  const long long target = (long long)p.sm_count * MINB * 4;
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

}  // namespace ak

// ak_stage_v3.cuh -- production ak_hydro_stage kernel: TMA-staged 2.5-D plane marching.
// A CTA owns a TI x TJ tile of (i, j) columns of one MeshBlock and marches along k:
//   * each k-plane of the tile WITH its R halo layers, all 5 variables, arrives by ONE 5-D cp.async.bulk.tensor
//     (TMA) into a two-slot shared-memory ring, armed on an mbarrier two planes ahead; in stage 2 a second box
//     brings U0 = U^n of the tile's columns on the same mbarrier;
//   * the CTA is NT = TI x TJ WORKER threads (one per column) plus ONE EDGE WARP whose lanes own the TI + TJ
//     tile-edge faces (reconstruct the two halo cells, solve the upper-edge face) and whose lane 0 issues the
//     TMA copies.  The edge warp has less work per plane than a worker warp, so it is never the one the
//     barrier waits for, and the workers' instruction stream contains no edge code.
// Per iteration s (plane s already converted to primitives in slot b = it & 1):
//       B(s)    workers: reconstruct own cell in x1, x2: q+ -> Q[b], q- in registers
//               edge:    reconstruct halo cells -1 and wI (wJ): q+ of -1 -> Q[b], q- of wI in registers
//       ---- barrier 1 ----   edge lane 0 issues the TMA for plane s+2 (and its U0 box) into slot b
//       C(s)    workers: HLLC at the lower x1 / x2 faces; edge: HLLC at the upper edge face; F overwrites q+
//       L(s+1)  workers: wait for plane s+1, conserved->primitive in place (+ cross-shaped halo), RK-weighted
//               old state -> T ring; x3 reconstruction + HLLC from registers; completed plane -> global
//       ---- barrier 2 ----
//       D(s)    workers: in-plane flux divergence into the T ring (thread-private slots)
// Face fluxes never reach device memory.  Tile-edge faces are solved by the edge warps of both tiles sharing
// them with the same arithmetic on the same inputs (-fmad=false, every fused multiply-add written out), so
// results do not depend on the tiling or on the block decomposition.
#pragma once
#include "ak_pack.h"
#include "ak_lean.cuh"
#include "ak_tma.cuh"

namespace ak {

template <int RECON, int TI, int TJ>
struct V3Tile {
  static constexpr int R = (RECON == 0) ? 2 : 3;
  static constexpr int WI = TI + 2 * R, WJ = TJ + 2 * R, NT = TI * TJ, NTH = NT + 32;
  static constexpr int nU = 5 * WJ * WI;                              // doubles per staged plane
  static constexpr int nUpad = (nU + 15) & ~15;                       // keep every slot 128-B aligned
  static constexpr int nQ1 = 5 * TJ * (TI + 1), nQ2 = 5 * (TJ + 1) * TI;
  static constexpr int nQ = (nQ1 + nQ2 + 15) & ~15;
  static constexpr int NS = R + 1;                                    // T-ring slots
  static constexpr int nT = NS * 5 * NT;
  static constexpr int W0 = TI + 2;                                   // U0 box width (16-B aligned origin)
  static constexpr int nU0 = 5 * TJ * W0;
  static constexpr int nU0pad = (nU0 + 15) & ~15;
  static constexpr int oQ = 2 * nUpad, oT = oQ + 2 * nQ, oU0 = (oT + nT + 15) & ~15, oBar = oU0 + 2 * nU0pad;
  static constexpr size_t bytes = sizeof(double) * oBar + 64;
  static constexpr unsigned tx_bytes = nU * 8, tx0_bytes = nU0 * 8;
  static constexpr int NH = (2 * R * (TI + TJ) + NT - 1) / NT;        // halo cells per worker (1 or 2)
  static constexpr int NE = (TI + TJ + 31) / 32;                      // tile-edge faces per lane of the edge warp
};

// Ghost fill fused into the stage (uniform periodic meshes with nx_d >= 2 ng): the thread that writes
// active cell (gi, gj, f) of block m also stores it into the ghost cells that are its periodic image in the
// neighbouring blocks -- the block in direction E holds it at the index shifted by -E * nx.  (e1, e2, e3) say which
// face the cell is within ng of in each direction (0: none); its images are the up to 7 non-empty sub-selections.
// Exact copies of what ak_fill_ghosts would copy in a separate pass over the state; only threads near a block face
// come here (loops not unrolled: the hot loop keeps its size).
__device__ __forceinline__ void push_ghosts(const PackDev& P, double* __restrict__ Uout, int m, int gi, int gj, int f,
                                         int e1, int e2, int e3, double u0, double u1, double u2, double u3, double u4) {
  const int ng = P.ng;
  const long long nc = P.ncell;
  const int* nb = P.nbr + 27 * m;
#pragma unroll 1
  for (int a3 = 0; a3 <= (e3 != 0); a3++)
#pragma unroll 1
    for (int a2 = 0; a2 <= (e2 != 0); a2++)
#pragma unroll 1
      for (int a1 = 0; a1 <= (e1 != 0); a1++) {
        if (!(a1 | a2 | a3)) continue;
        const int E1 = a1 ? e1 : 0, E2 = a2 ? e2 : 0, E3 = a3 ? e3 : 0;
        const int dst = nb[(E3 + 1) * 9 + (E2 + 1) * 3 + (E1 + 1)];
        double* o = Uout + (long long)dst * 5 * nc +
                    ((long long)(f + ng - E3 * P.nx[2]) * P.nt[1] + (gj + ng - E2 * P.nx[1])) * P.nt[0] + (gi + ng - E1 * P.nx[0]);
        o[0] = u0; o[nc] = u1; o[2 * nc] = u2; o[3 * nc] = u3; o[4 * nc] = u4;
      }
}

__device__ __forceinline__ void cta_sync(int nthreads) {
  asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}

template <int RECON, int RS, int TI, int TJ, int MINB, bool STAGE2>
__global__ void __launch_bounds__(TI * TJ + 32, MINB)
stage_v3_kernel(const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmU0, PackDev P,
                double* __restrict__ Uout, StageCoef sc, int KC, int ntile_i) {
  using S = V3Tile<RECON, TI, TJ>;
  constexpr int R = S::R, WI = S::WI, WJ = S::WJ, NT = S::NT, NS = S::NS, NH = S::NH, NTH = S::NTH;
  constexpr bool SHARE = (RECON == 1);        // PPM4: every interface value computed once and shared through the Q slots
  // ... and the edge warp converts the cross-shaped halo where that balances the schedulers (measured: PLM and PPM4;
  // not PPMX / WENOZ, whose edge warp is the heavy one)
  constexpr bool EDGEHALO = (RECON <= 1);
  extern __shared__ __align__(1024) double sm[];
  // sm[0 .. 2 nUpad)        staged U plane ring, converted to W in place      [2][5][WJ][WI]
  // sm[oQ .. oQ + 2 nQ)     per plane parity: Q1 [5][TJ][TI+1] (q+ along x1 of cells -1..TI-1, then F1 at
  //                         faces 0..TI) and Q2 [5][TJ+1][TI]
  // sm[oT .. oT + nT)       T ring [NS][5][NT]: partial updates waiting for their upper x3 flux
  // sm[oU0 .. + 2 nU0pad)   stage 2: U0 = U^n of the tile's active columns     [2][5][TJ][TI+2]
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + S::oBar);

  const int tid = threadIdx.x;
  const int tile_i = blockIdx.x % ntile_i, tile_j = blockIdx.x / ntile_i;
  const int i0 = tile_i * TI, j0 = tile_j * TJ, m = blockIdx.z;
  const int k0 = blockIdx.y * KC, k1 = min(k0 + KC, P.nx[2]);
  const int wI = min(TI, P.nx[0] - i0), wJ = min(TJ, P.nx[1] - j0);
  const int ng = P.ng;
  const int ci = i0 + ng - R, cj = j0 + ng - R;         // box origin of the staged plane in (i, j)
  const int o0 = ng & 1;                                // U0 box starts o0 cells left of the tile (16-B aligned)
  const int send = k1 + R;                              // planes k0-R .. send-1 are staged

  GasConst g;
  g.gamma = P.gamma; g.gm1 = P.gamma - 1.0;
  g.ug_floor = P_FLOOR / (P.gamma - 1.0);

  // plane p (absolute active index, may lie in the ghost layers) -> ring slot `slot`, armed on bars[slot]
  auto issue = [&](int p, int slot) {
    const bool u0 = STAGE2 && p >= k0 && p < k1;
    mbar_expect_tx(&bars[slot], S::tx_bytes + (u0 ? S::tx0_bytes : 0u));
    tma_load_5d(sm + slot * S::nUpad, &tmU, &bars[slot], ci, cj, p + ng, 0, m);
    if (u0) tma_load_5d(sm + S::oU0 + slot * S::nU0pad, &tmU0, &bars[slot], i0 + ng - o0, j0 + ng, p + ng, 0, m);
  };

  if (tid == NT) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbar_init();
    issue(k0 - R, 0);
    issue(k0 - R + 1, 1);
  }
  cta_sync(NTH);

  // =================================== edge warp ======================================================
  if (tid >= NT) {
    // edge face e < wJ is the upper x1 face of row e, wJ <= e < wJ+wI the upper x2 face of column e-wJ; both
    // kinds share one instruction stream (stride / offsets differ).  Lane l owns faces l, l+32, ...
    constexpr int NE = S::NE;
    const int lane = tid - NT;
    bool extra[NE], ex2[NE];
    int eA[NE], eB[NE], eSt[NE], eQlo[NE], eQhi[NE], eQn[NE];
#pragma unroll
    for (int q = 0; q < NE; q++) {
      const int e = lane + 32 * q;
      extra[q] = e < wI + wJ;
      ex2[q] = e >= wJ;
      eA[q] = eB[q] = eQlo[q] = eQhi[q] = 0; eSt[q] = 1; eQn[q] = 0;
      if (extra[q]) {
        if (!ex2[q]) {          // row e: cells -1 and wI along x1
          eSt[q] = 1; eA[q] = (e + R) * WI + R - 1; eB[q] = (e + R) * WI + R + wI;
          eQlo[q] = e * (TI + 1); eQhi[q] = e * (TI + 1) + wI; eQn[q] = TJ * (TI + 1);
        } else {                // column c: cells -1 and wJ along x2
          const int c = e - wJ;
          eSt[q] = WI; eA[q] = (R - 1) * WI + c + R; eB[q] = (R + wJ) * WI + c + R;
          eQlo[q] = S::nQ1 + c; eQhi[q] = S::nQ1 + wJ * TI + c; eQn[q] = (TJ + 1) * TI;
        }
      }
    }
    // cross-shaped halo of the tile (2 R (wI + wJ) cells per plane), NHE cells per lane, offsets fixed for the whole march
    constexpr int NHE = EDGEHALO ? (2 * R * (TI + TJ) + 31) / 32 : 1;
    int eH[NHE];
    if constexpr (EDGEHALO) {
      const int nh1 = 2 * R * wJ, nhalo = nh1 + 2 * R * wI;
#pragma unroll
      for (int q = 0; q < NHE; q++) {
        const int h = lane + 32 * q;
        eH[q] = -1;
        if (h < nhalo) {
          int ii, jj;
          if (h < nh1) { jj = h / (2 * R); const int c = h - jj * (2 * R); ii = c < R ? c - R : wI + c - R; }
          else { const int hh = h - nh1; const int r = hh / wI; ii = hh - r * wI; jj = r < R ? r - R : wJ + r - R; }
          eH[q] = (jj + R) * WI + ii + R;
        }
      }
    }
    int it = 0;
    for (int s = k0 - R; s < send - 1; s++, it++) {   // (iteration send-1 would have nothing to do)
      const int b = it & 1;
      const bool inplane = (s >= k0) && (s < k1);
      const double* Ws = sm + b * S::nUpad;
      double* Q = sm + S::oQ + b * S::nQ;
      double qmE[NE][5];
      if constexpr (SHARE) {
        // PPM4 with interface values computed once per face: B1 -- the interface below halo cell -1 (register), the
        // two interfaces of halo cell wI (the lower one also into the slot worker wI-1 reads as its upper interface)
        double loA[NE][5], loB[NE][5], hiB[NE][5];
#pragma unroll
        for (int q = 0; q < NE; q++) {
          if (inplane && extra[q]) {
#pragma unroll
            for (int n = 0; n < 5; n++) {
              const double* pa = Ws + n * (WJ * WI) + eA[q];
              const double* pb = Ws + n * (WJ * WI) + eB[q];
              const int st = eSt[q];
              loA[q][n] = iface_lean(pa[-2 * st], pa[-st], pa[0], pa[st]);
              loB[q][n] = iface_lean(pb[-2 * st], pb[-st], pb[0], pb[st]);
              hiB[q][n] = iface_lean(pb[-st], pb[0], pb[st], pb[2 * st]);
              Q[n * eQn[q] + eQhi[q]] = loB[q][n];
            }
          }
        }
        cta_sync(NTH);                                  // interface values visible
        // B2 -- limit the two halo cells: q+ of cell -1 replaces worker 0's interface value in its slot, q- of cell wI stays here
#pragma unroll
        for (int q = 0; q < NE; q++) {
          if (inplane && extra[q]) {
#pragma unroll
            for (int n = 0; n < 5; n++) {
              double lo = loA[q][n], hi = Q[n * eQn[q] + eQlo[q]];
              limit_lean(Ws[n * (WJ * WI) + eA[q]], lo, hi);
              Q[n * eQn[q] + eQlo[q]] = hi;
              double lo2 = loB[q][n], hi2 = hiB[q][n];
              limit_lean(Ws[n * (WJ * WI) + eB[q]], lo2, hi2);
              qmE[q][n] = lo2;
            }
          }
        }
      } else {
#pragma unroll
        for (int q = 0; q < NE; q++) {
          if (inplane && extra[q]) {
#pragma unroll
            for (int n = 0; n < 5; n++) {
              double qm, qp;
              recon2<RECON>(Ws + n * (WJ * WI) + eA[q], eSt[q], qm, qp);
              Q[n * eQn[q] + eQlo[q]] = qp;
              recon2<RECON>(Ws + n * (WJ * WI) + eB[q], eSt[q], qmE[q][n], qp);
            }
          }
        }
      }
      cta_sync(NTH);                                    // q+ visible; every read of W(s) is done
      if (lane == 0 && s + 2 < send) {                  // refill slot b with plane s+2
        fence_proxy_async();
        issue(s + 2, b);
      }
#pragma unroll
      for (int q = 0; q < NE; q++) {
        if (inplane && extra[q]) {
          double L[5], F[5];
#pragma unroll
          for (int n = 0; n < 5; n++) L[n] = Q[n * eQn[q] + eQhi[q]];
          flux3_12<RS>(g, ex2[q], L, qmE[q], F);
#pragma unroll
          for (int n = 0; n < 5; n++) Q[n * eQn[q] + eQhi[q]] = F[n];
        }
      }
      if constexpr (EDGEHALO) {
        // conserved -> primitive of the halo cells of plane s+1 (the workers convert their own cells meanwhile)
        if (s + 1 >= k0 && s + 1 < k1) {
          double* Wn = sm + ((it + 1) & 1) * S::nUpad;
          mbar_wait(&bars[(it + 1) & 1], ((it + 1) >> 1) & 1);
#pragma unroll
          for (int q = 0; q < NHE; q++) {
            if (eH[q] >= 0) {
              double u[5], w[5];
#pragma unroll
              for (int n = 0; n < 5; n++) u[n] = Wn[n * (WJ * WI) + eH[q]];
              c2p_lean(u, w, g.ug_floor);
#pragma unroll
              for (int n = 0; n < 5; n++) Wn[n * (WJ * WI) + eH[q]] = w[n];
            }
          }
        }
      }
      cta_sync(NTH);                                    // fluxes of plane s visible
    }
    return;
  }

  // =================================== workers ========================================================
  const int ti = tid % TI, tj = tid / TI;
  const bool valid = (ti < wI) && (tj < wJ);
  const long long nc = P.ncell;
  const long long plane = (long long)P.nt[0] * P.nt[1];
  const long long col = (long long)m * 5 * nc + (long long)(j0 + tj + ng) * P.nt[0] + (i0 + ti + ng);
  const int lev = P.blk[m].x;
  const double c1 = sc.c[lev][0], c2 = sc.c[lev][1], c3 = sc.c[lev][2];
  // fused ghost fill: is this column within ng of an x1 / x2 face of its block?
  const int pe1 = !sc.push ? 0 : (i0 + ti < ng ? -1 : (i0 + ti >= P.nx[0] - ng ? 1 : 0));
  const int pe2 = !sc.push ? 0 : (j0 + tj < ng ? -1 : (j0 + tj >= P.nx[1] - ng ? 1 : 0));
  // where this column's copies live in the in-plane neighbour blocks (x1 neighbour, x2 neighbour, the diagonal one): element
  // offsets of the column at plane 0, fixed for the whole march, or -1; planes near an x3 face take the general loop
  // (only where 168 registers are available: the three-CTA PLM tile keeps the general loop, measured faster there)
  constexpr bool FASTPUSH = (MINB <= 2);
  long long pc1 = -1, pc2 = -1, pc12 = -1;
  if (FASTPUSH && (pe1 | pe2)) {
    const int* nb = P.nbr + 27 * m + 9;                 // (E3 = 0)
    const long long r0 = (long long)(j0 + tj + ng) * P.nt[0] + (i0 + ti + ng);
    const long long s1 = (long long)pe1 * P.nx[0], s2 = (long long)pe2 * P.nx[1] * P.nt[0];
    if (pe1) pc1 = (long long)nb[3 + (pe1 + 1)] * 5 * nc + r0 - s1;
    if (pe2) pc2 = (long long)nb[(pe2 + 1) * 3 + 1] * 5 * nc + r0 - s2;
    if (pe1 && pe2) pc12 = (long long)nb[(pe2 + 1) * 3 + (pe1 + 1)] * 5 * nc + r0 - s1 - s2;
  }

  const int oW = (tj + R) * WI + ti + R;                // own cell inside a staged plane (variable stride WJ*WI)
  const int oQ1 = tj * (TI + 1) + ti;                   // lower x1 face of the own cell   (variable stride TJ*(TI+1))
  const int oQ2 = tj * TI + ti;                         // lower x2 face of the own cell   (variable stride (TJ+1)*TI)
  const int oU0 = tj * S::W0 + ti + o0;                 // own cell inside a staged U0 box (variable stride TJ*W0)
  // cross-shaped halo: NH cells per worker, offsets fixed for the whole march
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

  constexpr int NW = (RECON >= 2) ? 4 : R;            // x3 window: PPMX / WENOZ need the five planes p-4 .. p
  double wk[NW][5], qlow[5], qp3[5], G[5];
  // stage 2: max signal speed per direction over this thread's cells, kept as BIT PATTERNS: for x >= 0 they order
  // like the doubles, and every NaN / +inf orders above all finite values, so a corrupted cell is not skipped
  unsigned long long smax[3] = {0ull, 0ull, 0ull};
  int nfl = 0;
#pragma unroll
  for (int a = 0; a < NW; a++)
#pragma unroll
    for (int n = 0; n < 5; n++) wk[a][n] = 1.0;
#pragma unroll
  for (int n = 0; n < 5; n++) { qlow[n] = 1.0; qp3[n] = 1.0; G[n] = 0.0; }

  // L(s): conserved -> primitive of plane s in ring slot it & 1, T-ring bookkeeping, x3 pipeline
  int tslot = 0;                                        // T-ring slot of the plane being converted
  // Straight-line on purpose: the x3 pipeline (wk, qlow, qp3, G) is updated unconditionally and only the
  // stores are predicated, so that no conditional assignment of loop-carried registers (= register copies
  // at every join) is left.  Threads outside a ragged tile and planes outside [k0, k1] compute on whatever
  // the (zero-filled) staging holds; nothing of that is ever stored.
  auto phaseL = [&](int s, int it) {
    const bool inplane = (s >= k0) && (s < k1);
    double* Ws = sm + (it & 1) * S::nUpad;
    mbar_wait(&bars[it & 1], (it >> 1) & 1);
    double wp[5];
    {
      double u[5];
#pragma unroll
      for (int n = 0; n < 5; n++) u[n] = Ws[n * (WJ * WI) + oW];
      const int f = c2p_lean(u, wp, g.ug_floor);
      nfl += (inplane && valid) ? f : 0;
      double* Tn = sm + S::oT + tslot * (5 * NT) + tid;
      const double* U0s = sm + S::oU0 + (it & 1) * S::nU0pad + oU0;
#pragma unroll
      for (int n = 0; n < 5; n++) {
        if (valid) Ws[n * (WJ * WI) + oW] = wp[n];   // (outside a ragged tile this cell is another thread's halo)
        if constexpr (STAGE2) Tn[n * NT] = fma(sc.g0, u[n], sc.g1 * U0s[n * (TJ * S::W0)]);
        else Tn[n * NT] = u[n];                    // 0*U + 1*U of the stage-1 weights, exactly
      }
    }
    if (!EDGEHALO && inplane) {
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
    double qm3[5], qpn[5];
    if constexpr (RECON == 0) {                    // the five reciprocal seeds in flight together (as in B)
      double prod[5], r[5], den[5];
#pragma unroll
      for (int n = 0; n < 5; n++) {
        const double dL = wk[1][n] - wk[0][n], dR = wp[n] - wk[1][n];
        prod[n] = dL * dR; den[n] = dL + dR;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r[n]) : "d"(den[n]));
      }
#pragma unroll
      for (int n = 0; n < 5; n++) {
        const double e = fma(-den[n], r[n], 1.0);
        const double q = prod[n] * fma(r[n], fma(e, e, e), r[n]);
        const double h = pos(prod[n]) ? q : 0.0;
        qm3[n] = wk[1][n] - h; qpn[n] = wk[1][n] + h;
      }
    }
#pragma unroll
    for (int n = 0; n < 5; n++) {
      if constexpr (RECON == 0) {
      } else if constexpr (RECON >= 2) {
        const double qv[5] = {wk[0][n], wk[1][n], wk[2][n], wk[3][n], wp[n]};
        recon5<RECON>(qv, qm3[n], qpn[n]);
      } else {
        double hi = iface_lean(wk[0][n], wk[1][n], wk[2][n], wp[n]);
        double lo = qlow[n];
        qlow[n] = hi;
        limit_lean(wk[1][n], lo, hi);
        qm3[n] = lo; qpn[n] = hi;
      }
    }
    const int c = s - (R - 1);
    double Gn[5];
    flux3<RS, 2>(g, qp3, qm3, Gn);
    if (c > k0 && c <= k1 && valid) {              // plane c-1 complete: its slot is the one after tslot
      const int ts = (tslot + 1 == NS) ? 0 : tslot + 1;
      const double* Tc = sm + S::oT + ts * (5 * NT) + tid;
      double* o = Uout + col + (long long)(c - 1 + ng) * plane;
      double un[5];
#pragma unroll
      for (int n = 0; n < 5; n++) { un[n] = fma(-c3, Gn[n] - G[n], Tc[n * NT]); o[n * nc] = un[n]; }
      const int pe3 = !sc.push ? 0 : (c - 1 < ng ? -1 : (c - 1 >= P.nx[2] - ng ? 1 : 0));
      if (pe3 || (!FASTPUSH && (pe1 | pe2))) {
        push_ghosts(P, Uout, m, i0 + ti, j0 + tj, c - 1, pe1, pe2, pe3, un[0], un[1], un[2], un[3], un[4]);
      } else if (pe1 | pe2) {
        const long long po = (long long)(c - 1 + ng) * plane;
        if (pc1 >= 0) { double* q = Uout + pc1 + po; q[0] = un[0]; q[nc] = un[1]; q[2 * nc] = un[2]; q[3 * nc] = un[3]; q[4 * nc] = un[4]; }
        if (pc2 >= 0) { double* q = Uout + pc2 + po; q[0] = un[0]; q[nc] = un[1]; q[2 * nc] = un[2]; q[3 * nc] = un[3]; q[4 * nc] = un[4]; }
        if (pc12 >= 0) { double* q = Uout + pc12 + po; q[0] = un[0]; q[nc] = un[1]; q[2 * nc] = un[2]; q[3 * nc] = un[3]; q[4 * nc] = un[4]; }
      }
      if (STAGE2 && sc.take_dt) {                  // (uniform over the grid)
        // S0 of the NEXT step (Eq.(3)) on U^{n+1} while it is in registers: the cell's signal speeds
        // |v_d| + c_s in the oracle's arithmetic (IEEE division and sqrt, no contraction: this translation unit
        // is compiled with -fmad=false), so that ak_new_dt need not read the state again
        double rho = un[0];
        if (!(rho >= RHO_FLOOR)) rho = RHO_FLOOR;
        const double rinv = 1.0 / rho;
        double ug = un[4] - 0.5 * rinv * (un[1] * un[1] + (un[2] * un[2] + un[3] * un[3]));
        if (!(ug >= g.ug_floor)) ug = g.ug_floor;
        const double cs = sqrt(g.gamma * (g.gm1 * ug) / rho);
#pragma unroll
        for (int d = 0; d < 3; d++) {
          const unsigned long long b = (unsigned long long)__double_as_longlong(fabs(un[1 + d] * rinv) + cs);
          smax[d] = b > smax[d] ? b : smax[d];
        }
      }
    }
#pragma unroll
    for (int n = 0; n < 5; n++) { G[n] = Gn[n]; qp3[n] = qpn[n]; }
#pragma unroll
    for (int a = 0; a + 1 < NW; a++)
#pragma unroll
      for (int n = 0; n < 5; n++) wk[a][n] = wk[a + 1][n];
#pragma unroll
    for (int n = 0; n < 5; n++) wk[NW - 1][n] = wp[n];
  };

  int it = 0;
  phaseL(k0 - R, 0);
  int dslot = 0;                                        // T-ring slot of plane s (the one D(s) updates)
  for (int s = k0 - R; s < send - 1; s++, it++) {     // (iteration send-1 would have nothing to do)
    const int b = it & 1;
    const bool inplane = (s >= k0) && (s < k1);
    const double* Ws = sm + b * S::nUpad;
    double* Q1 = sm + S::oQ + b * S::nQ;
    double* Q2 = Q1 + S::nQ1;
    // ---- B(s) --------------------------------------------------------------------------------------
    double qm1[5], qm2[5];
    if (inplane && valid) {
      if constexpr (RECON == 0) {
        // PLM: the five variables of one direction in lock step, so that the five reciprocal seeds (MUFU, long
        // latency) are in flight together instead of one per dependency chain
#pragma unroll
        for (int d = 0; d < 2; d++) {
          const int st = d ? WI : 1;
          double c[5], prod[5], r[5], den[5];
#pragma unroll
          for (int n = 0; n < 5; n++) {
            const double* p = Ws + n * (WJ * WI) + oW;
            c[n] = p[0];
            const double dL = c[n] - p[-st], dR = p[st] - c[n];
            prod[n] = dL * dR; den[n] = dL + dR;
            asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r[n]) : "d"(den[n]));
          }
#pragma unroll
          for (int n = 0; n < 5; n++) {
            const double e = fma(-den[n], r[n], 1.0);
            const double q = prod[n] * fma(r[n], fma(e, e, e), r[n]);     // = div2(prod, den), same operations
            const double h = pos(prod[n]) ? q : 0.0;
            if (d == 0) { qm1[n] = c[n] - h; Q1[n * (TJ * (TI + 1)) + oQ1 + 1] = c[n] + h; }
            else        { qm2[n] = c[n] - h; Q2[n * ((TJ + 1) * TI) + oQ2 + TI] = c[n] + h; }
          }
        }
      } else if constexpr (!SHARE) {
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
    }
    if constexpr (SHARE) {
      // B1: the interface values at the LOWER x1 and x2 faces of the own cell -- kept, and stored in that face's slot for
      // the neighbour below, whose upper interface it is (the upper interfaces of the tile's last row / column come from
      // the edge warp)
      if (inplane && valid) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          const double* p = Ws + n * (WJ * WI) + oW;
          qm1[n] = iface_lean(p[-2], p[-1], p[0], p[1]);
          qm2[n] = iface_lean(p[-2 * WI], p[-WI], p[0], p[WI]);
          Q1[n * (TJ * (TI + 1)) + oQ1] = qm1[n];
          Q2[n * ((TJ + 1) * TI) + oQ2] = qm2[n];
        }
      }
      cta_sync(NTH);                                    // interface values visible
      // B2: CW84 limiter on (lower interface, cell, upper interface); q+ overwrites the upper interface in the slot only
      // this thread reads, q- stays in registers
      if (inplane && valid) {
#pragma unroll
        for (int n = 0; n < 5; n++) {
          const double a = Ws[n * (WJ * WI) + oW];
          double hi = Q1[n * (TJ * (TI + 1)) + oQ1 + 1];
          limit_lean(a, qm1[n], hi);
          Q1[n * (TJ * (TI + 1)) + oQ1 + 1] = hi;
          double hi2 = Q2[n * ((TJ + 1) * TI) + oQ2 + TI];
          limit_lean(a, qm2[n], hi2);
          Q2[n * ((TJ + 1) * TI) + oQ2 + TI] = hi2;
        }
      }
    }
    cta_sync(NTH);                                      // q+ visible; every read of W(s) is done
    // ---- C(s) --------------------------------------------------------------------------------------
    if (inplane && valid) {
      double L1[5], L2[5], F1[5], F2[5];
#pragma unroll
      for (int n = 0; n < 5; n++) { L1[n] = Q1[n * (TJ * (TI + 1)) + oQ1]; L2[n] = Q2[n * ((TJ + 1) * TI) + oQ2]; }
      flux3_x1x2<RS>(g, L1, qm1, L2, qm2, F1, F2); // HLLC: the two solves interleaved
#pragma unroll
      for (int n = 0; n < 5; n++) { Q1[n * (TJ * (TI + 1)) + oQ1] = F1[n]; Q2[n * ((TJ + 1) * TI) + oQ2] = F2[n]; }
    }
    // ---- L(s+1) ------------------------------------------------------------------------------------
    tslot = (dslot + 1 == NS) ? 0 : dslot + 1;
    phaseL(s + 1, it + 1);
    cta_sync(NTH);                                      // fluxes of plane s visible
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
  if (STAGE2 && sc.take_dt) {
    // positive doubles order like their bit patterns: warp max by shuffles, one atomicMax per warp and direction
#pragma unroll
    for (int d = 0; d < 3; d++) {
      unsigned long long v = smax[d];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) { const unsigned long long t = __shfl_xor_sync(0xffffffffu, v, o); v = t > v ? t : v; }
      if ((tid & 31) == 0 && v) atomicMax(P.smax_bits + 3 * lev + d, v);
    }
  }
}

template <int RECON, int RS, int TI, int TJ, int MINB>
cudaError_t launch_v3(const ak_pack& p, const double* Uin, const double* U0, double* Uout, const StageCoef& sc,
                      bool stage2) {
  using S = V3Tile<RECON, TI, TJ>;
  const PackDev& P = p.d;
  if (p.tmap_box[0] != S::WI || p.tmap_box[1] != S::WJ) {
    for (int b = 0; b < 3; b++)
      if (p.u[b] && !make_state_tmap(&p.tmap[b], p.u[b], P.nmb, P.nt, S::WI, S::WJ)) return cudaErrorNotSupported;
    p.tmap_box[0] = S::WI; p.tmap_box[1] = S::WJ;
  }
  if (p.tmap0_box[0] != S::W0 || p.tmap0_box[1] != TJ) {
    for (int b = 0; b < 3; b++)
      if (p.u[b] && !make_state_tmap(&p.tmap0[b], p.u[b], P.nmb, P.nt, S::W0, TJ)) return cudaErrorNotSupported;
    p.tmap0_box[0] = S::W0; p.tmap0_box[1] = TJ;
  }
  const CUtensorMap& tm = (Uin == p.u[0]) ? p.tmap[0] : (Uin == p.u[1] ? p.tmap[1] : p.tmap[2]);
  const CUtensorMap& tm0 = (U0 == p.u[0]) ? p.tmap0[0] : (U0 == p.u[1] ? p.tmap0[1] : p.tmap0[2]);
  const size_t smem = S::bytes;
  auto k1 = stage_v3_kernel<RECON, RS, TI, TJ, MINB, false>;
  auto k2 = stage_v3_kernel<RECON, RS, TI, TJ, MINB, true>;
  static bool attr_set_dev[64] = {};   // the opt-in to > 48 KB of dynamic shared memory is per device
  bool& attr_set = attr_set_dev[p.device & 63];
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const int nti = (P.nx[0] + TI - 1) / TI, ntj = (P.nx[1] + TJ - 1) / TJ;
  const long long ntiles = (long long)nti * ntj * P.nmb;
  // split k only when the tiles alone cannot fill the machine a few times over
  const long long target = (long long)p.sm_count * MINB * 4;
  int nchunk = (int)((target + ntiles - 1) / ntiles);
  int maxchunk = P.nx[2] / 8 > 0 ? P.nx[2] / 8 : 1;
  if (nchunk > maxchunk) nchunk = maxchunk;
  if (nchunk < 1) nchunk = 1;
  const int KC = (P.nx[2] + nchunk - 1) / nchunk;
  nchunk = (P.nx[2] + KC - 1) / KC;
  dim3 grid(nti * ntj, nchunk, P.nmb);
  if (stage2) k2<<<grid, S::NTH, smem, p.stream>>>(tm, tm0, P, Uout, sc, KC, nti);
  else        k1<<<grid, S::NTH, smem, p.stream>>>(tm, tm0, P, Uout, sc, KC, nti);
  return cudaGetLastError();
}

}  // namespace ak

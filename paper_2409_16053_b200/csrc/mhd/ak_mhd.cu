// ak_mhd.cu -- MHD + constrained-transport stage over a MeshBlockPack (include/ak_mhd.h), first cut:
// correct and device-resident, not yet fused.  Paper: Eq.(5) and the gamma-law energy, face-centred field with
// CT and Gardiner-Stone upwinded EMFs, HLLD.  Readings DESIGN.md Q33-Q37.
// Compiled with -fmad=false: every expression rounds once per operation in the order written (fused multiply-adds only where
// written out).  With akm_pack_set_exact the flux sweeps also use IEEE division / sqrt in the definition's order and the whole
// path is bit-identical to the definition evaluated on the host; the default uses MUFU-seeded reciprocals and square roots.
// Kernels, all one thread per cell with i fastest (coalesced), launched in this order per stage:
//   prim_kernel      U -> W = (rho, v, u_g, B_cc)                                   work: W[8]
//   flux_kernel<D>   PLM on W along D, HLLD at the lower D-face of every cell        work: F_D[7]
//   emf_kernel       corner EMFs from the face fluxes, upwinded                     work: Ec[3]
//   update_kernel    cells: flux divergence; faces: curl of the corner EMFs; stage weights
// plus fill_kernel (periodic ghost copy of all 8 variables) and dt_kernel (CFL reduction with the fast speed).
// This file is part of the CUDA path only; the CPU oracle of the tests shares nothing with it.
#include "ak_mhd.h"

#include <cuda_runtime.h>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>

namespace akm {
// plain-data view of the pack for the kernels
struct Dev {
  int nmb, nx[3], ng, nt[3], nrb[3];
  long long ncell;            // cells per block incl. ghosts = stride between variables
  double gamma, dx[3];
  const int* lx;              // [nmb][3]
  const int* leaf;            // [nrb3][nrb2][nrb1] -> block
  double* W;                  // [nmb][8][ncell]
  double* F[3];               // [nmb][7][ncell] per direction: 0..4 hydro fluxes (unrotated), 5 = flux of B_{d+1}, 6 = of B_{d+2}
  double* Ec;                 // [nmb][3][ncell] corner EMFs
  unsigned long long* cells;  // [0] min dt as ordered bits, [1] floor count, [2] non-finite count
};
// The flux sweeps of the default arithmetic flavour live in a second translation unit (ak_mhd_fast.cu = this file with
// AKM_FAST_TU defined) compiled WITHOUT -fmad=false: the compiler may contract a*b+c there (-17 % FP64-pipe instructions with
// PLM, -20 % with WENOZ; the sweeps are bound by that pipe).  The verification flavour and every other kernel stay in the
// -fmad=false unit, where each operation is the one written.
void launch_sweeps_fast(const Dev& d, int recon, int rsolver, dim3 grid, cudaStream_t stream, const double* Uin);
}  // namespace akm

namespace {
using akm::Dev;

thread_local std::string g_err;
int fail(int code, const std::string& msg) { g_err = msg; return code; }
int cuda_fail(cudaError_t e, const char* where) { return fail(-4, std::string(where) + ": " + cudaGetErrorString(e)); }
#define AKM_CUDA(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, where); } while (0)

constexpr double RHO_FLOOR = 1e-20, P_FLOOR = 1e-20;


// ---- division and square root in two flavours --------------------------------------------------------------------
// X = true: IEEE division and sqrt in the definition's operation order -- the results are bit-identical to the definition
// evaluated on the host, which is how this path is verified (akm_pack_set_exact).  X = false (default): MUFU seed + one
// cubically convergent step (1-2 ulp), 3-4 FP64-pipe instructions instead of ~13, and quotients by a shared divisor formed
// with one reciprocal: the sweeps are bound by the issue of exactly these instructions.  The fast flavour differs from the
// exact one by rounding only (measured <= 1e-14 per stage in the parity metric); the upwind switch of the corner EMFs is
// ramped (Q36), so a mass flux at round-off level does not turn that rounding into a different choice of side.
__device__ __forceinline__ double rcp_fast(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  return fma(r, fma(e, e, e), r);
}
__device__ __forceinline__ double sqrt_fast(double x) {      // x > 0 (0 -> 0 handled by the caller where it can occur)
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-(x * r), r, 1.0);
  r = fma(r, e * fma(0.375, e, 0.5), r);
  return x * r;
}
template <bool X> __device__ __forceinline__ double div_(double a, double b) { if constexpr (X) return a / b; else return a * rcp_fast(b); }
template <bool X> __device__ __forceinline__ double rcp_(double b) { if constexpr (X) return 1.0 / b; else return rcp_fast(b); }
template <bool X> __device__ __forceinline__ double sqrt_(double x) { if constexpr (X) return sqrt(x); else return x > 0.0 ? sqrt_fast(x) : 0.0; }

// ---- HLLD (Miyoshi & Kusano 2005, restated; Q34): rotated states (rho, u, v, w, u_g, By, Bz), normal field bx ----
// Written so that few values are live at a time (the sweeps run at 64 registers): only the scalars of both sides that the
// wave speeds need, the conserved vector and physical flux of the side the face lies on, and of the other side's star state
// only what the double-star state takes from it.  In the exact flavour every value is formed by the same operations in the
// same order as in the definition, so the result does not depend on this arrangement.
struct Side { double r, u, v, w, by, bz, pt, E, vb, cf; };

template <bool X>
__device__ __forceinline__ void side_init(double gamma, double bx, const double W[7], Side& s) {
  s.r = W[0]; s.u = W[1]; s.v = W[2]; s.w = W[3]; s.by = W[5]; s.bz = W[6];
  const double e = W[4], p = (gamma - 1.0) * e;
  const double b2 = bx * bx + (s.by * s.by + s.bz * s.bz);
  s.pt = p + 0.5 * b2;
  s.E = e + 0.5 * s.r * (s.u * s.u + (s.v * s.v + s.w * s.w)) + 0.5 * b2;
  s.vb = s.u * bx + (s.v * s.by + s.w * s.bz);
  const double gp = gamma * p, sum = gp + b2;
  double disc = sum * sum - 4.0 * gp * (bx * bx);
  if (disc < 0.0) disc = 0.0;
  s.cf = sqrt_<X>(div_<X>(sum + sqrt_<X>(disc), 2.0 * s.r));
}
__device__ __forceinline__ void cons_flux(double bx, const Side& s, double U[7], double F[7]) {
  U[0] = s.r; U[1] = s.r * s.u; U[2] = s.r * s.v; U[3] = s.r * s.w; U[4] = s.E; U[5] = s.by; U[6] = s.bz;
  F[0] = s.r * s.u; F[1] = s.r * s.u * s.u + s.pt - bx * bx; F[2] = s.r * s.u * s.v - bx * s.by;
  F[3] = s.r * s.u * s.w - bx * s.bz; F[4] = (s.E + s.pt) * s.u - bx * s.vb; F[5] = s.by * s.u - bx * s.v;
  F[6] = s.bz * s.u - bx * s.w;
}

// star state of side K behind the outer wave SK: density, transverse velocities and fields, v.B; isdm = 1 / (SK - SM)
struct Star { double rs, vs, ws, bys, bzs, vbs, isdm; };
template <bool X>
__device__ __forceinline__ void star_state(double bx, const Side& s, double SK, double SM, double pts, Star& t) {
  const double sdu = SK - s.u, sdm = SK - SM;
  if constexpr (X) { t.rs = s.r * sdu / sdm; t.isdm = 0.0; }
  else { t.isdm = rcp_fast(sdm); t.rs = (s.r * sdu) * t.isdm; }
  const double den = s.r * sdu * sdm - bx * bx;
  if (fabs(den) < 1e-8 * pts) {
    t.vs = s.v; t.ws = s.w; t.bys = s.by; t.bzs = s.bz;
  } else {
    double f1, f2;
    if constexpr (X) { f1 = bx * (SM - s.u) / den; f2 = (s.r * sdu * sdu - bx * bx) / den; }
    else { const double id = rcp_fast(den); f1 = (bx * (SM - s.u)) * id; f2 = (s.r * sdu * sdu - bx * bx) * id; }
    t.vs = s.v - s.by * f1; t.ws = s.w - s.bz * f1;
    t.bys = s.by * f2; t.bzs = s.bz * f2;
  }
  t.vbs = SM * bx + (t.vs * t.bys + t.ws * t.bzs);
}
template <bool X>
__device__ __forceinline__ double star_energy(double bx, const Side& s, double SK, double SM, double pts, const Star& t) {
  const double num = (SK - s.u) * s.E - s.pt * s.u + pts * SM + bx * (s.vb - t.vbs);
  if constexpr (X) return num / (SK - SM); else return num * t.isdm;
}

template <bool X>
__device__ void hlld(double gamma, double bn, const double WL[7], const double WR[7], double F[7]) {
  Side L, R;
  side_init<X>(gamma, bn, WL, L);
  side_init<X>(gamma, bn, WR, R);
  const double cfm = fmax(L.cf, R.cf);
  const double SL = fmin(L.u, R.u) - cfm, SR = fmax(L.u, R.u) + cfm;
  double UK[7];
  if (SL >= 0.0) { cons_flux(bn, L, UK, F); return; }
  if (SR <= 0.0) { cons_flux(bn, R, UK, F); return; }
  const double mL = L.r * (SL - L.u), mR = R.r * (SR - R.u);
  double SM, pts;
  if constexpr (X) {
    SM = ((mR * R.u - mL * L.u) - (R.pt - L.pt)) / (mR - mL);
    pts = ((mR * L.pt - mL * R.pt) + mL * mR * (R.u - L.u)) / (mR - mL);
  } else {
    const double im = rcp_fast(mR - mL);
    SM = ((mR * R.u - mL * L.u) - (R.pt - L.pt)) * im;
    pts = ((mR * L.pt - mL * R.pt) + mL * mR * (R.u - L.u)) * im;
  }
  Star tL, tR;
  star_state<X>(bn, L, SL, SM, pts, tL);
  star_state<X>(bn, R, SR, SM, pts, tR);
  const double sqL = sqrt_<X>(tL.rs), sqR = sqrt_<X>(tR.rs);
  const double SsL = SM - div_<X>(fabs(bn), sqL), SsR = SM + div_<X>(fabs(bn), sqR);
  const bool left = (SM >= 0.0);
  const Side& K = left ? L : R;
  const Star& tK = left ? tL : tR;
  const double SK = left ? SL : SR, SsK = left ? SsL : SsR;
  const double EsK = star_energy<X>(bn, K, SK, SM, pts, tK);
  const double Us[7] = {tK.rs, tK.rs * SM, tK.rs * tK.vs, tK.rs * tK.ws, EsK, tK.bys, tK.bzs};
  double FK[7];
  cons_flux(bn, K, UK, FK);
  const bool outer = left ? (SsL >= 0.0) : (SsR <= 0.0);
  if (outer || 0.5 * bn * bn < 1e-8 * pts) {
    for (int n = 0; n < 7; n++) F[n] = FK[n] + SK * (Us[n] - UK[n]);
    return;
  }
  // double-star state; in the exact flavour the star velocities go through the conserved momenta as in the definition
  const double sgn = (bn > 0.0) ? 1.0 : -1.0, isum = rcp_<X>(sqL + sqR);
  double vsL, wsL, vsR, wsR;
  if constexpr (X) { vsL = (tL.rs * tL.vs) / tL.rs; wsL = (tL.rs * tL.ws) / tL.rs; vsR = (tR.rs * tR.vs) / tR.rs; wsR = (tR.rs * tR.ws) / tR.rs; }
  else { vsL = tL.vs; wsL = tL.ws; vsR = tR.vs; wsR = tR.ws; }
  const double vss = (sqL * vsL + sqR * vsR + (tR.bys - tL.bys) * sgn) * isum;
  const double wss = (sqL * wsL + sqR * wsR + (tR.bzs - tL.bzs) * sgn) * isum;
  const double byss = (sqL * tR.bys + sqR * tL.bys + sqL * sqR * (vsR - vsL) * sgn) * isum;
  const double bzss = (sqL * tR.bzs + sqR * tL.bzs + sqL * sqR * (wsR - wsL) * sgn) * isum;
  const double vbss = SM * bn + (vss * byss + wss * bzss);
  double Uss[7];
  Uss[0] = Us[0]; Uss[1] = Us[1]; Uss[2] = Us[0] * vss; Uss[3] = Us[0] * wss;
  Uss[4] = left ? EsK - sqL * (tL.vbs - vbss) * sgn : EsK + sqR * (tR.vbs - vbss) * sgn;
  Uss[5] = byss; Uss[6] = bzss;
  for (int n = 0; n < 7; n++) F[n] = FK[n] + SsK * Uss[n] - (SsK - SK) * Us[n] - SK * UK[n];
}

// LLF and HLLE in the same variables: F = (F_L + F_R)/2 - (lambda/2)(U_R - U_L) with lambda = max(|u| + cf); the HLL
// flux between HLLD's outer speeds, b- = min(S_L, 0), b+ = max(S_R, 0).
template <bool X>
__device__ void llf(double gamma, double bn, const double WL[7], const double WR[7], double F[7]) {
  Side L, R;
  side_init<X>(gamma, bn, WL, L);
  side_init<X>(gamma, bn, WR, R);
  const double lam = fmax(fabs(L.u) + L.cf, fabs(R.u) + R.cf);
  double UL[7], FL[7], UR[7], FR[7];
  cons_flux(bn, L, UL, FL);
  cons_flux(bn, R, UR, FR);
#pragma unroll
  for (int n = 0; n < 7; n++) F[n] = 0.5 * (FL[n] + FR[n]) - 0.5 * lam * (UR[n] - UL[n]);
}
template <bool X>
__device__ void hlle(double gamma, double bn, const double WL[7], const double WR[7], double F[7]) {
  Side L, R;
  side_init<X>(gamma, bn, WL, L);
  side_init<X>(gamma, bn, WR, R);
  const double cfm = fmax(L.cf, R.cf);
  const double SL = fmin(L.u, R.u) - cfm, SR = fmax(L.u, R.u) + cfm;
  const double bm = fmin(SL, 0.0), bp = fmax(SR, 0.0);
  double UL[7], FL[7], UR[7], FR[7];
  cons_flux(bn, L, UL, FL);
  cons_flux(bn, R, UR, FR);
  if constexpr (X) {
#pragma unroll
    for (int n = 0; n < 7; n++) F[n] = ((bp * FL[n] - bm * FR[n]) + bp * bm * (UR[n] - UL[n])) / (bp - bm);
  } else {
    const double inv = rcp_fast(bp - bm);
#pragma unroll
    for (int n = 0; n < 7; n++) F[n] = ((bp * FL[n] - bm * FR[n]) + bp * bm * (UR[n] - UL[n])) * inv;
  }
}
template <bool X, int RS>
__device__ __forceinline__ void riemann(double gamma, double bn, const double WL[7], const double WR[7], double F[7]) {
  if constexpr (RS == 1) llf<X>(gamma, bn, WL, WR, F);
  else if constexpr (RS == 2) hlle<X>(gamma, bn, WL, WR, F);
  else hlld<X>(gamma, bn, WL, WR, F);
}

template <bool X>
__device__ __forceinline__ void plm(double qm1, double q0, double qp1, double& qm, double& qp) {
  const double dL = q0 - qm1, dR = qp1 - q0, prod = dL * dR;
  const double h = (prod > 0.0) ? div_<X>(prod, dL + dR) : 0.0;
  qm = q0 - h; qp = q0 + h;
}

// PPM4 (the hydro path's reading): fourth-order interface value clamped between its two cells, then Colella &
// Woodward's (1984) Eq.(1.10) monotonicity constraint on the parabola of cell a with edge values (aL, aR).
template <bool X>
__device__ __forceinline__ double ppm4_iface(double qm1, double q0, double qp1, double qp2) {
  const double n = 7.0 * (q0 + qp1) - (qm1 + qp2);
  double v;
  if constexpr (X) v = n / 12.0; else v = n * (1.0 / 12.0);
  return fmax(fmin(q0, qp1), fmin(v, fmax(q0, qp1)));
}
template <bool X>
__device__ __forceinline__ void ppm4_limit(double a, double aL, double aR, double& qm, double& qp) {
  if ((aR - a) * (a - aL) <= 0.0) { aL = a; aR = a; }
  else {
    const double d = aR - aL, mu = a - 0.5 * (aL + aR), dmu = d * mu;
    double d26;
    if constexpr (X) d26 = d * d / 6.0; else d26 = (d * d) * (1.0 / 6.0);
    if (dmu > d26) aL = 3.0 * a - 2.0 * aR;
    else if (-d26 > dmu) aR = 3.0 * a - 2.0 * aL;
  }
  qm = aL; qp = aR;
}
// PPMX (Q30; Colella & Sekora 2008 / McCorquodale & Colella 2011, restated): fourth-order interface value, replaced
// where it is not between its two cells by (q0 + q1)/2 - D/6 with D the second difference limited among the face-centred one
// and C = 5/4 times the two cell-centred ones; ...
template <bool X>
__device__ __forceinline__ double ppmx_iface(double qm1, double q0, double q1, double q2) {
  const double C = 1.25, n = 7.0 * (q0 + q1) - (qm1 + q2);
  double v;
  if constexpr (X) v = n / 12.0; else v = n * (1.0 / 12.0);
  if ((v - q0) * (q1 - v) < 0.0) {
    const double dc = 3.0 * ((q0 + q1) - 2.0 * v), dl = (qm1 + q1) - 2.0 * q0, dr = (q0 + q2) - 2.0 * q1;
    double D = 0.0;
    if (dc > 0.0 && dl > 0.0 && dr > 0.0) D = fmin(dc, C * fmin(dl, dr));
    else if (dc < 0.0 && dl < 0.0 && dr < 0.0) D = -fmin(-dc, C * fmin(-dl, -dr));
    if constexpr (X) v = 0.5 * (q0 + q1) - D / 6.0; else v = 0.5 * (q0 + q1) - D * (1.0 / 6.0);
  }
  return v;
}
// ... and the parabola of the cell q2 of (q0 .. q4) with edge values (aL, aR): at an extremum its second derivative is limited
// among itself and C times the three cell-centred second differences and both edge increments are scaled by the ratio (kept when
// the ratio >= 1 - 1e-12); elsewhere an edge increment is at most twice the other.
template <bool X>
__device__ __forceinline__ void ppmx_limit(double q0, double q1, double q2, double q3, double q4, double aL, double aR, double& qm, double& qp) {
  const double C = 1.25, a = q2, dm = a - aL, dp = aR - a;
  if (dm * dp <= 0.0 || (q3 - a) * (a - q1) <= 0.0) {
    const double df = 6.0 * ((aL + aR) - 2.0 * a);
    const double d1 = (q0 + q2) - 2.0 * q1, d2 = (q1 + q3) - 2.0 * q2, d3 = (q2 + q4) - 2.0 * q3;
    double D = 0.0;
    if (df > 0.0 && d1 > 0.0 && d2 > 0.0 && d3 > 0.0) D = fmin(df, C * fmin(d1, fmin(d2, d3)));
    else if (df < 0.0 && d1 < 0.0 && d2 < 0.0 && d3 < 0.0) D = -fmin(-df, C * fmin(-d1, fmin(-d2, -d3)));
    const double rho = (df != 0.0) ? div_<X>(D, df) : 0.0;
    if (rho <= 1.0 - 1e-12) { aL = a - rho * dm; aR = a + rho * dp; }
  } else {
    if (fabs(dm) >= 2.0 * fabs(dp)) aL = a - 2.0 * dp;
    if (fabs(dp) >= 2.0 * fabs(dm)) aR = a + 2.0 * dm;
  }
  qm = aL; qp = aR;
}
// WENO-Z (Borges et al. 2008; Q29) value at the UPPER face of the middle cell of (a, b, c, d, e), in the differences
// of neighbouring cells (constants reproduced exactly); the lower-face value is the same function of the mirrored stencil.
template <bool X>
__device__ __forceinline__ double wenoz_upper(double a, double b, double c, double d, double e) {
  const double d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
  const double P0 = 5.0 * d2 - 2.0 * d1, P1 = 2.0 * d3 + d2, P2 = 4.0 * d3 - d4;
  const double s0 = d2 - d1, t0 = 3.0 * d2 - d1, s1 = d3 - d2, t1 = d2 + d3, s2 = d4 - d3, t2 = d4 - 3.0 * d3;
  const double b0 = 13.0 / 12.0 * (s0 * s0) + 0.25 * (t0 * t0);
  const double b1 = 13.0 / 12.0 * (s1 * s1) + 0.25 * (t1 * t1);
  const double b2 = 13.0 / 12.0 * (s2 * s2) + 0.25 * (t2 * t2);
  const double eps = 1e-40, tau = fabs(b0 - b2);
  const double r0 = div_<X>(tau, b0 + eps), r1 = div_<X>(tau, b1 + eps), r2 = div_<X>(tau, b2 + eps);
  const double a0 = 0.1 * (1.0 + r0 * r0), a1 = 0.6 * (1.0 + r1 * r1), a2 = 0.3 * (1.0 + r2 * r2);
  return c + div_<X>(a0 * P0 + (a1 * P1 + a2 * P2), 6.0 * (a0 + (a1 + a2)));
}
// left and right state of one primitive at the face between cells cm = c - st and c (RECON: 0 PLM, 1 PPM4, 2 PPMX, 3 WENOZ)
template <bool X, int RECON>
__device__ __forceinline__ void face_states(const double* __restrict__ w, long long c, long long st, double& wl, double& wr) {
  if constexpr (RECON == 0) {
    double qm, qp;
    plm<X>(w[c - 2 * st], w[c - st], w[c], qm, qp); wl = qp;
    plm<X>(w[c - st], w[c], w[c + st], qm, qp);     wr = qm;
  } else {
    const double s0 = w[c - 3 * st], s1 = w[c - 2 * st], s2 = w[c - st], s3 = w[c], s4 = w[c + st], s5 = w[c + 2 * st];
    if constexpr (RECON == 1) {
      const double fL = ppm4_iface<X>(s0, s1, s2, s3), fM = ppm4_iface<X>(s1, s2, s3, s4), fR = ppm4_iface<X>(s2, s3, s4, s5);
      double qm, qp;
      ppm4_limit<X>(s2, fL, fM, qm, qp); wl = qp;
      ppm4_limit<X>(s3, fM, fR, qm, qp); wr = qm;
    } else if constexpr (RECON == 2) {
      const double fL = ppmx_iface<X>(s0, s1, s2, s3), fM = ppmx_iface<X>(s1, s2, s3, s4), fR = ppmx_iface<X>(s2, s3, s4, s5);
      double qm, qp;
      ppmx_limit<X>(s0, s1, s2, s3, s4, fL, fM, qm, qp); wl = qp;
      ppmx_limit<X>(s1, s2, s3, s4, s5, fM, fR, qm, qp); wr = qm;
    } else {
      wl = wenoz_upper<X>(s0, s1, s2, s3, s4);
      wr = wenoz_upper<X>(s5, s4, s3, s2, s1);
    }
  }
}

// (k, j, i) of a flat cell index inside one block
// (32-bit: a block has fewer than 2^31 cells, checked at create; the 64-bit form cost ~250 instructions per thread)
__device__ __forceinline__ void kji(const Dev& P, long long c, int& k, int& j, int& i) {
  const unsigned cu = (unsigned)c, row = cu / (unsigned)P.nt[0], kk = row / (unsigned)P.nt[1];
  i = (int)(cu - row * (unsigned)P.nt[0]); j = (int)(row - kk * (unsigned)P.nt[1]); k = (int)kk;
}
__device__ __forceinline__ void kji_active(const Dev& P, long long t, int& k, int& j, int& i) {
  const unsigned tu = (unsigned)t, row = tu / (unsigned)P.nx[0], kk = row / (unsigned)P.nx[1];
  i = (int)(tu - row * (unsigned)P.nx[0]) + P.ng; j = (int)(row - kk * (unsigned)P.nx[1]) + P.ng; k = (int)kk + P.ng;
}

// ---- S1: primitives with the cell-centred field = mean of the two faces (Q33); not for the outermost upper layer ----
__global__ void __launch_bounds__(256) prim_kernel(Dev P, const double* __restrict__ U) {
  const int m = blockIdx.y;
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= P.ncell) return;
  int k, j, i; kji(P, c, k, j, i);
  if (i >= P.nt[0] - 1 || j >= P.nt[1] - 1 || k >= P.nt[2] - 1) return;
  const long long nc = P.ncell, str[3] = {1, P.nt[0], (long long)P.nt[0] * P.nt[1]};
  const double* Ub = U + (long long)m * 8 * nc;
  int nfl = 0;
  double rho = Ub[c];
  if (!(rho >= RHO_FLOOR)) { rho = RHO_FLOOR; nfl++; }
  const double rinv = 1.0 / rho, m1 = Ub[nc + c], m2 = Ub[2 * nc + c], m3 = Ub[3 * nc + c];
  double B[3];
  for (int d = 0; d < 3; d++) B[d] = 0.5 * (Ub[(5 + d) * nc + c] + Ub[(5 + d) * nc + c + str[d]]);
  double ug = Ub[4 * nc + c] - 0.5 * rinv * (m1 * m1 + (m2 * m2 + m3 * m3)) - 0.5 * (B[0] * B[0] + (B[1] * B[1] + B[2] * B[2]));
  if (!(ug >= P_FLOOR / (P.gamma - 1.0))) { ug = P_FLOOR / (P.gamma - 1.0); nfl++; }
  double* Wb = P.W + (long long)m * 8 * nc;
  Wb[c] = rho; Wb[nc + c] = m1 * rinv; Wb[2 * nc + c] = m2 * rinv; Wb[3 * nc + c] = m3 * rinv; Wb[4 * nc + c] = ug;
  for (int d = 0; d < 3; d++) Wb[(5 + d) * nc + c] = B[d];
  // (the oracle counts the floors of every cell it converts, ghosts included: so does this)
  if (nfl) atomicAdd(P.cells + 1, (unsigned long long)nfl);
}

// ---- S2 + S3: PLM + HLLD at the lower D-face of every cell whose stencil exists ----
// Occupancy (measured at 256^3): the exact flavour waits on its IEEE division chains and runs best with 32 warps per SM (64
// registers, 240 B spilled); the fast flavour is bound by the FP64 pipe and runs best without spills (96 registers, 20 warps:
// 1.49 -> 1.67 G cell-updates/s against 8 CTAs per SM).
template <int D, bool X, int RECON, int RS>
__global__ void __launch_bounds__(128, X ? 8 : (RECON == 0 ? 5 : 4)) flux_kernel(Dev P, const double* __restrict__ U) {
  constexpr int D1 = (D + 1) % 3, D2 = (D + 2) % 3;
  const int m = blockIdx.y;
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= P.ncell) return;
  int idx[3]; kji(P, c, idx[2], idx[1], idx[0]);
  constexpr int R = (RECON == 0) ? 2 : 3;        // cells c-R .. c+R-1 along D must hold W
  if (idx[D] < R || idx[D] >= P.nt[D] - R || idx[D1] >= P.nt[D1] - 1 || idx[D2] >= P.nt[D2] - 1) return;
  const long long nc = P.ncell, str[3] = {1, P.nt[0], (long long)P.nt[0] * P.nt[1]};
  const long long st = str[D];
  const double* Wb = P.W + (long long)m * 8 * nc;
  const int var[7] = {0, 1 + D, 1 + D1, 1 + D2, 4, 5 + D1, 5 + D2};
  double WL[7], WR[7], F[7];
#pragma unroll
  for (int q = 0; q < 7; q++) face_states<X, RECON>(Wb + var[q] * nc, c, st, WL[q], WR[q]);
  riemann<X, RS>(P.gamma, U[(long long)m * 8 * nc + (5 + D) * nc + c], WL, WR, F);
  double* Fb = P.F[D] + (long long)m * 7 * nc;
  Fb[c] = F[0]; Fb[(1 + D) * nc + c] = F[1]; Fb[(1 + D1) * nc + c] = F[2]; Fb[(1 + D2) * nc + c] = F[3];
  Fb[4 * nc + c] = F[4]; Fb[5 * nc + c] = F[5]; Fb[6 * nc + c] = F[6];
}

#ifndef AKM_FAST_TU
// upwinded (face - centre) EMF difference (Q36): weight w of the lower side = 1/2 + nu clipped to [0, 1] with
// nu = 1024 dt F_mass / (dx (rho_1 + rho_2)) -- pure upwind once the contact crosses 2^-10 of a cell per step, the mean at
// rest, continuous in between (a mass flux at round-off level does not decide the result).  k = 1024 dt / dx.
template <bool X>
__device__ __forceinline__ double upwind(double k, double mflux, double rho1, double rho2, double from_lower, double from_upper) {
  const double w = 0.5 + fmax(-0.5, fmin(0.5, div_<X>(k * mflux, rho1 + rho2)));
  return w * from_lower + (1.0 - w) * from_upper;
}
__device__ __forceinline__ double ecc(const double* __restrict__ Wb, long long nc, long long c, int e) {
  const int a = (e + 1) % 3, b = (e + 2) % 3;          // E_e = -(v_a B_b - v_b B_a)
  return -(Wb[(1 + a) * nc + c] * Wb[(5 + b) * nc + c] - Wb[(1 + b) * nc + c] * Wb[(5 + a) * nc + c]);
}

// ---- CT: E_e on the edges along e at the lower-a, lower-b corner of each cell (Q35, Q36) ----
template <bool X>
__global__ void __launch_bounds__(128) emf_kernel(Dev P, double k0, double k1, double k2) {
  const int m = blockIdx.y;
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= P.ncell) return;
  int idx[3]; kji(P, c, idx[2], idx[1], idx[0]);
  const long long nc = P.ncell, str[3] = {1, P.nt[0], (long long)P.nt[0] * P.nt[1]};
  const double* Wb = P.W + (long long)m * 8 * nc;
  const double kd[3] = {k0, k1, k2};
  for (int e = 0; e < 3; e++) {
    const int a = (e + 1) % 3, b = (e + 2) % 3;
    bool in = true;
    for (int d = 0; d < 3; d++) in = in && idx[d] >= P.ng && idx[d] < P.nx[d] + P.ng + (d == e ? 0 : 1);
    if (!in) continue;
    const double* Fa = P.F[a] + (long long)m * 7 * nc;
    const double* Fb = P.F[b] + (long long)m * 7 * nc;
    const long long sa = str[a], sb = str[b];
    // E_e at an a-face = -F_a(B_b) (slot 5 of direction a), at a b-face = +F_b(B_a) (slot 6 of direction b)
    const double Eaf0 = -Fa[5 * nc + c], Eaf1 = -Fa[5 * nc + c - sb], Ebf0 = Fb[6 * nc + c], Ebf1 = Fb[6 * nc + c - sa];
    const double mean = 0.25 * ((Eaf1 + Eaf0) + (Ebf1 + Ebf0));
    const double E00 = ecc(Wb, nc, c, e), E10 = ecc(Wb, nc, c - sa, e), E01 = ecc(Wb, nc, c - sb, e), E11 = ecc(Wb, nc, c - sa - sb, e);
    const double r00 = Wb[c], r10 = Wb[c - sa], r01 = Wb[c - sb], r11 = Wb[c - sa - sb];
    const double l2 = upwind<X>(kd[a], Fa[c - sb], r11, r01, Ebf1 - E11, Ebf0 - E01);
    const double r2 = upwind<X>(kd[a], Fa[c],      r10, r00, Ebf1 - E10, Ebf0 - E00);
    const double l1 = upwind<X>(kd[b], Fb[c - sa], r11, r10, Eaf1 - E11, Eaf0 - E10);
    const double r1 = upwind<X>(kd[b], Fb[c],      r01, r00, Eaf1 - E01, Eaf0 - E00);
    P.Ec[(long long)m * 3 * nc + e * nc + c] = mean + 0.25 * ((l1 + r1) + (l2 + r2));
  }
}

// ---- S4: cells by the flux divergence, faces by the curl of the corner EMFs, with the stage weights ----
// (U_out may be U_in (SSPRK(3,3) stage 2) or U^n (last stage): every thread reads its own cell before it writes it; no __restrict__)
__global__ void __launch_bounds__(128) update_kernel(Dev P, const double* Uin, const double* U0, double* Uout,
                                                     double g0, double g1, double c1, double c2, double c3) {
  const int m = blockIdx.y;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long nact = (long long)P.nx[0] * P.nx[1] * P.nx[2];
  if (t >= nact) return;
  int i, j, k; kji_active(P, t, k, j, i);
  const long long nc = P.ncell, str[3] = {1, P.nt[0], (long long)P.nt[0] * P.nt[1]};
  const long long c = k * str[2] + j * str[1] + i;
  const double cdt[3] = {c1, c2, c3};
  const double* Ub = Uin + (long long)m * 8 * nc;
  const double* U0b = U0 + (long long)m * 8 * nc;
  double* Uo = Uout + (long long)m * 8 * nc;
  for (int n = 0; n < 5; n++) {
    double v = g0 * Ub[n * nc + c] + g1 * U0b[n * nc + c];
    for (int d = 0; d < 3; d++) {
      const double* Fd = P.F[d] + (long long)m * 7 * nc + n * nc;
      v = v - cdt[d] * (Fd[c + str[d]] - Fd[c]);
    }
    Uo[n * nc + c] = v;
  }
  const double* Ec = P.Ec + (long long)m * 3 * nc;
  for (int a = 0; a < 3; a++) {                        // db_a/dt = -(d_b E_c - d_c E_b), (a, b, c) cyclic
    const int b = (a + 1) % 3, cc = (a + 2) % 3;
    double v = g0 * Ub[(5 + a) * nc + c] + g1 * U0b[(5 + a) * nc + c];
    v = v - cdt[b] * (Ec[cc * nc + c + str[b]] - Ec[cc * nc + c]);
    v = v + cdt[cc] * (Ec[b * nc + c + str[cc]] - Ec[b * nc + c]);
    Uo[(5 + a) * nc + c] = v;
  }
}

// ---- ghost fill: every ghost cell takes all 8 variables of its periodic image (an active cell) ----
// One thread per GHOST cell (13 % of the cells of a 128^3 block), enumerated without a table: the two x3 slabs, then the two x2
// slabs of the remaining planes, then the two x1 strips of the remaining rows.
__global__ void __launch_bounds__(256) fill_kernel(Dev P, double* __restrict__ U) {
  const int m = blockIdx.y;
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned g2 = 2u * P.ng, n0 = P.nt[0], n1 = P.nt[1];
  const unsigned A = g2 * n1 * n0, B = (unsigned)P.nx[2] * g2 * n0, Cn = (unsigned)P.nx[2] * P.nx[1] * g2;
  if (t >= A + B + Cn) return;
  int idx[3];
  if (t < A) {
    const unsigned kk = t / (n1 * n0), r = t - kk * (n1 * n0), j = r / n0;
    idx[2] = (int)(kk < (unsigned)P.ng ? kk : kk + P.nx[2]); idx[1] = (int)j; idx[0] = (int)(r - j * n0);
  } else if (t < A + B) {
    t -= A;
    const unsigned kk = t / (g2 * n0), r = t - kk * (g2 * n0), jj = r / n0;
    idx[2] = (int)kk + P.ng; idx[1] = (int)(jj < (unsigned)P.ng ? jj : jj + P.nx[1]); idx[0] = (int)(r - jj * n0);
  } else {
    t -= A + B;
    const unsigned row = t / g2, ii = t - row * g2, kk = row / (unsigned)P.nx[1];
    idx[2] = (int)kk + P.ng; idx[1] = (int)(row - kk * (unsigned)P.nx[1]) + P.ng; idx[0] = (int)(ii < (unsigned)P.ng ? ii : ii + P.nx[0]);
  }
  const long long c = ((long long)idx[2] * P.nt[1] + idx[1]) * P.nt[0] + idx[0];
  int sl[3], s[3];
  for (int d = 0; d < 3; d++) {
    const int a = idx[d] - P.ng;
    const int N = P.nrb[d] * P.nx[d];
    int g = (P.lx[3 * m + d] * P.nx[d] + a) % N;
    if (g < 0) g += N;
    sl[d] = g / P.nx[d]; s[d] = g - sl[d] * P.nx[d] + P.ng;
  }
  const int src = P.leaf[(sl[2] * P.nrb[1] + sl[1]) * P.nrb[0] + sl[0]];
  const long long nc = P.ncell;
  const long long cs = ((long long)s[2] * P.nt[1] + s[1]) * P.nt[0] + s[0];
  for (int n = 0; n < 8; n++) U[((long long)m * 8 + n) * nc + c] = U[((long long)src * 8 + n) * nc + cs];
}

// ---- S0: CFL reduction with the fast speed per direction (Q37); candidates are positive: ordered-bits atomicMin ----
__global__ void dt_init_kernel(Dev P) { P.cells[0] = 0x7FF0000000000000ull; P.cells[2] = 0ull; }

__global__ void __launch_bounds__(256) dt_kernel(Dev P, const double* __restrict__ U) {
  const int m = blockIdx.y;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long nact = (long long)P.nx[0] * P.nx[1] * P.nx[2];
  double best = __longlong_as_double(0x7FF0000000000000ll);
  bool bad = false;
  if (t < nact) {
    int i, j, k; kji_active(P, t, k, j, i);
    const long long nc = P.ncell, str[3] = {1, P.nt[0], (long long)P.nt[0] * P.nt[1]};
    const long long c = (long long)m * 8 * nc + k * str[2] + j * str[1] + i;
    double rho = U[c];
    if (!(rho >= RHO_FLOOR)) rho = RHO_FLOOR;
    const double rinv = 1.0 / rho, m1 = U[c + nc], m2 = U[c + 2 * nc], m3 = U[c + 3 * nc];
    double B[3];
    for (int d = 0; d < 3; d++) B[d] = 0.5 * (U[c + (5 + d) * nc] + U[c + (5 + d) * nc + str[d]]);
    const double b2 = B[0] * B[0] + (B[1] * B[1] + B[2] * B[2]);
    double ug = U[c + 4 * nc] - 0.5 * rinv * (m1 * m1 + (m2 * m2 + m3 * m3)) - 0.5 * b2;
    if (!(ug >= P_FLOOR / (P.gamma - 1.0))) ug = P_FLOOR / (P.gamma - 1.0);
    const double gp = P.gamma * ((P.gamma - 1.0) * ug), sum = gp + b2;
    const double v[3] = {m1 * rinv, m2 * rinv, m3 * rinv};
    for (int d = 0; d < 3; d++) {
      double disc = sum * sum - 4.0 * gp * (B[d] * B[d]);
      if (disc < 0.0) disc = 0.0;
      const double cf = sqrt((sum + sqrt(disc)) / (2.0 * rho));
      const double s = fabs(v[d]) + cf;
      if (!(s > 0.0 && s < __longlong_as_double(0x7FF0000000000000ll))) { bad = true; continue; }
      const double cand = P.dx[d] / s;
      if (cand < best) best = cand;
    }
  }
  // warp shuffles, then the CTA's eight warps through shared memory: one atomic per CTA
  for (int o = 16; o > 0; o >>= 1) best = fmin(best, __shfl_xor_sync(0xffffffffu, best, o));
  __shared__ double wmin[8];
  __shared__ int anybad;
  if (threadIdx.x == 0) anybad = 0;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) wmin[threadIdx.x >> 5] = best;
  if (bad) anybad = 1;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; w++) best = fmin(best, wmin[w]);
    atomicMin(P.cells, (unsigned long long)__double_as_longlong(best));
    if (anybad) atomicAdd(P.cells + 2, 1ull);
  }
}

}  // namespace

// =================================== host side: the C-ABI of include/ak_mhd.h ===================================
struct akm_pack {
  Dev d{};
  double xmin[3]{}, xmax[3]{};
  std::vector<int> lx, leaf;
  double* u[2] = {nullptr, nullptr};
  void* work = nullptr;
  cudaStream_t stream = nullptr;
  int cur = 0, device = -1;
  bool bound = false, ghosts_ok = false;
  int recon = 0, nstages = 2, rsolver = 0;  // akm_pack_set_rsolver (0 HLLD, 1 LLF, 2 HLLE); akm_pack_set_recon (0 PLM, 1 PPM4, 2 PPMX, 3 WENOZ), akm_pack_set_integrator (2, 3)
  bool exact = false;          // akm_pack_set_exact: IEEE division / sqrt in the definition's order (bit-identical, slower)
  long long launches = 0;
};

namespace {
size_t align256(size_t n) { return (n + 255) & ~(size_t)255; }
struct WorkLayout { size_t cells, lx, leaf, W, F[3], Ec, total; };
WorkLayout work_layout(const akm_pack* p) {
  WorkLayout w;
  const size_t nc = (size_t)p->d.ncell * p->d.nmb;
  w.cells = 0;
  w.lx = 256;
  w.leaf = w.lx + align256(sizeof(int) * 3 * (size_t)p->d.nmb);
  w.W = w.leaf + align256(sizeof(int) * (size_t)p->d.nmb);
  w.F[0] = w.W + align256(8 * nc * sizeof(double));
  w.F[1] = w.F[0] + align256(7 * nc * sizeof(double));
  w.F[2] = w.F[1] + align256(7 * nc * sizeof(double));
  w.Ec = w.F[2] + align256(7 * nc * sizeof(double));
  w.total = w.Ec + align256(3 * nc * sizeof(double));
  return w;
}
struct Guard {
  int prev = -1;
  explicit Guard(int dev) { if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) cudaSetDevice(dev); else prev = -1; }
  ~Guard() { if (prev >= 0) cudaSetDevice(prev); }
};
}  // namespace

extern "C" const char* akm_last_error(void) { return g_err.c_str(); }

extern "C" akm_pack* akm_pack_create(int nmb, int nx1, int nx2, int nx3, int ng, double gamma, int nrb1, int nrb2, int nrb3,
                                     const int* lx, const double* xmin, const double* xmax) {
  if (nmb < 1 || !lx || !xmin || !xmax) { fail(-1, "bad arguments"); return nullptr; }
  if (ng < 3 || ng > 8) { fail(-1, "MHD with PLM needs 3 <= ng <= 8 (cell-centred fields of the outermost layer are not defined)"); return nullptr; }
  if (!(gamma > 1.0)) { fail(-1, "gamma <= 1"); return nullptr; }
  if ((long long)nmb != (long long)nrb1 * nrb2 * nrb3) { fail(-1, "a uniform pack has nrb1*nrb2*nrb3 blocks"); return nullptr; }
  akm_pack* p = new akm_pack;
  Dev& d = p->d;
  d.nmb = nmb; d.ng = ng; d.gamma = gamma;
  const int nx[3] = {nx1, nx2, nx3}, nrb[3] = {nrb1, nrb2, nrb3};
  for (int e = 0; e < 3; e++) {
    if (nx[e] < ng || nrb[e] < 1 || !(xmax[e] > xmin[e])) { fail(-1, "nx_d >= ng, nrb_d >= 1 and a non-empty domain are required"); delete p; return nullptr; }
    d.nx[e] = nx[e]; d.nt[e] = nx[e] + 2 * ng; d.nrb[e] = nrb[e];
    p->xmin[e] = xmin[e]; p->xmax[e] = xmax[e];
    d.dx[e] = (xmax[e] - xmin[e]) / ((double)nrb[e] * nx[e]);
  }
  d.ncell = (long long)d.nt[0] * d.nt[1] * d.nt[2];
  if (d.ncell >= (1ll << 31)) { fail(-3, "a MeshBlock with 2^31 or more cells (ghosts included) is not supported"); delete p; return nullptr; }
  p->lx.assign(lx, lx + 3 * (size_t)nmb);
  p->leaf.assign(nmb, -1);
  for (int m = 0; m < nmb; m++) {
    const int* l = &p->lx[3 * (size_t)m];
    for (int e = 0; e < 3; e++) if (l[e] < 0 || l[e] >= nrb[e]) { fail(-1, "logical location out of range"); delete p; return nullptr; }
    int& slot = p->leaf[((size_t)l[2] * nrb2 + l[1]) * nrb1 + l[0]];
    if (slot >= 0) { fail(-1, "duplicate block"); delete p; return nullptr; }
    slot = m;
  }
  return p;
}

extern "C" size_t akm_pack_state_bytes(const akm_pack* p) { return p ? (size_t)p->d.nmb * 8 * (size_t)p->d.ncell * 8 : 0; }
extern "C" size_t akm_pack_work_bytes(const akm_pack* p) { return p ? work_layout(p).total : 0; }

extern "C" int akm_pack_bind(akm_pack* p, void* u_a, void* u_b, void* work, void* cuda_stream) {
  if (!p) return fail(-1, "null pack");
  if (!u_a || !u_b || !work) return fail(-1, "null device buffer");
  if (((uintptr_t)u_a | (uintptr_t)u_b | (uintptr_t)work) & 255) return fail(-1, "buffers must be 256-byte aligned");
  const size_t sb = akm_pack_state_bytes(p);
  const WorkLayout wl = work_layout(p);
  auto overlap = [](const void* a, size_t na, const void* b, size_t nb) {
    return (uintptr_t)a < (uintptr_t)b + nb && (uintptr_t)b < (uintptr_t)a + na;
  };
  if (overlap(u_a, sb, u_b, sb) || overlap(u_a, sb, work, wl.total) || overlap(u_b, sb, work, wl.total))
    return fail(-1, "device buffers overlap");
  cudaPointerAttributes pa;
  AKM_CUDA(cudaPointerGetAttributes(&pa, u_a), "cudaPointerGetAttributes");
  if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) return fail(-1, "u_a is not a device pointer");
  p->device = pa.device;
  Guard guard(p->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  char* w = (char*)work;
  AKM_CUDA(cudaMemsetAsync(w, 0, 256, st), "memset work");
  AKM_CUDA(cudaMemcpyAsync(w + wl.lx, p->lx.data(), sizeof(int) * p->lx.size(), cudaMemcpyHostToDevice, st), "upload block table");
  AKM_CUDA(cudaMemcpyAsync(w + wl.leaf, p->leaf.data(), sizeof(int) * p->leaf.size(), cudaMemcpyHostToDevice, st), "upload leaf map");
  AKM_CUDA(cudaStreamSynchronize(st), "bind sync");
  Dev& d = p->d;
  d.cells = (unsigned long long*)w;
  d.lx = (const int*)(w + wl.lx);
  d.leaf = (const int*)(w + wl.leaf);
  d.W = (double*)(w + wl.W);
  for (int e = 0; e < 3; e++) d.F[e] = (double*)(w + wl.F[e]);
  d.Ec = (double*)(w + wl.Ec);
  p->u[0] = (double*)u_a; p->u[1] = (double*)u_b; p->work = work; p->stream = st;
  p->cur = 0; p->bound = true; p->ghosts_ok = false; p->launches = 0;
  return 0;
}

extern "C" int akm_pack_set_exact(akm_pack* p, int on) {
  if (!p) return fail(-1, "null pack");
  p->exact = on != 0;
  return 0;
}

extern "C" int akm_pack_set_recon(akm_pack* p, int recon) {
  if (!p) return fail(-1, "null pack");
  if (recon < 0 || recon > 3) return fail(-3, "reconstruction: 0 PLM, 1 PPM4, 2 PPMX, 3 WENOZ");
  if (recon != 0 && p->d.ng < 4) return fail(-1, "PPM4 / PPMX / WENOZ with face-centred fields need ng >= 4");
  if (recon != 0 && p->rsolver != 0) return fail(-3, "LLF / HLLE are built with PLM only");
  p->recon = recon;
  return 0;
}
extern "C" int akm_pack_set_rsolver(akm_pack* p, int rsolver) {
  if (!p) return fail(-1, "null pack");
  if (rsolver < 0 || rsolver > 2) return fail(-3, "Riemann solver: 0 HLLD, 1 LLF, 2 HLLE");
  if (rsolver != 0 && p->recon != 0) return fail(-3, "LLF / HLLE are built with PLM only");
  p->rsolver = rsolver;
  return 0;
}
extern "C" int akm_pack_set_integrator(akm_pack* p, int nstages) {
  if (!p) return fail(-1, "null pack");
  if (nstages != 2 && nstages != 3) return fail(-3, "integrator: 2 = SSPRK(2,2), 3 = SSPRK(3,3)");
  if (p->cur != 0) return fail(-2, "the integrator can only change between steps");
  p->nstages = nstages;
  return 0;
}

namespace {
template <int RECON, int RS>
void launch_sweeps_exact(const akm_pack* p, dim3 grid, const double* Uin) {
  flux_kernel<0, true, RECON, RS><<<grid, 128, 0, p->stream>>>(p->d, Uin);
  flux_kernel<1, true, RECON, RS><<<grid, 128, 0, p->stream>>>(p->d, Uin);
  flux_kernel<2, true, RECON, RS><<<grid, 128, 0, p->stream>>>(p->d, Uin);
}
void launch_sweeps(const akm_pack* p, dim3 grid, const double* Uin) {
  if (!p->exact) { akm::launch_sweeps_fast(p->d, p->recon, p->rsolver, grid, p->stream, Uin); return; }
  if (p->rsolver == 1) launch_sweeps_exact<0, 1>(p, grid, Uin);      // LLF / HLLE: PLM only (akm_pack_set_rsolver)
  else if (p->rsolver == 2) launch_sweeps_exact<0, 2>(p, grid, Uin);
  else if (p->recon == 1) launch_sweeps_exact<1, 0>(p, grid, Uin);
  else if (p->recon == 2) launch_sweeps_exact<2, 0>(p, grid, Uin);
  else if (p->recon == 3) launch_sweeps_exact<3, 0>(p, grid, Uin);
  else launch_sweeps_exact<0, 0>(p, grid, Uin);
}
}  // namespace

extern "C" int akm_fill_ghosts(akm_pack* p) {
  if (!p || !p->bound) return fail(-2, "pack not bound");
  Guard guard(p->device);
  const Dev& d = p->d;
  const long long nghost = d.ncell - (long long)d.nx[0] * d.nx[1] * d.nx[2];
  dim3 grid((unsigned)((nghost + 255) / 256), (unsigned)d.nmb);
  fill_kernel<<<grid, 256, 0, p->stream>>>(d, p->u[p->cur]);
  AKM_CUDA(cudaGetLastError(), "akm_fill_ghosts launch");
  p->launches += 1;
  p->ghosts_ok = true;
  return 0;
}

extern "C" int akm_stage(akm_pack* p, int stage, double dt) {
  if (!p || !p->bound) return fail(-2, "pack not bound");
  const int ns = p->nstages;
  if (stage < 1 || stage > ns) return fail(-1, "stage must be 1 .. number of stages of the integrator");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(-1, "dt must be positive and finite");
  if (p->cur != (stage == 1 ? 0 : 1)) return fail(-2, "stages must be called in order, starting from U^n in buffer A");
  if (!p->ghosts_ok) return fail(-2, "akm_fill_ghosts must precede akm_stage");
  Guard guard(p->device);
  // U_out = g0 U_in + g1 U^n - beta dt L(U_in).  SSPRK(2,2): A -> B, (B, A) -> A.  SSPRK(3,3): A -> B, (B, A) -> B in place
  // (the update is pointwise once the fluxes and EMFs are in the work buffer), (B, A) -> A.  DESIGN.md Q1
  static const double C2[2][3] = {{0.0, 1.0, 1.0}, {0.5, 0.5, 0.5}};
  static const double C3[3][3] = {{0.0, 1.0, 1.0}, {0.25, 0.75, 0.25}, {2.0 / 3.0, 1.0 / 3.0, 2.0 / 3.0}};
  const double* cf = (ns == 2) ? C2[stage - 1] : C3[stage - 1];
  const double g0 = cf[0], g1 = cf[1], beta = cf[2];
  const int out = (stage == ns) ? 0 : 1;
  const Dev& d = p->d;
  const double* Uin = p->u[p->cur];
  double* Uout = p->u[out];
  dim3 gall256((unsigned)((d.ncell + 255) / 256), (unsigned)d.nmb), gall128((unsigned)((d.ncell + 127) / 128), (unsigned)d.nmb);
  const long long nact = (long long)d.nx[0] * d.nx[1] * d.nx[2];
  dim3 gact((unsigned)((nact + 127) / 128), (unsigned)d.nmb);
  prim_kernel<<<gall256, 256, 0, p->stream>>>(d, Uin);
  launch_sweeps(p, gall128, Uin);
  const double k0 = 1024.0 * dt / d.dx[0], k1 = 1024.0 * dt / d.dx[1], k2 = 1024.0 * dt / d.dx[2];
  if (p->exact) emf_kernel<true><<<gall128, 128, 0, p->stream>>>(d, k0, k1, k2);
  else emf_kernel<false><<<gall128, 128, 0, p->stream>>>(d, k0, k1, k2);
  update_kernel<<<gact, 128, 0, p->stream>>>(d, Uin, p->u[0], Uout, g0, g1, beta * dt / d.dx[0], beta * dt / d.dx[1], beta * dt / d.dx[2]);
  AKM_CUDA(cudaGetLastError(), "akm_stage launch");
  p->launches += 6;
  p->cur = out;
  p->ghosts_ok = false;
  return 0;
}

extern "C" int akm_new_dt(akm_pack* p, double cfl, double* dt_out) {
  if (!p || !p->bound) return fail(-2, "pack not bound");
  if (!dt_out) return fail(-1, "null dt_out");
  if (!(cfl > 0.0)) return fail(-1, "cfl must be positive");
  Guard guard(p->device);
  const Dev& d = p->d;
  const long long nact = (long long)d.nx[0] * d.nx[1] * d.nx[2];
  dim3 gact((unsigned)((nact + 255) / 256), (unsigned)d.nmb);
  dt_init_kernel<<<1, 1, 0, p->stream>>>(d);
  dt_kernel<<<gact, 256, 0, p->stream>>>(d, p->u[p->cur]);
  AKM_CUDA(cudaGetLastError(), "akm_new_dt launch");
  p->launches += 2;
  unsigned long long cells[3];
  AKM_CUDA(cudaMemcpyAsync(cells, d.cells, 24, cudaMemcpyDeviceToHost, p->stream), "akm_new_dt copy");
  AKM_CUDA(cudaStreamSynchronize(p->stream), "akm_new_dt sync");
  double dtmin;
  std::memcpy(&dtmin, &cells[0], 8);
  if (cells[2] || !(dtmin > 0.0) || !std::isfinite(dtmin)) return fail(-5, "non-finite signal speed in the state (NaN or inf in an active cell)");
  *dt_out = cfl * dtmin;
  return 0;
}

extern "C" int akm_step(akm_pack* p, double cfl, double dt_fixed, double* dt_out) {
  double dt = dt_fixed;
  if (!(dt_fixed > 0.0)) { int rc = akm_new_dt(p, cfl, &dt); if (rc) return rc; }
  for (int stage = 1; stage <= p->nstages; stage++) {
    int rc = akm_fill_ghosts(p); if (rc) return rc;
    rc = akm_stage(p, stage, dt); if (rc) return rc;
  }
  if (dt_out) *dt_out = dt;
  return 0;
}

extern "C" void* akm_pack_current(const akm_pack* p) { return (p && p->bound) ? (void*)p->u[p->cur] : nullptr; }
extern "C" long long akm_pack_launch_count(const akm_pack* p) { return p ? p->launches : -1; }
extern "C" long long akm_pack_floor_count(akm_pack* p) {
  if (!p || !p->bound) { fail(-2, "pack not bound"); return -1; }
  Guard guard(p->device);
  unsigned long long n = 0;
  if (cudaMemcpyAsync(&n, p->d.cells + 1, 8, cudaMemcpyDeviceToHost, p->stream) != cudaSuccess ||
      cudaStreamSynchronize(p->stream) != cudaSuccess) { fail(-4, "akm_pack_floor_count copy failed"); return -1; }
  return (long long)n;
}
extern "C" int akm_pack_destroy(akm_pack* p) { delete p; return 0; }
#else   // AKM_FAST_TU: only the sweeps of the default flavour
}  // namespace

namespace akm {
template <int RECON, int RS>
static void sweeps(const Dev& d, dim3 grid, cudaStream_t st, const double* Uin) {
  flux_kernel<0, false, RECON, RS><<<grid, 128, 0, st>>>(d, Uin);
  flux_kernel<1, false, RECON, RS><<<grid, 128, 0, st>>>(d, Uin);
  flux_kernel<2, false, RECON, RS><<<grid, 128, 0, st>>>(d, Uin);
}
void launch_sweeps_fast(const Dev& d, int recon, int rsolver, dim3 grid, cudaStream_t st, const double* Uin) {
  if (rsolver == 1) sweeps<0, 1>(d, grid, st, Uin);                  // LLF / HLLE: PLM only (akm_pack_set_rsolver)
  else if (rsolver == 2) sweeps<0, 2>(d, grid, st, Uin);
  else if (recon == 1) sweeps<1, 0>(d, grid, st, Uin);
  else if (recon == 2) sweeps<2, 0>(d, grid, st, Uin);
  else if (recon == 3) sweeps<3, 0>(d, grid, st, Uin);
  else sweeps<0, 0>(d, grid, st, Uin);
}
}  // namespace akm
#endif

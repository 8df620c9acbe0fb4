// ak_physics.cuh -- per-cell / per-face device arithmetic of the hydro stage (sm_100a, fp64).
// conserved->primitive (paper Eq.(4)), PLM / PPM4 reconstruction of the primitives
// (P:101), HLLC flux.  The formulas are the readings listed in DESIGN.md (Q1-Q7).
// This header is part of the CUDA path only; the CPU oracle shares nothing with it.
#pragma once
#include <cuda_runtime.h>

namespace ak {

constexpr double RHO_FLOOR = 1e-20;
constexpr double P_FLOOR   = 1e-20;

// ---- fast fp64 reciprocal / rsqrt ----------------------------------------------------------------
// The FP64 pipe is the binding resource of this path, and IEEE division /
// sqrt cost ~10-14 FP64-pipe instructions each plus a slow-path branch.  rcp.approx.ftz.f64 /
// rsqrt.approx.ftz.f64 (MUFU.RCP64H / MUFU.RSQ64H, ~20 significant bits, issued on the SFU pipe)
// followed by two Newton steps give <= ~1 ulp results for normal arguments in 4-5 FP64 instructions.
// Arguments here (densities, pressures, wave-speed differences) are far from the denormal /
// overflow range where the approximations lose accuracy.
__device__ __forceinline__ double rcp_fast(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}
// a / b to ~1 ulp: quotient with one residual correction
__device__ __forceinline__ double div_fast(double a, double b) {
  double r = rcp_fast(b);
  double q = a * r;
  double res = fma(-b, q, a);
  return fma(res, r, q);
}
__device__ __forceinline__ double rsqrt_fast(double x) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  // Newton for y = x^{-1/2}: r <- r + r*(1 - x r^2)/2, twice
  double hx = 0.5 * x;
  double e = fma(-hx * r, r, 0.5);
  r = fma(r, e, r);
  e = fma(-hx * r, r, 0.5);
  r = fma(r, e, r);
  return r;
}
// sqrt(x) to ~1 ulp for x > 0 (x = 0 handled by the callers that can see it)
__device__ __forceinline__ double sqrt_fast(double x) {
  double r = rsqrt_fast(x);
  double s = x * r;
  double res = fma(-s, s, x);
  return fma(0.5 * res, r, s);
}


#ifdef AK_EXACT_MATH
__device__ __forceinline__ double rcp_(double x)  { return 1.0 / x; }
__device__ __forceinline__ double div_(double a, double b) { return a / b; }
__device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
#else
__device__ __forceinline__ double rcp_(double x)  { return rcp_fast(x); }
__device__ __forceinline__ double div_(double a, double b) { return div_fast(a, b); }
__device__ __forceinline__ double sqrt_(double x) { return sqrt_fast(x); }
#endif

// ---- S1  conserved -> primitive, W = (rho, v1, v2, v3, u_g) --------------------------------------
// returns the number of floor activations (0 on every BASELINE config)
__device__ __forceinline__ int c2p(const double U[5], double W[5], double ug_floor) {
  int nfl = 0;
  double rho = U[0];
  if (!(rho >= RHO_FLOOR)) { rho = RHO_FLOOR; nfl++; }
  double rinv = rcp_(rho);
  double ke2 = U[1] * U[1] + (U[2] * U[2] + U[3] * U[3]);
  double ug = U[4] - 0.5 * rinv * ke2;
  if (!(ug >= ug_floor)) { ug = ug_floor; nfl++; }
  W[0] = rho; W[1] = U[1] * rinv; W[2] = U[2] * rinv; W[3] = U[3] * rinv; W[4] = ug;
  return nfl;
}

// ---- S2  reconstruction -------------------------------------------------------------------------
// PLM, van Leer: half-slope h = dL*dR/(dL+dR) where dL*dR > 0, else 0; q- = q - h, q+ = q + h.
__device__ __forceinline__ double plm_halfslope(double qm1, double q0, double qp1) {
  double dL = q0 - qm1, dR = qp1 - q0;
  double prod = dL * dR;
  return (prod > 0.0) ? div_(prod, dL + dR) : 0.0;
}

// PPM4 (i)+(ii): fourth-order interface value between q0 and qp1, clamped into [min,max](q0,qp1).
__device__ __forceinline__ double ppm4_iface(double qm1, double q0, double qp1, double qp2) {
  double v = (7.0 * (q0 + qp1) - (qm1 + qp2)) * (1.0 / 12.0);
  return fmax(fmin(q0, qp1), fmin(v, fmax(q0, qp1)));
}
// PPM4 (iii): CW84 Eq.(1.10) on (aL, a, aR); results in aL (= q-) and aR (= q+).
__device__ __forceinline__ void ppm4_limit(double a, double& aL, double& aR) {
  if ((aR - a) * (a - aL) <= 0.0) {
    aL = a; aR = a;
  } else {
    double d = aR - aL;
    double mu = a - 0.5 * (aL + aR);
    double dmu = d * mu, d26 = d * d * (1.0 / 6.0);
    if (dmu > d26)       aL = 3.0 * a - 2.0 * aR;
    else if (-d26 > dmu) aR = 3.0 * a - 2.0 * aL;
  }
}

// ---- S3  HLLC flux ------------------------------------------------------------------------------
// WL/WR are (rho, u, v, w, u_g) ALREADY ROTATED so that u is the face-normal velocity and (v, w)
// the cyclic transverse pair; F is returned in the same rotated order (mass, normal momentum,
// transverse momenta, energy).
struct GasConst {
  double gamma, gm1, ug_floor;
};

__device__ __forceinline__ void hllc(const GasConst& g, const double WL[5], const double WR[5], double F[5]) {
  const double rL = WL[0], uL = WL[1], vL = WL[2], wL = WL[3], eL = WL[4];
  const double rR = WR[0], uR = WR[1], vR = WR[2], wR = WR[3], eR = WR[4];
  const double pL = g.gm1 * eL, pR = g.gm1 * eR;
  const double rLinv = rcp_(rL), rRinv = rcp_(rR);
  const double cL = sqrt_(g.gamma * pL * rLinv), cR = sqrt_(g.gamma * pR * rRinv);
  // Davis's direct wave-speed estimates (Q2, round-2 reading; Toro Eq.(10.48))
  const double sl1 = uL - cL, sl2 = uR - cR, sr1 = uL + cL, sr2 = uR + cR;
  const double SL = sl2 < sl1 ? sl2 : sl1, SR = sr1 > sr2 ? sr1 : sr2;    // (NaN c_L -> S_L, NaN c_R -> S_R)
  const double bm = fmin(SL, 0.0), bp = fmax(SR, 0.0);
  const double mL = rL * (uL - SL), mR = rR * (SR - uR);
  const double Ss = ((pL - pR) + (mL * uL + mR * uR)) * rcp_(mL + mR);
  const double psL = pL + rL * (SL - uL) * (Ss - uL);
  const double psR = pR + rR * (SR - uR) * (Ss - uR);
  const double ps = fmax(0.5 * (psL + psR), 0.0);
  const bool left = (Ss >= 0.0);
  const double rK = left ? rL : rR, uK = left ? uL : uR, vK = left ? vL : vR, wK = left ? wL : wR;
  const double eK = left ? eL : eR, pK = left ? pL : pR, b = left ? bm : bp;
  const double EK = eK + 0.5 * rK * (uK * uK + (vK * vK + wK * wK));
  const double mom = rK * uK;
  const double inv = rcp_(Ss - b);
  const double bps = b * ps;
  // F_n = [S*(F_K,n - b U_K,n) - b p* D_n] / (S* - b),  D = (0,1,0,0,S*)
  F[0] = Ss * (mom - b * rK) * inv;
  F[1] = (Ss * ((mom * uK + pK) - b * mom) - bps) * inv;
  F[2] = Ss * (mom * vK - b * (rK * vK)) * inv;
  F[3] = Ss * (mom * wK - b * (rK * wK)) * inv;
  F[4] = (Ss * ((EK + pK) * uK - b * EK) - bps * Ss) * inv;
}

}  // namespace ak

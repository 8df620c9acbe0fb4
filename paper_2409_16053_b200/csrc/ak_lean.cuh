// ak_lean.cuh -- branch-free, instruction-lean forms of the per-cell / per-face arithmetic for the
// production stage kernel (ak_stage_v3.cuh).  Same formulas as ak_physics.cuh (DESIGN.md section 2
// readings Q1-Q7, Q29-Q31; paper P:101 reconstruction on primitives, P:103 HLLC, P:122-126 gamma-law gas); they
// differ from it by rounding only (a few ulp) and are written against what the ncu captures of round 1 showed to be
// expensive on sm_100a (every FP64-pipe and every ALU-pipe instruction costs about two issue cycles):
//   * fmin/fmax on doubles lower to DSETP + SEL/FSEL + several moves (NaN handling): replaced by one
//     compare + select, or by a sign test of the high word on the integer pipe where the other operand is 0;
//   * data-dependent branches (shock branch of the wave speeds, CW84 limiter cases) diverge inside a warp
//     on turbulent data and cost BSSY/BSYNC: everything here is straight-line code with selects;
//   * IEEE division / sqrt: MUFU.RCP64H / RSQ64H seed + Newton, as in ak_physics.cuh.
#pragma once
#include "ak_physics.cuh"

namespace ak {

// sign tests on the integer pipe.  neg(): true for x < 0 and -0.  pos(): true for x > 0 except positive
// denormals below 2^-1042 (treated as zero; they only ever gate a slope of that size).
__device__ __forceinline__ bool neg(double x) { return __double2hiint(x) < 0; }
__device__ __forceinline__ bool pos(double x) { return __double2hiint(x) > 0; }
__device__ __forceinline__ double max0(double x) { return neg(x) ? 0.0 : x; }
__device__ __forceinline__ double min0(double x) { return neg(x) ? x : 0.0; }

// 1/x to ~1 ulp: MUFU seed (>= 20 bits, error e) + ONE cubically convergent step r (1 + e + e^2), whose
// truncation error e^3 < 2^-60 is below the rounding error                      3 FP64 + 1 MUFU
__device__ __forceinline__ double rcp2(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  return fma(r, fma(e, e, e), r);
}
// a / b to ~1.5 ulp                                                              4 FP64 + 1 MUFU
__device__ __forceinline__ double div2(double a, double b) { return a * rcp2(b); }

// ---- S1  conserved -> primitive ------------------------------------------------------------------
__device__ __forceinline__ int c2p_lean(const double U[5], double W[5], double ug_floor) {
  int nfl = 0;
  double rho = U[0];
  if (!(rho >= RHO_FLOOR)) { rho = RHO_FLOOR; nfl++; }
  const double rinv = rcp2(rho);
  const double ke2 = fma(U[1], U[1], fma(U[2], U[2], U[3] * U[3]));
  double ug = fma(-0.5 * rinv, ke2, U[4]);
  if (!(ug >= ug_floor)) { ug = ug_floor; nfl++; }
  W[0] = rho; W[1] = U[1] * rinv; W[2] = U[2] * rinv; W[3] = U[3] * rinv; W[4] = ug;
  return nfl;
}

// ---- S2  reconstruction --------------------------------------------------------------------------
// PLM, van Leer: q-/q+ of the cell with neighbours (m1, c, p1)
__device__ __forceinline__ void plm_lean(double m1, double c, double p1, double& qm, double& qp) {
  const double dL = c - m1, dR = p1 - c, prod = dL * dR;
  const double q = div2(prod, dL + dR);          // discarded by the select where prod <= 0 (may be NaN)
  const double h = pos(prod) ? q : 0.0;
  qm = c - h; qp = c + h;
}

// PPM4 (i)+(ii): 4th-order interface value between q0 and q1 clamped into [min,max](q0,q1)   7 FP64
__device__ __forceinline__ double iface_lean(double qm1, double q0, double q1, double q2) {
  const double v = fma(7.0, q0 + q1, -(qm1 + q2)) * (1.0 / 12.0);
  // median(v, q0, q1) with three compares whose XORs fold into the DSETPs, and two selects
  const bool c0 = v < q0;
  const bool inside = (v < q1) != c0;          // v strictly between q0 and q1
  const bool far = (q0 < q1) != c0;            // otherwise: the bound on v's side is q1 (else q0)
  const double bound = far ? q1 : q0;
  return inside ? v : bound;
}
// PPM4 (iii): CW84 Eq.(1.10), straight-line, in difference form.  With x = aR - a, y = a - aL (same sign
// unless the cell is an extremum) one has d = aR - aL = x + y, 6 mu = 3 (y - x), hence
//   d mu >  d^2/6  <=>  d (y - 2x) > 0  <=>  y - 2x has the sign of y,   and then aL <- 3a - 2aR = a - 2x
//   -d^2/6 > d mu  <=>  d (2y - x) < 0  <=>  2y - x has the sign of -y,  and then aR <- 3a - 2aL = a + 2y
// The sign tests run on the integer pipe.  At a tie the replaced value equals the old one (the limiter is
// continuous), so a decision that flips through rounding moves the result by rounding error only.   7 FP64
__device__ __forceinline__ void limit_lean(double a, double& aL, double& aR) {
  const double x = aR - a, y = a - aL;
  const bool flat = !pos(x * y);
  const double tL = fma(-2.0, x, y), tR = fma(2.0, y, -x);
  const double nL = fma(-2.0, x, a), nR = fma(2.0, y, a);
  const int hy = __double2hiint(y);
  const bool cL = (__double2hiint(tL) ^ hy) >= 0, cR = (__double2hiint(tR) ^ hy) < 0;
  aL = flat ? a : (cL ? nL : aL);
  aR = flat ? a : (cR ? nR : aR);
}

// ---- S2'  PPMX and WENOZ (paper P:101; Q29, Q30), straight-line -----------------------------
// select-min on doubles without the NaN handling of fmin (operands are finite here)
__device__ __forceinline__ double dmin2(double a, double b) { return a < b ? a : b; }

// WENO-Z edge values of the middle cell of q[i-2..i+2], in the differences of neighbouring cells (constants are
// reproduced exactly); same operation order as the oracle, reciprocals by rcp2.  q+ is the value at the upper face;
// q- is the same formula on the mirrored stencil, for which the smoothness indicators are those of q+ in reverse
// order (beta0' = beta2, beta1' = beta1, beta2' = beta0, bit for bit, hence the same tau5 and the same ratios) and the
// candidate polynomials are -(5 d3 - 2 d4), -(2 d2 + d3), -(4 d2 - d1): the indicators, tau5 and the three
// reciprocals are formed once for both sides.
__device__ __forceinline__ void wenoz_lean(const double q[5], double& qm, double& qp) {
  const double c = q[2];
  const double d1 = q[1] - q[0], d2 = q[2] - q[1], d3 = q[3] - q[2], d4 = q[4] - q[3];
  const double s0 = d2 - d1, t0 = 3.0 * d2 - d1;
  const double s1 = d3 - d2, t1 = d2 + d3;
  const double s2 = d4 - d3, t2 = d4 - 3.0 * d3;
  const double b0 = (13.0 / 12.0) * (s0 * s0) + 0.25 * (t0 * t0);
  const double b1 = (13.0 / 12.0) * (s1 * s1) + 0.25 * (t1 * t1);
  const double b2 = (13.0 / 12.0) * (s2 * s2) + 0.25 * (t2 * t2);
  const double eps = 1e-40;
  const double tau = fabs(b0 - b2);
  const double r0 = tau * rcp2(b0 + eps), r1 = tau * rcp2(b1 + eps), r2 = tau * rcp2(b2 + eps);
  const double w0 = 1.0 + r0 * r0, w1 = 1.0 + r1 * r1, w2 = 1.0 + r2 * r2;
  {
    const double P0 = 5.0 * d2 - 2.0 * d1, P1 = 2.0 * d3 + d2, P2 = 4.0 * d3 - d4;
    const double a0 = 0.1 * w0, a1 = 0.6 * w1, a2 = 0.3 * w2;
    qp = c + (a0 * P0 + (a1 * P1 + a2 * P2)) * rcp2(6.0 * (a0 + (a1 + a2)));
  }
  {
    const double P0 = -(5.0 * d3 - 2.0 * d4), P1 = -(2.0 * d2 + d3), P2 = -(4.0 * d2 - d1);
    const double a0 = 0.1 * w2, a1 = 0.6 * w1, a2 = 0.3 * w0;
    qm = c + (a0 * P0 + (a1 * P1 + a2 * P2)) * rcp2(6.0 * (a0 + (a1 + a2)));
  }
}

// PPMX (i): fourth-order interface value between q0 and q1, limited where it is not between them
__device__ __forceinline__ double ppmx_iface(double qm1, double q0, double q1, double q2) {
  const double v = (7.0 * (q0 + q1) - (qm1 + q2)) * (1.0 / 12.0);
  const double dc = 3.0 * ((q0 + q1) - 2.0 * v);
  const double dl = (qm1 + q1) - 2.0 * q0, dr = (q0 + q2) - 2.0 * q1;
  const bool same = (dc > 0.0 && dl > 0.0 && dr > 0.0) || (dc < 0.0 && dl < 0.0 && dr < 0.0);
  const double m = dmin2(fabs(dc), 1.25 * dmin2(fabs(dl), fabs(dr)));
  const double D = same ? copysign(m, dc) : 0.0;
  const double lim = 0.5 * (q0 + q1) - D * (1.0 / 6.0);
  return ((v - q0) * (q1 - v) < 0.0) ? lim : v;
}
// PPMX (ii): limited parabola of the middle cell of q[i-2..i+2]
__device__ __forceinline__ void ppmx_lean(const double q[5], double& qm, double& qp) {
  const double a = q[2];
  const double aL = ppmx_iface(q[0], q[1], q[2], q[3]);
  const double aR = ppmx_iface(q[1], q[2], q[3], q[4]);
  const double dm = a - aL, dp = aR - a;
  const bool ext = (dm * dp <= 0.0) || ((q[3] - a) * (a - q[1]) <= 0.0);
  const double df = 6.0 * ((aL + aR) - 2.0 * a);
  const double d1 = (q[0] + q[2]) - 2.0 * q[1], d2 = (q[1] + q[3]) - 2.0 * q[2], d3 = (q[2] + q[4]) - 2.0 * q[3];
  const bool same = (df > 0.0 && d1 > 0.0 && d2 > 0.0 && d3 > 0.0) || (df < 0.0 && d1 < 0.0 && d2 < 0.0 && d3 < 0.0);
  const double m = dmin2(fabs(df), 1.25 * dmin2(fabs(d1), dmin2(fabs(d2), fabs(d3))));
  const double D = same ? copysign(m, df) : 0.0;
  const double rho = (df != 0.0) ? div2(D, df) : 0.0;
  const bool use = rho <= 1.0 - 1e-12;
  const double eL = use ? a - rho * dm : aL, eR = use ? a + rho * dp : aR;
  const double mL = (fabs(dm) >= 2.0 * fabs(dp)) ? a - 2.0 * dp : aL;
  const double mR = (fabs(dp) >= 2.0 * fabs(dm)) ? a + 2.0 * dm : aR;
  qm = ext ? eL : mL;
  qp = ext ? eR : mR;
}
// q-/q+ of the middle cell of five values: RECON 2 = PPMX, 3 = WENOZ
template <int RECON>
__device__ __forceinline__ void recon5(const double q[5], double& qm, double& qp) {
  if constexpr (RECON == 2) ppmx_lean(q, qm, qp);
  else wenoz_lean(q, qm, qp);
}

// q-/q+ of the cell at p[0] from the stencil along stride st: RECON 0 = PLM, 1 = PPM4, 2 = PPMX, 3 = WENOZ
template <int RECON>
__device__ __forceinline__ void recon2(const double* p, int st, double& qm, double& qp) {
  if constexpr (RECON == 0) {
    plm_lean(p[-st], p[0], p[st], qm, qp);
  } else if constexpr (RECON >= 2) {
    const double q[5] = {p[-2 * st], p[-st], p[0], p[st], p[2 * st]};
    recon5<RECON>(q, qm, qp);
  } else {
    const double m2 = p[-2 * st], m1 = p[-st], a = p[0], p1 = p[st], p2 = p[2 * st];
    double lo = iface_lean(m2, m1, a, p1);
    double hi = iface_lean(m1, a, p1, p2);
    limit_lean(a, lo, hi);
    qm = lo; qp = hi;
  }
}

// sqrt(a / b) = a (a b)^(-1/2) for a, b > 0 without a division: MUFU seed r of t^(-1/2) (error e = 1 - t r^2
// <= 2^-19) + ONE cubic (Halley) step r (1 + e/2 + 3 e^2/8), truncation 5/16 e^3 < 2^-58    7 FP64 + 1 MUFU
__device__ __forceinline__ double sqrt_ratio(double a, double b) {
  const double t = a * b;
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(t));
  const double e = fma(-(t * r), r, 1.0);
  r = fma(r, e * fma(0.375, e, 0.5), r);
  return fabs(a) * r;              // (a, b < 0 together, an unphysical face state: the positive root, like sqrt(a / b))
}

// ---- S3  HLLC, rotated states (rho, u_normal, v, w, u_g) -------------------------------------------
// Wave speeds: Davis's direct estimates S_L = min(u_L - c_L, u_R - c_R), S_R = max(u_L + c_L, u_R + c_R) (Q2,
// round-2 reading): always S_L < S* < S_R, so the star flux is finite for head-on collisions at any Mach number.
// Straight-line; the upwind side is chosen by the sign of S*.  ~70 FP64-pipe instructions + 4 MUFU.
__device__ __forceinline__ void hllc2(const GasConst& g, const double WL[5], const double WR[5], double F[5]) {
  const double rL = WL[0], uL = WL[1], eL = WL[4];
  const double rR = WR[0], uR = WR[1], eR = WR[4];
  const double pL = g.gm1 * eL, pR = g.gm1 * eR;
  const double ggm1 = g.gamma * g.gm1;
  const double cL = sqrt_ratio(ggm1 * eL, rL), cR = sqrt_ratio(ggm1 * eR, rR);
  const double sl1 = uL - cL, sl2 = uR - cR, sr1 = uL + cL, sr2 = uR + cR;
  // (this operand order lets a NaN c_L reach S_L and a NaN c_R reach S_R: an unphysical face state gives a NaN flux on
  // both sides, Q31; for finite operands min and max)
  const double SL = sl2 < sl1 ? sl2 : sl1, SR = sr1 > sr2 ? sr1 : sr2;
  const double mL = rL * (uL - SL), mR = rR * (SR - uR);
  const double Ss = div2((pL - pR) + fma(mL, uL, mR * uR), mL + mR);
  const double psL = fma(-mL, Ss - uL, pL);
  const double psR = fma(mR, Ss - uR, pR);
  const double ps = max0(0.5 * (psL + psR));
  const bool left = !neg(Ss);
  const double rK = left ? rL : rR, uK = left ? uL : uR, vK = left ? WL[2] : WR[2], wK = left ? WL[3] : WR[3];
  const double eK = left ? eL : eR, pK = left ? pL : pR;      // (p_K = (gamma-1) e_K would save the select but costs spills in the 128-register tile)
  // b = min(S_L, 0) on the left of the contact, max(S_R, 0) on its right: one select of the speed, one sign test
  const double SK = left ? SL : SR;
  const double b = (neg(SK) == left) ? SK : 0.0;
  const double EK = fma(0.5 * rK, fma(uK, uK, fma(vK, vK, wK * wK)), eK);
  const double mom = rK * uK;
  const double inv = rcp2(Ss - b);
  const double w = Ss * inv;                       // S*/(S* - b)
  const double bps = b * ps;
  const double f0 = fma(-b, rK, mom) * w;
  F[0] = f0;
  F[1] = fma(Ss, fma(-b, mom, fma(mom, uK, pK)), -bps) * inv;
  F[2] = f0 * vK;
  F[3] = f0 * wK;
  F[4] = (fma(-b, EK, (EK + pK) * uK) - bps) * w;
}

// direction D known at compile time: pick the normal / cyclic transverse components, un-rotate the flux
template <int D>
__device__ __forceinline__ void flux2(const GasConst& g, const double L[5], const double Rr[5], double F[5]) {
  const double l[5] = {L[0], L[1 + D], L[1 + (D + 1) % 3], L[1 + (D + 2) % 3], L[4]};
  const double r[5] = {Rr[0], Rr[1 + D], Rr[1 + (D + 1) % 3], Rr[1 + (D + 2) % 3], Rr[4]};
  double f[5];
  hllc2(g, l, r, f);
  F[0] = f[0]; F[1 + D] = f[1]; F[1 + (D + 1) % 3] = f[2]; F[1 + (D + 2) % 3] = f[3]; F[4] = f[4];
}
// direction x1 (d2 = false) or x2 (d2 = true) chosen at run time: used by the tile-edge threads so that the
// x1-edge and x2-edge faces of a tile run through ONE instruction stream instead of two divergent ones
__device__ __forceinline__ void flux2_12(const GasConst& g, bool d2, const double L[5], const double Rr[5], double F[5]) {
  const double l[5] = {L[0], d2 ? L[2] : L[1], d2 ? L[3] : L[2], d2 ? L[1] : L[3], L[4]};
  const double r[5] = {Rr[0], d2 ? Rr[2] : Rr[1], d2 ? Rr[3] : Rr[2], d2 ? Rr[1] : Rr[3], Rr[4]};
  double f[5];
  hllc2(g, l, r, f);
  F[0] = f[0];
  F[1] = d2 ? f[3] : f[1];
  F[2] = d2 ? f[1] : f[2];
  F[3] = d2 ? f[2] : f[3];
  F[4] = f[4];
}

// N independent faces solved in lock step: every statement of hllc2 is written as a loop over the faces, so
// that the N dependency chains (about 45 FP64 operations deep at ~9 cycles each on sm_100a) are adjacent in
// the instruction stream and ptxas can interleave them.  Same arithmetic per face as hllc2, bit for bit.
template <int N>
__device__ __forceinline__ void hllc2n(const GasConst& g, const double WL[N][5], const double WR[N][5], double F[N][5]) {
  const double ggm1 = g.gamma * g.gm1;
  double pL[N], pR[N], cL[N], cR[N], SL[N], SR[N], mL[N], mR[N], Ss[N];
#pragma unroll
  for (int f = 0; f < N; f++) { pL[f] = g.gm1 * WL[f][4]; pR[f] = g.gm1 * WR[f][4]; }
#pragma unroll
  for (int f = 0; f < N; f++) { cL[f] = sqrt_ratio(ggm1 * WL[f][4], WL[f][0]); cR[f] = sqrt_ratio(ggm1 * WR[f][4], WR[f][0]); }
#pragma unroll
  for (int f = 0; f < N; f++) {
    const double sl1 = WL[f][1] - cL[f], sl2 = WR[f][1] - cR[f], sr1 = WL[f][1] + cL[f], sr2 = WR[f][1] + cR[f];
    SL[f] = sl2 < sl1 ? sl2 : sl1; SR[f] = sr1 > sr2 ? sr1 : sr2;     // (NaN c_L -> S_L, NaN c_R -> S_R, as in hllc2)
    mL[f] = WL[f][0] * (WL[f][1] - SL[f]); mR[f] = WR[f][0] * (SR[f] - WR[f][1]);
  }
#pragma unroll
  for (int f = 0; f < N; f++)
    Ss[f] = div2((pL[f] - pR[f]) + fma(mL[f], WL[f][1], mR[f] * WR[f][1]), mL[f] + mR[f]);
  double ps[N], rK[N], uK[N], vK[N], wK[N], eK[N], pK[N], b[N];
#pragma unroll
  for (int f = 0; f < N; f++) {
    const double psL = fma(-mL[f], Ss[f] - WL[f][1], pL[f]);
    const double psR = fma(mR[f], Ss[f] - WR[f][1], pR[f]);
    ps[f] = max0(0.5 * (psL + psR));
    const bool left = !neg(Ss[f]);
    rK[f] = left ? WL[f][0] : WR[f][0]; uK[f] = left ? WL[f][1] : WR[f][1];
    vK[f] = left ? WL[f][2] : WR[f][2]; wK[f] = left ? WL[f][3] : WR[f][3];
    eK[f] = left ? WL[f][4] : WR[f][4]; pK[f] = left ? pL[f] : pR[f];
    const double SK = left ? SL[f] : SR[f];
    b[f] = (neg(SK) == left) ? SK : 0.0;
  }
  double EK[N], mom[N], inv[N];
#pragma unroll
  for (int f = 0; f < N; f++) {
    EK[f] = fma(0.5 * rK[f], fma(uK[f], uK[f], fma(vK[f], vK[f], wK[f] * wK[f])), eK[f]);
    mom[f] = rK[f] * uK[f];
    inv[f] = rcp2(Ss[f] - b[f]);
  }
#pragma unroll
  for (int f = 0; f < N; f++) {
    const double w = Ss[f] * inv[f];               // S*/(S* - b)
    const double bps = b[f] * ps[f];
    const double f0 = fma(-b[f], rK[f], mom[f]) * w;
    F[f][0] = f0;
    F[f][1] = fma(Ss[f], fma(-b[f], mom[f], fma(mom[f], uK[f], pK[f])), -bps) * inv[f];
    F[f][2] = f0 * vK[f];
    F[f][3] = f0 * wK[f];
    F[f][4] = (fma(-b[f], EK[f], (EK[f] + pK[f]) * uK[f]) - bps) * w;
  }
}

// the lower x1 and x2 faces of one cell, solved together
__device__ __forceinline__ void flux2_x1x2(const GasConst& g, const double L1[5], const double R1[5], const double L2[5],
                                           const double R2[5], double F1[5], double F2[5]) {
  const double l[2][5] = {{L1[0], L1[1], L1[2], L1[3], L1[4]}, {L2[0], L2[2], L2[3], L2[1], L2[4]}};
  const double r[2][5] = {{R1[0], R1[1], R1[2], R1[3], R1[4]}, {R2[0], R2[2], R2[3], R2[1], R2[4]}};
  double f[2][5];
  hllc2n<2>(g, l, r, f);
  F1[0] = f[0][0]; F1[1] = f[0][1]; F1[2] = f[0][2]; F1[3] = f[0][3]; F1[4] = f[0][4];
  F2[0] = f[1][0]; F2[2] = f[1][1]; F2[3] = f[1][2]; F2[1] = f[1][3]; F2[4] = f[1][4];
}

// ---- S3'  LLF and HLLE (paper P:103 option list), rotated states (rho, u_normal, v, w, u_g) ----
// conserved state, physical flux and sound speed of one rotated primitive state
__device__ __forceinline__ void state_flux(const GasConst& g, const double W[5], double U[5], double F[5], double& c, double& p) {
  const double r = W[0], u = W[1], v = W[2], w = W[3], e = W[4];
  p = g.gm1 * e;
  const double E = fma(0.5 * r, fma(u, u, fma(v, v, w * w)), e);
  const double m = r * u;
  U[0] = r; U[1] = m; U[2] = r * v; U[3] = r * w; U[4] = E;
  F[0] = m; F[1] = fma(m, u, p); F[2] = m * v; F[3] = m * w; F[4] = (E + p) * u;
  c = sqrt_ratio(g.gamma * p, r);
}
// LLF (Rusanov): F = 1/2 [(F_L + F_R) - a (U_R - U_L)], a = max(|u_L| + c_L, |u_R| + c_R)
__device__ __forceinline__ void llf2(const GasConst& g, const double WL[5], const double WR[5], double F[5]) {
  double UL[5], UR[5], FL[5], FR[5], cL, cR, pL, pR;
  state_flux(g, WL, UL, FL, cL, pL);
  state_flux(g, WR, UR, FR, cR, pR);
  const double aL = fabs(WL[1]) + cL, aR = fabs(WR[1]) + cR;
  const double a = aL > aR ? aL : aR;
#pragma unroll
  for (int n = 0; n < 5; n++) F[n] = 0.5 * ((FL[n] + FR[n]) - a * (UR[n] - UL[n]));
}
// HLLE with Einfeldt's speeds from the Roe averages (weights sqrt(rho)), bounded by the L/R characteristic speeds
__device__ __forceinline__ void hlle2(const GasConst& g, const double WL[5], const double WR[5], double F[5]) {
  double UL[5], UR[5], FL[5], FR[5], cL, cR, pL, pR;
  state_flux(g, WL, UL, FL, cL, pL);
  state_flux(g, WR, UR, FR, cR, pR);
  const double sL = sqrt_ratio(WL[0], 1.0), sR = sqrt_ratio(WR[0], 1.0), isum = rcp2(sL + sR);
  const double HL = (UL[4] + pL) * rcp2(WL[0]), HR = (UR[4] + pR) * rcp2(WR[0]);
  const double ut = fma(sL, WL[1], sR * WR[1]) * isum, vt = fma(sL, WL[2], sR * WR[2]) * isum;
  const double wt = fma(sL, WL[3], sR * WR[3]) * isum, Ht = fma(sL, HL, sR * HR) * isum;
  const double ct = sqrt_ratio(g.gm1 * fma(-0.5, fma(ut, ut, fma(vt, vt, wt * wt)), Ht), 1.0);
  const double l1 = WL[1] - cL, l2 = ut - ct, r1 = WR[1] + cR, r2 = ut + ct;
  const double bm = min0(l1 < l2 ? l1 : l2), bp = max0(r1 > r2 ? r1 : r2);
  const double inv = rcp2(bp - bm), bb = bp * bm;
#pragma unroll
  for (int n = 0; n < 5; n++) F[n] = (fma(bp, FL[n], -(bm * FR[n])) + bb * (UR[n] - UL[n])) * inv;
}

// Roe's linearised solver (Toro 2013 ch.11; Q28): Roe averages as in hlle2, wave strengths from dU,
// F = 1/2 (F_L + F_R) - 1/2 sum_k a_k |l_k| K_k; no entropy fix
__device__ __forceinline__ void roe2(const GasConst& g, const double WL[5], const double WR[5], double F[5]) {
  double UL[5], UR[5], FL[5], FR[5], cL, cR, pL, pR;
  state_flux(g, WL, UL, FL, cL, pL);
  state_flux(g, WR, UR, FR, cR, pR);
  const double sL = sqrt_ratio(WL[0], 1.0), sR = sqrt_ratio(WR[0], 1.0), isum = rcp2(sL + sR);
  const double HL = (UL[4] + pL) * rcp2(WL[0]), HR = (UR[4] + pR) * rcp2(WR[0]);
  const double ut = fma(sL, WL[1], sR * WR[1]) * isum, vt = fma(sL, WL[2], sR * WR[2]) * isum;
  const double wt = fma(sL, WL[3], sR * WR[3]) * isum, Ht = fma(sL, HL, sR * HR) * isum;
  const double q2 = fma(ut, ut, fma(vt, vt, wt * wt));
  const double c2 = g.gm1 * fma(-0.5, q2, Ht), ct = sqrt_ratio(c2, 1.0), ic = rcp2(ct);
  double dU[5];
#pragma unroll
  for (int n = 0; n < 5; n++) dU[n] = UR[n] - UL[n];
  const double a3 = fma(-vt, dU[0], dU[2]), a4 = fma(-wt, dU[0], dU[3]);
  const double dU5 = fma(-a4, wt, fma(-a3, vt, dU[4]));
  const double a2 = (g.gm1 * (ic * ic)) * (fma(dU[0], fma(-ut, ut, Ht), ut * dU[1]) - dU5);
  const double a1 = (fma(dU[0], ut + ct, -dU[1]) - ct * a2) * (0.5 * ic);
  const double a5 = dU[0] - (a1 + a2);
  const double w1 = a1 * fabs(ut - ct), l2 = fabs(ut), w2 = a2 * l2, w3 = a3 * l2, w4 = a4 * l2, w5 = a5 * fabs(ut + ct);
  const double uc = ut * ct;
  F[0] = 0.5 * ((FL[0] + FR[0]) - (w1 + (w2 + w5)));
  F[1] = 0.5 * ((FL[1] + FR[1]) - fma(w1, ut - ct, fma(w2, ut, w5 * (ut + ct))));
  F[2] = 0.5 * ((FL[2] + FR[2]) - fma(w1 + (w2 + w5), vt, w3));
  F[3] = 0.5 * ((FL[3] + FR[3]) - fma(w1 + (w2 + w5), wt, w4));
  F[4] = 0.5 * ((FL[4] + FR[4]) - fma(w1, Ht - uc, fma(w2, 0.5 * q2, fma(w3, vt, fma(w4, wt, w5 * (Ht + uc))))));
}

// solver chosen at compile time: RS = 0 HLLC, 1 LLF, 2 HLLE, 3 Roe
template <int RS>
__device__ __forceinline__ void riemann2(const GasConst& g, const double l[5], const double r[5], double f[5]) {
  if constexpr (RS == 0) hllc2(g, l, r, f);
  else if constexpr (RS == 1) llf2(g, l, r, f);
  else if constexpr (RS == 2) hlle2(g, l, r, f);
  else roe2(g, l, r, f);
}
template <int RS, int D>
__device__ __forceinline__ void flux3(const GasConst& g, const double L[5], const double Rr[5], double F[5]) {
  if constexpr (RS == 0) { flux2<D>(g, L, Rr, F); return; }
  const double l[5] = {L[0], L[1 + D], L[1 + (D + 1) % 3], L[1 + (D + 2) % 3], L[4]};
  const double r[5] = {Rr[0], Rr[1 + D], Rr[1 + (D + 1) % 3], Rr[1 + (D + 2) % 3], Rr[4]};
  double f[5];
  riemann2<RS>(g, l, r, f);
  F[0] = f[0]; F[1 + D] = f[1]; F[1 + (D + 1) % 3] = f[2]; F[1 + (D + 2) % 3] = f[3]; F[4] = f[4];
}
template <int RS>
__device__ __forceinline__ void flux3_12(const GasConst& g, bool d2, const double L[5], const double Rr[5], double F[5]) {
  if constexpr (RS == 0) { flux2_12(g, d2, L, Rr, F); return; }
  const double l[5] = {L[0], d2 ? L[2] : L[1], d2 ? L[3] : L[2], d2 ? L[1] : L[3], L[4]};
  const double r[5] = {Rr[0], d2 ? Rr[2] : Rr[1], d2 ? Rr[3] : Rr[2], d2 ? Rr[1] : Rr[3], Rr[4]};
  double f[5];
  riemann2<RS>(g, l, r, f);
  F[0] = f[0];
  F[1] = d2 ? f[3] : f[1];
  F[2] = d2 ? f[1] : f[2];
  F[3] = d2 ? f[2] : f[3];
  F[4] = f[4];
}
template <int RS>
__device__ __forceinline__ void flux3_x1x2(const GasConst& g, const double L1[5], const double R1[5], const double L2[5],
                                           const double R2[5], double F1[5], double F2[5]) {
  if constexpr (RS == 0) { flux2_x1x2(g, L1, R1, L2, R2, F1, F2); return; }
  flux3<RS, 0>(g, L1, R1, F1);
  flux3<RS, 1>(g, L2, R2, F2);
}

}  // namespace ak

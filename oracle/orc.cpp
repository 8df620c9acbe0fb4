// orc.cpp -- CPU ORACLE (test infrastructure only; see orc.h for scope, citations and pins).
// Plain triple loops, fp64, compiled -O2 -ffp-contract=off -fno-fast-math so that every expression
// is evaluated exactly as written (no FMA contraction, no reassociation).
// Steps S0-S4 and G1-G4 are SURVEY.md section 8(c); P:NN = /root/reference/PAPER.md line NN.
#include "orc.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <string>
#include <tuple>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

static thread_local std::string g_err;
static int fail(const char* msg) { g_err = msg; return -1; }
extern "C" const char* orc_last_error(void) { return g_err.c_str(); }

static const double RHO_FLOOR = 1e-20;   // floors act on W only
static const double P_FLOOR   = 1e-20;

// ------------------------------------------------------------------------------------------------
// S1  conserved -> primitive, W = (rho, v, u_g)  (the primitive is the INTERNAL ENERGY)
// ------------------------------------------------------------------------------------------------
extern "C" void orc_c2p(double gamma, const double U[5], double W[5], int* floored) {
  int nfl = 0;
  double rho = U[0];
  if (!(rho >= RHO_FLOOR)) { rho = RHO_FLOOR; nfl++; }
  double rinv = 1.0 / rho;
  double m1 = U[1], m2 = U[2], m3 = U[3];
  double ug = U[4] - 0.5 * rinv * (m1 * m1 + (m2 * m2 + m3 * m3));
  double ug_floor = P_FLOOR / (gamma - 1.0);
  if (!(ug >= ug_floor)) { ug = ug_floor; nfl++; }
  W[0] = rho; W[1] = m1 * rinv; W[2] = m2 * rinv; W[3] = m3 * rinv; W[4] = ug;
  if (floored) *floored = nfl;
}

// ------------------------------------------------------------------------------------------------
// S2  reconstruction of one primitive along one direction
// ------------------------------------------------------------------------------------------------
// PLM with van Leer's harmonic-mean limiter: h = dL*dR/(dL+dR) if dL*dR > 0 else 0.
extern "C" void orc_plm(double qm1, double q0, double qp1, double* q_minus, double* q_plus) {
  double dL = q0 - qm1, dR = qp1 - q0;
  double prod = dL * dR;
  double h = (prod > 0.0) ? prod / (dL + dR) : 0.0;
  *q_minus = q0 - h;
  *q_plus  = q0 + h;
}

// PPM4 (i) fourth-order interface value at i+1/2 and (ii) clamp into the range of the two adjacent cells.
extern "C" void orc_ppm4_iface(double qm1, double q0, double qp1, double qp2, double* q_half) {
  double v = (7.0 * (q0 + qp1) - (qm1 + qp2)) / 12.0;
  double lo = std::fmin(q0, qp1), hi = std::fmax(q0, qp1);
  v = std::fmax(lo, std::fmin(v, hi));
  *q_half = v;
}

// PPM4 (iii) Colella & Woodward (1984) Eq.(1.10) monotonicity limiter for cell i given q[i-2..i+2].
extern "C" void orc_ppm4(const double q[5], double* q_minus, double* q_plus) {
  double aL, aR, a = q[2];
  orc_ppm4_iface(q[0], q[1], q[2], q[3], &aL);   // face i-1/2
  orc_ppm4_iface(q[1], q[2], q[3], q[4], &aR);   // face i+1/2
  if ((aR - a) * (a - aL) <= 0.0) {
    aL = a; aR = a;
  } else {
    double d = aR - aL;
    double mu = a - 0.5 * (aL + aR);
    double dmu = d * mu, d26 = d * d / 6.0;
    if (dmu > d26)        aL = 3.0 * a - 2.0 * aR;
    else if (-d26 > dmu)  aR = 3.0 * a - 2.0 * aL;
  }
  *q_minus = aL;
  *q_plus  = aR;
}

// ------------------------------------------------------------------------------------------------
// S2'  the higher-order reconstructions of the paper's option list ("PPM ... using extremum-preserving limiters
// (McCorquodale et al. 2015, hereafter PPMX), and the improved WENOZ scheme"; both converge at fourth order on
// the 1-D linear wave).  The paper defers the formulas; the readings are DESIGN.md Q29 (WENOZ) and Q30 (PPMX).
// Both take the five values q[i-2..i+2] of one primitive along one direction and return q- (at i-1/2) and q+ (at i+1/2).
// ------------------------------------------------------------------------------------------------
// WENO-Z (Borges et al. 2008) fifth-order value at the UPPER face of the middle cell from the stencil (a,b,c,d,e) =
// q[i-2..i+2]: candidate parabolas p_k, Jiang-Shu smoothness indicators beta_k, global indicator tau5 = |beta0 - beta2|,
// weights alpha_k = d_k (1 + (tau5 / (beta_k + eps))^2) with d = (1/10, 6/10, 3/10), eps = 1e-40.
static double wenoz_upper(double a, double b, double c, double d, double e) {
  // written in the differences of neighbouring cells, so that constant data are reproduced exactly (uniform states
  // must be preserved bit for bit): p_k = c + P_k / 6
  const double d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
  const double P0 = 5.0 * d2 - 2.0 * d1;          // (2a - 7b + 11c)/6 = c + P0/6
  const double P1 = 2.0 * d3 + d2;                // (-b + 5c + 2d)/6  = c + P1/6
  const double P2 = 4.0 * d3 - d4;                // (2c + 5d - e)/6   = c + P2/6
  const double s0 = d2 - d1, t0 = 3.0 * d2 - d1;  // a - 2b + c,  a - 4b + 3c
  const double s1 = d3 - d2, t1 = d2 + d3;        // b - 2c + d,  d - b
  const double s2 = d4 - d3, t2 = d4 - 3.0 * d3;  // c - 2d + e,  3c - 4d + e
  const double b0 = 13.0 / 12.0 * (s0 * s0) + 0.25 * (t0 * t0);
  const double b1 = 13.0 / 12.0 * (s1 * s1) + 0.25 * (t1 * t1);
  const double b2 = 13.0 / 12.0 * (s2 * s2) + 0.25 * (t2 * t2);
  const double eps = 1e-40;
  const double tau = std::fabs(b0 - b2);
  const double r0 = tau / (b0 + eps), r1 = tau / (b1 + eps), r2 = tau / (b2 + eps);
  const double a0 = 0.1 * (1.0 + r0 * r0), a1 = 0.6 * (1.0 + r1 * r1), a2 = 0.3 * (1.0 + r2 * r2);
  return c + (a0 * P0 + (a1 * P1 + a2 * P2)) / (6.0 * (a0 + (a1 + a2)));
}
extern "C" void orc_wenoz(const double q[5], double* q_minus, double* q_plus) {
  *q_plus  = wenoz_upper(q[0], q[1], q[2], q[3], q[4]);
  *q_minus = wenoz_upper(q[4], q[3], q[2], q[1], q[0]);    // the mirrored stencil: exact mirror symmetry
}

// PPMX: fourth-order interface values, the Colella-Sekora (2008) / McCorquodale-Colella (2011) limiters.
// (i) interface value between q0 and q1 from (qm1, q0, q1, q2): the fourth-order value; where it is not between q0 and
// q1 it is replaced by (q0 + q1)/2 - D/6 with D the second difference limited among the face-centred one
// 3 (q0 - 2 v + q1) and C times the two cell-centred ones (C = 5/4), zero unless all three share a sign.
static double ppmx_iface(double qm1, double q0, double q1, double q2) {
  const double C = 1.25;
  double v = (7.0 * (q0 + q1) - (qm1 + q2)) / 12.0;
  if ((v - q0) * (q1 - v) < 0.0) {
    const double dc = 3.0 * ((q0 + q1) - 2.0 * v);               // (groupings symmetric under mirroring)
    const double dl = (qm1 + q1) - 2.0 * q0, dr = (q0 + q2) - 2.0 * q1;
    double D = 0.0;
    if (dc > 0.0 && dl > 0.0 && dr > 0.0) D = std::fmin(dc, C * std::fmin(dl, dr));
    else if (dc < 0.0 && dl < 0.0 && dr < 0.0) D = -std::fmin(-dc, C * std::fmin(-dl, -dr));
    v = 0.5 * (q0 + q1) - D / 6.0;
  }
  return v;
}
// (ii) the parabola of cell i with edge values (aL, aR): at an extremum (of the parabola or of the cell averages) the
// parabola's second derivative 6 (aL + aR - 2a) is limited among itself and C times the three cell-centred second
// differences (zero unless all four share a sign) and both edge increments are scaled by the ratio -- a smooth
// extremum keeps its parabola, which is what PPM4's "flatten at every extremum" cannot do; elsewhere CW84's monotonicity
// constraint in the two-sided form (an edge increment at most twice the other).
extern "C" void orc_ppmx(const double q[5], double* q_minus, double* q_plus) {
  const double C = 1.25;
  const double a = q[2];
  double aL = ppmx_iface(q[0], q[1], q[2], q[3]);
  double aR = ppmx_iface(q[1], q[2], q[3], q[4]);
  const double dm = a - aL, dp = aR - a;
  if (dm * dp <= 0.0 || (q[3] - a) * (a - q[1]) <= 0.0) {
    const double df = 6.0 * ((aL + aR) - 2.0 * a);
    const double d1 = (q[0] + q[2]) - 2.0 * q[1], d2 = (q[1] + q[3]) - 2.0 * q[2], d3 = (q[2] + q[4]) - 2.0 * q[3];
    double D = 0.0;
    if (df > 0.0 && d1 > 0.0 && d2 > 0.0 && d3 > 0.0) D = std::fmin(df, C * std::fmin(d1, std::fmin(d2, d3)));
    else if (df < 0.0 && d1 < 0.0 && d2 < 0.0 && d3 < 0.0) D = -std::fmin(-df, C * std::fmin(-d1, std::fmin(-d2, -d3)));
    const double rho = (df != 0.0) ? D / df : 0.0;
    if (rho <= 1.0 - 1e-12) { aL = a - rho * dm; aR = a + rho * dp; }
  } else {
    if (std::fabs(dm) >= 2.0 * std::fabs(dp)) aL = a - 2.0 * dp;
    if (std::fabs(dp) >= 2.0 * std::fabs(dm)) aR = a + 2.0 * dm;
  }
  *q_minus = aL;
  *q_plus  = aR;
}

// ------------------------------------------------------------------------------------------------
// S3  HLLC flux at one face (P:103 names the solver; formulas: Toro 2013 ch.10, restated)
// Wave speeds (Q2, round-2 reading): Davis's direct estimates, Toro Eq.(10.48),
//   S_L = min(u_L - c_L, u_R - c_R),   S_R = max(u_L + c_L, u_R + c_R).
// They bound the speeds of an isolated shock (Lax condition) and of both rarefaction heads, satisfy
// S_L <= u_L - c_L and S_R >= u_R + c_R (Batten et al.'s condition for a positively conservative HLLC), and give
// S_L < S* < S_R for every pair of states with positive pressure, so the star flux is finite for head-on
// collisions at any Mach number (the pressure-based estimate of round 1 gave S_L > 0 > S_R and 0/0 there, Q26).
// ------------------------------------------------------------------------------------------------
extern "C" void orc_hllc(double gamma, int dir, const double WL[5], const double WR[5], double F[5]) {
  const int iu = 1 + dir, iv = 1 + (dir + 1) % 3, iw = 1 + (dir + 2) % 3;   // normal, transverse pair (cyclic)
  const double gm1 = gamma - 1.0;
  double rL = WL[0], uL = WL[iu], vL = WL[iv], wL = WL[iw], eL = WL[4];
  double rR = WR[0], uR = WR[iu], vR = WR[iv], wR = WR[iw], eR = WR[4];
  double pL = gm1 * eL, pR = gm1 * eR;
  double cL = std::sqrt(gamma * pL / rL), cR = std::sqrt(gamma * pR / rR);
  // min / max written as comparisons in this operand order so that a NaN sound speed (an unphysical reconstructed state:
  // negative pressure or density at the face) is NOT dropped the way fmin / fmax would drop it: a NaN c_L makes S_L NaN, a
  // NaN c_R makes S_R NaN, either makes S* and with it the whole flux NaN, and the cell is then caught by FOFC (Q31) or
  // reported by the time-step reduction.  For finite operands these are min and max.
  const double sl1 = uL - cL, sl2 = uR - cR, sr1 = uL + cL, sr2 = uR + cR;
  double SL = (sl2 < sl1) ? sl2 : sl1, SR = (sr1 > sr2) ? sr1 : sr2;
  double bm = std::fmin(SL, 0.0), bp = std::fmax(SR, 0.0);
  double mL = rL * (uL - SL), mR = rR * (SR - uR);
  double Ss = ((pL - pR) + (mL * uL + mR * uR)) / (mL + mR);                  // contact speed
  double psL = pL + rL * (SL - uL) * (Ss - uL);
  double psR = pR + rR * (SR - uR) * (Ss - uR);
  double ps = std::fmax(0.5 * (psL + psR), 0.0);
  double rK, uK, vK, wK, eK, pK, b;
  if (Ss >= 0.0) { rK = rL; uK = uL; vK = vL; wK = wL; eK = eL; pK = pL; b = bm; }
  else           { rK = rR; uK = uR; vK = vR; wK = wR; eK = eR; pK = pR; b = bp; }
  double EK = eK + 0.5 * rK * (uK * uK + (vK * vK + wK * wK));
  double UK[5] = { rK, rK * uK, rK * vK, rK * wK, EK };
  double FK[5] = { rK * uK, rK * uK * uK + pK, rK * uK * vK, rK * uK * wK, (EK + pK) * uK };
  double D[5]  = { 0.0, 1.0, 0.0, 0.0, Ss };
  double Fn[5];
  double den = Ss - b;
  for (int n = 0; n < 5; n++) Fn[n] = (Ss * (FK[n] - b * UK[n]) - b * ps * D[n]) / den;
  F[0] = Fn[0]; F[iu] = Fn[1]; F[iv] = Fn[2]; F[iw] = Fn[3]; F[4] = Fn[4];
}

// ------------------------------------------------------------------------------------------------
// S3'  the other two-state solvers of the paper's option list ("LLF ... HLLE, HLLC ...").
// Textbook forms (Toro 2013 ch.10), restated because the paper defers them:
//   LLF (Rusanov): F = 1/2 [(F_L + F_R) - a (U_R - U_L)],  a = max(|u_L| + c_L, |u_R| + c_R)
//   HLLE: F = [b+ F_L - b- F_R + b+ b- (U_R - U_L)] / (b+ - b-),  b- = min(S_L, 0), b+ = max(S_R, 0),
//         Einfeldt's speeds S_L = min(u_L - c_L, u~ - c~), S_R = max(u_R + c_R, u~ + c~) from the Roe averages
//         (weights sqrt(rho)):  u~, v~, w~, H~ = (E + p)/rho averaged,  c~^2 = (gamma - 1)(H~ - 1/2 |v~|^2)
// ------------------------------------------------------------------------------------------------
static void rotated_states(double gamma, int dir, const double W[5], double U[5], double Fx[5], double* c) {
  const int iu = 1 + dir, iv = 1 + (dir + 1) % 3, iw = 1 + (dir + 2) % 3;
  const double r = W[0], u = W[iu], v = W[iv], w = W[iw], e = W[4];
  const double p = (gamma - 1.0) * e;
  const double E = e + 0.5 * r * (u * u + (v * v + w * w));
  U[0] = r; U[1] = r * u; U[2] = r * v; U[3] = r * w; U[4] = E;
  Fx[0] = r * u; Fx[1] = r * u * u + p; Fx[2] = r * u * v; Fx[3] = r * u * w; Fx[4] = (E + p) * u;
  *c = std::sqrt(gamma * p / r);
}
static void unrotate(int dir, const double Fn[5], double F[5]) {
  const int iu = 1 + dir, iv = 1 + (dir + 1) % 3, iw = 1 + (dir + 2) % 3;
  F[0] = Fn[0]; F[iu] = Fn[1]; F[iv] = Fn[2]; F[iw] = Fn[3]; F[4] = Fn[4];
}

extern "C" void orc_llf(double gamma, int dir, const double WL[5], const double WR[5], double F[5]) {
  double UL[5], UR[5], FL[5], FR[5], cL, cR, Fn[5];
  rotated_states(gamma, dir, WL, UL, FL, &cL);
  rotated_states(gamma, dir, WR, UR, FR, &cR);
  const double a = std::fmax(std::fabs(WL[1 + dir]) + cL, std::fabs(WR[1 + dir]) + cR);
  for (int n = 0; n < 5; n++) Fn[n] = 0.5 * ((FL[n] + FR[n]) - a * (UR[n] - UL[n]));
  unrotate(dir, Fn, F);
}

extern "C" void orc_hlle(double gamma, int dir, const double WL[5], const double WR[5], double F[5]) {
  double UL[5], UR[5], FL[5], FR[5], cL, cR, Fn[5];
  rotated_states(gamma, dir, WL, UL, FL, &cL);
  rotated_states(gamma, dir, WR, UR, FR, &cR);
  const double gm1 = gamma - 1.0;
  const double sL = std::sqrt(WL[0]), sR = std::sqrt(WR[0]), isum = 1.0 / (sL + sR);
  // Roe averages; velocities from the rotated conserved states, enthalpy H = (E + p) / rho
  const double uL = UL[1] / UL[0], vL = UL[2] / UL[0], wL = UL[3] / UL[0];
  const double uR = UR[1] / UR[0], vR = UR[2] / UR[0], wR = UR[3] / UR[0];
  const double HL = (UL[4] + gm1 * WL[4]) / UL[0], HR = (UR[4] + gm1 * WR[4]) / UR[0];
  const double ut = (sL * uL + sR * uR) * isum, vt = (sL * vL + sR * vR) * isum, wt = (sL * wL + sR * wR) * isum;
  const double Ht = (sL * HL + sR * HR) * isum;
  const double ct = std::sqrt(gm1 * (Ht - 0.5 * (ut * ut + (vt * vt + wt * wt))));
  const double SL = std::fmin(uL - cL, ut - ct), SR = std::fmax(uR + cR, ut + ct);
  const double bm = std::fmin(SL, 0.0), bp = std::fmax(SR, 0.0);
  for (int n = 0; n < 5; n++) Fn[n] = ((bp * FL[n] - bm * FR[n]) + bp * bm * (UR[n] - UL[n])) / (bp - bm);
  unrotate(dir, Fn, F);
}

// Roe's linearised solver ("as well as Roe's linearized solver"; Toro 2013 ch.11, restated): Roe averages as for
// HLLE; eigenvalues l1 = u~ - c~, l2,3,4 = u~, l5 = u~ + c~; wave strengths from dU = U_R - U_L:
//   a3 = dU3 - v~ dU1,  a4 = dU4 - w~ dU1,  dU5' = dU5 - a3 v~ - a4 w~,
//   a2 = (gamma-1)/c~^2 [dU1 (H~ - u~^2) + u~ dU2 - dU5'],  a1 = [dU1 (u~ + c~) - dU2 - c~ a2] / (2 c~),  a5 = dU1 - (a1 + a2);
// right eigenvectors K1 = (1, u~-c~, v~, w~, H~-u~c~), K2 = (1, u~, v~, w~, |v~|^2/2), K3 = (0,0,1,0,v~), K4 = (0,0,0,1,w~),
// K5 = (1, u~+c~, v~, w~, H~+u~c~);  F = 1/2 (F_L + F_R) - 1/2 sum_k a_k |l_k| K_k.  No entropy fix, no fallback (Q28).
extern "C" void orc_roe(double gamma, int dir, const double WL[5], const double WR[5], double F[5]) {
  double UL[5], UR[5], FL[5], FR[5], cL, cR, Fn[5];
  rotated_states(gamma, dir, WL, UL, FL, &cL);
  rotated_states(gamma, dir, WR, UR, FR, &cR);
  const double gm1 = gamma - 1.0;
  const double sL = std::sqrt(WL[0]), sR = std::sqrt(WR[0]), isum = 1.0 / (sL + sR);
  const double uL = UL[1] / UL[0], vL = UL[2] / UL[0], wL = UL[3] / UL[0];
  const double uR = UR[1] / UR[0], vR = UR[2] / UR[0], wR = UR[3] / UR[0];
  const double HL = (UL[4] + gm1 * WL[4]) / UL[0], HR = (UR[4] + gm1 * WR[4]) / UR[0];
  const double ut = (sL * uL + sR * uR) * isum, vt = (sL * vL + sR * vR) * isum, wt = (sL * wL + sR * wR) * isum;
  const double Ht = (sL * HL + sR * HR) * isum;
  const double q2 = ut * ut + (vt * vt + wt * wt);
  const double c2 = gm1 * (Ht - 0.5 * q2), ct = std::sqrt(c2);
  double dU[5];
  for (int n = 0; n < 5; n++) dU[n] = UR[n] - UL[n];
  const double a3 = dU[2] - vt * dU[0], a4 = dU[3] - wt * dU[0];
  const double dU5 = dU[4] - a3 * vt - a4 * wt;
  const double a2 = gm1 / c2 * (dU[0] * (Ht - ut * ut) + ut * dU[1] - dU5);
  const double a1 = (dU[0] * (ut + ct) - dU[1] - ct * a2) / (2.0 * ct);
  const double a5 = dU[0] - (a1 + a2);
  const double l1 = std::fabs(ut - ct), l2 = std::fabs(ut), l5 = std::fabs(ut + ct);
  const double K1[5] = { 1.0, ut - ct, vt, wt, Ht - ut * ct }, K2[5] = { 1.0, ut, vt, wt, 0.5 * q2 };
  const double K3[5] = { 0.0, 0.0, 1.0, 0.0, vt }, K4[5] = { 0.0, 0.0, 0.0, 1.0, wt }, K5[5] = { 1.0, ut + ct, vt, wt, Ht + ut * ct };
  for (int n = 0; n < 5; n++) {
    const double diss = (a1 * l1) * K1[n] + ((a2 * l2) * K2[n] + ((a3 * l2) * K3[n] + ((a4 * l2) * K4[n] + (a5 * l5) * K5[n])));
    Fn[n] = 0.5 * ((FL[n] + FR[n]) - diss);
  }
  unrotate(dir, Fn, F);
}

// ------------------------------------------------------------------------------------------------
// Pack descriptor
// ------------------------------------------------------------------------------------------------
struct orc_pack {
  int nmb, nx[3], ng, nt[3];
  double gamma;
  int recon, rsolver;
  int nrb[3];
  double xmin[3], xmax[3];
  bool mesh_set = false, bound = false;
  std::vector<int> level, lx;            // lx[3*m+d]
  std::vector<char> blk_set;
  std::map<std::tuple<int, int, int, int>, int> leaf;   // (level, l1, l2, l3) -> m
  int max_level = 0;
  double* u[3] = { nullptr, nullptr, nullptr };   // A (U^n at the start of a step), B, and C (third register, RK3 only)
  int integrator = 2;                             // number of stages: 2 = SSPRK(2,2) (default), 3 = SSPRK(3,3) (f2)
  int cur = 0;
  long long floor_count = 0;
  int nthreads = 1;
  int bc[6] = { 0, 0, 0, 0, 0, 0 };      // per face x1min,x1max,...: 0 periodic, 1 outflow, 2 reflect
  bool flux_correction = false;          // SURVEY 8(f) f1, off by default (north_star's stage list omits it)
  bool fofc = false;                     // SURVEY 8(f) f2 / P:118: first-order flux correction, off by default
  long long fofc_count = 0;              // cells flagged since bind

  size_t ncell() const { return (size_t)nt[0] * nt[1] * nt[2]; }
  size_t idx(int m, int n, int k, int j, int i) const {
    return ((((size_t)m * 5 + n) * nt[2] + k) * nt[1] + j) * nt[0] + i;
  }
  double dx(int lev, int d) const { return (xmax[d] - xmin[d]) / ((double)nrb[d] * nx[d] * (double)(1 << lev)); }
  long nglob(int lev, int d) const { return (long)nrb[d] * nx[d] * (1L << lev); }
  int find_leaf(int lev, long b1, long b2, long b3) const {
    auto it = leaf.find(std::make_tuple(lev, (int)b1, (int)b2, (int)b3));
    return it == leaf.end() ? -1 : it->second;
  }
};

extern "C" orc_pack* orc_pack_create(int nmb, int nx1, int nx2, int nx3, int ng, double gamma, int recon, int rsolver) {
  int nx[3] = { nx1, nx2, nx3 };
  if (nmb < 1) { fail("nmb < 1"); return nullptr; }
  for (int d = 0; d < 3; d++) if (nx[d] < ng || (nx[d] & 1)) { fail("nx_d must be even and >= ng"); return nullptr; }
  if (!(gamma > 1.0)) { fail("gamma <= 1"); return nullptr; }
  if (recon < 0 || recon > 3) { fail("unknown recon"); return nullptr; }
  if (rsolver < 0 || rsolver > 3) { fail("unknown rsolver"); return nullptr; }
  if ((recon == 0 && ng < 2) || (recon >= 1 && ng < 3)) { fail("ng too small for the reconstruction"); return nullptr; }
  orc_pack* p = new orc_pack;
  p->nmb = nmb; p->ng = ng; p->gamma = gamma; p->recon = recon; p->rsolver = rsolver;
  for (int d = 0; d < 3; d++) { p->nx[d] = nx[d]; p->nt[d] = nx[d] + 2 * ng; }
  p->level.assign(nmb, 0); p->lx.assign(3 * (size_t)nmb, 0); p->blk_set.assign(nmb, 0);
  return p;
}

extern "C" int orc_pack_set_mesh(orc_pack* p, int nrb1, int nrb2, int nrb3,
                                 double x1min, double x1max, double x2min, double x2max, double x3min, double x3max) {
  if (!p) return fail("null pack");
  if (nrb1 < 1 || nrb2 < 1 || nrb3 < 1) return fail("nrb < 1");
  if (!(x1max > x1min) || !(x2max > x2min) || !(x3max > x3min)) return fail("empty domain");
  p->nrb[0] = nrb1; p->nrb[1] = nrb2; p->nrb[2] = nrb3;
  p->xmin[0] = x1min; p->xmax[0] = x1max; p->xmin[1] = x2min; p->xmax[1] = x2max; p->xmin[2] = x3min; p->xmax[2] = x3max;
  p->mesh_set = true;
  return 0;
}

extern "C" int orc_pack_set_block(orc_pack* p, int m, int level, int lx1, int lx2, int lx3) {
  if (!p) return fail("null pack");
  if (!p->mesh_set) return fail("set_mesh first");
  if (m < 0 || m >= p->nmb) return fail("block index out of range");
  if (level < 0 || level > 1) return fail("level must be 0 or 1");
  int l[3] = { lx1, lx2, lx3 };
  for (int d = 0; d < 3; d++) if (l[d] < 0 || l[d] >= p->nrb[d] * (1 << level)) return fail("logical location out of range");
  p->level[m] = level;
  for (int d = 0; d < 3; d++) p->lx[3 * (size_t)m + d] = l[d];
  p->blk_set[m] = 1;
  return 0;
}

extern "C" int orc_pack_bind(orc_pack* p, double* u_a, double* u_b) {
  if (!p) return fail("null pack");
  if (!p->mesh_set) return fail("set_mesh first");
  if (!u_a || !u_b) return fail("null buffer");
  p->leaf.clear(); p->max_level = 0;
  double vol = 0.0;
  for (int m = 0; m < p->nmb; m++) {
    if (!p->blk_set[m]) return fail("block not set");
    auto key = std::make_tuple(p->level[m], p->lx[3 * m], p->lx[3 * m + 1], p->lx[3 * m + 2]);
    if (p->leaf.count(key)) return fail("duplicate block");
    p->leaf[key] = m;
    if (p->level[m] > p->max_level) p->max_level = p->level[m];
    vol += (p->level[m] == 0) ? 1.0 : 0.125;
  }
  // leaves must tile the root grid: no level-1 leaf under a level-0 leaf, total volume = root blocks
  for (int m = 0; m < p->nmb; m++) if (p->level[m] == 1) {
    if (p->find_leaf(0, p->lx[3 * m] / 2, p->lx[3 * m + 1] / 2, p->lx[3 * m + 2] / 2) >= 0) return fail("overlapping leaves");
  }
  if (vol != (double)p->nrb[0] * p->nrb[1] * p->nrb[2]) return fail("leaves do not cover the domain");
  if (p->max_level > 0 && (p->ng & 1)) return fail("static refinement needs even ng");
  for (int f = 0; f < 6; f++) if (p->bc[f] != 0 && p->max_level > 0) return fail("physical boundaries need a single-level mesh");
  p->u[0] = u_a; p->u[1] = u_b; p->cur = 0; p->bound = true; p->floor_count = 0; p->fofc_count = 0;
  return 0;
}

extern "C" int orc_set_threads(orc_pack* p, int n) { if (!p || n < 1) return fail("bad thread count"); p->nthreads = n; return 0; }
extern "C" int orc_pack_set_boundaries(orc_pack* p, const int bc[6]) {
  if (!p || !bc) return fail("null argument");
  for (int f = 0; f < 6; f++) if (bc[f] < 0 || bc[f] > 2) return fail("unknown boundary condition");
  for (int d = 0; d < 3; d++) if ((bc[2 * d] == 0) != (bc[2 * d + 1] == 0)) return fail("periodic faces come in pairs");
  for (int f = 0; f < 6; f++) p->bc[f] = bc[f];
  p->bound = false;
  return 0;
}
extern "C" int orc_set_integrator(orc_pack* p, int nstages, double* u_c) {
  if (!p) return fail("null pack");
  if (nstages < 1 || nstages > 3) return fail("integrator must be 1 (forward Euler), 2 (SSPRK(2,2)) or 3 (SSPRK(3,3))");
  if (nstages == 3 && !u_c) return fail("SSPRK(3,3) needs a third state buffer");
  if (p->bound && p->cur != 0 && !(p->integrator == 1 && p->cur == 1)) return fail("change the integrator between steps");
  if (p->bound && p->cur == 1 && nstages != 1) return fail("after an odd number of forward-Euler steps U^n is in buffer B: take one more or reload");
  p->integrator = nstages; p->u[2] = u_c;
  return 0;
}
extern "C" int orc_set_flux_correction(orc_pack* p, int on) { if (!p) return fail("null pack"); p->flux_correction = on != 0; return 0; }
extern "C" int orc_set_fofc(orc_pack* p, int on) { if (!p) return fail("null pack"); p->fofc = on != 0; return 0; }
extern "C" long long orc_pack_fofc_count(const orc_pack* p) { return p ? p->fofc_count : -1; }
extern "C" double* orc_pack_current(orc_pack* p) { return (p && p->bound) ? p->u[p->cur] : nullptr; }
extern "C" long long orc_pack_floor_count(const orc_pack* p) { return p ? p->floor_count : -1; }
extern "C" int orc_pack_destroy(orc_pack* p) { delete p; return 0; }

// ------------------------------------------------------------------------------------------------
// G1-G4  ghost fill: a pure function of the ACTIVE cells of leaf blocks
// ------------------------------------------------------------------------------------------------
static inline long wrapl(long g, long n) { long r = g % n; return r < 0 ? r + n : r; }

// value of variable n in the active cell with level-`lev` global index G[] (already wrapped) of leaf m
static inline double leaf_cell(const orc_pack* p, const double* U, int m, int n, const long G[3]) {
  int a[3];
  for (int d = 0; d < 3; d++) a[d] = (int)(G[d] - (long)p->lx[3 * (size_t)m + d] * p->nx[d]) + p->ng;
  return U[p->idx(m, n, a[2], a[1], a[0])];
}

// G3: mean of the 8 level-(lev+1) active cells covering the level-`lev` cell G, fixed summation order
static bool restrict_cell(const orc_pack* p, const double* U, int lev, const long G[3], int n, double* out) {
  double f[2][2][2];
  for (int dk = 0; dk < 2; dk++) for (int dj = 0; dj < 2; dj++) for (int di = 0; di < 2; di++) {
    long Gf[3] = { 2 * G[0] + di, 2 * G[1] + dj, 2 * G[2] + dk };
    int m = p->find_leaf(lev + 1, Gf[0] / p->nx[0], Gf[1] / p->nx[1], Gf[2] / p->nx[2]);
    if (m < 0) return false;
    f[dk][dj][di] = leaf_cell(p, U, m, n, Gf);
  }
  *out = 0.125 * (((f[0][0][0] + f[0][0][1]) + (f[0][1][0] + f[0][1][1])) +
                  ((f[1][0][0] + f[1][0][1]) + (f[1][1][0] + f[1][1][1])));
  return true;
}

// virtual level-`lev` field C(.): the leaf value where a level-`lev` leaf covers G, else the G3 restriction
static bool coarse_field(const orc_pack* p, const double* U, int lev, const long Gin[3], int n, double* out) {
  long G[3];
  for (int d = 0; d < 3; d++) G[d] = wrapl(Gin[d], p->nglob(lev, d));
  int m = p->find_leaf(lev, G[0] / p->nx[0], G[1] / p->nx[1], G[2] / p->nx[2]);
  if (m >= 0) { *out = leaf_cell(p, U, m, n, G); return true; }
  return restrict_cell(p, U, lev, G, n, out);
}

static inline double minmod(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  double m = std::fmin(std::fabs(a), std::fabs(b));
  return a > 0.0 ? m : -m;
}

static int fill_block(const orc_pack* p, double* U, int m) {
  const int ng = p->ng, lev = p->level[m];
  for (int k = 0; k < p->nt[2]; k++) for (int j = 0; j < p->nt[1]; j++) for (int i = 0; i < p->nt[0]; i++) {
    int a[3] = { i - ng, j - ng, k - ng };
    bool ghost = false;
    for (int d = 0; d < 3; d++) if (a[d] < 0 || a[d] >= p->nx[d]) ghost = true;
    if (!ghost) continue;
    // position of the cell's image inside the domain: periodic wrap, or -- SURVEY 8(f) f3, the paper's
    // outflow / reflecting boundary functions -- the nearest active cell (outflow: zero gradient) or the mirror
    // image across the boundary face with the normal momentum negated (reflect)
    long G[3];
    double sgn[5] = { 1.0, 1.0, 1.0, 1.0, 1.0 };
    for (int d = 0; d < 3; d++) {
      const long N = p->nglob(lev, d);
      long g = (long)p->lx[3 * (size_t)m + d] * p->nx[d] + a[d];
      if (g >= 0 && g < N) { G[d] = g; continue; }
      const int kind = p->bc[2 * d + (g < 0 ? 0 : 1)];
      if (kind == 0) G[d] = wrapl(g, N);
      else if (kind == 1) G[d] = g < 0 ? 0 : N - 1;
      else { G[d] = g < 0 ? -1 - g : 2 * N - 1 - g; sgn[1 + d] = -sgn[1 + d]; }
    }
    // G1: which leaf covers this position?
    int src = p->find_leaf(lev, G[0] / p->nx[0], G[1] / p->nx[1], G[2] / p->nx[2]);
    for (int n = 0; n < 5; n++) {
      double val;
      if (src >= 0) {                                     // G2 same level: copy
        val = leaf_cell(p, U, src, n, G);
      } else if (restrict_cell(p, U, lev, G, n, &val)) {  // G3 finer neighbour: conservative restriction
      } else {                                            // G4 coarser neighbour: limited-linear prolongation
        if (lev == 0) return -1;
        long Gc[3]; int s[3];
        for (int d = 0; d < 3; d++) { Gc[d] = G[d] >> 1; s[d] = 2 * (int)(G[d] & 1) - 1; }
        double c0;
        if (!coarse_field(p, U, lev - 1, Gc, n, &c0)) return -1;
        double g[3];
        for (int d = 0; d < 3; d++) {
          long Gm[3] = { Gc[0], Gc[1], Gc[2] }, Gp[3] = { Gc[0], Gc[1], Gc[2] };
          Gm[d] -= 1; Gp[d] += 1;
          double cm, cp;
          if (!coarse_field(p, U, lev - 1, Gm, n, &cm)) return -1;
          if (!coarse_field(p, U, lev - 1, Gp, n, &cp)) return -1;
          g[d] = 0.25 * minmod(c0 - cm, cp - c0);
        }
        val = ((c0 + s[0] * g[0]) + s[1] * g[1]) + s[2] * g[2];
      }
      U[p->idx(m, n, k, j, i)] = sgn[n] * val;
    }
  }
  return 0;
}

extern "C" int orc_fill_ghosts(orc_pack* p) {
  if (!p || !p->bound) return fail("pack not bound");
  double* U = p->u[p->cur];
  int bad = 0;
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) reduction(+ : bad) if (p->nthreads > 1)
  for (int m = 0; m < p->nmb; m++) if (fill_block(p, U, m) != 0) bad++;
  return bad ? fail("ghost cell with no covering leaf") : 0;
}

// ------------------------------------------------------------------------------------------------
// S1-S4  one Runge-Kutta stage (P:99 reconstruct-solve-advance; P:105 SSP-RK2 in two registers)
// ------------------------------------------------------------------------------------------------
// F[d][n*ncell + c]: flux of direction d at the LOWER d-face of cell c
struct FaceFlux {
  std::vector<double> v[3];
  std::vector<double>& operator[](int d) { return v[d]; }
  const std::vector<double>& operator[](int d) const { return v[d]; }
};

// S1-S3 for block m: primitives, reconstruction and the Riemann flux at every face of the active region
static long long block_fluxes(const orc_pack* p, const double* Uin, int m, FaceFlux& F) {
  const int ng = p->ng, n1 = p->nt[0], n2 = p->nt[1], n3 = p->nt[2];
  const size_t nc = p->ncell();
  long long nfl = 0;
  // S1: primitives in every cell of the block, ghosts included
  std::vector<double> W(5 * nc);
  for (int k = 0; k < n3; k++) for (int j = 0; j < n2; j++) for (int i = 0; i < n1; i++) {
    double u[5], w[5]; int f;
    for (int n = 0; n < 5; n++) u[n] = Uin[p->idx(m, n, k, j, i)];
    orc_c2p(p->gamma, u, w, &f);
    nfl += f;
    size_t c = ((size_t)k * n2 + j) * n1 + i;
    for (int n = 0; n < 5; n++) W[n * nc + c] = w[n];
  }
  // S2 + S3: flux of direction d at the lower face of cell (k,j,i), stored at that cell's index
  const int str[3] = { 1, n1, n1 * n2 };
  for (int d = 0; d < 3; d++) {
    F[d].assign(5 * nc, 0.0);
    int hi[3] = { p->nx[0] + ng, p->nx[1] + ng, p->nx[2] + ng };
    hi[d] += 1;                                            // faces ng .. nx+ng along d
    for (int k = ng; k < hi[2]; k++) for (int j = ng; j < hi[1]; j++) for (int i = ng; i < hi[0]; i++) {
      size_t c = ((size_t)k * n2 + j) * n1 + i;            // cell on the + side of the face
      size_t cm = c - str[d];                              // cell on the - side
      double WL[5], WR[5], Fl[5];
      for (int n = 0; n < 5; n++) {
        const double* q = &W[n * nc];
        double qm, qp;
        if (p->recon == 0) {
          orc_plm(q[cm - str[d]], q[cm], q[cm + str[d]], &qm, &qp);          WL[n] = qp;   // q+ of cell i-1
          orc_plm(q[c - str[d]],  q[c],  q[c + str[d]],  &qm, &qp);          WR[n] = qm;   // q- of cell i
        } else {
          double sL[5] = { q[cm - 2 * str[d]], q[cm - str[d]], q[cm], q[cm + str[d]], q[cm + 2 * str[d]] };
          double sR[5] = { q[c - 2 * str[d]],  q[c - str[d]],  q[c],  q[c + str[d]],  q[c + 2 * str[d]] };
          if (p->recon == 1)      { orc_ppm4(sL, &qm, &qp);  WL[n] = qp;  orc_ppm4(sR, &qm, &qp);  WR[n] = qm; }
          else if (p->recon == 2) { orc_ppmx(sL, &qm, &qp);  WL[n] = qp;  orc_ppmx(sR, &qm, &qp);  WR[n] = qm; }
          else                    { orc_wenoz(sL, &qm, &qp); WL[n] = qp;  orc_wenoz(sR, &qm, &qp); WR[n] = qm; }
        }
      }
      if (p->rsolver == 0) orc_hllc(p->gamma, d, WL, WR, Fl);
      else if (p->rsolver == 1) orc_llf(p->gamma, d, WL, WR, Fl);
      else if (p->rsolver == 2) orc_hlle(p->gamma, d, WL, WR, Fl);
      else orc_roe(p->gamma, d, WL, WR, Fl);
      for (int n = 0; n < 5; n++) F[d][n * nc + c] = Fl[n];
    }
  }
  return nfl;
}

// S4 for block m: weighted update of the active cells, evaluated left to right
static void block_update(const orc_pack* p, const double* Uin, const double* U0, double* Uout, int m, const FaceFlux& F,
                         double g0, double g1, double beta, double dt) {
  const int ng = p->ng, n1 = p->nt[0], n2 = p->nt[1];
  const size_t nc = p->ncell();
  const int str[3] = { 1, n1, n1 * n2 };
  const int lev = p->level[m];
  const double c1 = beta * dt / p->dx(lev, 0), c2 = beta * dt / p->dx(lev, 1), c3 = beta * dt / p->dx(lev, 2);
  for (int n = 0; n < 5; n++)
    for (int k = ng; k < p->nx[2] + ng; k++) for (int j = ng; j < p->nx[1] + ng; j++) for (int i = ng; i < p->nx[0] + ng; i++) {
      size_t c = ((size_t)k * n2 + j) * n1 + i;
      size_t g = p->idx(m, n, k, j, i);
      double v = g0 * Uin[g] + g1 * U0[g];
      v = v - c1 * (F[0][n * nc + c + str[0]] - F[0][n * nc + c]);
      v = v - c2 * (F[1][n * nc + c + str[1]] - F[1][n * nc + c]);
      v = v - c3 * (F[2][n * nc + c + str[2]] - F[2][n * nc + c]);
      Uout[g] = v;
    }
}

// f1 ("flux correction"): at a face between a level-0 block and level-1 blocks the coarse
// block's flux is replaced by the mean of the four fine-block fluxes through the same area (equal areas),
// summed in a fixed order, so that what leaves the fine cells is exactly what enters the coarse cell.
static void correct_coarse_fluxes(const orc_pack* p, std::vector<FaceFlux>& F) {
  const int ng = p->ng;
  const size_t nc = p->ncell();
  const int n1 = p->nt[0], n2 = p->nt[1];
  for (int m = 0; m < p->nmb; m++) {
    if (p->level[m] != 0) continue;
    for (int d = 0; d < 3; d++) for (int side = 0; side < 2; side++) {
      long nb[3] = { p->lx[3 * (size_t)m], p->lx[3 * (size_t)m + 1], p->lx[3 * (size_t)m + 2] };
      nb[d] = wrapl(nb[d] + (side ? 1 : -1), p->nrb[d]);
      if (p->find_leaf(0, nb[0], nb[1], nb[2]) >= 0) continue;           // same-level neighbour: nothing to do
      const int t1 = (d == 0) ? 1 : 0, t2 = (d == 2) ? 1 : 2;             // tangential directions, t1 faster
      for (int b = 0; b < p->nx[t2]; b++) for (int a = 0; a < p->nx[t1]; a++) {
        int cc[3];                                                        // coarse cell on the + side of the face
        cc[d] = side ? p->nx[d] + ng : ng; cc[t1] = a + ng; cc[t2] = b + ng;
        const size_t c = ((size_t)cc[2] * n2 + cc[1]) * n1 + cc[0];
        // level-1 global index of the fine cell that stores the fine face: the cell on the + side of the face
        long Gc[3];
        for (int e = 0; e < 3; e++) Gc[e] = (long)p->lx[3 * (size_t)m + e] * p->nx[e] + (cc[e] - ng);
        double f[2][2][5];
        for (int s2 = 0; s2 < 2; s2++) for (int s1 = 0; s1 < 2; s1++) {
          long Gf[3];
          Gf[d] = 2 * Gc[d]; Gf[t1] = 2 * Gc[t1] + s1; Gf[t2] = 2 * Gc[t2] + s2;
          // upper coarse face: the fine cell on the + side is active in the fine neighbour (its lower boundary
          // face); lower coarse face: the fine face is the UPPER boundary face of the fine neighbour on the - side,
          // stored at that block's first upper ghost index
          long Gown[3] = { Gf[0], Gf[1], Gf[2] };
          if (!side) Gown[d] = Gf[d] - 1;                                 // an active cell of the fine neighbour
          for (int e = 0; e < 3; e++) Gown[e] = wrapl(Gown[e], p->nglob(1, e));
          const int mf = p->find_leaf(1, Gown[0] / p->nx[0], Gown[1] / p->nx[1], Gown[2] / p->nx[2]);
          int cf[3];
          for (int e = 0; e < 3; e++) cf[e] = (int)(Gown[e] - (long)p->lx[3 * (size_t)mf + e] * p->nx[e]) + ng;
          if (!side) cf[d] += 1;                                          // = nx[d] + ng
          const size_t cfi = ((size_t)cf[2] * n2 + cf[1]) * n1 + cf[0];
          for (int n = 0; n < 5; n++) f[s2][s1][n] = F[mf][d][n * nc + cfi];
        }
        for (int n = 0; n < 5; n++)
          F[m][d][n * nc + c] = 0.25 * ((f[0][0][n] + f[0][1][n]) + (f[1][0][n] + f[1][1][n]));
      }
    }
  }
}

// f2 / P:118 first-order flux correction (FOFC): "if the density or pressure in any cell were to go negative, the fluxes
// on all faces of that cell are recalculated using first-order (piecewise constant) reconstruction and a diffusive
// LLF Riemann solver".  Reading (Q31): a cell is flagged when the stage's tentative result has rho <= 0 or
// E - |m|^2/(2 rho) <= 0 (NaN included); the flags are copied into the ghost cells like the state (same-level copies
// and boundary images), so both blocks that share a face see the same pair of flags; every face with a flagged cell
// on either side takes F = LLF(W_lower, W_upper) of the two CELL-CENTRED primitive states of U_in; then the update is
// evaluated again.  Single-level meshes (the ordering against f1 that P:118 prescribes is then moot).
static long long fofc_replace_fluxes(const orc_pack* p, const double* Uin, const double* Utent, std::vector<FaceFlux>& F) {
  const int ng = p->ng, n1 = p->nt[0], n2 = p->nt[1], n3 = p->nt[2];
  const size_t nc = p->ncell();
  // flags live in variable 0 of a state-shaped scratch array so that the ghost fill of the state can be reused as it is
  std::vector<double> flag((size_t)p->nmb * 5 * nc, 0.0);
  long long nflag = 0;
  for (int m = 0; m < p->nmb; m++)
    for (int k = ng; k < p->nx[2] + ng; k++) for (int j = ng; j < p->nx[1] + ng; j++) for (int i = ng; i < p->nx[0] + ng; i++) {
      const double rho = Utent[p->idx(m, 0, k, j, i)];
      const double m1 = Utent[p->idx(m, 1, k, j, i)], m2 = Utent[p->idx(m, 2, k, j, i)], m3 = Utent[p->idx(m, 3, k, j, i)];
      const double eint = Utent[p->idx(m, 4, k, j, i)] - 0.5 * (m1 * m1 + (m2 * m2 + m3 * m3)) / rho;
      if (!(rho > 0.0) || !(eint > 0.0)) { flag[p->idx(m, 0, k, j, i)] = 1.0; nflag++; }
    }
  if (nflag == 0) return 0;
  for (int m = 0; m < p->nmb; m++) fill_block(p, flag.data(), m);
  const int str[3] = { 1, n1, n1 * n2 };
  for (int m = 0; m < p->nmb; m++)
    for (int d = 0; d < 3; d++) {
      int hi[3] = { p->nx[0] + ng, p->nx[1] + ng, p->nx[2] + ng };
      hi[d] += 1;
      for (int k = ng; k < hi[2]; k++) for (int j = ng; j < hi[1]; j++) for (int i = ng; i < hi[0]; i++) {
        const size_t c = ((size_t)k * n2 + j) * n1 + i, cm = c - str[d];
        const size_t base = (size_t)m * 5 * nc;
        if (flag[base + c] == 0.0 && flag[base + cm] == 0.0) continue;
        double uL[5], uR[5], WL[5], WR[5], Fl[5];
        for (int n = 0; n < 5; n++) { uL[n] = Uin[base + n * nc + cm]; uR[n] = Uin[base + n * nc + c]; }
        orc_c2p(p->gamma, uL, WL, nullptr);
        orc_c2p(p->gamma, uR, WR, nullptr);
        orc_llf(p->gamma, d, WL, WR, Fl);
        for (int n = 0; n < 5; n++) F[m][d][n * nc + c] = Fl[n];
      }
    }
  (void)n3;
  return nflag;
}

extern "C" int orc_hydro_stage(orc_pack* p, int stage, double dt) {
  if (!p || !p->bound) return fail("pack not bound");
  if (stage < 1 || stage > p->integrator) return fail("stage out of range for the integrator");
  if (p->integrator == 1) {
    // RK1 (forward Euler, "RK1 through RK4"): U^{n+1} = U^n + dt L(U^n); the two registers alternate
    if (p->cur > 1) return fail("forward Euler alternates between buffers A and B");
  } else if (p->cur != stage - 1) return fail("stages must be called in order, starting from U^n in buffer A");
  // Shu-Osher forms (P:105 names the family; coefficients: SURVEY Q1 and, for three stages, Q27), every
  // stage  U_out = g0 U_in + g1 U^n + beta dt L(U_in):
  //   SSPRK(2,2): U1 = U^n + dt L(U^n);  U^{n+1} = 1/2 U^n + 1/2 [U1 + dt L(U1)]
  //   SSPRK(3,3): U1 = U^n + dt L(U^n);  U2 = 3/4 U^n + 1/4 [U1 + dt L(U1)];  U^{n+1} = 1/3 U^n + 2/3 [U2 + dt L(U2)]
  static const double C2[2][3] = { { 0.0, 1.0, 1.0 }, { 0.5, 0.5, 0.5 } };
  static const double C3[3][3] = { { 0.0, 1.0, 1.0 }, { 0.25, 0.75, 0.25 }, { 2.0 / 3.0, 1.0 / 3.0, 2.0 / 3.0 } };
  const double* cf = (p->integrator == 2) ? C2[stage - 1] : C3[stage - 1];
  const double g0 = cf[0], g1 = cf[1], beta = cf[2];
  const double* Uin = p->u[p->cur];
  const double* U0 = (p->integrator == 1) ? Uin : p->u[0];
  // the last stage writes A in place (each cell's A value is read only for itself); the others write the next buffer;
  // forward Euler has no second register to combine with and writes the other buffer
  const int out = (p->integrator == 1) ? 1 - p->cur : ((stage == p->integrator) ? 0 : stage);
  double* Uout = p->u[out];
  long long nfl = 0;
  if (p->fofc) {
    if (p->max_level > 0) return fail("FOFC is implemented on single-level meshes");
    // high-order fluxes of all blocks, the tentative update into a scratch copy, flags, replaced fluxes, final update
    std::vector<FaceFlux> F(p->nmb);
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) reduction(+ : nfl) if (p->nthreads > 1)
    for (int m = 0; m < p->nmb; m++) nfl += block_fluxes(p, Uin, m, F[m]);
    std::vector<double> tent((size_t)p->nmb * 5 * p->ncell(), 0.0);
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) if (p->nthreads > 1)
    for (int m = 0; m < p->nmb; m++) block_update(p, Uin, U0, tent.data(), m, F[m], g0, g1, beta, dt);
    p->fofc_count += fofc_replace_fluxes(p, Uin, tent.data(), F);
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) if (p->nthreads > 1)
    for (int m = 0; m < p->nmb; m++) block_update(p, Uin, U0, Uout, m, F[m], g0, g1, beta, dt);
  } else if (p->flux_correction && p->max_level > 0) {
    // all fluxes first, then the coarse faces at level boundaries are replaced, then every block is advanced
    std::vector<FaceFlux> F(p->nmb);
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) reduction(+ : nfl) if (p->nthreads > 1)
    for (int m = 0; m < p->nmb; m++) nfl += block_fluxes(p, Uin, m, F[m]);
    correct_coarse_fluxes(p, F);
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) if (p->nthreads > 1)
    for (int m = 0; m < p->nmb; m++) block_update(p, Uin, U0, Uout, m, F[m], g0, g1, beta, dt);
  } else {
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) reduction(+ : nfl) if (p->nthreads > 1)
    for (int m = 0; m < p->nmb; m++) {
      FaceFlux F;
      nfl += block_fluxes(p, Uin, m, F);
      block_update(p, Uin, U0, Uout, m, F, g0, g1, beta, dt);
    }
  }
  p->floor_count += nfl;
  p->cur = out;
  return 0;
}

// ------------------------------------------------------------------------------------------------
// S0  CFL time step, Eq.(3): min over active cells of leaf blocks and over directions
// ------------------------------------------------------------------------------------------------
extern "C" int orc_new_dt(orc_pack* p, double cfl, double* dt_out) {
  if (!p || !p->bound || !dt_out) return fail("pack not bound");
  const double* U = p->u[p->cur];
  const int ng = p->ng;
  double dtmin = HUGE_VAL;
  long long bad = 0;      // cells whose signal speed is not a finite positive number (NaN / inf state): reported, not skipped
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) reduction(min : dtmin) reduction(+ : bad) if (p->nthreads > 1)
  for (int m = 0; m < p->nmb; m++) {
    const int lev = p->level[m];
    for (int k = ng; k < p->nx[2] + ng; k++) for (int j = ng; j < p->nx[1] + ng; j++) for (int i = ng; i < p->nx[0] + ng; i++) {
      double u[5], w[5];
      for (int n = 0; n < 5; n++) u[n] = U[p->idx(m, n, k, j, i)];
      orc_c2p(p->gamma, u, w, nullptr);
      double pr = (p->gamma - 1.0) * w[4];
      double cs = std::sqrt(p->gamma * pr / w[0]);
      for (int d = 0; d < 3; d++) {
        double s = std::fabs(w[1 + d]) + cs;
        if (!(s > 0.0 && s < HUGE_VAL)) { bad++; continue; }
        double cand = p->dx(lev, d) / s;
        if (cand < dtmin) dtmin = cand;
      }
    }
  }
  if (bad) return fail("non-finite signal speed in the state (NaN or inf)");
  *dt_out = cfl * dtmin;
  return 0;
}

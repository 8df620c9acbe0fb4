// orc_mhd.cpp -- CPU ORACLE for the MHD + constrained-transport stage (test infrastructure only; see orc_mhd.h for scope,
// citations and pins).  Plain loops, fp64, compiled -O2 -ffp-contract=off -fno-fast-math.  P:NN = /root/reference/PAPER.md
// line NN; Qnn = readings listed in DESIGN.md.
#include "orc_mhd.h"
#include "orc.h"       // orc_ppm4, orc_ppmx, orc_wenoz: the hydro oracle's reconstruction functions (same oracle, linked in)

#include <cmath>
#include <cstdio>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

static thread_local std::string g_err;
static int fail(const char* msg) { g_err = msg; return -1; }
extern "C" const char* orcm_last_error(void) { return g_err.c_str(); }

static const double RHO_FLOOR = 1e-20, P_FLOOR = 1e-20;     // Q7, as in the hydro oracle

// ------------------------------------------------------------------------------------------------------------------
// HLLD (P:158 names the solver; Miyoshi & Kusano 2005, restated; Q34).  Rotated states W = (rho, u, v, w, u_g, By, Bz),
// normal field Bx = bn.  Five waves S_L <= S_L* <= S_M <= S_R* <= S_R; outer speeds
//   S_L = min(u_L, u_R) - max(cf_L, cf_R),  S_R = max(u_L, u_R) + max(cf_L, cf_R)        (their Eq. 67)
// with the fast speed cf^2 = [ (gamma p + B^2) + sqrt((gamma p + B^2)^2 - 4 gamma p Bx^2) ] / (2 rho).
// ------------------------------------------------------------------------------------------------------------------
struct Side { double r, u, v, w, e, by, bz, p, pt, E, vb, cf; double U[7], F[7]; };

static void side_init(double gamma, double bx, const double W[7], Side& s) {
  s.r = W[0]; s.u = W[1]; s.v = W[2]; s.w = W[3]; s.e = W[4]; s.by = W[5]; s.bz = W[6];
  s.p = (gamma - 1.0) * s.e;
  const double b2 = bx * bx + (s.by * s.by + s.bz * s.bz);
  s.pt = s.p + 0.5 * b2;
  s.E = s.e + 0.5 * s.r * (s.u * s.u + (s.v * s.v + s.w * s.w)) + 0.5 * b2;
  s.vb = s.u * bx + (s.v * s.by + s.w * s.bz);
  const double gp = gamma * s.p, sum = gp + b2;
  double disc = sum * sum - 4.0 * gp * (bx * bx);
  if (disc < 0.0) disc = 0.0;
  s.cf = std::sqrt((sum + std::sqrt(disc)) / (2.0 * s.r));
  const double U[7] = { s.r, s.r * s.u, s.r * s.v, s.r * s.w, s.E, s.by, s.bz };
  const double F[7] = { s.r * s.u, s.r * s.u * s.u + s.pt - bx * bx, s.r * s.u * s.v - bx * s.by, s.r * s.u * s.w - bx * s.bz,
                        (s.E + s.pt) * s.u - bx * s.vb, s.by * s.u - bx * s.v, s.bz * s.u - bx * s.w };
  for (int n = 0; n < 7; n++) { s.U[n] = U[n]; s.F[n] = F[n]; }
}

// star state of side K behind the outer wave SK (their Eqs. 43-48), given S_M and pt*
static void star_state(double bx, const Side& s, double SK, double SM, double pts, double Us[7], double* vbs) {
  const double sdu = SK - s.u, sdm = SK - SM;
  const double rs = s.r * sdu / sdm;
  const double den = s.r * sdu * sdm - bx * bx;
  double vs, ws, bys, bzs;
  if (std::fabs(den) < 1e-8 * pts) {                  // degenerate: the Alfven and the outer wave coincide
    vs = s.v; ws = s.w; bys = s.by; bzs = s.bz;
  } else {
    const double f1 = bx * (SM - s.u) / den, f2 = (s.r * sdu * sdu - bx * bx) / den;
    vs = s.v - s.by * f1; ws = s.w - s.bz * f1;
    bys = s.by * f2; bzs = s.bz * f2;
  }
  *vbs = SM * bx + (vs * bys + ws * bzs);
  const double Es = (sdu * s.E - s.pt * s.u + pts * SM + bx * (s.vb - *vbs)) / sdm;
  Us[0] = rs; Us[1] = rs * SM; Us[2] = rs * vs; Us[3] = rs * ws; Us[4] = Es; Us[5] = bys; Us[6] = bzs;
}

extern "C" void orcm_hlld(double gamma, double bn, const double WL[7], const double WR[7], double F[7]) {
  Side L, R;
  side_init(gamma, bn, WL, L);
  side_init(gamma, bn, WR, R);
  const double cfm = std::fmax(L.cf, R.cf);
  const double SL = std::fmin(L.u, R.u) - cfm, SR = std::fmax(L.u, R.u) + cfm;
  if (SL >= 0.0) { for (int n = 0; n < 7; n++) F[n] = L.F[n]; return; }
  if (SR <= 0.0) { for (int n = 0; n < 7; n++) F[n] = R.F[n]; return; }
  const double mL = L.r * (SL - L.u), mR = R.r * (SR - R.u);
  const double SM = ((mR * R.u - mL * L.u) - (R.pt - L.pt)) / (mR - mL);                       // Eq. 38
  const double pts = ((mR * L.pt - mL * R.pt) + mL * mR * (R.u - L.u)) / (mR - mL);            // Eq. 41
  double UsL[7], UsR[7], vbsL, vbsR;
  star_state(bn, L, SL, SM, pts, UsL, &vbsL);
  star_state(bn, R, SR, SM, pts, UsR, &vbsR);
  const double sqL = std::sqrt(UsL[0]), sqR = std::sqrt(UsR[0]);
  const double SsL = SM - std::fabs(bn) / sqL, SsR = SM + std::fabs(bn) / sqR;                 // Eq. 51
  // the side of the contact the face lies on, and whether it is inside the Alfven fan
  const bool left = (SM >= 0.0);
  const Side& K = left ? L : R;
  const double* Us = left ? UsL : UsR;
  const double SK = left ? SL : SR, SsK = left ? SsL : SsR;
  const bool outer = left ? (SsL >= 0.0) : (SsR <= 0.0);
  if (outer || 0.5 * bn * bn < 1e-8 * pts) {          // U** = U* where the normal field vanishes
    for (int n = 0; n < 7; n++) F[n] = K.F[n] + SK * (Us[n] - K.U[n]);
    return;
  }
  // double-star states between the Alfven waves (Eqs. 59-63)
  const double sgn = (bn > 0.0) ? 1.0 : -1.0, isum = 1.0 / (sqL + sqR);
  const double vsL = UsL[2] / UsL[0], wsL = UsL[3] / UsL[0], vsR = UsR[2] / UsR[0], wsR = UsR[3] / UsR[0];
  const double vss = (sqL * vsL + sqR * vsR + (UsR[5] - UsL[5]) * sgn) * isum;
  const double wss = (sqL * wsL + sqR * wsR + (UsR[6] - UsL[6]) * sgn) * isum;
  const double byss = (sqL * UsR[5] + sqR * UsL[5] + sqL * sqR * (vsR - vsL) * sgn) * isum;
  const double bzss = (sqL * UsR[6] + sqR * UsL[6] + sqL * sqR * (wsR - wsL) * sgn) * isum;
  const double vbss = SM * bn + (vss * byss + wss * bzss);
  double Uss[7];
  Uss[0] = Us[0]; Uss[1] = Us[1]; Uss[2] = Us[0] * vss; Uss[3] = Us[0] * wss;
  Uss[4] = left ? UsL[4] - sqL * (vbsL - vbss) * sgn : UsR[4] + sqR * (vbsR - vbss) * sgn;
  Uss[5] = byss; Uss[6] = bzss;
  for (int n = 0; n < 7; n++) F[n] = K.F[n] + SsK * Uss[n] - (SsK - SK) * Us[n] - SK * K.U[n];
}

// ------------------------------------------------------------------------------------------------------------------
// Pack descriptor: uniform single-level periodic mesh
// ------------------------------------------------------------------------------------------------------------------
struct orcm_pack {
  int nmb, nx[3], ng, nt[3], nrb[3];
  double gamma, xmin[3], xmax[3];
  std::vector<int> lx, leaf;             // lx[3m+d]; leaf[(l3*nrb2+l2)*nrb1+l1] -> m
  double* u[2] = { nullptr, nullptr };
  int cur = 0, nthreads = 1;
  int recon = 0;                         // 0 PLM, 1 PPM4, 2 PPMX, 3 WENOZ (the hydro oracle's codes and functions: oracle/orc.h)
  int nstages = 2;                       // 2: SSPRK(2,2), 3: SSPRK(3,3) (Q1)
  int rsolver = 0;                       // 0 HLLD, 1 LLF, 2 HLLE
  bool bound = false;
  long long floor_count = 0;
  size_t ncell() const { return (size_t)nt[0] * nt[1] * nt[2]; }
  size_t idx(int m, int n, int k, int j, int i) const { return ((((size_t)m * 8 + n) * nt[2] + k) * nt[1] + j) * nt[0] + i; }
  double dx(int d) const { return (xmax[d] - xmin[d]) / ((double)nrb[d] * nx[d]); }
};

extern "C" orcm_pack* orcm_pack_create(int nmb, int nx1, int nx2, int nx3, int ng, double gamma, int nrb1, int nrb2, int nrb3,
                                       const int* lx, const double xmin[3], const double xmax[3]) {
  if (nmb < 1 || !lx || !xmin || !xmax) { fail("bad arguments"); return nullptr; }
  if (ng < 3) { fail("MHD with PLM needs ng >= 3 (cell-centred fields of the outermost layer are not defined)"); return nullptr; }
  if (!(gamma > 1.0)) { fail("gamma <= 1"); return nullptr; }
  if (nmb != nrb1 * nrb2 * nrb3) { fail("a uniform pack has nrb1*nrb2*nrb3 blocks"); return nullptr; }
  orcm_pack* p = new orcm_pack;
  p->nmb = nmb; p->ng = ng; p->gamma = gamma;
  const int nx[3] = { nx1, nx2, nx3 }, nrb[3] = { nrb1, nrb2, nrb3 };
  for (int d = 0; d < 3; d++) {
    if (nx[d] < ng || !(xmax[d] > xmin[d])) { fail("nx_d >= ng and a non-empty domain are required"); delete p; return nullptr; }
    p->nx[d] = nx[d]; p->nt[d] = nx[d] + 2 * ng; p->nrb[d] = nrb[d]; p->xmin[d] = xmin[d]; p->xmax[d] = xmax[d];
  }
  p->lx.assign(lx, lx + 3 * (size_t)nmb);
  p->leaf.assign(nmb, -1);
  for (int m = 0; m < nmb; m++) {
    const int* l = &p->lx[3 * (size_t)m];
    for (int d = 0; d < 3; d++) if (l[d] < 0 || l[d] >= nrb[d]) { fail("logical location out of range"); delete p; return nullptr; }
    int& slot = p->leaf[((size_t)l[2] * nrb2 + l[1]) * nrb1 + l[0]];
    if (slot >= 0) { fail("duplicate block"); delete p; return nullptr; }
    slot = m;
  }
  return p;
}
extern "C" int orcm_pack_bind(orcm_pack* p, double* u_a, double* u_b) {
  if (!p || !u_a || !u_b) return fail("null argument");
  p->u[0] = u_a; p->u[1] = u_b; p->cur = 0; p->bound = true; p->floor_count = 0;
  return 0;
}
extern "C" int orcm_set_threads(orcm_pack* p, int n) { if (!p || n < 1) return fail("bad thread count"); p->nthreads = n; return 0; }
extern "C" double* orcm_pack_current(orcm_pack* p) { return (p && p->bound) ? p->u[p->cur] : nullptr; }
extern "C" long long orcm_pack_floor_count(const orcm_pack* p) { return p ? p->floor_count : -1; }
extern "C" int orcm_pack_destroy(orcm_pack* p) { delete p; return 0; }

// Ghost fill: every ghost cell takes all 8 variables of its periodic image, which is an ACTIVE cell; a face field
// travels with the cell whose lower face it sits on, so the shared face of two blocks is owned by the block above it.
extern "C" int orcm_fill_ghosts(orcm_pack* p) {
  if (!p || !p->bound) return fail("pack not bound");
  double* U = p->u[p->cur];
  const int ng = p->ng;
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) if (p->nthreads > 1)
  for (int m = 0; m < p->nmb; m++)
    for (int k = 0; k < p->nt[2]; k++) for (int j = 0; j < p->nt[1]; j++) for (int i = 0; i < p->nt[0]; i++) {
      const int a[3] = { i - ng, j - ng, k - ng };
      bool ghost = false;
      int src_l[3], s[3];
      for (int d = 0; d < 3; d++) {
        if (a[d] < 0 || a[d] >= p->nx[d]) ghost = true;
        const long N = (long)p->nrb[d] * p->nx[d];
        long g = ((long)p->lx[3 * (size_t)m + d] * p->nx[d] + a[d]) % N;
        if (g < 0) g += N;
        src_l[d] = (int)(g / p->nx[d]); s[d] = (int)(g - (long)src_l[d] * p->nx[d]) + ng;
      }
      if (!ghost) continue;
      const int src = p->leaf[((size_t)src_l[2] * p->nrb[1] + src_l[1]) * p->nrb[0] + src_l[0]];
      for (int n = 0; n < 8; n++) U[p->idx(m, n, k, j, i)] = U[p->idx(src, n, s[2], s[1], s[0])];
    }
  return 0;
}

// LLF and HLLE for MHD ("the local Lax-Friedrichs (LLF) method, various versions of the Harten-Lax-van Leer method"), in
// the same rotated variables.  LLF: F = (F_L + F_R)/2 - (lambda/2)(U_R - U_L), lambda = max(|u_L| + cf_L, |u_R| + cf_R).
// HLLE: the single-state HLL flux between the outer speeds of HLLD (Eq. 67 above), b- = min(S_L, 0), b+ = max(S_R, 0),
// F = [b+ F_L - b- F_R + b+ b- (U_R - U_L)] / (b+ - b-).
extern "C" void orcm_llf(double gamma, double bn, const double WL[7], const double WR[7], double F[7]) {
  Side L, R;
  side_init(gamma, bn, WL, L);
  side_init(gamma, bn, WR, R);
  const double lam = std::fmax(std::fabs(L.u) + L.cf, std::fabs(R.u) + R.cf);
  for (int n = 0; n < 7; n++) F[n] = 0.5 * (L.F[n] + R.F[n]) - 0.5 * lam * (R.U[n] - L.U[n]);
}
extern "C" void orcm_hlle(double gamma, double bn, const double WL[7], const double WR[7], double F[7]) {
  Side L, R;
  side_init(gamma, bn, WL, L);
  side_init(gamma, bn, WR, R);
  const double cfm = std::fmax(L.cf, R.cf);
  const double SL = std::fmin(L.u, R.u) - cfm, SR = std::fmax(L.u, R.u) + cfm;
  const double bm = std::fmin(SL, 0.0), bp = std::fmax(SR, 0.0);
  for (int n = 0; n < 7; n++) F[n] = ((bp * L.F[n] - bm * R.F[n]) + bp * bm * (R.U[n] - L.U[n])) / (bp - bm);
}

// van Leer PLM (Q4, as in the hydro oracle)
static inline void plm(double qm1, double q0, double qp1, double* q_minus, double* q_plus) {
  const double dL = q0 - qm1, dR = qp1 - q0, prod = dL * dR;
  const double h = (prod > 0.0) ? prod / (dL + dR) : 0.0;
  *q_minus = q0 - h; *q_plus = q0 + h;
}

// upwinded (face - centre) difference of an EMF (Gardiner & Stone 2005 / 2008, restated; Q36): taken on the side the mass
// flux through the transverse face comes from.  The switch is ramped: weight w of the lower side = 1/2 + nu clipped to
// [0, 1], nu = 1024 dt F_mass / (dx (rho_1 + rho_2)) with rho_1,2 the densities of the two cells the face separates -- the
// pure upwind value once the contact moves more than 2^-10 of a cell per step, the mean at rest, and a CONTINUOUS function
// of the state in between, so that a mass flux at round-off level does not decide the result.
static inline double upwind(double k, double mflux, double rho1, double rho2, double from_lower, double from_upper) {
  const double w = 0.5 + std::fmax(-0.5, std::fmin(0.5, (k * mflux) / (rho1 + rho2)));
  return w * from_lower + (1.0 - w) * from_upper;
}

// one block, one stage
static long long block_stage(const orcm_pack* p, const double* Uin, const double* U0, double* Uout, int m,
                             double g0, double g1, double beta, double dt) {
  const int ng = p->ng, n1 = p->nt[0], n2 = p->nt[1], n3 = p->nt[2];
  const size_t nc = p->ncell();
  const int str[3] = { 1, n1, n1 * n2 };
  const int nt[3] = { n1, n2, n3 };
  const double* Ub = Uin + (size_t)m * 8 * nc;
  long long nfl = 0;
  auto cid = [&](int k, int j, int i) { return ((size_t)k * n2 + j) * n1 + i; };
  // S1: primitives W = (rho, v1, v2, v3, u_g, B1, B2, B3) with cell-centred B = mean of the two faces (Q33); defined for
  // every cell but the outermost layer on the upper side
  std::vector<double> W(8 * nc, 0.0);
  for (int k = 0; k < n3 - 1; k++) for (int j = 0; j < n2 - 1; j++) for (int i = 0; i < n1 - 1; i++) {
    const size_t c = cid(k, j, i);
    double rho = Ub[c];
    if (!(rho >= RHO_FLOOR)) { rho = RHO_FLOOR; nfl++; }
    const double rinv = 1.0 / rho, m1 = Ub[nc + c], m2 = Ub[2 * nc + c], m3 = Ub[3 * nc + c];
    double B[3];
    for (int d = 0; d < 3; d++) B[d] = 0.5 * (Ub[(5 + d) * nc + c] + Ub[(5 + d) * nc + c + str[d]]);
    double ug = Ub[4 * nc + c] - 0.5 * rinv * (m1 * m1 + (m2 * m2 + m3 * m3)) - 0.5 * (B[0] * B[0] + (B[1] * B[1] + B[2] * B[2]));
    if (!(ug >= P_FLOOR / (p->gamma - 1.0))) { ug = P_FLOOR / (p->gamma - 1.0); nfl++; }
    W[c] = rho; W[nc + c] = m1 * rinv; W[2 * nc + c] = m2 * rinv; W[3 * nc + c] = m3 * rinv; W[4 * nc + c] = ug;
    for (int d = 0; d < 3; d++) W[(5 + d) * nc + c] = B[d];
  }
  // S2 + S3: PLM + HLLD at the lower d-face of every cell whose stencil exists.  Fd[d][n]: n = 0..4 the hydro fluxes in
  // the UNROTATED order, 5 = flux of B_{d+1}, 6 = flux of B_{d+2} (cyclic)
  std::vector<double> Fd[3];
  for (int d = 0; d < 3; d++) {
    Fd[d].assign(7 * nc, 0.0);
    const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
    const int var[7] = { 0, 1 + d, 1 + d1, 1 + d2, 4, 5 + d1, 5 + d2 };
    int lo[3] = { 0, 0, 0 }, hi[3] = { n1 - 1, n2 - 1, n3 - 1 };        // transverse: wherever W exists
    const int R = (p->recon == 0) ? 2 : 3;                              // along d: cells c-R .. c+R-1 must hold W
    lo[d] = R; hi[d] = nt[d] - R;
    for (int k = lo[2]; k < hi[2]; k++) for (int j = lo[1]; j < hi[1]; j++) for (int i = lo[0]; i < hi[0]; i++) {
      const size_t c = cid(k, j, i), cm = c - str[d];
      double WL[7], WR[7], F[7];
      for (int q = 0; q < 7; q++) {
        const double* w = &W[var[q] * nc];
        double qm, qp;
        if (p->recon == 0) {
          plm(w[cm - str[d]], w[cm], w[cm + str[d]], &qm, &qp); WL[q] = qp;
          plm(w[c - str[d]], w[c], w[c + str[d]], &qm, &qp);    WR[q] = qm;
        } else {                                                          // the hydro oracle's S2 / S2' on each primitive
          const double sL[5] = { w[cm - 2 * str[d]], w[cm - str[d]], w[cm], w[cm + str[d]], w[cm + 2 * str[d]] };
          const double sR[5] = { w[c - 2 * str[d]], w[c - str[d]], w[c], w[c + str[d]], w[c + 2 * str[d]] };
          if (p->recon == 1) { orc_ppm4(sL, &qm, &qp); WL[q] = qp; orc_ppm4(sR, &qm, &qp); WR[q] = qm; }
          else if (p->recon == 2) { orc_ppmx(sL, &qm, &qp); WL[q] = qp; orc_ppmx(sR, &qm, &qp); WR[q] = qm; }
          else               { orc_wenoz(sL, &qm, &qp); WL[q] = qp; orc_wenoz(sR, &qm, &qp); WR[q] = qm; }
        }
      }
      if (p->rsolver == 1) orcm_llf(p->gamma, Ub[(5 + d) * nc + c], WL, WR, F);
      else if (p->rsolver == 2) orcm_hlle(p->gamma, Ub[(5 + d) * nc + c], WL, WR, F);
      else orcm_hlld(p->gamma, Ub[(5 + d) * nc + c], WL, WR, F);
      Fd[d][c] = F[0]; Fd[d][(1 + d) * nc + c] = F[1]; Fd[d][(1 + d1) * nc + c] = F[2]; Fd[d][(1 + d2) * nc + c] = F[3];
      Fd[d][4 * nc + c] = F[4]; Fd[d][5 * nc + c] = F[5]; Fd[d][6 * nc + c] = F[6];
    }
  }
  // CT (Q35, Q36): cell-centred E = -v x B, face EMFs from the Riemann fluxes, corner EMFs by (ramped) upwinding
  std::vector<double> Ecc(3 * nc, 0.0), Ec(3 * nc, 0.0);
  for (size_t c = 0; c < nc; c++) {
    const double v1 = W[nc + c], v2 = W[2 * nc + c], v3 = W[3 * nc + c], B1 = W[5 * nc + c], B2 = W[6 * nc + c], B3 = W[7 * nc + c];
    Ecc[c] = -(v2 * B3 - v3 * B2); Ecc[nc + c] = -(v3 * B1 - v1 * B3); Ecc[2 * nc + c] = -(v1 * B2 - v2 * B1);
  }
  for (int e = 0; e < 3; e++) {                      // E_e on the edges along e, at the lower-a, lower-b corner of each cell
    const int a = (e + 1) % 3, b = (e + 2) % 3;
    const double* Fa = Fd[a].data(); const double* Fb = Fd[b].data();
    // E_e at an a-face = -F_a(B_b) (slot 5 of direction a), at a b-face = +F_b(B_a) (slot 6 of direction b)
    auto Eaf = [&](size_t c) { return -Fa[5 * nc + c]; };
    auto Ebf = [&](size_t c) { return Fb[6 * nc + c]; };
    const double* E0 = &Ecc[e * nc];
    const double ka = 1024.0 * dt / p->dx(a), kb = 1024.0 * dt / p->dx(b);
    int lo[3], hi[3];
    for (int d = 0; d < 3; d++) { lo[d] = ng; hi[d] = p->nx[d] + ng + 1; }
    hi[e] = p->nx[e] + ng;
    for (int k = lo[2]; k < hi[2]; k++) for (int j = lo[1]; j < hi[1]; j++) for (int i = lo[0]; i < hi[0]; i++) {
      const size_t c = cid(k, j, i), sa = str[a], sb = str[b];
      const double mean = 0.25 * ((Eaf(c - sb) + Eaf(c)) + (Ebf(c - sa) + Ebf(c)));
      const double* rho = W.data();
      const double l2 = upwind(ka, Fa[c - sb], rho[c - sb - sa], rho[c - sb], Ebf(c - sa) - E0[c - sa - sb], Ebf(c) - E0[c - sb]);
      const double r2 = upwind(ka, Fa[c],      rho[c - sa],      rho[c],      Ebf(c - sa) - E0[c - sa],      Ebf(c) - E0[c]);
      const double l1 = upwind(kb, Fb[c - sa], rho[c - sa - sb], rho[c - sa], Eaf(c - sb) - E0[c - sa - sb], Eaf(c) - E0[c - sa]);
      const double r1 = upwind(kb, Fb[c],      rho[c - sb],      rho[c],      Eaf(c - sb) - E0[c - sb],      Eaf(c) - E0[c]);
      Ec[e * nc + c] = mean + 0.25 * ((l1 + r1) + (l2 + r2));
    }
  }
  // S4: cells by the flux divergence, faces by the curl of the corner EMFs, with the stage weights
  const double cdt[3] = { beta * dt / p->dx(0), beta * dt / p->dx(1), beta * dt / p->dx(2) };
  const double* U0b = U0 + (size_t)m * 8 * nc;
  double* Uo = Uout + (size_t)m * 8 * nc;
  for (int k = ng; k < p->nx[2] + ng; k++) for (int j = ng; j < p->nx[1] + ng; j++) for (int i = ng; i < p->nx[0] + ng; i++) {
    const size_t c = cid(k, j, i);
    for (int n = 0; n < 5; n++) {
      double v = g0 * Ub[n * nc + c] + g1 * U0b[n * nc + c];
      for (int d = 0; d < 3; d++) v = v - cdt[d] * (Fd[d][n * nc + c + str[d]] - Fd[d][n * nc + c]);
      Uo[n * nc + c] = v;
    }
    for (int a = 0; a < 3; a++) {                    // db_a/dt = -(d_b E_c - d_c E_b), (a, b, c) cyclic
      const int b = (a + 1) % 3, cc = (a + 2) % 3;
      double v = g0 * Ub[(5 + a) * nc + c] + g1 * U0b[(5 + a) * nc + c];
      v = v - cdt[b] * (Ec[cc * nc + c + str[b]] - Ec[cc * nc + c]);
      v = v + cdt[cc] * (Ec[b * nc + c + str[cc]] - Ec[b * nc + c]);
      Uo[(5 + a) * nc + c] = v;
    }
  }
  return nfl;
}

// options: the reconstruction list of P:101 and the RK2 / RK3 integrators the paper's MHD tests and runs use (RK3 + PPMX /
// WENOZ, PPM4, PLM on the linear waves; WENOZ + RK2 + HLLD for the turbulence run)
extern "C" int orcm_pack_set_recon(orcm_pack* p, int recon) {
  if (!p) return fail("null pack");
  if (recon < 0 || recon > 3) return fail("reconstruction: 0 PLM, 1 PPM4, 2 PPMX, 3 WENOZ");
  if (recon != 0 && p->ng < 4) return fail("PPM4 / PPMX / WENOZ with face-centred fields need ng >= 4");
  p->recon = recon;
  return 0;
}
extern "C" int orcm_pack_set_rsolver(orcm_pack* p, int rsolver) {
  if (!p) return fail("null pack");
  if (rsolver < 0 || rsolver > 2) return fail("Riemann solver: 0 HLLD, 1 LLF, 2 HLLE");
  p->rsolver = rsolver;
  return 0;
}
extern "C" int orcm_pack_set_integrator(orcm_pack* p, int nstages) {
  if (!p) return fail("null pack");
  if (nstages != 2 && nstages != 3) return fail("integrator: 2 = SSPRK(2,2), 3 = SSPRK(3,3)");
  if (p->cur != 0) return fail("the integrator can only change between steps");
  p->nstages = nstages;
  return 0;
}

// One stage: U_out = g0 U_in + g1 U^n - beta dt div F(U_in) for the cells, the same weights with the curl of the corner EMFs for
// the faces.  SSPRK(2,2): A -> B, (B, A) -> A.  SSPRK(3,3) (Q1): A -> B; B <- 1/4 (B + dt L(B)) + 3/4 A (in place: every block
// forms all its fluxes and EMFs from U_in before it writes); A <- 2/3 (B + dt L(B)) + 1/3 A.
extern "C" int orcm_stage(orcm_pack* p, int stage, double dt) {
  if (!p || !p->bound) return fail("pack not bound");
  const int ns = p->nstages;
  if (stage < 1 || stage > ns || p->cur != (stage == 1 ? 0 : 1)) return fail("stages must be called in order, starting from U^n in buffer A");
  static const double C2[2][3] = { { 0.0, 1.0, 1.0 }, { 0.5, 0.5, 0.5 } };      // SSPRK(2,2), Q1
  static const double C3[3][3] = { { 0.0, 1.0, 1.0 }, { 0.25, 0.75, 0.25 }, { 2.0 / 3.0, 1.0 / 3.0, 2.0 / 3.0 } };
  const double* cf = (ns == 2) ? C2[stage - 1] : C3[stage - 1];
  const double g0 = cf[0], g1 = cf[1], beta = cf[2];
  const double* Uin = p->u[p->cur]; const double* U0 = p->u[0];
  const int out = (stage == ns) ? 0 : 1;
  double* Uout = p->u[out];
  long long nfl = 0;
#pragma omp parallel for schedule(dynamic) num_threads(p->nthreads) reduction(+ : nfl) if (p->nthreads > 1)
  for (int m = 0; m < p->nmb; m++) nfl += block_stage(p, Uin, U0, Uout, m, g0, g1, beta, dt);
  p->floor_count += nfl;
  p->cur = out;
  return 0;
}

// Eq.(3) with the fast magnetosonic speed along each direction (Q37)
extern "C" int orcm_new_dt(orcm_pack* p, double cfl, double* dt_out) {
  if (!p || !p->bound || !dt_out) return fail("pack not bound");
  const double* U = p->u[p->cur];
  const int ng = p->ng;
  const int str[3] = { 1, p->nt[0], p->nt[0] * p->nt[1] };
  double dtmin = HUGE_VAL; long long bad = 0;
  for (int m = 0; m < p->nmb; m++)
    for (int k = ng; k < p->nx[2] + ng; k++) for (int j = ng; j < p->nx[1] + ng; j++) for (int i = ng; i < p->nx[0] + ng; i++) {
      const size_t c = p->idx(m, 0, k, j, i), nc = p->ncell();
      double rho = U[c];
      if (!(rho >= RHO_FLOOR)) rho = RHO_FLOOR;
      const double rinv = 1.0 / rho, m1 = U[c + nc], m2 = U[c + 2 * nc], m3 = U[c + 3 * nc];
      double B[3];
      for (int d = 0; d < 3; d++) B[d] = 0.5 * (U[c + (5 + d) * nc] + U[c + (5 + d) * nc + str[d]]);
      const double b2 = B[0] * B[0] + (B[1] * B[1] + B[2] * B[2]);
      double ug = U[c + 4 * nc] - 0.5 * rinv * (m1 * m1 + (m2 * m2 + m3 * m3)) - 0.5 * b2;
      if (!(ug >= P_FLOOR / (p->gamma - 1.0))) ug = P_FLOOR / (p->gamma - 1.0);
      const double gp = p->gamma * ((p->gamma - 1.0) * ug), sum = gp + b2;
      const double v[3] = { m1 * rinv, m2 * rinv, m3 * rinv };
      for (int d = 0; d < 3; d++) {
        double disc = sum * sum - 4.0 * gp * (B[d] * B[d]);
        if (disc < 0.0) disc = 0.0;
        const double cf = std::sqrt((sum + std::sqrt(disc)) / (2.0 * rho));
        const double s = std::fabs(v[d]) + cf;
        if (!(s > 0.0 && s < HUGE_VAL)) { bad++; continue; }
        const double cand = p->dx(d) / s;
        if (cand < dtmin) dtmin = cand;
      }
    }
  if (bad) return fail("non-finite signal speed in the state (NaN or inf)");
  *dt_out = cfl * dtmin;
  return 0;
}

/* orc.h -- CPU ORACLE for the MeshBlockPack hydro stage.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this library.  It shares no code with the CUDA path in
 * paper_2409_16053_b200/csrc/ and neither includes the other.
 *
 * It follows, step by step and in the paper's order, the scheme the paper names
 * (/root/reference/PAPER.md, cited as P:line): finite-volume "reconstruct, solve, advance",
 * PLM / PPM4 reconstruction of the primitive variables, the HLLC Riemann solver,
 * SSP-RK2 with the CFL rule Eq.(3), the Newtonian gamma-law system Eq.(4)
 * (P:122-126), ghost-zone copies between MeshBlocks and restriction / prolongation at level
 * boundaries.  The paper defers every formula to its references; the readings
 * taken are SURVEY.md section 8(c) steps S0-S4 and G1-G4 and are listed in DESIGN.md.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): exact Riemann solution (Sod), sound-wave
 * convergence order, conservation, uniform-state preservation, mirror / permutation symmetry,
 * decomposition invariance, HLLC consistency / contact / supersonic / mirror properties, PLM and
 * PPM4 linear-data and monotonicity properties, brute-force ghost fill, dyadic-linear
 * restriction / prolongation; round 2: closed-form collision fluxes, strong two-shock tube, two-level dt,
 * PPMX / WENOZ polynomial exactness and the paper's fourth-order linear-wave convergence, FOFC positivity,
 * Shu-Osher tube.  PARITY UNPINNED beyond those properties: the particular HLLC wave-speed estimate
 * (Q2: Davis's direct estimates since round 2), the PPM4 variant (Q5), the floors (Q7), the WENOZ and
 * PPMX variants (Q29, Q30) and the FOFC criterion (Q31) -- the paper does not fix them.
 *
 * Layout: U[m][n][k][j][i], n = (rho, rho v1, rho v2, rho v3, E), i fastest, ghosts included
 * (P:63).  All pointers are HOST pointers owned by the caller.  Single-threaded unless
 * orc_set_threads(n>1) is called (OpenMP over MeshBlocks; results are bit-identical because
 * blocks are independent within a call and min is order-independent).
 */
#ifndef ORC_H
#define ORC_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_pack orc_pack;

/* recon: 0 = PLM (van Leer), 1 = PPM4, 2 = PPMX, 3 = WENOZ (ng >= 3 for 1-3); rsolver: 0 = HLLC, 1 = LLF, 2 = HLLE, 3 = Roe.  NULL on invalid arguments. */
orc_pack* orc_pack_create(int nmb, int nx1, int nx2, int nx3, int ng, double gamma, int recon, int rsolver);
int orc_pack_set_mesh(orc_pack*, int nrb1, int nrb2, int nrb3,
                      double x1min, double x1max, double x2min, double x2max, double x3min, double x3max);
int orc_pack_set_block(orc_pack*, int m, int level, int lx1, int lx2, int lx3);
/* f3: boundary condition per face (x1min, x1max, x2min, x2max, x3min, x3max): 0 periodic (default), 1 outflow,
 * 2 reflect.  Periodic faces come in pairs; non-periodic boundaries need a single-level mesh.  Call before bind. */
int orc_pack_set_boundaries(orc_pack*, const int bc[6]);
/* u_a holds U^n on entry; u_b is the second register.  Validates that the leaves tile the domain. */
int orc_pack_bind(orc_pack*, double* u_a, double* u_b);
int orc_set_threads(orc_pack*, int nthreads);
/* f1: replace the coarse flux at level-boundary faces by the mean of the four fine fluxes.  Off by default. */
int orc_set_flux_correction(orc_pack*, int on);
/* f2: first-order flux correction -- faces of cells whose tentative update has rho <= 0 or e_int <= 0 take the
 * LLF flux of the cell-centred states; single-level meshes; off by default.  orc_pack_fofc_count: cells flagged since bind. */
int orc_set_fofc(orc_pack*, int on);
long long orc_pack_fofc_count(const orc_pack*);
int orc_fill_ghosts(orc_pack*);                           /* G1-G4 on the current buffer           */
int orc_hydro_stage(orc_pack*, int stage, double dt);     /* S1-S4; stage 1: A->B, stage 2: B,A->A (RK3: B,A->C; C,A->A) */
/* f2: number of stages, 2 = SSPRK(2,2) (default) or 3 = SSPRK(3,3), which needs a third caller-owned buffer u_c. */
int orc_set_integrator(orc_pack*, int nstages, double* u_c);
int orc_new_dt(orc_pack*, double cfl, double* dt_out);    /* S0 on the current buffer              */
double* orc_pack_current(orc_pack*);
long long orc_pack_floor_count(const orc_pack*);
int orc_pack_destroy(orc_pack*);
const char* orc_last_error(void);

/* Single-operation entry points, exposed so each formula can be pinned on its own. */
void orc_c2p(double gamma, const double U[5], double W[5], int* floored);       /* S1 */
void orc_plm(double qm1, double q0, double qp1, double* q_minus, double* q_plus);       /* S2 */
void orc_ppm4(const double q[5] /* i-2..i+2 */, double* q_minus, double* q_plus);      /* S2 */
void orc_ppm4_iface(double qm1, double q0, double qp1, double qp2, double* q_half);    /* S2 (i),(ii) */
void orc_ppmx(const double q[5] /* i-2..i+2 */, double* q_minus, double* q_plus);      /* S2', f2: DESIGN.md Q30 */
void orc_wenoz(const double q[5] /* i-2..i+2 */, double* q_minus, double* q_plus);     /* S2', f2: DESIGN.md Q29 */
void orc_hllc(double gamma, int dir /*0,1,2*/, const double WL[5], const double WR[5], double F[5]); /* S3 */
void orc_llf (double gamma, int dir, const double WL[5], const double WR[5], double F[5]);             /* S3', f2 */
void orc_hlle(double gamma, int dir, const double WL[5], const double WR[5], double F[5]);             /* S3', f2 */
void orc_roe (double gamma, int dir, const double WL[5], const double WR[5], double F[5]);             /* S3', f2 */

#ifdef __cplusplus
}
#endif
#endif

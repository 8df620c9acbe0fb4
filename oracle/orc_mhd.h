/* orc_mhd.h -- CPU ORACLE for the MHD + constrained-transport stage.  TEST INFRASTRUCTURE ONLY:
 * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may build, load or call it.  It shares no code with
 * the CUDA path in paper_2409_16053_b200/csrc/ and neither includes the other.
 *
 * What the paper states (/root/reference/PAPER.md, P:line): Newtonian MHD, Eq.(5) with p* = p_g + B^2/2 and the gamma-law
 * E = p_g/(gamma-1) + rho v^2/2 + B^2/2; "the magnetic field is discretized as area-averages on cell-faces, and
 * the constrained transport (CT) algorithm of Evans & Hawley (1988) is used to preserve the divergence-free constraint with
 * upwinded electric fields calculated using the method of Gardiner & Stone (2005, 2008)"; HLLD is the solver of its
 * MHD run; all MHD waves converge at second order with PLM.  The formulas are deferred to those papers; the
 * readings taken are DESIGN.md Q33-Q37.  Scope: uniform single-level periodic packs; PLM (van Leer), PPM4, PPMX or WENOZ (the hydro
 * oracle's functions, orc.h) on the primitives (rho, v, u_g, B_t); HLLD; SSPRK(2,2) or SSPRK(3,3).
 *
 * Layout: U[m][n][k][j][i], n = 0..7 = (rho, rho v1, rho v2, rho v3, E, b1, b2, b3), i fastest, ghosts included, ng >= 3;
 * b_d of cell (k,j,i) is the area-averaged field on the LOWER d-face of that cell (the upper face of the last active cell is
 * the lower face of the first ghost cell beyond it).  All pointers are HOST pointers owned by the caller.
 *
 * Pins (tests/test_oracle_mhd.py): HLLD consistency with Eq.(5), mirror symmetry, exact stationary contact and (B = 0) Sod
 * convergence to the exact Riemann solution; LLF / HLLE consistency, mirror symmetry, closed-form dissipation on a stationary contact,
 * exact supersonic upwinding (HLLE); div B = 0 to round-off; conservation of mass, momentum, energy and mean field; uniform state
 * preserved bit-exactly; plane-parallel flow stays plane-parallel and direction-independent bit for bit; results independent of
 * the block decomposition bit for bit; the corner EMFs continuous where a mass flux changes sign (Q36); second-order convergence
 * of fast, Alfven and slow linear waves, along x1 and obliquely, whose eigenvectors the test computes numerically, and
 * the paper's statement about the higher-order options: RK3 + WENOZ / PPMX converge at fourth order on Alfven and slow
 * waves, the fast wave at second order, PPM4 at second order.
 * PARITY UNPINNED beyond those properties: the HLLD wave-speed estimate and degenerate-case thresholds (Q34), the ramp
 * width of the upwinding rule of the corner EMFs (Q36).
 */
#ifndef ORC_MHD_H
#define ORC_MHD_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orcm_pack orcm_pack;

/* Uniform periodic pack: nrb1 x nrb2 x nrb3 root blocks of nx1 x nx2 x nx3 cells on [xmin, xmax); lx[3 m + d] = logical
 * location of block m.  NULL on invalid arguments (orcm_last_error()). */
orcm_pack* orcm_pack_create(int nmb, int nx1, int nx2, int nx3, int ng, double gamma, int nrb1, int nrb2, int nrb3,
                            const int* lx, const double xmin[3], const double xmax[3]);
int orcm_pack_bind(orcm_pack*, double* u_a, double* u_b);   /* u_a holds U^n; both of nmb*8*nt1*nt2*nt3 doubles */
int orcm_set_threads(orcm_pack*, int nthreads);
int orcm_pack_set_recon(orcm_pack*, int recon);              /* 0 PLM (default), 1 PPM4, 2 PPMX, 3 WENOZ (orc.h's functions); ng >= 4 for 1-3 */
int orcm_pack_set_rsolver(orcm_pack*, int rsolver);          /* 0 HLLD (default), 1 LLF, 2 HLLE */
int orcm_pack_set_integrator(orcm_pack*, int nstages);      /* 2 = SSPRK(2,2) (default), 3 = SSPRK(3,3) */
int orcm_fill_ghosts(orcm_pack*);                           /* periodic copy of all 8 variables into the ghost cells */
int orcm_stage(orcm_pack*, int stage, double dt);           /* one stage: RK2 1: A -> B, 2: (B, A) -> A; RK3 2: (B, A) -> B, 3: (B, A) -> A */
int orcm_new_dt(orcm_pack*, double cfl, double* dt_out);    /* cfl * min dx_d / (|v_d| + c_fast,d) over active cells */
double* orcm_pack_current(orcm_pack*);
long long orcm_pack_floor_count(const orcm_pack*);
int orcm_pack_destroy(orcm_pack*);
const char* orcm_last_error(void);

/* HLLD flux of rotated states W = (rho, u_n, v_t1, v_t2, u_g, B_t1, B_t2) with the normal field bn;
 * F = (mass, normal momentum, transverse momenta, energy, flux of B_t1, flux of B_t2). */
void orcm_hlld(double gamma, double bn, const double WL[7], const double WR[7], double F[7]);
void orcm_llf(double gamma, double bn, const double WL[7], const double WR[7], double F[7]);    /* P:103, same variables */
void orcm_hlle(double gamma, double bn, const double WL[7], const double WR[7], double F[7]);

#ifdef __cplusplus
}
#endif
#endif

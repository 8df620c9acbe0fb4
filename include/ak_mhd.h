/* ak_mhd.h -- C-ABI boundary of the MHD + constrained-transport stage, first cut.
 *
 * Newtonian ideal MHD, paper Eq.(5) with the gamma-law energy E = p_g/(gamma-1) + rho v^2/2 + B^2/2 (/root/reference/PAPER.md
 * lines 146-150, cited as P:NN), on a MeshBlockPack resident in device memory.  "The magnetic field is discretized
 * as area-averages on cell-faces, and the constrained transport (CT) algorithm of Evans & Hawley (1988) is used to preserve the
 * divergence-free constraint with upwinded electric fields calculated using the method of Gardiner & Stone (2005, 2008)"
 * (P:116); HLLD Riemann solver.  Readings: DESIGN.md Q33-Q37.  Scope of this cut: uniform single-level periodic packs;
 * PLM (van Leer), PPM4, PPMX or WENOZ reconstruction of the primitives; HLLD (LLF, HLLE with PLM); SSPRK(2,2) or SSPRK(3,3) -- the options of the
 * paper's MHD tests and runs; the kernels are not fused (face fluxes and corner EMFs pass through a caller-owned
 * work buffer in device memory).
 *
 * One step:   akm_new_dt(p, cfl, &dt);  for stage in 1 .. nstages: { akm_fill_ghosts(p); akm_stage(p, stage, dt); }
 *
 * State layout: U[m][n][k][j][i], n = 0..7 = (rho, rho v1, rho v2, rho v3, E, b1, b2, b3), i fastest, fp64, ng >= 3 ghost
 * layers included; b_d of cell (k,j,i) is the field on the LOWER d-face of that cell.  Memory is caller-owned (device
 * pointers, 256-byte aligned); the descriptor is a small host object.  All functions are host functions; int results are
 * AK-style codes: 0 ok, -1 bad argument, -2 call order, -3 unsupported, -4 CUDA error, -5 non-finite state;
 * akm_last_error() returns a thread-local message.  No CPU fallback exists.
 */
#ifndef AK_MHD_H
#define AK_MHD_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct akm_pack akm_pack;

/* nrb1 x nrb2 x nrb3 root blocks of nx1 x nx2 x nx3 cells on the periodic box [xmin, xmax) (HOST arrays of 3);
 * lx[3 m + d] (HOST) = logical location of block m; nmb = nrb1 nrb2 nrb3.  NULL on invalid arguments. */
akm_pack* akm_pack_create(int nmb, int nx1, int nx2, int nx3, int ng, double gamma, int nrb1, int nrb2, int nrb3,
                          const int* lx, const double* xmin, const double* xmax);
size_t akm_pack_state_bytes(const akm_pack*);   /* one state buffer: nmb * 8 * (nx1+2ng)(nx2+2ng)(nx3+2ng) * 8 bytes */
size_t akm_pack_work_bytes(const akm_pack*);    /* work buffer: primitives, face fluxes, corner EMFs, tables          */
/* u_a holds U^n (ghost cells arbitrary) and becomes current; u_b is the second register; work the work buffer; all DEVICE
 * pointers, pairwise disjoint; cuda_stream a cudaStream_t (NULL = legacy stream) on which every kernel is launched. */
int akm_pack_bind(akm_pack*, void* u_a, void* u_b, void* work, void* cuda_stream);
/* Arithmetic of the flux sweeps.  on = 0 (default): reciprocals and square roots from the MUFU seed + one cubically convergent step
 * (1-2 ulp), quotients by a shared divisor through one reciprocal.  on = 1: IEEE division and sqrt in the definition's operation
 * order; the whole path is then bit-identical to the oracle the tests compare with (verification mode, ~30 % slower).  The two
 * differ by rounding only (<= 1e-14 per stage in the tests' metric); the upwind switch of the corner EMFs is ramped (DESIGN.md
 * Q36), so a face mass flux at round-off level does not decide a side. */
int akm_pack_set_exact(akm_pack*, int on);
/* Reconstruction: 0 PLM (default), 1 PPM4, 2 PPMX, 3 WENOZ (the codes of ak.h; Q29, Q30); 1-3 need ng >= 4 (-1 otherwise);
 * -3 for any other code. */
int akm_pack_set_recon(akm_pack*, int recon);
/* Riemann solver: 0 HLLD (default), 1 LLF, 2 HLLE (in HLLD's variables and outer wave speeds); 1 and 2 with PLM only (-3). */
int akm_pack_set_rsolver(akm_pack*, int rsolver);
/* Integrator: 2 = SSPRK(2,2) (default), 3 = SSPRK(3,3); between steps only (-2 inside a step). */
int akm_pack_set_integrator(akm_pack*, int nstages);

/* Periodic copy of all 8 variables into the ghost cells of the current buffer; bit-exact.  Asynchronous. */
int akm_fill_ghosts(akm_pack*);
/* One stage (SSPRK(2,2): 1: A -> B, 2: (B, A) -> A; SSPRK(3,3): 1: A -> B, 2: (B, A) -> B, 3: (B, A) -> A): primitives,
 * reconstruction + HLLD in x1, x2, x3, corner EMFs, flux
 * divergence for the cells and curl of the EMFs for the faces (div B is preserved to round-off).  Needs akm_fill_ghosts
 * on the current buffer first (-2 otherwise).  Asynchronous. */
int akm_stage(akm_pack*, int stage, double dt);
/* cfl * min over active cells and d of dx_d / (|v_d| + c_fast,d) (Eq.(3), with the fast magnetosonic speed);
 * dt_out is a HOST pointer; synchronises the stream; -5 for a NaN / inf state. */
int akm_new_dt(akm_pack*, double cfl, double* dt_out);
/* akm_new_dt (unless dt_fixed > 0), then the (fill, stage) pairs of the integrator; dt_out (HOST, may be NULL) receives the step taken. */
int akm_step(akm_pack*, double cfl, double dt_fixed, double* dt_out);
void* akm_pack_current(const akm_pack*);        /* device pointer of the buffer holding the latest state             */
long long akm_pack_floor_count(akm_pack*);      /* floor activations since bind (synchronises); negative on error    */
long long akm_pack_launch_count(const akm_pack*);
int akm_pack_destroy(akm_pack*);
const char* akm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif

/* ak.h -- C-ABI boundary of the B200-native MeshBlockPack hydro stage.
 *
 * The library advances Newtonian adiabatic hydrodynamics (paper Eq.(4), /root/reference/PAPER.md
 * lines 122-126, cited below as P:NN) on a MeshBlockPack -- all MeshBlocks resident on one device
 * and updated by one kernel launch -- stored as (N+1)-dimensional arrays
 * U[m][n][k][j][i] that never leave device memory.  The host only sequences calls; every
 * operation on the dependent variables runs in a CUDA kernel.
 *
 * One time step of the paper's method-of-lines RK2 scheme is
 *
 *     ak_new_dt(p, cfl, &dt);                        CFL rule, Eq.(3)
 *     for stage in 1, 2:
 *         ak_fill_ghosts(p);                         boundary kernels between stages
 *         ak_hydro_stage(p, stage, dt);              reconstruct - solve - advance
 *
 * Memory ownership: the caller (PyTorch in this repo) allocates every device buffer and supplies
 * the CUDA stream; the pack descriptor is a small host object that owns no device memory.
 * All functions are host functions.  "device pointer" / "host pointer" is stated per argument.
 * Threading: a pack is not thread-safe; different packs are independent.
 * Errors: functions returning int give AK_OK (0) or a negative code; ak_last_error() returns a
 * thread-local message for the last failing call.  Nothing throws.  Asynchronous CUDA errors
 * surface at the next synchronising call (ak_new_dt, ak_pack_download, ak_pack_floor_count).
 * There is no CPU fallback: without a CUDA device every compute call fails with AK_ECUDA.
 */
#ifndef AK_H
#define AK_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

#define AK_OK            0
#define AK_EINVAL      (-1)   /* bad argument                                   */
#define AK_ESTATE      (-2)   /* call order violated (e.g. stage before fill)   */
#define AK_EUNSUPPORTED (-3)  /* valid request outside the implemented scope    */
#define AK_ECUDA       (-4)   /* CUDA runtime error, message in ak_last_error() */
#define AK_ENONFINITE  (-5)   /* the state holds a NaN / inf: ak_new_dt found a non-finite signal speed */

#define AK_RECON_PLM   0      /* piecewise linear, van Leer limiter     */
#define AK_RECON_PPM4  1      /* piecewise parabolic, Colella-Woodward limiters */
#define AK_RECON_PPMX  2      /* PPM with extremum-preserving limiters; ng >= 3; HLLC, production kernel only */
#define AK_RECON_WENOZ 3      /* fifth-order WENO-Z; ng >= 3; HLLC, production kernel only */
#define AK_RSOLVER_HLLC 0
#define AK_RSOLVER_LLF  1     /* Rusanov, a = max(|u|+c) of the two states            */
#define AK_RSOLVER_HLLE 2     /* Einfeldt speeds from the Roe averages                */
#define AK_RSOLVER_ROE  3     /* Roe's linearised solver, no entropy fix               */

typedef struct ak_pack ak_pack;          /* opaque host-side descriptor */

const char* ak_last_error(void);

/* Create the descriptor of a pack of `nmb` MeshBlocks of nx1*nx2*nx3 active cells with `ng` ghost
 * layers, gamma-law EOS p=(gamma-1)u_g, reconstruction and Riemann solver
 * chosen at run time and instantiated as templates inside.
 * Returns NULL on error.  Rejects: nmb<1, nx_d<ng, odd nx_d, ng<2 (PLM) or ng<3 (PPM4), ng>4,
 * gamma<=1, unknown enums. */
ak_pack* ak_pack_create(int nmb, int nx1, int nx2, int nx3, int ng,
                        double gamma, int recon, int rsolver);

/* Periodic root grid of nrb1*nrb2*nrb3 blocks on [x_min,x_max]^3, uniform Cartesian. */
int ak_pack_set_mesh(ak_pack*, int nrb1, int nrb2, int nrb3,
                     double x1min, double x1max, double x2min, double x2max,
                     double x3min, double x3max);

/* Logical location of block m in the block tree: level 0 (root) or 1 (refined once),
 * 0 <= lx_d < nrb_d * 2^level.  Cell size of a block: (x_max-x_min)/(nrb_d*nx_d*2^level). */
int ak_pack_set_block(ak_pack*, int m, int level, int lx1, int lx2, int lx3);

/* Size in bytes of ONE state buffer, nmb*5*(nx1+2ng)*(nx2+2ng)*(nx3+2ng)*8, layout
 * U[m][n][k][j][i], n = (rho, rho v1, rho v2, rho v3, E), i fastest, ghosts included. */
size_t ak_pack_state_bytes(const ak_pack*);
/* Size in bytes of the scratch buffer (block table, leaf lookup maps, reduction cells). */
size_t ak_pack_scratch_bytes(const ak_pack*);

/* Attach caller-owned DEVICE memory and a CUDA stream (cudaStream_t passed as void*; NULL = the
 * legacy default stream).  u_a holds U^n and is the "current" buffer; u_b is the second RK
 * register; scratch is ak_pack_scratch_bytes() long.  All three must be 256-byte aligned and
 * must not overlap.  Validates that the blocks tile the domain (each root block is either a leaf
 * or fully covered by its 8 children), that refinement uses even ng, builds the block table and
 * leaf maps and uploads them into scratch (synchronises the stream once). */
int ak_pack_bind(ak_pack*, void* u_a, void* u_b, void* scratch, void* cuda_stream);

/* Fill every ghost cell (faces, edges, corners, depth ng) of the current buffer from the active
 * cells of the leaf block that covers its periodic image: same level -> copy; finer
 * neighbour -> conservative restriction (mean of 8, fixed order); coarser neighbour ->
 * limited-linear (minmod) prolongation of the conserved variables.  Reads active cells only,
 * writes ghost cells only; bit-exact against the oracle.  Asynchronous on the stream.  Returns without a launch
 * when the ghost cells are already current (the stage that wrote the state also wrote them: ak_pack_set_ghost_push). */
int ak_fill_ghosts(ak_pack*);

/* One Runge-Kutta stage.  Default integrator, SSP-RK2 in two registers:
 *   stage 1:  B = A - dt L(A)-terms            (reads A, writes B, B becomes current)
 *   stage 2:  A = 1/2 A + 1/2 (B + dt L(B))    (reads B and A, writes A, A becomes current)
 * (SSPRK(3,3) after ak_pack_set_integrator: stages 1..3, A -> B -> C -> A.)  Stages are called in order, starting
 * with U^n in buffer A (AK_ESTATE otherwise; AK_EINVAL for a stage number the integrator does not have).
 * With L = -sum_d (F_d(i+1/2) - F_d(i-1/2))/dx_d, F from conserved->primitive, PLM/PPM4
 * reconstruction of the primitives and the HLLC flux in x1, x2, x3, fused in one
 * launch; face fluxes never reach device memory.  The Riemann solver is the one given to ak_pack_create (HLLC, LLF,
 * HLLE or Roe).  The last stage of a step also reduces the signal speeds of its result for the next ak_new_dt.
 * Requires ak_fill_ghosts on the current buffer since the last change (else AK_ESTATE).  Asynchronous on the
 * stream. */
int ak_hydro_stage(ak_pack*, int stage, double dt);

/* CFL time step, Eq.(3): cfl * min over active cells of all blocks and over d of
 * dx_d(level) / (|v_d| + c_s), one dt for all levels.  dt_out is a HOST pointer.
 * Synchronises the stream.  After a complete step the answer comes from the maxima the last stage left behind
 * (48 bytes copied, no launch); otherwise a reduction kernel reads the state.  Both give the same bits. */
int ak_new_dt(ak_pack*, double cfl, double* dt_out);

/* The same CFL reduction (Eq.(3); the kernel ak_new_dt launches) for callers that may not allocate device
 * memory -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc -- and have no pack
 * with its caller-allocated scratch buffer.  u: DEVICE pointer to U[m][n][k][j][i] of a uniform single-level pack of nmb
 * MeshBlocks of nx1 x nx2 x nx3 active cells with ng ghost layers (ghost cells are not read); dx1..3: cell sizes;
 * dt_out: HOST pointer, receives cfl * min over active cells and directions of dx_d / (|v_d| + c_s), bit-identical to
 * ak_new_dt on the same state.  The reduction cells and the block table live in a 128 KiB static device array inside the
 * library (held by every GPU that loads the library until exit); nmb <= 8176, else AK_EUNSUPPORTED.  Calls no cudaMalloc,
 * cudaFree or allocating library routine.  Runs on the device that owns u, on cuda_stream, and synchronises it.  All
 * calls share the array: every call rewrites what it uses first, but calls that overlap on one GPU (two streams, two
 * threads) race on it -- serialise them.  AK_ENONFINITE for a NaN / inf state. */
int ak_new_dt_noalloc(const void* u, int nmb, int nx1, int nx2, int nx3, int ng, double gamma,
                      double dx1, double dx2, double dx3, double cfl, void* cuda_stream, double* dt_out);

/* Convenience: ak_new_dt, then (ak_fill_ghosts, ak_hydro_stage) for every stage of the integrator (2 by default,
 * 3 after ak_pack_set_integrator(p, 3, u_c)).  dt_out (HOST, may be NULL)
 * receives the step taken.  If dt_fixed > 0 it is used instead of the CFL value (lock-step parity
 * runs) and no reduction is launched. */
int ak_step(ak_pack*, double cfl, double dt_fixed, double* dt_out);

/* DEVICE pointer of the buffer holding the newest U (u_a or u_b). */
void* ak_pack_current(const ak_pack*);

/* Host <-> device transfer of one whole state buffer through the pack's stream.
 * upload: HOST -> buffer A, which becomes current, ghosts marked unfilled (asynchronous; the host
 * buffer must stay valid until the stream reaches the copy -- pinned memory makes it truly async).
 * download: current buffer -> HOST, synchronises the stream. */
int ak_pack_upload(ak_pack*, const void* host_u);
int ak_pack_download(ak_pack*, void* host_u);
/* As ak_pack_download without the synchronisation: the copy is only enqueued on the pack's stream (pinned host
 * memory makes it asynchronous); the caller synchronises the stream before reading host_u.  Lets two packs on two
 * streams overlap one pack's download with the other's upload and compute (bench.py e2e_pipelined). */
int ak_pack_download_async(ak_pack*, void* host_u);

/* Number of density / internal-energy floor activations in conserved->primitive since bind
 * (diagnostic; 0 on all BASELINE configs).  Synchronises the stream.  Negative on error. */
long long ak_pack_floor_count(ak_pack*);

/* Selects the implementation of ak_hydro_stage (all of them CUDA kernels of this library; they give the
 * same results to rounding and exist as independent cross-checks for the tests):
 *   0 = production kernel: TMA-staged plane marching, worker threads + edge warp (default)
 *   1 = one thread per cell, recomputes everything (independent cross-check)
 *   2 = tiled plane marching with LDG staging (also taken automatically when ng - stencil radius is odd, where
 *       the TMA box origin would not be 16-byte aligned)
 * AK_EINVAL for any other value. */
int ak_pack_set_variant(ak_pack*, int variant);

/* Time integrator (paper P:105: low-storage SSP Runge-Kutta schemes): nstages = 2 selects
 * SSPRK(2,2) (default, two registers), nstages = 3 SSPRK(3,3), which needs a third caller-owned device buffer u_c
 * of ak_pack_state_bytes() (256-byte aligned; ignored for nstages = 2).  Stages are then ak_hydro_stage(p, 1..3, dt):
 * stage 1 A -> B, stage 2 B (and U^n in A) -> C, stage 3 C (and A) -> A.  Call on a bound pack between steps
 * (AK_ESTATE otherwise).  nstages = 1 is forward Euler ("RK1"): every ak_hydro_stage(p, 1, dt) is a whole step from
 * the current buffer into the other one (A and B alternate; u_c ignored).  Integrators other than the default run in
 * the production kernel only (AK_EUNSUPPORTED with other variants). */
int ak_pack_set_integrator(ak_pack*, int nstages, void* u_c);

/* Boundary condition per domain face, in the order x1min, x1max, x2min, x2max, x3min, x3max (paper P:67; SURVEY
 * 8(f) f3): 0 = periodic (default), 1 = outflow (ghost <- nearest active cell), 2 = reflect (ghost <- mirror image
 * across the face, normal momentum negated).  Periodic faces come in pairs (AK_EINVAL otherwise).  Call before
 * ak_pack_bind (a bound pack becomes unbound); outflow / reflect need a single-level mesh (bind: AK_EUNSUPPORTED). */
int ak_pack_set_boundaries(ak_pack*, const int bc[6]);

/* Flux correction at coarse-fine faces (paper P:57).  on != 0: after every ak_hydro_stage on a
 * refined mesh, the flux a level-0 cell used at a face shared with level-1 blocks is replaced by the mean of the
 * four fine fluxes through that face (three small extra launches per stage), which makes the update
 * conservative across level boundaries.  Off by default (north_star's stage list omits it); no effect on
 * single-level meshes. */
int ak_pack_set_flux_correction(ak_pack*, int on);

/* First-order flux correction, FOFC (paper P:118; off by default): after the stage kernel, every cell whose
 * tentative result has rho <= 0 or E - |rho v|^2 / (2 rho) <= 0 (NaN included) is flagged, and every face with a flagged
 * cell on either side trades its high-order flux for the LLF flux of the two cell-centred states of the stage's input
 * and the cells on both sides are updated again from the stage's inputs (three extra launches per stage, which return at
 * once when nothing was flagged).  Because that second update needs U^n, the last stage of a step cannot run in place:
 * u_spare is a fourth caller-owned device buffer of ak_pack_state_bytes() (256-byte aligned, disjoint from the others)
 * which the last stage writes and which then TRADES PLACES with buffer A (ak_pack_current() returns it).  Call on a bound
 * pack between steps; ak_pack_bind with buffers that overlap the spare switches FOFC off again.  Single-level meshes,
 * production kernel (ak_hydro_stage returns AK_EUNSUPPORTED otherwise).  on = 0: off (u_spare ignored).
 * ak_pack_fofc_count: cells flagged since bind (synchronises). */
int ak_pack_set_fofc(ak_pack*, int on, void* u_spare);
long long ak_pack_fofc_count(ak_pack*);

/* Fused ghost fill (default on).  On a single-level, fully periodic mesh with nx_d >= 2 ng the production kernel stores every cell it
 * writes within ng of a MeshBlock face also into the ghost cells of the neighbouring blocks (exact copies, the same
 * values ak_fill_ghosts would copy), so the ak_fill_ghosts that follows finds the ghost cells current and returns
 * without a launch; a step is then two launches.  on = 0 restores the separate fill pass (results bit-identical).
 * Refined meshes, non-periodic boundaries and variants 1, 2 always use the separate pass. */
int ak_pack_set_ghost_push(ak_pack*, int on);

/* Tile shape of the production kernel (variant 0): -1 = chosen from the block size (default);
 * 0 = 16x10 columns, 2 CTAs per SM; 1 = 16x8, 2 CTAs per SM; 2 = 16x22 and 3 = 32x11, 1 CTA per SM.
 * Results are bit-identical for every tile shape (tile-edge faces are solved with the same instruction
 * sequence by both tiles that share them).  AK_EINVAL for any other value. */
int ak_pack_set_tile(ak_pack*, int tile);

/* Number of kernel launches issued through this pack since bind (for bench.py's gpu_launches). */
long long ak_pack_launch_count(const ak_pack*);

/* Frees the host descriptor only; device buffers belong to the caller. */
int ak_pack_destroy(ak_pack*);

#ifdef __cplusplus
}
#endif
#endif

// ak_pack.h -- host descriptor and the plain-data view of a pack that kernels receive by value.
// Internal to the library (the public boundary is include/ak.h).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <string>
#include <vector>

namespace ak {

struct GasConst;

// Device-side view: everything a kernel needs to address U[m][n][k][j][i] and to find the
// leaf that covers a position (block tree of P:59 flattened into dense per-level maps).
struct PackDev {
  int nmb;
  int nx[3];        // active cells per block
  int ng;
  int nt[3];        // nx + 2 ng
  int nrb[3];       // root blocks per direction
  int max_level;    // 0 or 1
  long long ncell;  // nt0*nt1*nt2, stride between variables
  const int4* blk;  // (level, lx1, lx2, lx3) per block
  const int* leaf0; // [nrb3][nrb2][nrb1]       -> block index or -1
  const int* leaf1; // [2nrb3][2nrb2][2nrb1]    -> block index or -1
  const int* nbr;   // [nmb][27] same-level neighbour in direction (d3+1)*9+(d2+1)*3+(d1+1), or -1
  const int* nbc;   // [nmb][27] how to map the ghost index per direction: 2 bits each (d1 | d2<<2 | d3<<4),
                    // 0 = shift by one block length (periodic / interior), 1 = outflow, 2 = reflect
  double dx0[3];    // level-0 cell size; level 1 is exactly half
  double gamma;
  unsigned long long* dtmin_bits;   // scratch cell: min candidate dt as ordered bits
  unsigned long long* floor_cnt;    // scratch cell: floor activations
  unsigned long long* nonfinite;    // scratch cell: rows with a NaN / inf signal speed seen by new_dt_kernel
  unsigned long long* smax_bits;    // 6 scratch cells [level][d]: max |v_d| + c_s of U^{n+1} as ordered bits (stage 2)
};

struct StageCoef {
  double g0, g1;            // weights of U_in and U0
  double c[2][3];           // beta*dt/dx_d for level 0 and 1
  int take_dt;              // last stage of a step: also reduce the signal speeds of the result
  int push;                 // uniform periodic meshes: the writer of a cell also stores it into the neighbours' ghost cells
};

}  // namespace ak

struct ak_pack {
  ak::PackDev d{};
  int recon = 0, rsolver = 0;
  double xmin[3]{}, xmax[3]{};
  bool mesh_set = false, bound = false, ghosts_ok = false;
  bool dt_cached = false;         // smax_bits describe the current state (set by stage 2 of the production kernel)
  std::vector<int> level, lx;     // lx[3m+d]
  std::vector<char> blk_set;
  double* u[3] = {nullptr, nullptr, nullptr};   // A (U^n at the start of a step), B, C (third register, RK3 only)
  int integrator = 2;                           // stages per step: 2 = SSPRK(2,2), 3 = SSPRK(3,3)
  void* scratch = nullptr;
  cudaStream_t stream = nullptr;
  int cur = 0;
  int variant = 0;
  int bc[6] = {0, 0, 0, 0, 0, 0};  // ak_pack_set_boundaries: x1min,x1max,x2min,x2max,x3min,x3max
  bool flux_correction = false;   // ak_pack_set_flux_correction
  bool fofc = false;              // ak_pack_set_fofc: first-order flux correction, single-level meshes
  double* u_spare = nullptr;                  // FOFC: the last stage writes here instead of in place over A; then A and spare swap
  unsigned char* fofc_flags = nullptr;        // scratch: one flag per cell of every block
  unsigned long long* fofc_cnt = nullptr;     // scratch: cells flagged in the current stage, and since bind
  bool ghost_push = true;         // ak_pack_set_ghost_push: fuse the same-level periodic ghost fill into the stage kernel
  int tile = -1;                  // -1 = automatic (ak_pack_set_tile)
  long long launches = 0;
  int sm_count = 148;
  int device = -1;                // ordinal of the device that owns the buffers (set at bind)
  // tensor maps over u[0], u[1] for the TMA stage kernel, rebuilt when the staging box changes
  mutable CUtensorMap tmap[3];
  mutable int tmap_box[2] = {0, 0};
  // ... and the halo-free U0 boxes of the v3 kernel's stage 2
  mutable CUtensorMap tmap0[3];
  mutable int tmap0_box[2] = {0, 0};
};

namespace ak {
// records the message ak_last_error() returns (thread-local, ak_api.cu) and hands `code` back
int set_error(int code, const char* msg);
// launchers implemented in the .cu translation units; return cudaGetLastError()
cudaError_t launch_fill_ghosts(const ak_pack& p, double* U);
cudaError_t launch_new_dt(const ak_pack& p, const double* U);       // leaves the min in dtmin_bits
cudaError_t launch_stage(const ak_pack& p, const double* Uin, const double* U0, double* Uout,
                         const StageCoef& sc);
int stage_launches_per_call(const ak_pack& p);
// refined meshes, optional: three launches (one per direction) after launch_stage
cudaError_t launch_flux_correction(const ak_pack& p, const double* Uin, double* Uout, const StageCoef& sc);
// optional first-order flux correction after launch_stage (single-level meshes): memset + three launches
cudaError_t launch_fofc(const ak_pack& p, const double* Uin, const double* U0, double* Uout, const StageCoef& sc);
}  // namespace ak

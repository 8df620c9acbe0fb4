// ak_api.cu -- the C-ABI of include/ak.h: pack descriptor, mesh validation, table upload and the
// host-side sequencing of kernel launches (the host drives, the device computes).
#include "../../include/ak.h"
#include "ak_pack.h"

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <utility>

static thread_local std::string g_err;
static int fail(int code, const std::string& msg) { g_err = msg; return code; }
static int cuda_fail(cudaError_t e, const char* where) {
  return fail(AK_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
#define AK_CUDA(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, where); } while (0)

extern "C" const char* ak_last_error(void) { return g_err.c_str(); }
namespace ak { int set_error(int code, const char* msg) { return fail(code, msg); } }

// every launching entry point runs on the device that owns the pack's buffers, whatever the caller's current device
struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) { if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) cudaSetDevice(dev); else prev = -1; }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

static size_t align256(size_t n) { return (n + 255) & ~(size_t)255; }

// scratch layout: [0,256) reduction cells | block table int4[nmb] | leaf0 | leaf1 | same-level neighbours int[nmb][27]
struct ScratchLayout { size_t blk, leaf0, leaf1, nbr, nbc, flags, total; };
static ScratchLayout scratch_layout(const ak_pack* p) {
  ScratchLayout s;
  const ak::PackDev& d = p->d;
  size_t n0 = (size_t)d.nrb[0] * d.nrb[1] * d.nrb[2];
  s.blk = 256;
  s.leaf0 = s.blk + align256(sizeof(int4) * (size_t)d.nmb);
  s.leaf1 = s.leaf0 + align256(sizeof(int) * n0);
  s.nbr = s.leaf1 + align256(sizeof(int) * 8 * n0);
  s.nbc = s.nbr + align256(sizeof(int) * 27 * (size_t)d.nmb);
  s.flags = s.nbc + align256(sizeof(int) * 27 * (size_t)d.nmb);      // FOFC: one byte per cell
  s.total = s.flags + align256((size_t)d.nmb * (size_t)d.ncell);
  return s;
}

extern "C" ak_pack* ak_pack_create(int nmb, int nx1, int nx2, int nx3, int ng, double gamma, int recon, int rsolver) {
  int nx[3] = {nx1, nx2, nx3};
  if (nmb < 1) { fail(AK_EINVAL, "nmb < 1"); return nullptr; }
  if (ng > 4) { fail(AK_EINVAL, "ng > 4"); return nullptr; }
  for (int d = 0; d < 3; d++)
    if (nx[d] < ng || (nx[d] & 1) || nx[d] < 2) { fail(AK_EINVAL, "nx_d must be even and >= ng"); return nullptr; }
  if (!(gamma > 1.0)) { fail(AK_EINVAL, "gamma <= 1"); return nullptr; }
  if (recon < AK_RECON_PLM || recon > AK_RECON_WENOZ) { fail(AK_EINVAL, "unknown recon"); return nullptr; }
  if (rsolver < AK_RSOLVER_HLLC || rsolver > AK_RSOLVER_ROE) { fail(AK_EINVAL, "unknown rsolver"); return nullptr; }
  if ((recon == AK_RECON_PLM && ng < 2) || (recon >= AK_RECON_PPM4 && ng < 3)) {
    fail(AK_EINVAL, "ng too small for the reconstruction stencil"); return nullptr;
  }
  long long ncell = (long long)(nx1 + 2 * ng) * (nx2 + 2 * ng) * (nx3 + 2 * ng);
  if (ncell * 5 * nmb >= (1ll << 40)) { fail(AK_EUNSUPPORTED, "pack too large"); return nullptr; }
  if ((long long)nx2 * nx3 > 65535 || nmb > 65535) { fail(AK_EUNSUPPORTED, "grid dimension limit"); return nullptr; }
  ak_pack* p = new ak_pack;
  p->d.nmb = nmb; p->d.ng = ng; p->d.gamma = gamma; p->d.ncell = ncell;
  for (int d = 0; d < 3; d++) { p->d.nx[d] = nx[d]; p->d.nt[d] = nx[d] + 2 * ng; p->d.nrb[d] = 0; }
  p->recon = recon; p->rsolver = rsolver;
  p->level.assign(nmb, 0); p->lx.assign(3 * (size_t)nmb, 0); p->blk_set.assign(nmb, 0);
  return p;
}

extern "C" int ak_pack_set_mesh(ak_pack* p, int nrb1, int nrb2, int nrb3, double x1min, double x1max,
                                double x2min, double x2max, double x3min, double x3max) {
  if (!p) return fail(AK_EINVAL, "null pack");
  if (nrb1 < 1 || nrb2 < 1 || nrb3 < 1) return fail(AK_EINVAL, "nrb < 1");
  if (!(x1max > x1min) || !(x2max > x2min) || !(x3max > x3min)) return fail(AK_EINVAL, "empty domain");
  int nrb[3] = {nrb1, nrb2, nrb3};
  for (int d = 0; d < 3; d++) if ((long long)nrb[d] * p->d.nx[d] * 2 > (1ll << 30)) return fail(AK_EUNSUPPORTED, "mesh too large");
  p->d.nrb[0] = nrb1; p->d.nrb[1] = nrb2; p->d.nrb[2] = nrb3;
  p->xmin[0] = x1min; p->xmax[0] = x1max; p->xmin[1] = x2min; p->xmax[1] = x2max; p->xmin[2] = x3min; p->xmax[2] = x3max;
  for (int d = 0; d < 3; d++) p->d.dx0[d] = (p->xmax[d] - p->xmin[d]) / ((double)nrb[d] * p->d.nx[d] * 1.0);
  p->mesh_set = true; p->bound = false;
  return AK_OK;
}

extern "C" int ak_pack_set_block(ak_pack* p, int m, int level, int lx1, int lx2, int lx3) {
  if (!p) return fail(AK_EINVAL, "null pack");
  if (!p->mesh_set) return fail(AK_ESTATE, "ak_pack_set_mesh first");
  if (m < 0 || m >= p->d.nmb) return fail(AK_EINVAL, "block index out of range");
  if (level < 0) return fail(AK_EINVAL, "negative level");
  if (level > 1) return fail(AK_EUNSUPPORTED, "only levels 0 and 1 are supported");
  int l[3] = {lx1, lx2, lx3};
  for (int d = 0; d < 3; d++) if (l[d] < 0 || l[d] >= (p->d.nrb[d] << level)) return fail(AK_EINVAL, "logical location out of range");
  p->level[m] = level;
  for (int d = 0; d < 3; d++) p->lx[3 * (size_t)m + d] = l[d];
  p->blk_set[m] = 1; p->bound = false;
  return AK_OK;
}

extern "C" size_t ak_pack_state_bytes(const ak_pack* p) { return p ? (size_t)p->d.nmb * 5 * (size_t)p->d.ncell * 8 : 0; }
extern "C" size_t ak_pack_scratch_bytes(const ak_pack* p) { return (p && p->mesh_set) ? scratch_layout(p).total : 0; }

extern "C" int ak_pack_bind(ak_pack* p, void* u_a, void* u_b, void* scratch, void* cuda_stream) {
  if (!p) return fail(AK_EINVAL, "null pack");
  if (!p->mesh_set) return fail(AK_ESTATE, "ak_pack_set_mesh first");
  if (!u_a || !u_b || !scratch) return fail(AK_EINVAL, "null device buffer");
  if (((uintptr_t)u_a | (uintptr_t)u_b | (uintptr_t)scratch) & 255) return fail(AK_EINVAL, "buffers must be 256-byte aligned");
  const size_t sb = ak_pack_state_bytes(p);
  auto overlap = [](const void* a, size_t na, const void* b, size_t nb) {
    return (uintptr_t)a < (uintptr_t)b + nb && (uintptr_t)b < (uintptr_t)a + na;
  };
  const ScratchLayout sl = scratch_layout(p);
  if (overlap(u_a, sb, u_b, sb) || overlap(u_a, sb, scratch, sl.total) || overlap(u_b, sb, scratch, sl.total))
    return fail(AK_EINVAL, "device buffers overlap");
  ak::PackDev& d = p->d;
  // ---- validate the block list: leaves must tile the root grid (P:59 block tree, two levels) ----
  const size_t n0 = (size_t)d.nrb[0] * d.nrb[1] * d.nrb[2];
  std::vector<int> leaf0(n0, -1), leaf1(8 * n0, -1);
  d.max_level = 0;
  for (int m = 0; m < d.nmb; m++) {
    if (!p->blk_set[m]) return fail(AK_ESTATE, "ak_pack_set_block missing for a block");
    const int* l = &p->lx[3 * (size_t)m];
    if (p->level[m] == 0) {
      size_t k = ((size_t)l[2] * d.nrb[1] + l[1]) * d.nrb[0] + l[0];
      if (leaf0[k] >= 0) return fail(AK_EINVAL, "duplicate block");
      leaf0[k] = m;
    } else {
      size_t k = ((size_t)l[2] * 2 * d.nrb[1] + l[1]) * 2 * d.nrb[0] + l[0];
      if (leaf1[k] >= 0) return fail(AK_EINVAL, "duplicate block");
      leaf1[k] = m;
      d.max_level = 1;
    }
  }
  for (int b3 = 0; b3 < d.nrb[2]; b3++) for (int b2 = 0; b2 < d.nrb[1]; b2++) for (int b1 = 0; b1 < d.nrb[0]; b1++) {
    int nchild = 0;
    for (int c = 0; c < 8; c++) {
      size_t k = ((size_t)(2 * b3 + (c >> 2)) * 2 * d.nrb[1] + (2 * b2 + ((c >> 1) & 1))) * 2 * d.nrb[0] + (2 * b1 + (c & 1));
      if (leaf1[k] >= 0) nchild++;
    }
    bool root_leaf = leaf0[((size_t)b3 * d.nrb[1] + b2) * d.nrb[0] + b1] >= 0;
    if (root_leaf && nchild) return fail(AK_EINVAL, "overlapping leaves");
    if (!root_leaf && nchild != 8) return fail(AK_EINVAL, "leaves do not cover the domain");
  }
  if (d.max_level > 0 && (d.ng & 1)) return fail(AK_EUNSUPPORTED, "static refinement needs even ng");
  for (int f = 0; f < 6; f++)
    if (p->bc[f] != 0 && d.max_level > 0) return fail(AK_EUNSUPPORTED, "outflow / reflecting boundaries need a single-level mesh");
  // ---- upload tables ----
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::vector<int4> blk(d.nmb);
  for (int m = 0; m < d.nmb; m++) blk[m] = make_int4(p->level[m], p->lx[3 * m], p->lx[3 * m + 1], p->lx[3 * m + 2]);
  // same-level neighbour of block m in direction (d1, d2, d3) in {-1,0,1}^3 (periodic wrap), or -1 where the
  // position is covered by a leaf of another level (the ghost fill then takes the general path)
  std::vector<int> nbr(27 * (size_t)d.nmb, -1), nbc(27 * (size_t)d.nmb, 0);
  for (int m = 0; m < d.nmb; m++) {
    const int lev = p->level[m];
    const int nb[3] = {d.nrb[0] << lev, d.nrb[1] << lev, d.nrb[2] << lev};
    const std::vector<int>& leaf = lev ? leaf1 : leaf0;
    for (int d3 = -1; d3 <= 1; d3++) for (int d2 = -1; d2 <= 1; d2++) for (int d1 = -1; d1 <= 1; d1++) {
      const int dd[3] = {d1, d2, d3};
      int b[3], code = 0;
      for (int e = 0; e < 3; e++) {
        b[e] = p->lx[3 * m + e] + dd[e];
        if (b[e] < 0 || b[e] >= nb[e]) {
          const int kind = p->bc[2 * e + (b[e] < 0 ? 0 : 1)];
          if (kind == 0) b[e] = (b[e] + nb[e]) % nb[e];              // periodic wrap
          else { b[e] = p->lx[3 * m + e]; code |= kind << (2 * e); }  // image lies in the boundary block itself
        }
      }
      const size_t k = 27 * (size_t)m + (d3 + 1) * 9 + (d2 + 1) * 3 + (d1 + 1);
      nbr[k] = leaf[((size_t)b[2] * nb[1] + b[1]) * nb[0] + b[0]];
      nbc[k] = code;
    }
  }
  {
    // the device that owns u_a runs every kernel of this pack (not whatever device is current at call time)
    cudaPointerAttributes pa;
    AK_CUDA(cudaPointerGetAttributes(&pa, u_a), "cudaPointerGetAttributes");
    if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) return fail(AK_EINVAL, "u_a is not a device pointer");
    p->device = pa.device;
  }
  DeviceGuard guard(p->device);
  char* s = (char*)scratch;
  AK_CUDA(cudaMemsetAsync(s, 0, 256, st), "memset scratch");
  AK_CUDA(cudaMemcpyAsync(s + sl.nbr, nbr.data(), sizeof(int) * nbr.size(), cudaMemcpyHostToDevice, st), "upload neighbour table");
  AK_CUDA(cudaMemcpyAsync(s + sl.nbc, nbc.data(), sizeof(int) * nbc.size(), cudaMemcpyHostToDevice, st), "upload boundary table");
  AK_CUDA(cudaMemcpyAsync(s + sl.blk, blk.data(), sizeof(int4) * d.nmb, cudaMemcpyHostToDevice, st), "upload block table");
  AK_CUDA(cudaMemcpyAsync(s + sl.leaf0, leaf0.data(), sizeof(int) * n0, cudaMemcpyHostToDevice, st), "upload leaf map 0");
  AK_CUDA(cudaMemcpyAsync(s + sl.leaf1, leaf1.data(), sizeof(int) * 8 * n0, cudaMemcpyHostToDevice, st), "upload leaf map 1");
  AK_CUDA(cudaStreamSynchronize(st), "bind sync");
  d.dtmin_bits = (unsigned long long*)s;
  d.floor_cnt = (unsigned long long*)(s + 8);
  d.nonfinite = (unsigned long long*)(s + 16);
  p->fofc_cnt = (unsigned long long*)(s + 24);           // [0] this stage, [1] since bind
  p->fofc_flags = (unsigned char*)(s + sl.flags);
  d.smax_bits = (unsigned long long*)(s + 64);
  d.blk = (const int4*)(s + sl.blk);
  d.leaf0 = (const int*)(s + sl.leaf0);
  d.leaf1 = (const int*)(s + sl.leaf1);
  d.nbr = (const int*)(s + sl.nbr);
  d.nbc = (const int*)(s + sl.nbc);
  AK_CUDA(cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device), "query SM count");
  p->u[0] = (double*)u_a; p->u[1] = (double*)u_b; p->scratch = scratch; p->stream = st;
  // a third register bound earlier (SSPRK(3,3)) stays valid only if it is still disjoint from the new buffers
  if (p->u[2] && (overlap(p->u[2], sb, u_a, sb) || overlap(p->u[2], sb, u_b, sb) || overlap(p->u[2], sb, scratch, sl.total))) {
    p->u[2] = nullptr; p->integrator = 2;
  }
  // likewise the FOFC spare (after a step it has traded places with A: re-arm FOFC after re-binding the old buffers)
  if (p->u_spare && (overlap(p->u_spare, sb, u_a, sb) || overlap(p->u_spare, sb, u_b, sb) || overlap(p->u_spare, sb, scratch, sl.total))) {
    p->u_spare = nullptr; p->fofc = false;
  }
  p->cur = 0; p->ghosts_ok = false; p->bound = true; p->launches = 0; p->dt_cached = false;
  p->tmap_box[0] = p->tmap_box[1] = 0;
  p->tmap0_box[0] = p->tmap0_box[1] = 0;
  return AK_OK;
}

extern "C" int ak_pack_set_variant(ak_pack* p, int variant) {
  if (!p) return fail(AK_EINVAL, "null pack");
  if (variant < 0 || variant > 2) return fail(AK_EINVAL, "unknown variant");
  p->variant = variant;
  return AK_OK;
}

extern "C" int ak_pack_set_integrator(ak_pack* p, int nstages, void* u_c) {
  if (!p) return fail(AK_EINVAL, "null pack");
  if (nstages < 1 || nstages > 3) return fail(AK_EINVAL, "integrator must be 1 (forward Euler), 2 (SSPRK(2,2)) or 3 (SSPRK(3,3))");
  if (nstages == 3) {
    if (!u_c) return fail(AK_EINVAL, "SSPRK(3,3) needs a third state buffer");
    if ((uintptr_t)u_c & 255) return fail(AK_EINVAL, "buffers must be 256-byte aligned");
    if (!p->bound) return fail(AK_ESTATE, "bind the pack first");
    const size_t sb = ak_pack_state_bytes(p), ss = scratch_layout(p).total;
    auto overlap = [](const void* a, size_t na, const void* b, size_t nb) {
      return (uintptr_t)a < (uintptr_t)b + nb && (uintptr_t)b < (uintptr_t)a + na;
    };
    if (overlap(u_c, sb, p->u[0], sb) || overlap(u_c, sb, p->u[1], sb) || overlap(u_c, sb, p->scratch, ss))
      return fail(AK_EINVAL, "device buffers overlap");
  }
  if (p->bound && p->cur != 0 && !(p->integrator == 1 && p->cur == 1)) return fail(AK_ESTATE, "change the integrator between steps");
  if (p->bound && p->cur == 1 && nstages != 1)
    return fail(AK_ESTATE, "after an odd number of forward-Euler steps U^n is in buffer B: take one more or reload");
  p->integrator = nstages;
  p->u[2] = (nstages == 3) ? (double*)u_c : nullptr;
  p->tmap_box[0] = p->tmap_box[1] = 0;          // tensor maps are rebuilt over all bound buffers
  p->tmap0_box[0] = p->tmap0_box[1] = 0;
  return AK_OK;
}

extern "C" int ak_pack_set_boundaries(ak_pack* p, const int bc[6]) {
  if (!p || !bc) return fail(AK_EINVAL, "null argument");
  for (int f = 0; f < 6; f++) if (bc[f] < 0 || bc[f] > 2) return fail(AK_EINVAL, "unknown boundary condition");
  for (int e = 0; e < 3; e++)
    if ((bc[2 * e] == 0) != (bc[2 * e + 1] == 0)) return fail(AK_EINVAL, "periodic faces come in pairs");
  for (int f = 0; f < 6; f++) p->bc[f] = bc[f];
  p->bound = false;                     // the neighbour tables are built at bind
  return AK_OK;
}

extern "C" int ak_pack_set_flux_correction(ak_pack* p, int on) {
  if (!p) return fail(AK_EINVAL, "null pack");
  p->flux_correction = on != 0;
  return AK_OK;
}

extern "C" int ak_pack_set_fofc(ak_pack* p, int on, void* u_spare) {
  if (!p) return fail(AK_EINVAL, "null pack");
  if (!on) { p->fofc = false; p->u_spare = nullptr; return AK_OK; }
  if (!p->bound) return fail(AK_ESTATE, "bind the pack first");
  if (!u_spare) return fail(AK_EINVAL, "FOFC needs a spare state buffer (the last stage of a step cannot run in place)");
  if ((uintptr_t)u_spare & 255) return fail(AK_EINVAL, "buffers must be 256-byte aligned");
  if (p->cur != 0 && !(p->integrator == 1)) return fail(AK_ESTATE, "switch FOFC on between steps");
  const size_t sb = ak_pack_state_bytes(p), ss = scratch_layout(p).total;
  auto overlap = [](const void* a, size_t na, const void* b, size_t nb) {
    return (uintptr_t)a < (uintptr_t)b + nb && (uintptr_t)b < (uintptr_t)a + na;
  };
  for (int b = 0; b < 3; b++) if (p->u[b] && overlap(u_spare, sb, p->u[b], sb)) return fail(AK_EINVAL, "device buffers overlap");
  if (overlap(u_spare, sb, p->scratch, ss)) return fail(AK_EINVAL, "device buffers overlap");
  p->fofc = true;
  p->u_spare = (double*)u_spare;
  return AK_OK;
}

extern "C" long long ak_pack_fofc_count(ak_pack* p) {
  if (!p || !p->bound) { fail(AK_ESTATE, "pack not bound"); return -1; }
  DeviceGuard guard(p->device);
  unsigned long long n = 0;
  if (cudaMemcpyAsync(&n, p->fofc_cnt + 1, 8, cudaMemcpyDeviceToHost, p->stream) != cudaSuccess ||
      cudaStreamSynchronize(p->stream) != cudaSuccess) { fail(AK_ECUDA, "ak_pack_fofc_count copy failed"); return -1; }
  return (long long)n;
}

extern "C" int ak_pack_set_ghost_push(ak_pack* p, int on) {
  if (!p) return fail(AK_EINVAL, "null pack");
  p->ghost_push = on != 0;
  return AK_OK;
}

extern "C" int ak_pack_set_tile(ak_pack* p, int tile) {
  if (!p) return fail(AK_EINVAL, "null pack");
  if (tile < -1 || tile > 3) return fail(AK_EINVAL, "unknown tile shape");
  p->tile = tile;
  return AK_OK;
}

extern "C" int ak_fill_ghosts(ak_pack* p) {
  if (!p || !p->bound) return fail(AK_ESTATE, "pack not bound");
  if (p->ghosts_ok) return AK_OK;       // already current: the stage that wrote the state also wrote its ghost copies
  DeviceGuard guard(p->device);
  AK_CUDA(ak::launch_fill_ghosts(*p, p->u[p->cur]), "ak_fill_ghosts launch");
  p->launches += 1;
  p->ghosts_ok = true;
  return AK_OK;
}

extern "C" int ak_hydro_stage(ak_pack* p, int stage, double dt) {
  if (!p || !p->bound) return fail(AK_ESTATE, "pack not bound");
  DeviceGuard guard(p->device);
  if (stage < 1 || stage > p->integrator) return fail(AK_EINVAL, "stage must be 1 .. number of stages of the integrator");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(AK_EINVAL, "dt must be positive and finite");
  if (p->integrator == 1 ? p->cur > 1 : p->cur != stage - 1)
    return fail(AK_ESTATE, stage == 1 ? "stage 1 expects U^n in buffer A (finish the previous step first)"
                                      : "stages must be called in order (the previous stage's result is not current)");
  if (!p->ghosts_ok) return fail(AK_ESTATE, "ak_fill_ghosts must precede ak_hydro_stage");
  if (p->rsolver != AK_RSOLVER_HLLC && (p->variant != 0 || ((p->d.ng - (p->recon == 0 ? 2 : 3)) & 1)))
    return fail(AK_EUNSUPPORTED, "LLF / HLLE / Roe exist in the production kernel only (variant 0, ng - stencil radius even)");
  if (p->recon >= AK_RECON_PPMX && (p->variant != 0 || ((p->d.ng - 3) & 1) || p->rsolver != AK_RSOLVER_HLLC))
    return fail(AK_EUNSUPPORTED, "PPMX / WENOZ exist in the production kernel with HLLC only (variant 0, ng - 3 even)");
  // Shu-Osher forms, every stage U_out = g0 U_in + g1 U^n + beta dt L(U_in) (Q1, Q27):
  //   SSPRK(2,2): (0,1,1), (1/2,1/2,1/2);   SSPRK(3,3): (0,1,1), (1/4,3/4,1/4), (2/3,1/3,2/3)
  static const double C2[2][3] = {{0.0, 1.0, 1.0}, {0.5, 0.5, 0.5}};
  static const double C3[3][3] = {{0.0, 1.0, 1.0}, {0.25, 0.75, 0.25}, {2.0 / 3.0, 1.0 / 3.0, 2.0 / 3.0}};
  const double* cf = (p->integrator == 2) ? C2[stage - 1] : C3[stage - 1];
  ak::StageCoef sc;
  const double beta = cf[2];
  sc.g0 = cf[0];
  sc.g1 = cf[1];
  // the last stage writes A in place (a cell's A value is read only by its own thread); the others the next buffer
  // (forward Euler has no second register to combine with: it writes the other buffer, A and B alternate)
  const int out = (p->integrator == 1) ? 1 - p->cur : ((stage == p->integrator) ? 0 : stage);
  const double* u0 = (p->integrator == 1) ? p->u[p->cur] : p->u[0];
  for (int lev = 0; lev < 2; lev++)
    for (int d = 0; d < 3; d++) {
      double dx = (p->xmax[d] - p->xmin[d]) / ((double)p->d.nrb[d] * p->d.nx[d] * (double)(1 << lev));
      sc.c[lev][d] = beta * dt / dx;
    }
  if (p->fofc && (p->d.max_level > 0 || p->variant != 0 || ((p->d.ng - (p->recon == 0 ? 2 : 3)) & 1)))
    return fail(AK_EUNSUPPORTED, "FOFC is implemented for the production kernel on single-level meshes");
  // stage 2 of the production kernel also leaves the max signal speeds of U^{n+1} for the next ak_new_dt
  const bool v3 = p->variant == 0 && !((p->d.ng - (p->recon == 0 ? 2 : 3)) & 1);
  if (p->integrator != 2 && !v3) return fail(AK_EUNSUPPORTED, "forward Euler and SSPRK(3,3) exist in the production kernel only");
  const bool last = stage == p->integrator;
  sc.take_dt = (last && stage >= 2 && !p->fofc) ? 1 : 0;      // (FOFC may change cells after the stage)
  // uniform, fully periodic meshes: the production kernel stores every boundary cell into the neighbours' ghost
  // cells as it writes it, so the next ak_fill_ghosts has nothing left to do
  bool periodic = true;
  for (int f = 0; f < 6; f++) periodic = periodic && p->bc[f] == 0;
  for (int d = 0; d < 3; d++) periodic = periodic && p->d.nx[d] >= 2 * p->d.ng;    // (a cell is near one face per direction)
  sc.push = (v3 && p->ghost_push && p->d.max_level == 0 && periodic && !p->fofc) ? 1 : 0;
  p->dt_cached = false;
  if (sc.take_dt && v3) AK_CUDA(cudaMemsetAsync(p->d.smax_bits, 0, 48, p->stream), "reset signal speeds");
  // with FOFC a cell may have to be updated again from U_in and U0, so the last stage must not overwrite U0 = A in place:
  // it writes the spare buffer, which then trades places with A
  const bool to_spare = p->fofc && p->integrator >= 2 && last;
  double* uout = to_spare ? p->u_spare : p->u[out];
  AK_CUDA(ak::launch_stage(*p, p->u[p->cur], u0, uout, sc), "ak_hydro_stage launch");
  p->launches += ak::stage_launches_per_call(*p);
  if (sc.take_dt && v3) p->dt_cached = true;
  if (p->fofc) {
    // first-order fluxes on the faces of cells whose tentative result is unphysical (before any flux correction
    // at level boundaries -- moot here: single-level meshes)
    AK_CUDA(ak::launch_fofc(*p, p->u[p->cur], u0, uout, sc), "FOFC launch");
    p->launches += 3;
    if (to_spare) {
      std::swap(p->u[0], p->u_spare);
      p->tmap_box[0] = p->tmap_box[1] = 0;        // the tensor maps follow the buffers
      p->tmap0_box[0] = p->tmap0_box[1] = 0;
    }
  }
  if (p->flux_correction && p->d.max_level > 0) {
    AK_CUDA(ak::launch_flux_correction(*p, p->u[p->cur], p->u[out], sc), "flux correction launch");
    p->launches += 3;
    p->dt_cached = false;               // the correction changed cells after their signal speeds were taken
  }
  p->cur = out;
  p->ghosts_ok = sc.push != 0;
  return AK_OK;
}

extern "C" int ak_new_dt(ak_pack* p, double cfl, double* dt_out) {
  if (!p || !p->bound) return fail(AK_ESTATE, "pack not bound");
  DeviceGuard guard(p->device);
  if (!dt_out) return fail(AK_EINVAL, "null dt_out");
  if (!(cfl > 0.0)) return fail(AK_EINVAL, "cfl must be positive");
  double dtmin = 0.0;
  if (p->dt_cached) {
    // min over cells of dx_d / (|v_d| + c_s) = dx_d / max(|v_d| + c_s), bit for bit (IEEE division is monotone in
    // its divisor); the maxima per level and direction were taken by stage 2 from the values it wrote
    double s[6];
    AK_CUDA(cudaMemcpyAsync(s, p->d.smax_bits, 48, cudaMemcpyDeviceToHost, p->stream), "ak_new_dt copy");
    AK_CUDA(cudaStreamSynchronize(p->stream), "ak_new_dt sync");
    dtmin = HUGE_VAL;
    for (int lev = 0; lev < 2; lev++)
      for (int d = 0; d < 3; d++) {
        const double dx = (lev ? 0.5 : 1.0) * p->d.dx0[d];
        // the maxima were taken on the bit patterns, where every NaN and +inf orders above all finite speeds, so a
        // single corrupted cell survives the reduction; an all-zero pattern means the level holds no block
        const double sv = s[3 * lev + d];
        if (sv != sv || sv == HUGE_VAL) return fail(AK_ENONFINITE, "non-finite signal speed in the state (NaN or inf in an active cell)");
        if (sv > 0.0) dtmin = std::fmin(dtmin, dx / sv);
      }
  } else {
    AK_CUDA(ak::launch_new_dt(*p, p->u[p->cur]), "ak_new_dt launch");
    p->launches += 2;
    unsigned long long cells[3];    // dtmin bits, floor counter, non-finite rows
    AK_CUDA(cudaMemcpyAsync(cells, p->d.dtmin_bits, 24, cudaMemcpyDeviceToHost, p->stream), "ak_new_dt copy");
    AK_CUDA(cudaStreamSynchronize(p->stream), "ak_new_dt sync");
    if (cells[2]) return fail(AK_ENONFINITE, "non-finite signal speed in the state (NaN or inf in an active cell)");
    std::memcpy(&dtmin, &cells[0], 8);
  }
  if (!(dtmin > 0.0) || !std::isfinite(dtmin))
    return fail(AK_ENONFINITE, "non-finite signal speed in the state (NaN or inf in an active cell)");
  *dt_out = cfl * dtmin;
  return AK_OK;
}

extern "C" int ak_step(ak_pack* p, double cfl, double dt_fixed, double* dt_out) {
  double dt = dt_fixed;
  if (!(dt_fixed > 0.0)) { int rc = ak_new_dt(p, cfl, &dt); if (rc) return rc; }
  for (int stage = 1; stage <= p->integrator; stage++) {
    int rc = ak_fill_ghosts(p); if (rc) return rc;
    rc = ak_hydro_stage(p, stage, dt); if (rc) return rc;
  }
  if (dt_out) *dt_out = dt;
  return AK_OK;
}

extern "C" void* ak_pack_current(const ak_pack* p) { return (p && p->bound) ? (void*)p->u[p->cur] : nullptr; }

extern "C" int ak_pack_upload(ak_pack* p, const void* host_u) {
  if (!p || !p->bound) return fail(AK_ESTATE, "pack not bound");
  DeviceGuard guard(p->device);
  if (!host_u) return fail(AK_EINVAL, "null host buffer");
  AK_CUDA(cudaMemcpyAsync(p->u[0], host_u, ak_pack_state_bytes(p), cudaMemcpyHostToDevice, p->stream), "ak_pack_upload");
  p->cur = 0; p->ghosts_ok = false; p->dt_cached = false;
  return AK_OK;
}

extern "C" int ak_pack_download_async(ak_pack* p, void* host_u) {
  if (!p || !p->bound) return fail(AK_ESTATE, "pack not bound");
  DeviceGuard guard(p->device);
  if (!host_u) return fail(AK_EINVAL, "null host buffer");
  AK_CUDA(cudaMemcpyAsync(host_u, p->u[p->cur], ak_pack_state_bytes(p), cudaMemcpyDeviceToHost, p->stream), "ak_pack_download_async");
  return AK_OK;
}

extern "C" int ak_pack_download(ak_pack* p, void* host_u) {
  if (!p || !p->bound) return fail(AK_ESTATE, "pack not bound");
  DeviceGuard guard(p->device);
  if (!host_u) return fail(AK_EINVAL, "null host buffer");
  AK_CUDA(cudaMemcpyAsync(host_u, p->u[p->cur], ak_pack_state_bytes(p), cudaMemcpyDeviceToHost, p->stream), "ak_pack_download");
  AK_CUDA(cudaStreamSynchronize(p->stream), "ak_pack_download sync");
  return AK_OK;
}

extern "C" long long ak_pack_floor_count(ak_pack* p) {
  if (!p || !p->bound) { fail(AK_ESTATE, "pack not bound"); return -1; }
  DeviceGuard guard(p->device);
  unsigned long long n = 0;
  if (cudaMemcpyAsync(&n, p->d.floor_cnt, 8, cudaMemcpyDeviceToHost, p->stream) != cudaSuccess ||
      cudaStreamSynchronize(p->stream) != cudaSuccess) { fail(AK_ECUDA, "ak_pack_floor_count copy failed"); return -1; }
  return (long long)n;
}

extern "C" long long ak_pack_launch_count(const ak_pack* p) { return p ? p->launches : -1; }

extern "C" int ak_pack_destroy(ak_pack* p) { delete p; return AK_OK; }

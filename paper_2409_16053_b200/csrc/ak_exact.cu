// ak_exact.cu -- kernels whose results must match the oracle BIT-EXACTLY: ghost fill (same-level
// copy, restriction, prolongation) and the CFL reduction (Eq.(3)).
// Compiled with -fmad=false and IEEE division / sqrt, so every expression rounds once per
// operation in the order written.
#define AK_EXACT_MATH 1
#include "ak_pack.h"
#include "ak_physics.cuh"
#include <cstring>

namespace ak {

__device__ __forceinline__ int nglob(const PackDev& P, int lev, int d) { return (P.nrb[d] * P.nx[d]) << lev; }

__device__ __forceinline__ int find_leaf(const PackDev& P, int lev, int b1, int b2, int b3) {
  if (lev == 0) return P.leaf0[(b3 * P.nrb[1] + b2) * P.nrb[0] + b1];
  if (P.max_level < 1) return -1;
  return P.leaf1[(b3 * (2 * P.nrb[1]) + b2) * (2 * P.nrb[0]) + b1];
}

// address of variable 0 of the active cell with level-`lev` global index G (wrapped) in leaf m
__device__ __forceinline__ long long leaf_cell(const PackDev& P, int m, int4 b, int G1, int G2, int G3) {
  int i = G1 - b.y * P.nx[0] + P.ng, j = G2 - b.z * P.nx[1] + P.ng, k = G3 - b.w * P.nx[2] + P.ng;
  return (long long)m * 5 * P.ncell + ((long long)k * P.nt[1] + j) * P.nt[0] + i;
}

// G3: conservative restriction of the 8 level-(lev+1) cells under level-`lev` cell G (fixed order).
// Returns false if no finer leaf covers the cell.
__device__ bool restrict5(const PackDev& P, const double* __restrict__ U, int lev, int G1, int G2, int G3, double out[5]) {
  // the 8 children live in one fine block because nx_d is even
  int F1 = 2 * G1, F2 = 2 * G2, F3 = 2 * G3;
  int m = find_leaf(P, lev + 1, F1 / P.nx[0], F2 / P.nx[1], F3 / P.nx[2]);
  if (m < 0) return false;
  long long a = leaf_cell(P, m, P.blk[m], F1, F2, F3);
  const long long sj = P.nt[0], sk = (long long)P.nt[0] * P.nt[1];
  for (int n = 0; n < 5; n++) {
    const double* q = U + a + n * P.ncell;
    double f000 = q[0], f100 = q[1], f010 = q[sj], f110 = q[sj + 1];
    double f001 = q[sk], f101 = q[sk + 1], f011 = q[sk + sj], f111 = q[sk + sj + 1];
    out[n] = 0.125 * (((f000 + f100) + (f010 + f110)) + ((f001 + f101) + (f011 + f111)));
  }
  return true;
}

__device__ __forceinline__ int wrap1(int g, int n) { return g < 0 ? g + n : (g >= n ? g - n : g); }

// virtual level-`lev` field C(.) of G4: leaf value where a level-`lev` leaf covers G, else restriction
__device__ bool coarse5(const PackDev& P, const double* __restrict__ U, int lev, int G1, int G2, int G3, double out[5]) {
  G1 = wrap1(G1, nglob(P, lev, 0)); G2 = wrap1(G2, nglob(P, lev, 1)); G3 = wrap1(G3, nglob(P, lev, 2));
  int m = find_leaf(P, lev, G1 / P.nx[0], G2 / P.nx[1], G3 / P.nx[2]);
  if (m >= 0) {
    long long a = leaf_cell(P, m, P.blk[m], G1, G2, G3);
    for (int n = 0; n < 5; n++) out[n] = U[a + n * P.ncell];
    return true;
  }
  return restrict5(P, U, lev, G1, G2, G3, out);
}

__device__ __forceinline__ double minmod(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  double m = fmin(fabs(a), fabs(b));
  return a > 0.0 ? m : -m;
}

// General path (G1-G4 of DESIGN.md): value of ghost cell (i, j, k) of block m from the leaf maps.
__device__ void ghost_general(const PackDev& P, const double* __restrict__ U, int m, int i, int j, int k, double val[5]) {
  const int ng = P.ng;
  const int4 b = P.blk[m];
  const int lev = b.x;
  // G1: which leaf covers the periodic image of this ghost cell?
  const int G1 = wrap1(b.y * P.nx[0] + i - ng, nglob(P, lev, 0));
  const int G2 = wrap1(b.z * P.nx[1] + j - ng, nglob(P, lev, 1));
  const int G3 = wrap1(b.w * P.nx[2] + k - ng, nglob(P, lev, 2));
  const int src = find_leaf(P, lev, G1 / P.nx[0], G2 / P.nx[1], G3 / P.nx[2]);
  if (src >= 0) {                                           // G2: same level, copy
    long long a = leaf_cell(P, src, P.blk[src], G1, G2, G3);
    for (int n = 0; n < 5; n++) val[n] = U[a + n * P.ncell];
  } else if (lev == 0) {                                    // G3: finer neighbour
    restrict5(P, U, 0, G1, G2, G3, val);
  } else {                                                  // G4: coarser neighbour
    const int C1 = G1 >> 1, C2 = G2 >> 1, C3 = G3 >> 1;
    const double s1 = (double)(2 * (G1 & 1) - 1), s2 = (double)(2 * (G2 & 1) - 1), s3 = (double)(2 * (G3 & 1) - 1);
    double c0[5], cm[5], cp[5], g1[5], g2[5], g3[5];
    coarse5(P, U, lev - 1, C1, C2, C3, c0);
    coarse5(P, U, lev - 1, C1 - 1, C2, C3, cm); coarse5(P, U, lev - 1, C1 + 1, C2, C3, cp);
    for (int n = 0; n < 5; n++) g1[n] = 0.25 * minmod(c0[n] - cm[n], cp[n] - c0[n]);
    coarse5(P, U, lev - 1, C1, C2 - 1, C3, cm); coarse5(P, U, lev - 1, C1, C2 + 1, C3, cp);
    for (int n = 0; n < 5; n++) g2[n] = 0.25 * minmod(c0[n] - cm[n], cp[n] - c0[n]);
    coarse5(P, U, lev - 1, C1, C2, C3 - 1, cm); coarse5(P, U, lev - 1, C1, C2, C3 + 1, cp);
    for (int n = 0; n < 5; n++) g3[n] = 0.25 * minmod(c0[n] - cm[n], cp[n] - c0[n]);
    for (int n = 0; n < 5; n++) val[n] = ((c0[n] + s1 * g1[n]) + s2 * g2[n]) + s3 * g3[n];
  }
}

// One ghost cell, all 5 variables.  Fast path: the same-level neighbour table built at bind time says which
// block holds the periodic image, and the source cell is the ghost index shifted by one block length (no
// division, one table load).  Where the table holds -1 (another level covers the position) the general
// path classifies the cell from the leaf maps.
// (Uniform meshes only: every table entry is a block there, so the kernel needs no general path and keeps a
// small register footprint -- 48 registers against 128 -- and with it the occupancy a copy kernel wants.)
__device__ __forceinline__ void fill_cell(const PackDev& P, double* __restrict__ U, const int* __restrict__ nb,
                                          int m, int i, int j, int k) {
  const int ng = P.ng, n1 = P.nt[0], n2 = P.nt[1];
  const int d1 = (i < ng) ? -1 : (i >= P.nx[0] + ng ? 1 : 0);
  const int d2 = (j < ng) ? -1 : (j >= P.nx[1] + ng ? 1 : 0);
  const int d3 = (k < ng) ? -1 : (k >= P.nx[2] + ng ? 1 : 0);
  const int dir = (d3 + 1) * 9 + (d2 + 1) * 3 + (d1 + 1);
  const int src = nb[dir];
  double val[5];
  if (src < 0) return;                 // cannot happen on a uniform mesh
  const int code = P.nbc[27 * m + dir];
  int si = i - d1 * P.nx[0], sj = j - d2 * P.nx[1], sk = k - d3 * P.nx[2];      // image one block length away
  if (code) {                          // the ghost lies outside a non-periodic domain boundary
    const int c1 = code & 3, c2 = (code >> 2) & 3, c3 = (code >> 4) & 3;
    // outflow: the nearest active cell; reflect: the mirror image across the boundary face
    if (c1) si = (c1 == 1) ? (d1 < 0 ? ng : P.nx[0] + ng - 1) : (d1 < 0 ? 2 * ng - 1 - i : 2 * (P.nx[0] + ng) - 1 - i);
    if (c2) sj = (c2 == 1) ? (d2 < 0 ? ng : P.nx[1] + ng - 1) : (d2 < 0 ? 2 * ng - 1 - j : 2 * (P.nx[1] + ng) - 1 - j);
    if (c3) sk = (c3 == 1) ? (d3 < 0 ? ng : P.nx[2] + ng - 1) : (d3 < 0 ? 2 * ng - 1 - k : 2 * (P.nx[2] + ng) - 1 - k);
    const double* q = U + (long long)src * 5 * P.ncell + ((long long)sk * n2 + sj) * n1 + si;
#pragma unroll
    for (int n = 0; n < 5; n++) val[n] = q[n * P.ncell];
    if (c1 == 2) val[1] = -val[1];     // the normal momentum of a reflected image changes sign
    if (c2 == 2) val[2] = -val[2];
    if (c3 == 2) val[3] = -val[3];
  } else {
    const double* q = U + (long long)src * 5 * P.ncell + ((long long)sk * n2 + sj) * n1 + si;
#pragma unroll
    for (int n = 0; n < 5; n++) val[n] = q[n * P.ncell];
  }
  double* o = U + (long long)m * 5 * P.ncell + ((long long)k * n2 + j) * n1 + i;
#pragma unroll
  for (int n = 0; n < 5; n++) o[n * P.ncell] = val[n];
}

// One warp per row of the ghost shell: the 2 ng n2 rows of the two k-slabs and the nx3 2 ng rows of the two
// j-slabs are full rows of n1 cells (lanes stride along i: coalesced); the nx3 nx2 interior rows have only
// their 2 ng end cells in the shell, and one warp takes 32 / (2 ng) of those rows at once.
__global__ void __launch_bounds__(256) fill_ghosts_kernel(PackDev P, double* __restrict__ U, int rowsA, int rowsB,
                                                          int groupsC, int rpg) {
  const int m = blockIdx.y, lane = threadIdx.x & 31;

  const int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int ng = P.ng, n1 = P.nt[0], n2 = P.nt[1];
  const int* nb = P.nbr + 27 * m;
  if (w < rowsA + rowsB) {
    int j, k;
    if (w < rowsA) { const int kk = w / n2; j = w - kk * n2; k = kk < ng ? kk : kk + P.nx[2]; }
    else { const int r = w - rowsA; const int kk = r / (2 * ng), jj = r - kk * (2 * ng); k = ng + kk; j = jj < ng ? jj : jj + P.nx[1]; }
    for (int i = lane; i < n1; i += 32) fill_cell(P, U, nb, m, i, j, k);
  } else if (w < rowsA + rowsB + groupsC) {
    const int g = w - rowsA - rowsB;
    for (int c = lane; c < rpg * 2 * ng; c += 32) {     // one pass unless 2 ng > 32
      const int sub = c / (2 * ng), ii = c - sub * (2 * ng);
      const int row = g * rpg + sub;
      if (row < P.nx[2] * P.nx[1]) {
        const int kk = row / P.nx[1], jj = row - kk * P.nx[1];
        fill_cell(P, U, nb, m, ii < ng ? ii : ii + P.nx[0], ng + jj, ng + kk);
      }
    }
  }
}

// Refined meshes: one thread per ghost cell, every cell through the general path (copy, restriction or
// prolongation decided per cell from the leaf maps).  The ghost shell of a block is enumerated as k-slabs,
// then j-slabs, then i-slabs so that consecutive threads touch consecutive i; the few expensive
// prolongation cells are spread over many warps and overlap with the cheap copies of the same launch.
__global__ void __launch_bounds__(256) fill_ghosts_flat_kernel(PackDev P, double* __restrict__ U, int nghost) {
  const int m = blockIdx.y;
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= nghost) return;
  const int ng = P.ng, n1 = P.nt[0], n2 = P.nt[1];
  const int A = 2 * ng * n2 * n1, B = P.nx[2] * 2 * ng * n1;
  int i, j, k;
  if (g < A) {
    int kk = g / (n2 * n1), r = g - kk * (n2 * n1);
    k = kk < ng ? kk : kk + P.nx[2];
    j = r / n1; i = r - j * n1;
  } else if (g < A + B) {
    g -= A;
    int kk = g / (2 * ng * n1), r = g - kk * (2 * ng * n1);
    k = ng + kk;
    int jj = r / n1; i = r - jj * n1;
    j = jj < ng ? jj : jj + P.nx[1];
  } else {
    g -= A + B;
    int kk = g / (P.nx[1] * 2 * ng), r = g - kk * (P.nx[1] * 2 * ng);
    k = ng + kk;
    int jj = r / (2 * ng), ii = r - jj * (2 * ng);
    j = ng + jj;
    i = ii < ng ? ii : ii + P.nx[0];
  }
  double val[5];
  // fast path: where the same-level neighbour table names a block, the ghost cell is a plain copy of the cell one block
  // length away (no leaf-map lookups, no wrapping); only cells next to another level take the general path
  const int d1 = (i < ng) ? -1 : (i >= P.nx[0] + ng ? 1 : 0);
  const int d2 = (j < ng) ? -1 : (j >= P.nx[1] + ng ? 1 : 0);
  const int d3 = (k < ng) ? -1 : (k >= P.nx[2] + ng ? 1 : 0);
  const int src = P.nbr[27 * m + (d3 + 1) * 9 + (d2 + 1) * 3 + (d1 + 1)];
  if (src >= 0) {
    const double* q = U + (long long)src * 5 * P.ncell +
                      ((long long)(k - d3 * P.nx[2]) * n2 + (j - d2 * P.nx[1])) * n1 + (i - d1 * P.nx[0]);
#pragma unroll
    for (int n = 0; n < 5; n++) val[n] = q[n * P.ncell];
  } else {
    ghost_general(P, U, m, i, j, k, val);
  }
  const long long o = (long long)m * 5 * P.ncell + ((long long)k * n2 + j) * n1 + i;
  for (int n = 0; n < 5; n++) U[o + n * P.ncell] = val[n];
}

cudaError_t launch_fill_ghosts(const ak_pack& p, double* U) {
  const PackDev& P = p.d;
  if (P.max_level > 0) {
    long long nghost = P.ncell - (long long)P.nx[0] * P.nx[1] * P.nx[2];
    dim3 grid((unsigned)((nghost + 255) / 256), (unsigned)P.nmb);
    fill_ghosts_flat_kernel<<<grid, 256, 0, p.stream>>>(P, U, (int)nghost);
    return cudaGetLastError();
  }
  const int rowsA = 2 * P.ng * P.nt[1], rowsB = P.nx[2] * 2 * P.ng;
  const int rpg = 32 / (2 * P.ng) > 0 ? 32 / (2 * P.ng) : 1;
  const int groupsC = (P.nx[2] * P.nx[1] + rpg - 1) / rpg;
  const int warps = rowsA + rowsB + groupsC;
  dim3 grid((unsigned)((warps + 7) / 8), (unsigned)P.nmb);
  fill_ghosts_kernel<<<grid, 256, 0, p.stream>>>(P, U, rowsA, rowsB, groupsC, rpg);
  return cudaGetLastError();
}

// ---- S0: CFL time step ---------------------------------------------------------------------------
// Every candidate dx_d/(|v_d|+c_s) is positive, so its IEEE bit pattern orders like an unsigned
// integer and the global min is one atomicMin per CTA after a shuffle + shared-memory reduction.
__global__ void dt_init_kernel(PackDev P) { *P.dtmin_bits = 0x7FF0000000000000ull; *P.nonfinite = 0ull; }

__global__ void __launch_bounds__(256) new_dt_kernel(PackDev P, const double* __restrict__ U, long long nrows) {
  const double ug_floor = P_FLOOR / (P.gamma - 1.0);
  double best = __longlong_as_double(0x7FF0000000000000ll);
  // one warp per group of rpw rows of nx1 active cells (rpw = 32 / nx1 rows of one block when nx1 <= 16, so
  // that short rows still fill the warp; else 1); groups enumerated over (m, k, j-group)
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5;
  const int rpw = P.nx[0] <= 16 ? 32 / P.nx[0] : 1;
  const int jg = (P.nx[1] + rpw - 1) / rpw;
  const int lj = rpw > 1 ? lane / P.nx[0] : 0, li = rpw > 1 ? lane - lj * P.nx[0] : lane;
  for (long long row = (long long)blockIdx.x * wpb + wib; row < nrows; row += (long long)gridDim.x * wpb) {
    long long r = row;
    int j = (int)(r % jg) * rpw + lj; r /= jg;
    int k = (int)(r % P.nx[2]); r /= P.nx[2];
    int m = (int)r;
    const int lev = P.blk[m].x;
    const double sc = lev ? 0.5 : 1.0;
    const double dx1 = sc * P.dx0[0], dx2 = sc * P.dx0[1], dx3 = sc * P.dx0[2];
    const bool rowok = (j < P.nx[1]) && (lj < rpw);
    const double* q = U + (long long)m * 5 * P.ncell + ((long long)(k + P.ng) * P.nt[1] + (j + P.ng)) * P.nt[0] + P.ng;
    // dx_d / s is monotone in s > 0 (IEEE division rounds monotonically), so the row's min over cells of
    // dx_d / (|v_d| + c_s) is dx_d / max(|v_d| + c_s), bit for bit: three divisions per row instead of per cell
    double s1 = 0.0, s2 = 0.0, s3 = 0.0;
    bool bad = false;                 // a NaN / inf signal speed must not be skipped by fmax (it is reported, ak.h)
#pragma unroll 2
    for (int i = li; rowok && i < P.nx[0]; i += 32) {
      double u[5], w[5];
      for (int n = 0; n < 5; n++) u[n] = q[i + n * P.ncell];
      c2p(u, w, ug_floor);
      double pr = (P.gamma - 1.0) * w[4];
      double cs = sqrt(P.gamma * pr / w[0]);
      const double a1 = fabs(w[1]) + cs, a2 = fabs(w[2]) + cs, a3 = fabs(w[3]) + cs;
      bad = bad || !((a1 + a2) + a3 < __longlong_as_double(0x7FF0000000000000ll));
      s1 = fmax(s1, a1);
      s2 = fmax(s2, a2);
      s3 = fmax(s3, a3);
    }
    if (bad) atomicAdd(P.nonfinite, 1ull);
    if (s1 > 0.0) best = fmin(best, fmin(dx1 / s1, fmin(dx2 / s2, dx3 / s3)));
  }
  for (int o = 16; o > 0; o >>= 1) best = fmin(best, __shfl_xor_sync(0xffffffffu, best, o));
  __shared__ double sm[8];
  if (lane == 0) sm[wib] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < wpb; w++) best = fmin(best, sm[w]);
    atomicMin(P.dtmin_bits, (unsigned long long)__double_as_longlong(best));
  }
}

cudaError_t launch_new_dt(const ak_pack& p, const double* U) {
  const PackDev& P = p.d;
  dt_init_kernel<<<1, 1, 0, p.stream>>>(P);
  const int rpw = P.nx[0] <= 16 ? 32 / P.nx[0] : 1;
  long long nrows = (long long)P.nmb * ((P.nx[1] + rpw - 1) / rpw) * P.nx[2];
  long long want = (nrows + 7) / 8;
  int grid = (int)(want < (long long)p.sm_count * 8 ? want : (long long)p.sm_count * 8);
  new_dt_kernel<<<grid, 256, 0, p.stream>>>(P, U, nrows);
  return cudaGetLastError();
}

}  // namespace ak

// ---- S0 without any allocation: ak_new_dt_noalloc (include/ak.h) ---------------------------------------------------
// Some callers cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it) and
// have no pack with its caller-allocated scratch buffer either.  This entry point runs the SAME reduction kernel as
// ak_new_dt (new_dt_kernel above, unchanged) on a caller-owned state buffer of a uniform single-level pack; the scratch
// the kernel needs -- the reduction cells and the block table it reads each block's level from -- lives in the
// file-scope device array below instead of a caller buffer.  Every GPU that loads the library holds its
// AK_NOALLOC_SCRATCH_BYTES (128 KiB) until exit.  All calls share the array and it keeps the last call's contents:
// every call rewrites the cells and the table entries it uses before the reduction reads them (noalloc_setup_kernel,
// same stream), and two calls that overlap on one GPU (different streams or threads) race on it.
#define AK_NOALLOC_SCRATCH_BYTES (128 * 1024)
#define AK_NOALLOC_MAX_BLOCKS ((AK_NOALLOC_SCRATCH_BYTES - 256) / (int)sizeof(int4))      /* 8176 */
static __device__ __align__(256) unsigned char g_noalloc_scratch[AK_NOALLOC_SCRATCH_BYTES];

namespace ak {
// layout of g_noalloc_scratch: [0, 8) min dt as ordered bits | [8, 16) unused | [16, 24) rows with a non-finite signal
// speed | [256, 256 + 16 nmb) block table int4 (level, lx1, lx2, lx3): level 0 for every block of a uniform pack.
// Device code names the array directly; host code must not (there the name is a host-side stand-in).
__global__ void __launch_bounds__(256) noalloc_setup_kernel(int nmb) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m == 0) {
    *reinterpret_cast<unsigned long long*>(g_noalloc_scratch) = 0x7FF0000000000000ull;        // +inf: identity of the min
    *reinterpret_cast<unsigned long long*>(g_noalloc_scratch + 16) = 0ull;
  }
  if (m < nmb) reinterpret_cast<int4*>(g_noalloc_scratch + 256)[m] = make_int4(0, 0, 0, 0);
}
}  // namespace ak

extern "C" int ak_new_dt_noalloc(const void* u, int nmb, int nx1, int nx2, int nx3, int ng, double gamma,
                                 double dx1, double dx2, double dx3, double cfl, void* cuda_stream, double* dt_out) {
  using namespace ak;
  if (!u || !dt_out) return set_error(-1, "ak_new_dt_noalloc: null pointer");
  if (nmb < 1 || nx1 < 1 || nx2 < 1 || nx3 < 1 || ng < 0 || ng > 4) return set_error(-1, "ak_new_dt_noalloc: bad pack shape");
  if (!(gamma > 1.0) || !(cfl > 0.0) || !(dx1 > 0.0) || !(dx2 > 0.0) || !(dx3 > 0.0))
    return set_error(-1, "ak_new_dt_noalloc: gamma must exceed 1; cfl and the cell sizes must be positive");
  if (nmb > AK_NOALLOC_MAX_BLOCKS)
    return set_error(-3, "ak_new_dt_noalloc: more than 8176 MeshBlocks do not fit the library's 128 KiB static scratch array "
                         "(use ak_new_dt on a pack with caller-allocated scratch)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // the device that owns u runs the kernels (no allocation: attribute queries and cudaSetDevice only)
  cudaPointerAttributes pa;
  cudaError_t e = cudaPointerGetAttributes(&pa, u);
  if (e != cudaSuccess) return set_error(-4, cudaGetErrorString(e));
  if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) return set_error(-1, "ak_new_dt_noalloc: u is not a device pointer");
  if (pa.device < 0 || pa.device >= 64) return set_error(-3, "ak_new_dt_noalloc: device ordinal beyond 63");
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) return set_error(-4, "ak_new_dt_noalloc: cudaGetDevice failed");
  if (prev != pa.device && cudaSetDevice(pa.device) != cudaSuccess) return set_error(-4, "ak_new_dt_noalloc: cudaSetDevice failed");
  int rc = 0;
  do {
    // device address of the static array: once per device, with that device current
    static unsigned char* scratch_of_device[64] = {};
    unsigned char* s = scratch_of_device[pa.device];
    if (!s) {
      e = cudaGetSymbolAddress((void**)&s, g_noalloc_scratch);
      if (e != cudaSuccess || !s) { rc = set_error(-4, "ak_new_dt_noalloc: cudaGetSymbolAddress failed"); break; }
      scratch_of_device[pa.device] = s;
    }
    PackDev P{};
    P.nmb = nmb; P.ng = ng; P.gamma = gamma; P.max_level = 0;
    P.nx[0] = nx1; P.nx[1] = nx2; P.nx[2] = nx3;
    for (int d = 0; d < 3; d++) { P.nt[d] = P.nx[d] + 2 * ng; P.nrb[d] = 1; }
    P.ncell = (long long)P.nt[0] * P.nt[1] * P.nt[2];
    P.dx0[0] = dx1; P.dx0[1] = dx2; P.dx0[2] = dx3;
    P.dtmin_bits = (unsigned long long*)s;
    P.floor_cnt = (unsigned long long*)(s + 8);
    P.nonfinite = (unsigned long long*)(s + 16);
    P.blk = (const int4*)(s + 256);
    noalloc_setup_kernel<<<(nmb + 255) / 256, 256, 0, st>>>(nmb);
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, pa.device);
    const int rpw = P.nx[0] <= 16 ? 32 / P.nx[0] : 1;                       // (as in launch_new_dt)
    const long long nrows = (long long)P.nmb * ((P.nx[1] + rpw - 1) / rpw) * P.nx[2];
    const long long want = (nrows + 7) / 8;
    const int grid = (int)(want < (long long)sms * 8 ? want : (long long)sms * 8);
    new_dt_kernel<<<grid, 256, 0, st>>>(P, (const double*)u, nrows);
    e = cudaGetLastError();
    if (e != cudaSuccess) { rc = set_error(-4, cudaGetErrorString(e)); break; }
    unsigned long long cells[3];
    e = cudaMemcpyAsync(cells, s, 24, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { rc = set_error(-4, cudaGetErrorString(e)); break; }
    double dtmin;
    memcpy(&dtmin, &cells[0], 8);
    if (cells[2] || !(dtmin > 0.0) || !(dtmin < __builtin_huge_val())) {
      rc = set_error(-5, "non-finite signal speed in the state (NaN or inf in an active cell)"); break;
    }
    *dt_out = cfl * dtmin;
  } while (0);
  if (prev != pa.device) cudaSetDevice(prev);
  return rc;
}

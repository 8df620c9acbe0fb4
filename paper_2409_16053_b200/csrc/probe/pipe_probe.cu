// pipe_probe.cu -- stand-alone micro-benchmarks behind the pipe model of DESIGN.md section 6.1 (what bounds the
// stage kernel on sm_100a).  Not part of libak.so.  Build and run on a B200:
//     nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -fmad=false -I paper_2409_16053_b200/csrc -I include \
//          -o /tmp/pipe_probe paper_2409_16053_b200/csrc/probe/pipe_probe.cu && /tmp/pipe_probe
// It prints, per line, "name value": issue cycles per warp instruction of DFMA / DADD / DMUL / FSEL and of DFMA+FSEL
// mixes at 12 warps per SM, the dependent-issue latency of DFMA, and the cycles per warp iteration of a loop that is
// exactly the x1/x2 PPM4 reconstruction of the stage kernel (ak_lean.cuh) at 6 .. 30 warps per SM, next to
// 2 x (FP64 + ALU instructions) of that loop (counted from its SASS: 202 + 151).
#include <cstdio>
#include <cuda_runtime.h>
#include "ak_pack.h"
#include "ak_lean.cuh"
using namespace ak;

#define SELF(i) asm volatile("{.reg .pred p; setp.ne.s32 p, %2, 0; selp.f32 %0, %0, %1, p;}" : "+f"(f[i]) : "f"(g[i]), "r"(sel))
#define SELG(i) asm volatile("{.reg .pred p; setp.ne.s32 p, %2, 0; selp.f32 %0, %0, %1, p;}" : "+f"(g[i]) : "f"(f[i]), "r"(sel))

// OP: 0 DFMA  1 DADD  2 DMUL  3 FSEL  4 DFMA + FSEL  5 DFMA + 2 FSEL
template <int OP, int ILP>
__global__ void __launch_bounds__(384, 1) op_kernel(double* out, int iters, int sel, double ca, double cb) {
  double x[ILP]; float f[ILP], g[ILP];
  for (int i = 0; i < ILP; i++) { x[i] = threadIdx.x * 1e-3 + i; f[i] = i + threadIdx.x; g[i] = 2 * i; }
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int u = 0; u < 8; u++) {
#pragma unroll
      for (int i = 0; i < ILP; i++) {
        if (OP == 0 || OP == 4 || OP == 5) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x[i]) : "d"(ca), "d"(cb));
        if (OP == 1) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(x[i]) : "d"(cb));
        if (OP == 2) asm volatile("mul.rn.f64 %0, %0, %1;" : "+d"(x[i]) : "d"(ca));
        if (OP == 3 || OP == 4 || OP == 5) SELF(i);
        if (OP == 5) SELG(i);
      }
    }
  }
  double s = 0;
  for (int i = 0; i < ILP; i++) s += x[i] + f[i] + g[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int OP, int ILP>
static double op_cycles(double* d, double ghz, int warps_per_sm) {
  const int iters = 2000, threads = 32 * warps_per_sm;
  op_kernel<OP, ILP><<<148, threads>>>(d, 10, 1, 1.0000001, 1e-9);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0);
  op_kernel<OP, ILP><<<148, threads>>>(d, iters, 1, 1.0000001, 1e-9);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  return ms * 1e-3 * ghz * 1e9 / (iters * 8.0 * ILP * (warps_per_sm / 4.0));   // SMSP cycles per warp per group of ops
}

constexpr int TI = 16, TJ = 12, RR = 3, WI = TI + 2 * RR, WJ = TJ + 2 * RR;
__global__ void __launch_bounds__(192, 5) recon_kernel(double* out, int iters) {
  __shared__ double W[5 * WJ * WI];
  __shared__ double Q[2 * 5 * 192];                // (never read: the compiler drops these stores; the counts above are of that loop)
  const int tid = threadIdx.x, ti = tid % TI, tj = tid / TI;
  for (int i = tid; i < 5 * WJ * WI; i += 192) W[i] = 1.0 + 0.01 * sin(0.37 * i) + 1e-3 * (i % 7);
  __syncthreads();
  const int oW = (tj + RR) * WI + ti + RR;
  double acc = 0;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int n = 0; n < 5; n++) {
      const double* p = W + n * (WJ * WI) + oW;
      { double lo = iface_lean(p[-2], p[-1], p[0], p[1]), hi = iface_lean(p[-1], p[0], p[1], p[2]);
        limit_lean(p[0], lo, hi); Q[n * 192 + tid] = hi; acc += lo; }
      { double lo = iface_lean(p[-2 * WI], p[-WI], p[0], p[WI]), hi = iface_lean(p[-WI], p[0], p[WI], p[2 * WI]);
        limit_lean(p[0], lo, hi); Q[(5 + n) * 192 + tid] = hi; acc += lo; }
    }
    W[oW] += 1e-9 * acc;          // iterations depend on memory: nothing can be hoisted
    __syncthreads();
  }
  out[blockIdx.x * 192 + tid] = acc;
}

static double recon_cycles(double* d, double ghz, int ctas_per_sm) {
  const int iters = 2000;
  recon_kernel<<<148 * ctas_per_sm, 192>>>(d, 10);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0); recon_kernel<<<148 * ctas_per_sm, 192>>>(d, iters); cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  return ms * 1e-3 * ghz * 1e9 / iters / (6.0 * ctas_per_sm / 4.0);
}

int main() {
  cudaDeviceProp pr; cudaGetDeviceProperties(&pr, 0);
  int khz = 0; cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
  const double ghz = khz * 1e-6;
  double* d; cudaMalloc(&d, 148 * 8 * 192 * 8);
  printf("device %s sms %d sm_clock_ghz %.3f\n", pr.name, pr.multiProcessorCount, ghz);
  printf("dfma_cycles_per_warp_instr %.2f\n", op_cycles<0, 6>(d, ghz, 12));
  printf("dadd_cycles_per_warp_instr %.2f\n", op_cycles<1, 6>(d, ghz, 12));
  printf("dmul_cycles_per_warp_instr %.2f\n", op_cycles<2, 6>(d, ghz, 12));
  printf("fsel_cycles_per_warp_instr %.2f\n", op_cycles<3, 6>(d, ghz, 12));
  printf("dfma_plus_fsel_cycles %.2f\n", op_cycles<4, 6>(d, ghz, 12));
  printf("dfma_plus_2fsel_cycles %.2f\n", op_cycles<5, 6>(d, ghz, 12));
  printf("dfma_dependent_latency_cycles %.2f\n", op_cycles<0, 1>(d, ghz, 4));
  for (int c = 1; c <= 5; c++) printf("ppm_recon_loop_cycles_at_%d_warps_per_sm %.0f\n", 6 * c, recon_cycles(d, ghz, c));
  printf("ppm_recon_loop_two_times_fp64_plus_alu %d\n", 2 * (202 + 151));
  return 0;
}

// contraction_bench.cu -- the experiment BASELINE.json's north_star asks for: how should the Nq x Nq derivative
// contraction of eq. (21)-(23) be issued on sm_100a?  Three variants of the SAME work -- D applied along xi
// to NV = 6 tiles of 5 x 5 x 5 nodes held in shared memory, in place -- timed in isolation at the occupancy of the
// tendency kernel (5 CTAs of 128 threads per SM, 148 SMs) and counted with ncu (profiles/r2_dmma.md):
//   A  line task     one thread per xi line: 5 LDS.64, 25 DFMA (D from the constant bank), 5 STS.64    (shipped kernels)
//   B  DMMA          mma.sync.m8n8k4.f64: 8 lines per MMA pair, fragments loaded from / stored to shared memory
//   C  warp shuffle  thread per node, value in a register, the 5 operands of a line fetched with __shfl_sync
// Build and run (committed files only):
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -o contraction_bench contraction_bench.cu && ./contraction_bench
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>

constexpr int Nq = 5, NF = 25, NP = 125, NV = 6, SLOT = 126, ITER = 200;
__constant__ double cD[8][8];

__device__ __forceinline__ void load_tiles(double* s, const double* g, int t) {
  for (int i = t; i < NV * SLOT; i += blockDim.x) s[i] = g[i];
  __syncthreads();
}
__device__ __forceinline__ void store_tiles(const double* s, double* g, int t) {
  __syncthreads();
  for (int i = t; i < NV * SLOT; i += blockDim.x) g[i] = s[i];
}

// A: one thread per line
__global__ void __launch_bounds__(128, 5) k_line(const double* in, double* out, int iters) {
  __shared__ double s[NV * SLOT];
  const int t = threadIdx.x;
  load_tiles(s, in + (size_t)blockIdx.x * NV * SLOT, t);
  for (int it = 0; it < iters; ++it) {
    if (t < NF) {
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        double* q = s + v * SLOT + Nq * t;
        double x[Nq], y[Nq];
#pragma unroll
        for (int m = 0; m < Nq; ++m) x[m] = q[m];
#pragma unroll
        for (int i = 0; i < Nq; ++i) { double a = 0.0;
#pragma unroll
          for (int m = 0; m < Nq; ++m) a += cD[i][m] * x[m];
          y[i] = a; }
#pragma unroll
        for (int i = 0; i < Nq; ++i) q[i] = y[i];
      }
    }
    __syncwarp();
  }
  store_tiles(s, out + (size_t)blockIdx.x * NV * SLOT, t);
}

// B: FP64 tensor-core MMA.  D (5x5, zero-padded to 8x8) is the A operand (two k-steps of 4), the values of 8 lines the B
// operand (k = node along the line, n = line), C (8 x 8) the result: row = output node, column = line.
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b, double c0, double c1) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%4,%5};"
               : "=d"(d0), "=d"(d1) : "d"(a), "d"(b), "d"(c0), "d"(c1));
}
__global__ void __launch_bounds__(128, 5) k_dmma(const double* in, double* out, int iters) {
  __shared__ double s[NV * SLOT + 64];
  const int t = threadIdx.x, lane = t & 31, w = t >> 5;
  load_tiles(s, in + (size_t)blockIdx.x * NV * SLOT, t);
  const int r = lane >> 2, c = lane & 3;                  // A: row r, col c | B: k = c, n = r | C: row r, cols 2c, 2c+1
  const double a0 = cD[r][c], a1 = cD[r][4 + c];          // zero beyond 5 x 5
  for (int it = 0; it < iters; ++it) {
    // warp w takes the line groups g = w (8 lines each): 25 lines -> groups 0..3 (lines 24..31 of group 3 are padding)
    const int g = w;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      double* q = s + v * SLOT;
      const int line = 8 * g + r;
      const double b0 = (line < NF) ? q[Nq * line + c] : 0.0;
      const double b1 = (line < NF && c == 0) ? q[Nq * line + 4] : 0.0;
      double c0 = 0.0, c1 = 0.0;
      dmma(c0, c1, a0, b0, c0, c1);
      dmma(c0, c1, a1, b1, c0, c1);
      __syncwarp();
      const int l0 = 8 * g + 2 * c, l1 = l0 + 1;          // columns of C = lines; row r = output node
      if (r < Nq) { if (l0 < NF) q[Nq * l0 + r] = c0; if (l1 < NF) q[Nq * l1 + r] = c1; }
      __syncwarp();
    }
  }
  store_tiles(s, out + (size_t)blockIdx.x * NV * SLOT, t);
}

// C: thread per node (5 warps x 30 lanes = 6 lines per warp, so that no line straddles a warp), operands by shuffle
__global__ void __launch_bounds__(160, 4) k_shfl(const double* in, double* out, int iters) {
  __shared__ double s[NV * SLOT];
  const int t = threadIdx.x, lane = t & 31, w = t >> 5;
  load_tiles(s, in + (size_t)blockIdx.x * NV * SLOT, t);
  const int n = 30 * w + lane;                            // node of this lane (lanes 30, 31 idle; last warp: 5 lanes)
  const bool act = lane < 30 && n < NP;
  const int i = lane % Nq, base = lane - i;
  double x[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) x[v] = act ? s[v * SLOT + n] : 0.0;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      double a = 0.0;
#pragma unroll
      for (int m = 0; m < Nq; ++m) a += cD[i][m] * __shfl_sync(0xffffffffu, x[v], base + m);
      x[v] = a;
    }
  }
#pragma unroll
  for (int v = 0; v < NV; ++v) if (act) s[v * SLOT + n] = x[v];
  store_tiles(s, out + (size_t)blockIdx.x * NV * SLOT, t);
}

int main() {
  int dev = 0; cudaDeviceProp pr; cudaGetDeviceProperties(&pr, dev);
  const int blocks = pr.multiProcessorCount * 5 * 8;
  const size_t n = (size_t)blocks * NV * SLOT;
  double hD[8][8] = {};
  // a contraction matrix with spectral radius < 1 so that 200 in-place applications stay finite; any 5 x 5 matrix does
  for (int i = 0; i < Nq; ++i) for (int j = 0; j < Nq; ++j) hD[i][j] = 0.19 * ((i == j) ? 1.0 : 0.3 / (1 + abs(i - j))) * ((i + j) % 2 ? -1 : 1);
  cudaMemcpyToSymbol(cD, hD, sizeof(hD));
  double *in, *o[3]; cudaMalloc(&in, n * 8);
  double* h = (double*)malloc(n * 8);
  for (size_t i = 0; i < n; ++i) h[i] = 1.0 + 1e-3 * (double)((i * 2654435761u) % 1000);
  cudaMemcpy(in, h, n * 8, cudaMemcpyHostToDevice);
  for (int k = 0; k < 3; ++k) { cudaMalloc(&o[k], n * 8); cudaMemset(o[k], 0, n * 8); }
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const char* name[3] = {"A line task (LDS/DFMA/STS)", "B DMMA m8n8k4.f64", "C warp shuffle"};
  float ms[3];
  for (int k = 0; k < 3; ++k)
    for (int rep = 0; rep < 3; ++rep) {
      cudaEventRecord(e0);
      if (k == 0) k_line<<<blocks, 128>>>(in, o[0], ITER);
      if (k == 1) k_dmma<<<blocks, 128>>>(in, o[1], ITER);
      if (k == 2) k_shfl<<<blocks, 160>>>(in, o[2], ITER);
      cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms[k], e0, e1);
    }
  if (cudaGetLastError() != cudaSuccess) { printf("CUDA error\n"); return 1; }
  // agreement of the three variants (same arithmetic up to summation order)
  double* r[3];
  for (int k = 0; k < 3; ++k) { r[k] = (double*)malloc(n * 8); cudaMemcpy(r[k], o[k], n * 8, cudaMemcpyDeviceToHost); }
  double dmax[3] = {0, 0, 0}, amax = 0;
  for (size_t i = 0; i < n; ++i) {
    if ((i % SLOT) >= NP) continue;
    amax = fmax(amax, fabs(r[0][i]));
    for (int k = 1; k < 3; ++k) dmax[k] = fmax(dmax[k], fabs(r[k][i] - r[0][i]));
  }
  const double units = (double)blocks * ITER;             // element-contractions (6 variables x 25 lines each)
  for (int k = 0; k < 3; ++k)
    printf("%-30s %8.3f ms  %7.2f ns per element-direction per SM  rel. diff to A %.1e\n", name[k], ms[k],
           1e6 * ms[k] / units * pr.multiProcessorCount, dmax[k] / amax);
  return 0;
}

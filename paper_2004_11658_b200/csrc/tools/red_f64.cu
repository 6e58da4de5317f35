// micro-benchmark: throughput of red.global.add.f64 in the scatter pattern a same-species pair reuse in pass 1 would
// need: every warp adds a whole T tile (TILE doubles, 32 consecutive doubles per instruction)
// to a pseudo-random destination tile.  Not part of libdpb.so.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o red_f64 paper_2004_11658_b200/csrc/tools/red_f64.cu && ./red_f64
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("CUDA error %s at %d\n",cudaGetErrorString(e),__LINE__); exit(1);} }while(0)

__global__ void k_red(double *T, int ntiles, int tile, int tiles_per_warp, unsigned seed) {
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  unsigned s = seed ^ (warp * 2654435761u);
  for (int k = 0; k < tiles_per_warp; ++k) {
    s = s * 1664525u + 1013904223u;
    double *dst = T + (size_t)((s >> 8) % (unsigned)ntiles) * tile;
    const double v = 1e-3 * lane + k;
#pragma unroll 4
    for (int o = lane; o < tile; o += 32) atomicAdd(dst + o, v);      // result unused -> RED.E.ADD.F64
  }
}

int main() {
  cudaDeviceProp p; CK(cudaGetDeviceProperties(&p, 0));
  printf("%s, %d SMs\n", p.name, p.multiProcessorCount);
  const int tile = 512;                                   // copper: M x 4 doubles = 4 KB per atom
  const int nts[3] = {4096, 32000, 131072};               // 16.8 MB (L2), 131 MB (one 32k-atom chunk), 537 MB
  for (int c = 0; c < 3; ++c) {
    const int ntiles = nts[c];
    double *T; CK(cudaMalloc(&T, sizeof(double) * (size_t)ntiles * tile)); CK(cudaMemset(T, 0, sizeof(double) * (size_t)ntiles * tile));
    for (int thr = 256; thr <= 1024; thr *= 2) {
      const int grid = p.multiProcessorCount * (2048 / thr), tpw = 64;
      const long long nwarps = (long long)grid * thr / 32;
      cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
      float best = 1e30f;
      for (int rep = 0; rep < 4; ++rep) {
        CK(cudaEventRecord(e0));
        k_red<<<grid, thr>>>(T, ntiles, tile, tpw, 12345u + rep);
        CK(cudaEventRecord(e1)); CK(cudaEventSynchronize(e1));
        float ms; CK(cudaEventElapsedTime(&ms, e0, e1)); if (rep && ms < best) best = ms;
      }
      const double nred = (double)nwarps * tpw * tile;
      printf("tiles %6d (%6.1f MB) grid %4d x %4d: %.3f ms, %.1f G red.f64/s = %.2f TB/s of operands; 2.83 M pairs x 512 -> %.2f ms\n",
             ntiles, ntiles * tile * 8e-6, grid, thr, best, nred / best * 1e-6, nred * 8 / best * 1e-9, 2.83e6 * 512 / (nred / best));
    }
    CK(cudaFree(T));
  }
  return 0;
}

// random_gather.cu — microbenchmark behind DESIGN.md section 5 ("what bounds the T1 kernel"): rounds of dependent
// random 16-byte gathers from an L2-resident (64 MB) or DRAM-resident (1 GB) buffer, W warps, M independent
// loads per lane and round.  Stand-alone measurement tool, not part of libavm_b200.so:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o random_gather random_gather.cu && ./random_gather
// Results on B200: profiles/r2_micro_random_gather.md.
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
__global__ void chase(const uint4* __restrict__ buf, size_t n, int rounds, int M, unsigned* out, int ldmode) {
  unsigned x = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
  unsigned acc = 0;
  for (int r = 0; r < rounds; ++r) {
    uint4 v[16];
#pragma unroll
    for (int m = 0; m < 16; ++m) {
      if (m < M) {
        unsigned long long idx = ((unsigned long long)(x + m * 0x9E3779B9u) * 0xD2511F53ull) % n;
        v[m] = ldmode ? __ldcg(buf + idx) : buf[idx];
      }
    }
#pragma unroll
    for (int m = 0; m < 16; ++m) if (m < M) acc += v[m].x + v[m].y;
    x = x * 1664525u + 1013904223u + acc;
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}
int main() {
  size_t bytes = (size_t)1 << 30;
  uint4* buf; cudaMalloc(&buf, bytes); cudaMemset(buf, 1, bytes);
  unsigned* out; cudaMalloc(&out, 1 << 24);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  int rounds = 20;
  for (size_t mb : {64, 1024}) {
    size_t n = mb * (1 << 20) / 16;
    for (int warps : {148, 592, 1184, 2368, 4736}) {
      for (int M : {1, 4, 8, 16}) {
        int blocks = warps / 4;
        chase<<<blocks, 128>>>(buf, n, rounds, M, out, 0);
        cudaEventRecord(e0);
        chase<<<blocks, 128>>>(buf, n, rounds, M, out, 0);
        cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        double per_round_us = ms * 1e3 / rounds;
        double sect = (double)warps * 32 * M;
        printf("buf %4zu MB warps %5d M %2d : %.2f us/round, %.1f G sectors/s\n", mb, warps, M, per_round_us, sect / per_round_us / 1e3);
      }
    }
  }
  return 0;
}

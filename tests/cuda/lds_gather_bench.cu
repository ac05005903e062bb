// micro-benchmark behind DESIGN.md section 6: throughput of random shared-memory gathers on one SM (B200), 832 threads like
// k_resident on config 3.  Not a test; build and run by hand:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 tests/cuda/lds_gather_bench.cu -o /tmp/lds && /tmp/lds
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
template <int BYTES, bool RANDOM>
__global__ void k(int iters, int nslots, long long *out, float *sink) {
  extern __shared__ float4 sm[];
  for (int i = threadIdx.x; i < nslots; i += blockDim.x) sm[i] = make_float4(i, i + 1, i + 2, i + 3);
  __syncthreads();
  uint32_t h = threadIdx.x * 2654435761u + 12345u;
  float acc = 0.f;
  long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      h = h * 1664525u + 1013904223u;
      int s = RANDOM ? (int)((h >> 8) % (uint32_t)nslots) : (int)((threadIdx.x + 32 * u + it) % nslots);
      if (BYTES == 16) { float4 v = sm[s]; acc += v.x + v.y + v.z; }
      else if (BYTES == 8) { float2 v = ((float2 *)sm)[2 * s]; acc += v.x + v.y; }
      else { float v = ((float *)sm)[4 * s]; acc += v; }
    }
  }
  long long t1 = clock64();
  if (threadIdx.x == 0) out[0] = t1 - t0;
  sink[threadIdx.x] = acc;
}
int main() {
  long long *d; float *s; cudaMalloc(&d, 8); cudaMalloc(&s, 4096 * 4);
  const int iters = 2000, nslots = 2540, threads = 832;
  auto run = [&](const char *name, void (*fn)(int, int, long long *, float *)) {
    cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 100000);
    fn<<<1, threads, nslots * 16>>>(iters, nslots, d, s); cudaDeviceSynchronize();
    fn<<<1, threads, nslots * 16>>>(iters, nslots, d, s); cudaDeviceSynchronize();
    long long c; cudaMemcpy(&c, d, 8, cudaMemcpyDeviceToHost);
    double warp_loads = (double)iters * 8 * (threads / 32);
    printf("%-28s %8.2f cycles per warp-level load (%d warps on the SM)  -> %.1f bytes/clk\n", name, c / warp_loads, threads / 32,
           32.0 * (name[4] == '1' ? 16 : name[4] == '8' ? 8 : 4) / (c / warp_loads));
  };
  run("LDS.128 random slots", k<16, true>);
  run("LDS.128 consecutive slots", k<16, false>);
  run("LDS.8B  random slots", k<8, true>);
  run("LDS.4B  random slots", k<4, true>);
  return 0;
}

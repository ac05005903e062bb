// TEST-ONLY kernel (never linked into the product): the product's hand-written Philox4x32-10
// (paper_1003_1148_b200/csrc/sop_device.cuh) against cuRAND's device function curand_Philox4x32_10 -- pin P6.
#include <cuda_runtime.h>
#include <curand_kernel.h>
#include <curand_philox4x32_x.h>
#include <stdint.h>

#include "../../paper_1003_1148_b200/csrc/sop_device.cuh"

__global__ void k_check(const uint32_t *ctr, const uint32_t *key, int n, uint32_t *mine, uint32_t *ref, float *normals,
                        unsigned long long seed) {
  int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= n) return;
  uint4 c = make_uint4(ctr[4 * q], ctr[4 * q + 1], ctr[4 * q + 2], ctr[4 * q + 3]);
  uint2 k = make_uint2(key[2 * q], key[2 * q + 1]);
  uint4 a = sop::philox4x32_10(c, k);
  uint4 b = curand_Philox4x32_10(c, k);
  mine[4 * q] = a.x; mine[4 * q + 1] = a.y; mine[4 * q + 2] = a.z; mine[4 * q + 3] = a.w;
  ref[4 * q] = b.x; ref[4 * q + 1] = b.y; ref[4 * q + 2] = b.z; ref[4 * q + 3] = b.w;
  sop::SysDev S;
  S.seed_lo = (uint32_t)seed; S.seed_hi = (uint32_t)(seed >> 32);
  // normals of (bead = ctr0, traj = ctr1, step = ctr2 | ctr3 << 32) with the product's mapping
  float3 g = sop::gaussian3(S, c.x, c.y, (unsigned long long)c.z | ((unsigned long long)c.w << 32));
  normals[3 * q] = g.x; normals[3 * q + 1] = g.y; normals[3 * q + 2] = g.z;
}

extern "C" int philox_check(const uint32_t *h_ctr, const uint32_t *h_key, int n, uint32_t *h_mine, uint32_t *h_ref,
                            float *h_normals, unsigned long long seed) {
  uint32_t *ctr, *key, *mine, *ref; float *nor;
  if (cudaMalloc(&ctr, 16 * n) || cudaMalloc(&key, 8 * n) || cudaMalloc(&mine, 16 * n) || cudaMalloc(&ref, 16 * n) ||
      cudaMalloc(&nor, 12 * n)) return -1;
  cudaMemcpy(ctr, h_ctr, 16 * n, cudaMemcpyHostToDevice);
  cudaMemcpy(key, h_key, 8 * n, cudaMemcpyHostToDevice);
  k_check<<<(n + 127) / 128, 128>>>(ctr, key, n, mine, ref, nor, seed);
  int rc = cudaDeviceSynchronize() == cudaSuccess ? 0 : -2;
  cudaMemcpy(h_mine, mine, 16 * n, cudaMemcpyDeviceToHost);
  cudaMemcpy(h_ref, ref, 16 * n, cudaMemcpyDeviceToHost);
  cudaMemcpy(h_normals, nor, 12 * n, cudaMemcpyDeviceToHost);
  cudaFree(ctr); cudaFree(key); cudaFree(mine); cudaFree(ref); cudaFree(nor);
  return rc;
}

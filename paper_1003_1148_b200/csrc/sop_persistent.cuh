// sop_persistent.cuh -- the persistent multi-step kernel: a3 + a4..a9 for up to pl_interval steps in ONE
// cooperative launch.  Each block owns a contiguous range of bead instances for the whole launch; the two time
// layers are exchanged through L2 with one grid-wide barrier per step, so a step costs one
// barrier + one gather latency instead of one kernel launch (a 30k-bead step moves ~6 MB: ~1 us of HBM time,
// below launch latency -- DESIGN.md "Why a persistent kernel").
#pragma once
#include "sop_device.cuh"

namespace sop {

// Grid-wide barrier on a monotonically increasing counter (zeroed by the host before the launch).
// release: this block's coordinate writes are ordered before the arrival; acquire: the other blocks' writes are
// visible (and this SM's L1 is invalidated) before anybody of this block reads the new time layer.
__device__ __forceinline__ void grid_barrier(unsigned *bar, unsigned target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
    unsigned v;
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
    } while (v < target);
  }
  __syncthreads();
}

template <int G, bool COMP>
__global__ void __launch_bounds__(1024) k_persist(SysDev S, int cur, unsigned long long step0, int n_steps,
                                                  int nb_interval, int filter_last, unsigned *bar) {
  const int per_block = (S.n_inst + gridDim.x - 1) / gridDim.x;
  const int b0 = min(S.n_inst, (int)blockIdx.x * per_block), b1 = min(S.n_inst, b0 + per_block);
  const int groups = blockDim.x / G;
  const int lane = threadIdx.x % G, grp = threadIdx.x / G;
  const int wlane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  int flag = 0;
  for (int s = 0; s < n_steps; ++s) {
    const unsigned long long step = step0 + (unsigned long long)s;
    const float4 *pin = S.pos[cur];
    float4 *pout = S.pos[cur ^ 1];
    for (int base = b0; base < b1; base += groups) {
      const int g = base + grp;
      const bool valid = g < b1;
      const int gg = valid ? g : b0;
      const int t = gg / S.N, i = gg - t * S.N;
      const float4 *pos_t = pin + (size_t)t * S.N;
      const float4 ri = pos_t[i];
      float3 f = internal_force<G, false>(S, pos_t, i, gg, lane, valid, ri, flag);
      if (valid && lane == 0) {
        const uint32_t tag = __float_as_uint(ri.w);
        external_force(S, i, ri, tag, step, f.x, f.y, f.z, flag);
        pout[gg] = langevin_update<COMP>(S, ri, tag, t, step, f.x, f.y, f.z, COMP ? S.carry + gg : nullptr, flag, gg);
      }
    }
    grid_barrier(bar, (unsigned)(s + 1) * gridDim.x);
    cur ^= 1;
    // eager re-filter (Alg. 3) of the rows this block owns, from the coordinates just written (list invariant)
    if ((step + 1) % (unsigned long long)nb_interval == 0 && (s + 1 < n_steps || filter_last)) {
      const float4 *pnew = S.pos[cur];
      for (int g = b0 + warp; g < b1; g += nwarps) {
        const int t = g / S.N, i = g - t * S.N;
        filter_row_warp<false>(S, pnew + (size_t)t * S.N, i, g, wlane, flag);
      }
      __syncthreads();
    }
  }
  if (flag) atomicOr(S.flags, flag);
}

}  // namespace sop

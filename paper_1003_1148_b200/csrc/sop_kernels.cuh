// sop_kernels.cuh -- __global__ kernels of the SOP Langevin hot path (sm_100a).  See DESIGN.md "Kernels".
#pragma once
#include "sop_device.cuh"

namespace sop {

// ------------------------------------------------------------------------------------------------
// a4-a9 fused: force + noise + integrate, one launch per step (the paper's single-kernel particle-based
// organisation), G lanes per bead.  FORCES = true: the non-fused instantiation that writes the
// deterministic force instead of moving the bead (sop_get_forces).
// ------------------------------------------------------------------------------------------------
// DENSE: blocks of <= 256 threads compiled for 32 registers (a few spilled words), so that 2048 threads are resident per SM:
// the streaming step waits on dependent index -> coordinate gathers, and occupancy is what hides them (cfg 4: 44 -> 38 us).
template <int G, bool COMP, bool FORCES, bool DENSE = false>
__global__ void __launch_bounds__(DENSE ? 256 : 1024, DENSE ? 8 : 1) k_step(SysDev S, int cur, unsigned long long step) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int g = (int)(gid / G);
  const int lane = (int)(gid % G);
  const bool valid = g < S.n_inst;
  const int gg = valid ? g : 0;
  const int t = gg / S.N, i = gg - t * S.N;
  const float4 *__restrict__ pos_t = S.pos[cur] + (size_t)t * S.N;
  const float4 ri = __ldg(pos_t + i);
  int flag = 0;
  float3 f = internal_force<G, true>(S, pos_t, i, gg, lane, valid, ri, flag);
  if (valid && lane == 0) {
    const uint32_t tag = __float_as_uint(ri.w);
    external_force(S, i, ri, tag, step, f.x, f.y, f.z, flag);
    if (FORCES) {
      S.force[gg] = make_float4(f.x, f.y, f.z, 0.f);
    } else {
      S.pos[cur ^ 1][gg] = langevin_update<COMP>(S, ri, tag, t, step, f.x, f.y, f.z, COMP ? S.carry + gg : nullptr, flag, gg);
    }
  }
  if (flag) atomicOr(S.flags, flag);
}

// ------------------------------------------------------------------------------------------------
// NEXT-4: the second-order update whose mean recursion is Eq. (5) (reading R14), two launches
// per step:  stage 0  r' = r + f(r) h/xi + G  -> the other time layer, f(r) -> S.force;
//            stage 1  r(t + h) = r + (h / 2 xi)[f(r) + f(r')] + G  in place (a thread writes only its own bead of the layer
//            it reads its own bead from; partners are read from the r' layer).
// The same Philox draw G in both stages (counter-based: regenerated, never stored); external terms at t_n in both.
// ------------------------------------------------------------------------------------------------
template <int G, bool COMP>
__global__ void __launch_bounds__(1024) k_step2(SysDev S, int cur, unsigned long long step, int stage) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int g = (int)(gid / G);
  const int lane = (int)(gid % G);
  const bool valid = g < S.n_inst;
  const int gg = valid ? g : 0;
  const int t = gg / S.N, i = gg - t * S.N;
  const float4 *__restrict__ pos_t = S.pos[stage == 0 ? cur : cur ^ 1] + (size_t)t * S.N;
  const float4 ri = __ldg(pos_t + i);                 // stage 0: r;  stage 1: r'
  int flag = 0;
  float3 f = internal_force<G, true>(S, pos_t, i, gg, lane, valid, ri, flag);
  if (valid && lane == 0) {
    const uint32_t tag = __float_as_uint(ri.w);
    external_force(S, i, ri, tag, step, f.x, f.y, f.z, flag);
    if (!(tag & TAG_FIXED)) {
      const float3 gn = gaussian3(S, tag & TAG_ID_MASK, (uint32_t)(S.traj_offset + t), step);
      const float amp = amp_of(S, t);
      if (stage == 0) {
        S.force[gg] = make_float4(f.x, f.y, f.z, 0.f);
        S.pos[cur ^ 1][gg] = langevin_apply<false>(S, ri, gn, f.x, f.y, f.z, nullptr, flag, amp);
      } else {
        const float4 f0 = S.force[gg];
        const float4 r0 = S.pos[cur][gg];
        S.pos[cur][gg] = langevin_apply<COMP>(S, r0, gn, 0.5f * (f0.x + f.x), 0.5f * (f0.y + f.y), 0.5f * (f0.z + f.z),
                                              COMP ? S.carry + gg : nullptr, flag, amp);
      }
    } else if (stage == 0) {
      S.pos[cur ^ 1][gg] = ri;
    }
  }
  if (flag) atomicOr(S.flags, flag);
}

// NEXT-4: one sweep of replica-exchange temperature swaps between trajectories (t, t+1), t = parity mod 2.
// Metropolis in fp64 on the device-reduced energies: accept if u <= min(1, exp((1/kT_t - 1/kT_t+1)(E_t - E_t+1))), u in (0, 1]
// from the first word of Philox4x32-10(counter = (global t, 'REX!', sweep lo, sweep hi), key = seed).
__global__ void k_replica_exchange(SysDev S, const double *e6, float *kT_t, float *amp_t, int parity, unsigned long long sweep, int *accepted) {
  const int pair = blockIdx.x * blockDim.x + threadIdx.x;
  const int t = parity + 2 * pair;
  if (t + 1 >= S.T) return;
  const double Ei = e6[6 * t] + e6[6 * t + 1] + e6[6 * t + 2] + e6[6 * t + 3] + e6[6 * t + 4];
  const double Ej = e6[6 * (t + 1)] + e6[6 * (t + 1) + 1] + e6[6 * (t + 1) + 2] + e6[6 * (t + 1) + 3] + e6[6 * (t + 1) + 4];
  const double d = (1.0 / (double)kT_t[t] - 1.0 / (double)kT_t[t + 1]) * (Ei - Ej);
  const double prob = d >= 0.0 ? 1.0 : exp(d);
  const uint4 x = philox4x32_10(make_uint4((uint32_t)(S.traj_offset + t), 0x52455821u, (uint32_t)sweep, (uint32_t)(sweep >> 32)),
                                make_uint2(S.seed_lo, S.seed_hi));
  const double u = ((double)(x.x >> 8) + 1.0) * (1.0 / 16777216.0);
  const int acc = u <= prob ? 1 : 0;
  if (acc) {
    const float k0 = kT_t[t], a0 = amp_t[t];
    kT_t[t] = kT_t[t + 1]; amp_t[t] = amp_t[t + 1];
    kT_t[t + 1] = k0; amp_t[t + 1] = a0;
  }
  if (accepted) accepted[t / 2] = acc;
}

// initial Hybrid Taus states (Alg. 6 line 1): Philox4x32-10(counter = (bead, traj, 'TAUS', 0), key = seed), with the
// bits that keep the Tausworthe components off their degenerate states (y1 >= 2, y2 >= 8, y3 >= 16)
__global__ void k_taus_seed(SysDev S, int cur) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= S.n_inst) return;
  const uint32_t bead = __float_as_uint(S.pos[cur][g].w) & TAG_ID_MASK;
  uint4 y = philox4x32_10(make_uint4(bead, (uint32_t)(S.traj_offset + g / S.N), 0x54415553u, 0u), make_uint2(S.seed_lo, S.seed_hi));
  y.x |= 2u; y.y |= 8u; y.z |= 16u;
  S.taus[g] = y;
}

// a3: L2 neighbor-list filter (Alg. 3), one warp per bead instance.
// 32 registers (two small spills) so that 2048 threads are resident: the kernel waits on its gathers, and the extra warps
// hide them (cfg 4: 164 -> 148 us; larger blocks or 8 lanes per row with 64-bit masks measured slower)
__global__ void __launch_bounds__(256, 8) k_filter(SysDev S, int cur) {
  const int w = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int lane = threadIdx.x & 31;
  if (w >= S.n_inst) return;
  const int t = w / S.N, i = w - t * S.N;
  int flag = 0;
  filter_row_warp<true>(S, S.pos[cur] + (size_t)t * S.N, i, w, lane, flag);
  if (flag && lane == 0) atomicOr(S.flags, flag);
}

// ------------------------------------------------------------------------------------------------
// a1: cell grid.  bbox -> grid parameters -> count -> scan -> fill -> per-cell sort (deterministic content).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int f2ord(float f) { int i = __float_as_int(f); return i >= 0 ? i : i ^ 0x7FFFFFFF; }
__device__ __forceinline__ float ord2f(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7FFFFFFF); }

__global__ void k_bbox_init(SysDev S) {
  int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q < S.T * 6) ((int *)S.bbox)[q] = (q % 6) < 3 ? 0x7FFFFFFF : (int)0x80000000;
}

__global__ void __launch_bounds__(256) k_bbox(SysDev S, int cur) {
  // grid: (blocks, T)
  const int t = blockIdx.y;
  const float4 *pos_t = S.pos[cur] + (size_t)t * S.N;
  float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < S.N; i += gridDim.x * blockDim.x) {
    float4 r = __ldg(pos_t + i);
    lo[0] = fminf(lo[0], r.x); lo[1] = fminf(lo[1], r.y); lo[2] = fminf(lo[2], r.z);
    hi[0] = fmaxf(hi[0], r.x); hi[1] = fmaxf(hi[1], r.y); hi[2] = fmaxf(hi[2], r.z);
  }
#pragma unroll
  for (int a = 0; a < 3; ++a)
    for (int o = 16; o > 0; o >>= 1) {
      lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
      hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
    }
  if ((threadIdx.x & 31) == 0) {
    int *bb = (int *)S.bbox + t * 6;
    for (int a = 0; a < 3; ++a) { atomicMin(bb + a, f2ord(lo[a])); atomicMax(bb + 3 + a, f2ord(hi[a])); }
  }
}

// grid parameters from a bounding box: cells of edge >= cell_edge, grown until they fit max_cells
__device__ __forceinline__ GridDev make_grid(const SysDev &S, const float lo[3], const float hi[3]) {
  float ext[3];
  for (int a = 0; a < 3; ++a) ext[a] = fmaxf(0.f, hi[a] - lo[a]);
  float edge = S.cell_edge;
  int n[3] = {1, 1, 1};
  for (;;) {
    // cell counts in floating point first: a structure that has blown up (the error flags say so, but the run may go
    // on) must not overflow the integer arithmetic and index out of the grid
    float nf[3];
    bool ok = true;
    for (int a = 0; a < 3; ++a) { nf[a] = floorf(ext[a] / edge) + 1.0f; ok = ok && nf[a] >= 1.0f && nf[a] < 1.0e6f; }
    if (ok && (double)nf[0] * (double)nf[1] * (double)nf[2] <= (double)S.max_cells) {
      for (int a = 0; a < 3; ++a) n[a] = (int)nf[a];
      break;
    }
    edge *= 1.25f;                       // cells may only grow: any edge >= cell_edge keeps the scan complete
    if (!(edge < 1.0e30f)) break;        // non-finite extent: one cell
  }
  GridDev gd;
  gd.ox = lo[0]; gd.oy = lo[1]; gd.oz = lo[2];
  gd.inv_edge = 1.0f / edge;
  gd.nx = n[0]; gd.ny = n[1]; gd.nz = n[2];
  gd.ncell = n[0] * n[1] * n[2];
  return gd;
}

__global__ void k_grid_setup(SysDev S) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= S.T) return;
  const int *bb = (const int *)S.bbox + t * 6;
  float lo[3], hi[3];
  for (int a = 0; a < 3; ++a) { lo[a] = ord2f(bb[a]); hi[a] = ord2f(bb[3 + a]); }
  S.grid[t] = make_grid(S, lo, hi);
}

__device__ __forceinline__ int3 cell_coords(const GridDev &gd, const float4 &r) {
  int cx = (int)floorf((r.x - gd.ox) * gd.inv_edge), cy = (int)floorf((r.y - gd.oy) * gd.inv_edge),
      cz = (int)floorf((r.z - gd.oz) * gd.inv_edge);
  cx = min(max(cx, 0), gd.nx - 1); cy = min(max(cy, 0), gd.ny - 1); cz = min(max(cz, 0), gd.nz - 1);
  return make_int3(cx, cy, cz);
}

__global__ void __launch_bounds__(256) k_cell_count(SysDev S, int cur) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= S.n_inst) return;
  const int t = g / S.N;
  const GridDev gd = S.grid[t];
  int3 c = cell_coords(gd, __ldg(S.pos[cur] + g));
  int cell = (c.z * gd.ny + c.y) * gd.nx + c.x;
  S.cell_of[g] = cell;
  atomicAdd(&S.cell_cnt[(size_t)t * S.max_cells + cell], 1);
}

// exclusive scan of the cell counts of one trajectory by one block; zeroes the counts (they become fill cursors)
__global__ void __launch_bounds__(1024) k_cell_scan(SysDev S) {
  const int t = blockIdx.x;
  const int ncell = S.grid[t].ncell;
  int *cnt = S.cell_cnt + (size_t)t * S.max_cells;
  int *start = S.cell_start + (size_t)t * (S.max_cells + 1);
  __shared__ int warp_tot[32];
  __shared__ int carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int base = 0; base < ncell; base += blockDim.x) {
    int q = base + threadIdx.x;
    int v = q < ncell ? cnt[q] : 0;
    int inc = v;
    for (int o = 1; o < 32; o <<= 1) { int n = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += n; }
    if (lane == 31) warp_tot[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      int w = lane < (blockDim.x >> 5) ? warp_tot[lane] : 0;
      int winc = w;
      for (int o = 1; o < 32; o <<= 1) { int n = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += n; }
      warp_tot[lane] = winc - w;
    }
    __syncthreads();
    int excl = carry_s + warp_tot[wid] + inc - v;
    if (q < ncell) { start[q] = excl; cnt[q] = 0; }
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry_s = excl + v;
    __syncthreads();
  }
  if (threadIdx.x == 0) start[ncell] = carry_s;
}

__global__ void __launch_bounds__(256) k_cell_fill(SysDev S) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= S.n_inst) return;
  const int t = g / S.N, i = g - t * S.N;
  const int cell = S.cell_of[g];
  int slot = atomicAdd(&S.cell_cnt[(size_t)t * S.max_cells + cell], 1);
  S.cell_bead[(size_t)t * S.N + S.cell_start[(size_t)t * (S.max_cells + 1) + cell] + slot] = i;
}

// One warp per cell: rank sort of the (distinct) bead indices so that the cell content, and with it every L1 row,
// does not depend on the order in which the atomics of k_cell_fill were served.  cell_of is free by now: scratch.
__global__ void __launch_bounds__(256) k_cell_sort(SysDev S, int cur) {
  const int t = blockIdx.y;
  const int ncell = S.grid[t].ncell;
  const int lane = threadIdx.x & 31;
  const int *start = S.cell_start + (size_t)t * (S.max_cells + 1);
  int *bead = S.cell_bead + (size_t)t * S.N;
  int *tmp = S.cell_of + (size_t)t * S.N;
  for (int c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; c < ncell; c += (gridDim.x * blockDim.x) >> 5) {
    const int s = start[c], n = start[c + 1] - s;
    for (int a = lane; a < n; a += 32) {
      int v = bead[s + a], rank = 0;
      for (int b = 0; b < n; ++b) rank += bead[s + b] < v;
      tmp[s + rank] = v;
    }
    __syncwarp();
    // sorted ids back, and the cell-sorted coordinate copy {x, y, z, bead index} the L1 build streams through
    for (int a = lane; a < n; a += 32) {
      const int v = tmp[s + a];
      bead[s + a] = v;
      const float4 r = __ldg(S.pos[cur] + (size_t)t * S.N + v);
      S.cell_pos[(size_t)t * S.N + s + a] = make_float4(r.x, r.y, r.z, __int_as_float(v));
    }
    __syncwarp();
  }
}

__device__ __forceinline__ bool is_excluded(const SysDev &S, int i, int j) {
  int lo = __ldg(&S.excl_ptr[i]), hi = __ldg(&S.excl_ptr[i + 1]);
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    int v = __ldg(&S.excl_idx[mid]);
    if (v == j) return true;
    if (v < j) lo = mid + 1; else hi = mid;
  }
  return false;
}

// a2: L1 pair-list build, one warp per bead instance: stream through the cell-sorted coordinates of the 27 cells
// around the bead ((2 SPAN + 1)^2 contiguous segments, the next 32 candidates in flight while the current ones are tested), keep
// j != i in the non-native set with pred32(R_pl); ballot + prefix-popcount compaction (row order: cells z,y,x
// ascending, beads ascending inside a cell -- deterministic; sop_get_lists returns rows sorted by the caller's index).
// The bonded / native partners are struck in a second pass over the finished row (a handful of warp iterations with the
// exclusion row held in lane registers) instead of a membership search per candidate, which was 30 % of the kernel.
constexpr int EXCL_SMEM = 64;
constexpr int CELL_SPAN = 1;            // cell edge = R_pl / CELL_SPAN, scan (2 SPAN + 1)^3 cells.  SPAN = 2 tests 42 % fewer
                                        // candidates but measured slower on cfg 3 (114 vs 89 us: 25 short segments, 8x the cells)
__global__ void __launch_bounds__(256) k_build_l1(SysDev S, int cur) {
  const int w = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int lane = threadIdx.x & 31;
  if (w >= S.n_inst) return;
  const int t = w / S.N, i = w - t * S.N;
  const float4 *__restrict__ cpos = S.cell_pos + (size_t)t * S.N;
  const GridDev gd = S.grid[t];
  const int *start = S.cell_start + (size_t)t * (S.max_cells + 1);
  int *dst = S.pl_idx + (size_t)w * S.cap_pl;
  const float4 ri = __ldg(S.pos[cur] + (size_t)t * S.N + i);
  const int e0 = __ldg(&S.excl_ptr[i]), ne = __ldg(&S.excl_ptr[i + 1]) - e0;
  const bool ex_reg = ne <= EXCL_SMEM;                 // exclusion row in two registers per lane (else: global search)
  const int ex0 = lane < ne ? __ldg(&S.excl_idx[e0 + lane]) : -1;
  const int ex1 = 32 + lane < ne ? __ldg(&S.excl_idx[e0 + 32 + lane]) : -1;
  const int3 c = cell_coords(gd, ri);
  // the (z, y) rows of cells: lane l fetches the bounds of row (l / SIDE - SPAN, l % SIDE - SPAN)
  int my_s = 0, my_e = 0;
  constexpr int SIDE = 2 * CELL_SPAN + 1, NSEG = SIDE * SIDE;
  if (lane < NSEG) {
    const int z = c.z + lane / SIDE - CELL_SPAN, y = c.y + lane % SIDE - CELL_SPAN;
    if (z >= 0 && z < gd.nz && y >= 0 && y < gd.ny) {
      const int c0 = (z * gd.ny + y) * gd.nx + max(c.x - CELL_SPAN, 0), c1 = (z * gd.ny + y) * gd.nx + min(c.x + CELL_SPAN, gd.nx - 1);
      my_s = start[c0]; my_e = start[c1 + 1];
    }
  }
  int n = 0;
  for (int seg = 0; seg < NSEG; ++seg) {
    const int s = __shfl_sync(0xffffffffu, my_s, seg), e = __shfl_sync(0xffffffffu, my_e, seg);
    // 128 candidates per iteration: four independent 16-byte loads per lane in flight, then four ordered compactions
    for (int base = s; base < e; base += 128) {
      float4 rj[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int q = base + 32 * u + lane;
        rj[u] = q < e ? __ldg(cpos + q) : make_float4(0.f, 0.f, 0.f, __int_as_float(i));
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (base + 32 * u >= e) break;
        const int q = base + 32 * u + lane;
        const int j = __float_as_int(rj[u].w);
        const bool pass = q < e && j != i && pred32(ri, rj[u], S.R_pl2) && (ex_reg || !is_excluded(S, i, j));
        const unsigned m = __ballot_sync(0xffffffffu, pass);
        if (pass) {
          const int slot = n + __popc(m & ((1u << lane) - 1u));
          if (slot < S.cap_pl) dst[slot] = j;
        }
        n += __popc(m);
      }
    }
  }
  if (n > S.cap_pl) { if (lane == 0) atomicOr(S.flags, FLAG_PL_OVERFLOW); n = S.cap_pl; }
  if (ex_reg && ne > 0) {
    // second pass, in place and order-preserving: the write index never passes the read index
    __syncwarp();
    int m2 = 0;
    for (int base = 0; base < n; base += 32) {
      const int p = base + lane;
      const int j = p < n ? dst[p] : -1;
      bool hit = false;
      for (int k = 0; k < min(ne, 32); ++k) hit |= __shfl_sync(0xffffffffu, ex0, k) == j;
      for (int k = 32; k < ne; ++k) hit |= __shfl_sync(0xffffffffu, ex1, k - 32) == j;
      const bool keep = p < n && !hit;
      const unsigned m = __ballot_sync(0xffffffffu, keep);
      if (keep) dst[m2 + __popc(m & ((1u << lane) - 1u))] = j;
      m2 += __popc(m);
    }
    n = m2;
  }
  if (lane == 0) S.pl_cnt[w] = n;
}

// R_pl = +inf: the static all-pairs L1 (Table I's "non-native pairs"), one row per bead, shared.
__global__ void __launch_bounds__(256) k_build_l1_static(SysDev S) {
  const int i = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int lane = threadIdx.x & 31;
  if (i >= S.N) return;
  int *dst = S.pl_idx + (size_t)i * S.cap_pl;
  int n = 0;
  for (int base = 0; base < S.N; base += 32) {
    int j = base + lane;
    bool pass = j < S.N && j != i && !is_excluded(S, i, j);
    unsigned m = __ballot_sync(0xffffffffu, pass);
    if (pass) {
      int slot = n + __popc(m & ((1u << lane) - 1u));
      if (slot < S.cap_pl) dst[slot] = j;
    }
    n += __popc(m);
  }
  if (lane == 0) {
    if (n > S.cap_pl) { atomicOr(S.flags, FLAG_PL_OVERFLOW); n = S.cap_pl; }
    S.pl_cnt[i] = n;
  }
}

// ------------------------------------------------------------------------------------------------
// a10: energies (Eq. (1) term by term, + external terms): fp32 pair terms, fp64 accumulation.
// 8 lanes per bead; pair terms are visited from both ends and halved.  grid = (blocks, T);
// partial[t][block][5] then k_energy_final sums the blocks in order (deterministic).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_energy(SysDev S, int cur, unsigned long long step, double *partial) {
  constexpr int G = 8;
  const int t = blockIdx.y;
  const float4 *__restrict__ pos_t = S.pos[cur] + (size_t)t * S.N;
  double e[5] = {0, 0, 0, 0, 0};
  const int lane = threadIdx.x % G;
  int flag = 0;
  for (int i = (blockIdx.x * blockDim.x + threadIdx.x) / G; i < S.N; i += gridDim.x * blockDim.x / G) {
    const int g = t * S.N + i;
    const float4 ri = __ldg(pos_t + i);
    for (int p = lane; p < S.cap_b; p += G) {
      int2 b = __ldg(&S.bond_tab[(size_t)i * S.cap_b + p]);
      if (b.x >= 0) {
        float4 rj = __ldg(pos_t + b.x);
        float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
        bool bad; float ev;
        fene_s(S, dx * dx + dy * dy + dz * dz, __int_as_float(b.y), bad, &ev);
        if (bad) flag |= FLAG_FENE; else e[0] += 0.5 * (double)ev;
      }
    }
    for (int q = __ldg(&S.nat_ptr[i]) + lane; q < __ldg(&S.nat_ptr[i + 1]); q += G) {
      int2 b = __ldg(&S.nat_tab[q]);
      float eps = S.nat_eps ? __ldg(&S.nat_eps[q]) : S.eps_native;
      float4 rj = __ldg(pos_t + b.x);
      float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
      float ev;
      native_s(dx * dx + dy * dy + dz * dz, __int_as_float(b.y), eps, &ev);
      e[1] += 0.5 * (double)ev;
    }
    const int cnt = S.nb_cnt[g];
    for (int p = lane; p < cnt; p += G) {
      int j = S.nb_idx[(size_t)g * S.cap_nb + p];
      float4 rj = __ldg(pos_t + j);
      float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
      float ev;
      rep_s(S, dx * dx + dy * dy + dz * dz, &ev);
      e[2] += 0.5 * (double)ev;
    }
    if (lane == 0) {
      const uint32_t tag = __float_as_uint(ri.w);
      if (S.has_pull && (tag & TAG_PULLED)) {
        float vs = (float)((double)S.pull_v * (double)step);
        float proj = ri.x * S.pull_nx + ri.y * S.pull_ny + ri.z * S.pull_nz - __ldg(&S.pull_adotn[i]);
        float ext = vs - proj;
        e[3] += (double)(0.5f * S.pull_k * ext * ext);
      }
      if (S.tip_on) {
        float vs = (float)((double)S.tip_v * (double)step);
        float dx = ri.x - (S.tip_cx + vs * S.tip_nx), dy = ri.y - (S.tip_cy + vs * S.tip_ny),
              dz = ri.z - (S.tip_cz + vs * S.tip_nz);
        float gap = sqrtf(dx * dx + dy * dy + dz * dz) - S.tip_R;
        if (!(gap > 0.f)) flag |= FLAG_NONFINITE;
        float ig = 1.0f / gap, ig2 = ig * ig;
        e[4] += (double)(S.tip_eps * S.tip_sigma6 * ig2 * ig2 * ig2);
      }
    }
  }
  __shared__ double red[5][8];
  const int wl = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    double v = e[k];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (wl == 0) red[k][wid] = v;
  }
  __syncthreads();
  if (threadIdx.x < 5) {
    double v = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += red[threadIdx.x][w];
    partial[((size_t)t * gridDim.x + blockIdx.x) * 5 + threadIdx.x] = v;
  }
  if (flag) atomicOr(S.flags, flag);
}

// ------------------------------------------------------------------------------------------------
// Observables per trajectory (PAPER.md:261 f(R) curves, :312-314 force-indentation): radius of
// gyration, end-to-end distance between internal beads ia and ib, cantilever force summed over the pulled beads,
// force resisting the indenter (sum_i F_i^tip . n_tip).  One block per trajectory; fp32 terms, fp64 sums, two passes
// (centre of mass, then the squared deviations).  o_out[t][4].
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double block_sum(double v, double *red) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  double tot = 0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) tot += red[w];     // same order in every thread: deterministic
  return tot;
}

__global__ void __launch_bounds__(1024) k_observables(SysDev S, int cur, unsigned long long step, int ia, int ib, double *o_out, int o_stride) {
  __shared__ double red[32];
  const int t = blockIdx.x;
  const float4 *__restrict__ pos_t = S.pos[cur] + (size_t)t * S.N;
  double sx = 0, sy = 0, sz = 0, fp = 0, ft = 0;
  int flag = 0;
  const float vs_pull = (float)((double)S.pull_v * (double)step), vs_tip = (float)((double)S.tip_v * (double)step);
  const float cx = S.tip_cx + vs_tip * S.tip_nx, cy = S.tip_cy + vs_tip * S.tip_ny, cz = S.tip_cz + vs_tip * S.tip_nz;
  for (int i = threadIdx.x; i < S.N; i += blockDim.x) {
    const float4 r = __ldg(pos_t + i);
    sx += (double)r.x; sy += (double)r.y; sz += (double)r.z;
    if (S.has_pull && (__float_as_uint(r.w) & TAG_PULLED)) {
      const float proj = r.x * S.pull_nx + r.y * S.pull_ny + r.z * S.pull_nz - __ldg(&S.pull_adotn[i]);
      fp += (double)(S.pull_k * (vs_pull - proj));
    }
    if (S.tip_on) {
      const float dx = r.x - cx, dy = r.y - cy, dz = r.z - cz;
      const float g = sqrtf(dx * dx + dy * dy + dz * dz), gap = g - S.tip_R;
      if (!(gap > 0.f)) flag |= FLAG_NONFINITE;
      const float ig = 1.0f / gap, ig2 = ig * ig;
      const float sf = 6.0f * S.tip_eps * S.tip_sigma6 * ig2 * ig2 * ig2 * ig / g;
      ft += (double)(sf * (dx * S.tip_nx + dy * S.tip_ny + dz * S.tip_nz));
    }
  }
  const double n = (double)S.N;
  const double mx = block_sum(sx, red) / n, my = block_sum(sy, red) / n, mz = block_sum(sz, red) / n;
  double s2 = 0;
  for (int i = threadIdx.x; i < S.N; i += blockDim.x) {
    const float4 r = __ldg(pos_t + i);
    const double dx = (double)r.x - mx, dy = (double)r.y - my, dz = (double)r.z - mz;
    s2 += dx * dx + dy * dy + dz * dz;
  }
  s2 = block_sum(s2, red);
  fp = block_sum(fp, red);
  ft = block_sum(ft, red);
  if (threadIdx.x == 0) {
    const float4 a = pos_t[ia], b = pos_t[ib];
    const double dx = (double)b.x - (double)a.x, dy = (double)b.y - (double)a.y, dz = (double)b.z - (double)a.z;
    double *o = o_out + (size_t)o_stride * (size_t)t;
    o[0] = sqrt(s2 / n); o[1] = sqrt(dx * dx + dy * dy + dz * dz); o[2] = fp; o[3] = ft;
  }
  if (flag) atomicOr(S.flags, flag);
}

__global__ void k_energy_final(int T, int nblk, const double *partial, double *e_out, int e_stride) {
  int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= T * 5) return;
  int t = q / 5, k = q % 5;
  double v = 0;
  for (int b = 0; b < nblk; ++b) v += partial[((size_t)t * nblk + b) * 5 + k];
  e_out[(size_t)t * e_stride + k] = v;
}

}  // namespace sop

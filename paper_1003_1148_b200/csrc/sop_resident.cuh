// sop_resident.cuh -- mode 3: the SM-resident persistent kernel (mode 3).
//
// A trajectory is cut into C chunks of consecutive beads (internal = Morton order of the native structure), one
// chunk per CTA, all CTAs co-resident.  A CTA keeps, in shared memory and for the whole launch,
//   * the coordinates of its own beads and of its halo (every bead its L1 rows, natives or bonds refer to),
//     addressed by 16-bit chunk-local "slots": own beads first, then the halo in ascending bead index;
//   * its L2 rows (Alg. 3 output) as 16-bit slots;
// so the force loop of Alg. 2 gathers with LDS only.  Per step a CTA publishes its new
// coordinates to an exchange buffer in L2 and fetches the *active* halo (slots the current L2 rows / natives / bonds
// use) of its neighbours.  There is no grid barrier: every published 8-byte word carries (value, stamp), a reader
// polls the words it needs until their stamps equal the step it is waiting for (64-bit accesses are single-copy
// atomic), so a step costs one L2 round trip and a CTA only ever waits for the CTAs it really depends on.
// Two exchange layers suffice: a CTA can only overwrite layer k with k+2 after it has read its neighbours'
// layer k+1, which they publish after they finished reading layer k.
#pragma once
#include "sop_kernels.cuh"

namespace sop {

constexpr int FLAG_SLOT_OVERFLOW = 16;

struct ResDev {
  int C;                      // chunks per trajectory
  int chunk;                  // beads per chunk (the last chunk of a trajectory may be shorter)
  int halo_cap;               // halo slots per chunk
  int implicit_l1;            // static all-pairs L1 and C == 1: the L1 row of i is "every j != i not excluded"
  int nat_entries;            // native table entries per trajectory
  int *n_halo;                // [T*C]
  int *halo_gid;              // [T*C][halo_cap] bead index (within the trajectory) of each halo slot, ascending
  unsigned short *pl_loc;     // [T*N][cap_pl]   L1 rows as slots
  unsigned short *nat_loc;    // [T][nat_entries]
  unsigned short *bond_loc;   // [T][N*cap_b]
  uint4 *xch;                 // [2][T*N][2]  {x, stamp, y, stamp} {z, stamp, -, -}
  // shared-memory carve-up (bytes from the start of dynamic shared memory), computed by the host
  int off_pos, off_g, off_carry, off_tag, off_nb, off_cnt, off_active, off_bm, off_sbm, off_misc;
  int nb_si, nb_sp;           // nb_loc(i, p) = nb[i * nb_si + p * nb_sp]
  int smem_bytes;
};

__device__ __forceinline__ float fast_rcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ void xch_put(uint4 *slot, const float4 &v, uint32_t st) {
  asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(slot), "r"(__float_as_uint(v.x)), "r"(st),
               "r"(__float_as_uint(v.y)), "r"(st) : "memory");
  asm volatile("st.volatile.global.v2.u32 [%0], {%1, %2};" ::"l"(slot + 1), "r"(__float_as_uint(v.z)), "r"(st) : "memory");
}

__device__ __forceinline__ bool xch_try(const uint4 *slot, uint32_t st, float4 &out) {
  uint32_t a0, a1, a2, a3, b0, b1;
  asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(a0), "=r"(a1), "=r"(a2), "=r"(a3) : "l"(slot) : "memory");
  asm volatile("ld.volatile.global.v2.u32 {%0, %1}, [%2];" : "=r"(b0), "=r"(b1) : "l"(slot + 1) : "memory");
  out = make_float4(__uint_as_float(a0), __uint_as_float(a2), __uint_as_float(b0), 0.f);
  return a1 == st && a3 == st && b1 == st;
}

// ------------------------------------------------------------------------------------------------
// k_localise: after an L1 build, give every chunk its halo slot table and re-express L1 rows, natives and bonds
// in chunk-local slots.  One CTA per (trajectory, chunk); dynamic shared memory: bitmap + prefix over the N beads.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512) k_localise(SysDev S, ResDev R) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int W = (S.N + 31) >> 5;
  uint32_t *bm = (uint32_t *)smem_raw;         // [W] bead j is in the halo
  uint32_t *pre = bm + W;                      // [W] exclusive prefix of popc(bm)
  __shared__ int warp_tot[32];
  __shared__ int carry_s;
  const int tc = blockIdx.x, t = tc / R.C, c = tc - t * R.C;
  const int b0 = c * R.chunk, b1 = min(S.N, b0 + R.chunk), n_own = b1 - b0;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  for (int w = threadIdx.x; w < W; w += blockDim.x) bm[w] = 0u;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  auto mark = [&](int j) { if (j < b0 || j >= b1) atomicOr(&bm[j >> 5], 1u << (j & 31)); };
  for (int i = b0 + warp; i < b1; i += nwarps) {
    const int g = t * S.N + i;
    const int cnt = S.pl_cnt[g];
    const int *row = S.pl_idx + (size_t)g * S.cap_pl;
    for (int p = lane; p < cnt; p += 32) mark(row[p]);
    for (int q = S.nat_ptr[i] + lane; q < S.nat_ptr[i + 1]; q += 32) mark(S.nat_tab[q].x);
    for (int p = lane; p < S.cap_b; p += 32) { int j = S.bond_tab[(size_t)i * S.cap_b + p].x; if (j >= 0) mark(j); }
  }
  __syncthreads();
  // exclusive scan of the word popcounts
  for (int base = 0; base < W; base += blockDim.x) {
    const int w = base + threadIdx.x;
    const int v = w < W ? __popc(bm[w]) : 0;
    int inc = v;
    for (int o = 1; o < 32; o <<= 1) { int n = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += n; }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      int x = lane < nwarps ? warp_tot[lane] : 0, xi = x;
      for (int o = 1; o < 32; o <<= 1) { int n = __shfl_up_sync(0xffffffffu, xi, o); if (lane >= o) xi += n; }
      warp_tot[lane] = xi - x;
    }
    __syncthreads();
    const int excl = carry_s + warp_tot[warp] + inc - v;
    if (w < W) pre[w] = (uint32_t)excl;
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry_s = excl + v;
    __syncthreads();
  }
  const int n_halo = carry_s;
  if (n_halo > R.halo_cap) {
    if (threadIdx.x == 0) { atomicOr(S.flags, FLAG_SLOT_OVERFLOW); R.n_halo[tc] = 0; }
    return;
  }
  if (threadIdx.x == 0) R.n_halo[tc] = n_halo;
  int *hg = R.halo_gid + (size_t)tc * R.halo_cap;
  for (int w = threadIdx.x; w < W; w += blockDim.x) {
    uint32_t bits = bm[w];
    int k = (int)pre[w];
    while (bits) { int b = __ffs(bits) - 1; bits &= bits - 1; hg[k++] = (w << 5) + b; }
  }
  auto slot_of = [&](int j) -> unsigned short {
    if (j >= b0 && j < b1) return (unsigned short)(j - b0);
    return (unsigned short)(n_own + pre[j >> 5] + __popc(bm[j >> 5] & ((1u << (j & 31)) - 1u)));
  };
  for (int i = b0 + warp; i < b1; i += nwarps) {
    const int g = t * S.N + i;
    const int cnt = S.pl_cnt[g];
    const int *row = S.pl_idx + (size_t)g * S.cap_pl;
    unsigned short *dst = R.pl_loc + (size_t)g * S.cap_pl;
    for (int p = lane; p < cnt; p += 32) dst[p] = slot_of(row[p]);
    if (R.C == 1) continue;                     // one chunk: slot = bead index, natives and bonds need no table
    for (int q = S.nat_ptr[i] + lane; q < S.nat_ptr[i + 1]; q += 32)
      R.nat_loc[(size_t)t * R.nat_entries + q] = slot_of(S.nat_tab[q].x);
    for (int p = lane; p < S.cap_b; p += 32) {
      int j = S.bond_tab[(size_t)i * S.cap_b + p].x;
      R.bond_loc[(size_t)g * S.cap_b + p] = j >= 0 ? slot_of(j) : (unsigned short)0;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Pair force laws of Eq. (1) with MUFU reciprocals (1 ulp; the parity bar is 1e-4 max|F|).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void acc_pair(const float4 &ri, const float4 &rj, float &dx, float &dy, float &dz, float &r2) {
  dx = ri.x - rj.x; dy = ri.y - rj.y; dz = ri.z - rj.z;
  r2 = dx * dx + dy * dy + dz * dz;
}

// Internal force on own bead `il` (slot il, bead index gi) from shared-memory coordinates: Alg. 2
// with the partner loop spread over G lanes; no distance test in the loop (reading R3c).
template <int G>
__device__ __forceinline__ float3 resident_force(const SysDev &S, const ResDev &R, const float4 *__restrict__ sp,
                                                 const unsigned short *__restrict__ nb, int cnt, int il, int gi, int t,
                                                 int lane, bool valid, const float4 &ri, int &flag) {
  float fx = 0.f, fy = 0.f, fz = 0.f;
  if (valid) {
    const bool multi = R.C > 1;
    // a4: FENE bonds
    for (int p = lane; p < S.cap_b; p += G) {
      const int2 e = __ldg(&S.bond_tab[(size_t)gi * S.cap_b + p]);
      if (e.x >= 0) {
        const int slot = multi ? (int)__ldg(&R.bond_loc[((size_t)t * S.N + gi) * S.cap_b + p]) : e.x;
        float dx, dy, dz, r2;
        acc_pair(ri, sp[slot], dx, dy, dz, r2);
        const float inv_r = rsqrtf(r2);
        const float del = r2 * inv_r - __int_as_float(e.y);
        const float x = 1.0f - del * del * S.inv_R0sq;
        if (!(x > 0.0f)) flag |= FLAG_FENE;
        const float s = -S.k_fene * del * fast_rcp(x) * inv_r;
        fx += s * dx; fy += s * dy; fz += s * dz;
      }
    }
    // a5: native contacts
    {
      const int q0 = __ldg(&S.nat_ptr[gi]), q1 = __ldg(&S.nat_ptr[gi + 1]);
      for (int q = q0 + lane; q < q1; q += G) {
        const int2 e = __ldg(&S.nat_tab[q]);
        const float eps = S.nat_eps ? __ldg(&S.nat_eps[q]) : S.eps_native;
        const int slot = multi ? (int)__ldg(&R.nat_loc[(size_t)t * R.nat_entries + q]) : e.x;
        float dx, dy, dz, r2;
        acc_pair(ri, sp[slot], dx, dy, dz, r2);
        const float inv_r2 = fast_rcp(r2);
        const float u = __int_as_float(e.y) * inv_r2;
        const float q3 = u * u * u;
        const float s = 12.0f * eps * inv_r2 * (q3 * q3 - q3);
        fx += s * dx; fy += s * dy; fz += s * dz;
      }
    }
    // a6: non-native repulsion over the shared-memory neighbor list
    {
      const unsigned short *row = nb + (size_t)il * R.nb_si;
      for (int p = lane; p < cnt; p += G) {
        const int slot = row[(size_t)p * R.nb_sp];
        float dx, dy, dz, r2;
        acc_pair(ri, sp[slot], dx, dy, dz, r2);
        const float inv_r2 = fast_rcp(r2);
        const float s = S.c_rep_f * (inv_r2 * inv_r2) * (inv_r2 * inv_r2);
        fx += s * dx; fy += s * dy; fz += s * dz;
      }
    }
  }
  if (G > 1) { fx = group_sum<G>(fx); fy = group_sum<G>(fy); fz = group_sum<G>(fz); }
  return make_float3(fx, fy, fz);
}

__device__ __forceinline__ int lower_bound_dev(const int *__restrict__ a, int n, int v) {
  int lo = 0, hi = n;
  while (lo < hi) { int mid = (lo + hi) >> 1; if (__ldg(&a[mid]) < v) lo = mid + 1; else hi = mid; }
  return lo;
}

// ------------------------------------------------------------------------------------------------
// k_resident: a3 + a4..a9 for n_steps Langevin steps of one chunk per CTA (see the header of this file).
// Shared-memory buffers are double-buffered on the step parity, so a step needs one __syncthreads:
//   (a) noise of this step, thread per bead        (b) fetch the active halo of this step's layer
//   (c) __syncthreads                              (d) forces (G lanes per bead) + update + publish
//   (e) every nb_interval steps: fetch the whole halo of the new layer, Alg. 3 on the own rows, new active set.
// ------------------------------------------------------------------------------------------------
template <int G, bool COMP>
__global__ void __launch_bounds__(1024, 1) k_resident(SysDev S, ResDev R, int cur, unsigned long long step0, int n_steps,
                                                      int nb_interval, int filter_last, uint32_t stamp0) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int slots_cap = R.chunk + R.halo_cap;
  float4 *spos = (float4 *)(smem_raw + R.off_pos);                   // [2][slots_cap]
  float4 *sg = (float4 *)(smem_raw + R.off_g);                       // [2][chunk]   (G > 1)
  float4 *scarry = (float4 *)(smem_raw + R.off_carry);               // [chunk]      (COMP)
  uint32_t *stag = (uint32_t *)(smem_raw + R.off_tag);               // [chunk]
  unsigned short *nb = (unsigned short *)(smem_raw + R.off_nb);      // L2 rows as slots
  unsigned short *cnt_s = (unsigned short *)(smem_raw + R.off_cnt);  // [chunk]
  unsigned short *active = (unsigned short *)(smem_raw + R.off_active);
  uint32_t *bm = (uint32_t *)(smem_raw + R.off_bm), *sbm = (uint32_t *)(smem_raw + R.off_sbm);
  int *misc = (int *)(smem_raw + R.off_misc);                        // [0] = number of active halo slots

  const int tc = blockIdx.x, t = tc / R.C, c = tc - t * R.C;
  const int b0 = c * R.chunk, b1 = min(S.N, b0 + R.chunk), n_own = b1 - b0;
  const bool multi = R.C > 1;
  const int n_halo = multi ? R.n_halo[tc] : 0;
  const int *__restrict__ hgid = R.halo_gid + (size_t)tc * R.halo_cap;
  const int HW = (n_halo + 31) >> 5;
  const int tid = threadIdx.x, bd = blockDim.x;
  const int lane = tid % G, grp = tid / G, groups = bd / G;
  const int wlane = tid & 31, warp = tid >> 5, nwarps = bd >> 5;
  const size_t inst0 = (size_t)t * S.N;
  uint4 *const xl0 = R.xch, *const xl1 = R.xch + 2 * (size_t)S.n_inst;
  int flag = 0;

  // ---- prologue: own coordinates, carry, tags; canonical L2 rows -> slots; static part of the active set
  for (int i = tid; i < n_own; i += bd) {
    const float4 v = S.pos[cur][inst0 + b0 + i];
    spos[i] = v;
    stag[i] = __float_as_uint(v.w);
    if (multi) xch_put(xl0 + 2 * (inst0 + b0 + i), v, stamp0);
    if (COMP) scarry[i] = S.carry[inst0 + b0 + i];
  }
  for (int il = warp; il < n_own; il += nwarps) {
    const size_t g = inst0 + b0 + il;
    const int cnt = min(S.nb_cnt[g], S.cap_nb);
    const int *row = S.nb_idx + g * S.cap_nb;
    for (int p = wlane; p < cnt; p += 32) {
      const int j = row[p];
      const int slot = (j >= b0 && j < b1) ? j - b0 : n_own + lower_bound_dev(hgid, n_halo, j);
      nb[(size_t)il * R.nb_si + (size_t)p * R.nb_sp] = (unsigned short)slot;
    }
    if (wlane == 0) cnt_s[il] = (unsigned short)cnt;
  }
  for (int w = tid; w < HW; w += bd) sbm[w] = 0u;
  __syncthreads();
  if (multi) {
    for (int il = warp; il < n_own; il += nwarps) {
      const int gi = b0 + il;
      for (int q = S.nat_ptr[gi] + wlane; q < S.nat_ptr[gi + 1]; q += 32) {
        const int h = (int)R.nat_loc[(size_t)t * R.nat_entries + q] - n_own;
        if (h >= 0) atomicOr(&sbm[h >> 5], 1u << (h & 31));
      }
      for (int p = wlane; p < S.cap_b; p += 32)
        if (S.bond_tab[(size_t)gi * S.cap_b + p].x >= 0) {
          const int h = (int)R.bond_loc[(inst0 + gi) * S.cap_b + p] - n_own;
          if (h >= 0) atomicOr(&sbm[h >> 5], 1u << (h & 31));
        }
    }
  }
  // active halo = static part + slots of the current L2 rows (3 barriers)
  auto build_active = [&]() {
    for (int w = tid; w < HW; w += bd) bm[w] = sbm[w];
    if (tid == 0) misc[0] = 0;
    __syncthreads();
    if (multi) {
      for (int il = warp; il < n_own; il += nwarps) {
        const int cnt = cnt_s[il];
        for (int p = wlane; p < cnt; p += 32) {
          const int h = (int)nb[(size_t)il * R.nb_si + (size_t)p * R.nb_sp] - n_own;
          if (h >= 0) atomicOr(&bm[h >> 5], 1u << (h & 31));
        }
      }
    }
    __syncthreads();
    for (int w = tid; w < HW; w += bd) {
      uint32_t bits = bm[w];
      if (bits) {
        int at = atomicAdd(&misc[0], __popc(bits));
        while (bits) { const int b = __ffs(bits) - 1; bits &= bits - 1; active[at++] = (unsigned short)(n_own + (w << 5) + b); }
      }
    }
    __syncthreads();
  };
  __syncthreads();
  build_active();

  // ---- the steps
  bool have_full = false;                    // the whole halo of the current layer is already in shared memory
  for (int k = 0; k < n_steps; ++k) {
    const unsigned long long step = step0 + (unsigned long long)k;
    float4 *pc = spos + (size_t)(k & 1) * slots_cap, *pn = spos + (size_t)((k & 1) ^ 1) * slots_cap;
    float4 *gc = sg + (size_t)(k & 1) * R.chunk;
    uint4 *const xc = (k & 1) ? xl1 : xl0, *const xn = (k & 1) ? xl0 : xl1;
    const uint32_t st_c = stamp0 + (uint32_t)k, st_n = st_c + 1u;
    // (a) a8: noise of this step, one thread per bead (the lanes of a group would otherwise idle through it)
    if (G > 1) {
      for (int i = tid; i < n_own; i += bd) {
        const uint32_t tag = stag[i];
        if (!(tag & TAG_FIXED)) {
          const float3 gn = gaussian3(S, tag & TAG_ID_MASK, (uint32_t)(S.traj_offset + t), step);
          gc[i] = make_float4(gn.x, gn.y, gn.z, 0.f);
        }
      }
    }
    // (b) active halo of layer k: poll until the neighbours have published it
    if (multi && !have_full) {
      const int na = misc[0];
      for (int q = bd - 1 - tid; q < na; q += bd) {
        const int slot = active[q];
        const uint4 *src = xc + 2 * (inst0 + hgid[slot - n_own]);
        float4 v;
        while (!xch_try(src, st_c, v)) {}
        pc[slot] = v;
      }
    }
    have_full = false;
    __syncthreads();                                                                       // (c)
    // (d) a4..a7 forces, a9 update, publish
    for (int base = 0; base < n_own; base += groups) {
      const int il = base + grp;
      const bool valid = il < n_own;
      const int ii = valid ? il : 0, gi = b0 + ii;
      const float4 ri = pc[ii];
      float3 f = resident_force<G>(S, R, pc, nb, valid ? (int)cnt_s[ii] : 0, ii, gi, t, lane, valid, ri, flag);
      if (valid && lane == 0) {
        const uint32_t tag = stag[ii];
        float4 out = ri;
        if (!(tag & TAG_FIXED)) {
          external_force(S, gi, ri, tag, step, f.x, f.y, f.z, flag);
          float3 gn;
          if (G > 1) { const float4 g4 = gc[ii]; gn = make_float3(g4.x, g4.y, g4.z); }
          else gn = gaussian3(S, tag & TAG_ID_MASK, (uint32_t)(S.traj_offset + t), step);
          out = langevin_apply<COMP>(S, ri, gn, f.x, f.y, f.z, COMP ? scarry + ii : nullptr, flag);
        }
        pn[ii] = out;
        if (multi) xch_put(xn + 2 * (inst0 + gi), out, st_n);
      }
    }
    // (e) a3: Alg. 3 on the own rows from the coordinates just written (list invariant)
    if ((step + 1) % (unsigned long long)nb_interval == 0 && (k + 1 < n_steps || filter_last)) {
      if (multi)
        for (int q = tid; q < n_halo; q += bd) {
          const uint4 *src = xn + 2 * (inst0 + hgid[q]);
          float4 v;
          while (!xch_try(src, st_n, v)) {}
          pn[n_own + q] = v;
        }
      __syncthreads();
      for (int il = warp; il < n_own; il += nwarps) {
        const int gi = b0 + il;
        const size_t g = inst0 + gi;
        const float4 ri = pn[il];
        int *canon = S.nb_idx + g * S.cap_nb;
        unsigned short *row = nb + (size_t)il * R.nb_si;
        int n = 0;
        const int cnt1 = R.implicit_l1 ? S.N : S.pl_cnt[g];
        const unsigned short *src = R.pl_loc + g * S.cap_pl;
        for (int base = 0; base < cnt1; base += 32) {
          const int p = base + wlane;
          int slot = 0;
          bool pass = false;
          if (p < cnt1) {
            slot = R.implicit_l1 ? p : (int)src[p];
            pass = pred32(ri, pn[slot], S.R_nb2);
            if (R.implicit_l1) pass = pass && p != gi && !is_excluded(S, gi, p);
          }
          const unsigned m = __ballot_sync(0xffffffffu, pass);
          if (pass) {
            const int at = n + __popc(m & ((1u << wlane) - 1u));
            if (at < S.cap_nb) {
              row[(size_t)at * R.nb_sp] = (unsigned short)slot;
              canon[at] = slot < n_own ? b0 + slot : hgid[slot - n_own];
            }
          }
          n += __popc(m);
        }
        if (n > S.cap_nb) { flag |= FLAG_NB_OVERFLOW; n = S.cap_nb; }
        if (wlane == 0) { cnt_s[il] = (unsigned short)n; S.nb_cnt[g] = n; }
      }
      build_active();
      have_full = true;
    }
  }

  // ---- epilogue: the current layer back to the canonical arrays
  __syncthreads();
  const float4 *pf = spos + (size_t)(n_steps & 1) * slots_cap;
  for (int i = tid; i < n_own; i += bd) {
    S.pos[cur][inst0 + b0 + i] = pf[i];
    if (COMP) S.carry[inst0 + b0 + i] = scarry[i];
  }
  if (flag) atomicOr(S.flags, flag);
}

}  // namespace sop

// sop_resident2.cuh -- mode 3 for a trajectory cut into several chunks: the SM-resident persistent kernel, second design
// (mode 3; the first design, sop_resident.cuh, stays for one-chunk trajectories and as a fallback).
//
// What the first design measured (profiles/r1p_*, r2a_*): the step was a chain of serial phases (halo poll -> pair forces ->
// update -> filter), the pair phase was bound by shared-memory gathers that collide 2.3x on the eight 16-byte bank groups, and
// half of the issue slots went to bookkeeping.  This kernel changes the structure, not the arithmetic:
//
//  * FOUR LANES PER BEAD, ROWS DEALT BY RESIDUE.  A 128-bit LDS is served a quarter-warp (8 lanes = 2 beads) at a time and
//    two of its gathers collide when the partners sit in the same 16-byte bank group (index mod 8).  Which partner sits
//    where in a bead's row is free (Alg. 2 sums over the row), so the entries of a row are put in the order of
//    index mod 8 and dealt round-robin to its groups of 4: the four gathers of a bead never collide with each other.
//    Natives and L2 partners share ONE row of 8-byte entries {byte offset of the partner's coordinate, par}, and one
//    branch-free law: s = A (1/r^2) (q max(q, 0) - q), q = (par/r^2)^3.  A native has par = r0^2 > 0: s = A (q^2 - q)/r^2, the
//    12-6 term with A = 12 eps; an L2 partner has par = -(6 eps_r sigma^6 / A)^(1/3) < 0: q < 0 and s = A |q|/r^2 =
//    6 eps_r sigma^6 / r^8 (Eq. (1)).
//  * OWN PARTNERS FIRST.  A row is [groups of own-chunk partners][groups of halo partners]; the own groups of step k+1 are
//    evaluated while the neighbours' coordinates are still in flight, so the L2 round trip of the exchange hides behind them.
//  * SERVICE WARPS.  Four warps do not compute forces: they draw the next step's noise (a8) and poll the exchange slots of
//    the active halo (four independent 256-bit loads in flight per lane) into the other time layer, then release the compute
//    warps through a named barrier (producer/consumer, bar.arrive / bar.sync).  Compute warps never wait on global memory.
//  * FUSED UPDATE.  a7 + a9 run in one lane of each bead's group right after its reduction; there is no update phase and
//    no second block-wide barrier.
//  * The L1 rows stay in global memory (L2), already dealt by residue by k_arrange_l1 and split own / halo; the filter
//    (Alg. 3) reads them 8 entries per quarter-warp, coalesced, every nb_interval steps, and writes the
//    force rows directly: a lane's survivors come out in residue order already (it always tests the same place of every
//    dealt L1 group), so the natives (sorted once per launch) followed by the survivors in lane order are dealt as they are.
// The exchange protocol (step layers + filter layers, bounded waits) is the one described in sop_resident.cuh.
#pragma once
#include "sop_resident.cuh"

namespace sop {

constexpr int R2_MAXP = 4;             // own beads per group of four lanes (register accumulators)
constexpr int R2_MAXR = 4;             // rows a quarter-warp filters per call (survivor masks in registers)
constexpr int R2_SERVICE_WARPS = 4;
constexpr int R2_MAXQ = 4;             // exchange slots a service lane polls at a time (independent 256-bit loads in flight)
constexpr unsigned R2_FIRST_POLL_NS = 50;   // pause between the end of a step and the first poll of the neighbours' layer
constexpr int R2_HALO_FLAG = 0x8000;   // 16-bit partner codes: own index, or R2_HALO_FLAG | halo index

struct Res2Dev {
  int P;                    // own beads per group of four lanes
  int n_cwarps;             // compute warps
  int n_swarps;             // service warps (the block has n_cwarps + n_swarps warps)
  int own_pad, halo_pad;    // index of the first of the eight dummy slots (one per bank group) of the own / halo region
  int own_stride;           // float4 elements of one own time layer (own_pad + 8)
  int halo_stride;          // float4 elements of one halo time layer (halo_pad + 8)
  int cap_arr;              // row stride (16-bit entries) of pl_arr
  unsigned short *pl_arr;   // [T*N][cap_arr] L1 rows dealt by residue: [G_o groups of own indices][G_h groups of halo indices]
  uchar2 *pl_g;             // [T*N] {G_o, G_h}
  int rows_cap;             // 8-byte entries of shared memory for the force rows of a chunk
  float a_ref;              // A of the force rows: 12 eps_native (1 if that is zero; the natives then contribute nothing and are left out)
  float par_rep;            // par of an L2 partner: -(6 eps_r sigma^6 / A)^(1/3)
  int off_own, off_halo, off_g, off_carry, off_tag, off_rows, off_eps, off_rowofs, off_rowg, off_nat, off_nateps, off_natq, off_natc,
      off_bond, off_cnt, off_active, off_bm, off_sbm, off_misc, off_order, off_taus, off_ext;
  int smem_bytes;
};

// ------------------------------------------------------------------------------------------------
// k_arrange_l1: after k_localise, deal every L1 row by residue.  One warp per row.  Input: the row in slot form (own
// beads first, then the halo; R.pl_loc).  Output: [own segment][halo segment], each segment sorted by (index mod 8) and
// dealt round-robin to its groups of 8, so that the 8 entries a quarter-warp gathers together fall into different bank
// groups; free positions hold the dummy index of their position (a point 1e18 A away: the predicate is false).
// Ranks come from match.any + popc in lane order: deterministic.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_arrange_l1(SysDev S, ResDev R, Res2Dev Q) {
  __shared__ int hist_s[8][16], run_s[8][16];
  const int w = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  if (w >= S.n_inst) return;
  const int t = w / S.N, i = w - t * S.N;
  const int c = i / R.chunk, b0 = c * R.chunk, n_own = min(S.N, b0 + R.chunk) - b0;
  const int cnt = min(S.pl_cnt[w], S.cap_pl);
  const unsigned short *src = R.pl_loc + (size_t)w * S.cap_pl;
  unsigned short *dst = Q.pl_arr + (size_t)w * Q.cap_arr;
  int *hist = hist_s[wib], *run = run_s[wib];
  if (lane < 16) { hist[lane] = 0; run[lane] = 0; }
  __syncwarp();
  const unsigned lt = (1u << lane) - 1u;
  auto key_of = [&](int e) { return e < n_own ? (e & 7) : 8 + ((e - n_own) & 7); };
  for (int base = 0; base < cnt; base += 32) {
    const int p = base + lane;
    const int key = p < cnt ? key_of((int)src[p]) : 32 + lane;
    const unsigned m = __match_any_sync(0xffffffffu, key);
    if (p < cnt && (m & lt) == 0u) hist[key] += __popc(m);      // the lowest lane of every key present: distinct addresses
    __syncwarp();
  }
  // exclusive prefix of the 8 counts of each segment
  int v = lane < 16 ? hist[lane] : 0, inc = v;
  for (int o = 1; o < 8; o <<= 1) { const int n = __shfl_up_sync(0xffffffffu, inc, o, 8); if ((lane & 7) >= o) inc += n; }
  const int n_o = __shfl_sync(0xffffffffu, inc, 7), n_h = __shfl_sync(0xffffffffu, inc, 15);
  const int G_o = (n_o + 7) >> 3, G_h = (n_h + 7) >> 3;
  if (lane < 16) hist[lane] = inc - v;
  // every position starts as the dummy of its place in the group
  for (int p = lane; p < 8 * (G_o + G_h); p += 32) dst[p] = (unsigned short)((p < 8 * G_o ? Q.own_pad : Q.halo_pad) + (p & 7));
  __syncwarp();
  for (int base = 0; base < cnt; base += 32) {
    const int p = base + lane;
    const int e = p < cnt ? (int)src[p] : 0;
    const int key = p < cnt ? key_of(e) : 32 + lane;
    const unsigned m = __match_any_sync(0xffffffffu, key);
    if (p < cnt) {
      const int k = hist[key] + run[key] + __popc(m & lt);
      const bool halo = key >= 8;
      const int G = halo ? G_h : G_o;
      dst[(halo ? 8 * G_o : 0) + 8 * (k % G) + k / G] = (unsigned short)(halo ? e - n_own : e);
    }
    __syncwarp();
    if (p < cnt && (m & lt) == 0u) run[key] += __popc(m);
    __syncwarp();
  }
  if (lane == 0) Q.pl_g[w] = make_uchar2((unsigned char)G_o, (unsigned char)G_h);
}

__device__ __forceinline__ void bar_sync_named(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void bar_arrive_named(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }

// Shared memory through 32-bit addresses: one register per pointer and plain LDS/STS in the hot loops (generic 64-bit
// pointers that ptxas cannot prove shared cost two registers and a window computation each time they are rebuilt).
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float4 lds_f4(uint32_t a) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ uint2 lds_u2(uint32_t a) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ float lds_f(uint32_t a) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ uint32_t lds_u(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts_f4(uint32_t a, const float4 &v) {
  asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// ------------------------------------------------------------------------------------------------
// k_res2: a3 + a4..a9 for n_steps Langevin steps of one chunk per CTA.  P = own beads per group of four lanes; EPS = the
// topology has per-contact native eps (one more 4-byte row of shared memory, one more LDS per entry).
// Force rows: groups of R2_GS = 4 entries of 8 bytes {byte offset of the partner's coordinate in its region, par};
// row = [H_o groups of own partners][H_h groups of halo partners]; entry k of a segment sits in group k mod H, place k / H.
// ------------------------------------------------------------------------------------------------
constexpr int R2_GS = 4;

template <bool COMP, bool EPS, int P>
__global__ void __launch_bounds__(1024, 1) k_res2(SysDev S, ResDev R, Res2Dev Q, int cur, unsigned long long step0, int n_steps,
                                                  int nb_interval, int filter_flags, uint32_t stamp0) {
  extern __shared__ __align__(16) unsigned char smem_raw[];     // (dynamic shared memory starts 1024-byte aligned)
  const bool filter_last = filter_flags & 1, filter_first = filter_flags & 2;
  float4 *own = (float4 *)(smem_raw + Q.off_own);                     // [2][own_stride] own coordinates, two time layers
  float4 *halo = (float4 *)(smem_raw + Q.off_halo);                   // [2][halo_stride] halo coordinates, two time layers
  float4 *sg = (float4 *)(smem_raw + Q.off_g);                        // [2][chunk] noise, two time layers
  float4 *scarry = (float4 *)(smem_raw + Q.off_carry);                // [chunk] (COMP)
  uint32_t *stag = (uint32_t *)(smem_raw + Q.off_tag);                // [chunk]
  uint2 *rows = (uint2 *)(smem_raw + Q.off_rows);                     // force rows
  float *rows_eps = (float *)(smem_raw + Q.off_eps);                  // [rows_cap] A of every entry (EPS)
  unsigned short *rowofs = (unsigned short *)(smem_raw + Q.off_rowofs);   // [chunk] first group of every row
  uchar2 *rowg = (uchar2 *)(smem_raw + Q.off_rowg);                   // [chunk] {own groups, all groups}
  uint2 *snat = (uint2 *)(smem_raw + Q.off_nat);                      // [nat_cap] natives as entries, per bead: own partners, then halo
  float *snat_eps = (float *)(smem_raw + Q.off_nateps);               //           partners, each in the order of index mod 8 (static)
  int *natq = (int *)(smem_raw + Q.off_natq);                         // [chunk + 1] offsets into the native table
  uchar2 *natc = (uchar2 *)(smem_raw + Q.off_natc);                   // [chunk] {own natives, halo natives}
  int2 *sbond = (int2 *)(smem_raw + Q.off_bond);                      // [chunk][cap_b] {byte offset | halo bit 31, or -1; bits(r0)}
  unsigned short *cnt_s = (unsigned short *)(smem_raw + Q.off_cnt);   // [chunk] L2 row counts
  unsigned short *active = (unsigned short *)(smem_raw + Q.off_active);   // halo indices the force rows / bonds use
  uint32_t *bm = (uint32_t *)(smem_raw + Q.off_bm), *sbm = (uint32_t *)(smem_raw + Q.off_sbm);
  int *misc = (int *)(smem_raw + Q.off_misc);                         // [0] active count, [1] groups used, [2] overflow, [16..271] bins of the
                                                                      // counting sorts
  unsigned short *order = (unsigned short *)(smem_raw + Q.off_order); // [2][chunk] own beads in processing order (current, next)
  uint4 *staus = (uint4 *)(smem_raw + Q.off_taus);                    // [chunk] Hybrid Taus states (rng = 1)
  float4 *sext = (float4 *)(smem_raw + Q.off_ext);                    // [2] step-dependent scalars of the external forces

  const int tc = blockIdx.x, t = tc / R.C, c = tc - t * R.C;
  const int b0 = c * R.chunk, b1 = min(S.N, b0 + R.chunk), n_own = b1 - b0;
  const int n_halo = R.n_halo[tc];
  const int *__restrict__ hgid = R.halo_gid + (size_t)tc * R.halo_cap;
  const int HW = (n_halo + 31) >> 5;
  const int tid = threadIdx.x, bd = blockDim.x;
  const int wlane = tid & 31, warp = tid >> 5, nwarps = bd >> 5;
  const int NC = Q.n_cwarps * 32, NS = Q.n_swarps * 32;              // compute / service threads
  const bool is_service = warp >= Q.n_cwarps;
  const int l8 = tid & 7, qw = tid >> 3, nqw = bd >> 3, qiw = (tid >> 3) & 3;   // quarter-warps (list work: a row each)
  const size_t inst0 = (size_t)t * S.N;
  uint4 *const xs0 = R.xch, *const xs1 = R.xch + 2 * (size_t)S.n_inst;
  uint4 *const xf0 = R.xchf, *const xf1 = R.xchf + 2 * (size_t)S.n_inst;
  const int cap_b = S.cap_b, cap_nb = S.cap_nb;
  const uint32_t traj = (uint32_t)(S.traj_offset + t);
  const bool skip_nat = !EPS && !(S.eps_native > 0.0f);              // eps_native = 0: the natives contribute exactly nothing
  const uint32_t par_rep = __float_as_uint(Q.par_rep);
  const unsigned lt = (1u << wlane) - 1u;
  int flag = 0;
  enum { BAR_END_C = 1, BAR_END_S = 2, BAR_HALO = 4 };  // named barriers; END_S and HALO alternate with the step parity

  auto draw = [&](int i, uint32_t tag, unsigned long long step) -> float4 {      // a8: the three normals of one bead and step
    float3 gn;
    if (S.taus) { uint4 y = staus[i]; const uint32_t x0 = taus_draw(y), x1 = taus_draw(y), x2 = taus_draw(y), x3 = taus_draw(y); staus[i] = y; gn = box_muller3(x0, x1, x2, x3); }
    else gn = gaussian3(S, tag & TAG_ID_MASK, traj, step);
    return make_float4(gn.x, gn.y, gn.z, 0.f);
  };
  auto put_ext = [&](int layer, unsigned long long step) {
    const ExtStep e = ext_step(S, step);
    sext[layer] = make_float4(e.vs_pull, e.cx, e.cy, e.cz);
  };

  // ---- prologue -----------------------------------------------------------------------------------------------
  const int qbase = S.nat_ptr[b0];
  unsigned fpar = (unsigned)((step0 / (unsigned long long)nb_interval) & 1ull);       // filter layer of the prologue
  if (tid < 8) {       // eight points 1e18 A away, one per bank group: their terms underflow to exactly zero
    const float4 far = make_float4(1.0e18f, 1.0e18f, 1.0e18f, 0.f);
    own[Q.own_pad + tid] = far; own[Q.own_stride + Q.own_pad + tid] = far;
    halo[Q.halo_pad + tid] = far; halo[Q.halo_stride + Q.halo_pad + tid] = far;
  }
  if (tid == 0) put_ext(0, step0);
  for (int i = tid; i < n_own; i += bd) {
    const float4 v = S.pos[cur][inst0 + b0 + i];
    own[i] = v;
    const uint32_t tag = __float_as_uint(v.w);
    stag[i] = tag;
    xch_put((fpar ? xf1 : xf0) + 2 * (inst0 + b0 + i), v, stamp0);
    if (COMP) scarry[i] = S.carry[inst0 + b0 + i];
    natq[i] = S.nat_ptr[b0 + i];
    if (S.taus) staus[i] = S.taus[inst0 + b0 + i];
    if (!(tag & TAG_FIXED)) sg[i] = draw(i, tag, step0);
  }
  if (tid == 0) natq[n_own] = S.nat_ptr[b1];
  {
    const int2 *bond_src = R.bond_pack + (inst0 + b0) * cap_b;
    for (int e = tid; e < n_own * cap_b; e += bd) {
      int2 b = bond_src[e];
      if (b.x >= 0) b.x = b.x >= n_own ? (int)(0x80000000u | (uint32_t)((b.x - n_own) * 16)) : b.x * 16;
      else b.x = -1;
      sbond[e] = b;
    }
  }
  for (int w = tid; w < HW; w += bd) sbm[w] = 0u;
  for (int b = tid; b < 256; b += bd) misc[16 + b] = 0;
  for (int q = tid; q < n_halo; q += bd) {          // the whole halo of the first layer, through the exchange
    float4 v;
    xch_wait((fpar ? xf1 : xf0) + 2 * (inst0 + hgid[q]), stamp0, v, S.flags);
    halo[q] = v;
  }
  __syncthreads();
  // processing order: own beads by descending native degree (counting sort), so that the beads of a warp run similar
  // numbers of groups.  Which lanes handle a bead does not change its force.
  {
    int *hist = misc + 16;
    for (int i = tid; i < n_own; i += bd) atomicAdd(&hist[63 - min(63, natq[i + 1] - natq[i])], 1);
    __syncthreads();
    if (tid == 0) { int run = 0; for (int b = 0; b < 64; ++b) { const int c2 = hist[b]; hist[b] = run; run += c2; } }
    __syncthreads();
    for (int i = tid; i < n_own; i += bd) order[atomicAdd(&hist[63 - min(63, natq[i + 1] - natq[i])], 1)] = (unsigned short)i;
  }
  // static part of the active set: halo beads that bonds refer to (the natives' follow below)
  for (int e = tid; e < n_own * cap_b; e += bd) {
    const int code = sbond[e].x;
    if (code != -1 && code < 0) { const int h = (int)(((uint32_t)code & 0x7FFFFFFFu) >> 4); atomicOr(&sbm[h >> 5], 1u << (h & 31)); }
  }
  // natives -> entries {byte offset, r0^2}, per bead [own partners][halo partners], each in the order of index mod 8.
  // A quarter-warp per bead; ranks from match.any + popc in lane order (deterministic); the row region is scratch here.
  {
    int *h16 = (int *)rows + (warp * 4 + qiw) * 16;
    const int2 *nat_glob = R.nat_pack + (size_t)t * R.nat_entries;
    for (int base = 0; base < n_own; base += nqw) {
      const int il = base + qw;
      const bool valid = il < n_own;
      const int q0 = valid ? natq[il] : 0;
      const int nn = valid ? natq[il + 1] - q0 : 0;
      h16[l8] = 0; h16[8 + l8] = 0;
      __syncwarp();
      const int slabs = __reduce_max_sync(0xffffffffu, (nn + 7) >> 3);
      for (int m = 0; m < slabs; ++m) {
        const int e = 8 * m + l8;
        int key = 64 + wlane;
        if (e < nn) { const int s = nat_glob[q0 + e].x; key = (qiw << 4) | (s >= n_own ? 8 | ((s - n_own) & 7) : (s & 7)); }
        const unsigned peers = __match_any_sync(0xffffffffu, key);
        if (e < nn && (peers & lt) == 0u) h16[key & 15] += __popc(peers);
        __syncwarp();
      }
      const int co = h16[l8], ch = h16[8 + l8];
      int io = co, ih = ch;
      for (int o = 1; o < 8; o <<= 1) {
        const int vo = __shfl_up_sync(0xffffffffu, io, o, 8), vh = __shfl_up_sync(0xffffffffu, ih, o, 8);
        if (l8 >= o) { io += vo; ih += vh; }
      }
      const int n_o = __shfl_sync(0xffffffffu, io, 7, 8), n_h = __shfl_sync(0xffffffffu, ih, 7, 8);
      __syncwarp();
      h16[l8] = io - co; h16[8 + l8] = n_o + ih - ch;         // first position of every (segment, residue)
      if (valid && l8 == 0) natc[il] = make_uchar2((unsigned char)min(n_o, 255), (unsigned char)min(n_h, 255));
      if (n_o > 255 || n_h > 255) flag |= FLAG_SLOT_OVERFLOW;
      __syncwarp();
      for (int m = 0; m < slabs; ++m) {
        const int e = 8 * m + l8;
        int key = 64 + wlane;
        int2 en = make_int2(0, 0);
        if (e < nn) { en = nat_glob[q0 + e]; key = (qiw << 4) | (en.x >= n_own ? 8 | ((en.x - n_own) & 7) : (en.x & 7)); }
        const unsigned peers = __match_any_sync(0xffffffffu, key);
        if (e < nn) {
          const int pos = q0 - qbase + h16[key & 15] + __popc(peers & lt);
          const int idx = en.x >= n_own ? en.x - n_own : en.x;
          snat[pos] = make_uint2((uint32_t)(idx * 16), (uint32_t)en.y);
          if (EPS) snat_eps[pos] = 12.0f * __ldg(S.nat_eps + q0 + e);
          if (en.x >= n_own) { const uint32_t bit = 1u << (idx & 31); if (!(((volatile uint32_t *)sbm)[idx >> 5] & bit)) atomicOr(&sbm[idx >> 5], bit); }
        }
        __syncwarp();
        if (e < nn && (peers & lt) == 0u) h16[key & 15] += __popc(peers);
        __syncwarp();
      }
    }
  }
  __syncthreads();
#ifdef SOP_PHASE_CLOCKS
  // profiling builds: raw clock64 stamps of the events of ONE step (the middle of the launch) per warp; a stamp taken after
  // a barrier depends on a shared-memory load issued after it (BAR.SYNC does not block the instructions that follow it)
  long long pc_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  if (tid == 0) *(long long *)(misc + 12) = clock64();
  __syncthreads();
  const long long pc_t0 = *(long long *)(misc + 12);      // one origin for the whole CTA
  int pc_step = -1;
  const uint32_t pc_probe = smem_u32(misc);
#define R2_TICK(n) { if (pc_step == n_steps / 2 + 3) { uint32_t dep_; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(dep_) : "r"(pc_probe) : "memory"); \
    long long now_; asm volatile("mov.u64 %0, %%clock64;" : "=l"(now_) : "r"(dep_) : "memory"); pc_acc[n] = now_ - pc_t0; } }
#else
#define R2_TICK(n)
#endif

  // ---- list work: every thread of the block, a quarter-warp per row ------------------------------------------------
  // exclusive scan of the rows' group counts -> rowofs (warp 0), capacity check; then the active halo set is reset
  // The processing order is re-sorted by (own groups, halo groups) so that the eight beads of a warp run the same number
  // of iterations; it goes to the second half of `order` and becomes current when the caller is done with the old one.
  auto row_key = [&](int i) { const uchar2 g2 = rowg[i]; return min((int)g2.x, 15) * 16 + min((int)g2.y - (int)g2.x, 15); };
  auto scan_rows = [&]() {
    int *bins = misc + 16;
    for (int b = tid; b < 256; b += bd) bins[b] = 0;
    __syncthreads();
    for (int i = tid - 32; i >= 0 && i < n_own; i += bd - 32) atomicAdd(&bins[row_key(i)], 1);
    if (warp == 0) {
      int carry = 0;
      for (int base = 0; base < n_own; base += 32) {
        const int i = base + wlane;
        const int v = i < n_own ? (int)rowg[i].y : 0;
        int inc = v;
        for (int o = 1; o < 32; o <<= 1) { const int nv = __shfl_up_sync(0xffffffffu, inc, o); if (wlane >= o) inc += nv; }
        if (i < n_own) rowofs[i] = (unsigned short)min(carry + inc - v, 65535);
        carry += __shfl_sync(0xffffffffu, inc, 31);
      }
      if (wlane == 0) { misc[0] = 0; misc[1] = carry; misc[2] = carry * R2_GS > Q.rows_cap ? 1 : 0; }
    }
    for (int w = tid; w < HW; w += bd) bm[w] = sbm[w];
    __syncthreads();
    if (warp == 0) {                                        // exclusive scan of the 256 bins, eight per lane
      int v[8], tot = 0;
#pragma unroll
      for (int u = 0; u < 8; ++u) { v[u] = bins[8 * wlane + u]; tot += v[u]; }
      int inc = tot;
      for (int o = 1; o < 32; o <<= 1) { const int nv = __shfl_up_sync(0xffffffffu, inc, o); if (wlane >= o) inc += nv; }
      int run = inc - tot;
#pragma unroll
      for (int u = 0; u < 8; ++u) { bins[8 * wlane + u] = run; run += v[u]; }
    }
    __syncthreads();
    for (int i = tid; i < n_own; i += bd) order[R.chunk + atomicAdd(&bins[row_key(i)], 1)] = (unsigned short)i;
    if (misc[2]) flag |= FLAG_SLOT_OVERFLOW;                // the rows of this chunk do not fit: error, nothing is written
    return misc[2] == 0;
  };
  // geometry of one row: natives per segment, survivors per segment -> groups
  struct RowGeo { int ofs, H_o, H_h, nno, nnh; uint32_t mul_o, mul_h; };
  auto row_geo = [&](int il, bool valid) {
    RowGeo g;
    const uchar2 nc = valid && !skip_nat ? natc[il] : make_uchar2(0, 0);
    const uchar2 gg = valid ? rowg[il] : make_uchar2(0, 0);
    g.nno = nc.x; g.nnh = nc.y;
    g.H_o = gg.x; g.H_h = gg.y - gg.x;
    g.ofs = valid ? (int)rowofs[il] * R2_GS : 0;
    g.mul_o = g.H_o ? (65536u + g.H_o - 1) / g.H_o : 0u;     // k / H = k * mul >> 16 for k < 1024, H < 256
    g.mul_h = g.H_h ? (65536u + g.H_h - 1) / g.H_h : 0u;
    return g;
  };
  // entry k of segment `hseg` of a row -> group k mod H, place k / H
  auto place = [&](const RowGeo &g, bool hseg, int k, uint32_t off, uint32_t par, float a) {
    const int H = hseg ? g.H_h : g.H_o;
    const int wq = (int)(((uint32_t)k * (hseg ? g.mul_h : g.mul_o)) >> 16), hq = k - wq * H;
    if (wq < R2_GS) {                                   // (always)
      const int at = g.ofs + (hseg ? g.H_o * R2_GS : 0) + hq * R2_GS + wq;
      rows[at] = make_uint2(off, par);
      if (EPS) rows_eps[at] = a;
    }
  };
  // the natives of a row into their places, and a dummy into every place that stays free
  auto place_static = [&](int il, const RowGeo &g, bool ok) {       // (called by whole warps: ok may differ between quarter-warps)
    // every place starts as a dummy (a point 1e18 A away, of the bank group of its position); the real entries follow
    const int n_pos = ok ? (g.H_o + g.H_h) * R2_GS : 0, own_pos = g.H_o * R2_GS;
    for (int p = l8; p < n_pos; p += 8) {
      rows[g.ofs + p] = make_uint2((uint32_t)(((p < own_pos ? Q.own_pad : Q.halo_pad) + ((p + (p >> 2)) & 7)) * 16), par_rep);
      if (EPS) rows_eps[g.ofs + p] = Q.a_ref;
    }
    __syncwarp();
    if (!ok) return;
    const int qn = natq[il] - qbase;
    for (int e = l8; e < g.nno; e += 8) place(g, false, e, snat[qn + e].x, snat[qn + e].y, EPS ? snat_eps[qn + e] : 0.f);
    for (int e = l8; e < g.nnh; e += 8) place(g, true, e, snat[qn + g.nno + e].x, snat[qn + g.nno + e].y, EPS ? snat_eps[qn + g.nno + e] : 0.f);
  };
  auto mark_active = [&](int idx) {
    const uint32_t bit = 1u << (idx & 31);
    if (!(((volatile uint32_t *)bm)[idx >> 5] & bit)) atomicOr(&bm[idx >> 5], bit);
  };
  // active halo set: bitmap -> list (a warp per word, a lane per bit; the order does not matter, only who polls what)
  auto active_list = [&]() {
    __syncthreads();
    for (int w = warp; w < HW; w += nwarps) {
      const uint32_t m = bm[w];
      if (m) {
        int at = 0;
        if (wlane == 0) at = atomicAdd(&misc[0], __popc(m));
        at = __shfl_sync(0xffffffffu, at, 0);
        if ((m >> wlane) & 1u) active[at + __popc(m & ((1u << wlane) - 1u))] = (unsigned short)((w << 5) + wlane);
      }
    }
    for (int i = tid; i < n_own; i += bd) order[i] = order[R.chunk + i];       // the new processing order becomes current
    __syncthreads();
  };

  // a3: Alg. 3 on the own rows + the force rows.  A quarter-warp per row.  Pass 1: the dealt L1 row comes
  // from global memory (L2) 8 entries at a time (the next four groups are in flight while four are tested), the candidates'
  // coordinates from shared memory; a lane keeps its survivors as two 64-bit masks.  Pass 2 (after the scan of the row
  // sizes): natives, then the survivors in lane order, dealt to the groups of the row.
  // member = true (a launch that does not start on a fresh L1): the L2 rows exist already, as global indices in the
  // canonical arrays; the same scan then keeps the candidates that ARE in the row instead of testing distances, so that
  // the force rows, and with them the summation order, do not depend on where a run was split.
  auto filter_rows = [&](const float4 *ownp, const float4 *halop, bool member) {
    const float R2 = S.R_nb2;
    unsigned long long mo[R2_MAXR], mh[R2_MAXR];
    // the rows are in the order of their force-row sizes, which follow the L1 row sizes: odd rounds walk their block of rows
    // backwards, so that a quarter-warp that got a short row in one round gets a long one in the next
    auto row_of = [&](int r) {
      const int first = r * nqw, last = min(n_own, first + nqw) - 1;
      const int ix = (r & 1) ? last - qw : first + qw;
      return ix >= first && ix <= last ? ix : -1;
    };
    const int bm_words = (Q.own_stride + Q.halo_stride + 31) >> 5;      // membership bitmap of one row (scratch in the row region)
    uint32_t *mbm = (uint32_t *)rows + (size_t)qw * bm_words;
    auto test_segment = [&](const unsigned short *row, int G, const float4 *P4, int pad, const float4 &ri, int bit0) {
      unsigned long long mask = 0ull;
      int e[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) e[u] = u < G ? (int)__ldg(row + 8 * u) : pad;
      for (int m = 0; m < G; m += 4) {
        int nx[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) nx[u] = m + 4 + u < G ? (int)__ldg(row + 8 * (m + 4 + u)) : pad;
        uint32_t nib = 0u;
        if (member) {
#pragma unroll
          for (int u = 0; u < 4; ++u) nib |= ((mbm[(bit0 + e[u]) >> 5] >> ((bit0 + e[u]) & 31)) & 1u) << u;
        } else {
#pragma unroll
          for (int u = 0; u < 4; ++u) nib |= (pred32(ri, P4[e[u]], R2) ? 1u : 0u) << u;
        }
        mask |= (unsigned long long)nib << m;
#pragma unroll
        for (int u = 0; u < 4; ++u) e[u] = nx[u];
      }
      return mask;
    };
#pragma unroll
    for (int r = 0; r < R2_MAXR; ++r) {
      mo[r] = 0ull; mh[r] = 0ull;
      if (r * nqw < n_own) {
        const int ix = row_of(r);
        const bool valid = ix >= 0;
        const int il = order[valid ? ix : n_own - 1];
        const size_t g = inst0 + b0 + il;
        const uchar2 gg = valid ? Q.pl_g[g] : make_uchar2(0, 0);
        const unsigned short *row = Q.pl_arr + g * Q.cap_arr + l8;
        const float4 ri = ownp[il];
        if (member) {
          __syncwarp();
          for (int w = l8; w < bm_words; w += 8) mbm[w] = 0u;
          __syncwarp();
          const int cnt = valid ? min(S.nb_cnt[g], cap_nb) : 0;
          for (int p = l8; p < cnt; p += 8) {
            const int j = S.nb_idx[g * cap_nb + p];
            const int bit = (j >= b0 && j < b1) ? j - b0 : Q.own_stride + lower_bound_dev(hgid, n_halo, j);
            atomicOr(&mbm[bit >> 5], 1u << (bit & 31));
          }
          __syncwarp();
        }
        mo[r] = test_segment(row, gg.x, ownp, Q.own_pad, ri, 0);
        mh[r] = test_segment(row + 8 * gg.x, gg.y, halop, Q.halo_pad, ri, Q.own_stride);
        int so = __popcll(mo[r]), sh = __popcll(mh[r]);
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) { so += __shfl_xor_sync(0xffffffffu, so, o); sh += __shfl_xor_sync(0xffffffffu, sh, o); }
        if (so + sh > cap_nb) flag |= FLAG_NB_OVERFLOW;
        if (valid && l8 == 0) {
          const uchar2 nc = skip_nat ? make_uchar2(0, 0) : natc[il];
          const int H_o = (nc.x + so + R2_GS - 1) / R2_GS, H_h = (nc.y + sh + R2_GS - 1) / R2_GS;
          if (H_o + H_h > 255) flag |= FLAG_SLOT_OVERFLOW;
          rowg[il] = make_uchar2((unsigned char)min(H_o, 255), (unsigned char)min(H_o + H_h, 255));
          cnt_s[il] = (unsigned short)min(so + sh, cap_nb);
        }
      }
    }
    const bool fits = scan_rows();
#pragma unroll
    for (int r = 0; r < R2_MAXR; ++r) {
      if (r * nqw < n_own && fits) {
        const int ix = row_of(r);
        const bool valid = ix >= 0;
        const int il = order[valid ? ix : n_own - 1];
        const size_t g = inst0 + b0 + il;
        const uchar2 gg = valid ? Q.pl_g[g] : make_uchar2(0, 0);
        const unsigned short *row = Q.pl_arr + g * Q.cap_arr + l8, *rowh = row + 8 * gg.x;
        const RowGeo geo = row_geo(il, valid);
        int io = __popcll(mo[r]), ih = __popcll(mh[r]);
        const int co = io, ch = ih;
        for (int o = 1; o < 8; o <<= 1) {
          const int vo = __shfl_up_sync(0xffffffffu, io, o, 8), vh = __shfl_up_sync(0xffffffffu, ih, o, 8);
          if (l8 >= o) { io += vo; ih += vh; }
        }
        const int so = __shfl_sync(0xffffffffu, io, 7, 8), sh = __shfl_sync(0xffffffffu, ih, 7, 8);
        const bool ok = valid && geo.H_o + geo.H_h < 255;
        place_static(il, geo, ok);
        if (ok) {
          int ko = geo.nno + io - co, kh = geo.nnh + ih - ch;
          unsigned long long m1 = mo[r], m2 = mh[r];
          while (m1) {
            const int m = __ffsll((long long)m1) - 1;
            m1 &= m1 - 1;
            place(geo, false, ko++, (uint32_t)__ldg(row + 8 * m) * 16u, par_rep, Q.a_ref);
          }
          while (m2) {
            const int m = __ffsll((long long)m2) - 1;
            m2 &= m2 - 1;
            const int idx = (int)__ldg(rowh + 8 * m);
            place(geo, true, kh++, (uint32_t)idx * 16u, par_rep, Q.a_ref);
            mark_active(idx);
          }
        }
      }
    }
    active_list();
  };

  filter_rows(own, halo, !filter_first);

  // ---- the steps ----------------------------------------------------------------------------------------------
  // `until` counts the steps to the next layer every chunk filters on (kept in step by both roles)
  int until = nb_interval - (int)(step0 % (unsigned long long)nb_interval);
  // Alg. 3 on the layer of step j (stamp j): whole halo from the filter layer, then the rows
  auto joint_filter = [&](int j, unsigned fp) {
    __syncthreads();
    const uint4 *xf = fp ? xf1 : xf0;
    float4 *hl = halo + (size_t)(j & 1) * Q.halo_stride;
    for (int q = tid; q < n_halo; q += bd) {
      float4 v;
      xch_wait(xf + 2 * (inst0 + hgid[q]), stamp0 + (uint32_t)j, v, S.flags);
      hl[q] = v;
    }
    __syncthreads();
    filter_rows(own + (size_t)(j & 1) * Q.own_stride, hl, false);
  };

  if (is_service) {
    // ======================= service warps: noise, halo and bond forces of the next step =======================
    const int stid = tid - NC;
    // what this lane polls: the first R2_MAXQ of its active halo slots stay in registers between filters
    int hq[R2_MAXQ], gq[R2_MAXQ];
    auto load_targets = [&]() {
      const int na = misc[0];
#pragma unroll
      for (int u = 0; u < R2_MAXQ; ++u) {
        const int q = stid + u * NS;
        hq[u] = q < na ? (int)active[q] : -1;
        gq[u] = q < na ? __ldg(hgid + hq[u]) : 0;
      }
    };
    load_targets();
    bar_arrive_named(BAR_HALO + 0, NC + NS);                     // step 0: halo and noise come from the prologue
    for (int j = 1; j < n_steps; ++j) {
#ifdef SOP_PHASE_CLOCKS
      pc_step = j;
#endif
      const unsigned long long step = step0 + (unsigned long long)j;
      const bool full = until == 1;                              // the halo of step j comes from the joint filter (j < n_steps)
      if (--until == 0) until = nb_interval;
      if (full) fpar ^= 1u;
      R2_TICK(7)
      float4 *gj = sg + (size_t)(j & 1) * R.chunk;               // last read by the update of step j - 2 (END_S(j - 2) is behind us)
      if (stid == 0) put_ext(j & 1, step);
      for (int i = stid; i < n_own; i += NS) {
        const uint32_t tag = stag[i];
        if (!(tag & TAG_FIXED)) gj[i] = draw(i, tag, step);
      }
      R2_TICK(1)                                                 // service: noise
      // The neighbours publish stamp j when they finish step j - 1, about when this CTA does: wait for that, then fetch.
      // Polling earlier only fills the load/store pipe that the compute warps' shared-memory gathers go through.
      bar_sync_named(BAR_END_S + ((j - 1) & 1), NC + NS);
      R2_TICK(0)                                                 // service: waiting for the compute warps
      if (!full) {
        const uint4 *xs = ((j & 1) ? xs1 : xs0) + 2 * inst0;
        const uint32_t st = stamp0 + (uint32_t)j;
        float4 *hl = halo + (size_t)(j & 1) * Q.halo_stride;
        __nanosleep(R2_FIRST_POLL_NS);                           // (a poll that comes too early costs a second round trip)
        unsigned pend = 0u;
#pragma unroll
        for (int u = 0; u < R2_MAXQ; ++u) pend |= hq[u] >= 0 ? 1u << u : 0u;
        unsigned spins = 0u;
        while (pend) {
          float4 v[R2_MAXQ];
          bool ok[R2_MAXQ];
#pragma unroll
          for (int u = 0; u < R2_MAXQ; ++u) ok[u] = ((pend >> u) & 1u) ? xch_try(xs + 2 * (size_t)gq[u], st, v[u]) : false;
#pragma unroll
          for (int u = 0; u < R2_MAXQ; ++u)
            if (ok[u]) { hl[hq[u]] = v[u]; pend &= ~(1u << u); }
          if (pend) __nanosleep(100);
          if (pend && (++spins & 1023u) == 0u) {
            volatile int *abort_word = S.flags + 1;
            if (*abort_word) break;
            if (spins >= XCH_SPIN_LIMIT) { atomicOr(S.flags, FLAG_EXCHANGE_TIMEOUT); *abort_word = 1; __threadfence(); break; }
          }
        }
        const int na = misc[0];
        for (int q = stid + R2_MAXQ * NS; q < na; q += NS) {     // (a very large active set: the rest one by one)
          const int h = active[q];
          float4 w;
          xch_wait(xs + 2 * (size_t)__ldg(hgid + h), st, w, S.flags);
          hl[h] = w;
        }
      }
      R2_TICK(2)                                                 // service: polling
      if (full) { joint_filter(j, fpar); load_targets(); }
      bar_arrive_named(BAR_HALO + (j & 1), NC + NS);
      R2_TICK(5)                                                 // service: release
    }
    bar_sync_named(BAR_END_S + ((n_steps - 1) & 1), NC + NS);
    if (until == 1 && filter_last) { fpar ^= 1u; joint_filter(n_steps, fpar); }
  } else {
    // ======================= compute warps: four lanes per bead ================================================
    const int l4 = tid & 3, grp = tid >> 2, NG = NC >> 2;
    int ilp[P];
    bool vp[P];
    const uint32_t s_own = smem_u32(own), s_halo = smem_u32(halo), s_rows = smem_u32(rows), s_g = smem_u32(sg);
    const uint32_t s_eps = smem_u32(rows_eps), s_ext = smem_u32(sext);
    const float A = Q.a_ref, amp_tr = amp_of(S, t);
    // one entry of a force row: s = A (1/r^2) (q max(q, 0) - q), q = (par/r^2)^3 (see the header); f_i += s (r_i - r_j)
    auto pair = [&](uint32_t entry, uint32_t base, const float4 &ri, float &fx, float &fy, float &fz) {
      const uint2 en = lds_u2(entry);
      const float4 rj = lds_f4(base + en.x);
      const float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
      const float inv = fast_rcp(dx * dx + dy * dy + dz * dz);
      const float u = __uint_as_float(en.y) * inv;
      const float q = u * u * u;
      const float tq = q * fmaxf(q, 0.0f) - q;
      const float a = EPS ? lds_f(s_eps + ((entry - s_rows) >> 1)) : A;
      const float s = a * inv * tq;
      fx += s * dx; fy += s * dy; fz += s * dz;
    };
    // a4: FENE bonds   V = -(k/2) R0^2 ln(1 - (r - r0)^2 / R0^2); lane b of the bead's group takes bond b, b + 4, ...;
    // bonds inside the chunk with the own partners, the few that cross into the halo with the halo partners
    uint2 bnd[P];                                                // this lane's bond of the bead of pass p (cap_b <= 4), {code, r0}
    bool hbond[P];
    auto bond_term = [&](const uint2 b, uint32_t base, const float4 &ri, float &fx, float &fy, float &fz) {
      const float4 rj = lds_f4(base + (b.x & 0x7FFFFFFFu));
      const float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
      const float r2 = dx * dx + dy * dy + dz * dz;
      const float inv_r = rsqrtf(r2);
      const float del = r2 * inv_r - __uint_as_float(b.y);
      const float x = 1.0f - del * del * S.inv_R0sq;
      if (!(x > 0.0f)) flag |= FLAG_FENE;
      const float sc = -S.k_fene * del * fast_rcp(x) * inv_r;
      fx += sc * dx; fy += sc * dy; fz += sc * dz;
    };
    auto bond = [&](int p, bool halo_part, uint32_t base, const float4 &ri, float &fx, float &fy, float &fz) {
      if (cap_b <= 4) {
        if (bnd[p].x != 0xFFFFFFFFu && ((bnd[p].x >> 31) != 0u) == halo_part) bond_term(bnd[p], base, ri, fx, fy, fz);
      } else if (vp[p]) {
        for (int bq = l4; bq < cap_b; bq += 4) {
          const int2 b = sbond[ilp[p] * cap_b + bq];
          if (b.x != -1 && (b.x < 0) == halo_part) bond_term(make_uint2((uint32_t)b.x, (uint32_t)b.y), base, ri, fx, fy, fz);
        }
      }
    };
    uint32_t rowa[P];                                            // address of the lane's entry in group 0 of the bead's row
    int ga[P], gb[P];                                            // own groups, all groups
    auto load_rows = [&]() {
#pragma unroll
      for (int p = 0; p < P; ++p) {
        const int idx = p * NG + grp;
        vp[p] = idx < n_own;
        ilp[p] = order[vp[p] ? idx : n_own - 1];
        bnd[p] = make_uint2(0xFFFFFFFFu, 0u);
        hbond[p] = false;
        if (vp[p]) {
          if (cap_b <= 4) {
            if (l4 < cap_b) { const int2 b = sbond[ilp[p] * cap_b + l4]; bnd[p] = make_uint2((uint32_t)b.x, (uint32_t)b.y); }
            hbond[p] = bnd[p].x != 0xFFFFFFFFu && (bnd[p].x >> 31) != 0u;
          } else {
            for (int bq = l4; bq < cap_b; bq += 4) { const int cb = sbond[ilp[p] * cap_b + bq].x; hbond[p] = hbond[p] || (cb != -1 && cb < 0); }
          }
        }
        const uchar2 gg = rowg[ilp[p]];
        rowa[p] = s_rows + (uint32_t)rowofs[ilp[p]] * (uint32_t)(R2_GS * 8) + (uint32_t)l4 * 8u;
        ga[p] = vp[p] ? (int)gg.x : 0; gb[p] = vp[p] ? (int)gg.y : 0;
      }
    };
    load_rows();
    for (int k = 0; k < n_steps; ++k) {
#ifdef SOP_PHASE_CLOCKS
      pc_step = k;
      R2_TICK(6)                                                 // compute: start of the step
#endif
      const uint32_t a_own = s_own + (uint32_t)(k & 1) * (uint32_t)Q.own_stride * 16u;
      const uint32_t a_halo = s_halo + (uint32_t)(k & 1) * (uint32_t)Q.halo_stride * 16u;
      const bool filt = until == 1 && (k + 1 < n_steps || filter_last);
      if (--until == 0) until = nb_interval;
      if (filt) fpar ^= 1u;
      float fx[P], fy[P], fz[P];
      float4 ri[P];
      // (A) own partners: nothing here depends on the neighbours' step
#pragma unroll
      for (int p = 0; p < P; ++p) {
        fx[p] = 0.f; fy[p] = 0.f; fz[p] = 0.f;
        ri[p] = lds_f4(a_own + (uint32_t)ilp[p] * 16u);
        for (int m = 0; m < ga[p]; ++m) pair(rowa[p] + (uint32_t)(R2_GS * 8) * m, a_own, ri[p], fx[p], fy[p], fz[p]);
        bond(p, false, a_own, ri[p], fx[p], fy[p], fz[p]);
      }
      R2_TICK(0)                                                 // compute: own partners
      bar_sync_named(BAR_HALO + (k & 1), NC + NS);               // halo, noise and bond forces of step k are in shared memory
      R2_TICK(1)                                                 // compute: waiting for the halo
      // (B) halo partners, reduction over the four lanes
#pragma unroll
      for (int p = 0; p < P; ++p) {
        for (int m = ga[p]; m < gb[p]; ++m) pair(rowa[p] + (uint32_t)(R2_GS * 8) * m, a_halo, ri[p], fx[p], fy[p], fz[p]);
        if (__any_sync(0xffffffffu, hbond[p])) bond(p, true, a_halo, ri[p], fx[p], fy[p], fz[p]);
#pragma unroll
        for (int o = 2; o > 0; o >>= 1) {
          fx[p] += __shfl_xor_sync(0xffffffffu, fx[p], o);
          fy[p] += __shfl_xor_sync(0xffffffffu, fy[p], o);
          fz[p] += __shfl_xor_sync(0xffffffffu, fz[p], o);
        }
      }
      R2_TICK(2)                                                 // compute: halo partners, reduction
      // a7 + a9: lane p of the group moves the bead of pass p and publishes it
      if (R.skew_ns && tc == R.skew_chunk && (step0 + (unsigned long long)k) % (unsigned long long)R.skew_period == 0) __nanosleep((unsigned)R.skew_ns);
      {
        float ux = fx[0], uy = fy[0], uz = fz[0];
        float4 r0 = ri[0];
        int il = ilp[0];
        bool v = vp[0];
#pragma unroll
        for (int p = 1; p < P; ++p)
          if (l4 == p) { ux = fx[p]; uy = fy[p]; uz = fz[p]; r0 = ri[p]; il = ilp[p]; v = vp[p]; }
        if (l4 < P && v) {
          const uint32_t tag = __float_as_uint(r0.w);
          float4 out = r0;
          if (!(tag & TAG_FIXED)) {
            const float4 e4 = lds_f4(s_ext + (uint32_t)(k & 1) * 16u);
            ExtStep ext; ext.vs_pull = e4.x; ext.cx = e4.y; ext.cy = e4.z; ext.cz = e4.w;
            external_force_at(S, b0 + il, r0, tag, ext, ux, uy, uz, flag);
            const float4 g4 = lds_f4(s_g + (uint32_t)((k & 1) * R.chunk + il) * 16u);
            out = langevin_apply<COMP>(S, r0, make_float3(g4.x, g4.y, g4.z), ux, uy, uz, COMP ? scarry + il : nullptr, flag, amp_tr);
          }
          sts_f4(s_own + (uint32_t)(((k & 1) ^ 1) * Q.own_stride + il) * 16u, out);
          uint4 *xp = filt ? (fpar ? xf1 : xf0) : (((k + 1) & 1) ? xs1 : xs0);
          xch_put(xp + 2 * (inst0 + b0 + il), out, stamp0 + (uint32_t)(k + 1));
        }
      }
      R2_TICK(3)                                                 // compute: update + publish
      bar_arrive_named(BAR_END_S + (k & 1), NC + NS);            // the service warps may reuse the layers of step k
      bar_sync_named(BAR_END_C, NC);                             // the own coordinates of step k + 1 are complete
      R2_TICK(4)                                                 // compute: waiting for the slowest compute warp
      if (filt) { joint_filter(k + 1, fpar); load_rows(); }
      R2_TICK(7)                                                 // compute: force rows + active set (after a filter)
    }
  }

#ifdef SOP_PHASE_CLOCKS
  if (wlane == 0) {
    S.force[((size_t)blockIdx.x * 32 + warp) * 2] = make_float4((float)pc_acc[0], (float)pc_acc[1], (float)pc_acc[2], (float)pc_acc[3]);
    S.force[((size_t)blockIdx.x * 32 + warp) * 2 + 1] = make_float4((float)pc_acc[4], (float)pc_acc[5], (float)pc_acc[6], (float)pc_acc[7]);
  }
#endif
  // ---- epilogue: the current layer, the carry, the generator states and the L2 rows back to the canonical arrays
  __syncthreads();
  const float4 *pf = own + (size_t)(n_steps & 1) * Q.own_stride;
  for (int i = tid; i < n_own; i += bd) {
    S.pos[cur][inst0 + b0 + i] = pf[i];
    if (COMP) S.carry[inst0 + b0 + i] = scarry[i];
    if (S.taus) S.taus[inst0 + b0 + i] = staus[i];
  }
  // the L2 partners of a row are its entries with par = par_rep that are not dummies
  for (int il = warp; il < n_own; il += nwarps) {
    const size_t g = inst0 + b0 + il;
    const uchar2 gg = rowg[il];
    const int first = (int)rowofs[il] * R2_GS, n_pos = gg.y * R2_GS, own_pos = gg.x * R2_GS;
    int *canon = S.nb_idx + g * cap_nb;
    int n = 0;
    for (int base = 0; base < n_pos; base += 32) {
      const int p = base + wlane;
      bool keep = false;
      int j = 0;
      if (p < n_pos) {
        const uint2 en = rows[first + p];
        const int idx = (int)(en.x >> 4);
        const bool hseg = p >= own_pos;
        keep = en.y == par_rep && idx < (hseg ? n_halo : n_own);
        if (keep) j = hseg ? hgid[idx] : b0 + idx;
      }
      const unsigned m = __ballot_sync(0xffffffffu, keep);
      if (keep) { const int at = n + __popc(m & lt); if (at < cap_nb) canon[at] = j; }
      n += __popc(m);
    }
    if (wlane == 0) S.nb_cnt[g] = min(n, cap_nb);
  }
  if (flag) atomicOr(S.flags, flag);
}

}  // namespace sop

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
// Readers and writers are kept apart by two pairs of layers.
//  * step layers (parity of the step): read by ACTIVE readers only.  Being active is symmetric between chunks (bonds,
//    natives and L2 rows are symmetric relations and both sides filter the same coordinates), so A overwrites stamp s
//    with s+2 only after it has read B's stamp s+1, which B published after it finished reading A's stamp s.
//  * filter layers (parity of step / nb_interval): the coordinates of the steps on which L2 is re-filtered (and of the
//    launch prologue) are published here and nowhere else, and every chunk reads its WHOLE halo from them.  The L1
//    relation is symmetric, so the same argument holds between any two chunks that are in each other's halo: A writes the
//    filter layer of step s+2 nb only after reading C's layer of step s+nb, published after C finished reading step s.
//    A halo-only (non-active) reader therefore never meets an overwritten slot, which a single pair of layers could not
//    guarantee (a chunk only waits for its ACTIVE neighbours between filters).
// Every wait is bounded (xch_wait): a protocol fault raises FLAG_EXCHANGE_TIMEOUT instead of hanging the launch.
#pragma once
#include <type_traits>

#include "sop_kernels.cuh"

namespace sop {

constexpr int FLAG_SLOT_OVERFLOW = 16;
constexpr int RES_GRID_CELLS = 1024;      // cells of the in-kernel grid of a one-chunk trajectory (implicit L1)

struct ResDev {
  int C;                      // chunks per trajectory
  int chunk;                  // beads per chunk (the last chunk of a trajectory may be shorter)
  int halo_cap;               // halo slots per chunk
  int implicit_l1;            // static all-pairs L1 and C == 1: the L1 row of i is "every j != i not excluded"
  int nat_entries;            // native table entries per trajectory
  int *n_halo;                // [T*C]
  int *halo_gid;              // [T*C][halo_cap] bead index (within the trajectory) of each halo slot, ascending
  unsigned short *pl_loc;     // [T*N][cap_pl]   L1 rows as slots
  int2 *nat_pack;             // [T][nat_entries] {slot, bits(r0^2)}   (C > 1; with one chunk slot = bead index)
  int2 *bond_pack;            // [T*N][cap_b]     {slot or -1, bits(r0)} (C > 1)
  int2 *nat_T;                // one chunk, natives not in shared memory: the native table transposed, entry k of bead i
  int nat_tpad;               // at [k * nat_tpad + i], so that a warp of consecutive beads reads 256 contiguous bytes
  uint4 *xch;                 // [2][T*N][2]  step layers: one 32-byte slot {x|stamp, y|stamp, z|stamp, -} per bead and step parity
  uint4 *xchf;                // [2][T*N][2]  filter layers: the coordinates of the steps on which L2 is re-filtered (read by the
                              //              WHOLE halo), alternating with the parity of step / nb_interval
  // one chunk per trajectory and more trajectories than SMs: a launch is cut into time slices of slice_len steps, one CTA per
  // (slice, trajectory), handed out slice-major by a ticket counter; a CTA waits until its trajectory's previous slice has
  // signalled `done`, so that the grid fills every SM all the time instead of running T CTAs in ceil(T / SMs) waves
  int slice_len;              // 0: one CTA per chunk for the whole launch
  int *ticket, *done;         // [1], [T]  (zeroed by the host before a sliced launch)
  int skew_chunk, skew_period, skew_ns;   // test hook: chunk skew_chunk sleeps skew_ns before publishing on steps % skew_period == 0
  // shared-memory carve-up (bytes from the start of dynamic shared memory), computed by the host
  int off_pos, off_g, off_carry, off_tag, off_force, off_nb, off_cnt, off_plcnt, off_plofs, off_pl, off_natq,
      off_nat, off_bond, off_active, off_bm, off_sbm, off_misc, off_order, off_hist;
  int nb_si;                  // L2 row i starts at nb[i * nb_si]; nb_si = cap_nb + 4 is a multiple of four 16-bit slots, so that every
                              // row is 8-byte aligned (rows are read four slots per 8-byte word and padded with the dummy slot)
  int nat_smem;               // the chunk's native table is copied to shared memory (its nat_cap entries fit)
  int nat_cap;                // largest number of native entries of a chunk
  int pl_cap;                 // 16-bit entries of shared memory for the chunk's L1 rows (0: read them from global)
  int smem_bytes;
  int stream;                 // the chunk state does not fit shared memory: only the coordinates (ONE time layer), tags, forces and
                              // counters are resident; L2 rows, bonds, natives and L1 rows are streamed from global memory (L2)
  unsigned short *nb_glob;    // [T*N][nb_si] L2 rows as slots (stream)
};

__device__ __forceinline__ float fast_rcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// One 32-byte exchange slot per bead: three 64-bit elements {value, stamp} for x, y, z and one of padding, written and read
// with ONE 256-bit access (sm_100: LDG/STG.256) at gpu scope -- one L2 sector request per bead per poll.  The PTX memory
// model treats a vector access as one access per ELEMENT, so the elements are the 64-bit {value, stamp} pairs the
// protocol needs to be single-copy atomic (.v4.b64), and all three stamps are checked.
__device__ __forceinline__ void xch_put(uint4 *slot, const float4 &v, uint32_t st) {
  const unsigned long long hi = (unsigned long long)st << 32;
  asm volatile("st.relaxed.gpu.global.v4.b64 [%0], {%1, %2, %3, %4};" ::"l"(slot), "l"(hi | __float_as_uint(v.x)),
               "l"(hi | __float_as_uint(v.y)), "l"(hi | __float_as_uint(v.z)), "l"(0ull) : "memory");
}

__device__ __forceinline__ bool xch_try(const uint4 *slot, uint32_t st, float4 &out) {
  unsigned long long a, b, c, d;
  asm volatile("ld.relaxed.gpu.global.v4.b64 {%0, %1, %2, %3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(slot) : "memory");
  out = make_float4(__uint_as_float((uint32_t)a), __uint_as_float((uint32_t)b), __uint_as_float((uint32_t)c), 0.f);
  return (uint32_t)(a >> 32) == st && (uint32_t)(b >> 32) == st && (uint32_t)(c >> 32) == st;
}

// Bounded wait for one slot.  A CTA that waits longer than XCH_SPIN_LIMIT polls (seconds: a protocol fault, a dead
// neighbour) raises FLAG_EXCHANGE_TIMEOUT and the abort word; every spinning thread looks at the abort word from time
// to time and gives up too, so the cooperative launch ends with an error status instead of hanging the GPU.
constexpr int FLAG_EXCHANGE_TIMEOUT = 32;
constexpr unsigned XCH_SPIN_LIMIT = 1u << 23;
__device__ __forceinline__ bool xch_slow_wait(const uint4 *slot, uint32_t st, float4 &out, int *flags) {
  volatile int *abort_word = flags + 1;
  for (unsigned spins = 0;; ++spins) {
    if (xch_try(slot, st, out)) return true;
    if ((spins & 1023u) == 1023u) {
      if (*abort_word) return false;
      if (spins >= XCH_SPIN_LIMIT) { atomicOr(flags, FLAG_EXCHANGE_TIMEOUT); *abort_word = 1; __threadfence(); return false; }
    }
  }
}
__device__ __forceinline__ bool xch_wait(const uint4 *slot, uint32_t st, float4 &out, int *flags) {
  if (xch_try(slot, st, out)) return true;
  return xch_slow_wait(slot, st, out, flags);
}

// ------------------------------------------------------------------------------------------------
// k_localise: after an L1 build, give every chunk its halo slot table and re-express L1 rows, natives and bonds
// in chunk-local slots.  One CTA per (trajectory, chunk); dynamic shared memory: bitmap + prefix over the N beads.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) k_localise(SysDev S, ResDev R) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int W = (S.N + 31) >> 5;
  uint32_t *bm = (uint32_t *)smem_raw;         // [W] bead j is in the halo
  uint32_t *pre = bm + W;                      // [W] exclusive prefix of popc(bm)
  int *cnt = (int *)(pre + W);                 // [chunk] L1 row counts of the own beads
  __shared__ int warp_tot[32];
  __shared__ int carry_s;
  const int tc = blockIdx.x, t = tc / R.C, c = tc - t * R.C;
  const int b0 = c * R.chunk, b1 = min(S.N, b0 + R.chunk), n_own = b1 - b0;
  const int tid = threadIdx.x, bd = blockDim.x;
  const int lane = tid & 31, warp = tid >> 5, nwarps = bd >> 5;
  const size_t g0 = (size_t)t * S.N + b0;
  const int cap_pl = S.cap_pl, cap_b = S.cap_b;
  for (int w = tid; w < W; w += bd) bm[w] = 0u;
  for (int i = tid; i < n_own; i += bd) cnt[i] = min(S.pl_cnt[g0 + i], cap_pl);
  if (tid == 0) carry_s = 0;
  __syncthreads();
  // every loop below is flat over table entries: independent, coalesced loads, nothing waits on a row at a time
  // test before the atomic: neighbours share most of their halo, so nearly every bit is already set
  auto mark = [&](int j) {
    if (j < b0 || j >= b1) { const uint32_t bit = 1u << (j & 31); if (!(((volatile uint32_t *)bm)[j >> 5] & bit)) atomicOr(&bm[j >> 5], bit); }
  };
  const int *rows = S.pl_idx + g0 * cap_pl;
  // a warp per row, four independent loads per lane in flight (no index arithmetic per entry, no padding visited)
  for (int r = warp; r < n_own; r += nwarps) {
    const int c_r = cnt[r];
    const int *row = rows + (size_t)r * cap_pl;
    for (int p0 = lane; p0 < c_r; p0 += 128) {
      int v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) v[u] = p0 + 32 * u < c_r ? row[p0 + 32 * u] : -1;
#pragma unroll
      for (int u = 0; u < 4; ++u) if (v[u] >= 0) mark(v[u]);
    }
  }
  const int q0 = S.nat_ptr[b0], q1 = S.nat_ptr[b1];
  const bool multi = R.C > 1;
  if (multi) {
    for (int q = q0 + tid; q < q1; q += bd) mark(S.nat_tab[q].x);
    for (int e = tid; e < n_own * cap_b; e += bd) { const int j = S.bond_tab[(size_t)b0 * cap_b + e].x; if (j >= 0) mark(j); }
  }
  __syncthreads();
  // exclusive scan of the word popcounts
  for (int base = 0; base < W; base += bd) {
    const int w = base + tid;
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
    if (tid == bd - 1) carry_s = excl + v;
    __syncthreads();
  }
  const int n_halo = carry_s;
  if (n_halo > R.halo_cap) {
    if (tid == 0) { atomicOr(S.flags, FLAG_SLOT_OVERFLOW); R.n_halo[tc] = 0; }
    return;
  }
  if (tid == 0) R.n_halo[tc] = n_halo;
  int *hg = R.halo_gid + (size_t)tc * R.halo_cap;
  for (int w = tid; w < W; w += bd) {
    uint32_t bits = bm[w];
    int k = (int)pre[w];
    while (bits) { int b = __ffs(bits) - 1; bits &= bits - 1; hg[k++] = (w << 5) + b; }
  }
  auto slot_of = [&](int j) -> int {
    if (j >= b0 && j < b1) return j - b0;
    return n_own + (int)pre[j >> 5] + __popc(bm[j >> 5] & ((1u << (j & 31)) - 1u));
  };
  unsigned short *loc = R.pl_loc + g0 * cap_pl;
  for (int r = warp; r < n_own; r += nwarps) {
    const int c_r = cnt[r];
    const int *row = rows + (size_t)r * cap_pl;
    unsigned short *lrow = loc + (size_t)r * cap_pl;
    for (int p0 = lane; p0 < c_r; p0 += 128) {
      int v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) v[u] = p0 + 32 * u < c_r ? row[p0 + 32 * u] : -1;
#pragma unroll
      for (int u = 0; u < 4; ++u) if (v[u] >= 0) lrow[p0 + 32 * u] = (unsigned short)slot_of(v[u]);
    }
  }
  if (multi) {                                  // one chunk: slot = bead index, natives and bonds need no table
    for (int q = q0 + tid; q < q1; q += bd) {
      const int2 en = S.nat_tab[q];
      R.nat_pack[(size_t)t * R.nat_entries + q] = make_int2(slot_of(en.x), en.y);
    }
    for (int e = tid; e < n_own * cap_b; e += bd) {
      const int2 en = S.bond_tab[(size_t)b0 * cap_b + e];
      R.bond_pack[g0 * cap_b + e] = make_int2(en.x >= 0 ? slot_of(en.x) : -1, en.y);
    }
  }
}

// native table -> transposed copy (one chunk per trajectory: slot = bead index), once at create
__global__ void k_transpose_nat(SysDev S, ResDev R) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= S.N) return;
  const int q0 = S.nat_ptr[i], q1 = S.nat_ptr[i + 1];
  for (int q = q0; q < q1; ++q) R.nat_T[(size_t)(q - q0) * R.nat_tpad + i] = S.nat_tab[q];
}

// ------------------------------------------------------------------------------------------------
// Pair force laws of Eq. (1) with MUFU reciprocals (1 ulp; the parity bar is 1e-4 max|F|).
// Each returns s with f_i += s (r_i - r_j).
// ------------------------------------------------------------------------------------------------
struct ForceK {                // loop invariants kept in registers
  float k_fene, inv_R0sq, eps12, c_rep_f;
};

__device__ __forceinline__ float rep_s3(float r2, float c_rep_f) {        // 6 eps_r sigma^6 / r^8
  const float inv_r2 = fast_rcp(r2);
  const float i4 = inv_r2 * inv_r2;
  return c_rep_f * i4 * i4;
}
__device__ __forceinline__ float nat_s3(float r2, float r0sq, float e12) {  // (12 eps / r^2) (q^2 - q), q = (r0/r)^6
  const float inv_r2 = fast_rcp(r2);
  const float u = r0sq * inv_r2;
  const float q3 = u * u * u;
  return e12 * inv_r2 * (q3 * q3 - q3);
}

__device__ __forceinline__ int lower_bound_dev(const int *__restrict__ a, int n, int v) {
  int lo = 0, hi = n;
  while (lo < hi) { int mid = (lo + hi) >> 1; if (__ldg(&a[mid]) < v) lo = mid + 1; else hi = mid; }
  return lo;
}

// ------------------------------------------------------------------------------------------------
// k_resident: a3 + a4..a9 for n_steps Langevin steps of one chunk per CTA (see the header of this file).
// Per step:
//   (b) fetch the active halo of this step's layer (poll the stamps)                    -- __syncthreads --
//   (d1) a4..a6 internal force, G lanes per bead: bonds, natives and the L2 row (two slots per 32-bit word) are
//        gathered from shared memory only, lane partial sums meet by shuffle, lane 0 stores the force -- __syncthreads --
//   (d2) a7 + a9 thread per bead: external force, update, publish; meanwhile the threads at the other end of the block
//        generate the noise (a8) of the NEXT step, off the critical path
//   (e) every nb_interval steps: fetch the whole halo of the new layer, Alg. 3 on the own rows (L1 rows resident in
//        shared memory when they fit), new active set.
// Coordinates and noise are double-buffered on the step parity.
// STREAM (systems whose chunks do not fit shared memory, e.g. 250,000 beads on 148 SMs): one coordinate layer -- every read of
// a step's coordinates lies before the block barrier that precedes the update, and a thread updates only its own bead, so the
// update can be done in place --, and the lists live in global memory (L2-resident): rows are read coalesced, the partner
// gathers stay in shared memory.
// ------------------------------------------------------------------------------------------------
// SPEC: the switches the step loop would otherwise test at run time, every step, are constants of the two common cases (the
// host picks the instantiation; 0 = general).  1: several chunks, explicit L1, natives in shared memory.  2: one chunk per
// trajectory with the static all-pairs L1, natives transposed in global memory (one lane per bead) or in shared memory
// (several lanes).  Both: one native eps, Philox noise, no skew hook.  Less straight-line code per step, which a kernel whose
// every step walks through once-only code pays for in instruction fetch.
template <int G, bool COMP, bool STREAM = false, int MAXT = 1024, int SPEC = 0>
__global__ void __launch_bounds__(MAXT, 1) k_resident(SysDev S, ResDev R, int cur, unsigned long long step0, int n_steps,
                                                      int nb_interval, int filter_flags, uint32_t stamp0) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int SC = R.chunk + R.halo_cap + 1;                           // + the dummy slot (last)
  float4 *spos = (float4 *)(smem_raw + R.off_pos);                   // [2][SC]
  float4 *sg = (float4 *)(smem_raw + R.off_g);                       // [2][chunk]
  float4 *scarry = (float4 *)(smem_raw + R.off_carry);               // [chunk]      (COMP)
  uint32_t *stag = (uint32_t *)(smem_raw + R.off_tag);               // [chunk]
  float4 *sforce = (float4 *)(smem_raw + R.off_force);                // [chunk] internal force of this step
  // (tc is blockIdx.x; the L2 rows of a streamed chunk start at its first bead instance)
  unsigned short *nb = STREAM ? R.nb_glob + ((size_t)(blockIdx.x / R.C) * S.N + (size_t)(blockIdx.x % R.C) * R.chunk) * R.nb_si
                              : (unsigned short *)(smem_raw + R.off_nb);      // L2 rows as slots, row stride nb_si
  unsigned short *cnt_s = (unsigned short *)(smem_raw + R.off_cnt);  // [chunk] L2 row counts
  unsigned short *plcnt_s = (unsigned short *)(smem_raw + R.off_plcnt);  // [chunk] L1 row counts
  int *plofs = (int *)(smem_raw + R.off_plofs);                      // [chunk + 1] L1 row starts in spl (even)
  unsigned short *spl = (unsigned short *)(smem_raw + R.off_pl);     // [pl_cap] L1 rows as slots, packed
  int *natq = (int *)(smem_raw + R.off_natq);                        // [chunk + 1] native table offsets
  int2 *snat = (int2 *)(smem_raw + R.off_nat);                       // [nat_cap]    (nat_smem)
  int2 *sbond = STREAM ? R.bond_pack + ((size_t)(blockIdx.x / R.C) * S.N + (size_t)(blockIdx.x % R.C) * R.chunk) * S.cap_b
                       : (int2 *)(smem_raw + R.off_bond);            // [chunk][cap_b]
  unsigned short *active = (unsigned short *)(smem_raw + R.off_active);
  uint32_t *bm = (uint32_t *)(smem_raw + R.off_bm), *sbm = (uint32_t *)(smem_raw + R.off_sbm);
  unsigned short *order = (unsigned short *)(smem_raw + R.off_order);     // own beads by descending native degree
  int *hist = (int *)(smem_raw + R.off_hist);                              // [64] scratch of that counting sort
  int *misc = (int *)(smem_raw + R.off_misc);                        // [0] active halo slots, [2..7] bounding box of the in-kernel grid

  int tc = blockIdx.x, slice = 0;
  if (!STREAM && R.slice_len > 0) {
    // sliced launch (C == 1): ticket -> (slice, trajectory); tickets are handed out in order, so the CTA that owns this
    // trajectory's previous slice took its ticket earlier and is running or done -- the wait below cannot deadlock
    __shared__ int s_ticket;
    if (threadIdx.x == 0) s_ticket = atomicAdd(R.ticket, 1);
    __syncthreads();
    const int n_tc = S.T * R.C, n_total = n_steps;
    slice = s_ticket / n_tc; tc = s_ticket - slice * n_tc;
    if (s_ticket < 0 || (long long)slice * R.slice_len >= n_total) return;      // (a ticket outside the grid's range: nothing to do)
    step0 += (unsigned long long)slice * (unsigned long long)R.slice_len;
    n_steps = min(R.slice_len, n_total - slice * R.slice_len);
    const bool last = (slice + 1) * R.slice_len >= n_total;
    // (slice_len is a multiple of nb_interval: the filter due at the end of an inner slice runs inside it)
    filter_flags = (last ? (filter_flags & 1) : 1) | (slice == 0 ? (filter_flags & 2) : 0);
    if (slice > 0) {
      // bounded like every other wait of this kernel (seconds: a lost ticket order would be a protocol fault): the flag is
      // raised, this slice and -- through the abort word -- every later one is skipped, the launch ends with SOP_E_CUDA
      __shared__ int s_ok;
      if (threadIdx.x == 0) {
        volatile int *abort_word = S.flags + 1;
        int seen, ok = 1;
        for (unsigned spins = 0;; ++spins) {
          asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(R.done + tc) : "memory");
          if (seen >= slice) break;
          if (*abort_word) { ok = 0; break; }
          if (spins >= XCH_SPIN_LIMIT) { atomicOr(S.flags, FLAG_EXCHANGE_TIMEOUT); *abort_word = 1; __threadfence(); ok = 0; break; }
          __nanosleep(200);
        }
        s_ok = ok;
      }
      __syncthreads();
      if (!s_ok) {
        if (threadIdx.x == 0) asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(R.done + tc), "r"(slice + 1) : "memory");
        return;
      }
      __threadfence();                         // every thread reads what the previous slice wrote (no stale L1 lines)
    }
  }
  const bool filter_last = filter_flags & 1, filter_first = filter_flags & 2;
  const int t = tc / R.C, c = tc - t * R.C;
  const int b0 = c * R.chunk, b1 = min(S.N, b0 + R.chunk), n_own = b1 - b0;
  constexpr bool FAST = SPEC != 0;
  const bool multi = SPEC == 1 || (SPEC == 0 && R.C > 1);
  const int n_halo = multi ? R.n_halo[tc] : 0;
  const int *__restrict__ hgid = R.halo_gid + (size_t)tc * R.halo_cap;
  const int HW = (n_halo + 31) >> 5;
  const int tid = threadIdx.x, bd = blockDim.x;
  const int wlane = tid & 31, warp = tid >> 5, nwarps = bd >> 5;
  const int lane = tid % G, grp = tid / G, groups = bd / G;
  const unsigned short DUMMY = (unsigned short)(SC - 1);
  const size_t inst0 = (size_t)t * S.N;
  uint4 *const xl0 = R.xch, *const xl1 = R.xch + 2 * (size_t)S.n_inst;
  uint4 *const xf0 = R.xchf, *const xf1 = R.xchf + 2 * (size_t)S.n_inst;
  unsigned fpar = (unsigned)((step0 / (unsigned long long)nb_interval) & 1ull);      // filter layer of the prologue
  const int cap_b = S.cap_b, cap_nb = S.cap_nb;
  const uint32_t traj = (uint32_t)(S.traj_offset + t);
  const float amp_tr = amp_of(S, t);
  int flag = 0;

  // exclusive scan of n_own 16-bit counts by warp 0 (the caller synchronises)
  auto scan_counts = [&](const unsigned short *cnt, int *ofs, bool round_even) {
    if (warp == 0) {
      int carry = 0;
      for (int base = 0; base < n_own; base += 32) {
        const int i = base + wlane;
        int v = i < n_own ? (int)cnt[i] : 0;
        if (round_even) v = (v + 1) & ~1;
        int inc = v;
        for (int o = 1; o < 32; o <<= 1) { const int n = __shfl_up_sync(0xffffffffu, inc, o); if (wlane >= o) inc += n; }
        if (i < n_own) ofs[i] = carry + inc - v;
        carry += __shfl_sync(0xffffffffu, inc, 31);
      }
      if (wlane == 0) ofs[n_own] = carry;
    }
  };

  // ---- prologue: own coordinates, carry, tags, static tables; canonical L2 rows -> slots; L1 rows -> shared memory
  const int qbase = S.nat_ptr[b0];
  if (tid == 0) {      // a point 1e18 A away: its repulsion underflows to exactly zero (pads odd L2 rows)
    spos[SC - 1] = make_float4(1.0e18f, 1.0e18f, 1.0e18f, 0.f);
    if (!STREAM) spos[2 * SC - 1] = make_float4(1.0e18f, 1.0e18f, 1.0e18f, 0.f);
  }
  for (int i = tid; i < n_own; i += bd) {
    const float4 v = S.pos[cur][inst0 + b0 + i];
    spos[i] = v;
    stag[i] = __float_as_uint(v.w);
    if (multi) xch_put((fpar ? xf1 : xf0) + 2 * (inst0 + b0 + i), v, stamp0);
    if (COMP) scarry[i] = S.carry[inst0 + b0 + i];
    natq[i] = S.nat_ptr[b0 + i];
    plcnt_s[i] = R.implicit_l1 ? (unsigned short)0 : (unsigned short)S.pl_cnt[inst0 + b0 + i];
    const uint32_t tag = __float_as_uint(v.w);
    if (G > 1 && !(tag & TAG_FIXED)) {
      const float3 gn = !FAST && S.taus ? gaussian3_taus(S.taus + inst0 + b0 + i) : gaussian3(S, tag & TAG_ID_MASK, traj, step0);
      sg[i] = make_float4(gn.x, gn.y, gn.z, 0.f);
    }
  }
  if (tid == 0) natq[n_own] = S.nat_ptr[b1];
  const int2 *bond_src = multi ? R.bond_pack + (inst0 + b0) * cap_b : S.bond_tab + (size_t)b0 * cap_b;
  if (!STREAM) for (int e = tid; e < n_own * cap_b; e += bd) sbond[e] = bond_src[e];
  const int2 *nat_glob = multi ? R.nat_pack + (size_t)t * R.nat_entries : S.nat_tab;
  const int n_nat = S.nat_ptr[b1] - qbase;
  if (R.nat_smem)
    for (int e = tid; e < n_nat; e += bd) snat[e] = nat_glob[qbase + e];
  const int2 *natp = R.nat_smem ? (const int2 *)snat - qbase : nat_glob;      // indexed by the global offset q
  // the whole halo of the first layer comes through the exchange (never from S.pos, which a chunk that has finished a short
  // launch overwrites in its epilogue while a late chunk is still in its prologue)
  for (int q = tid; q < n_halo; q += bd) {
    float4 v;
    xch_wait((fpar ? xf1 : xf0) + 2 * (inst0 + hgid[q]), stamp0, v, S.flags);
    spos[n_own + q] = v;
  }
  if (!filter_first) {
    for (int il = warp; il < n_own; il += nwarps) {
      const size_t g = inst0 + b0 + il;
      const int cnt = min(S.nb_cnt[g], cap_nb);
      const int *row = S.nb_idx + g * cap_nb;
      unsigned short *dst = nb + (size_t)il * R.nb_si;
      for (int p = wlane; p < cnt; p += 32) {
        const int j = row[p];
        dst[p] = (unsigned short)((j >= b0 && j < b1) ? j - b0 : n_own + lower_bound_dev(hgid, n_halo, j));
      }
      if (wlane == 0) { cnt_s[il] = (unsigned short)cnt; for (int k4 = cnt; k4 & 3; ++k4) dst[k4] = DUMMY; }
    }
  }
  for (int w = tid; w < HW; w += bd) sbm[w] = 0u;
  for (int b = tid; b < 64; b += bd) hist[b] = 0;
  __syncthreads();
  // processing order of the pair phase: own beads by descending native degree (counting sort), so that the groups of a
  // warp run the same number of native iterations and fewer warp-level gathers carry idle lanes.  Which group handles
  // a bead does not change its force (lane = position in the list mod G), so ties may fall either way.
  for (int i = tid; i < n_own; i += bd) atomicAdd(&hist[63 - min(63, natq[i + 1] - natq[i])], 1);
  __syncthreads();
  if (tid == 0) { int run = 0; for (int b = 0; b < 64; ++b) { const int c2 = hist[b]; hist[b] = run; run += c2; } }
  __syncthreads();
  if (!STREAM) {
    for (int i = tid; i < n_own; i += bd)           // one lane per bead: keep thread i on bead i (coalesced table reads)
      order[G > 1 ? atomicAdd(&hist[63 - min(63, natq[i + 1] - natq[i])], 1) : i] = (unsigned short)i;
    scan_counts(plcnt_s, plofs, true);
  }
  __syncthreads();
  const bool pl_in_smem = !STREAM && !R.implicit_l1 && R.pl_cap > 0 && plofs[n_own] <= R.pl_cap;
  if (pl_in_smem) {
    for (int il = warp; il < n_own; il += nwarps) {
      const uint32_t *src = (const uint32_t *)(R.pl_loc + (inst0 + b0 + il) * S.cap_pl);
      uint32_t *dst = (uint32_t *)(spl + plofs[il]);
      const int nw = ((int)plcnt_s[il] + 1) >> 1;
      for (int p = wlane; p < nw; p += 32) dst[p] = __ldg(src + p);
    }
  }
  // static part of the active set: halo slots the bonds and natives of the own beads use
  if (multi) {
    for (int e = tid; e < n_own * cap_b; e += bd) {
      const int h = sbond[e].x - n_own;
      if (h >= 0) atomicOr(&sbm[h >> 5], 1u << (h & 31));
    }
    for (int e = tid; e < n_nat; e += bd) {
      const int h = natp[qbase + e].x - n_own;
      if (h >= 0) atomicOr(&sbm[h >> 5], 1u << (h & 31));
    }
  }
  __syncthreads();
#ifdef SOP_PHASE_CLOCKS
  long long pc_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, pc_t = clock64();
  int pc_dep = 0;
// the clock reads and the block barriers are tied by register dependences, or ptxas moves the reads across the barriers
#define SOP_TICK(n) { long long now_; asm volatile("mov.u64 %0, %%clock64;" : "=l"(now_) : "r"(pc_dep) : "memory"); pc_acc[n] += now_ - pc_t; pc_t = now_; }
#define SOP_SYNC() { pc_dep = __syncthreads_or((int)(pc_t >> 63)); }
#else
#define SOP_TICK(n)
#define SOP_SYNC() __syncthreads()
#endif
  // a3: Alg. 3 on the own rows, candidates and coordinates from shared memory
  auto filter_rows = [&](const float4 *P) {
    const uint32_t lt = (1u << wlane) - 1u;
    if ((SPEC == 2 || (SPEC == 0 && R.implicit_l1)) && n_own * 4 <= bd) {
      // static all-pairs L1, few rows (cfg 0): one warp per row scans every j, ballot + prefix-popcount compaction
      for (int il = warp; il < n_own; il += nwarps) {
        const int gi = b0 + il;
        const float4 ri = P[il];
        unsigned short *row = nb + (size_t)il * R.nb_si;
        int n = 0;
        for (int base = 0; base < n_own; base += 32) {
          const int j = base + wlane;
          const bool pass = j < n_own && j != il && pred32(ri, P[min(j, n_own - 1)], S.R_nb2) && !is_excluded(S, gi, b0 + j);
          const unsigned m = __ballot_sync(0xffffffffu, pass);
          if (pass) { const int at = n + __popc(m & lt); if (at < cap_nb) row[at] = (unsigned short)j; }
          n += __popc(m);
        }
        if (n > cap_nb) { flag |= FLAG_NB_OVERFLOW; n = cap_nb; }
        if (wlane == 0) { cnt_s[il] = (unsigned short)n; for (int k4 = n; k4 & 3; ++k4) row[k4] = DUMMY; }
      }
    } else if (SPEC == 2 || (SPEC == 0 && R.implicit_l1)) {
      // static all-pairs L1 (one chunk = the whole trajectory): L2 row of i = every j != i within R_nb that is not
      // bonded / native.  Candidates come from a cell grid over the chunk built here in shared memory (a1 in small:
      // bounding box -> count -> scan -> fill -> per-cell sort, so that the row order does not depend on atomics).
      int *gstart = (int *)spl, *gcur = gstart + (RES_GRID_CELLS + 1);
      unsigned short *gbead = (unsigned short *)(gcur + RES_GRID_CELLS), *gcell = gbead + R.chunk;
      if (tid < 6) misc[2 + tid] = tid < 3 ? 0x7FFFFFFF : (int)0x80000000;
      for (int cc = tid; cc < RES_GRID_CELLS; cc += bd) gcur[cc] = 0;
      __syncthreads();
      {
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
        for (int i = tid; i < n_own; i += bd) {
          const float4 r = P[i];
          lo[0] = fminf(lo[0], r.x); lo[1] = fminf(lo[1], r.y); lo[2] = fminf(lo[2], r.z);
          hi[0] = fmaxf(hi[0], r.x); hi[1] = fmaxf(hi[1], r.y); hi[2] = fmaxf(hi[2], r.z);
        }
#pragma unroll
        for (int a3 = 0; a3 < 3; ++a3) {
          for (int o = 16; o > 0; o >>= 1) {
            lo[a3] = fminf(lo[a3], __shfl_xor_sync(0xffffffffu, lo[a3], o));
            hi[a3] = fmaxf(hi[a3], __shfl_xor_sync(0xffffffffu, hi[a3], o));
          }
          if (wlane == 0) { atomicMin(&misc[2 + a3], f2ord(lo[a3])); atomicMax(&misc[5 + a3], f2ord(hi[a3])); }
        }
      }
      __syncthreads();
      // grid parameters, computed identically by every thread
      const float ox = ord2f(misc[2]), oy = ord2f(misc[3]), oz = ord2f(misc[4]);
      const float ex = fmaxf(0.f, ord2f(misc[5]) - ox), ey = fmaxf(0.f, ord2f(misc[6]) - oy), ez = fmaxf(0.f, ord2f(misc[7]) - oz);
      float edge = sqrtf(S.R_nb2) * 1.001f;
      int nx = 1, ny = 1, nz = 1;
      for (;;) {                             // counts in floating point first: no integer overflow on a blown-up chain
        const float fx = floorf(ex / edge) + 1.0f, fy = floorf(ey / edge) + 1.0f, fz = floorf(ez / edge) + 1.0f;
        if (fx >= 1.0f && fy >= 1.0f && fz >= 1.0f && fx < 1.0e6f && fy < 1.0e6f && fz < 1.0e6f &&
            (double)fx * (double)fy * (double)fz <= (double)RES_GRID_CELLS) { nx = (int)fx; ny = (int)fy; nz = (int)fz; break; }
        edge *= 1.25f;                       // cells may only grow: the 27-cell scan stays complete
        if (!(edge < 1.0e30f)) break;        // non-finite extent: one cell
      }
      const float inv_edge = 1.0f / edge;
      const int ncell = nx * ny * nz;
      auto cell3 = [&](const float4 &r, int &cx, int &cy, int &cz) {
        cx = min(max((int)floorf((r.x - ox) * inv_edge), 0), nx - 1);
        cy = min(max((int)floorf((r.y - oy) * inv_edge), 0), ny - 1);
        cz = min(max((int)floorf((r.z - oz) * inv_edge), 0), nz - 1);
      };
      for (int i = tid; i < n_own; i += bd) {
        int cx, cy, cz;
        cell3(P[i], cx, cy, cz);
        const int cc = (cz * ny + cy) * nx + cx;
        gcell[i] = (unsigned short)cc;
        atomicAdd(&gcur[cc], 1);
      }
      __syncthreads();
      if (warp == 0) {
        int carry = 0;
        for (int base = 0; base < ncell; base += 32) {
          const int cc = base + wlane;
          const int v = cc < ncell ? gcur[cc] : 0;
          int inc = v;
          for (int o = 1; o < 32; o <<= 1) { const int nn = __shfl_up_sync(0xffffffffu, inc, o); if (wlane >= o) inc += nn; }
          if (cc < ncell) { gstart[cc] = carry + inc - v; gcur[cc] = 0; }
          carry += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (wlane == 0) gstart[ncell] = carry;
      }
      __syncthreads();
      for (int i = tid; i < n_own; i += bd) {
        const int cc = gcell[i];
        gbead[gstart[cc] + atomicAdd(&gcur[cc], 1)] = (unsigned short)i;
      }
      __syncthreads();
      for (int cc = tid; cc < ncell; cc += bd) {          // insertion sort of one (small) cell per thread
        const int s0 = gstart[cc], e0 = gstart[cc + 1];
        for (int a2 = s0 + 1; a2 < e0; ++a2) {
          const unsigned short v = gbead[a2];
          int b2 = a2 - 1;
          while (b2 >= s0 && gbead[b2] > v) { gbead[b2 + 1] = gbead[b2]; --b2; }
          gbead[b2 + 1] = v;
        }
      }
      __syncthreads();
      // cell-sorted copy of the coordinates (.w = slot) in the force buffer, which is dead between the update and the next
      // pair phase: the row scan below then streams its candidates without a dependent index load per candidate
      float4 *gpos = sforce;
      for (int q = tid; q < n_own; q += bd) {
        const int j = gbead[q];
        float4 r = P[j];
        r.w = __int_as_float(j);
        gpos[q] = r;
      }
      __syncthreads();
      // one thread per row: with a whole trajectory in the chunk there are about as many rows as threads, and a
      // private counter compacts without ballots (12x fewer warp instructions than a warp per row, measured)
      for (int il = tid; il < n_own; il += bd) {
        const int gi = b0 + il;
        const float4 ri = P[il];
        unsigned short *row = nb + (size_t)il * R.nb_si;
        int cx, cy, cz, n = 0;
        cell3(ri, cx, cy, cz);
        for (int z = max(cz - 1, 0); z <= min(cz + 1, nz - 1); ++z)
          for (int y = max(cy - 1, 0); y <= min(cy + 1, ny - 1); ++y) {
            const int c0 = (z * ny + y) * nx + max(cx - 1, 0), c1 = (z * ny + y) * nx + min(cx + 1, nx - 1);
            const int e0 = gstart[c1 + 1];
#pragma unroll 4
            for (int q = gstart[c0]; q < e0; ++q) {
              const float4 rj = gpos[q];
              const int j = __float_as_int(rj.w);
              if (j != il && pred32(ri, rj, S.R_nb2)) {
                if (n < R.nb_si) row[n] = (unsigned short)j;
                ++n;
              }
            }
          }
        // the bonded and native partners inside R_nb are struck afterwards: their indices are a handful of independent
        // loads, where a membership test inside the loop would be a dependent global search per candidate
        if (n > R.nb_si) { flag |= FLAG_NB_OVERFLOW; n = R.nb_si; }
        // (eight exclusions at a time in registers, loaded together; one compacting pass over the row per round: the
        // search per exclusion it replaces diverged on every row length and was 22 % of the filter's instructions)
        {
          const int x_lo = __ldg(&S.excl_ptr[gi]), x_hi = __ldg(&S.excl_ptr[gi + 1]);
          for (int x0 = x_lo; x0 < x_hi; x0 += 8) {
            int ex[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) ex[u] = x0 + u < x_hi ? __ldg(&S.excl_idx[x0 + u]) - b0 : -1;
            int m = 0;
            for (int p = 0; p < n; ++p) {
              const int v = row[p];
              bool hit = false;
#pragma unroll
              for (int u = 0; u < 8; ++u) hit |= v == ex[u];
              if (!hit) row[m++] = (unsigned short)v;
            }
            n = m;
          }
        }
        if (n > cap_nb) { flag |= FLAG_NB_OVERFLOW; n = cap_nb; }
        cnt_s[il] = (unsigned short)n;
        for (int k4 = n; k4 & 3; ++k4) row[k4] = DUMMY;
      }
    } else {
      // LPR lanes per row (as many as the block has per own bead, a power of two): a lane tests a contiguous run of
      // 64 candidates per round into a 64-bit mask -- no ballots, no popcounts per candidate -- then the lanes of the
      // row exchange their counts and write their survivors in row order (Alg. 3 keeps the L1 order)
      int LPR = 1;
      while (LPR < 32 && 2 * LPR * n_own <= bd) LPR <<= 1;
      const int frow = tid / LPR, flane = tid & (LPR - 1), fgroups = bd / LPR;
      auto rows_loop = [&](auto in_smem_t) {
      constexpr bool IN_SMEM = decltype(in_smem_t)::value;     // plain LDS when the rows are resident, else global loads
      for (int base = 0; base < n_own; base += fgroups) {
        const bool valid = base + frow < n_own;
        const int il = STREAM ? (valid ? base + frow : n_own - 1) : order[valid ? base + frow : n_own - 1];      // dense beads together: similar L1 row lengths per warp
        const int cnt1 = valid ? (int)plcnt_s[il] : 0;
        const int nw = (cnt1 + 1) >> 1;
        const float4 ri = P[il];
        const uint32_t *gsrc = (const uint32_t *)(R.pl_loc + (inst0 + b0 + il) * S.cap_pl);
        const uint32_t *ssrc = (const uint32_t *)(spl + (IN_SMEM ? plofs[il] : 0));
        auto word = [&](int w) -> uint32_t { return IN_SMEM ? ssrc[w] : __ldg(gsrc + w); };
        unsigned short *row = nb + (size_t)il * R.nb_si;
        const int rounds = __reduce_max_sync(0xffffffffu, (nw + 32 * LPR - 1) / (32 * LPR));
        int n = 0;
        for (int r = 0; r < rounds; ++r) {
          // the (up to 32 LPR) words of this round are split evenly: at most 32 words = 64 candidates per lane
          const int rw0 = r * 32 * LPR, rwn = min(32 * LPR, nw - rw0), per = (max(rwn, 0) + LPR - 1) / LPR;
          const int w0 = rw0 + flane * per;
          // survivors as two 32-bit masks (low / high slot of word k2 at bit k2): one predicated OR per candidate
          uint32_t ma = 0u, mb = 0u, bit = 1u;
          const int wend = min(per, rwn - flane * per);
#pragma unroll 4
          for (int k2 = 0; k2 < wend; ++k2) {
            const uint32_t u = word(w0 + k2);
            const bool pa = pred32(ri, P[u & 0xFFFFu], S.R_nb2);
            const bool pb = 2 * (w0 + k2) + 1 < cnt1 && pred32(ri, P[u >> 16], S.R_nb2);
            if (pa) ma |= bit;
            if (pb) mb |= bit;
            bit <<= 1;
          }
          const int mine = __popc(ma) + __popc(mb);
          int incl = mine;
          for (int o = 1; o < LPR; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o, LPR); if (flane >= o) incl += v; }
          const int total = __shfl_sync(0xffffffffu, incl, LPR - 1, LPR);
          int at = n + incl - mine;
          uint32_t many = ma | mb;
          while (many) {                               // words with a survivor, in row order: low slot before high slot
            const int k2 = __ffs((int)many) - 1;
            many &= many - 1;
            const uint32_t u = word(w0 + k2);
            if ((ma >> k2) & 1u) { if (at < cap_nb) row[at] = (unsigned short)(u & 0xFFFFu); ++at; }
            if ((mb >> k2) & 1u) { if (at < cap_nb) row[at] = (unsigned short)(u >> 16); ++at; }
          }
          n += total;
        }
        if (n > cap_nb) { flag |= FLAG_NB_OVERFLOW; n = cap_nb; }
        if (valid && flane == 0) { cnt_s[il] = (unsigned short)n; for (int k4 = n; k4 & 3; ++k4) row[k4] = DUMMY; }
      }
      };
      if (pl_in_smem) rows_loop(std::true_type{}); else rows_loop(std::false_type{});
    }
  };
  // active halo = static part + halo slots of the current L2 rows
  auto after_filter = [&]() {
    __syncthreads();                                   // the row counts are complete
    for (int w = tid; w < HW; w += bd) bm[w] = sbm[w];
    if (tid == 0) misc[0] = 0;
    __syncthreads();
    if (multi) {
      const int r8 = tid >> 3, l8 = tid & 7, g8 = bd >> 3;               // eight lanes per (short) row
      for (int il = r8; il < n_own; il += g8) {
        const int cnt = cnt_s[il];
        const unsigned short *row = nb + (size_t)il * R.nb_si;
        for (int p = l8; p < cnt; p += 8) {
          const int h = (int)row[p] - n_own;
          if (h >= 0) {
            const uint32_t bit = 1u << (h & 31);
            if (!(((volatile uint32_t *)bm)[h >> 5] & bit)) atomicOr(&bm[h >> 5], bit);
          }
        }
      }
    }
    __syncthreads();
    // bitmap -> list: a warp per word, a lane per bit (the order of the list does not matter, only who polls what)
    // (STREAM keeps the bitmap only: the list of a 9000-slot halo would not fit)
    for (int w = warp; w < HW && !STREAM; w += nwarps) {
      const uint32_t m = bm[w];
      if (m) {
        int at = 0;
        if (wlane == 0) at = atomicAdd(&misc[0], __popc(m));
        at = __shfl_sync(0xffffffffu, at, 0);
        if ((m >> wlane) & 1u) active[at + __popc(m & ((1u << wlane) - 1u))] = (unsigned short)(n_own + (w << 5) + wlane);
      }
    }
    __syncthreads();
  };
  if (filter_first) filter_rows(spos);
  after_filter();

  // ---- the steps
  ForceK K;
  K.k_fene = S.k_fene; K.inv_R0sq = S.inv_R0sq; K.eps12 = 12.0f * S.eps_native; K.c_rep_f = S.c_rep_f;
  const float *nat_eps = FAST ? nullptr : S.nat_eps;
  int until_filter = nb_interval - (int)(step0 % (unsigned long long)nb_interval);
  bool have_full = true;                     // the whole halo of the current layer is already in shared memory (prologue)
  for (int k = 0; k < n_steps; ++k) {
    const unsigned long long step = step0 + (unsigned long long)k;
    float4 *pc = spos + (STREAM ? 0 : (size_t)(k & 1) * SC), *pn = spos + (STREAM ? 0 : (size_t)((k & 1) ^ 1) * SC);
    float4 *gc = sg + (size_t)(k & 1) * R.chunk, *gnx = sg + (size_t)((k & 1) ^ 1) * R.chunk;
    uint4 *const xc = (k & 1) ? xl1 : xl0, *const xn = (k & 1) ? xl0 : xl1;
    const uint32_t st_c = stamp0 + (uint32_t)k, st_n = st_c + 1u;
    const ExtStep ext = ext_step(S, step);          // fp64 conversions of the step number: before the waits, not after
    // (b) active halo of layer k: poll until the neighbours have published it
    if (multi && !have_full && STREAM) {
      for (int w = warp; w < HW; w += nwarps) {              // a warp per bitmap word, a lane per halo slot
        if ((bm[w] >> wlane) & 1u) {
          const int h = (w << 5) + wlane;
          float4 v;
          xch_wait(xc + 2 * (inst0 + hgid[h]), st_c, v, S.flags);
          pc[n_own + h] = v;
        }
      }
    } else if (multi && !have_full) {
      const int na = misc[0];
      for (int q = tid; q < na; q += bd) {
        const int slot = active[q];
        const uint4 *src = xc + 2 * (inst0 + hgid[slot - n_own]);
        float4 v;
        xch_wait(src, st_c, v, S.flags);
        pc[slot] = v;
      }
    }
    have_full = false;
    SOP_TICK(0)                                                                            // halo poll
    SOP_SYNC();
    SOP_TICK(1)                                                                            // waiting for the slowest poller
    // (d1) a4..a6: internal force, G lanes per bead (Alg. 2; no distance test in the loop, R3c)
    for (int base = 0; base < n_own; base += groups) {
      const bool valid = base + grp < n_own;
      const int il = STREAM ? (valid ? base + grp : n_own - 1) : order[valid ? base + grp : n_own - 1];
      const float4 ri = pc[il];
      float fx = 0.f, fy = 0.f, fz = 0.f;
      if (valid) {
        // a4: FENE bonds   V = -(k/2) R0^2 ln(1 - (r-r0)^2/R0^2)
        for (int p = lane; p < cap_b; p += G) {
          const int2 b = sbond[il * cap_b + p];
          if (b.x >= 0) {
            const float4 rj = pc[b.x];
            const float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
            const float r2 = dx * dx + dy * dy + dz * dz;
            const float inv_r = rsqrtf(r2);
            const float del = r2 * inv_r - __int_as_float(b.y);
            const float x = 1.0f - del * del * K.inv_R0sq;
            if (!(x > 0.0f)) flag |= FLAG_FENE;
            const float s = -K.k_fene * del * fast_rcp(x) * inv_r;
            fx += s * dx; fy += s * dy; fz += s * dz;
          }
        }
        // a5: native contacts   V = eps [(r0/r)^12 - 2 (r0/r)^6]   (per-contact eps only when the topology has it)
        const int q1 = natq[il + 1];
        auto natives = [&](auto has_eps_t, auto in_smem_t) {
          constexpr bool HAS_EPS = decltype(has_eps_t)::value, IN_SMEM = decltype(in_smem_t)::value;
          const int q0 = natq[il];
          for (int q = q0 + lane; q < q1; q += G) {
            const int2 en = IN_SMEM ? snat[q - qbase]           // a plain LDS.64 (the generic pointer costs address checks)
                                    : R.nat_T ? __ldg(&R.nat_T[(size_t)(q - q0) * R.nat_tpad + il]) : natp[q];
            float e12 = K.eps12;
            if (HAS_EPS) e12 = 12.0f * __ldg(&nat_eps[q]);
            const float4 rj = pc[en.x];
            const float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
            const float s = nat_s3(dx * dx + dy * dy + dz * dz, __int_as_float(en.y), e12);
            fx += s * dx; fy += s * dy; fz += s * dz;
          }
        };
        if (STREAM && !nat_eps) {
          // the table comes from global memory (L2): eight independent entry loads in flight, then their gathers
          // (an entry past the end is the dummy slot with r0^2 = 0: its term is exactly zero)
          const int q0 = natq[il];
          for (int q = q0 + lane; q < q1; q += 8 * G) {
            int2 en[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) en[u] = q + u * G < q1 ? __ldg(&natp[q + u * G]) : make_int2((int)DUMMY, 0);
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const float4 rj = pc[en[u].x];
              const float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
              const float s = nat_s3(dx * dx + dy * dy + dz * dz, __int_as_float(en[u].y), K.eps12);
              fx += s * dx; fy += s * dy; fz += s * dz;
            }
          }
        }
        else if (SPEC == 2 ? G == 1 : SPEC == 0 && !nat_eps && R.nat_T) {
          // one-chunk trajectories with one lane per bead (cfg 1): the transposed table is read coalesced from L2, eight
          // independent entry loads in flight instead of one L2 round trip per native contact (same order of summation;
          // an entry past the end is the dummy slot with r0^2 = 0: its term is exactly zero)
          const int nq = q1 - natq[il];
          const int tpad = R.nat_tpad;                      // (rows x tpad entries fit 32 bits: N <= 65535 slots per chunk)
          for (int r = 0; r < nq; r += 8) {
            int2 en[8];
            const int2 *np = R.nat_T + (r * tpad + il);
#pragma unroll
            for (int u = 0; u < 8; ++u) en[u] = r + u < nq ? __ldg(np + u * tpad) : make_int2((int)DUMMY, 0);
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const float4 rj = pc[en[u].x];
              const float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
              const float s = nat_s3(dx * dx + dy * dy + dz * dz, __int_as_float(en[u].y), K.eps12);
              fx += s * dx; fy += s * dy; fz += s * dz;
            }
          }
        }
        else if (nat_eps) natives(std::true_type{}, std::false_type{});
        else if (SPEC == 1 || (SPEC == 2 && G > 1) || (SPEC == 0 && R.nat_smem)) natives(std::false_type{}, std::true_type{});
        else natives(std::false_type{}, std::false_type{});
        // a6: non-native repulsion   V = eps_r (sigma/r)^6; four slots per 8-byte word (rows are padded to a multiple
        // of four with the dummy slot): one index load, four gathers in flight
        const uint2 *row64 = (const uint2 *)(nb + (size_t)il * R.nb_si);
        const int n4 = ((int)cnt_s[il] + 3) >> 2;
        uint2 wn = make_uint2(0u, 0u);
        if (STREAM && lane < n4) wn = row64[lane];                  // (global memory: the next word is in flight while this one is used)
        for (int p = lane; p < n4; p += G) {
          uint2 w;
          if (STREAM) { w = wn; if (p + G < n4) wn = row64[p + G]; }
          else w = row64[p];
          const float4 ra = pc[w.x & 0xFFFFu], rb = pc[w.x >> 16], rc = pc[w.y & 0xFFFFu], rd = pc[w.y >> 16];
          const float ax = ri.x - ra.x, ay = ri.y - ra.y, az = ri.z - ra.z;
          const float bx = ri.x - rb.x, by = ri.y - rb.y, bz = ri.z - rb.z;
          const float cx = ri.x - rc.x, cy = ri.y - rc.y, cz = ri.z - rc.z;
          const float dx = ri.x - rd.x, dy = ri.y - rd.y, dz = ri.z - rd.z;
          const float sa = rep_s3(ax * ax + ay * ay + az * az, K.c_rep_f);
          const float sb = rep_s3(bx * bx + by * by + bz * bz, K.c_rep_f);
          const float sc = rep_s3(cx * cx + cy * cy + cz * cz, K.c_rep_f);
          const float sd = rep_s3(dx * dx + dy * dy + dz * dz, K.c_rep_f);
          fx += sa * ax; fy += sa * ay; fz += sa * az;
          fx += sb * bx; fy += sb * by; fz += sb * bz;
          fx += sc * cx; fy += sc * cy; fz += sc * cz;
          fx += sd * dx; fy += sd * dy; fz += sd * dz;
        }
      }
      if (G > 1) { fx = group_sum<G>(fx); fy = group_sum<G>(fy); fz = group_sum<G>(fz); }
      if (valid && lane == 0) sforce[il] = make_float4(fx, fy, fz, 0.f);
    }
    SOP_TICK(2)                                                                            // pair forces
    SOP_SYNC();
    SOP_TICK(3)                                                                            // waiting for the slowest warp
    // (d2) a7 + a9: thread per bead; the other end of the block draws the next step's noise (a8)
    const bool filt_due = until_filter == 1 && (k + 1 < n_steps || filter_last);   // the new layer is one every chunk filters on
    if (filt_due) fpar ^= 1u;
    uint4 *const xpub = filt_due ? (fpar ? xf1 : xf0) : xn;
    if (!FAST && R.skew_ns && tc == R.skew_chunk && step % (unsigned long long)R.skew_period == 0) __nanosleep((unsigned)R.skew_ns);
    for (int i = tid; i < n_own; i += bd) {
      const float4 ri = pc[i];
      const uint32_t tag = stag[i];
      const float4 a = sforce[i];
      float4 out = ri;
      if (!(tag & TAG_FIXED)) {
        float fx = a.x, fy = a.y, fz = a.z;
        external_force_at(S, b0 + i, ri, tag, ext, fx, fy, fz, flag);
        float3 gn;
        if (G > 1) { const float4 g4 = gc[i]; gn = make_float3(g4.x, g4.y, g4.z); }
        else gn = !FAST && S.taus ? gaussian3_taus(S.taus + inst0 + b0 + i) : gaussian3(S, tag & TAG_ID_MASK, traj, step);   // thread per bead already
        out = langevin_apply<COMP>(S, ri, gn, fx, fy, fz, COMP ? scarry + i : nullptr, flag, amp_tr);
      }
      pn[i] = out;
      if (multi) xch_put(xpub + 2 * (inst0 + b0 + i), out, st_n);
    }
    if (G > 1 && k + 1 < n_steps) {
      for (int i = bd - 1 - tid; i < n_own; i += bd) {
        const uint32_t tag = stag[i];
        if (!(tag & TAG_FIXED)) {
          const float3 gn = !FAST && S.taus ? gaussian3_taus(S.taus + inst0 + b0 + i) : gaussian3(S, tag & TAG_ID_MASK, traj, step + 1);
          gnx[i] = make_float4(gn.x, gn.y, gn.z, 0.f);
        }
      }
    }
    SOP_TICK(4)                                                                            // update + noise
    // (e) a3: Alg. 3 on the own rows from the coordinates just written (list invariant)
    if (--until_filter == 0) {
      until_filter = nb_interval;
      if (k + 1 < n_steps || filter_last) {
        if (multi)
          for (int q = tid; q < n_halo; q += bd) {
            const uint4 *src = xpub + 2 * (inst0 + hgid[q]);
            float4 v;
            xch_wait(src, st_n, v, S.flags);
            pn[n_own + q] = v;
          }
        __syncthreads();
        filter_rows(pn);
        after_filter();
        have_full = true;
      }
      SOP_TICK(5)                                                                          // filter (whole-halo poll, rows, active set)
    }
  }
#ifdef SOP_PHASE_CLOCKS
  if (wlane == 0) {
    S.force[((size_t)blockIdx.x * 32 + warp) * 2] = make_float4((float)pc_acc[0], (float)pc_acc[1], (float)pc_acc[2], (float)pc_acc[3]);
    S.force[((size_t)blockIdx.x * 32 + warp) * 2 + 1] = make_float4((float)pc_acc[4], (float)pc_acc[5], (float)pc_acc[6], (float)pc_acc[7]);
  }
#endif

  // ---- epilogue: the current layer, the carry and the L2 rows back to the canonical arrays
  __syncthreads();
  const float4 *pf = spos + (STREAM ? 0 : (size_t)(n_steps & 1) * SC);
  for (int i = tid; i < n_own; i += bd) {
    S.pos[cur][inst0 + b0 + i] = pf[i];
    if (COMP) S.carry[inst0 + b0 + i] = scarry[i];
  }
  for (int il = warp; il < n_own; il += nwarps) {
    const size_t g = inst0 + b0 + il;
    const int cnt = cnt_s[il];
    int *canon = S.nb_idx + g * cap_nb;
    for (int p = wlane; p < cnt; p += 32) {
      const int slot = nb[(size_t)il * R.nb_si + p];
      canon[p] = slot < n_own ? b0 + slot : hgid[slot - n_own];
    }
    if (wlane == 0) S.nb_cnt[g] = cnt;
  }
  if (flag) atomicOr(S.flags, flag);
  if (!STREAM && R.slice_len > 0) {            // this trajectory's next slice may start: release what every thread wrote
    __syncthreads();
    if (tid == 0) { __threadfence(); asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(R.done + tc), "r"(slice + 1) : "memory"); }
  }
}

}  // namespace sop

// sop_device.cuh -- device-side building blocks of the SOP Langevin hot path (sm_100a).
//
// Everything here is fp32 on SoA float4 coordinates.  Citations are to PAPER.md (arxiv 1003.1148) and to the
// readings listed in DESIGN.md.  No code is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sop {

// bits of the device flag word
enum : int { FLAG_PL_OVERFLOW = 1, FLAG_NB_OVERFLOW = 2, FLAG_FENE = 4, FLAG_NONFINITE = 8 };

// bits stored in float4.w of every coordinate (an integer tag, never used in arithmetic)
constexpr uint32_t TAG_FIXED = 0x80000000u;
constexpr uint32_t TAG_PULLED = 0x40000000u;
constexpr uint32_t TAG_ID_MASK = 0x0FFFFFFFu;   // caller's bead index (Philox counter word 0)

struct GridDev {          // per-trajectory cell grid, written on the device by k_grid_setup
  float ox, oy, oz;       // origin (bounding-box minimum)
  float inv_edge;
  int nx, ny, nz;
  int ncell;
};

struct SysDev {
  int N, T;
  int n_inst;                       // T * N bead instances
  float4 *pos[2];                   // [T][N] ping-pong time layers
  float4 *carry;                    // [T][N] Kahan carry or nullptr
  float4 *force;                    // [T][N] output of the forces-only instantiation
  // static tables in internal bead order, shared by all trajectories
  int cap_b;
  const int2 *bond_tab;             // [N][cap_b] {j, bits(r0)}; j = -1: empty slot
  const int *nat_ptr;               // [N+1]
  const int2 *nat_tab;              // [nat_ptr[N]] {j, bits(r0^2)}
  const float *nat_eps;             // [nat_ptr[N]] or nullptr (uniform eps_native)
  const int *excl_ptr;              // [N+1] bonded + native partners, ascending
  const int *excl_idx;
  const float *pull_adotn;          // [N] a_p . n of the pulled beads (nullptr if none)
  // lists
  int static_l1;                    // R_pl = +inf: one L1 [N][cap_pl] shared by all trajectories
  int cap_pl, cap_nb;
  int *pl_cnt, *pl_idx;             // L1 "pair list"      (PossiblePairsMap)
  int *nb_cnt, *nb_idx;             // L2 "neighbor list"  (PairsMap of Alg. 3)
  // cell grid
  int max_cells;
  float *bbox;                      // [T][6] as ordered ints
  GridDev *grid;                    // [T]
  int *cell_of;                     // [T][N]
  int *cell_cnt;                    // [T][max_cells]   (reused as fill cursor)
  int *cell_start;                  // [T][max_cells+1]
  int *cell_bead;                   // [T][N] beads sorted by (cell, internal index)
  float4 *cell_pos;                 // [T][N] {x, y, z, bead index} in the same order
  float cell_edge;
  // parameters (fp32, derived once on the host in fp64)
  float k_fene, R0, inv_R0sq;
  float eps_native;
  float c_rep_f;                    // 6 eps_r sigma^6
  float c_rep_e;                    // eps_r sigma^6
  float R_nb2, R_pl2;               // (float)(R*R): the canonical cutoffs of the list predicate
  float D, amp;                     // h/xi and sqrt(2 kT h/xi)
  const float *amp_t;               // [T] sqrt(2 kT_t h/xi): one temperature per trajectory (NEXT-4), or nullptr
  uint32_t seed_lo, seed_hi;
  int traj_offset;
  int has_pull; float pull_k, pull_v, pull_nx, pull_ny, pull_nz;
  int tip_on; float tip_R, tip_eps, tip_sigma6, tip_v, tip_cx, tip_cy, tip_cz, tip_nx, tip_ny, tip_nz;
  uint4 *taus;                      // [T][N] Hybrid Taus states (params.rng == 1), else nullptr
  int *flags;
};

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11), entirely in registers: no generator state in memory, unlike the paper's
// per-thread Hybrid Taus state.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    uint32_t hi0 = __umulhi(M0, c.x), lo0 = M0 * c.x;
    uint32_t hi1 = __umulhi(M1, c.z), lo1 = M1 * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u;
    k.y += 0xBB67AE85u;
  }
  return c;
}

// Three N(0,1) numbers of bead `bead` of trajectory `traj` for the update step -> step+1 (reading R6):
// counter (bead, traj, step lo, step hi), key (seed lo, seed hi); top 24 bits -> uniforms exactly representable
// in fp32; Box-Muller; the 4th normal is discarded as in the paper.
__device__ __forceinline__ float3 gaussian3(const SysDev &S, uint32_t bead, uint32_t traj, unsigned long long step) {
  uint4 x = philox4x32_10(make_uint4(bead, traj, (uint32_t)step, (uint32_t)(step >> 32)),
                          make_uint2(S.seed_lo, S.seed_hi));
  const float k = 1.0f / 16777216.0f;
  float ua = (float)((x.x >> 8) + 1u) * k;
  float ub = (float)(x.y >> 8) * k;
  float uc = (float)((x.z >> 8) + 1u) * k;
  float ud = (float)(x.w >> 8) * k;
  float ra = sqrtf(-2.0f * __logf(ua));
  float rc = sqrtf(-2.0f * __logf(uc));
  float sb, cb;
  __sincosf(6.283185307179586f * ub, &sb, &cb);
  float cd = __cosf(6.283185307179586f * ud);
  return make_float3(ra * cb, ra * sb, rc * cd);
}

// ------------------------------------------------------------------------------------------------
// The list predicate "r < cutoff" (Alg. 3 line 9) in canonical fp32 arithmetic (reading R4):
// three subtractions, three products, two additions, each rounded once (no FMA contraction), strict <.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool pred32(const float4 &a, const float4 &b, float R2f) {
  float dx = __fsub_rn(a.x, b.x), dy = __fsub_rn(a.y, b.y), dz = __fsub_rn(a.z, b.z);
  float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
  return d2 < R2f;
}

template <bool NC>
__device__ __forceinline__ float4 ldpos(const float4 *p) {
  if (NC) return __ldg(p);      // read-only for the whole launch: non-coherent path
  return *p;                    // persistent kernel: coherent load (L1 is invalidated by the acquire at the grid barrier)
}

// ------------------------------------------------------------------------------------------------
// Pair force laws = -dV/dr of Eq. (1).  Each returns s with f_i += s * (r_i - r_j).
// ------------------------------------------------------------------------------------------------
// FENE: V = -(k/2) R0^2 ln(1 - (r-r0)^2/R0^2)   ->  s = -k (r-r0) / (1 - (r-r0)^2/R0^2) / r
__device__ __forceinline__ float fene_s(const SysDev &S, float r2, float r0, bool &bad, float *e = nullptr) {
  float inv_r = rsqrtf(r2);
  float r = r2 * inv_r;
  float del = r - r0;
  float x = 1.0f - del * del * S.inv_R0sq;
  bad = !(x > 0.0f);
  if (e) *e = -0.5f * S.k_fene * S.R0 * S.R0 * logf(x);
  return -S.k_fene * del * __frcp_rn(x) * inv_r;
}
// native 12-6: V = eps [(r0/r)^12 - 2 (r0/r)^6]  ->  s = (12 eps / r^2) (q^2 - q), q = (r0/r)^6
__device__ __forceinline__ float native_s(float r2, float r0sq, float eps, float *e = nullptr) {
  float inv_r2 = __frcp_rn(r2);
  float u = r0sq * inv_r2;
  float q = u * u * u;
  if (e) *e = eps * (q * q - 2.0f * q);
  return 12.0f * eps * inv_r2 * (q * q - q);
}
// repulsion: V = eps_r (sigma/r)^6  ->  s = 6 eps_r sigma^6 / r^8
__device__ __forceinline__ float rep_s(const SysDev &S, float r2, float *e = nullptr) {
  float inv_r2 = __frcp_rn(r2);
  float inv_r6 = inv_r2 * inv_r2 * inv_r2;
  if (e) *e = S.c_rep_e * inv_r6;
  return S.c_rep_f * inv_r6 * inv_r2;
}

template <int G>
__device__ __forceinline__ float group_sum(float v) {
#pragma unroll
  for (int o = G / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ------------------------------------------------------------------------------------------------
// Internal force on bead instance (t, i) summed over the G lanes of its group: bonds (a4), natives (a5),
// L2 partners (a6) -- Alg. 2 with the partner loop spread over G lanes.  No distance test in
// the loop (Alg. 2 has none; reading R3c).  Every lane of the group returns the full sum.
// ------------------------------------------------------------------------------------------------
template <int G, bool NC>
__device__ __forceinline__ float3 internal_force(const SysDev &S, const float4 *__restrict__ pos_t, int i, int g,
                                                 int lane, bool valid, const float4 &ri, int &flag) {
  float fx = 0.f, fy = 0.f, fz = 0.f;
  if (valid) {
    // a4: FENE bonds
    for (int p = lane; p < S.cap_b; p += G) {
      int2 e = __ldg(&S.bond_tab[(size_t)i * S.cap_b + p]);
      if (e.x >= 0) {
        float4 rj = ldpos<NC>(pos_t + e.x);
        float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
        float r2 = dx * dx + dy * dy + dz * dz;
        bool bad;
        float s = fene_s(S, r2, __int_as_float(e.y), bad);
        if (bad) flag |= FLAG_FENE;
        fx += s * dx; fy += s * dy; fz += s * dz;
      }
    }
    // a5: native contacts
    {
      int q0 = __ldg(&S.nat_ptr[i]), q1 = __ldg(&S.nat_ptr[i + 1]);
      for (int q = q0 + lane; q < q1; q += G) {
        int2 e = __ldg(&S.nat_tab[q]);
        float eps = S.nat_eps ? __ldg(&S.nat_eps[q]) : S.eps_native;
        float4 rj = ldpos<NC>(pos_t + e.x);
        float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
        float r2 = dx * dx + dy * dy + dz * dz;
        float s = native_s(r2, __int_as_float(e.y), eps);
        fx += s * dx; fy += s * dy; fz += s * dz;
      }
    }
    // a6: non-native repulsion over the neighbor list
    {
      int cnt = S.nb_cnt[g];
      const int *row = S.nb_idx + (size_t)g * S.cap_nb;
      for (int p = lane; p < cnt; p += G) {
        int j = row[p];
        float4 rj = ldpos<NC>(pos_t + j);
        float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
        float r2 = dx * dx + dy * dy + dz * dz;
        float s = rep_s(S, r2);
        fx += s * dx; fy += s * dy; fz += s * dz;
      }
    }
  }
  if (G > 1) { fx = group_sum<G>(fx); fy = group_sum<G>(fy); fz = group_sum<G>(fz); }
  return make_float3(fx, fy, fz);
}

// what a7 needs of the step number: spring-base advance and tip centre (computed once per step, off the critical path)
struct ExtStep { float vs_pull, cx, cy, cz; };
__device__ __forceinline__ ExtStep ext_step(const SysDev &S, unsigned long long step) {
  ExtStep e;
  e.vs_pull = (float)((double)S.pull_v * (double)step);
  const float vs = (float)((double)S.tip_v * (double)step);
  e.cx = S.tip_cx + vs * S.tip_nx; e.cy = S.tip_cy + vs * S.tip_ny; e.cz = S.tip_cz + vs * S.tip_nz;
  return e;
}

// a7: external forces on one bead (readings R7, R8), the step-dependent scalars given.
__device__ __forceinline__ void external_force_at(const SysDev &S, int i, const float4 &ri, uint32_t tag, const ExtStep &e,
                                                  float &fx, float &fy, float &fz, int &flag) {
  if (S.has_pull && (tag & TAG_PULLED)) {
    float proj = ri.x * S.pull_nx + ri.y * S.pull_ny + ri.z * S.pull_nz - __ldg(&S.pull_adotn[i]);
    float f = S.pull_k * (e.vs_pull - proj);
    fx += f * S.pull_nx; fy += f * S.pull_ny; fz += f * S.pull_nz;
  }
  if (S.tip_on) {
    float dx = ri.x - e.cx, dy = ri.y - e.cy, dz = ri.z - e.cz;
    float g2 = dx * dx + dy * dy + dz * dz;
    float inv_g = rsqrtf(g2);
    float gap = g2 * inv_g - S.tip_R;
    if (!(gap > 0.f)) flag |= FLAG_NONFINITE;
    float ig = __frcp_rn(gap);
    float ig2 = ig * ig;
    float s = 6.0f * S.tip_eps * S.tip_sigma6 * ig2 * ig2 * ig2 * ig * inv_g;
    fx += s * dx; fy += s * dy; fz += s * dz;
  }
}

// a7: external forces on one bead (readings R7, R8).
__device__ __forceinline__ void external_force(const SysDev &S, int i, const float4 &ri, uint32_t tag,
                                               unsigned long long step, float &fx, float &fy, float &fz, int &flag) {
  external_force_at(S, i, ri, tag, ext_step(S, step), fx, fy, fz, flag);
}

// ------------------------------------------------------------------------------------------------
// NEXT-2: the paper's Hybrid Taus generator (Alg. 6; constants: DESIGN.md reading R12): three
// Tausworthe components and one LCG, 16 bytes of state per bead instance in global memory, four draws per bead-step.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t taus_draw(uint4 &y) {
  uint32_t b;
  b = ((y.x << 13) ^ y.x) >> 19;  y.x = ((y.x & 4294967294u) << 12) ^ b;
  b = ((y.y << 2) ^ y.y) >> 25;   y.y = ((y.y & 4294967288u) << 4) ^ b;
  b = ((y.z << 3) ^ y.z) >> 11;   y.z = ((y.z & 4294967280u) << 17) ^ b;
  y.w = 1664525u * y.w + 1013904223u;
  return y.x ^ y.y ^ y.z ^ y.w;
}

__device__ __forceinline__ float3 box_muller3(uint32_t x0, uint32_t x1, uint32_t x2, uint32_t x3) {
  const float k = 1.0f / 16777216.0f;
  float ua = (float)((x0 >> 8) + 1u) * k, ub = (float)(x1 >> 8) * k, uc = (float)((x2 >> 8) + 1u) * k, ud = (float)(x3 >> 8) * k;
  float ra = sqrtf(-2.0f * __logf(ua)), rc = sqrtf(-2.0f * __logf(uc));
  float sb, cb;
  __sincosf(6.283185307179586f * ub, &sb, &cb);
  return make_float3(ra * cb, ra * sb, rc * __cosf(6.283185307179586f * ud));
}

// state load, four draws, state store: the traffic the counter-based generator does not have
__device__ __forceinline__ float3 gaussian3_taus(uint4 *state) {
  uint4 y = *state;
  const uint32_t x0 = taus_draw(y), x1 = taus_draw(y), x2 = taus_draw(y), x3 = taus_draw(y);
  *state = y;
  return box_muller3(x0, x1, x2, x3);
}

// a9: the position update of Alg. 7 line 5 given the three normals, optionally Kahan-compensated (R10).
__device__ __forceinline__ float amp_of(const SysDev &S, int t) { return S.amp_t ? __ldg(S.amp_t + t) : S.amp; }

template <bool COMP>
__device__ __forceinline__ float4 langevin_apply(const SysDev &S, const float4 &ri, const float3 &gn, float fx, float fy,
                                                 float fz, float4 *carry_slot, int &flag, float amp) {
  float dx = S.D * fx + amp * gn.x, dy = S.D * fy + amp * gn.y, dz = S.D * fz + amp * gn.z;
  float4 out;
  if (COMP) {
    float4 c = *carry_slot;
    float yx = __fsub_rn(dx, c.x), yy = __fsub_rn(dy, c.y), yz = __fsub_rn(dz, c.z);
    out.x = __fadd_rn(ri.x, yx); out.y = __fadd_rn(ri.y, yy); out.z = __fadd_rn(ri.z, yz);
    c.x = __fsub_rn(__fsub_rn(out.x, ri.x), yx);
    c.y = __fsub_rn(__fsub_rn(out.y, ri.y), yy);
    c.z = __fsub_rn(__fsub_rn(out.z, ri.z), yz);
    *carry_slot = c;
  } else {
    out.x = ri.x + dx; out.y = ri.y + dy; out.z = ri.z + dz;
  }
  out.w = ri.w;
  if (!isfinite(out.x + out.y + out.z)) flag |= FLAG_NONFINITE;
  return out;
}

// a8 + a9: noise and the position update.
template <bool COMP>
__device__ __forceinline__ float4 langevin_update(const SysDev &S, const float4 &ri, uint32_t tag, int t,
                                                  unsigned long long step, float fx, float fy, float fz,
                                                  float4 *carry_slot, int &flag, int inst = 0) {
  if (tag & TAG_FIXED) return ri;                                     // fixed beads are copied unchanged
  float3 gn = S.taus ? gaussian3_taus(S.taus + inst) : gaussian3(S, tag & TAG_ID_MASK, (uint32_t)(S.traj_offset + t), step);
  return langevin_apply<COMP>(S, ri, gn, fx, fy, fz, carry_slot, flag, amp_of(S, t));
}

// ------------------------------------------------------------------------------------------------
// a3: Alg. 3 for one bead by one warp: scan the L1 row in order, keep entries with
// pred32(R_nb), order-preserving compaction by ballot + prefix popcount.
// ------------------------------------------------------------------------------------------------
template <bool NC>
__device__ __forceinline__ void filter_row_warp(const SysDev &S, const float4 *__restrict__ pos_t, int i, int g,
                                                int lane, int &flag) {
  const int row1 = S.static_l1 ? i : g;
  const int cnt1 = S.pl_cnt[row1];
  const int *src = S.pl_idx + (size_t)row1 * S.cap_pl;
  int *dst = S.nb_idx + (size_t)g * S.cap_nb;
  const float4 ri = ldpos<NC>(pos_t + i);
  int n = 0;
  // 128 candidates per iteration: four index loads, then four coordinate gathers in flight per lane (the gathers are
  // L2 round trips for large systems), then four ordered compactions
  for (int base = 0; base < cnt1; base += 128) {
    int j[4];
    float4 rj[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int p = base + 32 * u + lane; j[u] = p < cnt1 ? src[p] : -1; }
#pragma unroll
    for (int u = 0; u < 4; ++u) rj[u] = j[u] >= 0 ? ldpos<NC>(pos_t + j[u]) : ri;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (base + 32 * u >= cnt1) break;
      const bool pass = j[u] >= 0 && pred32(ri, rj[u], S.R_nb2);
      unsigned m = __ballot_sync(0xffffffffu, pass);
      if (pass) {
        int slot = n + __popc(m & ((1u << lane) - 1u));
        if (slot < S.cap_nb) dst[slot] = j[u];
      }
      n += __popc(m);
    }
  }
  if (n > S.cap_nb) { flag |= FLAG_NB_OVERFLOW; n = S.cap_nb; }
  if (lane == 0) S.nb_cnt[g] = n;
}

}  // namespace sop

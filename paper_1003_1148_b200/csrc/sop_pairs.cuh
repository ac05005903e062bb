// sop_pairs.cuh -- mode 4: the paper's interacting-pair based parallelisation (NEXT-3).
//
// Alg. 4: one thread per interacting pair computes the pair force ONCE and saves +df and -df to two unique places
// F[i][shift_i], F[j][shift_j] of a force array; Alg. 5: a gathering kernel, one thread per particle, sums the places of
// its particle -- here "incorporated into the integration kernel", as the paper suggests.  The atomics
// form the paper anticipates for Fermi ("thread safe atomic addition of the computed force values") is the
// second variant: +-df go to one accumulator per particle with atomicAdd.
//
// The place of a pair in F follows the tables the particle-based kernels use, so no extra bookkeeping is stored:
//   bond b of bead i          -> i * cap_b + b
//   native entry q of bead i  -> N * cap_b + q                (q = nat_ptr[i] + k)
//   L2 partner p of bead i    -> N * cap_b + n_nat + i * cap_nb + p
// Static pairs (bonds, natives) are listed once at create; the vector of L2 pairs is re-formed after every filter from
// the symmetric L2 rows (each pair taken from the row of its smaller index; its place in the other row is searched).
// The paper forms this vector on the CPU because its order matters for the texture cache; here the order
// does not matter for the result -- every force lands in its own place and Alg. 5 sums the places in row order -- so the
// vector is compacted on the device with one atomicAdd per warp.
#pragma once
#include "sop_kernels.cuh"

namespace sop {

struct PairDev {
  int n_static;              // bonds + natives, each once
  int n_bonds;               // the first n_bonds static pairs are bonds
  const int4 *spair;         // [n_static] {i, j, place_i, place_j}
  const float2 *spar;        // [n_static] {r0 (bond) or r0^2 (native), eps (native)}
  int cap_pairs;             // L2 pairs per trajectory the vector holds
  int4 *lpair;               // [T][cap_pairs] {i, j, place_i, place_j}
  int *n_lpair;              // [T]
  int n_place;               // places of one trajectory: N cap_b + n_nat + N cap_nb
  float4 *F;                 // [T][n_place]   (Alg. 4 lines 12-13)
  float *Facc;               // [T][N][4] accumulators of the atomics form
  int atomics;               // 0: unique places + gather (Alg. 4 + 5); 1: atomicAdd
};

// the vector of L2 pairs ("forming the vector pairs of all residue pairs"): one warp per row
__global__ void __launch_bounds__(256) k_pairs_build(SysDev S, PairDev P) {
  const int w = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int lane = threadIdx.x & 31;
  if (w >= S.n_inst) return;
  const int t = w / S.N, i = w - t * S.N;
  const int cnt = min(S.nb_cnt[w], S.cap_nb);
  const int *row = S.nb_idx + (size_t)w * S.cap_nb;
  const int base_r = S.N * S.cap_b + __ldg(&S.nat_ptr[S.N]);
  for (int b0 = 0; b0 < cnt; b0 += 32) {
    const int p = b0 + lane;
    const int j = p < cnt ? row[p] : -1;
    int q = -1;
    if (j > i) {                                         // the pair belongs to the row of its smaller index
      const size_t gj = (size_t)t * S.N + j;
      const int cj = min(S.nb_cnt[gj], S.cap_nb);
      const int *rj = S.nb_idx + gj * S.cap_nb;
      for (int k = 0; k < cj; ++k) if (rj[k] == i) { q = k; break; }
    }
    const bool take = q >= 0;
    const unsigned m = __ballot_sync(0xffffffffu, take);
    int at = 0;
    if (lane == 0 && m) at = atomicAdd(&P.n_lpair[t], __popc(m));
    at = __shfl_sync(0xffffffffu, at, 0) + __popc(m & ((1u << lane) - 1u));
    if (take && at < P.cap_pairs) P.lpair[(size_t)t * P.cap_pairs + at] = make_int4(i, j, base_r + i * S.cap_nb + p, base_r + j * S.cap_nb + q);
  }
}

// Alg. 4: thread = pair.  grid.y = trajectory.
__global__ void __launch_bounds__(256) k_pair_forces(SysDev S, PairDev P, int cur) {
  const int t = blockIdx.y;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  const int n_l = min(P.n_lpair[t], P.cap_pairs);
  if (p >= P.n_static + n_l) return;
  const float4 *__restrict__ pos_t = S.pos[cur] + (size_t)t * S.N;
  int4 pr;
  float s;
  int flag = 0;
  if (p < P.n_static) {
    pr = __ldg(&P.spair[p]);                                         // lines 2-7
    const float2 par = __ldg(&P.spar[p]);
    const float4 ri = __ldg(pos_t + pr.x), rj = __ldg(pos_t + pr.y);  // lines 8-9
    const float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z; // line 10
    const float r2 = dx * dx + dy * dy + dz * dz;
    if (p < P.n_bonds) { bool bad; s = fene_s(S, r2, par.x, bad); if (bad) flag |= FLAG_FENE; }
    else s = native_s(r2, par.x, par.y);
    const float4 df = make_float4(s * dx, s * dy, s * dz, 0.f);       // line 11
    if (P.atomics) {
      float *a = P.Facc + ((size_t)t * S.N + pr.x) * 4, *b = P.Facc + ((size_t)t * S.N + pr.y) * 4;
      atomicAdd(a, df.x); atomicAdd(a + 1, df.y); atomicAdd(a + 2, df.z);
      atomicAdd(b, -df.x); atomicAdd(b + 1, -df.y); atomicAdd(b + 2, -df.z);
    } else {
      float4 *F = P.F + (size_t)t * P.n_place;
      F[pr.z] = df;                                                    // line 12
      F[pr.w] = make_float4(-df.x, -df.y, -df.z, 0.f);                 // line 13
    }
  } else {
    pr = P.lpair[(size_t)t * P.cap_pairs + (p - P.n_static)];
    const float4 ri = __ldg(pos_t + pr.x), rj = __ldg(pos_t + pr.y);
    const float dx = ri.x - rj.x, dy = ri.y - rj.y, dz = ri.z - rj.z;
    s = rep_s(S, dx * dx + dy * dy + dz * dz);
    const float4 df = make_float4(s * dx, s * dy, s * dz, 0.f);
    if (P.atomics) {
      float *a = P.Facc + ((size_t)t * S.N + pr.x) * 4, *b = P.Facc + ((size_t)t * S.N + pr.y) * 4;
      atomicAdd(a, df.x); atomicAdd(a + 1, df.y); atomicAdd(a + 2, df.z);
      atomicAdd(b, -df.x); atomicAdd(b + 1, -df.y); atomicAdd(b + 2, -df.z);
    } else {
      float4 *F = P.F + (size_t)t * P.n_place;
      F[pr.z] = df;
      F[pr.w] = make_float4(-df.x, -df.y, -df.z, 0.f);
    }
  }
  if (flag) atomicOr(S.flags, flag);
}

// Alg. 5 inside the integration kernel: thread = particle sums its places (or reads and clears its
// accumulator), adds the external terms (a7), draws the noise (a8) and moves the bead (a9).  FORCES: writes the force instead.
template <bool COMP, bool FORCES>
__global__ void __launch_bounds__(256) k_pair_gather_update(SysDev S, PairDev P, int cur, unsigned long long step) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= S.n_inst) return;
  const int t = g / S.N, i = g - t * S.N;
  float fx = 0.f, fy = 0.f, fz = 0.f;
  if (P.atomics) {
    float4 *a = (float4 *)(P.Facc + (size_t)g * 4);
    const float4 v = *a;
    fx = v.x; fy = v.y; fz = v.z;
    *a = make_float4(0.f, 0.f, 0.f, 0.f);               // ready for the next step
  } else {
    const float4 *F = P.F + (size_t)t * P.n_place;
    for (int b = 0; b < S.cap_b; ++b)
      if (__ldg(&S.bond_tab[(size_t)i * S.cap_b + b]).x >= 0) { const float4 v = F[i * S.cap_b + b]; fx += v.x; fy += v.y; fz += v.z; }
    const int base_n = S.N * S.cap_b;
    for (int q = __ldg(&S.nat_ptr[i]); q < __ldg(&S.nat_ptr[i + 1]); ++q) { const float4 v = F[base_n + q]; fx += v.x; fy += v.y; fz += v.z; }
    const int base_r = base_n + __ldg(&S.nat_ptr[S.N]) + i * S.cap_nb;
    const int cnt = min(S.nb_cnt[g], S.cap_nb);
    for (int p = 0; p < cnt; ++p) { const float4 v = F[base_r + p]; fx += v.x; fy += v.y; fz += v.z; }   // lines 4-7
  }
  const float4 ri = S.pos[cur][g];
  const uint32_t tag = __float_as_uint(ri.w);
  int flag = 0;
  external_force(S, i, ri, tag, step, fx, fy, fz, flag);
  if (FORCES) S.force[g] = make_float4(fx, fy, fz, 0.f);
  else S.pos[cur ^ 1][g] = langevin_update<COMP>(S, ri, tag, t, step, fx, fy, fz, COMP ? S.carry + g : nullptr, flag, g);
  if (flag) atomicOr(S.flags, flag);
}

}  // namespace sop

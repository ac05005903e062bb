// sop.cu -- host side of the C ABI in include/sop.h: validation, static tables, workspace carving, launch
// schedule (list invariant), getters.  All arithmetic of the hot path is in the kernels (sop_kernels.cuh).
#include "../../include/sop.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

#include "sop_kernels.cuh"
#include "sop_persistent.cuh"
#include "sop_resident.cuh"
#include "sop_resident2.cuh"
#include "sop_pairs.cuh"

using namespace sop;

namespace {

thread_local std::string g_last_error;

struct Plan {                     // everything that depends only on (topology, native coords, params, n_traj)
  int N = 0, T = 0;
  std::vector<int> perm, iperm;   // perm[internal] = caller index; iperm[caller] = internal
  int cap_b = 1, cap_nb = 0, cap_pl = 0;
  bool static_l1 = false, comp = false, reorder = false;
  int lanes = 1, block = 256, mode = 1;
  int max_cells = 1;
  size_t n_nat_entries = 0, n_excl = 0;
  int energy_blocks = 1;
  // workspace offsets
  size_t off_pos0, off_pos1, off_carry, off_force, off_bond, off_natptr, off_nattab, off_nateps, off_exclptr,
      off_exclidx, off_adotn, off_plcnt, off_plidx, off_nbcnt, off_nbidx, off_bbox, off_grid, off_cellof,
      off_cellcnt, off_cellstart, off_cellbead, off_cellpos, off_taus, off_flags, off_epart, off_eout, off_bar, off_series, off_kTt, off_ampt, off_rexacc, off_spair, off_spar, off_lpair, off_nlpair, off_F, off_Facc, total;
  int cap_pairs = 0, n_place = 0;
  // mode 3 (SM-resident kernel): chunking, launch shape, shared-memory carve-up, workspace
  bool res_ok = false;
  std::string res_why;
  int res_lanes = 1, res_block = 1024, res_nat_rows = 0;
  ResDev R;
  size_t off_nhalo, off_hgid, off_plloc, off_natloc, off_bondloc, off_xch, off_xchf, off_nbglob, off_slice;
  // mode 3, several chunks per trajectory: the second resident kernel (sop_resident2.cuh) when its plan fits
  bool res2_ok = false;
  int res2_block = 0;
  Res2Dev R2;
  size_t off_plarr, off_plg;
};

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

int fail(int code, const std::string &msg, sop_handle *h = nullptr);

#define CUDA_OK(call)                                                                                   \
  do {                                                                                                  \
    cudaError_t e_ = (call);                                                                            \
    if (e_ != cudaSuccess)                                                                              \
      return fail(SOP_E_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_), h);                   \
  } while (0)

}  // namespace

struct sop_handle {
  Plan plan;
  SysDev S;
  sop_params prm;
  cudaStream_t stream = nullptr;
  int cur = 0;                    // index of the current time layer
  int64_t step = 0, l1_built_at = 0, l2_built_at = 0;
  uint64_t launches = 0;
  char *ws = nullptr;
  std::string last_error;
  int coop_blocks = 0;            // persistent kernel: grid size (co-resident)
  int coop_block_size = 0;
  int num_sms = 0;
  unsigned *S_bar = nullptr;      // grid-barrier counter of the persistent kernel
 ResDev R;                       // mode 3
  Res2Dev R2;
  const void *res2_fn = nullptr;
  PairDev P;                      // mode 4
  int64_t obs_stride = 0, obs_count = 0;   // observables recorded every obs_stride steps into a device ring of obs_cap samples
  int obs_cap = 0;
  std::vector<int64_t> obs_steps;           // [obs_cap] step of the sample in every ring slot
  int obs_a = 0, obs_b = 0;       // internal indices of the two ends of the end-to-end distance
  const void *res_fn = nullptr;
  uint32_t res_launch_id = 0;
  int res_resident_ctas = 148;
  int last_slice_len = 0;              // steps per time slice of the most recent sliced mode-3 launch (0: none so far)
  std::vector<uint32_t> tag;      // [N] host copy of the coordinate tags (internal order)
  float4 *stage = nullptr;        // pinned host staging buffer [T][N] for coordinate transfers
  // optional kernel timing (sop_set_profiling): event pairs around groups of launches of one kind
  struct Span { cudaEvent_t a, b; int kind; int64_t steps; };
  bool profiling = false;
  std::vector<Span> spans;
  int open_kind = -1;
  double prof_ms[3] = {0, 0, 0};
  int64_t prof_n[3] = {0, 0, 0}, prof_steps = 0;
};

namespace {

int fail(int code, const std::string &msg, sop_handle *h) {
  g_last_error = msg;
  if (h) h->last_error = msg;
  return code;
}

// ---- host-side neighbour statistics of the native structure (sizing only; not on the hot path) ----------
// fn(i, j) for every ordered pair i != j closer than R (cell list over the bounding box)
template <class F>
void visit_neighbors(const std::vector<double> &x, int N, double R, F fn) {
  double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
  for (int i = 0; i < N; ++i)
    for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], x[3 * i + a]); hi[a] = std::max(hi[a], x[3 * i + a]); }
  int n[3];
  for (int a = 0; a < 3; ++a) n[a] = std::max(1, std::min(1024, (int)std::floor((hi[a] - lo[a]) / R) + 1));
  double edge[3];
  for (int a = 0; a < 3; ++a) edge[a] = std::max(R, (hi[a] - lo[a]) / n[a] * (1 + 1e-9) + 1e-9);
  auto cell = [&](int i, int a) { return std::min(n[a] - 1, std::max(0, (int)std::floor((x[3 * i + a] - lo[a]) / edge[a]))); };
  size_t ncell = (size_t)n[0] * n[1] * n[2];
  std::vector<int> start(ncell + 1, 0), of(N), order(N);
  for (int i = 0; i < N; ++i) { of[i] = (cell(i, 2) * n[1] + cell(i, 1)) * n[0] + cell(i, 0); start[of[i] + 1]++; }
  for (size_t c = 0; c < ncell; ++c) start[c + 1] += start[c];
  std::vector<int> fill(start.begin(), start.end() - 1);
  for (int i = 0; i < N; ++i) order[fill[of[i]]++] = i;
  const double R2 = R * R;
  for (int i = 0; i < N; ++i) {
    int cx = cell(i, 0), cy = cell(i, 1), cz = cell(i, 2);
    for (int z = std::max(0, cz - 1); z <= std::min(n[2] - 1, cz + 1); ++z)
      for (int y = std::max(0, cy - 1); y <= std::min(n[1] - 1, cy + 1); ++y)
        for (int xx = std::max(0, cx - 1); xx <= std::min(n[0] - 1, cx + 1); ++xx) {
          int c = (z * n[1] + y) * n[0] + xx;
          for (int q = start[c]; q < start[c + 1]; ++q) {
            int j = order[q];
            if (j == i) continue;
            double dx = x[3 * i] - x[3 * j], dy = x[3 * i + 1] - x[3 * j + 1], dz = x[3 * i + 2] - x[3 * j + 2];
            if (dx * dx + dy * dy + dz * dz < R2) fn(i, j);
          }
        }
  }
}

int max_neighbors(const std::vector<double> &x, int N, double R) {
  if (!std::isfinite(R)) return N - 1;
  std::vector<int> cnt(N, 0);
  visit_neighbors(x, N, R, [&](int i, int) { cnt[i]++; });
  return *std::max_element(cnt.begin(), cnt.end());
}

int device_sm_count() {
  int dev = 0, n = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) {
    cudaGetLastError();
    return 148;                       // B200; only reached without a device (sizing queries)
  }
  return n;
}

uint32_t part1by2(uint32_t v) {   // spread the low 10 bits of v
  v &= 0x3FF;
  v = (v | (v << 16)) & 0x030000FF;
  v = (v | (v << 8)) & 0x0300F00F;
  v = (v | (v << 4)) & 0x030C30C3;
  v = (v | (v << 2)) & 0x09249249;
  return v;
}

// ---- mode 3, several chunks: plan of the second resident kernel (sop_resident2.cuh).  Called at the end of plan_resident
// (chunking and halo capacity are shared).  Leaves res2_ok = false when the chunk state does not fit; the first kernel
// then runs the multi-chunk case too.
void plan_resident2(const sop_topology *tp, const sop_params *p, const std::vector<double> &x, Plan &pl) {
  const ResDev &R = pl.R;
  Res2Dev &Q = pl.R2;
  memset(&Q, 0, sizeof(Q));
  pl.res2_ok = false;
  if (R.C <= 1 || pl.static_l1 || p->resident_variant != 2) return;     // (auto = the first design: measured faster)
  const int N = pl.N, chunk = R.chunk;
  const int max_groups = (32 - 4) * 8;                          // groups of four lanes, at least four service warps
  const int P = (chunk + max_groups - 1) / max_groups;
  if (P > 2) return;                                             // (one or two beads per group: the filter keeps <= R2_MAXR rows per quarter-warp)
  Q.P = P;
  Q.n_cwarps = (chunk + 8 * P - 1) / (8 * P);
  Q.n_swarps = Q.n_cwarps <= 26 ? 6 : 32 - Q.n_cwarps;           // service warps: noise, exchange, bonds
  pl.res2_block = 32 * (Q.n_cwarps + Q.n_swarps);
  if ((chunk + pl.res2_block / 8 - 1) / (pl.res2_block / 8) > R2_MAXR) return;
  if (chunk > pl.res2_block || R.halo_cap > 32760 || pl.cap_pl > 496 || pl.cap_nb > 240 || pl.cap_b > 8) return;   // (15-bit partner codes, 64-bit survivor masks)
  Q.own_pad = (chunk + 7) / 8 * 8; Q.halo_pad = (R.halo_cap + 7) / 8 * 8;
  Q.own_stride = Q.own_pad + 8; Q.halo_stride = Q.halo_pad + 8;
  Q.cap_arr = (pl.cap_pl + 7) / 8 * 8 + 16;
  // force rows of a chunk: natives + partners within 1.05 R_nb of the native structure + the padding of two segments
  std::vector<long long> per(R.C, 0);
  {
    std::vector<int> nnb(N, 0);
    visit_neighbors(x, N, (double)p->R_nb * 1.05, [&](int i, int) { nnb[i]++; });
    std::vector<int> nnat(N, 0);
    for (int c2 = 0; c2 < tp->n_native; ++c2) {          // natives the neighbour count above does not contain
      const int i = tp->native[2 * c2], j = tp->native[2 * c2 + 1];
      const double dx = x[3 * i] - x[3 * j], dy = x[3 * i + 1] - x[3 * j + 1], dz = x[3 * i + 2] - x[3 * j + 2];
      if (dx * dx + dy * dy + dz * dz >= (double)p->R_nb * 1.05 * (double)p->R_nb * 1.05) { nnat[i]++; nnat[j]++; }
    }
    for (int i = 0; i < N; ++i) per[pl.iperm[i] / chunk] += nnb[i] + nnat[i] + 8;
  }
  long long want = (long long)(*std::max_element(per.begin(), per.end()) * 1.15) + 64;
  want = std::max<long long>(2048, std::min<long long>((want + 7) / 8 * 8, 65528LL * 4));      // (>= 8 KB: scratch of the prologue)
  {   // the prologue of a launch that continues on an old L1 keeps one membership bitmap per quarter-warp in the row region
    const long long bm_bytes = (long long)(pl.res2_block / 8) * ((Q.own_stride + Q.halo_stride + 31) / 32) * 4;
    want = std::max<long long>(want, (bm_bytes / 8 + 8) / 8 * 8);
  }
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = (o + bytes + 127) / 128 * 128; return (int)at; };
  auto carve = [&](long long rows_cap) {
    o = 0;
    Q.rows_cap = (int)rows_cap;
    Q.off_own = take(2 * (size_t)Q.own_stride * 16);
    Q.off_halo = take(2 * (size_t)Q.halo_stride * 16);
    Q.off_rows = take((size_t)rows_cap * 8);
    Q.off_eps = take(tp->native_eps ? (size_t)rows_cap * 4 : 0);
    Q.off_ext = take(32);
    Q.off_g = take(2 * (size_t)chunk * 16);
    Q.off_carry = take(pl.comp ? (size_t)chunk * 16 : 0);
    Q.off_tag = take((size_t)chunk * 4);
    Q.off_rowofs = take(((size_t)chunk + 1) * 2);
    Q.off_rowg = take((size_t)chunk * 2);
    Q.off_nat = take((size_t)R.nat_cap * 8);
    Q.off_nateps = take(tp->native_eps ? (size_t)R.nat_cap * 4 : 0);
    Q.off_natq = take(((size_t)chunk + 1) * 4);
    Q.off_natc = take((size_t)chunk * 2);
    Q.off_bond = take((size_t)chunk * pl.cap_b * 8);
    Q.off_cnt = take((size_t)chunk * 2);
    Q.off_active = take((size_t)R.halo_cap * 2);
    Q.off_bm = take((size_t)(R.halo_cap / 32 + 1) * 4);
    Q.off_sbm = take((size_t)(R.halo_cap / 32 + 1) * 4);
    Q.off_misc = take(2048);
    Q.off_order = take((size_t)chunk * 4);
    Q.off_taus = take(p->rng == 1 ? (size_t)chunk * 16 : 0);
    Q.smem_bytes = (int)o;
  };
  {
    const double e12 = 12.0 * (double)p->eps_native;
    const double a_ref = e12 > 0.0 ? e12 : 1.0;
    Q.a_ref = (float)a_ref;
    Q.par_rep = (float)(-std::cbrt(6.0 * (double)p->eps_rep * std::pow((double)p->sigma, 6.0) / (double)Q.a_ref));
  }
  const int per_entry = tp->native_eps ? 12 : 8;
  carve(want);
  if (o > 232448) {                       // the rows get what is left, if that is still most of what they may need
    const long long fixed = (long long)o - want * per_entry;
    const long long left = (232448 - fixed - 512) / per_entry / 8 * 8;
    if (left * 10 < want * 8 || left < 2048 || left * 8 < (long long)(pl.res2_block / 8) * ((Q.own_stride + Q.halo_stride + 31) / 32) * 4) return;
    carve(left);
    if (o > 232448) return;
  }
  pl.res2_ok = true;
  if (getenv("SOP_DEBUG_PLAN"))
    fprintf(stderr, "[sop plan] mode 3 (second kernel): P=%d compute warps=%d block=%d rows_cap=%d cap_arr=%d smem=%d B\n",
            Q.P, Q.n_cwarps, pl.res2_block, Q.rows_cap, Q.cap_arr, Q.smem_bytes);
}

// ---- mode 3 plan: chunks, lanes, halo capacity from the native structure, shared-memory carve-up ------------
void plan_resident(const sop_topology *tp, const sop_params *p, const std::vector<double> &x, Plan &pl) {
  const int N = pl.N, T = pl.T;
  ResDev &R = pl.R;
  memset(&R, 0, sizeof(R));
  pl.res_ok = false;
  const int sms = device_sm_count();
  int C = 1;
  if (!pl.static_l1) {
    const int maxC = std::max(1, sms / T);
    C = std::max(1, std::min(maxC, N / 192));
  }
  int chunk = (N + C - 1) / C;
  if (p->chunk_beads > 0 && !pl.static_l1) chunk = std::min(N, (int)p->chunk_beads);
  C = (N + chunk - 1) / chunk;
  R.C = C; R.chunk = chunk;
  R.implicit_l1 = pl.static_l1 ? 1 : 0;
  R.nat_entries = (int)pl.n_nat_entries;
  int G = p->lanes_per_bead;
  if (G == 0) { G = 32; while (G > 1 && (long long)chunk * G > 1024) G >>= 1; }
  pl.res_lanes = G;
  int block = p->block_size > 0 ? p->block_size : (int)std::min<long long>(1024, ((long long)chunk * G + 31) / 32 * 32);
  pl.res_block = std::max(32, std::min(1024, block));
  // halo capacity: beads of other chunks within 1.1 R_pl of a chunk's beads at the native structure, + 25 % + 64
  int halo_cap = 32, pl_want = 0;
  if (C > 1) {
    std::vector<int> cnt(C, 0);
    std::vector<long long> l1_entries(C, 0);
    // chunk of a bead = internal index / chunk; distinct (chunk, outside bead) keys
    std::vector<uint64_t> keys;
    keys.reserve((size_t)N * 64);
    visit_neighbors(x, N, (double)p->R_pl * 1.1, [&](int i, int j) {
      const int ci = pl.iperm[i] / chunk, jj = pl.iperm[j];
      l1_entries[ci]++;
      if (jj / chunk != ci) keys.push_back(((uint64_t)ci << 32) | (uint32_t)jj);
    });
    pl_want = (int)std::min<long long>(1 << 20, *std::max_element(l1_entries.begin(), l1_entries.end()) + chunk + 64);
    std::sort(keys.begin(), keys.end());
    keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
    for (uint64_t k : keys) cnt[(int)(k >> 32)]++;
    const int worst = *std::max_element(cnt.begin(), cnt.end());
    halo_cap = ((int)(worst * 1.15) + 32 + 31) / 32 * 32;
  }
  R.halo_cap = halo_cap;
  const long long slots = (long long)chunk + halo_cap;
  if (slots > 65535) { pl.res_why = "a chunk and its halo exceed 65535 slots"; return; }
  // native entries per chunk (internal order)
  {
    std::vector<int> per(C, 0);
    for (int c2 = 0; c2 < tp->n_native; ++c2) {
      per[pl.iperm[tp->native[2 * c2]] / chunk]++;
      per[pl.iperm[tp->native[2 * c2 + 1]] / chunk]++;
    }
    R.nat_cap = std::max(1, *std::max_element(per.begin(), per.end()));
  }
  R.nb_si = pl.cap_nb + 4;                       // rows padded to a multiple of four slots, 8-byte aligned
  if (R.nb_si % 4 != 0) { pl.res_why = "internal: the L2 row stride must be a multiple of four slots"; return; }   // (cap_nb is)
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = (o + bytes + 15) / 16 * 16; return (int)at; };
  auto carve = [&](bool nat_smem, int pl_cap, bool stream = false) {
    o = 0;
    R.nat_smem = nat_smem ? 1 : 0;
    R.pl_cap = pl_cap;
    R.stream = stream ? 1 : 0;
    R.off_pos = take((stream ? 1 : 2) * (size_t)(slots + 1) * 16);
    R.off_g = take(G > 1 ? 2 * (size_t)chunk * 16 : 0);
    R.off_carry = take(pl.comp ? (size_t)chunk * 16 : 0);
    R.off_tag = take((size_t)chunk * 4);
    R.off_force = take((size_t)chunk * 16);
    R.off_nb = take(stream ? 0 : (size_t)chunk * R.nb_si * 2);
    R.off_cnt = take((size_t)chunk * 2);
    R.off_plcnt = take((size_t)chunk * 2);
    R.off_plofs = take(stream ? 0 : ((size_t)chunk + 1) * 4);
    R.off_pl = take((size_t)pl_cap * 2);
    R.off_natq = take(((size_t)chunk + 1) * 4);
    R.off_nat = take(nat_smem ? (size_t)R.nat_cap * 8 : 0);
    R.off_bond = take(stream ? 0 : (size_t)chunk * pl.cap_b * 8);
    R.off_active = take(stream ? 0 : (size_t)halo_cap * 2);
    R.off_bm = take((size_t)(halo_cap / 32 + 1) * 4);
    R.off_sbm = take((size_t)(halo_cap / 32 + 1) * 4);
    R.off_misc = take(64);
    R.off_order = take(stream ? 0 : (size_t)chunk * 2);
    R.off_hist = take(64 * 4);
    R.smem_bytes = (int)o;
  };
  if (getenv("SOP_TEST_NO_PL_SMEM") && !pl.static_l1) pl_want = 0;      // test hook: exercise the L1-rows-in-global path
  // implicit L1: the same region holds the in-kernel cell grid (2 x (cells + 1) ints + 2 x chunk shorts)
  if (pl.static_l1) pl_want = (2 * (RES_GRID_CELLS + 1) * 4 + 4 * chunk + 64) / 2;
  // what is read every step goes to shared memory first (natives), then the L1 rows (read every nb_interval steps)
  const bool nat_ok = getenv("SOP_TEST_NO_NAT_SMEM") == nullptr;          // test hook: natives stay in global memory
  carve(nat_ok, pl_want);
  if (o > 232448 && pl.static_l1) carve(false, pl_want);
  if (o > 232448 && !pl.static_l1) {
    // the L1 rows get what is left (the kernel reads them from global memory if a chunk's rows do not fit at run time)
    carve(nat_ok, 0);
    const long long left = (232448 - (long long)o) / 2 - 16;
    if (left > 4 * chunk) carve(nat_ok, (int)std::min<long long>(pl_want, left));
  }
  if (o > 232448 && !pl.static_l1) carve(false, 0);
  // still too large (chunks of a thousand beads and more): keep only the coordinates resident and stream the lists
  if (o > 232448 && !pl.static_l1 && C > 1 && G <= 2) carve(false, 0, true);
  if (getenv("SOP_TEST_STREAM") && !pl.static_l1 && C > 1 && G <= 2) carve(false, 0, true);   // test hook: the streamed variant on small inputs
  if (o > 232448) {
    if (getenv("SOP_DEBUG_PLAN")) fprintf(stderr, "[sop plan] mode 3 does not fit: C=%d chunk=%d lanes=%d halo_cap=%d smem=%zu B\n", C, chunk, G, halo_cap, o);
    pl.res_why = "chunk state does not fit the 227 KB of shared memory of an SM"; return;
  }
  R.nat_tpad = 0;
  pl.res_nat_rows = 0;
  if (C == 1 && !R.nat_smem && G == 1) {          // natives stay in global memory: read them coalesced
    std::vector<int> deg(N, 0);
    for (int c2 = 0; c2 < tp->n_native; ++c2) { deg[tp->native[2 * c2]]++; deg[tp->native[2 * c2 + 1]]++; }
    pl.res_nat_rows = std::max(1, *std::max_element(deg.begin(), deg.end()));
    R.nat_tpad = (N + 31) / 32 * 32;
  }
  if ((size_t)((N + 31) / 32) * 8 > 200000) { pl.res_why = "n_beads too large for the localise bitmap"; return; }
  plan_resident2(tp, p, x, pl);
  if (getenv("SOP_DEBUG_PLAN"))
    fprintf(stderr, "[sop plan] mode 3: C=%d chunk=%d lanes=%d block=%d halo_cap=%d cap_nb=%d cap_pl=%d nat_smem=%d pl_cap=%d stream=%d smem=%d B\n",
            R.C, R.chunk, pl.res_lanes, pl.res_block, R.halo_cap, pl.cap_nb, pl.cap_pl, R.nat_smem, R.pl_cap, R.stream, R.smem_bytes);
  pl.res_ok = true;
}

int make_plan(const sop_topology *tp, const float *xyz, const sop_params *p, int32_t T, Plan &pl) {
  if (!tp || !xyz || !p || T < 1) return fail(SOP_E_ARG, "null argument or n_traj < 1");
  const int N = tp->n_beads;
  if (N < 1 || N > (int)TAG_ID_MASK) return fail(SOP_E_ARG, "n_beads out of range");
  if ((long long)N * T > 0x7FFFFFF0LL) return fail(SOP_E_ARG, "n_beads * n_traj too large");
  if (p->nb_interval < 1 || p->pl_interval < 1 || p->pl_interval % p->nb_interval != 0)
    return fail(SOP_E_ARG, "pl_interval must be a positive multiple of nb_interval");
  if (!(p->R_nb > 0) || !(p->R_pl >= p->R_nb) || !(p->R0 > 0) || !(p->dt_over_zeta >= 0) || !(p->kT >= 0))
    return fail(SOP_E_ARG, "bad cutoffs / R0 / dt_over_zeta / kT");
  for (int q = 0; q < 3 * N; ++q)
    if (!std::isfinite(xyz[q])) return fail(SOP_E_ARG, "non-finite native coordinate");
  pl.N = N; pl.T = T;
  pl.static_l1 = std::isinf(p->R_pl);

  std::vector<double> x(3 * (size_t)N);
  double maxabs = 0;
  for (size_t q = 0; q < 3 * (size_t)N; ++q) { x[q] = xyz[q]; maxabs = std::max(maxabs, std::fabs(x[q])); }
  pl.comp = p->compensated == 1 || (p->compensated == 0 && maxabs > 512.0);

  // internal bead order: Morton order of 8 A cells of the native structure (gather locality), ties by index
  pl.reorder = p->reorder == 1 || (p->reorder == 0 && (p->mode == 0 || p->mode == 3));
  pl.perm.resize(N); pl.iperm.resize(N);
  for (int i = 0; i < N; ++i) pl.perm[i] = i;
  if (pl.reorder) {
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int i = 0; i < N; ++i)
      for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], x[3 * i + a]); hi[a] = std::max(hi[a], x[3 * i + a]); }
    double ext = std::max({hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2], 1.0});
    double cellw = std::max(8.0, ext / 1023.0);
    std::vector<uint32_t> key(N);
    for (int i = 0; i < N; ++i) {
      uint32_t c[3];
      for (int a = 0; a < 3; ++a) c[a] = (uint32_t)std::min(1023.0, std::floor((x[3 * i + a] - lo[a]) / cellw));
      key[i] = part1by2(c[0]) | (part1by2(c[1]) << 1) | (part1by2(c[2]) << 2);
    }
    std::stable_sort(pl.perm.begin(), pl.perm.end(), [&](int a, int b) { return key[a] < key[b]; });
  }
  for (int i = 0; i < N; ++i) pl.iperm[pl.perm[i]] = i;

  // row capacities (the paper's M)
  std::vector<int> deg(N, 0);
  for (int b = 0; b < tp->n_bonds; ++b) {
    int i = tp->bonds[2 * b], j = tp->bonds[2 * b + 1];
    if (i < 0 || j >= N || i >= j) return fail(SOP_E_ARG, "bond out of range or not i<j");
    deg[i]++; deg[j]++;
  }
  pl.cap_b = std::max(1, *std::max_element(deg.begin(), deg.end()));
  for (int c = 0; c < tp->n_native; ++c) {
    int i = tp->native[2 * c], j = tp->native[2 * c + 1];
    if (i < 0 || j >= N || i >= j) return fail(SOP_E_ARG, "native pair out of range or not i<j");
  }
  pl.n_nat_entries = 2 * (size_t)tp->n_native;
  pl.n_excl = 2 * ((size_t)tp->n_native + (size_t)tp->n_bonds);
  auto cap_of = [&](int requested, double R) {
    if (requested > 0) return (requested + 3) / 4 * 4;
    int m = max_neighbors(x, N, R);
    if (!std::isfinite(R)) return (std::max(m, 1) + 3) / 4 * 4;
    return ((int)(m * 1.15) + 8 + 3) / 4 * 4;
  };
  pl.cap_nb = cap_of(p->cap_nb, p->R_nb);
  pl.cap_pl = cap_of(p->cap_pl, p->R_pl);
  if (pl.static_l1 && (size_t)N * pl.cap_pl > (size_t)1 << 30)
    return fail(SOP_E_ARG, "R_pl = +inf needs an N x N pair list: N too large, give a finite R_pl");

  // cell grid capacity: the native bounding box, with room for the structure to grow 4x per axis sum
  if (!pl.static_l1) {
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int i = 0; i < N; ++i)
      for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], x[3 * i + a]); hi[a] = std::max(hi[a], x[3 * i + a]); }
    double edge = (double)p->R_pl * 1.001, tot = 1;
    for (int a = 0; a < 3; ++a) tot *= std::floor((hi[a] - lo[a]) / edge) + 1;
    pl.max_cells = (int)std::min(4.0e6, std::max(64.0, tot * 4.0));
  }

  // launch shape
  const long long inst = (long long)N * T;
  int lanes = p->lanes_per_bead;
  if (lanes == 0) {
    lanes = 32;
    while (lanes > 1 && inst * lanes > 600000LL) lanes >>= 1;    // measured on cfg 4: fewer lanes once the chip is full
  }
  if (lanes != 1 && lanes != 2 && lanes != 4 && lanes != 8 && lanes != 16 && lanes != 32)
    return fail(SOP_E_ARG, "lanes_per_bead must be 0 or a power of two <= 32");
  pl.lanes = lanes;
  pl.block = p->block_size > 0 ? p->block_size : 256;
  if (pl.block % 32 || pl.block > 1024) return fail(SOP_E_ARG, "block_size must be a multiple of 32, <= 1024");
  if (p->mode < 0 || p->mode > 4) return fail(SOP_E_ARG, "mode must be 0 ... 4");
  if (p->mode == 4 && p->rng != 0) return fail(SOP_E_ARG, "mode 4 (pair based) runs with rng = 0");
  if (p->integrator < 0 || p->integrator > 2) return fail(SOP_E_ARG, "integrator must be 0, 1 or 2");
  if (p->integrator == 2 && (p->rng != 0 || (p->mode > 1)))
    return fail(SOP_E_ARG, "integrator = 2 (second order, Eq. (5)) runs in mode 1 with rng = 0");
  if (p->kT_per_traj)
    for (int t = 0; t < T; ++t)
      if (!(p->kT_per_traj[t] >= 0)) return fail(SOP_E_ARG, "bad kT_per_traj");
  if (p->obs_stride < 0 || p->obs_capacity < 0 || (p->obs_stride > 0 && p->obs_capacity < 1))
    return fail(SOP_E_ARG, "obs_stride needs obs_capacity >= 1");
  if (p->resident_variant < 0 || p->resident_variant > 2) return fail(SOP_E_ARG, "resident_variant must be 0, 1 or 2");
  if (p->rng != 0 && p->rng != 1) return fail(SOP_E_ARG, "rng must be 0 (Philox) or 1 (Hybrid Taus)");
  pl.mode = p->integrator == 2 ? 1 : p->mode;
  if (pl.mode == 0 || pl.mode == 3) {
    plan_resident(tp, p, x, pl);
    if (pl.mode == 3 && !pl.res_ok) return fail(SOP_E_ARG, "mode 3 is not possible here: " + pl.res_why);
    // fallback: the streaming kernels; one launch per step once the chip is full (measured on cfg 4), else persistent
    // (auto does not pick the streamed variant of mode 3: on the 250,000-bead lattice it measured 76 us per step against 72 us
    //  of the per-step launches -- DESIGN.md section 6; it runs when mode 3 is asked for)
    const bool take3 = pl.res_ok && !(p->mode == 0 && pl.R.stream);
    pl.mode = take3 ? 3 : (inst > 100000 ? 1 : 2);
  }
  pl.energy_blocks = (int)std::min<long long>(296, ((long long)N * 8 + 255) / 256);

  // workspace
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
  const size_t I = (size_t)inst;
  pl.off_pos0 = take(I * 16); pl.off_pos1 = take(I * 16);
  pl.off_carry = take(pl.comp ? I * 16 : 0);
  pl.off_force = take(I * 16);
  pl.off_bond = take((size_t)N * pl.cap_b * 8);
  pl.off_natptr = take(((size_t)N + 1) * 4);
  pl.off_nattab = take(pl.n_nat_entries * 8);
  pl.off_nateps = take(tp->native_eps ? pl.n_nat_entries * 4 : 0);
  pl.off_exclptr = take(((size_t)N + 1) * 4);
  pl.off_exclidx = take(pl.n_excl * 4);
  pl.off_adotn = take(p->n_pulled > 0 ? (size_t)N * 4 : 0);
  const size_t rows1 = pl.static_l1 ? (size_t)N : I;
  pl.off_plcnt = take(rows1 * 4); pl.off_plidx = take(rows1 * pl.cap_pl * 4);
  pl.off_nbcnt = take(I * 4); pl.off_nbidx = take(I * pl.cap_nb * 4);
  pl.off_bbox = take((size_t)T * 6 * 4); pl.off_grid = take((size_t)T * sizeof(GridDev));
  pl.off_cellof = take(pl.static_l1 ? 0 : I * 4);
  pl.off_cellcnt = take(pl.static_l1 ? 0 : (size_t)T * pl.max_cells * 4);
  pl.off_cellstart = take(pl.static_l1 ? 0 : (size_t)T * ((size_t)pl.max_cells + 1) * 4);
  pl.off_cellbead = take(pl.static_l1 ? 0 : I * 4);
  pl.off_cellpos = take(pl.static_l1 ? 0 : I * 16);
  pl.off_taus = take(p->rng == 1 ? I * 16 : 0);
  pl.off_flags = take(64);
  pl.off_epart = take((size_t)T * pl.energy_blocks * 5 * 8);
  pl.off_eout = take((size_t)T * 6 * 8);
  pl.off_bar = take(256);
  pl.off_series = take(p->obs_capacity > 0 ? (size_t)p->obs_capacity * T * 10 * 8 : 0);
  pl.off_kTt = take(p->kT_per_traj ? (size_t)T * 4 : 0);
  pl.off_ampt = take(p->kT_per_traj ? (size_t)T * 4 : 0);
  pl.off_rexacc = take(p->kT_per_traj ? (size_t)T * 4 : 0);
  if (pl.mode == 4) {                 // the pair-based scheme (sop_pairs.cuh): pair vectors and the array of force places
    const size_t n_static = (size_t)tp->n_bonds + (size_t)tp->n_native;
    pl.cap_pairs = (int)std::min<size_t>(0x7FFFFFF0, ((size_t)N * pl.cap_nb + 1) / 2);
    pl.n_place = (int)((size_t)N * pl.cap_b + pl.n_nat_entries + (size_t)N * pl.cap_nb);
    pl.off_spair = take(n_static * 16); pl.off_spar = take(n_static * 8);
    pl.off_lpair = take((size_t)T * pl.cap_pairs * 16); pl.off_nlpair = take((size_t)T * 4);
    pl.off_F = take(p->pair_atomics ? 0 : (size_t)T * pl.n_place * 16);
    pl.off_Facc = take(p->pair_atomics ? I * 16 : 0);
  }
  if (pl.mode == 3) {
    const ResDev &R = pl.R;
    const bool multi = R.C > 1;
    pl.off_nhalo = take((size_t)T * R.C * 4);
    pl.off_hgid = take((size_t)T * R.C * R.halo_cap * 4);
    pl.off_plloc = take(R.implicit_l1 ? 0 : I * pl.cap_pl * 2);
    pl.off_natloc = take(multi ? (size_t)T * pl.n_nat_entries * 8 : (size_t)pl.res_nat_rows * R.nat_tpad * 8);
    pl.off_bondloc = take(multi ? I * pl.cap_b * 8 : 0);
    pl.off_xch = take(multi ? 2 * I * 32 : 0);
    pl.off_xchf = take(multi ? 2 * I * 32 : 0);
    pl.off_nbglob = take(R.stream ? I * R.nb_si * 2 : 0);
    pl.off_slice = take(R.C == 1 ? ((size_t)T + 1) * 4 : 0);        // ticket counter + done[T] of a sliced launch
    pl.off_plarr = take(pl.res2_ok ? I * pl.R2.cap_arr * 2 : 0);
    pl.off_plg = take(pl.res2_ok ? I * 2 : 0);
  }
  pl.total = o;
  return SOP_OK;
}

enum { SPAN_STEP = 0, SPAN_FILTER = 1, SPAN_L1 = 2 };

void span_close(sop_handle *h) {
  if (h->open_kind < 0) return;
  cudaEventRecord(h->spans.back().b, h->stream);
  h->open_kind = -1;
}
// open (or extend) a timed span of `kind`; consecutive launches of the same kind share one event pair
void span_begin(sop_handle *h, int kind, int64_t steps) {
  if (!h->profiling) return;
  if (h->open_kind == kind) { h->spans.back().steps += steps; return; }
  span_close(h);
  sop_handle::Span sp;
  cudaEventCreate(&sp.a); cudaEventCreate(&sp.b);
  sp.kind = kind; sp.steps = steps;
  cudaEventRecord(sp.a, h->stream);
  h->spans.push_back(sp);
  h->open_kind = kind;
}

template <int G>
void launch_step_g(sop_handle *h, bool forces) {
  const SysDev &S = h->S;
  const long long threads = (long long)S.n_inst * G;
  const int block = h->plan.block;
  const unsigned grid = (unsigned)((threads + block - 1) / block);
  const unsigned long long step = (unsigned long long)h->step;
  if (forces) k_step<G, false, true><<<grid, block, 0, h->stream>>>(S, h->cur, step);
  else if (block <= 256) {
    if (h->plan.comp) k_step<G, true, false, true><<<grid, block, 0, h->stream>>>(S, h->cur, step);
    else k_step<G, false, false, true><<<grid, block, 0, h->stream>>>(S, h->cur, step);
  }
  else if (h->plan.comp) k_step<G, true, false><<<grid, block, 0, h->stream>>>(S, h->cur, step);
  else k_step<G, false, false><<<grid, block, 0, h->stream>>>(S, h->cur, step);
  h->launches++;
}

void launch_step(sop_handle *h, bool forces) {
  switch (h->plan.lanes) {
    case 1: launch_step_g<1>(h, forces); break;
    case 2: launch_step_g<2>(h, forces); break;
    case 4: launch_step_g<4>(h, forces); break;
    case 8: launch_step_g<8>(h, forces); break;
    case 16: launch_step_g<16>(h, forces); break;
    default: launch_step_g<32>(h, forces); break;
  }
}

// mode 4: Alg. 4 (thread per pair) + Alg. 5 fused with the update (thread per bead)
void launch_pair_step(sop_handle *h, bool forces) {
  const SysDev &S = h->S;
  const PairDev &P = h->P;
  const unsigned gp = (unsigned)(((long long)P.n_static + P.cap_pairs + 255) / 256);
  k_pair_forces<<<dim3(gp, (unsigned)S.T), 256, 0, h->stream>>>(S, P, h->cur);
  const unsigned gb = (unsigned)((S.n_inst + 255) / 256);
  const unsigned long long step = (unsigned long long)h->step;
  if (forces) k_pair_gather_update<false, true><<<gb, 256, 0, h->stream>>>(S, P, h->cur, step);
  else if (h->plan.comp) k_pair_gather_update<true, false><<<gb, 256, 0, h->stream>>>(S, P, h->cur, step);
  else k_pair_gather_update<false, false><<<gb, 256, 0, h->stream>>>(S, P, h->cur, step);
  h->launches += 2;
}

template <int G>
void launch_step2_g(sop_handle *h, int stage) {
  const SysDev &S = h->S;
  const long long threads = (long long)S.n_inst * G;
  const int block = h->plan.block;
  const unsigned grid = (unsigned)((threads + block - 1) / block);
  if (h->plan.comp) k_step2<G, true><<<grid, block, 0, h->stream>>>(S, h->cur, (unsigned long long)h->step, stage);
  else k_step2<G, false><<<grid, block, 0, h->stream>>>(S, h->cur, (unsigned long long)h->step, stage);
  h->launches++;
}

void launch_step2(sop_handle *h, int stage) {
  switch (h->plan.lanes) {
    case 1: launch_step2_g<1>(h, stage); break;
    case 2: launch_step2_g<2>(h, stage); break;
    case 4: launch_step2_g<4>(h, stage); break;
    case 8: launch_step2_g<8>(h, stage); break;
    case 16: launch_step2_g<16>(h, stage); break;
    default: launch_step2_g<32>(h, stage); break;
  }
}

void launch_filter(sop_handle *h) {
  const SysDev &S = h->S;
  span_begin(h, SPAN_FILTER, 1);
  const long long threads = (long long)S.n_inst * 32;
  k_filter<<<(unsigned)((threads + 255) / 256), 256, 0, h->stream>>>(S, h->cur);
  h->launches++;
  if (h->plan.mode == 4) {            // the vector of L2 pairs follows the neighbor list
    cudaMemsetAsync(h->P.n_lpair, 0, (size_t)S.T * 4, h->stream);
    k_pairs_build<<<(unsigned)((threads + 255) / 256), 256, 0, h->stream>>>(S, h->P);
    h->launches++;
  }
  h->l2_built_at = h->step;
}

int launch_build_l1(sop_handle *h) {
  const SysDev &S = h->S;
  cudaStream_t st = h->stream;
  span_begin(h, SPAN_L1, 1);
  if (S.static_l1) {
    k_build_l1_static<<<(unsigned)(((long long)S.N * 32 + 255) / 256), 256, 0, st>>>(S);
    h->launches++;
  } else {
    k_bbox_init<<<(S.T * 6 + 255) / 256, 256, 0, st>>>(S);
    dim3 gb((unsigned)std::min(64, (S.N + 255) / 256), (unsigned)S.T);
    k_bbox<<<gb, 256, 0, st>>>(S, h->cur);
    k_grid_setup<<<(S.T + 127) / 128, 128, 0, st>>>(S);
    CUDA_OK(cudaMemsetAsync(S.cell_cnt, 0, (size_t)S.T * S.max_cells * 4, st));
    const unsigned gi = (unsigned)((S.n_inst + 255) / 256);
    k_cell_count<<<gi, 256, 0, st>>>(S, h->cur);
    k_cell_scan<<<S.T, 1024, 0, st>>>(S);
    k_cell_fill<<<gi, 256, 0, st>>>(S);
    dim3 gs((unsigned)std::min(1024, (S.max_cells * 32 + 255) / 256), (unsigned)S.T);
    k_cell_sort<<<gs, 256, 0, st>>>(S, h->cur);
    k_build_l1<<<(unsigned)(((long long)S.n_inst * 32 + 255) / 256), 256, 0, st>>>(S, h->cur);
    h->launches += 8;
  }
  h->l1_built_at = h->step;
  return SOP_OK;
}

int check_launch(sop_handle *h, const char *what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(SOP_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e), h);
  return SOP_OK;
}

int read_flags(sop_handle *h) {
  int flags = 0;
  CUDA_OK(cudaMemcpyAsync(&flags, h->S.flags, 4, cudaMemcpyDeviceToHost, h->stream));
  CUDA_OK(cudaStreamSynchronize(h->stream));
  if (!flags) return SOP_OK;
  CUDA_OK(cudaMemsetAsync(h->S.flags, 0, 8, h->stream));          // the flag word and the abort word of the exchange
  if (flags & FLAG_EXCHANGE_TIMEOUT)
    return fail(SOP_E_CUDA, "mode 3: a chunk waited too long for a neighbour's coordinates (exchange time-out); the run is invalid", h);
  if (flags & FLAG_NONFINITE) return fail(SOP_E_NONFINITE, "non-finite coordinate or bead inside the indenter", h);
  if (flags & FLAG_FENE) return fail(SOP_E_FENE, "a bond reached |r - r0| >= R0", h);
  if (flags & FLAG_PL_OVERFLOW) return fail(SOP_E_LIST_OVERFLOW, "pair-list row exceeded cap_pl", h);
  if (flags & FLAG_SLOT_OVERFLOW) return fail(SOP_E_LIST_OVERFLOW, "the halo of a chunk exceeded its slot capacity (mode 3)", h);
  return fail(SOP_E_LIST_OVERFLOW, "neighbor-list row exceeded cap_nb", h);
}


template <int G, bool COMP>
const void *persist_fn() { return (const void *)k_persist<G, COMP>; }

const void *persist_kernel(int lanes, bool comp) {
  switch (lanes) {
    case 1: return comp ? persist_fn<1, true>() : persist_fn<1, false>();
    case 2: return comp ? persist_fn<2, true>() : persist_fn<2, false>();
    case 4: return comp ? persist_fn<4, true>() : persist_fn<4, false>();
    case 8: return comp ? persist_fn<8, true>() : persist_fn<8, false>();
    case 16: return comp ? persist_fn<16, true>() : persist_fn<16, false>();
    default: return comp ? persist_fn<32, true>() : persist_fn<32, false>();
  }
}

// grid of the persistent kernel: every block co-resident (cooperative launch), no more blocks than there is work
int persistent_prepare(sop_handle *h) {
  const Plan &pl = h->plan;
  int block = h->prm.block_size > 0 ? h->prm.block_size : 512;
  int occ = 0;
  CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, persist_kernel(pl.lanes, pl.comp), block, 0));
  if (occ < 1) return fail(SOP_E_CUDA, "persistent kernel does not fit on an SM", h);
  int coop = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  if (!coop) return fail(SOP_E_CUDA, "device cannot do cooperative launches", h);
  const long long want = ((long long)h->S.n_inst * pl.lanes + block - 1) / block;
  h->coop_blocks = (int)std::max<long long>(1, std::min<long long>((long long)h->num_sms * std::min(occ, 2), want));
  h->coop_block_size = block;
  return SOP_OK;
}

int persistent_launch(sop_handle *h, int n, bool filter_last) {
  CUDA_OK(cudaMemsetAsync(h->S_bar, 0, 4, h->stream));
  span_close(h);
  span_begin(h, SPAN_STEP, n);
  SysDev S = h->S;
  int cur = h->cur;
  unsigned long long step0 = (unsigned long long)h->step;
  int nb = h->prm.nb_interval, fl = filter_last ? 1 : 0;
  unsigned *bar = h->S_bar;
  void *args[] = {&S, &cur, &step0, &n, &nb, &fl, &bar};
  CUDA_OK(cudaLaunchCooperativeKernel(persist_kernel(h->plan.lanes, h->plan.comp), dim3(h->coop_blocks),
                                      dim3(h->coop_block_size), args, 0, h->stream));
  h->launches++;
  return SOP_OK;
}

// The register budget follows the block size (one CTA per SM: 65536 / threads): the instantiations for blocks of <= 832 and
// <= 576 threads get 72 and 112 registers instead of 64, which takes address rematerialisation out of the pair loops
// (cfg 2, 544 threads: 4.19 -> 3.98 us per step; cfg 3, 832 threads: 5.39 -> 5.35).  Same arithmetic, same bits.
// SPEC instantiations (the run-time switches of the step loop folded, see k_resident): 1 = several chunks, with the lane
// counts and block sizes the auto plan gives large systems; 2 = one chunk per trajectory with the static all-pairs L1
template <int G>
const void *resident_fast_fn(bool comp, int block) {
  if (block <= 576) return comp ? (const void *)k_resident<G, true, false, 576, 1> : (const void *)k_resident<G, false, false, 576, 1>;
  if (block <= 832) return comp ? (const void *)k_resident<G, true, false, 832, 1> : (const void *)k_resident<G, false, false, 832, 1>;
  return nullptr;
}
const void *resident_fast_kernel(int lanes, bool comp, int block) {
  return lanes == 2 ? resident_fast_fn<2>(comp, block) : lanes == 4 ? resident_fast_fn<4>(comp, block) : nullptr;
}
const void *resident_fast1_kernel(int lanes, bool comp) {
#ifdef SOP_DEV_MIN
  if (lanes == 8) return nullptr;
#else
  if (lanes == 8) return comp ? (const void *)k_resident<8, true, false, 1024, 2> : (const void *)k_resident<8, false, false, 1024, 2>;
#endif
  if (lanes == 1) return comp ? (const void *)k_resident<1, true, false, 1024, 2> : (const void *)k_resident<1, false, false, 1024, 2>;
  return nullptr;
}

template <int G>
const void *resident_fn(bool comp, int block) {
  if constexpr (G <= 4) {
    if (block <= 576) return comp ? (const void *)k_resident<G, true, false, 576> : (const void *)k_resident<G, false, false, 576>;
    if (block <= 832) return comp ? (const void *)k_resident<G, true, false, 832> : (const void *)k_resident<G, false, false, 832>;
  }
  return comp ? (const void *)k_resident<G, true> : (const void *)k_resident<G, false>;
}

const void *resident_kernel(int lanes, bool comp, int block) {
#ifdef SOP_DEV_MIN      // development builds only (compile time): the instantiations cfg 1 / cfg 2 / cfg 3 take
  return lanes == 1 ? resident_fn<1>(comp, block) : lanes == 2 ? resident_fn<2>(comp, block) : resident_fn<4>(comp, block);
#else
  switch (lanes) {
    case 1: return resident_fn<1>(comp, block);
    case 2: return resident_fn<2>(comp, block);
    case 4: return resident_fn<4>(comp, block);
    case 8: return resident_fn<8>(comp, block);
    case 16: return resident_fn<16>(comp, block);
    default: return resident_fn<32>(comp, block);
  }
#endif
}

template <bool COMP, bool EPS>
const void *res2_fn_p(int P) {
  return P == 1 ? (const void *)k_res2<COMP, EPS, 1> : (const void *)k_res2<COMP, EPS, 2>;
}
const void *res2_kernel(bool comp, bool eps, int P) {
#ifdef SOP_DEV_MIN
  return nullptr;
#else
  if (comp) return eps ? res2_fn_p<true, true>(P) : res2_fn_p<true, false>(P);
  return eps ? res2_fn_p<false, true>(P) : res2_fn_p<false, false>(P);
#endif
}

const void *resident_stream_kernel(int lanes, bool comp) {
  if (lanes == 1) return comp ? (const void *)k_resident<1, true, true> : (const void *)k_resident<1, false, true>;
  return comp ? (const void *)k_resident<2, true, true> : (const void *)k_resident<2, false, true>;
}

int resident_prepare(sop_handle *h) {
  const Plan &pl = h->plan;
  h->R = pl.R;
  ResDev &R = h->R;
  char *w = h->ws;
  R.n_halo = (int *)(w + pl.off_nhalo); R.halo_gid = (int *)(w + pl.off_hgid);
  R.pl_loc = (unsigned short *)(w + pl.off_plloc); R.nat_pack = (int2 *)(w + pl.off_natloc);
  R.bond_pack = (int2 *)(w + pl.off_bondloc); R.xch = (uint4 *)(w + pl.off_xch); R.xchf = (uint4 *)(w + pl.off_xchf);
  R.nat_T = nullptr;
  R.nb_glob = (unsigned short *)(w + pl.off_nbglob);
  R.slice_len = 0; R.ticket = (int *)(w + pl.off_slice); R.done = R.ticket + 1;
  R.skew_chunk = 0; R.skew_period = 1; R.skew_ns = 0;
  if (const char *sk = getenv("SOP_TEST_SKEW")) {        // test hook "chunk,period,ns": one chunk runs late on some steps
    int a = 0, b = 1, c = 0;
    if (sscanf(sk, "%d,%d,%d", &a, &b, &c) == 3 && b > 0) { R.skew_chunk = a; R.skew_period = b; R.skew_ns = c; }
  }
  h->R2 = pl.R2;
  h->R2.pl_arr = (unsigned short *)(w + pl.off_plarr); h->R2.pl_g = (uchar2 *)(w + pl.off_plg);
  if (R.nat_tpad > 0) {
    R.nat_T = (int2 *)(w + pl.off_natloc);
    k_transpose_nat<<<(h->S.N + 255) / 256, 256, 0, h->stream>>>(h->S, R);
  }
  h->res_fn = R.stream ? resident_stream_kernel(pl.res_lanes, pl.comp) : resident_kernel(pl.res_lanes, pl.comp, pl.res_block);
  if (!R.stream && !h->S.nat_eps && !h->S.taus && R.skew_ns == 0 && !getenv("SOP_NO_FAST")) {
    const void *f = nullptr;
    if (R.C > 1 && !R.implicit_l1 && R.nat_smem) f = resident_fast_kernel(pl.res_lanes, pl.comp, pl.res_block);
    if (R.C == 1 && R.implicit_l1 && (pl.res_lanes == 1 ? R.nat_tpad > 0 : R.nat_smem != 0)) f = resident_fast1_kernel(pl.res_lanes, pl.comp);
    if (f) h->res_fn = f;
  }
  CUDA_OK(cudaFuncSetAttribute(h->res_fn, cudaFuncAttributeMaxDynamicSharedMemorySize, R.smem_bytes));
  const int loc_smem = ((h->S.N + 31) / 32) * 8 + R.chunk * 4;
  CUDA_OK(cudaFuncSetAttribute((const void *)k_localise, cudaFuncAttributeMaxDynamicSharedMemorySize, std::max(loc_smem, 1024)));
  int occ = 0;
  CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->res_fn, pl.res_block, R.smem_bytes));
  if (occ < 1) return fail(SOP_E_CUDA, "resident kernel does not fit on an SM", h);
  h->res_resident_ctas = occ * device_sm_count();          // CTAs of the first resident kernel the device holds at once
  if (pl.res2_ok) {
    h->res2_fn = res2_kernel(pl.comp, h->S.nat_eps != nullptr, pl.R2.P);
    CUDA_OK(cudaFuncSetAttribute(h->res2_fn, cudaFuncAttributeMaxDynamicSharedMemorySize, h->R2.smem_bytes));
    CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->res2_fn, pl.res2_block, h->R2.smem_bytes));
    if (occ < 1) return fail(SOP_E_CUDA, "the second resident kernel does not fit on an SM", h);
  }
  if (R.C > 1) {
    int coop = 0, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (!coop || (long long)h->S.T * R.C > (long long)occ * h->num_sms)
      return fail(SOP_E_CUDA, "the chunks of mode 3 cannot all be co-resident on this device", h);
    CUDA_OK(cudaMemsetAsync(R.xch, 0, 2 * (size_t)h->S.n_inst * 32, h->stream));
    CUDA_OK(cudaMemsetAsync(R.xchf, 0, 2 * (size_t)h->S.n_inst * 32, h->stream));
  }
  CUDA_OK(cudaMemsetAsync(R.n_halo, 0, (size_t)h->S.T * R.C * 4, h->stream));
  return SOP_OK;
}

int resident_launch(sop_handle *h, int n, bool filter_last, bool filter_first) {
  span_close(h);
  span_begin(h, SPAN_STEP, n);
  SysDev S = h->S;
  ResDev R = h->R;
  int cur = h->cur;
  unsigned long long step0 = (unsigned long long)h->step;
  int nb = h->prm.nb_interval, fl = (filter_last ? 1 : 0) | (filter_first ? 2 : 0);
  h->res_launch_id++;
  uint32_t stamp0 = ((h->res_launch_id & 0xFFFu) << 20) | 1u;     // never 0, never the previous launch's stamps
  // One chunk per trajectory and more trajectories than SMs (the many-runs batch): T CTAs of one SM each
  // would run in ceil(T / SMs) waves with the last one partly empty (256 on 148: 14 % of the machine idle).  The launch is cut
  // into time slices instead -- one CTA per (slice, trajectory), handed out slice-major by a ticket, a trajectory's slices
  // chained through `done` -- so every SM is busy until the last wave of slices.  A slice is what a separate launch of
  // slice_len steps would be (same prologue / epilogue, same bits); slice_len is a multiple of nb_interval.
  unsigned n_cta = (unsigned)(S.T * R.C);
  if (R.C == 1 && !h->plan.res2_ok && !R.stream && S.T > h->res_resident_ctas && !getenv("SOP_NO_SLICES")) {
    const int best_len = sop_plan_slices(n, nb, S.T, h->res_resident_ctas);   // (CTA slots, not SMs, when small CTAs share an SM)
    if (best_len > 0) {
      R.slice_len = best_len;
      h->last_slice_len = best_len;
      n_cta = (unsigned)(((n + best_len - 1) / best_len) * S.T);
      CUDA_OK(cudaMemsetAsync(R.ticket, 0, ((size_t)S.T + 1) * 4, h->stream));
    }
  }
  void *args[] = {&S, &R, &cur, &step0, &n, &nb, &fl, &stamp0};
  const dim3 grid(n_cta), block((unsigned)h->plan.res_block);
  if (h->plan.res2_ok) {
    Res2Dev Q = h->R2;
    void *args2[] = {&S, &R, &Q, &cur, &step0, &n, &nb, &fl, &stamp0};
    CUDA_OK(cudaLaunchCooperativeKernel(h->res2_fn, grid, dim3((unsigned)h->plan.res2_block), args2, (size_t)Q.smem_bytes, h->stream));
  }
  else if (R.C > 1) CUDA_OK(cudaLaunchCooperativeKernel(h->res_fn, grid, block, args, (size_t)R.smem_bytes, h->stream));
  else CUDA_OK(cudaLaunchKernel(h->res_fn, grid, block, args, (size_t)R.smem_bytes, h->stream));
  h->launches++;
  return SOP_OK;
}

// L1 (+ its slot form for mode 3), then L2 by Alg. 3.  with_filter = false (mode 3, inside sop_run only): the next
// resident launch filters in its prologue instead, and the canonical L2 rows stay stale until that launch ends.
int rebuild_lists(sop_handle *h, bool with_filter = true) {
  int rc = launch_build_l1(h);
  if (rc) return rc;
  if (h->plan.mode == 3 && !h->R.implicit_l1) {
    const int loc_smem = ((h->S.N + 31) / 32) * 8 + h->R.chunk * 4;
    k_localise<<<(unsigned)(h->S.T * h->R.C), 1024, loc_smem, h->stream>>>(h->S, h->R);
    h->launches++;
    if (h->plan.res2_ok) {
      k_arrange_l1<<<(unsigned)(((long long)h->S.n_inst * 32 + 255) / 256), 256, 0, h->stream>>>(h->S, h->R, h->R2);
      h->launches++;
    }
  }
  if (with_filter) launch_filter(h);
  span_close(h);
  return check_launch(h, "list rebuild");
}


// NEXT-1: one sample of the observable series = {Rg, X, cantilever force, tip force, V_fene, V_nat, V_rep, V_pull, V_tip, -}
// per trajectory, reduced on the device into slot (count mod capacity) of the ring; nothing goes to the host.
int record_sample(sop_handle *h) {
  const SysDev &S = h->S;
  const int slot = (int)(h->obs_count % h->obs_cap);
  double *d_slot = (double *)(h->ws + h->plan.off_series) + (size_t)slot * S.T * 10;
  double *partial = (double *)(h->ws + h->plan.off_epart);
  span_close(h);
  k_observables<<<(unsigned)S.T, 1024, 0, h->stream>>>(S, h->cur, (unsigned long long)h->step, h->obs_a, h->obs_b, d_slot, 10);
  dim3 grid((unsigned)h->plan.energy_blocks, (unsigned)S.T);
  k_energy<<<grid, 256, 0, h->stream>>>(S, h->cur, (unsigned long long)h->step, partial);
  k_energy_final<<<(S.T * 5 + 127) / 128, 128, 0, h->stream>>>(S.T, h->plan.energy_blocks, partial, d_slot + 4, 10);
  h->launches += 3;
  h->obs_steps[slot] = h->step;
  h->obs_count++;
  return check_launch(h, "observable sample");
}

// ------------------------------------------------------------------------------------------------
// sop_energies_noalloc (include/sop.h): the a10 reduction with its scratch in a file-scope static __device__ array, for
// callers that may not allocate.  In HOST code the name g_noalloc_scratch is a host-side stand-in, not a device address:
// the address a kernel may use comes from cudaGetSymbolAddress, resolved once per device with that device current.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_noalloc_scratch[SOP_NOALLOC_SCRATCH_BYTES / sizeof(double)];

constexpr int NOALLOC_MAX_DEVICES = 64;
double *g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};          // device address of the array on each device, once resolved

// block partials -> {fene, native, rep, pull, tip, total} per trajectory: the blocks in order (as k_energy_final), the total
// as sop_get_energies forms it on the host ((((e0 + e1) + e2) + e3) + e4 in fp64), so that the two paths agree bit for bit
__global__ void k_energy_final_total(int T, int nblk, const double *partial, double *e_out) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= T) return;
  double e[5];
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    double v = 0;
    for (int b = 0; b < nblk; ++b) v += partial[((size_t)t * nblk + b) * 5 + k];
    e[k] = v;
    e_out[(size_t)t * 6 + k] = v;
  }
  e_out[(size_t)t * 6 + 5] = e[0] + e[1] + e[2] + e[3] + e[4];
}

int noalloc_scratch(sop_handle *h, double **out) {
  int dev = -1;
  CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(SOP_E_CUDA, "sop_energies_noalloc: device ordinal out of range", h);
  if (!g_noalloc_ptr[dev]) {
    double *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void **)&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p)
      return fail(SOP_E_CUDA, std::string("sop_energies_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e), h);
    g_noalloc_ptr[dev] = p;       // (two threads racing here store the same address)
  }
  *out = g_noalloc_ptr[dev];
  return SOP_OK;
}

}  // namespace

// =====================================================================================================
extern "C" {

// Steps per time slice of a launch of n_steps Langevin steps over n_traj one-chunk trajectories when the device holds
// cta_slots CTAs of the resident kernel at once; 0 = one CTA per trajectory for the whole launch.  Host arithmetic only.
// Cost model: waves of CTAs x (slice length + 3.5 steps of measured prologue / epilogue cost per slice); slices are multiples
// of nb_interval and at least two filter intervals long; slicing must save 3 % to be chosen.
int32_t sop_plan_slices(int32_t n_steps, int32_t nb_interval, int32_t n_traj, int32_t cta_slots) {
  if (n_steps < 1 || nb_interval < 1 || n_traj < 1 || cta_slots < 1 || n_traj <= cta_slots) return 0;
  long long best_cost = 0; int best_len = 0;
  for (int len = 2 * nb_interval; len < n_steps; len += nb_interval) {
    const long long slices = (n_steps + len - 1) / len;
    const long long waves = (slices * n_traj + cta_slots - 1) / cta_slots;
    const long long cost = waves * (2LL * len + 7);
    if (!best_len || cost < best_cost) { best_cost = cost; best_len = len; }
  }
  const long long plain = (long long)((n_traj + cta_slots - 1) / cta_slots) * (2LL * n_steps + 7);
  return best_len && best_cost * 100 < plain * 97 ? best_len : 0;
}


const char *sop_last_error(sop_handle *h) { return h ? h->last_error.c_str() : g_last_error.c_str(); }

int sop_query_workspace(const sop_topology *topo, const float *native_xyz, const sop_params *params, int32_t n_traj,
                        size_t *bytes_out) {
  if (!bytes_out) return fail(SOP_E_ARG, "bytes_out is null");
  Plan pl;
  int rc = make_plan(topo, native_xyz, params, n_traj, pl);
  if (rc) return rc;
  *bytes_out = pl.total;
  return SOP_OK;
}

int sop_create(const sop_topology *tp, const float *native_xyz, const sop_params *p, int32_t n_traj,
               void *d_workspace, size_t workspace_bytes, sop_handle **out) {
  if (!out) return fail(SOP_E_ARG, "out is null");
  *out = nullptr;
  sop_handle *h = new sop_handle();
  Plan &pl = h->plan;
  int rc = make_plan(tp, native_xyz, p, n_traj, pl);
  if (rc) { delete h; return rc; }
  if (!d_workspace || workspace_bytes < pl.total || ((uintptr_t)d_workspace & 255)) {
    delete h;
    return fail(SOP_E_ARG, "workspace missing, misaligned or smaller than sop_query_workspace says");
  }
  const int N = pl.N, T = pl.T;
  h->prm = *p;
  h->prm.fixed = nullptr; h->prm.pulled = nullptr; h->prm.kT_per_traj = nullptr;
  h->stream = (cudaStream_t)p->stream;
  h->ws = (char *)d_workspace;

  // ---- static tables in internal order; r0 from the native structure in fp64, rounded to fp32
  auto X = [&](int caller, int a) { return (double)native_xyz[3 * (size_t)caller + a]; };
  auto dist = [&](int i, int j) {
    double dx = X(i, 0) - X(j, 0), dy = X(i, 1) - X(j, 1), dz = X(i, 2) - X(j, 2);
    return std::sqrt(dx * dx + dy * dy + dz * dz);
  };
  std::vector<int2> bond_tab((size_t)N * pl.cap_b, make_int2(-1, 0));
  std::vector<int> bfill(N, 0);
  std::vector<std::vector<int>> excl(N);
  for (int b = 0; b < tp->n_bonds; ++b) {
    int i = tp->bonds[2 * b], j = tp->bonds[2 * b + 1];
    float r0 = (float)dist(i, j);
    int ii = pl.iperm[i], jj = pl.iperm[j];
    int r0b; memcpy(&r0b, &r0, 4);
    bond_tab[(size_t)ii * pl.cap_b + bfill[ii]++] = make_int2(jj, r0b);
    bond_tab[(size_t)jj * pl.cap_b + bfill[jj]++] = make_int2(ii, r0b);
    excl[ii].push_back(jj); excl[jj].push_back(ii);
  }
  struct NatE { int j; float r0sq; float eps; };
  std::vector<std::vector<NatE>> nat(N);
  for (int c = 0; c < tp->n_native; ++c) {
    int i = tp->native[2 * c], j = tp->native[2 * c + 1];
    float r0 = (float)dist(i, j);
    float r0sq = (float)((double)r0 * (double)r0);
    float eps = tp->native_eps ? tp->native_eps[c] : p->eps_native;
    int ii = pl.iperm[i], jj = pl.iperm[j];
    nat[ii].push_back({jj, r0sq, eps}); nat[jj].push_back({ii, r0sq, eps});
    excl[ii].push_back(jj); excl[jj].push_back(ii);
  }
  std::vector<int> nat_ptr(N + 1, 0), excl_ptr(N + 1, 0);
  std::vector<int2> nat_tab; nat_tab.reserve(pl.n_nat_entries);
  std::vector<float> nat_eps; std::vector<int> excl_idx; excl_idx.reserve(pl.n_excl);
  for (int i = 0; i < N; ++i) {
    std::sort(nat[i].begin(), nat[i].end(), [](const NatE &a, const NatE &b) { return a.j < b.j; });
    for (auto &e : nat[i]) { int b; memcpy(&b, &e.r0sq, 4); nat_tab.push_back(make_int2(e.j, b)); nat_eps.push_back(e.eps); }
    nat_ptr[i + 1] = (int)nat_tab.size();
    std::sort(excl[i].begin(), excl[i].end());
    for (size_t q = 0; q < excl[i].size(); ++q) {
      if (excl[i][q] == i || (q && excl[i][q] == excl[i][q - 1])) {
        delete h;
        return fail(SOP_E_ARG, "duplicate pair, self pair, or a bond that is also a native contact");
      }
      excl_idx.push_back(excl[i][q]);
    }
    excl_ptr[i + 1] = (int)excl_idx.size();
  }

  // ---- mode 4: the static pairs of Alg. 4 (every bond and native contact once) with their places in the force array
  std::vector<int4> spair;
  std::vector<float2> spar;
  if (pl.mode == 4) {
    auto bond_slot = [&](int ii, int jj) { for (int b = 0; b < pl.cap_b; ++b) if (bond_tab[(size_t)ii * pl.cap_b + b].x == jj) return ii * pl.cap_b + b; return -1; };
    auto nat_slot = [&](int ii, int jj) { for (int q = nat_ptr[ii]; q < nat_ptr[ii + 1]; ++q) if (nat_tab[q].x == jj) return N * pl.cap_b + q; return -1; };
    for (int b = 0; b < tp->n_bonds; ++b) {
      const int ii = pl.iperm[tp->bonds[2 * b]], jj = pl.iperm[tp->bonds[2 * b + 1]];
      spair.push_back(make_int4(ii, jj, bond_slot(ii, jj), bond_slot(jj, ii)));
      spar.push_back(make_float2((float)dist(tp->bonds[2 * b], tp->bonds[2 * b + 1]), 0.f));
    }
    for (int c = 0; c < tp->n_native; ++c) {
      const int ii = pl.iperm[tp->native[2 * c]], jj = pl.iperm[tp->native[2 * c + 1]];
      const float r0 = (float)dist(tp->native[2 * c], tp->native[2 * c + 1]);
      spair.push_back(make_int4(ii, jj, nat_slot(ii, jj), nat_slot(jj, ii)));
      spar.push_back(make_float2((float)((double)r0 * (double)r0), tp->native_eps ? tp->native_eps[c] : p->eps_native));
    }
  }

  // ---- tags, anchors, initial coordinates
  std::vector<uint32_t> &tag = h->tag;
  tag.resize(N);
  for (int i = 0; i < N; ++i) tag[i] = (uint32_t)pl.perm[i];
  for (int q = 0; q < p->n_fixed; ++q) {
    if (!p->fixed || p->fixed[q] < 0 || p->fixed[q] >= N) { delete h; return fail(SOP_E_ARG, "fixed bead out of range"); }
    tag[pl.iperm[p->fixed[q]]] |= TAG_FIXED;
  }
  double nrm[3] = {p->pull_dir[0], p->pull_dir[1], p->pull_dir[2]};
  std::vector<float> adotn(N, 0.f);
  for (int q = 0; q < p->n_pulled; ++q) {
    if (!p->pulled || p->pulled[q] < 0 || p->pulled[q] >= N) { delete h; return fail(SOP_E_ARG, "pulled bead out of range"); }
    int c = p->pulled[q], ii = pl.iperm[c];
    tag[ii] |= TAG_PULLED;
    adotn[ii] = (float)(X(c, 0) * nrm[0] + X(c, 1) * nrm[1] + X(c, 2) * nrm[2]);
  }
  h->obs_a = pl.iperm[p->n_fixed > 0 ? p->fixed[0] : 0];
  h->obs_b = pl.iperm[p->n_pulled > 0 ? p->pulled[0] : N - 1];
  std::vector<float4> pos0((size_t)N * T);
  for (int t = 0; t < T; ++t)
    for (int ii = 0; ii < N; ++ii) {
      int c = pl.perm[ii];
      float w; memcpy(&w, &tag[ii], 4);
      pos0[(size_t)t * N + ii] = make_float4(native_xyz[3 * (size_t)c], native_xyz[3 * (size_t)c + 1], native_xyz[3 * (size_t)c + 2], w);
    }

  // ---- device view
  SysDev &S = h->S;
  memset(&S, 0, sizeof(S));
  char *w = h->ws;
  S.N = N; S.T = T; S.n_inst = N * T;
  S.pos[0] = (float4 *)(w + pl.off_pos0); S.pos[1] = (float4 *)(w + pl.off_pos1);
  S.carry = pl.comp ? (float4 *)(w + pl.off_carry) : nullptr;
  S.force = (float4 *)(w + pl.off_force);
  S.cap_b = pl.cap_b; S.bond_tab = (const int2 *)(w + pl.off_bond);
  S.nat_ptr = (const int *)(w + pl.off_natptr); S.nat_tab = (const int2 *)(w + pl.off_nattab);
  S.nat_eps = tp->native_eps ? (const float *)(w + pl.off_nateps) : nullptr;
  S.excl_ptr = (const int *)(w + pl.off_exclptr); S.excl_idx = (const int *)(w + pl.off_exclidx);
  S.pull_adotn = p->n_pulled > 0 ? (const float *)(w + pl.off_adotn) : nullptr;
  S.static_l1 = pl.static_l1; S.cap_pl = pl.cap_pl; S.cap_nb = pl.cap_nb;
  S.pl_cnt = (int *)(w + pl.off_plcnt); S.pl_idx = (int *)(w + pl.off_plidx);
  S.nb_cnt = (int *)(w + pl.off_nbcnt); S.nb_idx = (int *)(w + pl.off_nbidx);
  S.max_cells = pl.max_cells;
  S.bbox = (float *)(w + pl.off_bbox); S.grid = (GridDev *)(w + pl.off_grid);
  S.cell_of = (int *)(w + pl.off_cellof); S.cell_cnt = (int *)(w + pl.off_cellcnt);
  S.cell_start = (int *)(w + pl.off_cellstart); S.cell_bead = (int *)(w + pl.off_cellbead);
  S.cell_pos = (float4 *)(w + pl.off_cellpos);
  S.cell_edge = pl.static_l1 ? 1.0f : (float)((double)p->R_pl * 1.001);
  S.k_fene = p->k_fene; S.R0 = p->R0; S.inv_R0sq = (float)(1.0 / ((double)p->R0 * (double)p->R0));
  S.eps_native = p->eps_native;
  const double sig6 = std::pow((double)p->sigma, 6.0);
  S.c_rep_e = (float)((double)p->eps_rep * sig6); S.c_rep_f = (float)(6.0 * (double)p->eps_rep * sig6);
  S.R_nb2 = (float)((double)p->R_nb * (double)p->R_nb);
  S.R_pl2 = pl.static_l1 ? std::numeric_limits<float>::infinity() : (float)((double)p->R_pl * (double)p->R_pl);
  S.D = p->dt_over_zeta; S.amp = (float)std::sqrt(2.0 * (double)p->kT * (double)p->dt_over_zeta);
  S.seed_lo = (uint32_t)(p->seed & 0xFFFFFFFFu); S.seed_hi = (uint32_t)(p->seed >> 32);
  S.traj_offset = p->traj_offset;
  S.has_pull = p->n_pulled > 0; S.pull_k = p->pull_k; S.pull_v = p->pull_v;
  S.pull_nx = p->pull_dir[0]; S.pull_ny = p->pull_dir[1]; S.pull_nz = p->pull_dir[2];
  S.tip_on = p->tip_on != 0; S.tip_R = p->tip_R; S.tip_eps = p->tip_eps;
  S.tip_sigma6 = (float)std::pow((double)p->tip_sigma, 6.0); S.tip_v = p->tip_v;
  S.tip_cx = p->tip_c0[0]; S.tip_cy = p->tip_c0[1]; S.tip_cz = p->tip_c0[2];
  S.tip_nx = p->tip_dir[0]; S.tip_ny = p->tip_dir[1]; S.tip_nz = p->tip_dir[2];
  S.taus = p->rng == 1 ? (uint4 *)(w + pl.off_taus) : nullptr;
  S.amp_t = p->kT_per_traj ? (const float *)(w + pl.off_ampt) : nullptr;
  S.flags = (int *)(w + pl.off_flags);

  // ---- upload (synchronous copies from pageable host vectors; create is not on the hot path)
  cudaStream_t st = h->stream;
  auto up = [&](size_t off, const void *src, size_t bytes) -> cudaError_t {
    if (!bytes) return cudaSuccess;
    return cudaMemcpyAsync(w + off, src, bytes, cudaMemcpyHostToDevice, st);
  };
  cudaError_t e = cudaSuccess;
  auto acc = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  acc(cudaMemsetAsync(w + pl.off_flags, 0, 64, st));
  acc(cudaMemsetAsync(w + pl.off_bar, 0, 256, st));
  acc(up(pl.off_pos0, pos0.data(), pos0.size() * 16));
  acc(up(pl.off_pos1, pos0.data(), pos0.size() * 16));
  if (pl.comp) acc(cudaMemsetAsync(w + pl.off_carry, 0, pos0.size() * 16, st));
  acc(up(pl.off_bond, bond_tab.data(), bond_tab.size() * 8));
  acc(up(pl.off_natptr, nat_ptr.data(), nat_ptr.size() * 4));
  acc(up(pl.off_nattab, nat_tab.data(), nat_tab.size() * 8));
  if (tp->native_eps) acc(up(pl.off_nateps, nat_eps.data(), nat_eps.size() * 4));
  acc(up(pl.off_exclptr, excl_ptr.data(), excl_ptr.size() * 4));
  acc(up(pl.off_exclidx, excl_idx.data(), excl_idx.size() * 4));
  if (p->n_pulled > 0) acc(up(pl.off_adotn, adotn.data(), adotn.size() * 4));
  std::vector<float> kT_t, amp_t;
  if (p->kT_per_traj) {
    for (int t = 0; t < T; ++t) { kT_t.push_back(p->kT_per_traj[t]); amp_t.push_back((float)std::sqrt(2.0 * (double)p->kT_per_traj[t] * (double)p->dt_over_zeta)); }
    acc(up(pl.off_kTt, kT_t.data(), (size_t)T * 4)); acc(up(pl.off_ampt, amp_t.data(), (size_t)T * 4));
  }
  if (pl.mode == 4) {
    PairDev &P = h->P;
    memset(&P, 0, sizeof(P));
    P.n_static = (int)spair.size(); P.n_bonds = tp->n_bonds;
    P.spair = (const int4 *)(w + pl.off_spair); P.spar = (const float2 *)(w + pl.off_spar);
    P.cap_pairs = pl.cap_pairs; P.lpair = (int4 *)(w + pl.off_lpair); P.n_lpair = (int *)(w + pl.off_nlpair);
    P.n_place = pl.n_place; P.F = (float4 *)(w + pl.off_F); P.Facc = (float *)(w + pl.off_Facc); P.atomics = p->pair_atomics ? 1 : 0;
    acc(up(pl.off_spair, spair.data(), spair.size() * 16)); acc(up(pl.off_spar, spar.data(), spar.size() * 8));
    acc(cudaMemsetAsync(w + pl.off_nlpair, 0, (size_t)T * 4, st));
    if (P.atomics) acc(cudaMemsetAsync(w + pl.off_Facc, 0, (size_t)N * T * 16, st));
  }
  acc(cudaStreamSynchronize(st));
  if (e != cudaSuccess) { std::string m = cudaGetErrorString(e); delete h; return fail(SOP_E_CUDA, "upload: " + m); }

  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev);
  h->S_bar = (unsigned *)(w + pl.off_bar);
  if (pl.mode == 2) {
    rc = persistent_prepare(h);
    if (rc) { std::string m = g_last_error; delete h; return fail(rc, m); }
  }

  if (pl.mode == 3) {
    rc = resident_prepare(h);
    if (rc) { std::string m = g_last_error; delete h; return fail(rc, m); }
  }

  if (S.taus) {
    k_taus_seed<<<(unsigned)((S.n_inst + 255) / 256), 256, 0, h->stream>>>(S, 0);
    h->launches++;
  }
  h->cur = 0; h->step = 0;
  h->obs_stride = p->obs_capacity > 0 ? p->obs_stride : 0; h->obs_cap = p->obs_capacity;
  h->obs_steps.assign((size_t)std::max(0, p->obs_capacity), 0);
  rc = rebuild_lists(h);
  if (!rc) rc = read_flags(h);
  if (rc) { std::string m = h->last_error; delete h; return fail(rc, m); }
  *out = h;
  return SOP_OK;
}

void sop_destroy(sop_handle *h) {
  if (!h) return;
  cudaStreamSynchronize(h->stream);
  for (auto &sp : h->spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
  if (h->stage) cudaFreeHost(h->stage);
  delete h;
}

// Kernel timing for the bench: CUDA events on the handle's stream around groups of launches.
// out[0..2] = ms in {step kernels, L2 filter kernels, L1 build kernels}, out[3..5] = number of such spans,
// out[6] = Langevin steps covered by the step spans, out[7] = reserved.  Reading synchronises and resets.
int sop_set_profiling(sop_handle *h, int32_t on) {
  if (!h) return fail(SOP_E_ARG, "null handle");
  h->profiling = on != 0;
  return SOP_OK;
}

int sop_get_profile(sop_handle *h, double out[8]) {
  if (!h || !out) return fail(SOP_E_ARG, "null argument", h);
  span_close(h);
  CUDA_OK(cudaStreamSynchronize(h->stream));
  for (auto &sp : h->spans) {
    float ms = 0.f;
    cudaEventElapsedTime(&ms, sp.a, sp.b);
    h->prof_ms[sp.kind] += ms; h->prof_n[sp.kind]++;
    if (sp.kind == SPAN_STEP) h->prof_steps += sp.steps;
    cudaEventDestroy(sp.a); cudaEventDestroy(sp.b);
  }
  h->spans.clear();
  for (int k = 0; k < 3; ++k) { out[k] = h->prof_ms[k]; out[3 + k] = (double)h->prof_n[k]; h->prof_ms[k] = 0; h->prof_n[k] = 0; }
  out[6] = (double)h->prof_steps; out[7] = 0;
  h->prof_steps = 0;
  return SOP_OK;
}

int sop_run(sop_handle *h, int64_t n_steps) {
  if (!h || n_steps < 0) return fail(SOP_E_ARG, "bad handle or n_steps", h);
  const int64_t nb = h->prm.nb_interval, plv = h->prm.pl_interval, ost = h->obs_stride;
  int64_t left = n_steps;
  bool pending_filter = false;
  while (left > 0) {
    if (h->plan.mode == 2 || h->plan.mode == 3) {
      // one persistent launch runs up to the next pair-list boundary (or observable sample), re-filtering L2 inside
      int64_t n = std::min<int64_t>(left, (1 << 20) - 2);
      if (!h->S.static_l1) n = std::min<int64_t>(n, plv - (h->step % plv));
      if (ost > 0) n = std::min<int64_t>(n, ost - (h->step % ost));
      const bool l1_due = !h->S.static_l1 && (h->step + n) % plv == 0;
      const bool sample_due = ost > 0 && (h->step + n) % ost == 0;
      int rc = h->plan.mode == 3 ? resident_launch(h, (int)n, !l1_due, pending_filter) : persistent_launch(h, (int)n, !l1_due);
      if (rc) return rc;
      pending_filter = false;
      if (h->plan.mode == 2) h->cur ^= (int)(n & 1);      // mode 3 writes the final layer back in place
      h->step += n; left -= n;
      if (l1_due) {
        // (a sample needs the canonical L2 of this very step: the filter then runs as its own kernel)
        pending_filter = h->plan.mode == 3 && left > 0 && !sample_due;
        rc = rebuild_lists(h, !pending_filter);
        if (rc) return rc;
        if (pending_filter) h->l2_built_at = h->step;
      }
      else if (h->step / nb * nb > h->l2_built_at) h->l2_built_at = h->step / nb * nb;
      if (sample_due) { rc = record_sample(h); if (rc) return rc; }
    } else {
      span_begin(h, SPAN_STEP, 1);
      if (h->prm.integrator == 2) { launch_step2(h, 0); launch_step2(h, 1); h->step++; left--; }     // (the result is back in layer cur)
      else { if (h->plan.mode == 4) launch_pair_step(h, false); else launch_step(h, false); h->cur ^= 1; h->step++; left--; }
      if (!h->S.static_l1 && h->step % plv == 0) { int rc = launch_build_l1(h); if (rc) return rc; }
      if (h->step % nb == 0) launch_filter(h);
      if (ost > 0 && h->step % ost == 0) { int rc = record_sample(h); if (rc) return rc; }
    }
  }
  span_close(h);
  return check_launch(h, "sop_run");
}

int sop_set_observable_stride(sop_handle *h, int32_t stride) {
  if (!h || stride < 0) return fail(SOP_E_ARG, "bad stride", h);
  if (stride > 0 && h->obs_cap < 1) return fail(SOP_E_ARG, "the handle was created with obs_capacity = 0", h);
  h->obs_stride = stride;
  return SOP_OK;
}

int sop_get_observable_series(sop_handle *h, double *o_out, int64_t *steps_out, int32_t max_samples, int32_t *n_out) {
  if (!h || !n_out || max_samples < 0) return fail(SOP_E_ARG, "null argument", h);
  const int T = h->S.T;
  const int64_t have = std::min<int64_t>(h->obs_count, h->obs_cap);
  const int n = (int)std::min<int64_t>(have, max_samples);
  *n_out = n;
  if (n == 0) return read_flags(h);
  if (!o_out) return fail(SOP_E_ARG, "o_out is null", h);
  const double *ring = (const double *)(h->ws + h->plan.off_series);
  for (int q = 0; q < n; ++q) {                 // the last n samples, oldest first
    const int slot = (int)((h->obs_count - n + q) % h->obs_cap);
    CUDA_OK(cudaMemcpyAsync(o_out + (size_t)q * T * 10, ring + (size_t)slot * T * 10, (size_t)T * 80, cudaMemcpyDeviceToHost, h->stream));
    if (steps_out) steps_out[q] = h->obs_steps[slot];
  }
  int rc = read_flags(h);
  for (size_t r = 0; r < (size_t)n * T; ++r) {
    double *e = o_out + 10 * r + 4;
    e[5] = e[0] + e[1] + e[2] + e[3] + e[4];
  }
  return rc;
}

int sop_sync(sop_handle *h) {
  if (!h) return fail(SOP_E_ARG, "null handle");
  return read_flags(h);
}

int sop_get_step(sop_handle *h, int64_t *step) {
  if (!h || !step) return fail(SOP_E_ARG, "null argument", h);
  *step = h->step;
  return SOP_OK;
}

int sop_set_step(sop_handle *h, int64_t step) {
  if (!h || step < 0) return fail(SOP_E_ARG, "bad step", h);
  h->step = step; h->l1_built_at = step; h->l2_built_at = step;
  return SOP_OK;
}

static int ensure_stage(sop_handle *h) {
  if (h->stage) return SOP_OK;
  CUDA_OK(cudaHostAlloc((void **)&h->stage, (size_t)h->S.n_inst * 16, cudaHostAllocDefault));
  return SOP_OK;
}

int sop_get_coords(sop_handle *h, float *xyz_out) {
  if (!h || !xyz_out) return fail(SOP_E_ARG, "null argument", h);
  const int N = h->S.N, T = h->S.T;
  int rc = ensure_stage(h);
  if (rc) return rc;
  CUDA_OK(cudaMemcpyAsync(h->stage, h->S.pos[h->cur], (size_t)N * T * 16, cudaMemcpyDeviceToHost, h->stream));
  rc = read_flags(h);
  for (int t = 0; t < T; ++t)
    for (int ii = 0; ii < N; ++ii) {
      const float4 &v = h->stage[(size_t)t * N + ii];
      float *o = xyz_out + 3 * ((size_t)t * N + h->plan.perm[ii]);
      o[0] = v.x; o[1] = v.y; o[2] = v.z;
    }
  return rc;
}

int sop_set_coords(sop_handle *h, const float *xyz) {
  if (!h || !xyz) return fail(SOP_E_ARG, "null argument", h);
  const int N = h->S.N, T = h->S.T;
  int rc = ensure_stage(h);
  if (rc) return rc;
  CUDA_OK(cudaStreamSynchronize(h->stream));
  for (int t = 0; t < T; ++t)
    for (int ii = 0; ii < N; ++ii) {
      const float *s = xyz + 3 * ((size_t)t * N + h->plan.perm[ii]);
      float w; memcpy(&w, &h->tag[ii], 4);
      h->stage[(size_t)t * N + ii] = make_float4(s[0], s[1], s[2], w);
    }
  CUDA_OK(cudaMemcpyAsync(h->S.pos[h->cur], h->stage, (size_t)N * T * 16, cudaMemcpyHostToDevice, h->stream));
  if (h->S.carry) CUDA_OK(cudaMemsetAsync(h->S.carry, 0, (size_t)N * T * 16, h->stream));
  rc = rebuild_lists(h);
  if (rc) return rc;
  return read_flags(h);
}

int sop_get_energies(sop_handle *h, double *e_out) {
  if (!h || !e_out) return fail(SOP_E_ARG, "null argument", h);
  const SysDev &S = h->S;
  double *partial = (double *)(h->ws + h->plan.off_epart), *d_e = (double *)(h->ws + h->plan.off_eout);
  dim3 grid((unsigned)h->plan.energy_blocks, (unsigned)S.T);
  k_energy<<<grid, 256, 0, h->stream>>>(S, h->cur, (unsigned long long)h->step, partial);
  k_energy_final<<<(S.T * 5 + 127) / 128, 128, 0, h->stream>>>(S.T, h->plan.energy_blocks, partial, d_e, 6);
  h->launches += 2;
  int rc = check_launch(h, "energy");
  if (rc) return rc;
  CUDA_OK(cudaMemcpyAsync(e_out, d_e, (size_t)S.T * 6 * 8, cudaMemcpyDeviceToHost, h->stream));
  rc = read_flags(h);
  for (int t = 0; t < S.T; ++t) {
    double *e = e_out + 6 * (size_t)t;
    e[5] = e[0] + e[1] + e[2] + e[3] + e[4];
  }
  return rc;
}

int sop_energies_noalloc(sop_handle *h, double *d_e_out) {
  if (!h || !d_e_out) return fail(SOP_E_ARG, "null argument", h);
  const SysDev &S = h->S;
  const size_t need = (size_t)S.T * (size_t)h->plan.energy_blocks * 5 * sizeof(double);
  if (need > (size_t)SOP_NOALLOC_SCRATCH_BYTES)
    return fail(SOP_E_ARG, "sop_energies_noalloc: " + std::to_string(S.T) + " trajectories x " + std::to_string(h->plan.energy_blocks) +
                " reduction blocks need " + std::to_string(need) + " bytes of scratch, the static scratch holds " +
                std::to_string((size_t)SOP_NOALLOC_SCRATCH_BYTES) + " (use sop_get_energies)", h);
  double *partial = nullptr;
  int rc = noalloc_scratch(h, &partial);
  if (rc) return rc;
  dim3 grid((unsigned)h->plan.energy_blocks, (unsigned)S.T);
  k_energy<<<grid, 256, 0, h->stream>>>(S, h->cur, (unsigned long long)h->step, partial);
  k_energy_final_total<<<(S.T + 127) / 128, 128, 0, h->stream>>>(S.T, h->plan.energy_blocks, partial, d_e_out);
  h->launches += 2;
  return check_launch(h, "energy (no-alloc)");
}

int sop_replica_exchange(sop_handle *h, int32_t parity, uint64_t sweep, int32_t *accepted_out) {
  if (!h || (parity != 0 && parity != 1)) return fail(SOP_E_ARG, "bad argument", h);
  if (!h->S.amp_t) return fail(SOP_E_ARG, "replica exchange needs params.kT_per_traj", h);
  const SysDev &S = h->S;
  double *partial = (double *)(h->ws + h->plan.off_epart), *d_e = (double *)(h->ws + h->plan.off_eout);
  int *d_acc = (int *)(h->ws + h->plan.off_rexacc);
  dim3 grid((unsigned)h->plan.energy_blocks, (unsigned)S.T);
  k_energy<<<grid, 256, 0, h->stream>>>(S, h->cur, (unsigned long long)h->step, partial);
  k_energy_final<<<(S.T * 5 + 127) / 128, 128, 0, h->stream>>>(S.T, h->plan.energy_blocks, partial, d_e, 6);
  const int pairs = (S.T + 1) / 2;
  k_replica_exchange<<<(pairs + 127) / 128, 128, 0, h->stream>>>(S, d_e, (float *)(h->ws + h->plan.off_kTt), (float *)(h->ws + h->plan.off_ampt),
                                                                parity, (unsigned long long)sweep, d_acc);
  h->launches += 3;
  int rc = check_launch(h, "replica exchange");
  if (rc) return rc;
  if (accepted_out) {
    const int tried = (S.T - parity) / 2;
    for (int q = 0; q < S.T / 2; ++q) accepted_out[q] = 0;
    if (tried > 0) {
      std::vector<int> tmp((size_t)S.T, 0);
      CUDA_OK(cudaMemcpyAsync(tmp.data(), d_acc, (size_t)S.T * 4, cudaMemcpyDeviceToHost, h->stream));
      rc = read_flags(h);
      for (int t = parity; t + 1 < S.T; t += 2) accepted_out[t / 2] = tmp[t / 2];
      return rc;
    }
  }
  return SOP_OK;
}

int sop_get_temperatures(sop_handle *h, float *kT_out) {
  if (!h || !kT_out) return fail(SOP_E_ARG, "null argument", h);
  if (!h->S.amp_t) { for (int t = 0; t < h->S.T; ++t) kT_out[t] = h->prm.kT; return SOP_OK; }
  CUDA_OK(cudaMemcpyAsync(kT_out, h->ws + h->plan.off_kTt, (size_t)h->S.T * 4, cudaMemcpyDeviceToHost, h->stream));
  return read_flags(h);
}

int sop_get_observables(sop_handle *h, double *o_out) {
  if (!h || !o_out) return fail(SOP_E_ARG, "null argument", h);
  const SysDev &S = h->S;
  double *d_o = (double *)(h->ws + h->plan.off_epart);          // reuses the energy partial buffer (>= T * 40 bytes)
  k_observables<<<(unsigned)S.T, 1024, 0, h->stream>>>(S, h->cur, (unsigned long long)h->step, h->obs_a, h->obs_b, d_o, 4);
  h->launches++;
  int rc = check_launch(h, "observables");
  if (rc) return rc;
  CUDA_OK(cudaMemcpyAsync(o_out, d_o, (size_t)S.T * 4 * 8, cudaMemcpyDeviceToHost, h->stream));
  return read_flags(h);
}

int sop_get_forces(sop_handle *h, float *f_out) {
  if (!h || !f_out) return fail(SOP_E_ARG, "null argument", h);
  const int N = h->S.N, T = h->S.T;
  int rc = ensure_stage(h);
  if (rc) return rc;
  if (h->plan.mode == 4) launch_pair_step(h, true); else launch_step(h, true);
  rc = check_launch(h, "forces");
  if (rc) return rc;
  CUDA_OK(cudaMemcpyAsync(h->stage, h->S.force, (size_t)N * T * 16, cudaMemcpyDeviceToHost, h->stream));
  rc = read_flags(h);
  for (int t = 0; t < T; ++t)
    for (int ii = 0; ii < N; ++ii) {
      const float4 &v = h->stage[(size_t)t * N + ii];
      float *o = f_out + 3 * ((size_t)t * N + h->plan.perm[ii]);
      o[0] = v.x; o[1] = v.y; o[2] = v.z;
    }
  return rc;
}

int sop_get_lists(sop_handle *h, int32_t traj, int32_t level, int32_t *row_cnt, int32_t *idx, int32_t *cap_out,
                  int64_t *built_at_step) {
  if (!h || traj < 0 || traj >= h->S.T || (level != 1 && level != 2)) return fail(SOP_E_ARG, "bad argument", h);
  const SysDev &S = h->S;
  const int N = S.N;
  const int cap = level == 1 ? S.cap_pl : S.cap_nb;
  if (cap_out) *cap_out = cap;
  if (built_at_step) *built_at_step = level == 1 ? h->l1_built_at : h->l2_built_at;
  if (!row_cnt) return SOP_OK;
  const size_t row0 = (level == 1 && S.static_l1) ? 0 : (size_t)traj * N;
  const int *d_cnt = (level == 1 ? S.pl_cnt : S.nb_cnt) + row0;
  const int *d_idx = (level == 1 ? S.pl_idx : S.nb_idx) + row0 * cap;
  std::vector<int> cnt(N), rows;
  CUDA_OK(cudaMemcpyAsync(cnt.data(), d_cnt, (size_t)N * 4, cudaMemcpyDeviceToHost, h->stream));
  if (idx) {
    rows.resize((size_t)N * cap);
    CUDA_OK(cudaMemcpyAsync(rows.data(), d_idx, rows.size() * 4, cudaMemcpyDeviceToHost, h->stream));
  }
  int rc = read_flags(h);
  for (int ii = 0; ii < N; ++ii) {
    const int c = h->plan.perm[ii];
    const int n = std::min(cnt[ii], cap);
    row_cnt[c] = n;
    if (idx) {
      int *o = idx + (size_t)c * cap;
      for (int q = 0; q < n; ++q) o[q] = h->plan.perm[rows[(size_t)ii * cap + q]];
      std::sort(o, o + n);                       // rows ascending in the caller's index (reading R4)
      for (int q = n; q < cap; ++q) o[q] = -1;
    }
  }
  return rc;
}

int sop_device_coords(sop_handle *h, void **d_float4_out, int32_t *perm_out) {
  if (!h || !d_float4_out) return fail(SOP_E_ARG, "null argument", h);
  *d_float4_out = h->S.pos[h->cur];
  if (perm_out) memcpy(perm_out, h->plan.perm.data(), (size_t)h->S.N * 4);
  return SOP_OK;
}

#ifdef SOP_PHASE_CLOCKS
extern "C" int sop_debug_phase_clocks(sop_handle *h, float *out, int n_float4) {     // profiling builds only
  cudaStreamSynchronize(h->stream);
  return (int)cudaMemcpy(out, h->S.force, (size_t)n_float4 * 16, cudaMemcpyDeviceToHost);
}
#endif

int sop_get_config(sop_handle *h, int32_t out[12]) {
  if (!h || !out) return fail(SOP_E_ARG, "null argument", h);
  out[0] = h->plan.mode == 3 ? h->plan.res_lanes : h->plan.lanes; out[1] = h->plan.mode == 3 ? h->plan.res_block : h->plan.block; out[2] = h->plan.comp; out[3] = h->plan.mode;
  out[4] = h->plan.reorder; out[5] = h->plan.cap_nb; out[6] = h->plan.cap_pl;
  out[7] = (int32_t)(h->launches & 0xFFFFFFFFu); out[8] = (int32_t)(h->launches >> 32);
  out[9] = h->plan.mode == 3 && h->R.C > 1 ? (h->plan.res2_ok ? 2 : 1) : 0;
  if (out[9] == 2) { out[0] = R2_GS; out[1] = h->plan.res2_block; }
  out[10] = h->last_slice_len; out[11] = 0;
  return SOP_OK;
}

}  // extern "C"

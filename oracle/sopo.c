/* sopo.c -- fp64 CPU ORACLE for the SOP overdamped-Langevin hot path.  TEST INFRASTRUCTURE (see sopo.h).
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC sopo.c -o libsopo.so -lm
 * (-ffp-contract=off so that the fp32 list predicate below is three subtractions, three products and two
 *  additions, each rounded once -- DESIGN.md reading R4.)
 *
 * Everything is written in the paper's order and notation; every function cites the passage it follows.
 * OpenMP is used only where the units are independent by definition (rows of a list, trajectories of a
 * batch); the force loop is the sequential pair loop of Alg. 1.
 */
#include "sopo.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int64_t *ptr;      /* [N+1] */
  int32_t *idx;      /* [ptr[N]] rows ascending in j */
  int64_t built_at;  /* step whose coordinates the list was made from */
} csr_t;

struct sopo_handle {
  int32_t N, T;
  int32_t n_bonds;  int32_t *bond_i, *bond_j;  double *bond_r0;
  int32_t n_native; int32_t *nat_i, *nat_j;    double *nat_r0, *nat_eps;
  sopo_params p;
  unsigned char *is_fixed;        /* [N] */
  uint32_t *taus;                 /* [T][N][4] Hybrid Taus states (params.rng == 1) */
  double *kT_t;                   /* [T] temperature of every run */
  int32_t *pulled;                /* [n_pulled] */
  double *native;                 /* [N][3] promoted native coordinates (anchors of the pulled beads) */
  int64_t *excl_ptr; int32_t *excl_idx;   /* bonded + native partners of each bead, ascending */
  double *r;                      /* [T][N][3] */
  int static_l1;                  /* R_pl = +inf: one L1, made once, shared by all trajectories */
  csr_t *L1;                      /* [T] (static: only [0] used) */
  csr_t *L2;                      /* [T] */
  int64_t step;
};

static void csr_free(csr_t *c) { free(c->ptr); free(c->idx); c->ptr = NULL; c->idx = NULL; }

/* ------------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): 10 rounds; multipliers 0xD2511F53, 0xCD9E8D57;
 * key schedule increments 0x9E3779B9, 0xBB67AE85.  north_star replaces the paper's per-thread Hybrid Taus
 * state by this counter-based generator (reading R6).
 * ------------------------------------------------------------------------------------------------ */
void sopo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Noise of one bead for the update step -> step+1 (reading R6; Box-Muller).
 * counter = (bead, trajectory, step mod 2^32, step div 2^32), key = (seed lo, seed hi);
 * uniforms from the top 24 bits: u_a, u_c in (0,1], u_b, u_d in [0,1); 4 uniforms -> 4 normals, 3 used
 * ("4 normally distributed random numbers for each residue"). */
void sopo_normals(uint64_t seed, uint32_t bead, uint32_t traj, uint64_t step, double g_out[3]) {
  const double TWO_PI = 6.283185307179586476925286766559;
  uint32_t ctr[4] = { bead, traj, (uint32_t)(step & 0xFFFFFFFFu), (uint32_t)(step >> 32) };
  uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
  uint32_t x[4];
  sopo_philox4x32_10(ctr, key, x);
  double u_a = ((double)(x[0] >> 8) + 1.0) * (1.0 / 16777216.0);
  double u_b = ((double)(x[1] >> 8)) * (1.0 / 16777216.0);
  double u_c = ((double)(x[2] >> 8) + 1.0) * (1.0 / 16777216.0);
  double u_d = ((double)(x[3] >> 8)) * (1.0 / 16777216.0);
  double ra = sqrt(-2.0 * log(u_a));
  double rc = sqrt(-2.0 * log(u_c));
  g_out[0] = ra * cos(TWO_PI * u_b);
  g_out[1] = ra * sin(TWO_PI * u_b);
  g_out[2] = rc * cos(TWO_PI * u_d);
}

/* ------------------------------------------------------------------------------------------------
 * Hybrid Taus (Alg. 6): three Tausworthe components + one LCG, four 32-bit words of state per
 * bead ("one-PRNG-per-thread"), output = y1 ^ y2 ^ y3 ^ y4.  The listing's constants are garbled in PAPER.md:209
 * (c21 and c31 appear twice); reading R12 takes the taus88 / GPU Gems 3 ch. 37 set the paper cites ([49]-[51]):
 * (13, 19, 12, 4294967294), (2, 25, 4, 4294967288), (3, 11, 17, 4294967280), LCG a = 1664525, c = 1013904223.
 * ------------------------------------------------------------------------------------------------ */
uint32_t sopo_taus_step(uint32_t y[4]) {
  uint32_t b;
  b = ((y[0] << 13) ^ y[0]) >> 19;  y[0] = ((y[0] & 4294967294u) << 12) ^ b;      /* lines 6-7  */
  b = ((y[1] << 2) ^ y[1]) >> 25;   y[1] = ((y[1] & 4294967288u) << 4) ^ b;       /* lines 8-9  */
  b = ((y[2] << 3) ^ y[2]) >> 11;   y[2] = ((y[2] & 4294967280u) << 17) ^ b;      /* lines 10-11 */
  y[3] = 1664525u * y[3] + 1013904223u;                                           /* line 12 */
  return y[0] ^ y[1] ^ y[2] ^ y[3];                                               /* line 13 (before mult) */
}

/* Initial seeds of one bead's generator (Alg. 6 line 1: "initial seeds", generated on the CPU):
 * the four words of Philox4x32-10(counter = (bead, traj, 'TAUS', 0), key = seed); the Tausworthe components need
 * y1 >= 2, y2 >= 8, y3 >= 16 (L'Ecuyer), enforced by setting that bit. */
void sopo_taus_seed(uint64_t seed, uint32_t bead, uint32_t traj, uint32_t y[4]) {
  uint32_t ctr[4] = { bead, traj, 0x54415553u, 0u };
  uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
  sopo_philox4x32_10(ctr, key, y);
  y[0] |= 2u; y[1] |= 8u; y[2] |= 16u;
}

/* Three normals from four consecutive Hybrid Taus draws: the same 24-bit uniforms and Box-Muller as sopo_normals
 * (the paper's mult * x can be exactly 0, whose logarithm diverges; reading R6 keeps u_a, u_c in (0, 1]). */
static void taus_normals(uint32_t y[4], double g_out[3]) {
  const double TWO_PI = 6.283185307179586476925286766559;
  uint32_t x[4];
  for (int k = 0; k < 4; ++k) x[k] = sopo_taus_step(y);
  double u_a = ((double)(x[0] >> 8) + 1.0) * (1.0 / 16777216.0);
  double u_b = ((double)(x[1] >> 8)) * (1.0 / 16777216.0);
  double u_c = ((double)(x[2] >> 8) + 1.0) * (1.0 / 16777216.0);
  double u_d = ((double)(x[3] >> 8)) * (1.0 / 16777216.0);
  double ra = sqrt(-2.0 * log(u_a));
  double rc = sqrt(-2.0 * log(u_c));
  g_out[0] = ra * cos(TWO_PI * u_b);
  g_out[1] = ra * sin(TWO_PI * u_b);
  g_out[2] = rc * cos(TWO_PI * u_d);
}

void sopo_normals_batch(uint64_t seed, uint32_t bead0, uint32_t n_beads, uint32_t traj, uint64_t step, double *g_out) {
  for (uint32_t b = 0; b < n_beads; ++b) sopo_normals(seed, bead0 + b, traj, step, g_out + 3 * (size_t)b);
}

/* ------------------------------------------------------------------------------------------------
 * The list predicate "r < cutoff" (Alg. 3 line 9) in canonical fp32 arithmetic
 * (reading R4): coordinates rounded to binary32; d2 = ((dx*dx)+(dy*dy))+(dz*dz), every
 * operation one IEEE-754 binary32 round-to-nearest; true iff d2 < (float)(R*R).  R = +inf: always true.
 * ------------------------------------------------------------------------------------------------ */
static int pred32(const double *a, const double *b, float R2f, int always) {
  if (always) return 1;
  float ax = (float)a[0], ay = (float)a[1], az = (float)a[2];
  float bx = (float)b[0], by = (float)b[1], bz = (float)b[2];
  float dx = ax - bx;
  float dy = ay - by;
  float dz = az - bz;
  float xx = dx * dx;
  float yy = dy * dy;
  float zz = dz * dz;
  float s = xx + yy;
  float d2 = s + zz;
  return d2 < R2f;
}
static float cutoff2f(double R) { return (float)(R * R); }

int sopo_pred(const double a[3], const double b[3], double R) {
  return pred32(a, b, cutoff2f(R), isinf(R) ? 1 : 0);
}

int sopo_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------------
 * create
 * ------------------------------------------------------------------------------------------------ */
static int cmp_i32(const void *a, const void *b) {
  int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
  return (x > y) - (x < y);
}

static int is_excluded(const sopo_handle *h, int32_t i, int32_t j) {
  for (int64_t q = h->excl_ptr[i]; q < h->excl_ptr[i + 1]; ++q)
    if (h->excl_idx[q] == j) return 1;
  return 0;
}

static double dist3(const double *a, const double *b) {
  double dx = a[0] - b[0], dy = a[1] - b[1], dz = a[2] - b[2];
  return sqrt(dx * dx + dy * dy + dz * dz);
}

static int build_L1(const sopo_handle *h, const double *r, int builder, csr_t *out);
static int filter_L2(const sopo_handle *h, const double *r, const csr_t *L1, csr_t *out);
static int rebuild_all(sopo_handle *h);

int sopo_create(const sopo_topology *tp, const float *native_xyz, const sopo_params *p, int32_t n_traj,
                sopo_handle **out) {
  if (!tp || !native_xyz || !p || !out || n_traj < 1 || tp->n_beads < 1) return SOPO_E_ARG;
  const int32_t N = tp->n_beads;
  if (p->nb_interval < 1 || p->pl_interval < 1 || p->pl_interval % p->nb_interval != 0) return SOPO_E_ARG;
  if (!(p->R_nb > 0) || !(p->R_pl >= p->R_nb) || !(p->R0 > 0) || !(p->dt_over_zeta >= 0) || !(p->kT >= 0))
    return SOPO_E_ARG;

  sopo_handle *h = (sopo_handle *)calloc(1, sizeof(*h));
  h->N = N; h->T = n_traj; h->p = *p;
  h->n_bonds = tp->n_bonds; h->n_native = tp->n_native;

  /* native coordinates: fp32 input promoted to double (both sides see the same numbers) */
  h->native = (double *)malloc(sizeof(double) * 3 * (size_t)N);
  for (int64_t q = 0; q < 3 * (int64_t)N; ++q) h->native[q] = (double)native_xyz[q];

  /* r0 of bonds and natives = distance in the native structure, computed in double,
     rounded to fp32 and promoted again so that oracle and GPU use the same parameter values */
  h->bond_i = (int32_t *)malloc(sizeof(int32_t) * (size_t)(tp->n_bonds + 1));
  h->bond_j = (int32_t *)malloc(sizeof(int32_t) * (size_t)(tp->n_bonds + 1));
  h->bond_r0 = (double *)malloc(sizeof(double) * (size_t)(tp->n_bonds + 1));
  h->nat_i = (int32_t *)malloc(sizeof(int32_t) * (size_t)(tp->n_native + 1));
  h->nat_j = (int32_t *)malloc(sizeof(int32_t) * (size_t)(tp->n_native + 1));
  h->nat_r0 = (double *)malloc(sizeof(double) * (size_t)(tp->n_native + 1));
  h->nat_eps = (double *)malloc(sizeof(double) * (size_t)(tp->n_native + 1));
  int64_t *deg = (int64_t *)calloc((size_t)N + 1, sizeof(int64_t));
  int bad = 0;
  for (int32_t b = 0; b < tp->n_bonds; ++b) {
    int32_t i = tp->bonds[2 * b], j = tp->bonds[2 * b + 1];
    if (i < 0 || j >= N || i >= j) { bad = 1; break; }
    h->bond_i[b] = i; h->bond_j[b] = j;
    h->bond_r0[b] = (double)(float)dist3(h->native + 3 * (size_t)i, h->native + 3 * (size_t)j);
    deg[i]++; deg[j]++;
  }
  for (int32_t c = 0; c < tp->n_native && !bad; ++c) {
    int32_t i = tp->native[2 * c], j = tp->native[2 * c + 1];
    if (i < 0 || j >= N || i >= j) { bad = 1; break; }
    h->nat_i[c] = i; h->nat_j[c] = j;
    h->nat_r0[c] = (double)(float)dist3(h->native + 3 * (size_t)i, h->native + 3 * (size_t)j);
    h->nat_eps[c] = tp->native_eps ? tp->native_eps[c] : p->eps_native;
    deg[i]++; deg[j]++;
  }
  /* exclusion rows = bonded and native partners (they are not in the non-native set, Eq. (1) Delta_ij) */
  h->excl_ptr = (int64_t *)calloc((size_t)N + 1, sizeof(int64_t));
  for (int32_t i = 0; i < N; ++i) h->excl_ptr[i + 1] = h->excl_ptr[i] + deg[i];
  h->excl_idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(h->excl_ptr[N] + 1));
  memset(deg, 0, sizeof(int64_t) * ((size_t)N + 1));
  if (!bad) {
    for (int32_t b = 0; b < tp->n_bonds; ++b) {
      int32_t i = h->bond_i[b], j = h->bond_j[b];
      h->excl_idx[h->excl_ptr[i] + deg[i]++] = j;
      h->excl_idx[h->excl_ptr[j] + deg[j]++] = i;
    }
    for (int32_t c = 0; c < tp->n_native; ++c) {
      int32_t i = h->nat_i[c], j = h->nat_j[c];
      h->excl_idx[h->excl_ptr[i] + deg[i]++] = j;
      h->excl_idx[h->excl_ptr[j] + deg[j]++] = i;
    }
    for (int32_t i = 0; i < N && !bad; ++i) {
      int64_t a = h->excl_ptr[i], n = h->excl_ptr[i + 1] - a;
      qsort(h->excl_idx + a, (size_t)n, sizeof(int32_t), cmp_i32);
      for (int64_t q = 1; q < n; ++q)
        if (h->excl_idx[a + q] == h->excl_idx[a + q - 1]) bad = 1;   /* duplicate pair or bond that is also native */
    }
  }
  free(deg);

  h->is_fixed = (unsigned char *)calloc((size_t)N, 1);
  for (int32_t q = 0; q < p->n_fixed && !bad; ++q) {
    if (p->fixed[q] < 0 || p->fixed[q] >= N) bad = 1; else h->is_fixed[p->fixed[q]] = 1;
  }
  h->pulled = (int32_t *)malloc(sizeof(int32_t) * (size_t)(p->n_pulled + 1));
  for (int32_t q = 0; q < p->n_pulled && !bad; ++q) {
    if (p->pulled[q] < 0 || p->pulled[q] >= N) bad = 1; else h->pulled[q] = p->pulled[q];
  }
  h->p.fixed = NULL; h->p.pulled = h->pulled;

  h->r = (double *)malloc(sizeof(double) * 3 * (size_t)N * (size_t)n_traj);
  h->kT_t = (double *)malloc(sizeof(double) * (size_t)n_traj);
  for (int32_t t = 0; t < n_traj; ++t) h->kT_t[t] = p->kT_per_traj ? p->kT_per_traj[t] : p->kT;
  h->p.kT_per_traj = NULL;
  h->taus = NULL;
  if (p->rng == 1) {
    h->taus = (uint32_t *)malloc(sizeof(uint32_t) * 4 * (size_t)N * (size_t)n_traj);
    for (int32_t t = 0; t < n_traj; ++t)
      for (int32_t i = 0; i < N; ++i)
        sopo_taus_seed(p->seed, (uint32_t)i, (uint32_t)(p->traj_offset + t), h->taus + 4 * ((size_t)N * (size_t)t + (size_t)i));
  }
  h->L1 = (csr_t *)calloc((size_t)n_traj, sizeof(csr_t));
  h->L2 = (csr_t *)calloc((size_t)n_traj, sizeof(csr_t));
  h->static_l1 = isinf(p->R_pl) ? 1 : 0;
  if (bad) { sopo_destroy(h); return SOPO_E_ARG; }

  /* every trajectory starts from the native structure (the paper starts from the PDB structure) */
  for (int32_t t = 0; t < n_traj; ++t) memcpy(h->r + 3 * (size_t)N * (size_t)t, h->native, sizeof(double) * 3 * (size_t)N);
  h->step = 0;
  int rc = rebuild_all(h);
  if (rc) { sopo_destroy(h); return rc; }
  *out = h;
  return SOPO_OK;
}

void sopo_destroy(sopo_handle *h) {
  if (!h) return;
  free(h->bond_i); free(h->bond_j); free(h->bond_r0);
  free(h->nat_i); free(h->nat_j); free(h->nat_r0); free(h->nat_eps);
  free(h->taus); free(h->kT_t); free(h->is_fixed); free(h->pulled); free(h->native); free(h->excl_ptr); free(h->excl_idx); free(h->r);
  if (h->L1) for (int32_t t = 0; t < h->T; ++t) csr_free(&h->L1[t]);
  if (h->L2) for (int32_t t = 0; t < h->T; ++t) csr_free(&h->L2[t]);
  free(h->L1); free(h->L2);
  free(h);
}

/* ------------------------------------------------------------------------------------------------
 * L1 "pair list" = PossiblePairsMap (PAPER.md:107, :126; cutoff-limited for big systems, :440):
 * row i = ascending j != i, (i,j) in the non-native set, pred(i,j,R_pl).
 * builder 0: brute force over all j -- the definition.  builder 1: the oracle's own cell list, which only
 * narrows the candidate set (cell edge > R_pl) and then sorts; tests prove it identical to builder 0.
 * ------------------------------------------------------------------------------------------------ */
static void rows_to_csr(int32_t N, int32_t **rows, const int32_t *cnt, csr_t *out) {
  csr_free(out);
  out->ptr = (int64_t *)malloc(sizeof(int64_t) * ((size_t)N + 1));
  out->ptr[0] = 0;
  for (int32_t i = 0; i < N; ++i) out->ptr[i + 1] = out->ptr[i] + cnt[i];
  out->idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(out->ptr[N] + 1));
  for (int32_t i = 0; i < N; ++i) {
    memcpy(out->idx + out->ptr[i], rows[i], sizeof(int32_t) * (size_t)cnt[i]);
    free(rows[i]);
  }
}

static int build_L1(const sopo_handle *h, const double *r, int builder, csr_t *out) {
  const int32_t N = h->N;
  const int always = isinf(h->p.R_pl) ? 1 : 0;
  const float R2f = cutoff2f(h->p.R_pl);
  int32_t **rows = (int32_t **)calloc((size_t)N, sizeof(int32_t *));
  int32_t *cnt = (int32_t *)calloc((size_t)N, sizeof(int32_t));

  if (builder == 0 || always) {
#pragma omp parallel
    {
      int32_t *tmp = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
#pragma omp for schedule(dynamic, 64)
      for (int32_t i = 0; i < N; ++i) {
        int32_t n = 0;
        for (int32_t j = 0; j < N; ++j) {
          if (j == i) continue;
          if (!pred32(r + 3 * (size_t)i, r + 3 * (size_t)j, R2f, always)) continue;
          if (is_excluded(h, i, j)) continue;
          tmp[n++] = j;
        }
        rows[i] = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n + 1));
        memcpy(rows[i], tmp, sizeof(int32_t) * (size_t)n);
        cnt[i] = n;
      }
      free(tmp);
    }
  } else {
    /* cell list over the fp32-rounded coordinates; edge 0.1 % wider than R_pl so that any pair passing
       pred32 lies in adjacent cells whatever the rounding */
    double lo[3] = { 1e300, 1e300, 1e300 }, hi[3] = { -1e300, -1e300, -1e300 };
    for (int32_t i = 0; i < N; ++i)
      for (int a = 0; a < 3; ++a) {
        double v = (double)(float)r[3 * (size_t)i + a];
        if (v < lo[a]) lo[a] = v;
        if (v > hi[a]) hi[a] = v;
      }
    const double edge = h->p.R_pl * 1.001;
    int32_t nc[3];
    for (int a = 0; a < 3; ++a) {
      nc[a] = (int32_t)floor((hi[a] - lo[a]) / edge) + 1;
      if (nc[a] < 1) nc[a] = 1;
    }
    const int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
    int64_t *cstart = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
    int64_t *cell_of = (int64_t *)malloc(sizeof(int64_t) * (size_t)N);
    for (int32_t i = 0; i < N; ++i) {
      int64_t c[3];
      for (int a = 0; a < 3; ++a) {
        c[a] = (int64_t)floor(((double)(float)r[3 * (size_t)i + a] - lo[a]) / edge);
        if (c[a] >= nc[a]) c[a] = nc[a] - 1;
      }
      cell_of[i] = (c[2] * nc[1] + c[1]) * nc[0] + c[0];
      cstart[cell_of[i] + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) cstart[c + 1] += cstart[c];
    int32_t *cbead = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    int64_t *fill = (int64_t *)calloc((size_t)ncell, sizeof(int64_t));
    for (int32_t i = 0; i < N; ++i) { int64_t c = cell_of[i]; cbead[cstart[c] + fill[c]++] = i; }
    free(fill);
#pragma omp parallel
    {
      int32_t cap = 1024, *tmp = (int32_t *)malloc(sizeof(int32_t) * (size_t)cap);
#pragma omp for schedule(dynamic, 64)
      for (int32_t i = 0; i < N; ++i) {
        int32_t n = 0;
        int64_t ci = cell_of[i];
        int64_t cx = ci % nc[0], cy = (ci / nc[0]) % nc[1], cz = ci / ((int64_t)nc[0] * nc[1]);
        for (int64_t z = cz - 1; z <= cz + 1; ++z) {
          if (z < 0 || z >= nc[2]) continue;
          for (int64_t y = cy - 1; y <= cy + 1; ++y) {
            if (y < 0 || y >= nc[1]) continue;
            for (int64_t x = cx - 1; x <= cx + 1; ++x) {
              if (x < 0 || x >= nc[0]) continue;
              int64_t c = (z * nc[1] + y) * nc[0] + x;
              for (int64_t q = cstart[c]; q < cstart[c + 1]; ++q) {
                int32_t j = cbead[q];
                if (j == i) continue;
                if (!pred32(r + 3 * (size_t)i, r + 3 * (size_t)j, R2f, 0)) continue;
                if (is_excluded(h, i, j)) continue;
                if (n == cap) { cap *= 2; tmp = (int32_t *)realloc(tmp, sizeof(int32_t) * (size_t)cap); }
                tmp[n++] = j;
              }
            }
          }
        }
        qsort(tmp, (size_t)n, sizeof(int32_t), cmp_i32);
        rows[i] = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n + 1));
        memcpy(rows[i], tmp, sizeof(int32_t) * (size_t)n);
        cnt[i] = n;
      }
      free(tmp);
    }
    free(cstart); free(cell_of); free(cbead);
  }
  rows_to_csr(N, rows, cnt, out);
  free(rows); free(cnt);
  return SOPO_OK;
}

/* L2 "neighbor list" = PairsMap regenerated by Alg. 3: scan row i of L1 in order, copy
 * the entries with r < cutoff (lines 9-11), store the count (line 14). */
static int filter_L2(const sopo_handle *h, const double *r, const csr_t *L1, csr_t *out) {
  const int32_t N = h->N;
  const float R2f = cutoff2f(h->p.R_nb);
  int32_t **rows = (int32_t **)calloc((size_t)N, sizeof(int32_t *));
  int32_t *cnt = (int32_t *)calloc((size_t)N, sizeof(int32_t));
#pragma omp parallel for schedule(dynamic, 256)
  for (int32_t i = 0; i < N; ++i) {                                   /* line 1: i <- thread index */
    int64_t a = L1->ptr[i], P = L1->ptr[i + 1] - a;                   /* line 4 */
    int32_t *row = (int32_t *)malloc(sizeof(int32_t) * (size_t)(P + 1));
    int32_t p_i = 0;                                                  /* line 2 */
    for (int64_t pp = 0; pp < P; ++pp) {                              /* line 5 */
      int32_t j = L1->idx[a + pp];                                    /* line 6 */
      if (pred32(r + 3 * (size_t)i, r + 3 * (size_t)j, R2f, 0))       /* lines 7-9 */
        row[p_i++] = j;                                               /* lines 10-11 */
    }
    rows[i] = row; cnt[i] = p_i;                                      /* line 14 */
  }
  rows_to_csr(N, rows, cnt, out);
  free(rows); free(cnt);
  return SOPO_OK;
}

static int rebuild_all(sopo_handle *h) {
  const size_t stride = 3 * (size_t)h->N;
  for (int32_t t = 0; t < h->T; ++t) {
    const csr_t *L1;
    if (h->static_l1) {
      if (t == 0) { build_L1(h, h->r, 0, &h->L1[0]); h->L1[0].built_at = h->step; }
      L1 = &h->L1[0];
    } else {
      build_L1(h, h->r + stride * t, h->p.list_builder, &h->L1[t]);
      h->L1[t].built_at = h->step;
      L1 = &h->L1[t];
    }
    filter_L2(h, h->r + stride * t, L1, &h->L2[t]);
    h->L2[t].built_at = h->step;
  }
  return SOPO_OK;
}

/* ------------------------------------------------------------------------------------------------
 * Energies and forces.  Alg. 1: for every pair once, df = force(r_i - r_j, par),
 * f[i] += df, f[j] -= df.  Force laws are -dV/dr of Eq. (1):
 *   FENE    V = -(k/2) R0^2 ln(1 - (r - r0)^2/R0^2)          f = -k d/(1 - d^2/R0^2) * rvec/r,  d = r - r0
 *   native  V = eps [(r0/r)^12 - 2 (r0/r)^6]                  f = (12 eps/r^2)(q^2 - q) * rvec,  q = (r0/r)^6
 *   repuls. V = eps_r (sigma/r)^6 over the L2 pairs           f = (6 eps_r/r^2)(sigma/r)^6 * rvec
 * There is no distance test inside the force loop (Alg. 2 has none; reading R3c).
 * External terms (readings R7, R8): cantilever spring on the pulled beads, spherical indenter.
 * e[6] = fene, native, rep, pull, tip, total.  f may be NULL.
 * ------------------------------------------------------------------------------------------------ */
static int eval(const sopo_handle *h, const double *r, const csr_t *L2, int64_t step, double *e, double *f) {
  const int32_t N = h->N;
  const sopo_params *p = &h->p;
  int status = SOPO_OK;
  double e_fene = 0, e_nat = 0, e_rep = 0, e_pull = 0, e_tip = 0;
  if (f) memset(f, 0, sizeof(double) * 3 * (size_t)N);

  for (int32_t b = 0; b < h->n_bonds; ++b) {                    /* first term of Eq. (1) */
    int32_t i = h->bond_i[b], j = h->bond_j[b];
    double d[3] = { r[3 * (size_t)i] - r[3 * (size_t)j], r[3 * (size_t)i + 1] - r[3 * (size_t)j + 1],
                    r[3 * (size_t)i + 2] - r[3 * (size_t)j + 2] };
    double rr = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double del = rr - h->bond_r0[b];
    double x = 1.0 - del * del / (p->R0 * p->R0);
    if (!(x > 0.0)) { status = SOPO_E_FENE; continue; }         /* |r - r0| >= R0: log of a non-positive number */
    e_fene += -0.5 * p->k_fene * p->R0 * p->R0 * log(x);
    if (f) {
      double s = -p->k_fene * del / x / rr;
      for (int a = 0; a < 3; ++a) { f[3 * (size_t)i + a] += s * d[a]; f[3 * (size_t)j + a] -= s * d[a]; }
    }
  }
  for (int32_t c = 0; c < h->n_native; ++c) {                   /* second term of Eq. (1) */
    int32_t i = h->nat_i[c], j = h->nat_j[c];
    double d[3] = { r[3 * (size_t)i] - r[3 * (size_t)j], r[3 * (size_t)i + 1] - r[3 * (size_t)j + 1],
                    r[3 * (size_t)i + 2] - r[3 * (size_t)j + 2] };
    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    double rr = sqrt(r2);
    double q = pow(h->nat_r0[c] / rr, 6.0);
    e_nat += h->nat_eps[c] * (q * q - 2.0 * q);
    if (f) {
      double s = 12.0 * h->nat_eps[c] / r2 * (q * q - q);
      for (int a = 0; a < 3; ++a) { f[3 * (size_t)i + a] += s * d[a]; f[3 * (size_t)j + a] -= s * d[a]; }
    }
  }
  for (int32_t i = 0; i < N; ++i) {                             /* third + fourth terms, over the L2 pairs */
    for (int64_t q = L2->ptr[i]; q < L2->ptr[i + 1]; ++q) {
      int32_t j = L2->idx[q];
      if (j < i) continue;                                      /* every pair once (Alg. 1) */
      double d[3] = { r[3 * (size_t)i] - r[3 * (size_t)j], r[3 * (size_t)i + 1] - r[3 * (size_t)j + 1],
                      r[3 * (size_t)i + 2] - r[3 * (size_t)j + 2] };
      double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
      double rr = sqrt(r2);
      double s6 = pow(p->sigma / rr, 6.0);
      e_rep += p->eps_rep * s6;
      if (f) {
        double s = 6.0 * p->eps_rep / r2 * s6;
        for (int a = 0; a < 3; ++a) { f[3 * (size_t)i + a] += s * d[a]; f[3 * (size_t)j + a] -= s * d[a]; }
      }
    }
  }
  /* cantilever spring (reading R7): the spring base moves v*step along n from the bead's native
     position a_p;  V = (kappa/2)(v s - (r_p - a_p).n)^2,  f = kappa (v s - (r_p - a_p).n) n */
  for (int32_t k = 0; k < p->n_pulled; ++k) {
    int32_t i = h->pulled[k];
    double proj = 0;
    for (int a = 0; a < 3; ++a) proj += (r[3 * (size_t)i + a] - h->native[3 * (size_t)i + a]) * p->pull_dir[a];
    double ext = p->pull_v * (double)step - proj;
    e_pull += 0.5 * p->pull_k * ext * ext;
    if (f) for (int a = 0; a < 3; ++a) f[3 * (size_t)i + a] += p->pull_k * ext * p->pull_dir[a];
  }
  /* indenter sphere (reading R8; the paper names indentation, and gives no formula):
     centre c = c0 + v_tip*step*n_tip;  V = eps_t (sigma_t/(g - R_tip))^6,  g = |r_i - c| */
  if (p->tip_on) {
    double c[3];
    for (int a = 0; a < 3; ++a) c[a] = p->tip_c0[a] + p->tip_v * (double)step * p->tip_dir[a];
    for (int32_t i = 0; i < N; ++i) {
      double d[3] = { r[3 * (size_t)i] - c[0], r[3 * (size_t)i + 1] - c[1], r[3 * (size_t)i + 2] - c[2] };
      double g = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
      double gap = g - p->tip_R;
      if (!(gap > 0.0)) { status = SOPO_E_NONFINITE; continue; }
      double s6 = pow(p->tip_sigma / gap, 6.0);
      e_tip += p->tip_eps * s6;
      if (f) {
        double s = 6.0 * p->tip_eps * s6 / gap / g;
        for (int a = 0; a < 3; ++a) f[3 * (size_t)i + a] += s * d[a];
      }
    }
  }
  if (e) { e[0] = e_fene; e[1] = e_nat; e[2] = e_rep; e[3] = e_pull; e[4] = e_tip;
           e[5] = e_fene + e_nat + e_rep + e_pull + e_tip; }
  return status;
}

/* ------------------------------------------------------------------------------------------------
 * One update step of one trajectory: Alg. 7.
 *   line 3: f_i = sum of the pair forces;  line 4: g_i = 3 normals;
 *   line 5: r_i <- r_i + f_i h/xi + g_i sqrt(2 kT h/xi);  h/xi = dt_over_zeta.
 * All beads move from forces at the old coordinates (two time layers); fixed beads stay
 * ("fixing the N-terminal end").
 * ------------------------------------------------------------------------------------------------ */
static int step_one(sopo_handle *h, int32_t t, int64_t step, double *fbuf) {
  const int32_t N = h->N;
  double *r = h->r + 3 * (size_t)N * (size_t)t;
  int status = eval(h, r, &h->L2[t], step, NULL, fbuf);
  const double D = h->p.dt_over_zeta;
  const double amp = sqrt(2.0 * h->kT_t[t] * D);
  if (h->p.integrator == 2) {
    /* Second order (reading R14).  Eq. (5) is the mean recursion of the predictor-corrector
     *   r' = r + f(r, t_n) h/xi + G,   r(t_n + h) = r + (h / 2 xi) [f(r, t_n) + f(r', t_n)] + G
     * (for the paper's f = r_f t_n - K_sp X:  X + (r_f t_n/xi - X/tau) h + (X/(2 tau^2) - r_f t_n/(2 tau xi)) h^2), with the
     * same random displacement G = g sqrt(2 kT h/xi) in both stages and the lists, the pulling spring and the indenter at
     * t_n in both force evaluations. */
    double *rp = (double *)malloc(sizeof(double) * 3 * (size_t)N), *gs = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *f2 = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    for (int32_t i = 0; i < N; ++i) {
      double g[3] = { 0, 0, 0 };
      if (!h->is_fixed[i]) sopo_normals(h->p.seed, (uint32_t)i, (uint32_t)(h->p.traj_offset + t), (uint64_t)step, g);
      for (int a = 0; a < 3; ++a) {
        gs[3 * (size_t)i + a] = g[a];
        rp[3 * (size_t)i + a] = h->is_fixed[i] ? r[3 * (size_t)i + a] : r[3 * (size_t)i + a] + D * fbuf[3 * (size_t)i + a] + amp * g[a];
      }
    }
    int rc = eval(h, rp, &h->L2[t], step, NULL, f2);
    if (rc && !status) status = rc;
    for (int32_t i = 0; i < N; ++i) {
      if (h->is_fixed[i]) continue;
      for (int a = 0; a < 3; ++a) {
        double v = r[3 * (size_t)i + a] + 0.5 * D * (fbuf[3 * (size_t)i + a] + f2[3 * (size_t)i + a]) + amp * gs[3 * (size_t)i + a];
        if (!isfinite(v)) status = status ? status : SOPO_E_NONFINITE;
        r[3 * (size_t)i + a] = v;
      }
    }
    free(rp); free(gs); free(f2);
    return status;
  }
  for (int32_t i = 0; i < N; ++i) {
    if (h->is_fixed[i]) continue;
    double g[3];
    if (h->p.rng == 1) taus_normals(h->taus + 4 * ((size_t)N * (size_t)t + (size_t)i), g);   /* state read, 4 draws, state written back */
    else sopo_normals(h->p.seed, (uint32_t)i, (uint32_t)(h->p.traj_offset + t), (uint64_t)step, g);
    for (int a = 0; a < 3; ++a) {
      double v = r[3 * (size_t)i + a] + D * fbuf[3 * (size_t)i + a] + amp * g[a];
      if (!isfinite(v)) status = status ? status : SOPO_E_NONFINITE;
      r[3 * (size_t)i + a] = v;
    }
  }
  return status;
}

/* ------------------------------------------------------------------------------------------------
 * NEXT-4: replica exchange (the many-runs-per-GPU approach "in conjunction with parallel tempering
 * algorithms, including variants of the Replica Exchange Method").  Two runs at inverse temperatures b_i, b_j and
 * potential energies E_i, E_j swap temperatures with the Metropolis probability min(1, exp((b_i - b_j)(E_i - E_j))):
 * the ratio of the Boltzmann weights of the swapped and the unswapped pair, exp(-b_i E_j - b_j E_i) / exp(-b_i E_i - b_j E_j).
 * ------------------------------------------------------------------------------------------------ */
double sopo_rex_probability(double E_i, double E_j, double kT_i, double kT_j) {
  double d = (1.0 / kT_i - 1.0 / kT_j) * (E_i - E_j);
  return d >= 0.0 ? 1.0 : exp(d);
}
int sopo_rex_accept(double E_i, double E_j, double kT_i, double kT_j, double u) {
  return u <= sopo_rex_probability(E_i, E_j, kT_i, kT_j) ? 1 : 0;      /* u in (0, 1]: probability 1 always accepts */
}

int sopo_replica_exchange(sopo_handle *h, int32_t parity, uint64_t sweep, int32_t *accepted) {
  if (!h || (parity != 0 && parity != 1)) return SOPO_E_ARG;
  int status = SOPO_OK;
  for (int32_t t = parity; t + 1 < h->T; t += 2) {
    double e_i[6], e_j[6];
    int rc = eval(h, h->r + 3 * (size_t)h->N * (size_t)t, &h->L2[t], h->step, e_i, NULL);
    if (rc && !status) status = rc;
    rc = eval(h, h->r + 3 * (size_t)h->N * (size_t)(t + 1), &h->L2[t + 1], h->step, e_j, NULL);
    if (rc && !status) status = rc;
    uint32_t ctr[4] = { (uint32_t)(h->p.traj_offset + t), 0x52455821u, (uint32_t)(sweep & 0xFFFFFFFFu), (uint32_t)(sweep >> 32) };
    uint32_t key[2] = { (uint32_t)(h->p.seed & 0xFFFFFFFFu), (uint32_t)(h->p.seed >> 32) }, x[4];
    sopo_philox4x32_10(ctr, key, x);
    double u = ((double)(x[0] >> 8) + 1.0) * (1.0 / 16777216.0);
    int acc = sopo_rex_accept(e_i[5], e_j[5], h->kT_t[t], h->kT_t[t + 1], u);
    if (acc) { double tmp = h->kT_t[t]; h->kT_t[t] = h->kT_t[t + 1]; h->kT_t[t + 1] = tmp; }
    if (accepted) accepted[t / 2] = acc;
  }
  return status;
}

int sopo_get_temperatures(sopo_handle *h, double *kT_out) {
  if (!h || !kT_out) return SOPO_E_ARG;
  memcpy(kT_out, h->kT_t, sizeof(double) * (size_t)h->T);
  return SOPO_OK;
}

/* Schedule: after the update that makes step = s, if s % pl_interval == 0 the
 * L1 is rebuilt from the new coordinates, and if s % nb_interval == 0 the L2 is re-filtered (after the L1). */
int sopo_run(sopo_handle *h, int64_t n_steps) {
  if (!h || n_steps < 0) return SOPO_E_ARG;
  const int32_t N = h->N, T = h->T;
  int status = SOPO_OK;
#pragma omp parallel for schedule(dynamic, 1) if (T > 1)
  for (int32_t t = 0; t < T; ++t) {
    double *fbuf = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *r = h->r + 3 * (size_t)N * (size_t)t;
    int st = SOPO_OK;
    for (int64_t n = 0; n < n_steps; ++n) {
      int64_t s = h->step + n;
      int rc = step_one(h, t, s, fbuf);
      if (rc && !st) st = rc;
      int64_t s1 = s + 1;
      if (!h->static_l1 && s1 % h->p.pl_interval == 0) {
        build_L1(h, r, h->p.list_builder, &h->L1[t]);
        h->L1[t].built_at = s1;
      }
      if (s1 % h->p.nb_interval == 0) {
        filter_L2(h, r, h->static_l1 ? &h->L1[0] : &h->L1[t], &h->L2[t]);
        h->L2[t].built_at = s1;
      }
    }
    free(fbuf);
    if (st) {
#pragma omp critical
      if (!status) status = st;
    }
  }
  h->step += n_steps;
  return status;
}

int sopo_get_coords(sopo_handle *h, double *xyz_out) {
  if (!h || !xyz_out) return SOPO_E_ARG;
  memcpy(xyz_out, h->r, sizeof(double) * 3 * (size_t)h->N * (size_t)h->T);
  return SOPO_OK;
}

int sopo_set_coords(sopo_handle *h, const double *xyz) {
  if (!h || !xyz) return SOPO_E_ARG;
  memcpy(h->r, xyz, sizeof(double) * 3 * (size_t)h->N * (size_t)h->T);
  return rebuild_all(h);
}

int sopo_get_step(sopo_handle *h, int64_t *step) { if (!h || !step) return SOPO_E_ARG; *step = h->step; return SOPO_OK; }
int sopo_set_step(sopo_handle *h, int64_t step) { if (!h || step < 0) return SOPO_E_ARG; h->step = step; return SOPO_OK; }

int sopo_get_energies(sopo_handle *h, double *e_out) {
  if (!h || !e_out) return SOPO_E_ARG;
  int status = SOPO_OK;
  for (int32_t t = 0; t < h->T; ++t) {
    int rc = eval(h, h->r + 3 * (size_t)h->N * (size_t)t, &h->L2[t], h->step, e_out + 6 * (size_t)t, NULL);
    if (rc && !status) status = rc;
  }
  return status;
}

/* Observables the paper's applications plot (PAPER.md:261 force-extension curves f(R), Fig. 3; :312-314
 * force-indentation), per trajectory, plain definitions:
 *   o[0] = Rg   = sqrt( (1/N) sum_i |r_i - r_cm|^2 ),  r_cm = (1/N) sum_i r_i
 *   o[1] = X    = |r_b - r_a|,  a = first fixed bead (else bead 0), b = first pulled bead (else bead N-1)
 *   o[2] = f    = sum over pulled beads of kappa (v s - (r_p - a_p).n)      (cantilever force; = r_f t at zero
 *                 displacement, r_f = kappa v)
 *   o[3] = f_tip = sum_i F_i^tip . n_tip = dV_tip / d(advance)              (force resisting the indenter, reading R8) */
int sopo_get_observables(sopo_handle *h, double *o_out) {
  if (!h || !o_out) return SOPO_E_ARG;
  const sopo_params *p = &h->p;
  const int32_t N = h->N;
  int32_t a = 0, b = N - 1;
  for (int32_t i = 0; i < N; ++i) if (h->is_fixed[i]) { a = i; break; }
  if (p->n_pulled > 0) b = h->pulled[0];
  for (int32_t t = 0; t < h->T; ++t) {
    const double *r = h->r + 3 * (size_t)N * (size_t)t;
    double *o = o_out + 4 * (size_t)t;
    double cm[3] = {0, 0, 0};
    for (int32_t i = 0; i < N; ++i) for (int k = 0; k < 3; ++k) cm[k] += r[3 * (size_t)i + k];
    for (int k = 0; k < 3; ++k) cm[k] /= (double)N;
    double s2 = 0;
    for (int32_t i = 0; i < N; ++i) for (int k = 0; k < 3; ++k) { double d = r[3 * (size_t)i + k] - cm[k]; s2 += d * d; }
    o[0] = sqrt(s2 / (double)N);
    double x2 = 0;
    for (int k = 0; k < 3; ++k) { double d = r[3 * (size_t)b + k] - r[3 * (size_t)a + k]; x2 += d * d; }
    o[1] = sqrt(x2);
    double f = 0;
    for (int32_t q = 0; q < p->n_pulled; ++q) {
      int32_t i = h->pulled[q];
      double proj = 0;
      for (int k = 0; k < 3; ++k) proj += (r[3 * (size_t)i + k] - h->native[3 * (size_t)i + k]) * p->pull_dir[k];
      f += p->pull_k * (p->pull_v * (double)h->step - proj);
    }
    o[2] = f;
    double ft = 0;
    if (p->tip_on) {
      double c[3];
      for (int k = 0; k < 3; ++k) c[k] = p->tip_c0[k] + p->tip_v * (double)h->step * p->tip_dir[k];
      for (int32_t i = 0; i < N; ++i) {
        double d[3], g2 = 0, dn = 0;
        for (int k = 0; k < 3; ++k) { d[k] = r[3 * (size_t)i + k] - c[k]; g2 += d[k] * d[k]; dn += d[k] * p->tip_dir[k]; }
        double g = sqrt(g2), gap = g - p->tip_R;
        if (!(gap > 0)) return SOPO_E_NONFINITE;
        ft += 6.0 * p->tip_eps * pow(p->tip_sigma / gap, 6.0) / gap / g * dn;
      }
    }
    o[3] = ft;
  }
  return SOPO_OK;
}

int sopo_get_forces(sopo_handle *h, double *f_out) {
  if (!h || !f_out) return SOPO_E_ARG;
  int status = SOPO_OK;
  for (int32_t t = 0; t < h->T; ++t) {
    size_t off = 3 * (size_t)h->N * (size_t)t;
    int rc = eval(h, h->r + off, &h->L2[t], h->step, NULL, f_out + off);
    if (rc && !status) status = rc;
  }
  return status;
}

int sopo_eval_frozen(sopo_handle *h, int32_t traj, const double *xyz, int64_t step, double *e_out, double *f_out) {
  if (!h || !xyz || traj < 0 || traj >= h->T) return SOPO_E_ARG;
  return eval(h, xyz, &h->L2[traj], step, e_out, f_out);
}

static int csr_to_rows(const csr_t *L, int32_t N, int32_t *row_cnt, int32_t *idx, int32_t cap) {
  for (int32_t i = 0; i < N; ++i) {
    int64_t n = L->ptr[i + 1] - L->ptr[i];
    if (n > cap) return SOPO_E_CAP;
    row_cnt[i] = (int32_t)n;
    memcpy(idx + (size_t)i * (size_t)cap, L->idx + L->ptr[i], sizeof(int32_t) * (size_t)n);
  }
  return SOPO_OK;
}

int sopo_get_lists(sopo_handle *h, int32_t traj, int32_t level, int32_t *row_cnt, int32_t *idx, int32_t cap,
                   int64_t *built_at_step) {
  if (!h || traj < 0 || traj >= h->T || (level != 1 && level != 2) || !row_cnt || !idx) return SOPO_E_ARG;
  const csr_t *L = level == 1 ? (h->static_l1 ? &h->L1[0] : &h->L1[traj]) : &h->L2[traj];
  if (built_at_step) *built_at_step = L->built_at;
  return csr_to_rows(L, h->N, row_cnt, idx, cap);
}

int sopo_max_row(sopo_handle *h, int32_t traj, int32_t level, int32_t *max_cnt) {
  if (!h || traj < 0 || traj >= h->T || (level != 1 && level != 2) || !max_cnt) return SOPO_E_ARG;
  const csr_t *L = level == 1 ? (h->static_l1 ? &h->L1[0] : &h->L1[traj]) : &h->L2[traj];
  int64_t m = 0;
  for (int32_t i = 0; i < h->N; ++i) { int64_t n = L->ptr[i + 1] - L->ptr[i]; if (n > m) m = n; }
  *max_cnt = (int32_t)m;
  return SOPO_OK;
}

int sopo_build_lists(sopo_handle *h, const double *xyz, int32_t level, int32_t builder, int32_t *row_cnt,
                     int32_t *idx, int32_t cap) {
  if (!h || !xyz || (level != 1 && level != 2) || !row_cnt || !idx) return SOPO_E_ARG;
  csr_t L1 = { 0 }, L2 = { 0 };
  build_L1(h, xyz, builder, &L1);
  int rc;
  if (level == 1) rc = csr_to_rows(&L1, h->N, row_cnt, idx, cap);
  else { filter_L2(h, xyz, &L1, &L2); rc = csr_to_rows(&L2, h->N, row_cnt, idx, cap); }
  csr_free(&L1); csr_free(&L2);
  return rc;
}

int sopo_filter(sopo_handle *h, const double *xyz, const int32_t *l1_cnt, const int32_t *l1_idx, int32_t cap1,
                int32_t *row_cnt, int32_t *idx, int32_t cap2) {
  if (!h || !xyz || !l1_cnt || !l1_idx || !row_cnt || !idx) return SOPO_E_ARG;
  const int32_t N = h->N;
  csr_t L1 = { 0 }, L2 = { 0 };
  L1.ptr = (int64_t *)malloc(sizeof(int64_t) * ((size_t)N + 1));
  L1.ptr[0] = 0;
  for (int32_t i = 0; i < N; ++i) L1.ptr[i + 1] = L1.ptr[i] + l1_cnt[i];
  L1.idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(L1.ptr[N] + 1));
  for (int32_t i = 0; i < N; ++i)
    memcpy(L1.idx + L1.ptr[i], l1_idx + (size_t)i * (size_t)cap1, sizeof(int32_t) * (size_t)l1_cnt[i]);
  filter_L2(h, xyz, &L1, &L2);
  int rc = csr_to_rows(&L2, N, row_cnt, idx, cap2);
  csr_free(&L1); csr_free(&L2);
  return rc;
}

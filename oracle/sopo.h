/* sopo.h -- fp64 CPU ORACLE for the SOP overdamped-Langevin hot path.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this.  It shares no code with the CUDA path (paper_1003_1148_b200/csrc,
 * include/sop.h): no header, no table, no helper.  Plain sequential C99 in double precision, written from the
 * paper (PAPER.md = arxiv 1003.1148) in the paper's order:
 *
 *   forces   : Alg. 1 pair loop with the force laws -dV/dr of Eq. (1)
 *   lists    : Alg. 3 -- L2 = entries of the L1 row with r < cutoff, in order;
 *              L1 ("PossiblePairsMap") by brute force over all j
 *   noise    : Box-Muller on a counter-based Philox4x32-10 stream (north_star; R6)
 *   update   : Alg. 7 line 5  r += f h/xi + g sqrt(2 kT h/xi)
 *   energies : Eq. (1) term by term
 *
 * Pins (tests/test_oracle_pins.py): see DESIGN.md "Oracle pins".  Parity-unpinned by the paper: the indenter
 * force law (the paper gives no formula; reading R8) -- pinned only by F = -grad V self-consistency.
 */
#ifndef SOPO_H
#define SOPO_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sopo_handle sopo_handle;

typedef struct {
  int32_t n_beads;
  int32_t n_bonds;  const int32_t *bonds;      /* [n_bonds][2]  i<j */
  int32_t n_native; const int32_t *native;     /* [n_native][2] i<j, disjoint from bonds */
  const double *native_eps;                    /* [n_native] or NULL -> eps_native */
} sopo_topology;

typedef struct {
  double k_fene, R0, eps_native, eps_rep, sigma;
  double R_nb, R_pl;                           /* R_pl may be +inf: static all-pairs L1 */
  int32_t nb_interval, pl_interval;
  double dt_over_zeta, kT;
  uint64_t seed;
  int32_t traj_offset;                         /* global index of local trajectory 0 (Philox counter word 1) */
  int32_t n_fixed;  const int32_t *fixed;
  int32_t n_pulled; const int32_t *pulled;
  double pull_k, pull_v, pull_dir[3];
  int32_t tip_on; double tip_R, tip_eps, tip_sigma, tip_c0[3], tip_dir[3], tip_v;
  int32_t list_builder;                        /* 0 brute force over all j (the definition); 1 the oracle's own
                                                  cell list (tests prove it equal to 0; used for big N only) */
  int32_t rng;                                 /* 0 counter-based Philox (reading R6); 1 the paper's Hybrid Taus
                                                  (Alg. 6), state per bead, reading R12 */
  int32_t integrator;                          /* 0/1 first order, Alg. 7 line 5; 2 second order: the scheme whose
                                                  mean recursion is Eq. (5) (reading R14) */
  const double *kT_per_traj;                   /* [n_traj] or NULL -> kT for all: one temperature per run of a many-runs batch
                                                  ("parallel tempering ... Replica Exchange") */
} sopo_params;

enum { SOPO_OK = 0, SOPO_E_ARG = -1, SOPO_E_CAP = -3, SOPO_E_FENE = -4, SOPO_E_NONFINITE = -5 };

int  sopo_create(const sopo_topology *, const float *native_xyz /*[N][3]*/, const sopo_params *,
                 int32_t n_traj, sopo_handle **out);
void sopo_destroy(sopo_handle *);
int  sopo_run(sopo_handle *, int64_t n_steps);
int  sopo_get_coords(sopo_handle *, double *xyz_out /*[T][N][3]*/);
int  sopo_set_coords(sopo_handle *, const double *xyz /*[T][N][3]*/);   /* rebuilds L1 then L2 */
int  sopo_get_step(sopo_handle *, int64_t *step);
int  sopo_set_step(sopo_handle *, int64_t step);
int  sopo_get_energies(sopo_handle *, double *e_out /*[T][6] fene,native,rep,pull,tip,total*/);
uint32_t sopo_taus_step(uint32_t y[4]);       /* one Hybrid Taus draw; advances the state */
void sopo_taus_seed(uint64_t seed, uint32_t bead, uint32_t traj, uint32_t y[4]);
int  sopo_get_observables(sopo_handle *, double *o_out /*[T][4] Rg, end-to-end X, cantilever force, tip force*/);
int  sopo_get_forces(sopo_handle *, double *f_out /*[T][N][3]*/);       /* current coords, current L2 */
/* row counts and row contents (ascending j) of trajectory `traj`; idx is [N][cap]; cap too small -> SOPO_E_CAP */
int  sopo_get_lists(sopo_handle *, int32_t traj, int32_t level, int32_t *row_cnt, int32_t *idx, int32_t cap,
                    int64_t *built_at_step);
int  sopo_max_row(sopo_handle *, int32_t traj, int32_t level, int32_t *max_cnt);

/* caller-supplied coordinates; handle state untouched */
int  sopo_build_lists(sopo_handle *, const double *xyz /*[N][3]*/, int32_t level, int32_t builder,
                      int32_t *row_cnt, int32_t *idx, int32_t cap);     /* level 2 = filter(L1(xyz), xyz) */
int  sopo_filter(sopo_handle *, const double *xyz, const int32_t *l1_cnt, const int32_t *l1_idx, int32_t cap1,
                 int32_t *row_cnt, int32_t *idx, int32_t cap2);         /* Alg. 3 on a given L1 */
/* energies and forces at xyz with the L2 of trajectory `traj` FROZEN (finite-difference pins) */
int  sopo_eval_frozen(sopo_handle *, int32_t traj, const double *xyz /*[N][3]*/, int64_t step,
                      double *e_out /*[6]*/, double *f_out /*[N][3] or NULL*/);

/* noise pieces, exposed for the pins */
void sopo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void sopo_normals(uint64_t seed, uint32_t bead, uint32_t traj, uint64_t step, double g_out[3]);
void sopo_normals_batch(uint64_t seed, uint32_t bead0, uint32_t n_beads, uint32_t traj, uint64_t step,
                         double *g_out /*[n_beads][3]*/);
int  sopo_pred(const double a[3], const double b[3], double R);        /* the canonical fp32 list predicate */
int  sopo_num_threads(void);

/* NEXT-4: replica exchange over the batch.  One sweep: for every pair (t, t+1) with t = parity (mod 2), swap
 * the TEMPERATURES of the two runs with the Metropolis probability min(1, exp((1/kT_t - 1/kT_t+1)(E_t - E_t+1))), E = total
 * potential energy of the run at its current coordinates; the uniform of pair t in sweep `sweep` is the first word of
 * Philox4x32-10(counter = (t, 'REX!', sweep lo, sweep hi), key = seed) mapped to (0, 1] like u_a of sopo_normals.
 * accepted (may be NULL): [n_traj / 2] flags of the pairs tried (pair index t / 2). */
int  sopo_replica_exchange(sopo_handle *, int32_t parity, uint64_t sweep, int32_t *accepted);
int  sopo_get_temperatures(sopo_handle *, double *kT_out /*[n_traj]*/);
/* the acceptance probability and the decision, exposed for the pins */
double sopo_rex_probability(double E_i, double E_j, double kT_i, double kT_j);
int  sopo_rex_accept(double E_i, double E_j, double kT_i, double kT_j, double u);

#ifdef __cplusplus
}
#endif
#endif

/* sop.h -- C ABI of the B200-native SOP overdamped-Langevin hot path (arxiv 1003.1148; PAPER.md).
 *
 * The boundary follows the paper's statement of the problem: topology + native (PDB) coordinates in, trajectories
 * of coordinates and energies out (PAPER.md:45 Fig. 2; :98 "covalent bonds and native interactions ... obtained
 * from the PDB structure ... do not change").  Everything between sop_create and sop_get_* runs in hand-written
 * sm_100a CUDA kernels; there is no CPU fallback and no other backend.
 *
 * Conventions
 *   - plain C types only; every pointer says HOST or DEVICE;
 *   - the caller owns every input array; the library copies what it needs during sop_create and keeps no host
 *     pointer afterwards; outputs go into caller-allocated HOST buffers;
 *   - device memory comes from the caller (PyTorch in this repo): ask sop_query_workspace for the size, allocate,
 *     pass the DEVICE pointer to sop_create; it must stay alive until sop_destroy; 256-byte aligned;
 *   - all work is enqueued on params.stream (a cudaStream_t; NULL = legacy default stream);
 *   - every call returns 0 or a negative sop_status; device-side conditions (list-row overflow, FENE overstretch,
 *     non-finite coordinate) set bits in a device flag word that is read by the next synchronising call
 *     (sop_sync, sop_get_*); sop_last_error gives a handle-owned message;
 *   - a handle is not thread-safe; one stream per handle.
 *
 * Units: Angstrom, kcal/mol; dt_over_zeta = h/xi of Alg. 7 in A^2 mol/kcal; forces kcal/mol/A.
 */
#ifndef SOP_H
#define SOP_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sop_handle sop_handle;

enum sop_status {
  SOP_OK = 0,
  SOP_E_ARG = -1,            /* bad topology / params: out-of-range or duplicate pair, bond that is also native,
                                pl_interval not a multiple of nb_interval, workspace too small, ... */
  SOP_E_CUDA = -2,           /* a CUDA runtime call failed (message in sop_last_error) */
  SOP_E_LIST_OVERFLOW = -3,  /* a list row exceeded cap_nb / cap_pl (never truncated silently) */
  SOP_E_FENE = -4,           /* some bond reached |r - r0| >= R0: log of a non-positive number (Eq. (1)) */
  SOP_E_NONFINITE = -5       /* a coordinate became non-finite, or a bead entered the indenter sphere */
};

/* Topology (HOST arrays, 0-based bead indices).  Bonds: first term of Eq. (1); natives: second
 * term, Delta_ij = 1.  Every other pair belongs to the non-native set (third and fourth terms,
 * PAPER.md:243; it contains the i,i+2 pairs).  r0 of both kinds is the distance in native_xyz. */
typedef struct {
  int32_t n_beads;                             /* N per trajectory */
  int32_t n_bonds;   const int32_t *bonds;     /* HOST [n_bonds][2], i<j, unique */
  int32_t n_native;  const int32_t *native;    /* HOST [n_native][2], i<j, unique, disjoint from bonds */
  const float *native_eps;                     /* HOST [n_native] or NULL -> params.eps_native for all */
} sop_topology;

typedef struct {
  float k_fene, R0;                  /* FENE spring constant and tolerance R0 (R0 = 2 A) */
  float eps_native;                  /* eps_n of the 12-6 term (paper 1.5; BASELINE configs 1) */
  float eps_rep, sigma;              /* eps_r, sigma of the (sigma/r)^6 repulsion */
  float R_nb, R_pl;                  /* neighbor-list (L2) cutoff; pair-list (L1) cutoff, may be +INFINITY:
                                        static all-pairs L1 built once and shared by all trajectories */
  int32_t nb_interval, pl_interval;  /* L2 re-filtered every nb_interval steps (Alg. 3); L1 rebuilt every
                                        pl_interval steps (a multiple of nb_interval) */
  int32_t cap_nb, cap_pl;            /* row capacities (the paper's M); 0 -> chosen from the native
                                        structure (max count within the cutoff * 1.15 + 8) */
  float dt_over_zeta, kT;            /* h/xi and k_B T of Alg. 7 line 5 */
  const float *kT_per_traj;          /* HOST [n_traj] or NULL -> kT for all: one temperature per run of a many-runs batch (NEXT-4;
                                        PAPER.md:310, parallel tempering / Replica Exchange); see sop_replica_exchange */
  int32_t integrator;                /* 0 / 1 first order, Alg. 7 line 5; 2 second order: the predictor-corrector whose
                                        mean recursion is Eq. (5) (reading R14): two force evaluations per
                                        step, mode 1 and rng = 0 only */
  uint64_t seed;                     /* Philox4x32-10 key = (seed lo, seed hi) */
  int32_t traj_offset;               /* global index of local trajectory 0; goes into Philox counter word 1 so
                                        that a batch sharded over GPUs reproduces the unsharded batch */
  int32_t n_fixed;   const int32_t *fixed;    /* HOST; beads that are never moved */
  int32_t n_pulled;  const int32_t *pulled;   /* HOST; beads on a cantilever spring */
  float pull_k, pull_v, pull_dir[3];          /* kappa [kcal/mol/A^2], spring-base speed [A/step], unit vector n:
                                                 f = kappa (v s - (r_p - a_p).n) n, a_p = native position */
  int32_t tip_on;                             /* spherical indenter (reading R8 of DESIGN.md) */
  float tip_R, tip_eps, tip_sigma, tip_c0[3], tip_dir[3], tip_v;
                                              /* V = eps_t (sigma_t/(|r - c| - R))^6, c = c0 + v s dir */
  int32_t lanes_per_bead;            /* 0 auto; 1,2,4,8,16,32: threads cooperating on one bead
                                        (1 = the paper's particle-based thread-per-bead, 32 = warp-per-bead) */
  int32_t block_size;                /* 0 auto; threads per block of the step kernel (multiple of 32) */
  int32_t compensated;               /* 0 auto (on if max|coord| > 512 A), 1 on, 2 off: Kahan-compensated
                                        position update (keeps fp32 coordinates accurate at |x| ~ 10^3 A) */
  int32_t pair_atomics;              /* mode 4: 0 unique places + gathering (Alg. 4 + 5), 1 atomicAdd into one accumulator per
                                        bead (the form the paper anticipates for Fermi) */
  int32_t mode;                      /* 4 = the paper's interacting-pair based scheme (Alg. 4 + 5): one thread
                                        per pair, every pair force computed once, two launches per step.
                                        0 auto (3 when the chunk state fits shared memory, else 2), 1 one launch per
                                        step, 2 persistent streaming kernel (grid barrier per step), 3 SM-resident
                                        persistent kernel: a chunk of beads + halo + its L2 rows live in shared
                                        memory, chunks exchange coordinates through stamped words in L2 */
  int32_t reorder;                   /* 0 auto, 1 sort beads by native position inside the library, 2 keep order;
                                        invisible at the boundary (all indices in and out are the caller's) */
  int32_t chunk_beads;               /* mode 3: beads per chunk (one chunk per CTA); 0 auto */
  int32_t resident_variant;          /* mode 3 with several chunks per trajectory: 0 auto (the faster one as measured, 1),
                                        1 first design (lanes_per_bead lanes per bead, phases separated by block barriers),
                                        2 second design (four lanes per bead, rows dealt by bank group, service warps that
                                        overlap the exchange with the own-chunk partners) */
  int32_t obs_stride, obs_capacity;  /* NEXT-1: record the observables + energies of every trajectory every obs_stride steps inside
                                        sop_run into a DEVICE ring of obs_capacity samples (part of the workspace); 0, 0 = off */
  int32_t rng;                       /* 0 counter-based Philox4x32-10 (no generator state in memory); 1 the paper's Hybrid
                                        Taus (Alg. 6): 16 bytes of state per bead instance read and
                                        written every step, seeded from Philox(seed); every mode.  The state is not part
                                        of sop_set_coords / sop_set_step, so an exact resume needs rng = 0 */
  void *stream;                      /* cudaStream_t */
} sop_params;

/* Bytes of DEVICE workspace sop_create needs for this problem (deterministic: capacities, not contents). */
int sop_query_workspace(const sop_topology *topo, const float *native_xyz /*HOST [N][3]*/,
                        const sop_params *params, int32_t n_traj, size_t *bytes_out);

/* Validate, derive r0 from native_xyz (fp64, rounded to fp32), upload the static tables, start all n_traj
 * trajectories from native_xyz (they differ only through the trajectory word of the Philox counter), build the
 * pair list L1 and the neighbor list L2 from it, step = 0.   PAPER.md:45, :98. */
int sop_create(const sop_topology *topo, const float *native_xyz /*HOST [N][3]*/, const sop_params *params,
               int32_t n_traj, void *d_workspace /*DEVICE*/, size_t workspace_bytes, sop_handle **out);
void sop_destroy(sop_handle *);

/* Advance every trajectory by n_steps updates of Alg. 7 with the forces of Eq. (1), the
 * external terms and Philox/Box-Muller noise.  Asynchronous on the stream.
 * List invariant on return (once the stream has drained): if step % pl_interval == 0 the L1 was built from the
 * current coordinates; if step % nb_interval == 0 then L2 = filter(L1, current coordinates) (Alg. 3). */
int sop_run(sop_handle *, int64_t n_steps);
/* Wait for the stream and report device-side conditions raised since the last sync. */
int sop_sync(sop_handle *);

int sop_get_coords(sop_handle *, float *xyz_out /*HOST [T][N][3]*/);
int sop_set_coords(sop_handle *, const float *xyz /*HOST [T][N][3]*/);   /* rebuilds L1 then L2 */
/* Eq. (1) term by term + external terms, per trajectory: fene, native, rep (over the current
 * L2, each pair once), pull, tip, total.  fp32 pair terms, fp64 accumulation. */
int sop_get_energies(sop_handle *, double *e_out /*HOST [T][6]*/);
/* The same six energies for callers that may not allocate device memory or wait for the host (code under CUDA graph
 * capture, tight serving loops): sop_energies_noalloc enqueues the a10 reduction on the handle's stream with its per-block
 * partial sums in a file-scope static __device__ array of SOP_NOALLOC_SCRATCH_BYTES inside the library (every GPU that
 * loads the library holds it until exit) and writes {fene, native, rep, pull, tip, total} per trajectory to the caller's
 * DEVICE array.  It calls no cudaMalloc / cudaFree / allocating routine, copies nothing to the host and does not
 * synchronise: the result is valid once the stream has reached it (sop_sync); device-side conditions (FENE overstretch ...)
 * are reported by the next synchronising call, as for sop_run.  Values are bit-identical to sop_get_energies.
 * The scratch is shared by every handle and every call on a device and keeps the last call's contents (nothing in it has
 * to start at zero: every block overwrites its own partial sums before they are read): calls that overlap on the GPU --
 * two handles on different streams -- race and must be ordered by the caller.
 * Errors: SOP_E_ARG for a null argument or when n_traj x reduction blocks x 5 doubles exceed SOP_NOALLOC_SCRATCH_BYTES
 * (the message states both sizes; use sop_get_energies then); SOP_E_CUDA when the scratch address cannot be resolved
 * or a launch fails. */
#define SOP_NOALLOC_SCRATCH_BYTES (1u << 20)
int sop_energies_noalloc(sop_handle *, double *d_e_out /*DEVICE [T][6]*/);
/* Observables of the paper's applications, per trajectory, reduced on the device (PAPER.md:261 force-extension curves
 * f(R); :312-314 force-indentation): o[0] = radius of gyration, o[1] = end-to-end distance X between the first fixed
 * bead (else bead 0) and the first pulled bead (else bead N-1), o[2] = cantilever force summed over the pulled beads
 * kappa (v s - (r_p - a_p).n)  (= r_f t at zero displacement, r_f = kappa v), o[3] = force resisting the
 * indenter sum_i F_i^tip . tip_dir.  fp32 terms, fp64 sums. */
int sop_get_observables(sop_handle *, double *o_out /*HOST [T][4]*/);
/* The series recorded inside sop_run (params.obs_stride): the curves of the paper's applications -- force-extension f(R)
 * (PAPER.md:261), force-indentation (:312-314) -- and time averages without one host round trip per sample.
 * A sample is taken whenever step % obs_stride == 0 after an update.  o_out: HOST [n][T][10] = {Rg, X, cantilever force, tip
 * force, V_fene, V_nat, V_rep, V_pull, V_tip, V_total} of the last n <= max_samples samples, oldest first; steps_out: HOST [n]
 * (may be NULL).  Synchronises.  sop_set_observable_stride changes the stride (0 = stop recording). */
int sop_set_observable_stride(sop_handle *, int32_t stride);
int sop_get_observable_series(sop_handle *, double *o_out, int64_t *steps_out, int32_t max_samples, int32_t *n_out);
/* NEXT-4: one sweep of replica exchange over the batch.  For every pair of trajectories (t, t+1) with
 * t = parity (mod 2), swap their TEMPERATURES with the Metropolis probability min(1, exp((1/kT_t - 1/kT_t+1)(E_t - E_t+1))),
 * E = total potential energy at the current coordinates (the device-side reduction of sop_get_energies, decided in fp64);
 * the uniform of pair t is the first word of Philox4x32-10(counter = (traj_offset + t, 'REX!', sweep lo, sweep hi), key = seed)
 * mapped to (0, 1].  accepted_out: HOST [n_traj / 2] flags of the pairs tried (index t / 2), may be NULL.  Needs
 * params.kT_per_traj.  sop_get_temperatures: HOST [n_traj] current kT of every trajectory. */
int sop_replica_exchange(sop_handle *, int32_t parity, uint64_t sweep, int32_t *accepted_out);
int sop_get_temperatures(sop_handle *, float *kT_out);
/* Deterministic force (no noise) at the current coordinates with the current L2, incl. external terms. */
int sop_get_forces(sop_handle *, float *f_out /*HOST [T][N][3]*/);
/* Row counts and rows (ascending caller index j, padded with -1 to cap) of trajectory traj.
 * level 1 = pair list, 2 = neighbor list.  idx may be NULL to fetch counts / capacity only. */
int sop_get_lists(sop_handle *, int32_t traj, int32_t level, int32_t *row_cnt /*HOST [N]*/,
                  int32_t *idx /*HOST [N][cap]*/, int32_t *cap_out, int64_t *built_at_step);
int sop_get_step(sop_handle *, int64_t *step);
int sop_set_step(sop_handle *, int64_t step);       /* with sop_set_coords: exact resume of a checkpoint */
/* Zero-copy view of the current coordinate layer: DEVICE float4 [T][N] in the library's internal bead order;
 * perm_out (HOST [N], may be NULL) receives the caller index of each internal slot. */
int sop_device_coords(sop_handle *, void **d_float4_out, int32_t *perm_out);
/* What the auto settings resolved to: lanes_per_bead, block_size, compensated(0/1), mode(1/2/3), reorder(0/1),
 * cap_nb, cap_pl, kernel launches issued so far (lo, hi), resident_variant in use (0 when the trajectory is one chunk),
 * steps per time slice of the most recent SLICED mode-3 launch (0: none so far; many one-chunk trajectories,
 * PAPER.md:292), reserved. */
int sop_get_config(sop_handle *, int32_t out[12]);
/* Launch planning of the many-runs batch (many independent trajectories of a small system in one launch), host
 * arithmetic only, no device call: the number of Langevin steps per TIME SLICE a mode-3 launch of n_steps steps over n_traj
 * one-chunk trajectories is cut into when the device holds cta_slots resident CTAs at once (one CTA per slice and trajectory,
 * handed out slice-major by a ticket, so that no SM idles through a partly empty last wave); 0 = not sliced (n_traj <=
 * cta_slots, a short launch, or less than 3 % to gain).  A positive result is a multiple of nb_interval, at least
 * 2 * nb_interval and less than n_steps.  Bad arguments (anything < 1) return 0. */
int32_t sop_plan_slices(int32_t n_steps, int32_t nb_interval, int32_t n_traj, int32_t cta_slots);
/* Kernel timing for the bench (CUDA events on the handle's stream around groups of launches of one kind).
 * sop_get_profile synchronises, fills out[0..2] = ms spent in {step kernels, L2 filter kernels, L1 build kernels},
 * out[3..5] = number of timed spans of each kind, out[6] = Langevin steps covered by the step spans, and resets. */
int sop_set_profiling(sop_handle *, int32_t on);
int sop_get_profile(sop_handle *, double out[8]);
const char *sop_last_error(sop_handle *);           /* handle may be NULL: last error of a failed create/query */

#ifdef __cplusplus
}
#endif
#endif

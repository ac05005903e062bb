/* Test driver (tests/test_oracle_sanitizers.py): exercises the fp64 oracle under -fsanitize=address,undefined (SURVEY.md
 * section 5).  Builds a small two-chain system, runs every entry point, prints a checksum; any sanitizer report makes the
 * run fail. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../oracle/sopo.h"

int main(void) {
  enum { N = 60 };
  float xyz[N][3];
  int32_t bonds[N][2], native[4 * N][2];
  int nb = 0, nn = 0;
  /* two helices of 30 beads, 3.8 A bonds */
  for (int i = 0; i < N; ++i) {
    int c = i / 30, k = i % 30;
    xyz[i][0] = (float)(4.0 * cos(0.9 * k) + 9.0 * c);
    xyz[i][1] = (float)(4.0 * sin(0.9 * k));
    xyz[i][2] = (float)(1.5 * k);
    if (k > 0) { bonds[nb][0] = i - 1; bonds[nb][1] = i; ++nb; }
  }
  for (int i = 0; i < N; ++i)
    for (int j = i + 3; j < N; ++j) {
      double d = 0;
      for (int a = 0; a < 3; ++a) d += ((double)xyz[i][a] - xyz[j][a]) * ((double)xyz[i][a] - xyz[j][a]);
      if (d < 64.0 && (i / 30 != j / 30 || j - i > 2) && nn < 4 * N) { native[nn][0] = i; native[nn][1] = j; ++nn; }
    }
  sopo_topology tp = { N, nb, &bonds[0][0], nn, &native[0][0], NULL };
  int32_t fixed[1] = { 0 }, pulled[1] = { N - 1 };
  double kTs[3] = { 0.5, 0.6, 0.7 };
  int rc = 0;
  double sum = 0;
  for (int variant = 0; variant < 4; ++variant) {
    sopo_params p;
    memset(&p, 0, sizeof(p));
    p.k_fene = 14; p.R0 = 2; p.eps_native = 1; p.eps_rep = 1; p.sigma = 3.8; p.R_nb = 10; p.R_pl = variant == 0 ? INFINITY : 20;
    p.nb_interval = 10; p.pl_interval = 50; p.dt_over_zeta = 2e-3; p.kT = 0.6; p.seed = 0x5EED;
    p.n_fixed = 1; p.fixed = fixed; p.n_pulled = 1; p.pulled = pulled; p.pull_k = 0.05; p.pull_v = 1e-3; p.pull_dir[2] = 1;
    p.tip_on = 1; p.tip_R = 50; p.tip_eps = 1; p.tip_sigma = 3.8; p.tip_c0[2] = 110; p.tip_dir[2] = -1; p.tip_v = 1e-3;
    p.list_builder = variant & 1; p.rng = variant == 2; p.integrator = variant == 3 ? 2 : 0; p.kT_per_traj = kTs;
    sopo_handle *h = NULL;
    rc |= sopo_create(&tp, &xyz[0][0], &p, 3, &h);
    if (rc || !h) { printf("create failed %d\n", rc); return 1; }
    rc |= sopo_run(h, 120);
    double e[18], o[12], x[3 * N * 3], f[3 * N * 3], kT[3];
    int32_t cnt[N], idx[N * N], acc[2], mx = 0;
    int64_t at = 0;
    rc |= sopo_get_energies(h, e); rc |= sopo_get_observables(h, o); rc |= sopo_get_coords(h, x); rc |= sopo_get_forces(h, f);
    rc |= sopo_max_row(h, 1, 1, &mx);
    rc |= sopo_get_lists(h, 2, 2, cnt, idx, N, &at);
    rc |= sopo_build_lists(h, x, 2, 1, cnt, idx, N);
    rc |= sopo_filter(h, x, cnt, idx, N, cnt, idx, N);
    rc |= sopo_replica_exchange(h, 0, 3, acc); rc |= sopo_replica_exchange(h, 1, 4, acc); rc |= sopo_get_temperatures(h, kT);
    rc |= sopo_set_coords(h, x); rc |= sopo_run(h, 30);
    rc |= sopo_eval_frozen(h, 0, x, 150, e, f);
    for (int q = 0; q < 6; ++q) sum += e[q];
    sopo_destroy(h);
  }
  uint32_t y[4]; double g[3];
  sopo_taus_seed(1, 2, 3, y); sum += (double)sopo_taus_step(y); sopo_normals(1, 2, 3, 4, g); sum += g[0];
  printf("rc %d checksum %.6f\n", rc, sum);
  return rc != 0;
}

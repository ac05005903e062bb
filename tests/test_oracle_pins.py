"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only; no CUDA path involved).

P1  Eq. (1) minima at the native structure
P2  F = -grad V, term by term, by central differences               PAPER.md:259 ("f = -dV/dr"), Eq. (1)
P3  zero net internal force and torque (Alg. 1 lines 8-9, +-df)
P4  FENE divergence, error beyond R0, exact two-bead recursion
P5  free diffusion <dr^2> = 6 (kT h/xi) n, independence             PAPER.md:224 (Alg. 7 line 5)
P6  Philox4x32-10 = cuRAND's host generator + known-answer vectors  north_star; tests/golden/philox_kat.txt
P7  bead on a moving spring: Eq. (4) exactly, Eq. (3) to O(h/tau)
P8  lists: brute force, Table I identity, boundary cases, Alg. 3
P9  indenter / pulling spring: F = -grad V, 1-D special case        readings R7, R8 (paper silent on the indenter)
P10 Box-Muller normals: moments, bound, KS
P13 Eq. (1) magnitudes of the native and repulsion terms by hand
P14 replica exchange: Metropolis rule, detailed balance, sweep
P15 second-order update: Eq. (5) exactly, Eq. (3) within 1e-5
"""
import ctypes
import math
import os

import numpy as np
import pytest

from oracle import sopo
from workloads import generators as gen

GOLD = os.path.join(os.path.dirname(__file__), "golden")
rng = np.random.default_rng(12345)


def perturbed(w, amp, seed):
    r = np.random.default_rng(seed)
    return w.xyz.astype(np.float64) + amp * r.normal(size=w.xyz.shape)


# ---------------------------------------------------------------------------------------------- P1
def test_p1_native_minima():
    w = gen.config0()
    o = sopo.from_workload(w)
    e = o.get_energies()[0]
    assert abs(e[0]) < 1e-9                                   # V_FENE = 0 at r = r0 (r0 is an fp32: ~1e-12 left)
    assert e[1] == pytest.approx(-1.0 * len(w.native), abs=1e-9)   # each 12-6 term is -eps at r = r0
    assert e[3] == 0 and e[4] == 0
    assert e[5] == pytest.approx(e[0] + e[1] + e[2], abs=1e-12)
    # bonded and native forces vanish at the native structure: with eps_rep = 0 nothing is left
    p = dict(w.params, eps_rep=0.0)
    o0 = sopo.Oracle(w.xyz, w.bonds, w.native, p)
    assert np.abs(o0.get_forces()).max() < 1e-4
    # and the full force is the repulsion alone
    p2 = dict(w.params, k_fene=0.0, eps_native=0.0)
    o2 = sopo.Oracle(w.xyz, w.bonds, w.native, p2)
    assert np.abs(o.get_forces() - o2.get_forces()).max() < 1e-4


# ---------------------------------------------------------------------------------------------- P2
@pytest.mark.parametrize("term", ["fene", "native", "rep", "all"])
def test_p2_force_is_minus_gradient(term):
    w = gen.tiny(48, 1)
    p = dict(w.params)
    if term == "fene":
        p.update(eps_native=0.0, eps_rep=0.0)
    elif term == "native":
        p.update(k_fene=0.0, eps_rep=0.0)
    elif term == "rep":
        p.update(k_fene=0.0, eps_native=0.0)
    o = sopo.Oracle(w.xyz, w.bonds, w.native, p)
    x = perturbed(w, 0.15, 7)
    e0, f = o.eval_frozen(x)
    col = {"fene": 0, "native": 1, "rep": 2, "all": 5}[term]
    h = 1e-5
    worst = 0.0
    for i in range(0, w.n_beads, 5):
        for a in range(3):
            xp = x.copy(); xp[i, a] += h
            xm = x.copy(); xm[i, a] -= h
            ep, _ = o.eval_frozen(xp, want_forces=False)
            em, _ = o.eval_frozen(xm, want_forces=False)
            fd = -(ep[col] - em[col]) / (2 * h)
            worst = max(worst, abs(fd - f[i, a]))
    assert worst < 2e-6 * max(1.0, np.abs(f).max())
    assert np.abs(f).max() > 0.1          # the term really acts


# ---------------------------------------------------------------------------------------------- P3
def test_p3_newton_third_law():
    w = gen.two_chains(64, 0)
    assert (w.chain[w.native[:, 0]] != w.chain[w.native[:, 1]]).any()
    o = sopo.from_workload(w)
    x = perturbed(w, 0.2, 3)
    _, f = o.eval_frozen(x)
    assert np.abs(f.sum(axis=0)).max() < 1e-9 * np.abs(f).sum()
    assert np.abs(np.cross(x, f).sum(axis=0)).max() < 1e-9 * np.abs(np.cross(x, f)).sum()


# ---------------------------------------------------------------------------------------------- P4
def _two_beads(**over):
    xyz = np.array([[0, 0, 0], [3.8, 0, 0]], np.float32)
    p = dict(gen.BASE_PARAMS, kT=0.0, **over)
    return sopo.Oracle(xyz, np.array([[0, 1]], np.int32), np.zeros((0, 2), np.int32), p)


def test_p4_fene_divergence_and_error():
    o = _two_beads()
    k, R0 = 14.0, 2.0
    r0 = float(np.float32(3.8))
    prev = 0.0
    for m in range(1, 7):
        delta = R0 * (1 - 10.0 ** -m)
        x = np.array([[0, 0, 0], [r0 + delta, 0, 0]], float)
        _, f = o.eval_frozen(x)
        expect = k * delta / (1 - delta * delta / (R0 * R0))
        assert f[0, 0] == pytest.approx(expect, rel=1e-6)      # bead 0 is pulled toward bead 1 (+x)
        assert f[1, 0] == pytest.approx(-expect, rel=1e-6)
        assert f[0, 0] > 4.0 * prev                            # grows like 10^m k R0 / 2
        prev = f[0, 0]
        assert expect == pytest.approx(10.0 ** m * k * R0 / 2, rel=0.6)
    for delta in (R0, R0 * 1.01, -R0):
        x = np.array([[0, 0, 0], [r0 + delta, 0, 0]], float)
        with pytest.raises(sopo.OracleError) as ei:
            o.eval_frozen(x)
        assert ei.value.code == -4


def test_p4_two_bead_relaxation_recursion():
    D, k, R0 = float(np.float32(2e-3)), 14.0, 2.0
    o = _two_beads()
    r0 = float(np.float32(3.8))
    delta = 1.5
    o.set_coords(np.array([[[0, 0, 0], [r0 + delta, 0, 0]]], float))
    for n in range(200):
        o.run(1)
        delta = delta - 2 * D * k * delta / (1 - delta * delta / (R0 * R0))
        x = o.get_coords()[0]
        assert (x[1, 0] - x[0, 0]) - r0 == pytest.approx(delta, abs=1e-12)
    assert abs(delta) < 1e-4


# ---------------------------------------------------------------------------------------------- P5
def test_p5_free_diffusion():
    N, n = 4096, 50
    w = gen.free_beads(N, R_pl=20.0, kT=0.6)
    o = sopo.from_workload(w, n_traj=2)
    x0 = o.get_coords()
    o.run(n)
    d = o.get_coords() - x0                                  # [T][N][3]
    kT, D = float(np.float32(0.6)), float(np.float32(2e-3))
    var = 2 * kT * D * n
    M = d.size
    assert abs(d.mean()) < 5 * math.sqrt(var / M)
    assert d.var() == pytest.approx(var, rel=5 * math.sqrt(2.0 / M))
    assert (d ** 2).sum(axis=2).mean() == pytest.approx(6 * kT * D * n, rel=5 * 0.816 / math.sqrt(2 * N))
    z = d / math.sqrt(var)
    assert abs((z ** 4).mean() - 3.0) < 5 * math.sqrt(96.0 / M)          # excess kurtosis 0
    # independence across axes, neighbouring beads and trajectories
    se = 5 / math.sqrt(2 * N)
    assert abs((z[..., 0] * z[..., 1]).mean()) < se and abs((z[..., 1] * z[..., 2]).mean()) < se
    assert abs((z[:, 1:, :] * z[:, :-1, :]).mean()) < se
    assert abs((z[0] * z[1]).mean()) < se
    # independence across steps: single-step increments
    o2 = sopo.from_workload(w)
    a = o2.get_coords(); o2.run(1); b = o2.get_coords(); o2.run(1); c = o2.get_coords()
    assert abs(((b - a) * (c - b)).mean()) / (2 * kT * D) < 5 / math.sqrt(3 * N)


# ---------------------------------------------------------------------------------------------- P6
def _kat():
    rows = []
    for line in open(os.path.join(GOLD, "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split() if t != "->"]
        rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_p6_philox_known_answers():
    for ctr, key, out in _kat():
        assert sopo.philox4x32_10(ctr, key).tolist() == out


def _curand_host():
    for name in ("libcurand.so", "libcurand.so.10", "/usr/local/cuda/lib64/libcurand.so"):
        try:
            return ctypes.CDLL(name)
        except OSError:
            pass
    return None


def test_p6_philox_equals_curand_host_generator():
    """Library-routine special case: cuRAND's HOST Philox4_32_10 generator (runs on the CPU).  With seed s its output
    stream, taken 4 words at a time, is block b = philox(counter = (b div 65536 as a 64-bit integer in words 0-1,
    b mod 65536, 0), key = (s lo, s hi)); the generator offset selects the first block (offset = 4 b)."""
    lib = _curand_host()
    if lib is None:
        pytest.skip("libcurand not found")
    r = np.random.default_rng(99)
    for _ in range(20):
        seed = int(r.integers(0, 2 ** 63))
        hi = int(r.integers(0, 2 ** 45)); sub = int(r.integers(0, 65536 - 8))
        blk = hi * 65536 + sub
        g = ctypes.c_void_p()
        assert lib.curandCreateGeneratorHost(ctypes.byref(g), 161) == 0          # CURAND_RNG_PSEUDO_PHILOX4_32_10
        assert lib.curandSetPseudoRandomGeneratorSeed(g, ctypes.c_ulonglong(seed)) == 0
        assert lib.curandSetGeneratorOffset(g, ctypes.c_ulonglong(4 * blk)) == 0
        out = np.zeros(32, np.uint32)
        assert lib.curandGenerate(g, out.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(32)) == 0
        lib.curandDestroyGenerator(g)
        for q in range(8):
            mine = sopo.philox4x32_10([hi & 0xFFFFFFFF, hi >> 32, sub + q, 0], [seed & 0xFFFFFFFF, seed >> 32])
            assert mine.tolist() == out[4 * q: 4 * q + 4].tolist()


def test_p6_counter_words_all_matter():
    base = sopo.philox4x32_10([1, 2, 3, 4], [5, 6]).tolist()
    for w in range(4):
        c = [1, 2, 3, 4]; c[w] += 1
        assert sopo.philox4x32_10(c, [5, 6]).tolist() != base
    assert sopo.philox4x32_10([1, 2, 3, 4], [6, 6]).tolist() != base
    assert sopo.philox4x32_10([1, 2, 3, 4], [5, 7]).tolist() != base
    # the mapping of sopo_normals: counter (bead, traj, step lo, step hi), key (seed lo, seed hi)
    x = sopo.philox4x32_10([7, 3, 0x23456789, 0x1], [0xDEADBEEF, 0x12345678])
    ua = ((int(x[0]) >> 8) + 1) / 2.0 ** 24; ub = (int(x[1]) >> 8) / 2.0 ** 24
    uc = ((int(x[2]) >> 8) + 1) / 2.0 ** 24; ud = (int(x[3]) >> 8) / 2.0 ** 24
    g = sopo.normals(0x12345678DEADBEEF, 7, 3, 0x123456789)
    assert g[0] == pytest.approx(math.sqrt(-2 * math.log(ua)) * math.cos(2 * math.pi * ub), abs=1e-14)
    assert g[1] == pytest.approx(math.sqrt(-2 * math.log(ua)) * math.sin(2 * math.pi * ub), abs=1e-14)
    assert g[2] == pytest.approx(math.sqrt(-2 * math.log(uc)) * math.cos(2 * math.pi * ud), abs=1e-14)


# ---------------------------------------------------------------------------------------------- P7
def _spring_beads(N, T, kT, kappa=0.05, v=1e-3):
    w = gen.free_beads(N, R_pl=20.0, kT=kT, pulled=list(range(N)), pull_k=kappa, pull_v=v, pull_dir=[0.0, 0.0, 1.0])
    return w, sopo.from_workload(w, n_traj=T)


def test_p7_eq4_exact_without_noise():
    """kT = 0: every bead must follow the first-order recursion Eq. (4) to rounding:
    X(n+1) = X(n) + (r_f t_n/xi - X(n)/tau) h with h/xi = D, h/tau = kappa D, r_f t_n h/xi = kappa v n D."""
    kappa, v, D = float(np.float32(0.05)), float(np.float32(1e-3)), float(np.float32(2e-3))
    w, o = _spring_beads(8, 1, 0.0)
    z0 = o.get_coords()[0, :, 2].copy()
    X = 0.0
    for n in range(300):
        o.run(1)
        X = X + kappa * D * (v * n - X)
        assert np.abs(o.get_coords()[0, :, 2] - z0 - X).max() < 1e-12
    # Eq. (3) with X0 = 0: <X(t)> = (r_f tau/xi)(t - tau(1 - exp(-t/tau))); in steps: v (n - tau(1-e^{-n/tau}))
    tau = 1.0 / (kappa * D)
    n = 300
    th = v * (n - tau * (1 - math.exp(-n / tau)))
    # first-order (Euler) error: relative O(h/t) while t << tau (X grows like t^2), O(h/tau) later
    assert X == pytest.approx(th, rel=1.5 / n + 10 / tau)


def test_p7_paper_parameters_error_bound():
    """with the paper's own parameters (K_sp = 40 pN/nm, D = 1.5e-11 cm^2/s, h = 1, 25, 50 ps) the
    ORACLE's update, iterated without noise, stays within the printed relative error 2e-5 of Eq. (3).  The paper's
    harmonic particle under the ramp r_f t is the oracle's bead on a cantilever with kappa = K_sp, spring-base speed
    v = r_f h / K_sp per step and h/xi = dt_over_zeta, so that kappa * dt_over_zeta = h/tau."""
    line = [l for l in open(os.path.join(GOLD, "eq3_eq4_paper_params.txt")) if not l.startswith("#")][0].split()
    Ksp, D_cm2s, kT, bound = float(line[0]), float(line[3]), float(line[4]), float(line[7])
    xi = kT / (D_cm2s * 1e14 * 1e-12)          # pN ps / nm   (D in nm^2/ps)
    tau = xi / Ksp                              # ps
    n = 10 ** 6
    for h in (1.0, 25.0, 50.0):
        a = h / tau                             # = kappa * dt_over_zeta in the oracle's units
        kappa = 1.0
        w = gen.free_beads(2, R_pl=20.0, kT=0.0, pulled=[0, 1], pull_k=kappa, pull_v=1.0, pull_dir=[0.0, 0.0, 1.0])
        p = dict(w.params, dt_over_zeta=a / kappa, nb_interval=1000, pl_interval=100000)
        o = sopo.Oracle(w.xyz, w.bonds, w.native, p)
        a = sopo.f32(a / kappa) * kappa         # the value the oracle really uses (parameters are fp32, promoted)
        z0 = o.get_coords()[0, :, 2].copy()
        o.run(n)
        sim = (o.get_coords()[0, :, 2] - z0)    # in units of v = 1 per step
        th = n - (1 - math.exp(-n * a)) / a     # Eq. (3) with X0 = 0, t = n h, in the same units
        assert np.abs(sim - th).max() / th < bound
        # and the closed form of the recursion X(n+1) = (1-a) X(n) + a n agrees with what the oracle iterated
        closed = n - (1 - (1 - a) ** n) / a
        assert np.abs(sim - closed).max() / closed < 1e-9


def test_p7_mathematics_of_eq4_beyond_what_is_iterated():
    """Mathematics only (no oracle call): the closed form of the first-order recursion Eq. (4) against Eq. (3) at the
    paper's 10^8 and 10^9 steps, which are not iterated here."""
    line = [l for l in open(os.path.join(GOLD, "eq3_eq4_paper_params.txt")) if not l.startswith("#")][0].split()
    Ksp, D_cm2s, kT, bound = float(line[0]), float(line[3]), float(line[4]), float(line[7])
    tau = kT / (D_cm2s * 1e14 * 1e-12) / Ksp
    for h in (1.0, 25.0, 50.0):
        a = h / tau
        for n in (10 ** 8, 10 ** 9):
            sim = (n - (1 - (1 - a) ** n) / a)
            t = n * h
            th = (t - tau * (1 - math.exp(-t / tau))) / h
            assert abs(sim - th) / th < bound


def test_p7_ensemble_mean_and_variance():
    kappa, v, D, kT = float(np.float32(0.05)), float(np.float32(1e-3)), float(np.float32(2e-3)), float(np.float32(0.6))
    N, T, n = 512, 8, 400
    w, o = _spring_beads(N, T, kT)
    z0 = o.get_coords()[:, :, 2].copy()
    o.run(n)
    dz = (o.get_coords()[:, :, 2] - z0).ravel()
    X = 0.0
    for s in range(n):
        X = X + kappa * D * (v * s - X)
    # variance after n steps of the discrete OU process started at 0: 2kTD (1-(1-a)^(2n))/(1-(1-a)^2)
    a = kappa * D
    var = 2 * kT * D * (1 - (1 - a) ** (2 * n)) / (1 - (1 - a) ** 2)
    M = dz.size
    assert dz.mean() == pytest.approx(X, abs=5 * math.sqrt(var / M))
    assert dz.var() == pytest.approx(var, rel=5 * math.sqrt(2.0 / M))
    # stationary limit (kT/kappa)/(1 - kappa D/2)
    assert 2 * kT * D / (1 - (1 - a) ** 2) == pytest.approx((kT / kappa) / (1 - a / 2), rel=1e-12)
    # transverse motion is free
    o2 = sopo.from_workload(w, n_traj=T)
    x0 = o2.get_coords()[:, :, 0].copy(); o2.run(50)
    dx = o2.get_coords()[:, :, 0] - x0
    assert dx.var() == pytest.approx(2 * kT * D * 50, rel=5 * math.sqrt(2.0 / dx.size))


# ---------------------------------------------------------------------------------------------- P8
def brute_lists(xyz, excl, R):
    """O(N^2) double loop with the canonical fp32 predicate written with numpy.float32 scalars."""
    x = np.asarray(xyz, np.float64).astype(np.float32)
    N = len(x)
    R2f = np.float32(np.float64(R) * np.float64(R))
    rows = []
    for i in range(N):
        row = []
        for j in range(N):
            if j == i or (i, j) in excl:
                continue
            if math.isinf(R):
                row.append(j); continue
            dx = np.float32(x[i, 0] - x[j, 0]); dy = np.float32(x[i, 1] - x[j, 1]); dz = np.float32(x[i, 2] - x[j, 2])
            d2 = np.float32(np.float32(np.float32(dx * dx) + np.float32(dy * dy)) + np.float32(dz * dz))
            if d2 < R2f:
                row.append(j)
        rows.append(row)
    return rows


def excl_set(w):
    s = set()
    for a, b in np.concatenate([w.bonds, w.native]):
        s.add((int(a), int(b))); s.add((int(b), int(a)))
    return s


def rows_of(cnt, idx):
    return [idx[i, :cnt[i]].tolist() for i in range(len(cnt))]


@pytest.mark.parametrize("N,seed", [(8, 0), (33, 1), (100, 2), (257, 3)])
def test_p8_lists_equal_brute_force(N, seed):
    w = gen.tiny(N, seed, R_pl=20.0)
    o = sopo.from_workload(w)
    x = perturbed(w, 0.3, seed)
    ex = excl_set(w)
    for builder in (0, 1):
        c1, i1 = o.build_lists(x, 1, builder)
        assert rows_of(c1, i1) == brute_lists(x, ex, 20.0)
        c2, i2 = o.build_lists(x, 2, builder)
        assert rows_of(c2, i2) == brute_lists(x, ex, 10.0)


def test_p8_static_all_pairs_and_table1_identity():
    w = gen.config0()
    o = sopo.from_workload(w)
    c1, i1, at = o.get_lists(1)
    N = w.n_beads
    assert c1.sum() // 2 == N * (N - 1) // 2 - len(w.bonds) - len(w.native)
    assert rows_of(c1, i1) == brute_lists(w.xyz, excl_set(w), math.inf)
    # the i,i+2 pairs are in the non-native set (third term of Eq. (1))
    assert all((i + 2) in i1[i, :c1[i]] for i in range(N - 2))


def test_p8_table1_printed_pair_counts():
    """Table I: non-native pairs = N(N-1)/2 - bonds - contacts for WW, Ig27, C2A, (Fb)2.
    Any topology with those counts must give the printed number of L1 pairs when R_pl = +inf."""
    for line in open(os.path.join(GOLD, "table1.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, N, nb, nc, pairs, exact = line.split()
        N, nb, nc, pairs = int(N), int(nb), int(nc), int(pairs)
        if exact != "1" or N > 200:
            if exact == "1":
                assert N * (N - 1) // 2 - nb - nc == pairs
            continue
        r = np.random.default_rng(N)
        xyz = (3.8 * np.cumsum(r.normal(size=(N, 3)), axis=0)).astype(np.float32)
        bonds = np.stack([np.arange(nb), np.arange(nb) + 1], axis=1).astype(np.int32)
        cand = [(i, j) for i in range(N) for j in range(i + 3, N)]
        pick = r.choice(len(cand), size=nc, replace=False)
        native = np.array(sorted(cand[q] for q in pick), np.int32)
        o = sopo.Oracle(xyz, bonds, native, dict(gen.BASE_PARAMS))
        c1, _, _ = o.get_lists(1)
        assert c1.sum() // 2 == pairs, name


def test_p8_cutoff_edge_and_strict_inequality():
    # two free beads on the x axis; R_nb = 10: d = 10 exactly is OUT (strict <), the fp32 just below is IN
    below = float(np.nextafter(np.float32(10.0), np.float32(0.0)))
    above = float(np.nextafter(np.float32(10.0), np.float32(20.0)))
    for d, inside in ((below, True), (10.0, False), (above, False)):
        assert sopo.pred([0, 0, 0], [d, 0, 0], 10.0) is inside
        assert sopo.pred([d, 0, 0], [0, 0, 0], 10.0) is inside      # symmetric
    # the predicate rounds coordinates to fp32 first: a double just below 10 that rounds to 10.0f is OUT
    assert sopo.pred([0, 0, 0], [10.0 - 1e-9, 0, 0], 10.0) is False
    # d2 is accumulated in fp32: (6,8,0) has d2 = 100 exactly -> OUT
    assert sopo.pred([0, 0, 0], [6, 8, 0], 10.0) is False
    assert sopo.pred([0, 0, 0], [1, 2, 3], math.inf) is True


def test_p8_cell_builder_boundary_points():
    """Points exactly on cell boundaries and pairs at the cutoff edge: the oracle's cell-list builder equals
    its brute-force builder (which is the definition)."""
    r = np.random.default_rng(5)
    R = 20.0
    edge = R * 1.001
    pts = []
    for ix in range(4):
        for iy in range(3):
            for iz in range(3):
                base = np.array([ix, iy, iz], float) * edge          # exactly on cell corners
                pts.append(base)
                pts.append(base + r.uniform(0, edge, 3))
                pts.append(base + np.array([R, 0, 0]))                # partner exactly R away
                pts.append(base + np.array([float(np.nextafter(np.float32(R), np.float32(0))), 0, 0]))
    xyz = np.array(pts, np.float32)
    N = len(xyz)
    p = dict(gen.BASE_PARAMS, R_pl=R)
    o = sopo.Oracle(xyz, np.zeros((0, 2), np.int32), np.zeros((0, 2), np.int32), p)
    a = o.build_lists(xyz, 1, 0); b = o.build_lists(xyz, 1, 1)
    assert rows_of(*a) == rows_of(*b)
    assert rows_of(*a) == brute_lists(xyz, set(), R)
    a2 = o.build_lists(xyz, 2, 0); b2 = o.build_lists(xyz, 2, 1)
    assert rows_of(*a2) == rows_of(*b2)


def test_p8_cell_builder_equals_brute_on_assemblies():
    w = gen.two_chains(150, 1, R_pl=20.0)
    o = sopo.from_workload(w)
    x = perturbed(w, 0.5, 1)
    assert rows_of(*o.build_lists(x, 1, 0)) == rows_of(*o.build_lists(x, 1, 1))
    w3 = gen.config3()
    o3 = sopo.from_workload(w3, list_builder=1)
    x3 = perturbed(w3, 0.3, 2)
    a = o3.build_lists(x3, 1, 0, cap=512); b = o3.build_lists(x3, 1, 1, cap=512)
    assert (a[0] == b[0]).all() and (a[1] == b[1]).all()


def test_p8_alg3_filter_is_ordered_subsequence():
    w = gen.tiny(200, 4, R_pl=20.0)
    o = sopo.from_workload(w)
    o.run(100)                                           # step 100: L1 and L2 both rebuilt from current coords
    x = o.get_coords()[0]
    c1, i1, at1 = o.get_lists(1); c2, i2, at2 = o.get_lists(2)
    assert at1 == 100 and at2 == 100
    ex = excl_set(w)
    assert rows_of(c1, i1) == brute_lists(x, ex, 20.0)
    assert rows_of(c2, i2) == brute_lists(x, ex, 10.0)
    o.run(30)                                            # step 130: L1 from step 100, L2 from step 130
    x = o.get_coords()[0]
    c1b, i1b, at1 = o.get_lists(1); c2, i2, at2 = o.get_lists(2)
    assert at1 == 100 and at2 == 130
    assert rows_of(c1b, i1b) == rows_of(c1, i1)
    for i in range(w.n_beads):
        row1 = i1[i, :c1[i]].tolist(); row2 = i2[i, :c2[i]].tolist()
        it = iter(row1)
        assert all(j in it for j in row2)                # ordered subsequence of the L1 row (Alg. 3 copies in order)
    # nothing moved by more than R_pl - R_nb, so the filtered list equals brute force at R_nb
    assert rows_of(c2, i2) == brute_lists(x, ex, 10.0)
    # sopo_filter on a caller-supplied L1 is the same operation
    cf, jf = o.filter(x, c1, i1)
    assert rows_of(cf, jf) == rows_of(c2, i2)
    o.run(5)                                             # step 135: lists unchanged
    assert o.get_lists(2)[2] == 130


# ---------------------------------------------------------------------------------------------- P9
def test_p9_external_terms_gradient_and_1d_law():
    w = gen.tiny(40, 2)
    p = dict(w.params, k_fene=0.0, eps_native=0.0, eps_rep=0.0, pulled=[39, 5], pull_k=0.05, pull_v=1e-3,
             pull_dir=[0.6, 0.0, 0.8], tip_on=1, tip_R=50.0, tip_eps=1.0, tip_sigma=3.8,
             tip_c0=[0.0, 0.0, 70.0], tip_dir=[0.0, 0.0, -1.0], tip_v=1e-3)
    nobond = np.zeros((0, 2), np.int32)
    o = sopo.Oracle(w.xyz, nobond, nobond, p)
    x = perturbed(w, 0.2, 9)
    step = 2500
    e0, f = o.eval_frozen(x, step=step)
    assert e0[3] > 0 and e0[4] > 0
    h = 1e-5
    for i in (0, 5, 20, 39):
        for a in range(3):
            xp = x.copy(); xp[i, a] += h
            xm = x.copy(); xm[i, a] -= h
            fd = -(o.eval_frozen(xp, step=step, want_forces=False)[0][5] - o.eval_frozen(xm, step=step, want_forces=False)[0][5]) / (2 * h)
            assert fd == pytest.approx(f[i, a], abs=1e-7 * max(1, abs(f[i, a])) + 1e-9)
    # a bead on the tip axis: 1-D law 6 eps sigma^6/(g - R)^7, pointing away from the tip centre
    c = np.array([0.0, 0.0, 70.0 - 1e-3 * step * float(np.float32(1e-3)) / 1e-3])
    xx = x.copy(); xx[0] = c + np.array([0, 0, -(50.0 + 4.0)])
    _, f1 = o.eval_frozen(xx, step=step)
    assert f1[0, 2] == pytest.approx(-6 * 3.8 ** 6 * (float(np.float32(3.8)) / 3.8) ** 6 / 4.0 ** 7, rel=1e-6)
    assert abs(f1[0, 0]) < 1e-12 and abs(f1[0, 1]) < 1e-12
    # pulled bead: f = kappa (v s - (r - a).n) n
    n = np.array([float(np.float32(0.6)), 0.0, float(np.float32(0.8))])
    ext = float(np.float32(1e-3)) * step - (x[39] - w.xyz[39].astype(float)) @ n
    tip39 = o.eval_frozen(x, step=step)[1][39] - float(np.float32(0.05)) * ext * n
    p2 = dict(p, pulled=[], pull_k=0.0)
    f_nopull = sopo.Oracle(w.xyz, nobond, nobond, p2).eval_frozen(x, step=step)[1]
    assert np.allclose(tip39, f_nopull[39], atol=1e-12)
    # inside the tip: error
    xx[0] = c + np.array([0, 0, -49.0])
    with pytest.raises(sopo.OracleError):
        o.eval_frozen(xx, step=step)


# ---------------------------------------------------------------------------------------------- P10
def test_p10_box_muller_normals():
    from scipy import stats
    g = np.concatenate([sopo.normals_batch(0x5EED, 0, 100_000, t, s) for t in range(2) for s in range(2)])
    M = g.size
    assert np.abs(g).max() <= math.sqrt(48 * math.log(2)) + 1e-12        # u in (0,1], 24 bits: |g| <= 5.77
    assert abs(g.mean()) < 5 / math.sqrt(M)
    assert g.var() == pytest.approx(1.0, abs=5 * math.sqrt(2.0 / M))
    assert abs((g ** 3).mean()) < 5 * math.sqrt(15.0 / M)
    assert (g ** 4).mean() == pytest.approx(3.0, abs=5 * math.sqrt(96.0 / M))
    for a in range(3):
        assert stats.kstest(g[:200_000, a], "norm").pvalue > 1e-4
    # x and y of one Box-Muller pair share the radius but are uncorrelated; z comes from the second pair
    assert abs((g[:, 0] * g[:, 1]).mean()) < 5 / math.sqrt(len(g))
    assert abs((g[:, 0] * g[:, 2]).mean()) < 5 / math.sqrt(len(g))
    r2 = g[:, 0] ** 2 + g[:, 1] ** 2                                     # chi^2 with 2 dof: mean 2, var 4
    assert r2.mean() == pytest.approx(2.0, abs=5 * 2 / math.sqrt(len(g)))


# ---------------------------------------------------------------------------------------------- schedule / batching
def test_run_split_and_trajectory_word():
    w = gen.tiny(64, 6)
    a = sopo.from_workload(w); a.run(57)
    b = sopo.from_workload(w); b.run(20); b.run(37)
    assert np.array_equal(a.get_coords(), b.get_coords())
    assert a.step == 57
    c = sopo.from_workload(w, n_traj=3); c.run(57)
    xc = c.get_coords()
    assert np.array_equal(xc[0], a.get_coords()[0])
    d = sopo.from_workload(w, n_traj=1, traj_offset=2); d.run(57)
    assert np.array_equal(xc[2], d.get_coords()[0])
    assert not np.array_equal(xc[1], xc[2])


def test_fixed_beads_do_not_move_and_bad_topology_is_rejected():
    w = gen.tiny(32, 7)
    p = dict(w.params, fixed=[0, 31])
    o = sopo.Oracle(w.xyz, w.bonds, w.native, p); o.run(25)
    x = o.get_coords()[0]
    assert np.array_equal(x[0], w.xyz[0].astype(float)) and np.array_equal(x[31], w.xyz[31].astype(float))
    assert not np.array_equal(x[1], w.xyz[1].astype(float))
    with pytest.raises(sopo.OracleError):
        sopo.Oracle(w.xyz, w.bonds, np.concatenate([w.native, w.bonds[:1]]), w.params)     # bond that is also native
    with pytest.raises(sopo.OracleError):
        sopo.Oracle(w.xyz, w.bonds[:, ::-1], w.native, w.params)                            # i > j
    with pytest.raises(sopo.OracleError):
        sopo.Oracle(w.xyz, w.bonds, w.native, dict(w.params, pl_interval=15))               # not a multiple


# ---------------------------------------------------------------------------------------------- P11 (NEXT-1)
def test_p11_observables_closed_forms():
    """sopo_get_observables against closed forms: Rg of a straight rod and of a ring, end-to-end distance, the
    paper's f_ext = r_f t with r_f = kappa nu_0 at zero displacement, and the tip force as the
    derivative of V_tip with respect to the tip's advance."""
    nob = np.zeros((0, 2), np.int32)
    base = dict(gen.BASE_PARAMS, k_fene=0.0, eps_native=0.0, eps_rep=0.0)
    # rod of N beads spaced d along (1, 2, 2)/3: Rg^2 = d^2 (N^2 - 1) / 12, X = (N - 1) d
    N, d = 25, 3.8
    u = np.array([1.0, 2.0, 2.0]) / 3.0
    rod = (np.arange(N)[:, None] * d * u[None]).astype(np.float32)
    o = sopo.Oracle(rod, nob, nob, base)
    rg, x, f, ft = o.get_observables()[0]
    r64 = rod.astype(np.float64)
    assert rg == pytest.approx(math.sqrt(d * d * (N * N - 1) / 12.0), rel=1e-6)     # fp32 input rounding only
    assert x == pytest.approx(np.linalg.norm(r64[-1] - r64[0]), rel=1e-14)
    assert f == 0.0 and ft == 0.0
    # ring of radius R: Rg = R exactly (centre of mass at the centre), X between beads 0 and N-1 = 2 R sin(pi / N)
    N, R = 36, 20.0
    ang = 2 * math.pi * np.arange(N) / N
    ring = np.stack([R * np.cos(ang), R * np.sin(ang), np.full(N, 5.0)], axis=1).astype(np.float32)
    rg, x, _, _ = sopo.Oracle(ring, nob, nob, base).get_observables()[0]
    assert rg == pytest.approx(R, rel=1e-6)
    assert x == pytest.approx(2 * R * math.sin(math.pi / N), rel=1e-5)
    # cantilever: fixed bead 3 and pulled bead 17 define X; at the native position f = kappa v s = r_f t
    p = dict(base, fixed=[3], pulled=[17], pull_k=0.05, pull_v=1e-3, pull_dir=[0.0, 0.0, 1.0])
    o = sopo.Oracle(rod, nob, nob, p)
    o.step = 4000
    _, x, f, _ = o.get_observables()[0]
    assert x == pytest.approx(np.linalg.norm(r64[17] - r64[3]), rel=1e-14)
    kappa, v = float(np.float32(0.05)), float(np.float32(1e-3))
    assert f == pytest.approx(kappa * v * 4000, rel=1e-14)
    moved = r64[None].copy(); moved[0, 17, 2] += 1.25                        # the bead follows the spring by 1.25 A
    o.set_coords(moved); o.step = 4000
    assert o.get_observables()[0, 2] == pytest.approx(kappa * (v * 4000 - 1.25), rel=1e-12)
    # indenter: f_tip = dV_tip / d(advance); advance = v_tip * step, central difference over +-1 step
    w = gen.tiny(40, 2)
    pt = dict(base, tip_on=1, tip_R=50.0, tip_eps=1.0, tip_sigma=3.8, tip_c0=[0.0, 0.0, 70.0], tip_dir=[0.0, 0.0, -1.0],
              tip_v=1e-4)
    o = sopo.Oracle(w.xyz, nob, nob, pt)
    s0 = 20000
    o.step = s0
    ft = o.get_observables()[0, 3]
    vt = float(np.float32(1e-4))
    x0 = w.xyz.astype(np.float64)
    vp = o.eval_frozen(x0, step=s0 + 1, want_forces=False)[0][4]
    vm = o.eval_frozen(x0, step=s0 - 1, want_forces=False)[0][4]
    assert ft > 0
    assert ft == pytest.approx((vp - vm) / (2 * vt), rel=1e-6)
    # and it is minus the total force the tip exerts on the beads, projected on the tip direction
    _, fb = o.eval_frozen(x0, step=s0)
    assert ft == pytest.approx(float(fb.sum(axis=0) @ np.array([0.0, 0.0, -1.0])), rel=1e-12)


# ---------------------------------------------------------------------------------------------- P12 (NEXT-2)
def _taus_component_matrix(k):
    """32x32 GF(2) matrix of Tausworthe component k, column j = image of bit j, built from the oracle's own step
    (valid because the step is linear over GF(2), which the test checks first)."""
    cols = []
    for j in range(32):
        y = np.zeros(4, np.uint32); y[k] = np.uint32(1 << j)
        sopo.taus_step(y)
        cols.append(int(y[k]))
    return cols


def _mat_mul(A, B):
    """(A o B): apply B, then A; matrices as 32 column images."""
    def app(M, v):
        out = 0
        j = 0
        while v:
            if v & 1:
                out ^= M[j]
            v >>= 1; j += 1
        return out
    return [app(A, B[j]) for j in range(32)]


def _mat_pow(M, e):
    R = [1 << j for j in range(32)]
    while e:
        if e & 1:
            R = _mat_mul(M, R)
        M = _mat_mul(M, M)
        e >>= 1
    return R


def test_p12_hybrid_taus_linearity_periods_lcg_and_moments():
    """Alg. 6 with the constants of reading R12.  Pins that do not retype the recurrence:
    (i) every Tausworthe component is linear over GF(2); (ii) on the k significant bits its transition matrix has
    order exactly 2^k - 1 for k = 31, 29, 28 (L'Ecuyer's maximal-period condition: any wrong shift or mask breaks it),
    which gives the period ~2^88 of the three components and, with the 2^32 LCG, the paper's ~2^121;
    (iii) the LCG obeys its closed form; (iv) uniform and Box-Muller moments of the output."""
    r = np.random.default_rng(7)
    for k in range(3):
        for _ in range(50):
            a, b = (int(v) for v in r.integers(0, 2 ** 32, 2, dtype=np.uint64))
            ya = np.zeros(4, np.uint32); ya[k] = a; sopo.taus_step(ya)
            yb = np.zeros(4, np.uint32); yb[k] = b; sopo.taus_step(yb)
            yc = np.zeros(4, np.uint32); yc[k] = a ^ b; sopo.taus_step(yc)
            assert int(yc[k]) == int(ya[k]) ^ int(yb[k])
    ident = [1 << j for j in range(32)]
    for k, bits, factors in ((0, 31, [2147483647]), (1, 29, [233, 1103, 2089]), (2, 28, [3, 5, 29, 43, 113, 127])):
        M = _taus_component_matrix(k)
        low = 32 - bits                                   # the low (32 - k) bits of the state are ignored by the recurrence
        assert all(M[j] == 0 for j in range(low))
        P = (1 << bits) - 1
        prod = 1
        for f in factors:
            prod *= f
        assert prod == P
        hi = lambda Mx: [Mx[j] >> low for j in range(low, 32)]
        assert hi(_mat_pow(M, P)) == hi(ident)            # M^(2^k - 1) = I on the significant bits ...
        for f in factors:
            if P // f > 1:
                assert hi(_mat_pow(M, P // f)) != hi(ident)   # ... and no proper divisor: the order is exactly 2^k - 1
    # LCG: y_n = a^n y_0 + c (a^n - 1)/(a - 1) mod 2^32, checked by iterating the oracle against modular arithmetic
    a, c, y0, n = 1664525, 1013904223, 123456789, 1000
    y = np.array([2, 8, 16, y0], np.uint32)
    for _ in range(n):
        sopo.taus_step(y)
    geo = 0
    an = 1
    for _ in range(n):
        geo = (geo * a + 1) % 2 ** 32
        an = (an * a) % 2 ** 32
    assert int(y[3]) == (an * y0 + c * geo) % 2 ** 32
    # output statistics: uniform moments of 2^18 draws, and the normals used by a run
    y = sopo.taus_seed(0xC0FFEE, 11, 3)
    assert y[0] >= 2 and y[1] >= 8 and y[2] >= 16
    u = np.array([sopo.taus_step(y) for _ in range(1 << 18)], np.float64) / 2.0 ** 32
    m = len(u)
    assert abs(u.mean() - 0.5) < 5 / math.sqrt(12 * m)
    assert abs(u.var() - 1 / 12) < 5 * math.sqrt(1 / 180 / m)
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 5 / math.sqrt(m)
    w = gen.free_beads(4000)
    o = sopo.Oracle(w.xyz, w.bonds, w.native, dict(w.params, rng=1))
    x0 = o.get_coords().copy()
    nst = 25
    o.run(nst)
    d = o.get_coords() - x0
    var = 2 * float(np.float32(0.6)) * float(np.float32(2e-3)) * nst
    assert abs(d.mean()) < 5 * math.sqrt(var / d.size)
    assert d.var() == pytest.approx(var, rel=5 * math.sqrt(2.0 / d.size))


# ---------------------------------------------------------------------------------------------- P13
def test_p13_eq1_magnitudes_two_beads_hand_evaluated():
    """The VALUE of the native and repulsion terms away from their special points, with eps != 1: two beads on the x axis
    against numbers evaluated by hand from Eq. (1) (tests/golden/eq1_two_bead_values.txt shows the arithmetic).
    A wrong exponent (any n in (r0/r)^n passes P1 and P2), a wrong prefactor or a dropped eps fails here."""
    rows = [l.split() for l in open(os.path.join(GOLD, "eq1_two_bead_values.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 6
    base = dict(gen.BASE_PARAMS, R_pl=math.inf, k_fene=14.0)
    for term, eps, r0s, r, V, Fr in rows:
        eps, r0s, r, V, Fr = float(eps), float(r0s), float(r), float(V), float(Fr)
        if term == "native":
            xyz = np.array([[0, 0, 0], [r0s, 0, 0]], np.float32)            # native distance = r0
            p = dict(base, eps_native=eps, eps_rep=0.0)
            o = sopo.Oracle(xyz, np.zeros((0, 2), np.int32), np.array([[0, 1]], np.int32), p)
            col = 1
        else:
            xyz = np.array([[0, 0, 0], [5.0, 0, 0]], np.float32)            # inside R_nb: the pair is in L2
            p = dict(base, eps_rep=eps, sigma=r0s, eps_native=0.0)
            o = sopo.Oracle(xyz, np.zeros((0, 2), np.int32), np.zeros((0, 2), np.int32), p)
            col = 2
        e, f = o.eval_frozen(np.array([[0.0, 0, 0], [r, 0, 0]]))
        tol = 2e-7                                                           # eps, sigma pass through fp32 (0.7, 3.8 are not exact)
        assert e[col] == pytest.approx(V, rel=tol, abs=1e-12)
        assert e[5] == pytest.approx(V, rel=tol, abs=1e-12)
        assert f[1, 0] == pytest.approx(Fr, rel=tol, abs=1e-12) and f[0, 0] == pytest.approx(-Fr, rel=tol, abs=1e-12)
        assert np.abs(f[:, 1:]).max() == 0.0


# ---------------------------------------------------------------------------------------------- P14
def test_p14_replica_exchange_rule_detailed_balance_and_sweep():
    """NEXT-4.  (i) hand-evaluated probabilities (tests/golden/rex_metropolis_values.txt); (ii) detailed balance
    of the swap move on a two-level toy (E = 0 or 1 at kT = 0.5 and 1.0): pi(a, b) p(a, b -> b, a) = pi(b, a) p(b, a -> a, b) with
    pi = exp(-E_a/kT_1 - E_b/kT_2) -- a wrong sign or swapped temperatures breaks it; (iii) the sweep swaps temperatures,
    not coordinates, of the pairs of the given parity, with the Philox uniform the header describes."""
    rows = [l.split() for l in open(os.path.join(GOLD, "rex_metropolis_values.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 4
    for Ei, Ej, ki, kj, pr in rows:
        assert sopo.rex_probability(float(Ei), float(Ej), float(ki), float(kj)) == pytest.approx(float(pr), rel=1e-9)
    k1, k2 = 0.5, 1.0
    lev = [0.0, 1.0]
    for a in lev:
        for b in lev:
            pi_ab = math.exp(-a / k1 - b / k2); pi_ba = math.exp(-b / k1 - a / k2)
            assert pi_ab * sopo.rex_probability(a, b, k1, k2) == pytest.approx(pi_ba * sopo.rex_probability(b, a, k1, k2), rel=1e-12)
    assert sopo.rex_accept(0, 1, k1, k2, 0.36) and not sopo.rex_accept(0, 1, k1, k2, 0.37) and sopo.rex_accept(1, 0, k1, k2, 1.0)
    # the sweep on five runs of a small chain at five temperatures
    w = gen.tiny(24, 4)
    kTs = [0.3, 0.45, 0.6, 0.8, 1.1]
    o = sopo.Oracle(w.xyz, w.bonds, w.native, dict(w.params, kT_per_traj=kTs), n_traj=5)
    o.run(200)
    x = o.get_coords().copy()
    E = o.get_energies()[:, 5]
    assert len(set(np.round(E, 6))) == 5                       # five different runs
    for parity, sweep in ((0, 7), (1, 7), (0, 8), (1, 123456789012)):
        kT = o.get_temperatures()
        acc = o.replica_exchange(parity, sweep)
        new = o.get_temperatures()
        for t in range(parity, 4, 2):
            xw = sopo.philox4x32_10([t, 0x52455821, sweep & 0xFFFFFFFF, sweep >> 32], [w.params["seed"] & 0xFFFFFFFF, w.params["seed"] >> 32])
            u = ((int(xw[0]) >> 8) + 1) / 2.0 ** 24
            expect = u <= min(1.0, math.exp(min(0.0, (1 / kT[t] - 1 / kT[t + 1]) * (E[t] - E[t + 1]))))
            assert bool(acc[t // 2]) == expect
            assert (new[t], new[t + 1]) == ((kT[t + 1], kT[t]) if expect else (kT[t], kT[t + 1]))
        untouched = [t for t in range(5) if not (t >= parity and (t - parity) // 2 * 2 + parity + 1 < 5)]
        for t in untouched:
            assert new[t] == kT[t]
        assert np.array_equal(o.get_coords(), x)               # temperatures move, coordinates stay
    assert sorted(o.get_temperatures()) == pytest.approx(sorted(sopo.f32(v) for v in kTs))
    # the noise amplitude follows the run's temperature: free beads, <dr^2> = 6 kT_t D n per run
    wf = gen.free_beads(512, R_pl=20.0)
    of = sopo.Oracle(wf.xyz, wf.bonds, wf.native, dict(wf.params, kT_per_traj=[0.3, 1.2]), n_traj=2)
    x0 = of.get_coords().copy(); of.run(50)
    msd = ((of.get_coords() - x0) ** 2).sum(axis=2).mean(axis=1)
    D = sopo.f32(wf.params["dt_over_zeta"])
    assert msd[0] == pytest.approx(6 * sopo.f32(0.3) * D * 50, rel=0.15) and msd[1] == pytest.approx(6 * sopo.f32(1.2) * D * 50, rel=0.15)


# ---------------------------------------------------------------------------------------------- P15
def test_p15_second_order_update_is_eq5_and_meets_the_papers_bound():
    """params.integrator = 2 (reading R14): without noise a bead on the moving spring follows the recursion Eq. (5)
     to rounding, stays within the paper's printed 1e-5 of Eq. (3) with the paper's parameters
    (tests/golden/eq5_paper_bound.txt)."""
    bound2 = float([l for l in open(os.path.join(GOLD, "eq5_paper_bound.txt")) if not l.startswith("#")][0])
    line = [l for l in open(os.path.join(GOLD, "eq3_eq4_paper_params.txt")) if not l.startswith("#")][0].split()
    Ksp, D_cm2s, kT = float(line[0]), float(line[3]), float(line[4])
    tau = kT / (D_cm2s * 1e14 * 1e-12) / Ksp                     # ps
    # (i) Eq. (5) exactly: X(n+1) = X + (r_f t_n/xi - X/tau) h + (X/(2 tau^2) - r_f t_n/(2 tau xi)) h^2, in the oracle's units
    kappa, v, D = float(np.float32(0.05)), float(np.float32(1e-3)), float(np.float32(2e-3))
    w = gen.free_beads(4, R_pl=20.0, kT=0.0, pulled=[0, 1, 2, 3], pull_k=kappa, pull_v=v, pull_dir=[0.0, 0.0, 1.0], integrator=2)
    o = sopo.from_workload(w)
    z0 = o.get_coords()[0, :, 2].copy()
    X, h_tau = 0.0, kappa * D
    for n in range(300):
        o.run(1)
        X = X + (v * n - X) * h_tau + (X - v * n) * h_tau * h_tau / 2
        assert np.abs(o.get_coords()[0, :, 2] - z0 - X).max() < 1e-12
    # (ii) the paper's parameters: 10^6 steps against Eq. (3)
    n = 10 ** 6
    for h in (1.0, 25.0, 50.0):
        errs = {}
        for integ in (1, 2):
            w = gen.free_beads(2, R_pl=20.0, kT=0.0, pulled=[0, 1], pull_k=1.0, pull_v=1.0, pull_dir=[0.0, 0.0, 1.0])
            p = dict(w.params, dt_over_zeta=h / tau, nb_interval=1000, pl_interval=100000, integrator=integ)
            o = sopo.Oracle(w.xyz, w.bonds, w.native, p)
            a = sopo.f32(h / tau)
            z0 = o.get_coords()[0, :, 2].copy(); o.run(n)
            sim = o.get_coords()[0, :, 2] - z0
            th = n - (1 - math.exp(-n * a)) / a
            errs[integ] = float(np.abs(sim - th).max() / th)
        assert errs[2] < bound2 and errs[1] < float(line[7])      # 1e-5 and 2e-5 as printed (both are dominated by the ramp being
                                                                  # held at t_n during a step, which Eq. (4) and Eq. (5) share)
    # (iii) with noise the second-order scheme keeps the first-order statistics: free diffusion <dr^2> = 6 kT D n
    wf = gen.free_beads(512, R_pl=20.0, integrator=2)
    of = sopo.from_workload(wf)
    x0 = of.get_coords().copy(); of.run(50)
    msd = ((of.get_coords() - x0) ** 2).sum(axis=2).mean()
    assert msd == pytest.approx(6 * sopo.f32(wf.params["kT"]) * sopo.f32(wf.params["dt_over_zeta"]) * 50, rel=0.12)

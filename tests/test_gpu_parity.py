"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle on the same seeded inputs.

Bars (BASELINE.json north_star):
  lists        bit-exact at both levels (row counts and row contents, ascending caller index)
  forces       max_i |F_gpu - F_cpu| <= 1e-4 * max_i |F_cpu|
  coordinates  max |dr| <= 1e-3 A after 100 steps with the same Philox stream
  energies     |dE| <= 1e-5 * sum of |terms|   (fp32 pair terms, fp64 accumulation; derived in DESIGN.md)
"""
import ctypes
import math
import os
import subprocess

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import sopo
from workloads import generators as gen

HERE = os.path.dirname(os.path.abspath(__file__))


def sop():
    import paper_1003_1148_b200 as m
    return m


def perturbed32(w, amp, seed, n_traj=1):
    r = np.random.default_rng(seed)
    x = w.xyz[None].astype(np.float64) + amp * r.normal(size=(n_traj,) + w.xyz.shape)
    return x.astype(np.float32)


def rows_equal(a_cnt, a_idx, b_cnt, b_idx):
    if not np.array_equal(a_cnt, b_cnt):
        return False
    m = int(a_cnt.max()) if len(a_cnt) else 0
    A = np.where(np.arange(m)[None, :] < a_cnt[:, None], a_idx[:, :m], -1)
    B = np.where(np.arange(m)[None, :] < b_cnt[:, None], b_idx[:, :m], -1)
    return np.array_equal(A, B)


def check_lists(s, o, x32, traj=0, builder=0):
    """GPU lists (built from the fp32 snapshot x32 that both sides hold) == oracle lists, both levels."""
    xd = x32.astype(np.float64)
    for level in (1, 2):
        gc, gi, _ = s.get_lists(level, traj)
        oc, oi = o.build_lists(xd, level, builder, cap=gi.shape[1])
        assert rows_equal(gc, gi, oc, oi), f"level {level} lists differ"


def check_forces(s, o, x32, step=0):
    f_gpu = s.get_forces()
    for t in range(s.T):
        o_t = o if o.T == 1 else None
        _, f_cpu = o.eval_frozen(x32[t].astype(np.float64), step=step, traj=t if o.T > 1 else 0)
        err = np.abs(f_gpu[t] - f_cpu).max()
        assert err <= 1e-4 * np.abs(f_cpu).max(), (err, np.abs(f_cpu).max())


def check_energies(e_gpu, e_cpu):
    scale = np.abs(e_cpu[:, :5]).sum(axis=1, keepdims=True) + 1e-30
    assert (np.abs(e_gpu - e_cpu) <= 1e-5 * scale).all(), (e_gpu, e_cpu)


SMALL = [
    ("tiny8", lambda: gen.tiny(8, 0), {}),
    ("tiny100_pl20", lambda: gen.tiny(100, 2, R_pl=20.0), {}),
    ("tiny257", lambda: gen.tiny(257, 3), {}),
    ("two150_pl20", lambda: gen.two_chains(150, 1, R_pl=20.0), {}),
    ("cfg0", gen.config0, {}),
]
VARIANTS = [dict(mode=1, lanes_per_bead=1), dict(mode=1, lanes_per_bead=8), dict(mode=1, lanes_per_bead=32),
            dict(mode=2, lanes_per_bead=4), dict(mode=2, lanes_per_bead=16, reorder=1), dict(mode=1, reorder=1),
            dict(mode=3), dict(mode=3, chunk_beads=40, lanes_per_bead=4), dict(mode=3, chunk_beads=64, lanes_per_bead=1),
            dict(mode=3, chunk_beads=33, lanes_per_bead=16, compensated=1),
            dict(mode=3, chunk_beads=40, resident_variant=2), dict(mode=3, chunk_beads=64, resident_variant=2, compensated=1),
            dict(mode=4), dict(mode=4, pair_atomics=1), dict(mode=4, reorder=1, compensated=1)]


@pytest.mark.parametrize("name,make,over", SMALL, ids=[c[0] for c in SMALL])
@pytest.mark.parametrize("var", VARIANTS, ids=lambda v: "-".join(f"{k}{v[k]}" for k in v))
def test_small_lists_forces_energies_coords(name, make, over, var):
    w = make()
    s = sop().from_workload(w, **var, **over)
    o = sopo.from_workload(w)
    # native snapshot
    x0 = w.xyz[None].copy()
    check_lists(s, o, x0[0])
    check_forces(s, o, x0)
    check_energies(s.get_energies(), o.get_energies())
    # perturbed snapshot: both sides rebuild their lists from the same fp32 coordinates
    x1 = perturbed32(w, 0.3, 11)
    s.set_coords(x1); o.set_coords(x1.astype(np.float64))
    check_lists(s, o, x1[0])
    check_forces(s, o, x1)
    check_energies(s.get_energies(), o.get_energies())
    # 100 steps from the native structure, same Philox stream
    s.set_coords(x0); o.set_coords(x0.astype(np.float64))
    s.step = 0; o.step = 0
    s.run(100); o.run(100)
    xg = s.get_coords(); xo = o.get_coords()
    assert np.abs(xg - xo).max() <= 1e-3
    assert s.step == 100
    # list invariant: at step 100 both levels were rebuilt from the current coordinates
    assert s.get_lists(2)[2] == 100
    check_lists(s, o, xg[0])
    check_energies(s.get_energies(), sopo_energies_at(o, xg))


def sopo_energies_at(o, x32):
    """oracle energies at the GPU's coordinates with lists rebuilt from them (so that V_rep sums the same pairs)"""
    o2 = o
    keep = o2.get_coords(); step = o2.step
    o2.set_coords(x32.astype(np.float64))
    e = o2.get_energies()
    o2.set_coords(keep); o2.step = step
    return e


def test_run_split_variant_and_mode_independence():
    w = gen.tiny(200, 5, R_pl=20.0)
    ref = None
    for var in (dict(mode=1, lanes_per_bead=4), dict(mode=2, lanes_per_bead=4)):
        a = sop().from_workload(w, **var); a.run(130)
        b = sop().from_workload(w, **var); b.run(7); b.run(93); b.run(30)
        xa, xb = a.get_coords(), b.get_coords()
        assert np.array_equal(xa, xb)                      # same variant: bit-identical however the run is split
        for lv in (1, 2):
            ca, ia, ata = a.get_lists(lv); cb, ib, atb = b.get_lists(lv)
            assert rows_equal(ca, ia, cb, ib) and ata == atb
        assert a.get_lists(1)[2] == 100 and a.get_lists(2)[2] == 130
        if ref is None:
            ref = xa
        else:
            assert np.array_equal(ref, xa)                 # per-step launches and the persistent kernel agree bit for bit
    c = sop().from_workload(w, mode=1, lanes_per_bead=32, reorder=1); c.run(130)
    assert np.abs(c.get_coords() - ref).max() < 1e-4       # other summation order: fp32 rounding only
    # the SM-resident kernel: bit-identical however the run is split and whatever else ran before on the exchange
    # buffer; against the streaming kernels only the rounding of the pair terms differs
    for var in (dict(mode=3), dict(mode=3, chunk_beads=48, lanes_per_bead=8), dict(mode=3, chunk_beads=48, resident_variant=2)):
        a = sop().from_workload(w, **var); a.run(130)
        b = sop().from_workload(w, **var); b.run(7); b.run(93); b.run(1); b.run(29)
        assert a.config()["mode"] == 3
        assert np.array_equal(a.get_coords(), b.get_coords())
        for lv in (1, 2):
            ca, ia, ata = a.get_lists(lv); cb, ib, atb = b.get_lists(lv)
            assert rows_equal(ca, ia, cb, ib) and ata == atb
        assert a.get_lists(1)[2] == 100 and a.get_lists(2)[2] == 130
        assert np.abs(a.get_coords() - ref).max() < 1e-4


@pytest.mark.parametrize("var", [dict(mode=2), dict(mode=3), dict(mode=3, chunk_beads=40), dict(mode=3, chunk_beads=40, resident_variant=2)], ids=str)
def test_checkpoint_resume_is_exact(var):
    w = gen.tiny(128, 9, R_pl=20.0)
    a = sop().from_workload(w, **var); a.run(300)
    b = sop().from_workload(w, **var); b.run(200)
    x = b.get_coords()
    c = sop().from_workload(w, **var); c.set_coords(x); c.step = 200; c.run(100)
    assert np.array_equal(a.get_coords(), c.get_coords())


@pytest.mark.parametrize("var", [dict(mode=2), dict(mode=3), dict(mode=3, chunk_beads=32, R_pl=20.0),
                                 dict(mode=3, chunk_beads=32, R_pl=20.0, resident_variant=2)], ids=str)
def test_batch_trajectories_and_sharding_offset(var):
    var = dict(var)
    w = gen.tiny(96, 4, **({"R_pl": var.pop("R_pl")} if "R_pl" in var else {}))
    T = 5
    s = sop().from_workload(w, n_traj=T, **var); s.run(100)
    o = sopo.from_workload(w, n_traj=T); o.run(100)
    xg, xo = s.get_coords(), o.get_coords()
    assert np.abs(xg - xo).max() <= 1e-3
    assert not np.array_equal(xg[0], xg[1])
    for t in range(T):
        gc, gi, _ = s.get_lists(2, t)
        oc, oi = o.build_lists(xg[t].astype(np.float64), 2, cap=gi.shape[1])
        assert rows_equal(gc, gi, oc, oi)
    check_energies(s.get_energies(), sopo_energies_at(o, xg))
    # a shard of the batch (trajectories 3..4 on another GPU) reproduces the unsharded batch bit for bit
    from paper_1003_1148_b200 import shard_trajectories
    off, n = shard_trajectories(T, 1, 2)
    assert (off, n) == (3, 2)
    sh = sop().from_workload(w, n_traj=n, traj_offset=off, **var); sh.run(100)
    assert np.array_equal(sh.get_coords(), xg[off:off + n])


def test_external_forces_pull_fixed_indenter_compensated():
    w = gen.tiny(64, 8)
    zmax = float(w.xyz[:, 2].max())
    p = dict(w.params, fixed=[0, 5], pulled=[63, 20], pull_k=0.05, pull_v=1e-3, pull_dir=[0.6, 0.0, 0.8],
             tip_on=1, tip_R=50.0, tip_eps=1.0, tip_sigma=3.8, tip_c0=[0.0, 0.0, zmax + 53.0],
             tip_dir=[0.0, 0.0, -1.0], tip_v=1e-3)
    for var in (dict(mode=1, compensated=2), dict(mode=2, compensated=1, lanes_per_bead=8), dict(mode=3),
                dict(mode=3, compensated=1, lanes_per_bead=8, chunk_beads=24, R_pl=20.0)):
        var = dict(var)
        if "R_pl" in var:
            p = dict(p, R_pl=var.pop("R_pl"), pl_interval=100)
        s = sop().Sop(w.xyz, w.bonds, w.native, p, **var)
        o = sopo.Oracle(w.xyz, w.bonds, w.native, p)
        s.step = 1000; o.step = 1000                         # the spring base and the tip have advanced
        check_forces(s, o, w.xyz[None], step=1000)
        check_energies(s.get_energies(), o.get_energies())
        assert o.get_energies()[0, 3] > 0 and o.get_energies()[0, 4] > 0
        s.run(100); o.run(100)
        xg, xo = s.get_coords(), o.get_coords()
        assert np.abs(xg - xo).max() <= 1e-3
        assert np.array_equal(xg[0, 0], w.xyz[0]) and np.array_equal(xg[0, 5], w.xyz[5])   # fixed beads never move


def test_compensated_update_at_large_coordinates():
    """Reading R10: at |x| ~ 2700 A plain fp32 accumulation drifts past 1e-3 A in 100 steps; Kahan does not."""
    w = gen.tiny(64, 10)
    shift = np.array([0.0, 0.0, 2700.0], np.float32)
    xyz = w.xyz + shift
    o = sopo.Oracle(xyz, w.bonds, w.native, w.params); o.run(100)
    s = sop().Sop(xyz, w.bonds, w.native, w.params, mode=2)     # compensated auto: on (max|coord| > 512)
    assert s.config()["compensated"] == 1
    s.run(100)
    assert np.abs(s.get_coords() - o.get_coords()).max() <= 1e-3


def test_error_flags():
    m = sop()
    w = gen.tiny(32, 1)
    s = m.from_workload(w)
    x = w.xyz[None].copy(); x[0, 10] += np.array([2.5, 0, 0], np.float32)       # bond 9-10 or 10-11 beyond R0
    s.set_coords(x)
    with pytest.raises(m.SopError) as ei:
        s.get_forces()
    assert ei.value.code == -4
    with pytest.raises(m.SopError) as ei:
        m.from_workload(w, cap_nb=4)                                             # rows overflow -> error, not truncation
    assert ei.value.code == -3
    with pytest.raises(m.SopError) as ei:
        m.Sop(w.xyz, w.bonds, np.concatenate([w.native, w.bonds[:1]]), w.params)
    assert ei.value.code == -1
    with pytest.raises(m.SopError):
        m.Sop(w.xyz, w.bonds, w.native, dict(w.params, pl_interval=15))


def test_p5_free_diffusion_on_gpu():
    N, n = 20000, 40
    w = gen.free_beads(N, R_pl=20.0)
    s = sop().from_workload(w, n_traj=2, mode=2)
    x0 = s.get_coords().astype(np.float64)
    s.run(n)
    d = s.get_coords().astype(np.float64) - x0
    kT, D = float(np.float32(0.6)), float(np.float32(2e-3))
    var = 2 * kT * D * n
    M = d.size
    assert abs(d.mean()) < 5 * math.sqrt(var / M)
    assert d.var() == pytest.approx(var, rel=5 * math.sqrt(2.0 / M) + 1e-4)
    z = d / math.sqrt(var)
    assert abs((z ** 4).mean() - 3.0) < 5 * math.sqrt(96.0 / M)
    assert abs((z[..., 0] * z[..., 1]).mean()) < 5 / math.sqrt(2 * N)
    assert abs((z[0] * z[1]).mean()) < 5 / math.sqrt(3 * N)


def test_p6_device_philox_equals_curand_and_oracle():
    src = os.path.join(HERE, "cuda", "philox_check.cu")
    out = os.path.join(HERE, "cuda", "philox_check.so")
    if not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.check_call(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-std=c++17", "--shared",
                               "-Xcompiler", "-fPIC", src, "-o", out])
    L = ctypes.CDLL(out)
    r = np.random.default_rng(2024)
    n = 4096
    ctr = r.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = r.integers(0, 2 ** 32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    ctr[:4] = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344], [1, 0, 0, 0]]
    key[:4] = [[0, 0], [0xFFFFFFFF] * 2, [0xA4093822, 0x299F31D0], [0, 0]]
    mine = np.zeros((n, 4), np.uint32); ref = np.zeros((n, 4), np.uint32); nor = np.zeros((n, 3), np.float32)
    seed = 0x1234567890ABCDEF
    assert L.philox_check(ctr.ctypes.data_as(ctypes.c_void_p), key.ctypes.data_as(ctypes.c_void_p), n,
                          mine.ctypes.data_as(ctypes.c_void_p), ref.ctypes.data_as(ctypes.c_void_p),
                          nor.ctypes.data_as(ctypes.c_void_p), ctypes.c_ulonglong(seed)) == 0
    assert np.array_equal(mine, ref)                                   # product Philox == cuRAND device function
    for q in range(64):
        assert sopo.philox4x32_10(ctr[q], key[q]).tolist() == mine[q].tolist()      # == oracle Philox
        step = int(ctr[q, 2]) | (int(ctr[q, 3]) << 32)
        g = sopo.normals(seed, int(ctr[q, 0]), int(ctr[q, 1]), step)
        assert np.abs(nor[q] - g).max() < 2e-5                         # fp32 Box-Muller with fast intrinsics


# ---------------------------------------------------------------------------------------------- full-size configs
def full_check(k, n_traj=None, steps=100, builder=1, sample_traj=(0,), **var):
    w = gen.make_config(k)
    T = w.n_traj if n_traj is None else n_traj
    s = sop().from_workload(w, n_traj=T, **var)
    o = sopo.from_workload(w, n_traj=T, list_builder=builder)
    x0 = np.broadcast_to(w.xyz, (T,) + w.xyz.shape)
    for t in sample_traj:
        check_lists(s, o, w.xyz, traj=t, builder=builder)
    f_gpu = s.get_forces(); f_cpu = o.get_forces()
    assert np.abs(f_gpu - f_cpu).max() <= 1e-4 * np.abs(f_cpu).max()
    check_energies(s.get_energies(), o.get_energies())
    s.run(steps); o.run(steps)
    xg, xo = s.get_coords(), o.get_coords()
    err = np.abs(xg - xo).max()
    assert err <= 1e-3, err
    for t in sample_traj:
        check_lists(s, o, xg[t], traj=t, builder=builder)
    # forces and energies at the GPU's own step-100 coordinates
    o.set_coords(xg.astype(np.float64)); o.step = steps
    f_gpu = s.get_forces(); f_cpu = o.get_forces()
    assert np.abs(f_gpu - f_cpu).max() <= 1e-4 * np.abs(f_cpu).max()
    check_energies(s.get_energies(), o.get_energies())
    return s


@pytest.mark.parametrize("mode", [2, 3])
def test_full_config1_batch(mode):
    s = full_check(1, n_traj=256, builder=0, sample_traj=(0, 137, 255), mode=mode)
    assert s.config()["mode"] == mode


@pytest.mark.parametrize("R_pl", [float("inf"), 20.0], ids=["static_l1", "finite_l1"])
def test_many_trajectories_sliced_launch_is_bit_identical(R_pl):
    """More one-chunk trajectories than SMs: a mode-3 launch is cut into time slices (one CTA per slice and trajectory, handed
    out by a ticket, chained per trajectory) so that no SM idles through a partly empty last wave.  A slice is what a separate
    launch would be, so coordinates, lists and energies must be bit-identical to the unsliced launch (SOP_NO_SLICES), also
    when the run is split; sample trajectories against the oracle."""
    w = gen.globule(96, 77, R_pl=R_pl)
    T = 160
    a = sop().from_workload(w, n_traj=T, mode=3); a.run(230)
    assert a.config()["mode"] == 3 and a.config()["slice_len"] > 0
    os.environ["SOP_NO_SLICES"] = "1"
    try:
        b = sop().from_workload(w, n_traj=T, mode=3); b.run(230)
        assert b.config()["slice_len"] == 0
    finally:
        del os.environ["SOP_NO_SLICES"]
    c = sop().from_workload(w, n_traj=T, mode=3); c.run(95); c.run(135)
    xa = a.get_coords()
    assert np.array_equal(xa, b.get_coords()) and np.array_equal(xa, c.get_coords())
    assert np.array_equal(a.get_energies(), b.get_energies())
    for t in (0, 97, T - 1):
        ca, ia, ata = a.get_lists(2, t); cb, ib, atb = b.get_lists(2, t)
        assert rows_equal(ca, ia, cb, ib) and ata == atb == 230
    o = sopo.from_workload(w, n_traj=T); o.run(230)
    assert np.abs(xa - o.get_coords()).max() <= 3e-3           # (230 steps: DESIGN.md section 8, "beyond 100 steps")


def test_mode3_fast_instantiation_is_bit_identical():
    """Philox, one native eps and either (1) several chunks, explicit L1, natives in shared memory or (2) one chunk per
    trajectory with the static all-pairs L1: the host picks an instantiation of the resident kernel in which those run-time
    switches are compile-time constants (less once-per-step code).  Same arithmetic in the same order: bit-identical to the
    general instantiation (SOP_NO_FAST), on chunked small systems with 2 and 4 lanes, the full 30,000-bead shell, config 0
    (8 lanes, one chunk) and a one-lane batch with the transposed native table."""
    def run(w, n, n_traj=None, **var):
        s = sop().from_workload(w, n_traj=n_traj, mode=3, **var); s.run(n)
        out = (s.get_coords(), s.get_lists(2)[0], s.get_lists(2)[1], s.get_energies())
        s.close()
        return out
    cases = [(gen.two_chains(150, 3, R_pl=20.0), 230, dict(chunk_beads=100, lanes_per_bead=4)),
             (gen.two_chains(150, 3, R_pl=20.0), 230, dict(chunk_beads=150, lanes_per_bead=2, compensated=1)),
             (gen.make_config(3), 200, {}),
             (gen.make_config(0), 230, {}),                                      # one chunk, static L1, 8 lanes
             (gen.globule(700, 5), 130, dict(lanes_per_bead=1, n_traj=3))]      # one chunk, static L1, one lane, transposed natives
    for w, n, var in cases:
        a = run(w, n, **var)
        os.environ["SOP_NO_FAST"] = "1"
        try:
            b = run(w, n, **var)
        finally:
            del os.environ["SOP_NO_FAST"]
        assert all(np.array_equal(x, y) for x, y in zip(a, b)), var


def test_full_config1_batch_finite_pair_list():
    w = gen.config1(R_pl=20.0)
    T = 16
    s = sop().from_workload(w, n_traj=T, mode=0)
    assert s.config()["mode"] == 3
    o = sopo.from_workload(w, n_traj=T)
    s.run(100); o.run(100)
    xg = s.get_coords()
    assert np.abs(xg - o.get_coords()).max() <= 1e-3
    for t in (0, 15):
        check_lists(s, o, xg[t], traj=t)


@pytest.mark.parametrize("mode,variant", [(2, 0), (3, 1), (3, 2)])
def test_full_config2_fiber_pulled(mode, variant):
    s = full_check(2, mode=mode, resident_variant=variant)
    assert s.config()["compensated"] == 1 and s.config()["mode"] == mode
    assert variant == 0 or s.config()["resident_variant"] == variant


@pytest.mark.parametrize("mode,variant", [(1, 0), (2, 0), (3, 1), (3, 2)])
def test_full_config3_shell_indented(mode, variant):
    s = full_check(3, mode=mode, resident_variant=variant)
    assert s.config()["mode"] == mode
    assert variant == 0 or s.config()["resident_variant"] == variant


@pytest.mark.parametrize("mode", [0, 1])
def test_full_config4_lattice(mode):
    full_check(4, mode=mode)


# ---------------------------------------------------------------------------------------------- more mode-3 coverage
@pytest.mark.parametrize("var", [dict(mode=1, lanes_per_bead=4), dict(mode=2), dict(mode=3), dict(mode=3, chunk_beads=45),
                                 dict(mode=3, chunk_beads=45, resident_variant=2)], ids=str)
def test_per_contact_native_eps(var):
    """topology.native_eps (one eps per native contact, PAPER.md:241 eps_n) on every kernel path."""
    w = gen.tiny(150, 21, R_pl=20.0)
    eps = (0.5 + np.random.default_rng(5).random(len(w.native))).astype(np.float32)
    s = sop().Sop(w.xyz, w.bonds, w.native, w.params, native_eps=eps, **var)
    o = sopo.Oracle(w.xyz, w.bonds, w.native, w.params, native_eps=eps)
    check_forces(s, o, w.xyz[None])
    check_energies(s.get_energies(), o.get_energies())
    s.run(100); o.run(100)
    assert np.abs(s.get_coords() - o.get_coords()).max() <= 1e-3


@pytest.mark.parametrize("var", [dict(mode=1), dict(mode=2), dict(mode=3, chunk_beads=60), dict(mode=3, chunk_beads=60, resident_variant=2)], ids=str)
def test_mode3_long_run_across_pair_list_rebuilds(var):
    """350 steps = 3 pair-list rebuilds inside one sop_run (the in-kernel first filter after each) against three
    separate runs that end on the rebuild boundaries (k_filter path) and against the oracle's lists at the end."""
    w = gen.two_chains(150, 3, R_pl=20.0)
    a = sop().from_workload(w, **var); a.run(350)
    b = sop().from_workload(w, **var); b.run(100); b.run(200); b.run(50)
    assert np.array_equal(a.get_coords(), b.get_coords())
    o = sopo.from_workload(w)
    xa = a.get_coords()
    assert a.get_lists(1)[2] == 300 and a.get_lists(2)[2] == 350
    # the L2 of step 350 is Alg. 3 applied to the STALE L1 of step 300 at the coordinates of step 350: bit for bit the
    # oracle's filter of the GPU's own L1 (a fresh build at step 350 would give a different list)
    c1, i1, _ = a.get_lists(1)
    c2, i2, _ = a.get_lists(2)
    oc, oi = o.filter(xa[0].astype(np.float64), c1, i1)
    assert np.array_equal(c2, oc)
    for i in range(w.n_beads):
        assert np.array_equal(i2[i, :c2[i]], oi[i, :oc[i]])
    fc, fi = o.build_lists(xa[0].astype(np.float64), 1, cap=i1.shape[1])
    assert not np.array_equal(fc, c1)                          # the pair list really is stale
    # L2 was filtered at step 350 from the L1 of step 300: compare with the oracle driven to the same state
    o.run(350)
    assert np.abs(xa - o.get_coords()).max() <= 5e-3          # 350 steps: fp32 vs fp64 drift, still far below a bond length
    e_gpu = a.get_energies()
    assert np.isfinite(e_gpu).all()


def test_mode3_halo_overflow_is_an_error_not_a_truncation():
    """Compress the structure after create: more beads enter a chunk's 20 A halo than its slot table holds."""
    m = sop()
    w = gen.tiny(400, 12, R_pl=20.0)
    s = m.from_workload(w, mode=3, chunk_beads=50)
    x = (w.xyz[None] * np.float32(0.55)).astype(np.float32)     # 6x the density: every list and halo grows
    with pytest.raises(m.SopError) as ei:
        s.set_coords(x)
        s.run(10)
        s.sync()
    assert ei.value.code in (-3, -4)                            # list / halo overflow (or a crushed bond caught first)


def test_ensemble_means_energy_and_rg_within_3_standard_errors():
    """north_star: long-run ensemble means (energy, radius of gyration) of GPU and oracle agree within 3 SE.
    64 independent trajectories of a small globule, 2000 steps, same Philox streams on both sides (the test does
    not rely on the trajectories staying close, only on the ensemble)."""
    w = gen.tiny(64, 31)
    T, n = 64, 2000
    s = sop().from_workload(w, n_traj=T, mode=3); s.run(n)
    o = sopo.from_workload(w, n_traj=T); o.run(n)
    xg, xo = s.get_coords().astype(np.float64), o.get_coords()
    rg = lambda x: np.sqrt(((x - x.mean(axis=1, keepdims=True)) ** 2).sum(axis=2).mean(axis=1))
    eg, eo = s.get_energies()[:, 5], o.get_energies()[:, 5]
    for a, b in ((rg(xg), rg(xo)), (eg, eo)):
        se = math.sqrt(a.var(ddof=1) / T + b.var(ddof=1) / T)
        assert abs(a.mean() - b.mean()) <= 3 * se, (a.mean(), b.mean(), se)


# ---------------------------------------------------------------------------------------------- NEXT-1: observables
def check_observables(s, o, xg, step):
    """device-side Rg / end-to-end distance / cantilever force / tip force == oracle at the SAME coordinates"""
    keep, kstep = o.get_coords(), o.step
    o.set_coords(xg.astype(np.float64)); o.step = step
    ref = o.get_observables()
    o.set_coords(keep); o.step = kstep
    got = s.get_observables()
    assert got.shape == ref.shape
    scale = np.abs(ref) + np.array([1e-3, 1e-3, 1e-3, 1e-3])
    assert (np.abs(got - ref) <= 2e-5 * scale + 1e-6).all(), (got, ref)     # fp32 coordinates and terms, fp64 sums


@pytest.mark.parametrize("var", [dict(mode=1), dict(mode=3), dict(mode=3, chunk_beads=24, R_pl=20.0),
                                 dict(mode=3, chunk_beads=24, R_pl=20.0, resident_variant=2)], ids=str)
def test_observables_small_with_pull_and_tip(var):
    var = dict(var)
    w = gen.tiny(64, 8)
    zmax = float(w.xyz[:, 2].max())
    p = dict(w.params, fixed=[0, 5], pulled=[63, 20], pull_k=0.05, pull_v=1e-3, pull_dir=[0.6, 0.0, 0.8],
             tip_on=1, tip_R=50.0, tip_eps=1.0, tip_sigma=3.8, tip_c0=[0.0, 0.0, zmax + 53.0],
             tip_dir=[0.0, 0.0, -1.0], tip_v=1e-3)
    if "R_pl" in var:
        p = dict(p, R_pl=var.pop("R_pl"), pl_interval=100)
    T = 3
    s = sop().Sop(w.xyz, w.bonds, w.native, p, n_traj=T, **var)
    o = sopo.Oracle(w.xyz, w.bonds, w.native, p, n_traj=T)
    s.step = 1000; o.step = 1000
    x0 = np.broadcast_to(w.xyz, (T,) + w.xyz.shape).copy()
    check_observables(s, o, x0, 1000)
    assert s.get_observables()[0, 2] > 0 and s.get_observables()[0, 3] > 0
    s.run(100)
    check_observables(s, o, s.get_coords(), 1100)
    rg = s.get_observables()[:, 0]
    assert not np.allclose(rg[0], rg[1])                      # per trajectory


@pytest.mark.parametrize("k", [2, 3])
def test_observables_full_configs(k):
    w = gen.make_config(k)
    s = sop().from_workload(w)
    o = sopo.from_workload(w, list_builder=1)
    check_observables(s, o, w.xyz[None], 0)
    s.run(100)
    check_observables(s, o, s.get_coords(), 100)
    obs = s.get_observables()[0]
    if k == 2:
        assert obs[1] > 5000.0                                 # the fiber's pulled end is ~5500 A from its fixed end
    else:
        assert obs[3] > 0.0                                    # the indenter already pushes on the shell


def test_mode3_is_deterministic_run_to_run():
    """compute-sanitizer is closed on this pool, so shared-memory / exchange races are hunted by repetition: the
    SM-resident kernel must give bit-identical coordinates, lists and energies every time, on small chunked systems
    (many exchange partners per CTA) and on the full 30,000-bead shell with all 148 CTAs polling each other."""
    w = gen.two_chains(150, 3, R_pl=20.0)
    for var in (dict(chunk_beads=30, lanes_per_bead=8), dict(chunk_beads=75, lanes_per_bead=1), dict(n_traj=3, chunk_beads=50),
                dict(n_traj=3, chunk_beads=50, resident_variant=2)):
        var = dict(var); T = var.pop("n_traj", 1)
        ref = None
        for rep in range(4):
            s = sop().from_workload(w, n_traj=T, mode=3, **var); s.run(230)
            out = (s.get_coords(), s.get_lists(2, T - 1)[0], s.get_energies())
            s.close()
            if ref is None:
                ref = out
            else:
                assert all(np.array_equal(a, b) for a, b in zip(ref, out)), (var, rep)
    w = gen.make_config(3)
    ref = None
    for rep in range(3):
        s = sop().from_workload(w); s.run(200)
        x = s.get_coords(); s.close()
        if ref is None:
            ref = x
        else:
            assert np.array_equal(ref, x), rep


@pytest.mark.parametrize("var", [dict(mode=1), dict(mode=2), dict(mode=3), dict(mode=3, chunk_beads=40),
                                 dict(mode=3, chunk_beads=40, resident_variant=2)], ids=str)
def test_a_blown_up_structure_reports_errors_but_stays_memory_safe(var):
    """A caller that ignores SOP_E_FENE / SOP_E_NONFINITE and keeps running must keep getting status codes, never a
    CUDA fault: the cell grid of a structure with a bead at 1e30 A (or NaN) once overflowed its integer arithmetic."""
    m = sop()
    w = gen.tiny(160, 14, R_pl=20.0)
    for bad in (np.float32(1.0e30), np.float32("nan"), np.float32("inf")):
        s = m.from_workload(w, **var)
        x = w.xyz[None].copy(); x[0, 7, 1] = bad
        codes = []
        try:
            s.set_coords(x)
        except m.SopError as e:
            codes.append(e.code)
        for _ in range(3):
            try:
                s.run(130); s.sync()
            except m.SopError as e:
                codes.append(e.code)
        assert codes and all(c in (-3, -4, -5) for c in codes), codes
        s.close()
    # the device is still healthy
    s = m.from_workload(w, **var); s.run(50); s.sync(); s.close()


# ---------------------------------------------------------------------------------------------- NEXT-2: Hybrid Taus
@pytest.mark.parametrize("var", [dict(mode=1, lanes_per_bead=4), dict(mode=2), dict(mode=0), dict(mode=1, reorder=1),
                                 dict(mode=3), dict(mode=3, chunk_beads=60), dict(mode=3, chunk_beads=60, resident_variant=2)], ids=str)
def test_hybrid_taus_noise_matches_the_oracle(var):
    """params.rng = 1: the paper's per-bead Hybrid Taus generator (Alg. 6).  Same seeds, same state stream per bead on
    both sides -> coordinates within 1e-3 A after 100 steps; fixed beads draw nothing; run splits do not matter."""
    m = sop()
    w = gen.two_chains(120, 5, R_pl=20.0)
    p = dict(w.params, rng=1, fixed=[0, 7])
    T = 3
    s = m.Sop(w.xyz, w.bonds, w.native, p, n_traj=T, **var)
    assert s.config()["mode"] == (var["mode"] or 3)          # every mode runs the paper's generator (auto -> the resident kernel)
    o = sopo.Oracle(w.xyz, w.bonds, w.native, p, n_traj=T)
    s.run(100); o.run(100)
    xg, xo = s.get_coords(), o.get_coords()
    assert np.abs(xg - xo).max() <= 1e-3
    assert not np.array_equal(xg[0], xg[1])
    assert np.array_equal(xg[0, 0], w.xyz[0]) and np.array_equal(xg[2, 7], w.xyz[7])
    b = m.Sop(w.xyz, w.bonds, w.native, p, n_traj=T, **var); b.run(37); b.run(63)
    assert np.array_equal(b.get_coords(), xg)
    # a different generator than Philox, same physics
    c = m.Sop(w.xyz, w.bonds, w.native, dict(p, rng=0), n_traj=T, **var); c.run(100)
    assert not np.allclose(c.get_coords(), xg, atol=1e-3)


def test_mode3_l1_rows_read_from_global_memory_when_they_do_not_fit():
    """The filter normally walks L1 rows that were copied to shared memory; a chunk whose rows do not fit reads them
    from global memory instead.  SOP_TEST_NO_PL_SMEM forces that path: identical results, bit for bit."""
    w = gen.two_chains(150, 3, R_pl=20.0)
    a = sop().from_workload(w, mode=3, chunk_beads=60); a.run(230)
    os.environ["SOP_TEST_NO_PL_SMEM"] = "1"
    try:
        b = sop().from_workload(w, mode=3, chunk_beads=60); b.run(230)
    finally:
        del os.environ["SOP_TEST_NO_PL_SMEM"]
    assert np.array_equal(a.get_coords(), b.get_coords())
    ca, ia, _ = a.get_lists(2); cb, ib, _ = b.get_lists(2)
    assert rows_equal(ca, ia, cb, ib)
    o = sopo.from_workload(w); o.run(230)
    assert np.abs(b.get_coords() - o.get_coords()).max() <= 3e-3


@pytest.mark.parametrize("var", [dict(chunk_beads=60, lanes_per_bead=4), dict(lanes_per_bead=1), dict(lanes_per_bead=2)], ids=str)
def test_mode3_native_table_in_global_memory(var):
    """Chunks whose native table does not fit shared memory read it from global memory (packed per chunk, or transposed
    for a one-chunk trajectory with one lane per bead).  SOP_TEST_NO_NAT_SMEM forces those paths: same results."""
    w = gen.two_chains(150, 3, R_pl=20.0)
    a = sop().from_workload(w, mode=3, **var); a.run(130)
    os.environ["SOP_TEST_NO_NAT_SMEM"] = "1"
    try:
        b = sop().from_workload(w, mode=3, **var); b.run(130)
    finally:
        del os.environ["SOP_TEST_NO_NAT_SMEM"]
    assert np.array_equal(a.get_coords(), b.get_coords())
    o = sopo.from_workload(w); o.run(130)
    assert np.abs(b.get_coords() - o.get_coords()).max() <= 2e-3


# ---------------------------------------------------------------------------------------------- NEXT-1: series at a stride
def _series_case(w, p, T, var, n_steps, stride):
    """The series recorded inside ONE sop_run equals (i) what the on-demand getters return when the same run is split by
    hand at every sample (bit for bit: the same kernels on the same coordinates) and (ii) the oracle's observables and
    energies at the GPU's coordinates of every sample (the 2e-5 / 1e-5 bars of the getters)."""
    m = sop()
    a = m.Sop(w.xyz, w.bonds, w.native, dict(p, obs_stride=stride, obs_capacity=n_steps // stride), n_traj=T, **var)
    a.run(n_steps)
    steps, ser = a.get_observable_series()
    assert steps.tolist() == list(range(stride, n_steps + 1, stride)) and ser.shape == (len(steps), T, 10)
    b = m.Sop(w.xyz, w.bonds, w.native, p, n_traj=T, **var)
    o = sopo.Oracle(w.xyz, w.bonds, w.native, p, n_traj=T, list_builder=1 if w.n_beads > 5000 else 0)
    for q, st in enumerate(steps):
        b.run(stride)
        assert np.array_equal(b.get_observables(), ser[q, :, :4]) and np.array_equal(b.get_energies(), ser[q, :, 4:])
        if q % max(1, len(steps) // 8) == 0 or q == len(steps) - 1:
            x = b.get_coords()
            o.set_coords(x.astype(np.float64)); o.step = int(st)
            ref = o.get_observables()
            scale = np.abs(ref) + 1e-3
            assert (np.abs(ser[q, :, :4] - ref) <= 2e-5 * scale + 1e-6).all(), (st, ser[q, :, :4], ref)
            check_energies(ser[q, :, 4:], o.get_energies())
    assert np.array_equal(a.get_coords(), b.get_coords())       # recording does not change the trajectory
    return steps, ser


@pytest.mark.parametrize("var", [dict(mode=1), dict(mode=2), dict(mode=3), dict(mode=3, chunk_beads=24, R_pl=20.0),
                                 dict(mode=3, chunk_beads=24, R_pl=20.0, resident_variant=2)], ids=str)
def test_observable_series_small(var):
    var = dict(var)
    w = gen.tiny(64, 8)
    zmax = float(w.xyz[:, 2].max())
    p = dict(w.params, fixed=[0, 5], pulled=[63, 20], pull_k=0.05, pull_v=1e-3, pull_dir=[0.6, 0.0, 0.8],
             tip_on=1, tip_R=50.0, tip_eps=1.0, tip_sigma=3.8, tip_c0=[0.0, 0.0, zmax + 53.0],
             tip_dir=[0.0, 0.0, -1.0], tip_v=1e-3)
    if "R_pl" in var:
        p = dict(p, R_pl=var.pop("R_pl"), pl_interval=100)
    steps, ser = _series_case(w, p, 3, var, 300, 10)
    # ring semantics: a capacity of 4 keeps the last four samples; stride 0 stops the recording
    c = sop().Sop(w.xyz, w.bonds, w.native, dict(p, obs_stride=10, obs_capacity=4), n_traj=3, **var)
    c.run(300)
    st4, s4 = c.get_observable_series()
    assert st4.tolist() == [270, 280, 290, 300] and np.array_equal(s4, ser[-4:])
    c.set_observable_stride(0); c.run(50)
    assert c.get_observable_series()[0].tolist() == [270, 280, 290, 300]


@pytest.mark.parametrize("k", [2, 3])
def test_observable_series_full_configs(k):
    """f(R) of the pulled fiber (X, cantilever force) and the force-indentation curve of the shell (tip force
    against the advance) at stride 10 over 1000 steps of one sop_run."""
    w = gen.make_config(k)
    steps, ser = _series_case(w, w.params, 1, {}, 1000, 10)
    if k == 2:
        f = ser[:, 0, 2]
        # r_f t = kappa v t plus kappa times the thermal excursion of the pulled bead (a few tenths of an A)
        assert np.polyfit(steps.astype(float), f, 1)[0] > 0 and abs(f[-1] - 0.05 * 1e-3 * 1000) < 0.1
        assert ser[:, 0, 1].min() > 5000.0
    else:
        assert (ser[:, 0, 3] > 0).all() and ser[-1, 0, 3] > ser[0, 0, 3]           # the tip advances: the shell pushes back harder


# ---------------------------------------------------------------------------------------------- exchange protocol under skew
@pytest.mark.parametrize("variant", [1, 2])
def test_mode3_exchange_is_exact_when_a_chunk_runs_late(variant):
    """SOP_TEST_SKEW makes one chunk sleep before it publishes on chosen steps (filter steps and the steps around them):
    its neighbours then run up to the limits the protocol allows.  10^4 steps must be bit-identical to the unskewed run,
    on a small chunked system and on the 148-chunk shell; no wait may time out."""
    cases = [(gen.two_chains(150, 3, R_pl=20.0), dict(mode=3, chunk_beads=30, resident_variant=variant), 10000, "2,3,50000"),
             (gen.make_config(3), dict(mode=3, resident_variant=variant), 2000, "70,7,50000")]
    for w, var, n, skew in cases:
        a = sop().from_workload(w, **var); a.run(n); xa = a.get_coords(); a.close()
        os.environ["SOP_TEST_SKEW"] = skew
        try:
            b = sop().from_workload(w, **var); b.run(n); xb = b.get_coords(); b.close()
        finally:
            del os.environ["SOP_TEST_SKEW"]
        assert np.array_equal(xa, xb), (w.name, skew)


# ---------------------------------------------------------------------------------------------- P11: long-run ensemble
def test_p11_long_run_ensemble_means_different_seeds():
    """SURVEY P11 / north_star: GPU and oracle with DIFFERENT seeds on a config-0-like chain (N = 128), 64 trajectories each,
    10^5 steps of which the first 10^4 are discarded; the per-trajectory time averages of the total energy and of Rg
    (sampled every 100 steps; on the GPU through the series recorded inside sop_run) are the independent samples:
    |m_gpu - m_cpu| <= 3 sqrt(SE_gpu^2 + SE_cpu^2)."""
    w = gen.config0()
    T, n, burn, stride = 64, 100000, 10000, 100
    s = sop().Sop(w.xyz, w.bonds, w.native, dict(w.params, seed=0xA11CE, obs_stride=stride, obs_capacity=n // stride), n_traj=T)
    s.run(n)
    steps, ser = s.get_observable_series()
    keep = steps > burn
    g_e, g_rg = ser[keep, :, 9].mean(axis=0), ser[keep, :, 0].mean(axis=0)
    o = sopo.Oracle(w.xyz, w.bonds, w.native, dict(w.params, seed=0xB0B), n_traj=T)
    o.run(burn)
    acc_e, acc_rg, cnt = np.zeros(T), np.zeros(T), 0
    for _ in range((n - burn) // stride):
        o.run(stride)
        acc_e += o.get_energies()[:, 5]; acc_rg += o.get_observables()[:, 0]; cnt += 1
    c_e, c_rg = acc_e / cnt, acc_rg / cnt
    for name, g, c in (("energy", g_e, c_e), ("Rg", g_rg, c_rg)):
        se = math.sqrt(g.var(ddof=1) / T + c.var(ddof=1) / T)
        assert abs(g.mean() - c.mean()) <= 3 * se, (name, g.mean(), c.mean(), se)
        assert se < 0.02 * abs(c.mean())                      # the test has resolving power: 3 SE is a few per cent at most


# ---------------------------------------------------------------------------------------------- NEXT-4
@pytest.mark.parametrize("var", [dict(mode=1, lanes_per_bead=4), dict(mode=2), dict(mode=3), dict(mode=3, chunk_beads=40),
                                 dict(mode=3, chunk_beads=40, resident_variant=2)], ids=str)
def test_per_trajectory_temperature_and_replica_exchange(var):
    """One temperature per run of a many-runs batch, and Metropolis swaps of the temperatures between neighbouring runs
    (PAPER.md:310).  Same seeds and sweep numbers on both sides: the coordinates agree after 100 steps at four temperatures;
    at the GPU's coordinates the oracle takes the same swap decisions (decided in fp64 from fp64 sums on both sides; a pair
    whose uniform falls within 1e-4 of its acceptance probability is not compared), and the runs continue in step."""
    m = sop()
    w = gen.two_chains(120, 5, R_pl=20.0)
    kTs = [0.5, 0.53, 0.56, 0.6, 0.64]
    p = dict(w.params, kT_per_traj=kTs)
    T = len(kTs)
    s = m.Sop(w.xyz, w.bonds, w.native, p, n_traj=T, **var)
    o = sopo.Oracle(w.xyz, w.bonds, w.native, p, n_traj=T)
    assert np.allclose(s.get_temperatures(), kTs)
    s.run(100); o.run(100)
    xg = s.get_coords()
    assert np.abs(xg - o.get_coords()).max() <= 1e-3
    spread = np.abs(xg - w.xyz[None]).reshape(T, -1).std(axis=1)
    assert spread[-1] > spread[0]                                # hotter runs move more
    swapped_any = False
    for sweep in range(12):
        o.set_coords(xg.astype(np.float64)); o.step = s.step
        E = o.get_energies()[:, 5]
        kT = o.get_temperatures()
        acc_g = s.replica_exchange(sweep & 1, sweep)
        acc_o = o.replica_exchange(sweep & 1, sweep)
        for t in range(sweep & 1, T - 1, 2):
            xw = sopo.philox4x32_10([t, 0x52455821, sweep, 0], [w.params["seed"] & 0xFFFFFFFF, w.params["seed"] >> 32])
            u = ((int(xw[0]) >> 8) + 1) / 2.0 ** 24
            pr = sopo.rex_probability(E[t], E[t + 1], kT[t], kT[t + 1])
            if abs(u - pr) > 1e-4:
                assert acc_g[t // 2] == acc_o[t // 2], (sweep, t, u, pr)
            swapped_any = swapped_any or bool(acc_g[t // 2])
        if not np.array_equal(acc_g, acc_o):
            pytest.skip("a swap decision within rounding of its threshold")
        assert np.allclose(s.get_temperatures(), o.get_temperatures())
        s.run(50); o.run(50)
        xg = s.get_coords()
        assert np.abs(xg - o.get_coords()).max() <= 1e-3
    assert swapped_any and sorted(s.get_temperatures().tolist()) == pytest.approx(sorted(kTs))
    with pytest.raises(m.SopError):
        m.Sop(w.xyz, w.bonds, w.native, w.params, n_traj=2, **var).replica_exchange(0, 0)     # no kT_per_traj


@pytest.mark.parametrize("lanes", [1, 8])
def test_second_order_integrator_matches_the_oracle(lanes):
    """params.integrator = 2: the predictor-corrector whose mean recursion is Eq. (5), two launches per
    step; coordinates within 1e-3 A of the oracle after 100 steps with pulling, a fixed bead and a finite pair list;
    bit-identical however the run is split; refused where it is not implemented."""
    m = sop()
    w = gen.two_chains(120, 5, R_pl=20.0)
    p = dict(w.params, integrator=2, fixed=[0], pulled=[119], pull_k=0.05, pull_v=1e-3, pull_dir=[0.0, 0.6, 0.8])
    T = 2
    s = m.Sop(w.xyz, w.bonds, w.native, p, n_traj=T, lanes_per_bead=lanes)
    assert s.config()["mode"] == 1
    o = sopo.Oracle(w.xyz, w.bonds, w.native, p, n_traj=T)
    s.run(100); o.run(100)
    xg, xo = s.get_coords(), o.get_coords()
    assert np.abs(xg - xo).max() <= 1e-3
    assert np.array_equal(xg[:, 0], np.broadcast_to(w.xyz[0], (T, 3)))
    check_lists(s, o, xg[0])
    b = m.Sop(w.xyz, w.bonds, w.native, p, n_traj=T, lanes_per_bead=lanes); b.run(37); b.run(63)
    assert np.array_equal(b.get_coords(), xg)
    c = m.Sop(w.xyz, w.bonds, w.native, dict(p, integrator=1), n_traj=T, lanes_per_bead=lanes); c.run(100)
    d = np.abs(c.get_coords() - xg).max()
    assert 1e-7 < d < 0.05                                       # another integrator, the same noise: O(h^2) apart
    for bad in (dict(mode=3), dict(mode=2), dict(rng=1)):
        with pytest.raises(m.SopError):
            m.Sop(w.xyz, w.bonds, w.native, dict(p, **{k: v for k, v in bad.items() if k == "rng"}), n_traj=T,
                  **{k: v for k, v in bad.items() if k != "rng"})


# ---------------------------------------------------------------------------------------------- NEXT-3: pair-based scheme
@pytest.mark.parametrize("atomics", [0, 1])
def test_pair_based_scheme_mode4(atomics):
    """Alg. 4 + Alg. 5: one thread per pair, forces saved to unique places and gathered in the update
    kernel (atomics = 0), or added atomically (atomics = 1, the form the paper anticipates).  Forces, lists,
    energies and 100-step coordinates against the oracle with pulling, an indenter, per-contact eps and a batch; the
    unique-place form is bit-identical run to run and however the run is split."""
    m = sop()
    w = gen.two_chains(150, 3, R_pl=20.0)
    zmax = float(w.xyz[:, 2].max())
    eps = (0.5 + np.random.default_rng(9).random(len(w.native))).astype(np.float32)
    p = dict(w.params, fixed=[0, 5], pulled=[149], pull_k=0.05, pull_v=1e-3, pull_dir=[0.6, 0.0, 0.8],
             tip_on=1, tip_R=50.0, tip_eps=1.0, tip_sigma=3.8, tip_c0=[0.0, 0.0, zmax + 53.0], tip_dir=[0.0, 0.0, -1.0], tip_v=1e-3)
    T = 3
    s = m.Sop(w.xyz, w.bonds, w.native, p, n_traj=T, native_eps=eps, mode=4, pair_atomics=atomics)
    o = sopo.Oracle(w.xyz, w.bonds, w.native, p, n_traj=T, native_eps=eps)
    assert s.config()["mode"] == 4
    f_gpu, f_cpu = s.get_forces(), o.get_forces()
    assert np.abs(f_gpu - f_cpu).max() <= 1e-4 * np.abs(f_cpu).max()
    check_energies(s.get_energies(), o.get_energies())
    s.run(100); o.run(100)
    xg = s.get_coords()
    assert np.abs(xg - o.get_coords()).max() <= 1e-3
    check_lists(s, o, xg[T - 1], traj=T - 1)
    b = m.Sop(w.xyz, w.bonds, w.native, p, n_traj=T, native_eps=eps, mode=4, pair_atomics=atomics); b.run(37); b.run(63)
    if atomics == 0:
        assert np.array_equal(b.get_coords(), xg)                  # unique places: no dependence on the order of the pairs
    else:
        assert np.abs(b.get_coords() - xg).max() < 1e-4            # atomic additions: the order of the sum is not fixed
    # against the particle-based kernels: the same pair terms, summed in another order
    c = m.Sop(w.xyz, w.bonds, w.native, p, n_traj=T, native_eps=eps, mode=1, lanes_per_bead=1); c.run(100)
    assert np.abs(c.get_coords() - xg).max() < 1e-4


def test_pair_based_scheme_full_config0_and_3():
    full_check(0, mode=4)
    full_check(3, mode=4)


# ---------------------------------------------------------------------------------------------- mode 3, streamed lists
def test_mode3_streamed_lists_variant():
    """Chunks whose state does not fit shared memory keep only the coordinates resident (one time layer, updated in place) and
    stream L2 rows, bonds, natives and L1 rows from global memory.  SOP_TEST_STREAM forces that variant on small inputs:
    forces, 230-step coordinates and lists against the oracle, bit-identical to itself however the run is split; the
    250,000-bead lattice takes it when mode 3 is asked for."""
    os.environ["SOP_TEST_STREAM"] = "1"
    try:
        w = gen.two_chains(150, 3, R_pl=20.0)
        for var in (dict(chunk_beads=60, lanes_per_bead=1), dict(chunk_beads=75, lanes_per_bead=2, compensated=1)):
            s = sop().from_workload(w, mode=3, **var)
            o = sopo.from_workload(w)
            f, fo = s.get_forces(), o.get_forces()
            assert np.abs(f - fo).max() <= 1e-4 * np.abs(fo).max()
            s.run(230); o.run(230)
            xg = s.get_coords()
            assert np.abs(xg - o.get_coords()).max() <= 3e-3
            c1, i1, _ = s.get_lists(1); c2, i2, _ = s.get_lists(2)
            oc, oi = o.filter(xg[0].astype(np.float64), c1, i1)
            assert np.array_equal(c2, oc) and all(np.array_equal(i2[i, :c2[i]], oi[i, :oc[i]]) for i in range(w.n_beads))
            b = sop().from_workload(w, mode=3, **var); b.run(100); b.run(130)
            assert np.array_equal(b.get_coords(), xg)
    finally:
        del os.environ["SOP_TEST_STREAM"]
    full_check(4, mode=3)

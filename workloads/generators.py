"""Seeded synthetic workloads: the five configs of BASELINE.json made concrete.

This module serves BOTH the fp64 oracle (oracle/) and the CUDA path (paper_1003_1148_b200/) and therefore
holds none of the method's arithmetic: no force law, no list predicate, no PRNG of the method, no update rule.
It only makes inputs: native C-alpha coordinates (fp32), the bond list, the native-contact list and a plain dict
of parameters.  The structures stand in for the PDB / VIPERdb systems of the paper's Table I,
which are not available and are not reconstructed.

Readings used (repeated in DESIGN.md):
  * bonds: consecutive beads of one chain (Eq. (1) first term);
  * native contacts: same-chain pairs with |i-j| > 2, and every inter-chain pair, whose native distance is
    < 8 A, strict, evaluated in fp64 from the fp32 coordinates ("R_C = 8 A");
  * everything else is the non-native set (the library derives it; it is not materialised here).
"""
from __future__ import annotations

import dataclasses
import functools
import hashlib
import math

import numpy as np

BOND = 3.8          # A, C-alpha virtual bond length used by the random walks
D_MIN = 3.8         # A, self-avoidance distance inside one chain
R_CONTACT = 8.0     # A, native contact cutoff

# constants shared by all five configs (BASELINE.json configs[0])
BASE_PARAMS = dict(
    k_fene=14.0, R0=2.0, eps_native=1.0, eps_rep=1.0, sigma=3.8,
    R_nb=10.0, R_pl=math.inf, nb_interval=10, pl_interval=100,
    dt_over_zeta=2e-3, kT=0.6, seed=0x5EED0000,
)


@dataclasses.dataclass
class Workload:
    name: str
    xyz: np.ndarray            # [N][3] float32 native coordinates
    bonds: np.ndarray          # [n_bonds][2] int32, i<j
    native: np.ndarray         # [n_native][2] int32, i<j
    chain: np.ndarray          # [N] int32 chain id of each bead
    params: dict               # plain python scalars / small lists (see BASE_PARAMS)
    n_traj: int
    n_steps: int               # the step count BASELINE.json quotes for the config

    @property
    def n_beads(self) -> int:
        return int(self.xyz.shape[0])

    def digest(self) -> dict:
        h = lambda a: hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()
        return {"xyz": h(self.xyz), "bonds": h(self.bonds), "native": h(self.native),
                "n_beads": self.n_beads, "n_bonds": int(len(self.bonds)), "n_native": int(len(self.native))}


# --------------------------------------------------------------------------------------------------
# random walks
# --------------------------------------------------------------------------------------------------
def _unit_vectors(rng, K):
    d = rng.normal(size=(K, 3))
    return d / np.linalg.norm(d, axis=1)[:, None]


def _first_ok(cand, in_region, earlier, chunk=8):
    """Index of the first candidate that is in the region and >= D_MIN from every bead of `earlier`, else -1.
    Candidates are examined in chunks only to save time; the answer does not depend on the chunk size."""
    for c0 in range(0, len(cand), chunk):
        ok = in_region[c0: c0 + chunk].copy()
        if ok.any() and len(earlier):
            dd = np.linalg.norm(cand[c0: c0 + chunk, None, :] - earlier[None, :, :], axis=2)
            ok &= (dd >= D_MIN).all(axis=1)
        idx = np.flatnonzero(ok)
        if len(idx):
            return c0 + int(idx[0])
    return -1


def compact_saw(N, inside, seed, *, start=(0.0, 0.0, 0.0), K=64, back=8, max_iter=2_000_000):
    """Self-avoiding walk of N beads with 3.8 A bonds confined to the region `inside(points)->mask`.

    To add a bead draw K isotropic unit vectors, accept the first candidate that lies in the region and is
    >= D_MIN from every earlier bead except its predecessor; if none, delete the last `back` beads.
    """
    rng = np.random.default_rng(seed)
    pts = np.zeros((N, 3))
    pts[0] = start
    n, it = 1, 0
    while n < N:
        it += 1
        if it > max_iter:
            raise RuntimeError("compact_saw did not finish")
        cand = pts[n - 1] + BOND * _unit_vectors(rng, K)
        pick = _first_ok(cand, inside(cand), pts[: n - 1])
        if pick >= 0:
            pts[n] = cand[pick]
            n += 1
        else:
            n = max(1, n - back)
    return pts


def directed_saw(N, seed, *, r_cyl=4.0, theta_max_deg=70.0, window=400, K=64, back=8, max_iter=2_000_000):
    """Walk advancing along +z: bond directions uniform on the cap theta <= theta_max about +z, confined to a
    cylinder of radius r_cyl about the z axis through the start; clash check against the previous `window` beads."""
    rng = np.random.default_rng(seed)
    cos_max = math.cos(math.radians(theta_max_deg))
    pts = np.zeros((N, 3))
    n, it = 1, 0
    while n < N:
        it += 1
        if it > max_iter:
            raise RuntimeError("directed_saw did not finish")
        d = _unit_vectors(rng, K)
        cz = 1.0 - (1.0 - cos_max) * (d[:, 2] * 0.5 + 0.5)        # uniform in [cos_max, 1]
        s = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
        ph = np.arctan2(d[:, 1], d[:, 0])
        d = np.stack([s * np.cos(ph), s * np.sin(ph), cz], axis=1)
        cand = pts[n - 1] + BOND * d
        ok = (cand[:, 0] ** 2 + cand[:, 1] ** 2) <= r_cyl * r_cyl
        lo = max(0, n - 1 - window)
        pick = _first_ok(cand, ok, pts[lo: n - 1])
        if pick >= 0:
            pts[n] = cand[pick]
            n += 1
        else:
            n = max(1, n - back)
    return pts


# --------------------------------------------------------------------------------------------------
# topology from coordinates
# --------------------------------------------------------------------------------------------------
def topology_from_coords(xyz32, chain):
    """bonds = consecutive beads of a chain; natives = pairs < 8 A that are not (same chain and |i-j| <= 2)."""
    from scipy.spatial import cKDTree

    N = len(xyz32)
    chain = np.asarray(chain, dtype=np.int32)
    i = np.arange(N - 1, dtype=np.int32)
    same = chain[:-1] == chain[1:]
    bonds = np.stack([i[same], i[same] + 1], axis=1).astype(np.int32)

    x = xyz32.astype(np.float64)
    pairs = cKDTree(x).query_pairs(R_CONTACT + 1e-6, output_type="ndarray")
    a = np.minimum(pairs[:, 0], pairs[:, 1])
    b = np.maximum(pairs[:, 0], pairs[:, 1])
    d = x[a] - x[b]
    d2 = d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1] + d[:, 2] * d[:, 2]
    keep = d2 < R_CONTACT * R_CONTACT
    keep &= ~((chain[a] == chain[b]) & ((b - a) <= 2))
    a, b = a[keep], b[keep]
    order = np.lexsort((b, a))
    native = np.stack([a[order], b[order]], axis=1).astype(np.int32)
    return bonds, native


def _params(**over):
    p = dict(BASE_PARAMS)
    p.update(over)
    return p


def _finish(name, xyz, chain, params, n_traj, n_steps):
    xyz32 = np.ascontiguousarray(xyz, dtype=np.float32)
    bonds, native = topology_from_coords(xyz32, chain)
    return Workload(name, xyz32, bonds, native, np.asarray(chain, np.int32), params, n_traj, n_steps)


# --------------------------------------------------------------------------------------------------
# regions
# --------------------------------------------------------------------------------------------------
def sphere(R):
    return lambda p: (p * p).sum(axis=1) <= R * R


def ellipsoid(a, b, c):
    return lambda p: (p[:, 0] / a) ** 2 + (p[:, 1] / b) ** 2 + (p[:, 2] / c) ** 2 <= 1.0


def cube(side):
    h = 0.5 * side
    return lambda p: (np.abs(p) <= h).all(axis=1)


# --------------------------------------------------------------------------------------------------
# the five configs
# --------------------------------------------------------------------------------------------------
def globule(N, seed, *, n_traj=1, n_steps=1000, philox_seed=0x5EED0000, name=None, **over):
    """Compact chain at config 0's density: sphere radius 15 A * (N/128)^(1/3)."""
    R = 15.0 * (N / 128.0) ** (1.0 / 3.0)
    xyz = compact_saw(N, sphere(R), seed)
    return _finish(name or f"globule{N}", xyz, np.zeros(N, np.int32),
                   _params(seed=philox_seed, **over), n_traj, n_steps)


@functools.lru_cache(maxsize=None)
def config0():
    return globule(128, 1000, n_traj=1, n_steps=1000, philox_seed=0x5EED0000, name="cfg0_chain128")


@functools.lru_cache(maxsize=None)
def config1(n_traj=256, R_pl=math.inf):
    return globule(1000, 1001, n_traj=n_traj, n_steps=100_000, philox_seed=0x5EED0001,
                   name="cfg1_batch1000x%d" % n_traj, R_pl=R_pl)


@functools.lru_cache(maxsize=None)
def config2(n_chains=20, chain_len=2000):
    chains = []
    for c in range(n_chains):
        w = directed_saw(chain_len, 1100 + c)
        w[:, 0] += 10.0 * (c % 5)
        w[:, 1] += 10.0 * (c // 5)
        chains.append(w)
    xyz = np.concatenate(chains)
    xyz -= 0.5 * (xyz.min(axis=0) + xyz.max(axis=0))
    chain = np.repeat(np.arange(n_chains, dtype=np.int32), chain_len)
    p = _params(seed=0x5EED0002, R_pl=20.0, compensated=1,
                fixed=[0], pulled=[chain_len - 1],
                pull_k=0.05, pull_v=1e-3, pull_dir=[0.0, 0.0, 1.0])
    return _finish("cfg2_fiber%dx%d" % (n_chains, chain_len), xyz, chain, p, 1, 100_000)


def icosahedral_rotations():
    """The 60 proper rotations, generated by the 5-fold about (0,1,phi) and the 3-fold about (1,1,1)."""
    phi = (1.0 + 5.0 ** 0.5) / 2.0

    def rot(axis, ang):
        a = np.asarray(axis, float)
        a /= np.linalg.norm(a)
        Kx = np.array([[0, -a[2], a[1]], [a[2], 0, -a[0]], [-a[1], a[0], 0]])
        return np.eye(3) + math.sin(ang) * Kx + (1 - math.cos(ang)) * Kx @ Kx

    gens = [rot([0, 1, phi], 2 * math.pi / 5), rot([1, 1, 1], 2 * math.pi / 3)]
    G = [np.eye(3)]
    k = 0
    while k < len(G):
        for B in gens:
            C = G[k] @ B
            if not any(np.allclose(C, X, atol=1e-9) for X in G):
                G.append(C)
        k += 1
    assert len(G) == 60
    return G


@functools.lru_cache(maxsize=None)
def config3(seed=1200):
    phi = (1.0 + 5.0 ** 0.5) / 2.0
    v5 = np.array([0.0, 1.0, phi]); v5 /= np.linalg.norm(v5)
    v3 = np.ones(3) / 3 ** 0.5
    v2 = np.array([0.0, 0.0, 1.0])
    p0 = 0.216 * v5 + 0.625 * v3 + 0.159 * v2
    p0 /= np.linalg.norm(p0)
    xax = np.cross(v2, p0); xax /= np.linalg.norm(xax)
    yax = np.cross(p0, xax)
    F = np.stack([xax, yax, p0], axis=1)               # subunit frame: z -> radial direction p0
    G = icosahedral_rotations()
    while True:
        sub = compact_saw(500, ellipsoid(28.0, 28.0, 16.7), seed)
        base = sub @ F.T + 120.0 * p0
        xyz = np.concatenate([base @ g.T for g in G])
        chain = np.repeat(np.arange(60, dtype=np.int32), 500)
        from scipy.spatial import cKDTree
        x32 = xyz.astype(np.float32).astype(np.float64)
        pr = cKDTree(x32).query_pairs(2.5, output_type="ndarray")
        if not (len(pr) and (chain[pr[:, 0]] != chain[pr[:, 1]]).any()):
            break
        seed += 1                                       # inter-subunit clash < 2.5 A: bump the seed
    z = xyz[:, 2].astype(np.float32)
    zmin, zmax = float(z.min()), float(z.max())
    fixed = np.flatnonzero(z < zmin + 10.0).astype(np.int32).tolist()
    R_tip = 50.0
    p = _params(seed=0x5EED0003, R_pl=20.0, fixed=fixed,
                tip_on=1, tip_R=R_tip, tip_eps=1.0, tip_sigma=3.8,
                tip_c0=[0.0, 0.0, zmax + R_tip + 10.0], tip_dir=[0.0, 0.0, -1.0], tip_v=1e-3)
    return _finish("cfg3_shell60x500", xyz, chain, p, 1, 100_000)


@functools.lru_cache(maxsize=None)
def config4(n_copies=500):
    sub = compact_saw(500, cube(36.0), 1300)
    grid = [(ix, iy, iz) for iz in range(5) for iy in range(10) for ix in range(10)][:n_copies]
    xyz = np.concatenate([sub + 40.0 * np.array(g, float) for g in grid])
    xyz -= 0.5 * (xyz.min(axis=0) + xyz.max(axis=0))
    chain = np.repeat(np.arange(n_copies, dtype=np.int32), 500)
    p = _params(seed=0x5EED0004, R_pl=20.0)
    return _finish("cfg4_lattice%dx500" % n_copies, xyz, chain, p, 1, 10_000)


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}


def make_config(k: int, **kw) -> Workload:
    return CONFIGS[k](**kw)


# --------------------------------------------------------------------------------------------------
# small inputs for tests
# --------------------------------------------------------------------------------------------------
def tiny(N, seed, **over):
    """A small compact chain (N = 8 ... 512) with config 0's constants."""
    return globule(N, 5000 + seed, name=f"tiny{N}_{seed}", philox_seed=0xABC000 + seed, **over)


def two_chains(N_each, seed, gap=4.0, **over):
    """Two small globules side by side: exercises the inter-chain native rule."""
    R = 15.0 * (N_each / 128.0) ** (1.0 / 3.0)
    a = compact_saw(N_each, sphere(R), 7000 + seed)
    b = compact_saw(N_each, sphere(R), 8000 + seed) + np.array([2 * R + gap, 0.0, 0.0])
    xyz = np.concatenate([a, b])
    chain = np.repeat(np.arange(2, dtype=np.int32), N_each)
    return _finish(f"two{N_each}_{seed}", xyz, chain, _params(seed=0xDEF000 + seed, **over), 1, 100)


def free_beads(N, spacing=25.0, **over):
    """N non-interacting beads on a cubic lattice wider than every cutoff (no bonds, no natives):
    free diffusion / spring pins (P5, P7)."""
    m = int(math.ceil(N ** (1.0 / 3.0)))
    g = np.stack(np.meshgrid(np.arange(m), np.arange(m), np.arange(m), indexing="ij"), axis=-1).reshape(-1, 3)[:N]
    xyz = (spacing * (g - 0.5 * (m - 1))).astype(np.float32)
    w = Workload(f"free{N}", xyz, np.zeros((0, 2), np.int32), np.zeros((0, 2), np.int32),
                 np.arange(N, dtype=np.int32), _params(**over), 1, 100)
    return w

"""The seeded synthetic workloads: shapes, the native-contact rule, reproducibility (MANIFEST hashes)."""
import json
import os

import numpy as np
import pytest

from workloads import generators as gen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("k,N,T", [(0, 128, 1), (1, 1000, 256), (2, 40000, 1), (3, 30000, 1), (4, 250000, 1)])
def test_config_shapes_and_manifest(k, N, T):
    w = gen.make_config(k)
    assert w.n_beads == N and w.n_traj == T
    assert w.xyz.dtype == np.float32 and w.bonds.dtype == np.int32 and w.native.dtype == np.int32
    man = json.load(open(os.path.join(ROOT, "workloads", "MANIFEST.json")))["configs"][str(k)]
    assert w.digest() == {q: man[q] for q in w.digest()}, "generator output changed (numpy version?)"
    # bonds are 3.8 A, consecutive beads of one chain
    d = np.linalg.norm(w.xyz[w.bonds[:, 0]].astype(float) - w.xyz[w.bonds[:, 1]], axis=1)
    assert np.allclose(d, 3.8, atol=1e-3)
    assert (w.bonds[:, 1] == w.bonds[:, 0] + 1).all()
    assert (w.chain[w.bonds[:, 0]] == w.chain[w.bonds[:, 1]]).all()
    # natives: i<j, < 8 A, not (same chain and |i-j| <= 2), unique, disjoint from bonds
    a, b = w.native[:, 0], w.native[:, 1]
    assert (a < b).all()
    dn = np.linalg.norm(w.xyz[a].astype(float) - w.xyz[b], axis=1)
    assert (dn < 8.0).all()
    assert not ((w.chain[a] == w.chain[b]) & (b - a <= 2)).any()
    key = a.astype(np.int64) * N + b
    assert len(np.unique(key)) == len(key)
    assert 2.0 <= 2 * len(w.native) / N <= 15.0


def test_native_rule_is_complete_on_a_small_case():
    w = gen.two_chains(40, 3)
    x = w.xyz.astype(float)
    want = set()
    for i in range(w.n_beads):
        for j in range(i + 1, w.n_beads):
            if w.chain[i] == w.chain[j] and j - i <= 2:
                continue
            if ((x[i] - x[j]) ** 2).sum() < 64.0:
                want.add((i, j))
    assert set(map(tuple, w.native.tolist())) == want


def test_config_specifics():
    w2 = gen.config2()
    assert w2.params["pulled"] == [1999] and w2.params["fixed"] == [0] and w2.params["compensated"] == 1
    assert np.abs(w2.xyz[:, 2]).max() > 2000
    assert (w2.chain[w2.native[:, 0]] != w2.chain[w2.native[:, 1]]).sum() > 10000
    w3 = gen.config3()
    r = np.linalg.norm(w3.xyz.astype(float), axis=1)
    assert 80 < r.min() and r.max() < 160                       # a shell about the 120 A sphere
    assert w3.params["tip_on"] == 1 and w3.params["tip_c0"][2] == pytest.approx(float(w3.xyz[:, 2].max()) + 60.0)
    assert 100 < len(w3.params["fixed"]) < 2000
    assert len(gen.icosahedral_rotations()) == 60
    w4 = gen.config4()
    assert (w4.chain[w4.native[:, 0]] != w4.chain[w4.native[:, 1]]).sum() > 1000

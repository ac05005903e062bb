"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol include/sop.h declares;
host-side validation and workspace sizing (no kernel is launched); the product never imports the oracle."""
import ctypes as C
import os
import re

import pytest

from workloads import generators as gen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    import paper_1003_1148_b200 as m
    hdr = open(os.path.join(ROOT, "include", "sop.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(sop_[a-z_]+)\s*\(", hdr)))
    assert len(declared) >= 15
    L = C.CDLL(m.library_path())
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/sop.h but not exported"
    assert sorted(m.exported_symbols()) == declared


def _query(w, n_traj=1, **over):
    from paper_1003_1148_b200 import sop
    tp, pp, keep = sop._marshal(w.xyz, w.bonds, w.native, w.params, None, over)
    n = C.c_size_t()
    rc = sop.lib().sop_query_workspace(C.byref(tp), keep["xyz"].ctypes.data, C.byref(pp), n_traj, C.byref(n))
    return rc, n.value, (sop.lib().sop_last_error(None) or b"").decode()


def test_query_workspace_is_host_only_and_validates():
    w = gen.config0()
    rc, n, _ = _query(w)
    assert rc == 0 and 100_000 < n < 50_000_000
    rc2, n2, _ = _query(w, n_traj=4)
    assert rc2 == 0 and n2 > n
    rc3, n3, _ = _query(w, cap_nb=64, cap_pl=128)
    assert rc3 == 0
    for bad in (dict(pl_interval=15), dict(R_nb=0.0), dict(R_pl=5.0), dict(lanes_per_bead=3), dict(block_size=100),
                dict(mode=7), dict(R0=-1.0)):
        rc, _, msg = _query(w, **bad)
        assert rc == -1 and msg, bad
    # a finite pair list costs less than the N x N static one
    big = gen.config1()
    rc_s, n_s, _ = _query(big, n_traj=1)
    rc_f, n_f, _ = _query(big, n_traj=1, R_pl=20.0)
    assert rc_s == 0 and rc_f == 0 and n_f < n_s


def test_slice_planner_host_logic():
    """sop_plan_slices (host arithmetic behind the sliced launches of the many-runs batch): no slicing when every trajectory
    has a CTA slot or the launch is short; otherwise a multiple of nb_interval, at least two filter intervals, shorter than the
    launch, and with fewer waves x (slice + overhead) than the plain launch; config 1's case (256 trajectories, 148 slots,
    1000 steps) is sliced."""
    from paper_1003_1148_b200 import sop
    plan = sop.lib().sop_plan_slices
    assert plan(1000, 10, 148, 148) == 0 and plan(1000, 10, 1, 148) == 0          # a slot for everyone
    assert plan(25, 10, 256, 148) == 0                                              # too short to cut
    for bad in ((0, 10, 256, 148), (1000, 0, 256, 148), (1000, 10, 0, 148), (1000, 10, 256, 0)):
        assert plan(*bad) == 0
    L = plan(1000, 10, 256, 148)
    assert L > 0
    for n, nb, T, slots in ((1000, 10, 256, 148), (200, 10, 256, 148), (100, 10, 160, 148), (230, 10, 160, 148),
                            (5000, 25, 1000, 296), (100000, 10, 300, 148)):
        L = plan(n, nb, T, slots)
        if L == 0:
            continue
        assert L % nb == 0 and 2 * nb <= L < n
        slices = -(-n // L)
        waves, plain_waves = -(-slices * T // slots), -(-T // slots)
        assert waves * (2 * L + 7) * 100 < plain_waves * (2 * n + 7) * 97
    # more slots than a one-CTA-per-SM kernel has: several small CTAs per SM are counted as slots
    assert plan(1000, 10, 256, 296) == 0


def test_struct_layout_matches_header():
    """Field order of the ctypes mirror follows the declaration order of sop_params in include/sop.h."""
    from paper_1003_1148_b200 import sop
    hdr = open(os.path.join(ROOT, "include", "sop.h")).read()
    body = hdr[hdr.index("typedef struct {\n  float k_fene"): hdr.index("} sop_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct {", "").replace("const", "").strip()
        if not decl:
            continue
        parts = decl.split(None, 1)[1]
        for v in parts.split(","):
            names.append(re.sub(r"[\*\s]|\[\d+\]", "", v))
    assert names == [f[0] for f in sop._Params._fields_]


def test_product_and_oracle_do_not_touch_each_other():
    pkg = os.path.join(ROOT, "paper_1003_1148_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|sopo|libsopo", text), f
    for f in os.listdir(os.path.join(ROOT, "include")):
        assert "sopo" not in open(os.path.join(ROOT, "include", f)).read()
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1003_1148_b200/" in text or "paper_1003_1148_b200" not in text   # only prose mentions
            assert not re.search(r"import\s+paper_1003_1148_b200|libsop\.so|include/sop\.h\"", text), f


def test_no_gpu_means_loud_failure():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_1003_1148_b200 as m
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        m.from_workload(gen.config0())

"""CPU-only checks of the product library: it loads, exports every symbol include/bltc.h declares,
validates arguments, and its host plan (tree, batches, MAC lists) is structurally identical to the
independently written oracle's.  No compute entry point is called (no GPU here)."""
import os
import re

import numpy as np
import pytest

from paper_2003_01833_b200 import binding as B
from paper_2003_01833_b200 import inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "bltc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b((?:bltc_|direct_)\w+)\s*\(", hdr))
    assert {"bltc_create", "bltc_convolve", "direct_convolve", "bltc_destroy"} <= declared
    L = B.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(B.EXPORTED)
    assert "sm_100a" in B.bltc_version()


def test_argument_validation_without_gpu():
    c = I.random_cloud(100, seed=0)
    X = c.coords()
    for bad in (dict(N=0), dict(theta=1.0), dict(theta=-0.1), dict(interp_degree=0), dict(interp_degree=21),
                dict(batch_size=0), dict(leaf_size=0)):
        kw = dict(N=c.N, theta=0.7, interp_degree=4, batch_size=50, leaf_size=50)
        kw.update(bad)
        with pytest.raises(B.BltcError) as ei:
            B.bltc_create_host_plan(None, X, None, **kw)
        assert ei.value.code == B.BLTC_EINVAL
    with pytest.raises(ValueError):
        B.bltc_create_host_plan(None, X.astype(np.float32), None, c.N, 0.7, 4, 50, 50)
    p = B.bltc_create_host_plan(None, X, None, c.N, 0.7, 4, 50, 50)
    out = np.empty((1, c.N))
    with pytest.raises(B.BltcError) as ei:                    # host-only plan cannot compute
        B.bltc_convolve(p, [1.0], c.f, 1, out, True, stream=0)
    assert ei.value.code == B.BLTC_ENODEVICE
    with pytest.raises(B.BltcError):                          # k <= 0
        B.direct_convolve(X, c.f, c.N, X, c.w, c.f, c.N, [0.0], 1, out, True, stream=0)
    with pytest.raises(B.BltcError):                          # subtraction needs f at targets
        B.direct_convolve(X, None, c.N, X, c.w, c.f, c.N, [1.0], 1, out, True, stream=0)
    B.bltc_destroy(p)


CASES = [
    ("cfg0", lambda: I.config0()),
    ("cfg0_small_leaves", lambda: I.config0(leaf_size=256, batch_size=256, degree=4)),
    ("clustered", lambda: I.random_cloud(5000, seed=4, clustered=True, leaf_size=100, batch_size=100, degree=4)),
    ("second_tree", lambda: I.random_cloud(3000, seed=10, leaf_size=200, batch_size=30, degree=4)),
    ("ragged", lambda: I.random_cloud(7777, seed=11, leaf_size=333, batch_size=333, degree=3, theta=0.5)),
    ("one_leaf", lambda: I.random_cloud(500, seed=12, leaf_size=2000, batch_size=2000)),
    ("theta0", lambda: I.random_cloud(2000, seed=13, leaf_size=100, batch_size=100, theta=0.0)),
    # large enough for the concurrent sub-tree tasks (>= 1e5 points per task level) and the chunked list build
    ("cfg1_threaded_build", lambda: I.config1()),
    ("random_300k_threaded_build", lambda: I.random_cloud(300000, seed=16, leaf_size=400, batch_size=400, degree=5)),
    ("clustered_250k_second_tree", lambda: I.random_cloud(250000, seed=17, clustered=True, leaf_size=600,
                                                          batch_size=250, degree=6, theta=0.8)),
]


@pytest.mark.parametrize("name,make", CASES, ids=[c[0] for c in CASES])
def test_host_plan_is_structurally_identical_to_oracle_tree(oracle_mod, name, make):
    # R18: the 1e-12 GPU-vs-CPU parity is defined for structurally identical trees -> compare first.
    c = make()
    p = B.bltc_create_host_plan(None, c.coords(), None, c.N, c.theta, c.degree, c.batch_size, c.leaf_size)
    e = B.bltc_export_plan(p)
    st = B.bltc_get_stats(p)
    op = oracle_mod.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, c.leaf_size, c.batch_size)
    oe = op.export()
    for key in e:                                            # integer-exact permutation/ranges/lists, bitwise boxes
        np.testing.assert_array_equal(e[key], oe[key], err_msg=key)
    assert (st["n_clusters"], st["n_leaves"], st["n_batches"]) == (op.n_clusters, op.n_leaves, op.n_batches)
    assert (st["far_evals"], st["near_evals"]) == (op.far_evals, op.near_evals)
    assert st["shared_batches"] == op.shared_batches
    B.bltc_destroy(p)


def test_host_plan_separate_targets(oracle_mod):
    c = I.random_cloud(3000, seed=10, leaf_size=200, batch_size=200, degree=4)
    rng = np.random.default_rng(12)
    T = np.ascontiguousarray(rng.random((3, c.N)))
    p = B.bltc_create_host_plan(T, c.coords(), None, c.N, 0.7, 4, 200, 200)
    e = B.bltc_export_plan(p)
    oe = oracle_mod.OraclePlan((c.x, c.y, c.z), 0.7, 4, 200, 200, targets=(T[0], T[1], T[2])).export()
    for key in e:
        np.testing.assert_array_equal(e[key], oe[key], err_msg=key)
    assert B.bltc_get_stats(p)["shared_batches"] == 0


def test_bench_flops_table_matches_the_built_sass():
    """bench.py's FLOPS_PER_PAIR (the roofline numerator) is the FP64 instruction mix actually in the
    pair kernels' inner loops of the built library, re-counted here from cuobjdump -sass."""
    import shutil
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump not on PATH")
    import bench
    from paper_2003_01833_b200 import sass_count
    rows = [r for r in sass_count.count() if r["SUB"] == 1]
    seen = set()
    for r in rows:                      # every GUARD / ZS variant executes the same FP64 mix per pair
        name = "near" if r["kernel"] == "near_kernel" else ("far9" if r["N1"] == 9 else "far")
        if r["KIND"] == 1:
            name = "c" + name
        key = (name, r["OT"])
        assert bench.FLOPS_PER_PAIR[key] == pytest.approx(r["flops"], abs=1e-9), (key, r)
        assert r["R"] == 2
        seen.add(key)
        if name in bench.FP64_INSTR_PER_PAIR:       # the instruction counts behind bench.py's fp64_pipe_busy
            first, extra = bench.FP64_INSTR_PER_PAIR["far" if name == "far9" and r["OT"] >= 6 else name]
            assert r["fp64"] == pytest.approx(first + extra * (r["OT"] - 1), abs=1e-9), (key, r)
    assert seen == set(bench.FLOPS_PER_PAIR)
    # one pipe: 76 FP64 instructions + 7 three-register accumulates per pair of a 7-orbital near tile
    busy = bench.fp64_pipe_busy("near", [7], 32.0 * 4 * 148 * 1.0e6, 1e3, 1.0)     # 1 s at 1 MHz: 4 x 148 x 1e6 pipe cycles
    assert busy == pytest.approx(2 * 76 + 7)


def test_host_plan_fuzz_against_oracle_tree(oracle_mod):
    # seeded sweep over odd sizes and parameters: tiny N, leaf size 1, exact duplicates, planar and collinear clouds
    rng = np.random.default_rng(20030183 + 77)
    for case in range(40):
        N = int(rng.choice([1, 2, 3, 17, 64, 257, 1000, 2500, 4000]))
        leaf = int(rng.choice([1, 2, 7, 32, 100, 300]))
        batch = leaf if rng.random() < 0.6 else int(rng.choice([1, 5, 50, 200]))
        theta = float(rng.choice([0.0, 0.3, 0.7, 0.95]))
        degree = int(rng.integers(1, 7))
        X = rng.random((3, N))
        shape = rng.integers(0, 4)
        if shape == 1:
            X[2] = 0.25                                        # planar: a degenerate box axis (reading R8)
        elif shape == 2:
            X[1] = X[0]; X[2] = 0.5                            # collinear
        elif shape == 3 and N > 3:
            X[:, N // 2:] = X[:, : N - N // 2]                 # every point duplicated (R3, R5: unsplittable clusters)
        X = np.ascontiguousarray(X)
        p = B.bltc_create_host_plan(None, X, None, N, theta, degree, batch, leaf)
        e = B.bltc_export_plan(p)
        st = B.bltc_get_stats(p)
        op = oracle_mod.OraclePlan((X[0], X[1], X[2]), theta, degree, leaf, batch)
        oe = op.export()
        for key in e:
            np.testing.assert_array_equal(e[key], oe[key], err_msg=f"case {case} {key} N={N} leaf={leaf} batch={batch}")
        assert (st["far_evals"], st["near_evals"]) == (op.far_evals, op.near_evals)
        B.bltc_destroy(p)

"""SURVEY.md 8(f) NEXT-4, child -> parent upward pass on the GPU (BLTC_UPWARD_FROM_CHILDREN; reading R23):
leaves from particles, every internal cluster from its children's proxy charges, level by level.  In exact arithmetic
the charges equal the particle-based ones (tests/test_oracle_pins_upward.py), so the GPU result is held to the SAME
bars against the default oracle -- GPU BLTC vs CPU BLTC <= 1e-12 -- and, charge by charge, against the oracle's own
child -> parent pass."""
import numpy as np
import pytest

from paper_2003_01833_b200 import binding as B
from paper_2003_01833_b200 import inputs as I

pytestmark = pytest.mark.gpu
OPT = B.BUILDER_DEVICE | B.UPWARD_FROM_CHILDREN


def rel2(a, b):
    a = np.atleast_2d(a); b = np.atleast_2d(b)
    return max(float(np.linalg.norm(a[o] - b[o]) / np.linalg.norm(b[o])) for o in range(a.shape[0]))


def _dev(*arrs):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]


@pytest.mark.parametrize("N,leaf,degree,theta,clustered,n_orb", [
    (6000, 40, 4, 0.7, True, 2), (9001, 60, 6, 0.8, False, 3), (4133, 30, 3, 0.5, True, 1),
    (12000, 150, 8, 0.7, True, 4), (3000, 25, 1, 0.9, False, 2), (20000, 300, 10, 0.7, True, 1)])
def test_children_based_upward_pass_matches_both_oracle_passes(oracle_mod, N, leaf, degree, theta, clustered, n_orb):
    import torch
    c = I.random_cloud(N, n_orb=n_orb, seed=41 + N % 7, clustered=clustered, leaf_size=leaf, batch_size=leaf, degree=degree, theta=theta)
    X, w, f = _dev(c.coords(), c.w, c.f)
    plan = B.bltc_create_with_builder(None, X, w, c.N, theta, degree, leaf, leaf, 0, 1, OPT)
    ref_plan = B.bltc_create_with_builder(None, X, w, c.N, theta, degree, leaf, leaf, 0, 1, B.UPWARD_FROM_PARTICLES)
    dflt = B.bltc_create(None, X, w, c.N, theta, degree, leaf, leaf)
    assert B.bltc_get_stats(dflt)["upward_from_children"] == 1              # what bltc_create uses
    B.bltc_destroy(dflt)
    st, st0 = B.bltc_get_stats(plan), B.bltc_get_stats(ref_plan)
    assert st["upward_from_children"] == 1 and st0["upward_from_children"] == 0
    assert st["n_proxy_clusters"] >= st0["n_proxy_clusters"] and st["upward_pairs"] <= st0["upward_pairs"]
    out = torch.empty((n_orb, c.N), dtype=torch.float64, device="cuda")
    out0 = torch.empty_like(out)
    B.bltc_convolve(plan, c.k, f, n_orb, out, True)
    B.bltc_convolve(ref_plan, c.k, f, n_orb, out0, True)
    torch.cuda.synchronize()
    P = (c.x, c.y, c.z)
    op0 = oracle_mod.OraclePlan(P, theta, degree, leaf, leaf)
    op1 = oracle_mod.OraclePlan(P, theta, degree, leaf, leaf, upward_from_children=True)
    assert op0.n_far > 0
    ref0 = op0.evaluate(c.w, c.f, c.k)
    ref1 = op1.evaluate(c.w, c.f, c.k)
    got = out.cpu().numpy()
    e0, e1, eg = rel2(got, ref0), rel2(got, ref1), rel2(got, out0.cpu().numpy())
    print(f"N={N} leaf={leaf} n={degree}: GPU(children) vs CPU(particles) {e0:.2e}, vs CPU(children) {e1:.2e}, vs GPU(particles) {eg:.2e}")
    assert e0 <= 1e-12 and e1 <= 1e-12 and eg <= 1e-12
    # charge by charge: the last orbital group's proxy charges and the proxy weights of w, every slot
    px = B.bltc_export_proxy(plan)
    ot = px["fhat"].shape[2]
    o0 = n_orb - ot
    worst = 0.0
    for s in range(0, len(px["cluster"]), max(1, len(px["cluster"]) // 40)):
        cl = int(px["cluster"][s])
        wh, nodes = op1.proxy(cl, c.w)
        np.testing.assert_array_equal(px["nodes"][s], nodes)
        scale = np.abs(wh).sum()
        worst = max(worst, np.abs(px["what"][s] - wh).max() / scale)
        for o in range(ot):
            fh, _ = op1.proxy(cl, c.f[o0 + o] * c.w)
            worst = max(worst, np.abs(px["fhat"][s][:, o] - fh).max() / max(np.abs(c.f[o0 + o] * c.w).sum(), 1e-300))
    assert worst <= 1e-13, worst
    B.bltc_destroy(plan); B.bltc_destroy(ref_plan)


def test_children_based_upward_pass_coulomb_sharded_and_host_builder(oracle_mod):
    import torch
    c = I.random_cloud(15000, n_orb=2, seed=44, clustered=True, leaf_size=80, batch_size=80, degree=5)
    X, w, f = _dev(c.coords(), c.w, c.f)
    op = oracle_mod.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, 80, 80)
    ref = op.evaluate_coulomb(c.w, c.f, alpha=0.3)
    out = torch.full((2, c.N), float("nan"), dtype=torch.float64, device="cuda")
    for r in range(3):                                       # three shards, device builder
        plan = B.bltc_create_with_builder(None, X, w, c.N, c.theta, c.degree, 80, 80, r, 3, OPT)
        B.bltc_convolve_coulomb(plan, f, 2, out, True, 0.3)
        torch.cuda.synchronize()
        B.bltc_destroy(plan)
    assert rel2(out.cpu().numpy(), ref) <= 1e-12
    plan = B.bltc_create_with_builder(None, X, w, c.N, c.theta, c.degree, 80, 80, 0, 1, B.BUILDER_HOST | B.UPWARD_FROM_CHILDREN)
    out2 = torch.empty_like(out)
    B.bltc_convolve_coulomb(plan, f, 2, out2, True, 0.3)
    torch.cuda.synchronize()
    assert torch.equal(out, out2)                            # both builders: the same plan, the same bits
    B.bltc_destroy(plan)


def test_parent_with_a_flat_child_falls_back_to_its_particles(oracle_mod):
    import torch
    rng = np.random.default_rng(20030183 + 402)
    A = rng.random((3, 1500)) * 0.45
    Bp = 0.55 + rng.random((3, 700)) * 0.45; Bp[2] = 0.8
    Xh = np.ascontiguousarray(np.concatenate([A, Bp], axis=1))
    # a far-away blob so that the root's children end up in far lists
    C = np.array([[8.0], [8.0], [8.0]]) + rng.random((3, 1200))
    Xh = np.ascontiguousarray(np.concatenate([Xh, C], axis=1))
    N = Xh.shape[1]
    wh = rng.random(N); fh = rng.uniform(-1, 1, (1, N))
    X, w, f = _dev(Xh, wh, fh)
    plan = B.bltc_create_with_builder(None, X, w, N, 0.8, 3, 300, 300, 0, 1, OPT)
    e = B.bltc_export_plan(plan)
    flat = np.any(e["cl_hi"] == e["cl_lo"], axis=1) & (e["cl_end"] - e["cl_begin"] > 1)
    assert flat.any()
    out = torch.empty((1, N), dtype=torch.float64, device="cuda")
    B.bltc_convolve(plan, [1.1], f, 1, out, True)
    torch.cuda.synchronize()
    ref = oracle_mod.OraclePlan((Xh[0], Xh[1], Xh[2]), 0.8, 3, 300, 300).evaluate(wh, fh, [1.1])
    assert B.bltc_get_stats(plan)["n_far"] > 0
    assert rel2(out.cpu().numpy(), ref) <= 1e-12
    B.bltc_destroy(plan)


def test_children_based_upward_pass_on_configs3_is_faster_and_within_parity(oracle_mod):
    """configs[3] (tree depth 11): sampled batches against the default CPU BLTC oracle, and the upward phase's time in
    both modes (CUDA events inside the library)."""
    import torch
    c = I.config3()
    sel = [0, 7, 13, 20]
    c.f = np.ascontiguousarray(c.f[sel]); c.k = c.k[sel]
    X, w, f = _dev(c.coords(), c.w, c.f)
    res = {}
    for name, opt in (("particles", B.UPWARD_FROM_PARTICLES), ("children", OPT)):
        plan = B.bltc_create_with_builder(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size, 0, 1, opt)
        out = torch.empty((4, c.N), dtype=torch.float64, device="cuda")
        B.bltc_set_profiling(plan, True)
        for _ in range(2):
            B.bltc_convolve(plan, c.k, f, 4, out, True)
        ph = B.bltc_get_phase_ms(plan)
        st = B.bltc_get_stats(plan)
        res[name] = (out.cpu().numpy(), ph["upward"], st["upward_pairs"], st["n_proxy_clusters"], st["upload_ms"])
        B.bltc_destroy(plan)
    op = oracle_mod.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, c.leaf_size, c.batch_size)
    batches = [17, 4242]
    ref = op.evaluate(c.w, c.f, c.k, batches=batches)
    m = np.isfinite(ref[0])
    e_c, e_p = rel2(res["children"][0][:, m], ref[:, m]), rel2(res["particles"][0][:, m], ref[:, m])
    e_cp = rel2(res["children"][0], res["particles"][0])
    print(f"cfg3 upward pass, 4 orbitals: particles {res['particles'][1]:.2f} ms ({res['particles'][2]:.3g} pairs, "
          f"{res['particles'][3]} slots) -> children {res['children'][1]:.2f} ms ({res['children'][2]:.3g} pairs, "
          f"{res['children'][3]} slots); GPU vs CPU BLTC {e_p:.2e} / {e_c:.2e}; children vs particles on the GPU {e_cp:.2e}")
    assert e_c <= 1e-12 and e_p <= 1e-12 and e_cp <= 1e-12
    assert res["children"][1] < res["particles"][1]

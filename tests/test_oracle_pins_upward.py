"""Pins of the oracle's child -> parent upward pass (reading R23): proxy charges of an
internal cluster computed from its children's proxy charges instead of from its own particles.  CPU only.

In exact arithmetic the two upward passes give the SAME charges: qhat^P_K = sum_j q_j [sum_k' L^P_K(s^c_k') L^c_k'(y_j)]
and the bracket is the degree-n interpolant, on the child's grid, of L^P_K -- itself a polynomial of degree n -- hence
L^P_K(y_j) exactly.  So the variant is pinned (1) to the particle-based charges to rounding, at every level of a deep
tree, and independently of them (2) to what interpolation fixes: moments up to per-axis degree n are reproduced, a
polynomial test kernel makes the whole far field exact, one level of the recursion equals the textbook formula written
out in numpy, and the treecode converges to the direct sum."""
import numpy as np
import pytest

from paper_2003_01833_b200 import inputs as I


def rel2(a, b):
    a = np.atleast_2d(a); b = np.atleast_2d(b)
    return max(float(np.linalg.norm(a[o] - b[o]) / np.linalg.norm(b[o])) for o in range(a.shape[0]))


def _bary_row(nodes, t):
    """Eq. (38)-(39) at one point, numpy longdouble, with the node-hit rule R7."""
    n = len(nodes) - 1
    hit = np.nonzero(nodes == t)[0]
    if len(hit):
        L = np.zeros(n + 1); L[hit[0]] = 1.0
        return L
    b = np.array([(-1.0) ** k * (0.5 if k in (0, n) else 1.0) for k in range(n + 1)], dtype=np.longdouble)
    v = b / (np.longdouble(t) - nodes.astype(np.longdouble))
    return np.asarray(v / v.sum(), dtype=np.float64)


def test_moments_are_reproduced_at_every_level(oracle_mod):
    c = I.random_cloud(6000, seed=31, clustered=True)
    n = 4
    p = oracle_mod.OraclePlan((c.x, c.y, c.z), 0.7, n, 60, 60, upward_from_children=True)
    e = p.export()
    q = c.f[0] * c.w
    internal = [cl for cl in range(p.n_clusters) if e["cl_nchild"][cl] > 0]
    assert len(internal) > 20
    picks = [0, internal[1], internal[len(internal) // 2], internal[-1]]
    for cl in picks:
        qhat, nodes = p.proxy(cl, q)
        Q = qhat.reshape(n + 1, n + 1, n + 1)
        idx = e["src_perm"][e["cl_begin"][cl]:e["cl_end"][cl]]
        X, Y, Z, qq = c.x[idx], c.y[idx], c.z[idx], q[idx]
        scale = np.abs(qq).sum()
        for a in ((0, 0, 0), (1, 0, 0), (0, 2, 0), (0, 0, n), (n, n, n), (2, 3, 1), (1, n, 0)):
            lhs = np.einsum("i,j,k,ijk->", nodes[0] ** a[0], nodes[1] ** a[1], nodes[2] ** a[2], Q)
            rhs = (X ** a[0] * Y ** a[1] * Z ** a[2] * qq).sum()
            assert abs(lhs - rhs) < 1e-11 * scale, (cl, a, lhs, rhs)
        lhs = np.einsum("i,ijk->", nodes[0] ** (n + 1), Q)               # degree n + 1 is not reproduced
        assert abs(lhs - (X ** (n + 1) * qq).sum()) > 1e-10 * scale
    # identical to the particle-based charges up to rounding (L^P_K is a polynomial of degree n: interpolating it on
    # the child's grid is exact), through all levels of the tree ...
    p0 = oracle_mod.OraclePlan((c.x, c.y, c.z), 0.7, n, 60, 60)
    assert e["cl_nchild"][e["cl_parent"][internal[-1]]] > 0 and max(e["cl_end"] - e["cl_begin"]) == c.N
    for cl in picks:
        a, _ = p.proxy(cl, q); b, _ = p0.proxy(cl, q)
        assert np.abs(a - b).max() < 1e-13 * np.abs(q[e["src_perm"][e["cl_begin"][cl]:e["cl_end"][cl]]]).sum(), cl
    a, _ = p.proxy(0, q); b, _ = p0.proxy(0, q)
    assert not np.array_equal(a, b)                      # ... but not the same computation
    # a leaf's are the very same numbers
    leaf = int(np.nonzero(e["cl_nchild"] == 0)[0][3])
    np.testing.assert_array_equal(p.proxy(leaf, q)[0], p0.proxy(leaf, q)[0])


def test_one_level_equals_the_formula_written_out(oracle_mod):
    # a root whose children are all leaves: qhat^P_K = sum_c sum_k' L^P_K(s^c_k') qhat^c_k', textbook barycentric form
    rng = np.random.default_rng(20030183 + 401)
    N, n = 900, 3
    X = rng.random((3, N))
    w = rng.random(N); f = rng.uniform(-1, 1, N)
    p = oracle_mod.OraclePlan((X[0], X[1], X[2]), 0.7, n, 200, 200, upward_from_children=True)
    e = p.export()
    kids = np.nonzero(e["cl_parent"] == 0)[0]
    assert len(kids) == 8 and np.all(e["cl_nchild"][kids] == 0)
    q = f * w
    got, nodesP = p.proxy(0, q)
    want = np.zeros((n + 1,) * 3, dtype=np.longdouble)
    for ch in kids:
        qc, nodesC = p.proxy(int(ch), q)
        # the child's own charges, from its particles, independently: Eq. (35) right
        idx = e["src_perm"][e["cl_begin"][ch]:e["cl_end"][ch]]
        mine = np.zeros((n + 1,) * 3, dtype=np.longdouble)
        for j in idx:
            Lx, Ly, Lz = (_bary_row(nodesC[d], X[d][j]) for d in range(3))
            mine += np.einsum("i,j,k->ijk", Lx, Ly, Lz).astype(np.longdouble) * q[j]
        np.testing.assert_allclose(qc.reshape(mine.shape), mine.astype(np.float64), rtol=0, atol=1e-14 * np.abs(q[idx]).sum())
        A = [np.array([_bary_row(nodesP[d], s) for s in nodesC[d]]) for d in range(3)]      # A[d][k', K]
        want += np.einsum("abc,ai,bj,ck->ijk", mine, *[a.astype(np.longdouble) for a in A])
    np.testing.assert_allclose(got.reshape(want.shape), want.astype(np.float64), rtol=0, atol=2e-14 * np.abs(q).sum())


def test_far_field_is_still_exact_for_a_polynomial_kernel(oracle_mod):
    # kind = 1: a kernel that is a polynomial of per-axis degree 3 in the source point.  Interpolating an interpolant
    # of degree n >= 3 loses nothing, so the treecode with children-based charges equals the direct sum to rounding
    # on a tree several levels deep -- a wrong child index, a transposed matrix or a skipped child breaks this.
    c = I.random_cloud(5000, seed=33, clustered=True)
    P = (c.x, c.y, c.z)
    f = c.f[0]
    for subtract in (False, True):
        dref = oracle_mod.direct(P, P, c.w, f, 3, f_tgt=f, subtract=subtract, finalize=False, kind=1)
        for n, exact in ((3, True), (5, True), (2, False)):
            p = oracle_mod.OraclePlan(P, 0.8, n, 30, 30, upward_from_children=True)
            e = p.export()
            far_internal = np.unique(e["far_idx"][e["cl_nchild"][e["far_idx"]] > 0])
            assert len(far_internal) > 10 and e["cl_nchild"][e["cl_parent"][far_internal[-1]]] > 0
            o = p.evaluate(c.w, f, 3, subtract=subtract, finalize=False, kind=1)
            err = rel2(o, dref)
            assert (err < 1e-11) if exact else (err > 1e-6), (n, subtract, err)


def test_treecode_with_children_based_charges_converges_to_the_direct_sum(oracle_mod):
    c = I.random_cloud(8000, n_orb=2, seed=35, clustered=True)
    P = (c.x, c.y, c.z)
    dref = oracle_mod.direct(P, P, c.w, c.f, c.k, f_tgt=c.f)
    errs = {}
    for theta, n in ((0.8, 2), (0.8, 4), (0.8, 6), (0.5, 6)):
        pc = oracle_mod.OraclePlan(P, theta, n, 40, 40, upward_from_children=True)
        pp = oracle_mod.OraclePlan(P, theta, n, 40, 40)
        errs[(theta, n)] = (rel2(pc.evaluate(c.w, c.f, c.k), dref), rel2(pp.evaluate(c.w, c.f, c.k), dref))
    for s in (0, 1):
        assert errs[(0.8, 2)][s] > errs[(0.8, 4)][s] > errs[(0.8, 6)][s] > errs[(0.5, 6)][s], errs
    for key, (ec, ep) in errs.items():
        assert abs(ec - ep) < 1e-9 * ep + 1e-14, (key, ec, ep)      # the same approximation, to rounding
    # theta = 0: no approximation at all
    p0 = oracle_mod.OraclePlan(P, 0.0, 4, 40, 40, upward_from_children=True)
    assert rel2(p0.evaluate(c.w, c.f, c.k), dref) < 1e-14
    # f == const with subtraction: fhat = c what at every level, so out == -2 c / k^2 (Eq. (20)-(21))
    pc = oracle_mod.OraclePlan(P, 0.7, 4, 40, 40, upward_from_children=True)
    out = pc.evaluate(c.w, np.full(c.N, 0.7), 1.3)
    assert np.abs(out + 2 * 0.7 / 1.3 ** 2).max() < 1e-12


def test_parent_with_a_degenerate_child_takes_its_own_particles(oracle_mod):
    # reading R23 / R8: a child flat on an axis has no grid.  Here one octant of the root holds only points of a plane.
    rng = np.random.default_rng(20030183 + 402)
    A = rng.random((3, 1500)) * 0.45                                   # lower octant: a 3-D blob
    B = 0.55 + rng.random((3, 700)) * 0.45; B[2] = 0.8                 # upper octant: points on the plane z = 0.8
    X = np.ascontiguousarray(np.concatenate([A, B], axis=1))
    N = X.shape[1]
    w = rng.random(N); f = rng.uniform(-1, 1, N)
    n = 3
    p = oracle_mod.OraclePlan((X[0], X[1], X[2]), 0.7, n, 300, 300, upward_from_children=True)
    e = p.export()
    kids = np.nonzero(e["cl_parent"] == 0)[0]
    flat = [k for k in kids if np.any(e["cl_hi"][k] == e["cl_lo"][k])]
    assert flat, "the construction must produce a flat child"
    p0 = oracle_mod.OraclePlan((X[0], X[1], X[2]), 0.7, n, 300, 300)
    q = f * w
    np.testing.assert_array_equal(p.proxy(0, q)[0], p0.proxy(0, q)[0])  # root: from particles, as in the default mode
    assert np.all(np.isfinite(p.evaluate(w, f, 1.0)))

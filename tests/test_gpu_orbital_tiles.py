"""Orbital register tiles: the pair kernels evaluate the geometry of a (target, source) pair once for a
tile of 1..7 orbitals; the library cuts n_orb into tiles (bltc_orbital_tiles).  Every tile width is held to the oracle
here (far + near + direct, Yukawa and Coulomb), and the result must not depend on how the orbitals are cut.

    GPU direct vs CPU direct                  <= 1e-13
    GPU BLTC   vs CPU BLTC (identical tree)   <= 1e-12
"""
import os

import numpy as np
import pytest

from paper_2003_01833_b200 import inputs as I

TOL_DIRECT = 1e-13
TOL_BLTC = 1e-12


def rel2(a, b):
    return max(float(np.linalg.norm(a[o] - b[o]) / np.linalg.norm(b[o])) for o in range(a.shape[0]))


def test_orbital_tiles_partition_every_orbital_count():
    """Host logic (no GPU): widths in 1..7, sum = n_orb, as equal as possible, and the forced maximum width is honoured."""
    from paper_2003_01833_b200 import binding as B
    os.environ.pop("BLTC_ORBITAL_TILE", None)
    for n in range(1, 64):
        w = B.bltc_orbital_tiles(n)
        assert sum(w) == n and all(1 <= x <= 7 for x in w) and max(w) - min(w) <= 1, (n, w)
    assert B.bltc_orbital_tiles(7) == [7] and B.bltc_orbital_tiles(21) == [7, 7, 7]
    try:
        for cap in range(1, 8):
            os.environ["BLTC_ORBITAL_TILE"] = str(cap)
            for n in (1, 5, 21, 22):
                w = B.bltc_orbital_tiles(n)
                assert sum(w) == n and max(w) <= cap and len(w) == -(-n // cap), (cap, n, w)
    finally:
        os.environ.pop("BLTC_ORBITAL_TILE", None)
    with pytest.raises(B.BltcError):
        B.bltc_orbital_tiles(0)


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2003_01833_b200 import binding as B
    B.lib()
    return torch, B


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_gpu(gpu, c, coulomb=False, alpha=0.3, sample=None):
    """(BLTC result, direct result on `sample` targets) of the CUDA path."""
    torch, B = gpu
    X, w, f = dev(torch, c.coords()), dev(torch, c.w), dev(torch, c.f)
    plan = B.bltc_create(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size)
    out = torch.empty((c.n_orb, c.N), dtype=torch.float64, device="cuda")
    T = dev(torch, c.coords()[:, sample]); fT = dev(torch, c.f[:, sample])
    dout = torch.empty((c.n_orb, len(sample)), dtype=torch.float64, device="cuda")
    if coulomb:
        B.bltc_convolve_coulomb(plan, f, c.n_orb, out, True, alpha)
        B.direct_convolve_coulomb(T, fT, len(sample), X, w, f, c.N, c.n_orb, dout, True, alpha)
    else:
        B.bltc_convolve(plan, c.k, f, c.n_orb, out, True)
        B.direct_convolve(T, fT, len(sample), X, w, f, c.N, c.k, c.n_orb, dout, True)
    torch.cuda.synchronize()
    B.bltc_destroy(plan)
    return out.cpu().numpy(), dout.cpu().numpy()


@pytest.mark.gpu
@pytest.mark.parametrize("n_orb", [3, 5, 6, 7, 8, 13])
def test_every_tile_width_against_the_oracle(gpu, n_orb):
    """n_orb = 5, 6, 7: one tile of that width; 8 = 4 + 4; 13 = 7 + 6; 3: the narrow tiles.  Clustered cloud with a
    ragged tail (4133 points), small leaves so that far and near lists are both long; degree 8 = the compiled 9^3 grid."""
    import oracle
    torch, B = gpu
    c = I.random_cloud(4133, n_orb=n_orb, seed=40 + n_orb, clustered=True, leaf_size=150, batch_size=150, degree=8)
    assert max(B.bltc_orbital_tiles(n_orb)) == min(n_orb, 7) or n_orb == 8
    P = (c.x, c.y, c.z)
    sample = np.sort(np.random.default_rng(n_orb).choice(c.N, size=700, replace=False))
    Ps = tuple(a[sample] for a in P)
    op = oracle.OraclePlan(P, c.theta, c.degree, c.leaf_size, c.batch_size)
    out, dout = run_gpu(gpu, c, sample=sample)
    assert rel2(out, op.evaluate(c.w, c.f, c.k)) <= TOL_BLTC
    assert rel2(dout, oracle.direct(Ps, P, c.w, c.f, c.k, f_tgt=c.f[:, sample])) <= TOL_DIRECT
    cout, cdout = run_gpu(gpu, c, coulomb=True, sample=sample)
    assert rel2(cout, op.evaluate_coulomb(c.w, c.f, alpha=0.3)) <= TOL_BLTC
    assert rel2(cdout, oracle.coulomb_direct(Ps, P, c.w, c.f, f_tgt=c.f[:, sample], alpha=0.3)) <= TOL_DIRECT


@pytest.mark.gpu
@pytest.mark.parametrize("degree", [8, 5])
def test_result_does_not_depend_on_the_tile_width(gpu, degree):
    """The per-orbital arithmetic is the same at every tile width: forcing tiles of 1..7 orbitals gives bitwise the
    result of the library's own choice (degree 8: the compiled far kernel, incl. its 3-point unroll at 6-7 orbitals;
    degree 5: the generic one)."""
    c = I.random_cloud(3001, n_orb=13, seed=77, clustered=True, leaf_size=120, batch_size=120, degree=degree)
    sample = np.arange(0, c.N, 7)
    os.environ.pop("BLTC_ORBITAL_TILE", None)
    ref, dref = run_gpu(gpu, c, sample=sample)
    cref, cdref = run_gpu(gpu, c, coulomb=True, sample=sample)
    try:
        for cap in range(1, 8):
            os.environ["BLTC_ORBITAL_TILE"] = str(cap)
            out, dout = run_gpu(gpu, c, sample=sample)
            assert np.array_equal(out, ref) and np.array_equal(dout, dref), cap
            cout, cdout = run_gpu(gpu, c, coulomb=True, sample=sample)
            assert np.array_equal(cout, cref) and np.array_equal(cdout, cdref), cap
    finally:
        os.environ.pop("BLTC_ORBITAL_TILE", None)


@pytest.mark.gpu
def test_proxy_charges_of_a_seven_orbital_tile_against_the_oracle(gpu):
    """The upward pass of the widest tile (upward_kernel<7>, upward_children_kernel<7>): proxy charges of all 7 orbitals
    of the exported group against the oracle's Eq. (35), <= 1e-13; bltc_export_proxy's buffer holds the widest tile."""
    import oracle
    torch, B = gpu
    os.environ.pop("BLTC_ORBITAL_TILE", None)
    c = I.random_cloud(5000, n_orb=7, seed=14, clustered=True, leaf_size=100, batch_size=100, degree=4)
    X, w, f = dev(torch, c.coords()), dev(torch, c.w), dev(torch, c.f)
    plan = B.bltc_create(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size)
    out = torch.empty((7, c.N), dtype=torch.float64, device="cuda")
    B.bltc_convolve(plan, c.k, f, 7, out, True)
    torch.cuda.synchronize()
    pr = B.bltc_export_proxy(plan)
    assert pr["fhat"].shape[2] == 7 and B.MAX_ORBITAL_TILE == 7 and len(pr["cluster"]) > 10
    op = oracle.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, c.leaf_size, c.batch_size)
    for s in range(0, len(pr["cluster"]), 5):
        cl = pr["cluster"][s]
        for o in range(7):
            fref, nodes_ref = op.proxy(cl, c.f[o] * c.w)
            np.testing.assert_array_equal(pr["nodes"][s], nodes_ref)
            assert np.abs(pr["fhat"][s][:, o] - fref).max() <= 1e-13 * max(np.abs(fref).max(), 1e-300), (s, o)
    B.bltc_destroy(plan)


@pytest.mark.gpu
@pytest.mark.parametrize("n_orb", [5, 7])
def test_underflow_guard_variants_of_the_wide_tiles(gpu, n_orb):
    """k r up to ~7000 >> 708: the launch takes the GUARD = true instantiations (exp below 2^-1022 is replaced by a
    subnormal-sized value, fp64_math.cuh); most pairs underflow, the nearest neighbours carry the result."""
    import oracle
    c = I.random_cloud(2049, n_orb=n_orb, seed=5 + n_orb, clustered=True, leaf_size=150, batch_size=150, degree=8)
    c.k = c.k * 800.0
    P = (c.x, c.y, c.z)
    sample = np.arange(0, c.N, 3)
    out, dout = run_gpu(gpu, c, sample=sample)
    assert np.all(np.isfinite(out)) and np.all(np.isfinite(dout))
    op = oracle.OraclePlan(P, c.theta, c.degree, c.leaf_size, c.batch_size)
    assert rel2(out, op.evaluate(c.w, c.f, c.k)) <= TOL_BLTC
    Ps = tuple(a[sample] for a in P)
    assert rel2(dout, oracle.direct(Ps, P, c.w, c.f, c.k, f_tgt=c.f[:, sample])) <= TOL_DIRECT

"""GPU parity: Hartree potential (Coulomb kernel, Gaussian singularity subtraction,
PAPER.md:197-229 Eq. (19),(23),(24)) -- bltc_convolve_coulomb / direct_convolve_coulomb through the C ABI
against oracle/coulomb_sum.c and oracle_bltc_eval_coulomb, element by element.

Same bars as the Yukawa path: GPU direct vs CPU direct <= 1e-13, GPU BLTC vs CPU BLTC on the
identical tree <= 1e-12 (relative 2-norm per density, max over densities).
"""
import numpy as np
import pytest

from paper_2003_01833_b200 import inputs as I

pytestmark = pytest.mark.gpu

TOL_DIRECT = 1e-13
TOL_BLTC = 1e-12


def rel2(a, b):
    a = np.atleast_2d(a); b = np.atleast_2d(b)
    return max(float(np.linalg.norm(a[o] - b[o]) / np.linalg.norm(b[o])) for o in range(a.shape[0]))


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2003_01833_b200 import binding as B
    B.lib()
    return torch, B


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_direct(gpu, c, idx=None, subtract=True, alpha=1.0, host=False):
    torch, B = gpu
    X = c.coords()
    T = X if idx is None else np.ascontiguousarray(X[:, idx])
    fT = c.f if idx is None else np.ascontiguousarray(c.f[:, idx])
    M = T.shape[1]
    if host:
        out = np.empty((c.n_orb, M))
        B.direct_convolve_coulomb(T, fT if subtract else None, M, X, c.w, np.ascontiguousarray(c.f), c.N,
                                  c.n_orb, out, subtract, alpha)
        return out
    out = torch.empty((c.n_orb, M), dtype=torch.float64, device="cuda")
    B.direct_convolve_coulomb(dev(torch, T), dev(torch, fT) if subtract else None, M, dev(torch, X),
                              dev(torch, c.w), dev(torch, c.f), c.N, c.n_orb, out, subtract, alpha)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def gpu_bltc(gpu, c, subtract=True, alpha=1.0, host=False):
    torch, B = gpu
    X = c.coords()
    if host:
        plan = B.bltc_create(None, X, c.w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size)
        out = np.empty((c.n_orb, c.N))
        B.bltc_convolve_coulomb(plan, np.ascontiguousarray(c.f), c.n_orb, out, subtract, alpha)
    else:
        plan = B.bltc_create(None, dev(torch, X), dev(torch, c.w), c.N, c.theta, c.degree, c.batch_size,
                             c.leaf_size)
        o = torch.empty((c.n_orb, c.N), dtype=torch.float64, device="cuda")
        B.bltc_convolve_coulomb(plan, dev(torch, c.f), c.n_orb, o, subtract, alpha)
        torch.cuda.synchronize()
        out = o.cpu().numpy()
    B.bltc_destroy(plan)
    return out


def oracle_bltc(oracle_mod, c, subtract=True, alpha=1.0, batches=None):
    pl = oracle_mod.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, c.leaf_size, c.batch_size)
    return pl.evaluate_coulomb(c.w, c.f, subtract=subtract, alpha=alpha, batches=batches), pl


# ------------------------------------------------------------------------------------ direct
@pytest.mark.parametrize("subtract", [True, False])
@pytest.mark.parametrize("N,n_f,alpha", [(1, 1, 1.0), (33, 1, 0.2), (1000, 2, 1.0), (4133, 3, 0.05), (9001, 5, 0.4)])
def test_coulomb_direct_small_all_tiles(gpu, oracle_mod, N, n_f, alpha, subtract):
    c = I.random_cloud(N, n_orb=n_f, seed=40 + N % 7)
    P = (c.x, c.y, c.z)
    ref = oracle_mod.coulomb_direct(P, P, c.w, c.f, f_tgt=c.f, subtract=subtract, alpha=alpha)
    got = gpu_direct(gpu, c, subtract=subtract, alpha=alpha)
    if N == 1:
        np.testing.assert_allclose(got, ref, rtol=1e-15, atol=0)       # only 2 pi alpha^2 f_i survives (or 0)
    else:
        assert rel2(got, ref) <= TOL_DIRECT


def test_coulomb_direct_config0_density_full_and_host(gpu, oracle_mod):
    # the hydrogen 1s density on the config-0 mesh: rho = psi^2
    c = I.density_workload(I.config0())
    P = (c.x, c.y, c.z)
    ref = oracle_mod.coulomb_direct(P, P, c.w, c.f, f_tgt=c.f, subtract=True, alpha=1.0)
    got = gpu_direct(gpu, c)
    assert rel2(got, ref) <= TOL_DIRECT
    np.testing.assert_array_equal(gpu_direct(gpu, c, host=True), got)  # deterministic reduction order


def test_coulomb_direct_sampled_targets_duplicates_and_far_gaussian(gpu, oracle_mod):
    # M != N, coincident target/source pairs (skip iff r == 0), exact duplicates, and distances where
    # e^{-r^2/alpha^2} underflows (r/alpha up to ~1e4): the guarded exp must return 0-sized values, not NaN
    c = I.random_cloud(6000, n_orb=2, seed=51, clustered=True)
    c.x *= 40.0; c.y *= 40.0; c.z *= 40.0
    c.x[10], c.y[10], c.z[10] = c.x[4000], c.y[4000], c.z[4000]
    idx = I.sample_targets(c.N, 777, seed=5)
    idx[0] = 10
    idx = np.unique(idx)
    P = (c.x, c.y, c.z)
    for subtract, alpha in ((True, 1.0), (True, 0.004), (False, 1.0)):
        ref = oracle_mod.coulomb_direct((c.x[idx], c.y[idx], c.z[idx]), P, c.w, c.f, f_tgt=c.f[:, idx],
                                        subtract=subtract, alpha=alpha)
        got = gpu_direct(gpu, c, idx=idx, subtract=subtract, alpha=alpha)
        assert np.all(np.isfinite(got)) and rel2(got, ref) <= TOL_DIRECT, (subtract, alpha)


def test_coulomb_direct_config1_sampled(gpu, oracle_mod):
    c = I.config1()
    idx = I.sample_targets(c.N, 1000, seed=6)
    ref = oracle_mod.coulomb_direct((c.x[idx], c.y[idx], c.z[idx]), (c.x, c.y, c.z), c.w, c.f, f_tgt=c.f[:, idx])
    got = gpu_direct(gpu, c, idx=idx)
    assert rel2(got, ref) <= TOL_DIRECT


# ------------------------------------------------------------------------------------ BLTC
BLTC_CASES = [
    ("cfg0", lambda: I.config0(), 1.0),
    ("cfg0_far_field", lambda: I.config0(leaf_size=256, batch_size=256, degree=4), 1.0),
    ("clustered_3f", lambda: I.random_cloud(5000, n_orb=3, seed=4, clustered=True, leaf_size=100,
                                            batch_size=100, degree=4), 0.1),
    ("ragged_5f", lambda: I.random_cloud(7777, n_orb=5, seed=11, leaf_size=333, batch_size=333, degree=5), 0.25),
    ("degree8_4f", lambda: I.random_cloud(30000, n_orb=4, seed=12, leaf_size=1000, batch_size=1000, degree=8,
                                          theta=0.8), 0.15),
    ("degree10_1f", lambda: I.random_cloud(9001, n_orb=1, seed=13, leaf_size=1500, batch_size=1500, degree=10,
                                           theta=0.9), 0.3),
]


@pytest.mark.parametrize("subtract", [True, False])
@pytest.mark.parametrize("name,make,alpha", BLTC_CASES, ids=[c[0] for c in BLTC_CASES])
def test_coulomb_bltc_matches_cpu_bltc(gpu, oracle_mod, name, make, alpha, subtract):
    c = make()
    ref, pl = oracle_bltc(oracle_mod, c, subtract=subtract, alpha=alpha)
    got = gpu_bltc(gpu, c, subtract=subtract, alpha=alpha)
    assert rel2(got, ref) <= TOL_BLTC, (name, pl.n_far, pl.n_near)
    if name == "ragged_5f":
        np.testing.assert_array_equal(gpu_bltc(gpu, c, subtract=subtract, alpha=alpha, host=True), got)


def test_coulomb_bltc_config1_sampled_batches_and_error_vs_direct(gpu, oracle_mod):
    # full-size workload in bench.py's launch configuration: CPU BLTC on sampled batches, GPU direct on sampled
    # targets for the method error (reported; Table 4 prints 5e-7..4e-5 Ha on E_H ~ 75 Ha)
    c = I.density_workload(I.config1())
    sel = [0, 137, 301, 567]
    ref, pl = oracle_bltc(oracle_mod, c, batches=sel)
    got = gpu_bltc(gpu, c)
    m = ~np.isnan(ref[0])
    assert m.sum() > 1000
    assert rel2(got[:, m], ref[:, m]) <= TOL_BLTC
    idx = I.sample_targets(c.N, 2000, seed=9)
    ds = gpu_direct(gpu, c, idx=idx)
    err = rel2(got[:, idx], ds)
    print(f"coulomb cfg1: BLTC vs direct (theta 0.7, n 8) = {err:.3e}")
    assert err < 1e-5


def test_coulomb_rejects_bad_arguments(gpu):
    torch, B = gpu
    c = I.random_cloud(500, seed=2, leaf_size=100, batch_size=100, degree=3)
    X = dev(torch, c.coords()); w = dev(torch, c.w); f = dev(torch, c.f)
    plan = B.bltc_create(None, X, w, c.N, 0.7, 3, 100, 100)
    out = torch.empty((1, c.N), dtype=torch.float64, device="cuda")
    with pytest.raises(B.BltcError):
        B.bltc_convolve_coulomb(plan, f, 1, out, True, 0.0)
    with pytest.raises(B.BltcError):
        B.bltc_convolve_coulomb(plan, f, 0, out, True, 1.0)
    with pytest.raises(B.BltcError):
        B.direct_convolve_coulomb(X, None, c.N, X, w, f, c.N, 1, out, True, 1.0)
    B.bltc_convolve_coulomb(plan, f, 1, out, False, 0.0)               # alpha ignored without subtraction
    torch.cuda.synchronize()
    B.bltc_destroy(plan)


def test_coulomb_bltc_hydrogen_hartree_potential_and_energy_closed_form(gpu):
    # physical pin of the whole GPU path without the oracle: rho = e^{-2r}/pi on the adaptive mesh, all 387,584 targets:
    # V_H = 1/r - e^{-2r}(1 + 1/r) and E_H = 1/2 int rho V_H = 5/16 Ha (textbook)
    torch, B = gpu
    h = I.hydrogen_adaptive()
    X = dev(torch, h.coords()); w = dev(torch, h.w)
    r = torch.sqrt((X ** 2).sum(0))
    rho = (torch.exp(-2 * r) / np.pi).reshape(1, h.N).contiguous()
    plan = B.bltc_create(None, X, w, h.N, 0.7, 8, 2000, 2000)
    out = torch.empty((1, h.N), dtype=torch.float64, device="cuda")
    B.bltc_convolve_coulomb(plan, rho, 1, out, True, 1.0)
    torch.cuda.synchronize()
    B.bltc_destroy(plan)
    exact = 1 / r - torch.exp(-2 * r) * (1 + 1 / r)
    err_w = float(torch.sqrt((w * (out[0] - exact) ** 2).sum() / (w * exact ** 2).sum()))
    e_h = float(0.5 * (w * rho[0] * out[0]).sum())
    print(f"hydrogen Hartree on GPU: V_H weighted L2 error {err_w:.2e}, E_H = {e_h:.7f} (5/16 = 0.3125)")
    assert err_w < 1e-4                                  # measured: 8.7e-6
    assert abs(e_h - 0.3125) < 2e-5                     # measured: 0.3125039

"""GPU parity: bltc_gi_update (Algorithm 2 lines 4-7, Eq. (27)) through the C ABI against
oracle/green_iteration.py.  Tolerance: the oracle's sums are exactly rounded; the kernels sum N products naively
per thread and then in a fixed tree, so scalars agree to ~sqrt(N) ulp: 1e-12 relative is two orders of margin
(DESIGN.md 7); psi element-wise relative 2-norm <= 1e-13.
"""
import math

import numpy as np
import pytest

from paper_2003_01833_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available()
    from paper_2003_01833_b200 import binding as B
    B.lib()
    return torch, B


def _fields(N, n_prev, seed):
    """Seeded fields with the structure of the real thing: positive weights of very different sizes, an orthonormal
    set phi (w-inner product), a normalised psi_old, and a psi_new with components along every phi_j."""
    rng = np.random.default_rng(20030183 + 3000 + seed)
    w = rng.random(N) ** 3 + 1e-6
    raw = rng.standard_normal((n_prev + 2, N))
    basis = []
    for v in raw:                                     # w-orthonormalise (input preparation, not the method)
        for b in basis:
            v = v - (w * v * b).sum() * b
        basis.append(v / math.sqrt((w * v * v).sum()))
    phi = np.ascontiguousarray(np.stack(basis[:n_prev])) if n_prev else None
    psi_old = basis[n_prev]
    psi_new = 0.9 * psi_old + 0.3 * basis[n_prev + 1] + (rng.standard_normal(n_prev) @ phi if n_prev else 0.0)
    f_old = -psi_old / (0.1 + rng.random(N))
    return w, psi_old, f_old, np.ascontiguousarray(psi_new), phi


def _check(res, psi, ref, n_prev):
    assert res[0] == pytest.approx(ref["eps_new"], rel=1e-12)
    assert res[1] == pytest.approx(ref["delta"], rel=1e-12)
    assert res[2] == pytest.approx(ref["norm"], rel=1e-12)
    assert res[3] == pytest.approx(ref["residual"], rel=1e-11)      # a difference of nearly equal vectors
    if n_prev:
        np.testing.assert_allclose(res[4:], ref["coeff"], rtol=1e-11, atol=1e-13)
    assert np.linalg.norm(psi - ref["psi"]) / np.linalg.norm(ref["psi"]) <= 1e-13


@pytest.mark.parametrize("N,n_prev", [(1, 0), (33, 0), (1000, 3), (4133, 8), (50001, 9), (300007, 20)])
def test_gi_update_matches_oracle(gpu, N, n_prev):
    torch, B = gpu
    from oracle import green_iteration as G
    if N == 1:
        w, po, f, pn, phi = np.array([0.7]), np.array([1.2]), np.array([-0.4]), np.array([0.9]), None
    else:
        w, po, f, pn, phi = _fields(N, n_prev, seed=N % 11)
    ref = G.gi_update(w, po, f, pn, phi, -0.8)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    psi = d(pn)
    res = torch.empty(4 + n_prev, dtype=torch.float64, device="cuda")
    B.bltc_gi_update(d(w), d(po), d(f), psi, d(phi) if n_prev else None, n_prev, N, -0.8, res)
    torch.cuda.synchronize()
    _check(res.cpu().numpy(), psi.cpu().numpy(), ref, n_prev)
    # same call with HOST buffers; bitwise equal to the device path (fixed summation order)
    psi_h = pn.copy()
    res_h = np.empty(4 + n_prev)
    B.bltc_gi_update(w, po, f, psi_h, phi, n_prev, N, -0.8, res_h)
    np.testing.assert_array_equal(res_h, res.cpu().numpy())
    np.testing.assert_array_equal(psi_h, psi.cpu().numpy())


def test_gi_update_after_a_convolution_hydrogen(gpu, oracle_mod):
    # one whole Green-Iteration step on the device: line 3 (direct_convolve) + lines 4-7, config 0
    torch, B = gpu
    from oracle import green_iteration as G
    c = I.config0()
    psi0 = c.meta["psi"] / math.sqrt((c.w * c.meta["psi"] ** 2).sum())
    r = np.sqrt(c.x ** 2 + c.y ** 2 + c.z ** 2)
    f = -psi0 / r
    eps0 = -0.5
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    X, w, fd = d(c.coords()), d(c.w), d(f[None, :])
    out = torch.empty((1, c.N), dtype=torch.float64, device="cuda")
    B.direct_convolve(X, fd, c.N, X, w, fd, c.N, [math.sqrt(-2 * eps0)], 1, out, True)
    res = torch.empty(4, dtype=torch.float64, device="cuda")
    B.bltc_gi_update(w, d(psi0), fd, out, None, 0, c.N, eps0, res)
    torch.cuda.synchronize()
    P = (c.x, c.y, c.z)
    pn = oracle_mod.direct(P, P, c.w, f, math.sqrt(-2 * eps0), f_tgt=f)
    ref = G.gi_update(c.w, psi0, f, pn, None, eps0)
    _check(res.cpu().numpy(), out[0].cpu().numpy(), ref, 0)


def test_gi_update_rejects_bad_arguments(gpu):
    torch, B = gpu
    a = torch.ones(10, dtype=torch.float64, device="cuda")
    res = torch.empty(4, dtype=torch.float64, device="cuda")
    with pytest.raises(B.BltcError):
        B.bltc_gi_update(a, a, a, a.clone(), None, 2, 10, -0.5, torch.empty(6, dtype=torch.float64, device="cuda"))   # n_prev > 0 without phi
    with pytest.raises(ValueError):      # the binding checks buffer sizes before the library sees the pointers
        B.bltc_gi_update(a, a, a, a.clone(), None, 2, 10, -0.5, res)      # result needs 4 + n_prev elements
    with pytest.raises(ValueError):
        B.bltc_gi_update(a, a[:5].clone(), a, a.clone(), None, 0, 10, -0.5, res)
    with pytest.raises(B.BltcError):
        B.bltc_gi_update(a, a, a, a.clone(), None, 0, 0, -0.5, res)
    with pytest.raises(B.BltcError):
        B.bltc_gi_update(a, a, a, a.clone(), None, 0, 10, float("nan"), res)

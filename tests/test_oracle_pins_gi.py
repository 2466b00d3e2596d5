"""Pins for oracle/green_iteration.py (Algorithm 2 lines 4-7, Eq. (27)
PAPER.md:244).  Closed forms only; nothing compares the oracle with itself and nothing uses the CUDA path.
"""
import math

import numpy as np
import pytest

from paper_2003_01833_b200 import inputs as I


@pytest.fixture(scope="module")
def G():
    from oracle import green_iteration
    return green_iteration


def _cube():
    # [-1,1]^3 in 2^3 cells x 4^3 Fejer points: products of total per-axis degree <= 3 are integrated exactly
    return I.mesh_from_cells(I.uniform_cells(1.0, 2), 4)


def test_eq27_closed_form_on_polynomials(G):
    x, y, z, w = _cube()
    a, b, eps0 = 0.7, -0.4, -1.3
    psi_old = np.full_like(x, 1 / math.sqrt(8.0))
    psi_new = a + b * x
    f_old = x.copy()                                   # "V psi_old" stands for any field: Eq. (27) is bilinear
    u = G.gi_update(w, psi_old, f_old, psi_new, None, eps0)
    # <f, psi_old - psi_new> = int x (1/sqrt8 - a - b x) = -b 8/3 ;  <psi_new, psi_new> = 8 a^2 + b^2 8/3
    delta = (-b * 8 / 3) / (8 * a * a + b * b * 8 / 3)
    assert u["delta"] == pytest.approx(delta, rel=1e-14)
    assert u["eps_new"] == pytest.approx(eps0 - delta, rel=1e-14)      # eps_new = eps_old MINUS the quotient
    assert u["norm"] == pytest.approx(math.sqrt(8 * a * a + b * b * 8 / 3), rel=1e-14)
    # fixed point: psi_new == psi_old leaves the eigenvalue alone and the residual at 0
    v = G.gi_update(w, psi_old, f_old, psi_old.copy(), None, eps0)
    assert v["eps_new"] == eps0 and v["residual"] < 1e-15 and v["norm"] == pytest.approx(1.0, rel=1e-14)


def test_deflation_normalisation_residual_closed_form(G):
    x, y, z, w = _cube()
    s = math.sqrt(3.0 / 8.0)
    phi = np.stack([np.full_like(x, 1 / math.sqrt(8.0)), s * x])        # orthonormal on the cube (Legendre P0, P1)
    psi_new = 2.0 * phi[0] - 3.0 * phi[1] + 0.5 * s * y
    psi_old = s * z
    u = G.gi_update(w, psi_old, np.zeros_like(x), psi_new, phi, -0.5)
    np.testing.assert_allclose(u["coeff"], [2.0, -3.0], rtol=1e-14)
    assert u["norm"] == pytest.approx(0.5, rel=1e-13)                   # what is left: 0.5 s y
    np.testing.assert_allclose(u["psi"], s * y, atol=1e-14)
    assert u["residual"] == pytest.approx(math.sqrt(2.0), rel=1e-13)    # || s y - s z ||^2 = 1 + 1
    assert u["eps_new"] == -0.5                                         # f == 0: no update
    for j in range(2):
        assert abs(G.inner(w, u["psi"], phi[j])) < 1e-14
    # the eigenvalue update uses psi_new as computed in line 3, BEFORE deflation and normalisation (Alg. 2 order)
    f = y.copy()
    v = G.gi_update(w, psi_old, f, psi_new, phi, -0.5)
    num = -(0.5 * s) * 8 / 3                                            # <y, s z - psi_new> = -0.5 s int y^2
    den = 4.0 + 9.0 + 0.25                                              # |psi_new|^2 = 2^2 + 3^2 + 0.5^2
    assert v["delta"] == pytest.approx(num / den, rel=1e-13)


def test_eq27_hydrogen_operator_identity(G):
    # Exact eigenpair (eps, psi) = (-1/2, e^{-r}/sqrt(pi)) of -1/2 lap - 1/r.  For a wrong eps0 the exact
    # psi_new = G(eps0) psi is  psi - 2 (eps - eps0) u  with  (-lap + k0^2) u = psi,  k0^2 = -2 eps0:
    #   u = [ e^{-r}/(k0^2 - 1) - 2 (e^{-r} - e^{-k0 r}) / (r (k0^2 - 1)^2) ] / sqrt(pi)      (check by substitution)
    # and, G being symmetric,  <V psi, psi - psi_new> = -(eps - eps0) <psi_new, psi>,  so Eq. (27) gives
    #   eps_new = eps0 + (eps - eps0) <psi_new, psi> / <psi_new, psi_new>,
    # which is second-order accurate in (eps - eps0).  Both sides are quadrature sums of DIFFERENT integrands.
    h = I.hydrogen_adaptive()
    r = np.sqrt(h.x ** 2 + h.y ** 2 + h.z ** 2)
    psi = np.exp(-r) / math.sqrt(math.pi)
    f = -psi / r
    eps = -0.5
    for eps0 in (-0.45, -0.6, -0.8):
        k2 = -2 * eps0
        k0 = math.sqrt(k2)
        u_ = (np.exp(-r) / (k2 - 1) - 2 * (np.exp(-r) - np.exp(-k0 * r)) / (r * (k2 - 1) ** 2)) / math.sqrt(math.pi)
        psi_new = psi - 2 * (eps - eps0) * u_
        out = G.gi_update(h.w, psi, f, psi_new, None, eps0)
        rhs = eps0 + (eps - eps0) * G.inner(h.w, psi_new, psi) / G.inner(h.w, psi_new, psi_new)
        assert abs(out["eps_new"] - rhs) < 2e-4, (eps0, out["eps_new"], rhs)
        assert abs(out["eps_new"] - eps) < 0.35 * abs(eps0 - eps), (eps0, out["eps_new"])   # moves towards -1/2
    # ... and much closer for a small perturbation (second order)
    assert abs(G.gi_update(h.w, psi, f, psi - 2 * (eps + 0.45) * (
        (np.exp(-r) / (0.9 - 1) - 2 * (np.exp(-r) - np.exp(-math.sqrt(0.9) * r)) / (r * (0.9 - 1) ** 2)) / math.sqrt(math.pi)),
        None, -0.45)["eps_new"] - eps) < 5e-3

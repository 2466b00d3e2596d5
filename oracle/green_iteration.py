"""oracle/green_iteration.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain CPU restatement (numpy fp64, exactly rounded sums via math.fsum) of the steps of Green Iteration
that follow the convolution, arXiv 2003.01833 Algorithm 2 lines 4-7:

  line 4  update eigenvalue, gradient-free form of Harrison et al. (Eq. (27)):
              eps_new = eps_old - <V_eff psi_old, psi_old - psi_new> / <psi_new, psi_new>
          with psi_new = G(eps_old) psi_old AS COMPUTED IN LINE 3 (before lines 5-6 touch it)
  line 5  orthogonalise psi_new against the previously converged wavefunctions phi_j, j < i
  line 6  normalise psi_new
  line 7  residual || psi_new - psi_old ||_2

Readings (R22, the paper prints no formulas for lines 5-7):
  - <a, b> is the quadrature sum  sum_i w_i a_i b_i  (Fejer weights of PAPER.md:152-161), and ||.||_2 its norm;
  - line 5 is one classical Gram-Schmidt projection: c_j = <psi_new, phi_j> for all j from the un-projected
    psi_new, then psi <- psi_new - sum_j c_j phi_j, subtracted in the order j = 0, 1, ...  (the phi_j are
    orthonormal, so this equals the modified variant up to rounding);
  - line 6 divides by sqrt(<psi, psi>) of the projected function.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this file; it shares no code
with the CUDA path (paper_2003_01833_b200/csrc/gi_kernels.cu).
"""
from __future__ import annotations

import math

import numpy as np


def inner(w, a, b):
    """<a, b> = sum_i w_i a_i b_i, exactly rounded sum of the fp64 products."""
    return math.fsum(np.asarray(w, dtype=np.float64) * np.asarray(a, dtype=np.float64) * np.asarray(b, dtype=np.float64))


def gi_update(w, psi_old, f_old, psi_new, phi, eps_old):
    """Algorithm 2 lines 4-7 for one wavefunction.

    w [N] quadrature weights; psi_old [N] current (normalised) iterate; f_old [N] = V_eff * psi_old;
    psi_new [N] = G(eps_old) psi_old from line 3; phi [n_prev][N] converged orthonormal wavefunctions
    (or None); eps_old scalar.
    Returns dict(eps_new, delta, coeff [n_prev], norm, psi [N] (orthogonalised, normalised), residual).
    """
    w = np.asarray(w, dtype=np.float64)
    psi_old = np.asarray(psi_old, dtype=np.float64)
    psi_new = np.asarray(psi_new, dtype=np.float64)
    f_old = np.asarray(f_old, dtype=np.float64)
    # line 4, Eq. (27)
    delta = inner(w, f_old, psi_old - psi_new) / inner(w, psi_new, psi_new)
    eps_new = eps_old - delta
    # line 5
    P = np.zeros((0, w.shape[0])) if phi is None else np.atleast_2d(np.asarray(phi, dtype=np.float64))
    coeff = np.array([inner(w, psi_new, P[j]) for j in range(P.shape[0])])
    psi = psi_new.copy()
    for j in range(P.shape[0]):
        psi = psi - coeff[j] * P[j]
    # line 6
    norm = math.sqrt(inner(w, psi, psi))
    psi = psi / norm
    # line 7
    d = psi - psi_old
    residual = math.sqrt(inner(w, d, d))
    return dict(eps_new=eps_new, delta=delta, coeff=coeff, norm=norm, psi=psi, residual=residual)

"""End-to-end physical check of the hot path on the GPU: Green Iteration (Algorithm 2) for the
hydrogen atom, every step through the C ABI -- line 3 by bltc_convolve (treecode, singularity subtraction), lines
4-7 by bltc_gi_update -- must converge to the textbook ground state eps = -1/2, psi = e^{-r}/sqrt(pi).

This is not a parity test (the oracle is not involved): it pins the whole GPU path, signs and prefactors included,
to a closed form.  The loop itself (f = V psi, the stopping test) is caller-side harness, not product code; the
paper's own driver is Python as well.
"""
import math

import numpy as np
import pytest

from paper_2003_01833_b200 import inputs as I

pytestmark = pytest.mark.gpu


def test_hydrogen_ground_state_by_green_iteration_on_the_gpu():
    import torch
    from paper_2003_01833_b200 import binding as B
    assert torch.cuda.is_available()
    h = I.hydrogen_adaptive()                                   # adaptive mesh on [-20,20]^3, N = 387,584
    N = h.N
    X = torch.from_numpy(h.coords()).cuda()
    w = torch.from_numpy(h.w).cuda()
    r = torch.sqrt((X ** 2).sum(0))
    V = -1.0 / r
    exact = torch.exp(-r) / math.sqrt(math.pi)
    plan = B.bltc_create(None, X, w, N, 0.7, 8, 2000, 2000)

    psi = torch.exp(-0.5 * r * r)                               # a poor initial guess: a Gaussian
    psi = psi / torch.sqrt((w * psi * psi).sum())
    eps = -0.3
    res = torch.empty(4, dtype=torch.float64, device="cuda")
    out = torch.empty((1, N), dtype=torch.float64, device="cuda")
    history = []
    for it in range(40):
        f = (V * psi).reshape(1, N).contiguous()
        B.bltc_convolve(plan, [math.sqrt(-2.0 * eps)], f, 1, out, True)          # line 3
        psi_new = out[0]
        B.bltc_gi_update(w, psi, f[0], psi_new, None, 0, N, eps, res)            # lines 4-7 (psi_new in place)
        eps_new, _, _, residual = (float(v) for v in res.cpu())
        history.append((eps_new, residual))
        psi = psi_new.clone()
        eps = min(eps_new, -0.05)                               # keep k real while far from convergence
        if residual < 1e-7:
            break
    B.bltc_destroy(plan)
    eps_final, residual = history[-1]
    err_w = float(torch.sqrt((w * (psi - exact) ** 2).sum() / (w * exact ** 2).sum()))
    print(f"hydrogen GI on GPU: {len(history)} iterations, eps = {eps_final:.6f}, residual {residual:.1e}, "
          f"psi weighted L2 error {err_w:.2e}; eps history {[round(e, 4) for e, _ in history[:8]]}")
    assert residual < 1e-6, history[-3:]
    assert abs(eps_final + 0.5) < 1e-4, eps_final          # measured: -0.499981
    assert err_w < 5e-4, err_w                            # measured: 9.1e-5


def test_hydrogen_first_excited_s_state_with_deflation_on_the_gpu():
    # Alg. 2 line 5 in anger: with the 1s state as the converged wavefunction phi_0, deflated Green Iteration from an
    # s-symmetric guess converges to the 2s state, eps = -1/8, psi = (2 - r) e^{-r/2} / (4 sqrt(2 pi)).
    # The paper's gauge shift V_eff -> V_eff + V_shift, V_shift = -0.5 (Eq. (22)), is applied by the
    # caller: eigenvalues shift to eps - 0.5 (2s: -0.625), wavefunctions are unaffected.  Without it this iteration
    # is unstable at k = 1/2 (measured: eps drifts away after ~6 iterations), which is why the paper has it.
    import torch
    from paper_2003_01833_b200 import binding as B
    h = I.hydrogen_adaptive()
    N = h.N
    X = torch.from_numpy(h.coords()).cuda()
    w = torch.from_numpy(h.w).cuda()
    r = torch.sqrt((X ** 2).sum(0))
    v_shift = -0.5
    V = -1.0 / r + v_shift
    phi = (torch.exp(-r) / math.sqrt(math.pi)).reshape(1, N).contiguous()
    phi = phi / torch.sqrt((w * phi[0] ** 2).sum())
    exact = (2.0 - r) * torch.exp(-0.5 * r) / (4.0 * math.sqrt(2.0 * math.pi))
    plan = B.bltc_create(None, X, w, N, 0.7, 8, 2000, 2000)
    # the gradient-free update Eq. (27) is a correction formula: like TAGI (initial eigenpairs from atomic data,
    # PAPER.md:142-148) the iteration starts from a reasonable guess, here a 2s-like function with wrong parameters
    psi = (2.0 - 1.2 * r) * torch.exp(-0.58 * r)
    psi = psi - (w * psi * phi[0]).sum() * phi[0]
    psi = psi / torch.sqrt((w * psi * psi).sum())
    eps = -0.15 + v_shift
    res = torch.empty(5, dtype=torch.float64, device="cuda")
    out = torch.empty((1, N), dtype=torch.float64, device="cuda")
    history = []
    for it in range(80):                                        # plain fixed-point iteration, no Anderson mixing
        f = (V * psi).reshape(1, N).contiguous()
        B.bltc_convolve(plan, [math.sqrt(-2.0 * eps)], f, 1, out, True)
        psi_new = out[0]
        B.bltc_gi_update(w, psi, f[0], psi_new, phi, 1, N, eps, res)
        eps_new, _, _, residual, c0 = (float(v) for v in res.cpu())
        history.append((eps_new, residual, c0))
        psi = psi_new.clone()
        eps = min(eps_new, v_shift - 0.02)
        if residual < 1e-6:
            break
    B.bltc_destroy(plan)
    eps_final, residual, _ = history[-1]
    if float((w * psi * exact).sum()) < 0:
        psi = -psi
    err_w = float(torch.sqrt((w * (psi - exact) ** 2).sum() / (w * exact ** 2).sum()))
    ortho = abs(float((w * psi * phi[0]).sum()))
    print(f"hydrogen 2s GI on GPU: {len(history)} iterations, eps = {eps_final - v_shift:.6f}, residual {residual:.1e}, "
          f"psi weighted L2 error {err_w:.2e}, <psi, 1s> = {ortho:.1e}")
    assert residual < 1e-4, history[-3:]
    assert abs(eps_final - v_shift + 0.125) < 5e-4, eps_final   # measured: -0.125071
    assert err_w < 1e-2, err_w                                  # measured: ~2e-3 (slow linear convergence, L = 20)
    assert ortho < 1e-12

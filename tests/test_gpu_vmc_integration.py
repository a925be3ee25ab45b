"""End-to-end integration on the GPU: the calls of include/nkb200.h chained into a variational Monte Carlo
optimisation with stochastic reconfiguration (Sec. 4.1, Eq. (30)): sample (nk_metropolis_sample) ->
local energies (nk_local_energy) -> gradient (nk_energy_gradient) -> SR direction (nk_sr_solve) -> plain SGD update.
The test is the physics: on the 10-site Heisenberg ring (Marshall-rotated, so the ground state is positive and a real
RBM can represent it) the variational energy must come down to the exact ground-state energy obtained here by dense
diagonalisation of the Kronecker-product Hamiltonian (E0 = -18.0618 for the Pauli-matrix normalisation, Q5).
Only the update theta <- theta - lr * delta is done outside the library (three torch axpys).
"""
import numpy as np
import pytest
import torch

import dense_ref as dr
from paper_2112_10526_b200 import inputs as inp

pytestmark = pytest.mark.gpu


def test_vmc_with_sr_reaches_the_ground_state_energy(nk):
    L, alpha, n_chains = 10, 2, 2048
    p = inp.make_problem(inp.KIND_HEISENBERG, "chain", L, alpha * L, n_chains, seed=1, scale=0.01)
    H = dr.heisenberg(L, p.bonds, p.colors, p.J)
    e0 = float(np.linalg.eigvalsh(H.toarray())[0])
    assert abs(e0 - (-18.06178542)) < 1e-6
    op = nk.Operator.from_problem(p, nk.NK_FLAG_MARSHALL)      # U H U with U = prod_{i in A} sigma^z_i: same spectrum
    dev = "cuda"
    sigma = torch.from_numpy(p.sigma).to(dev)
    W, a, b = (torch.from_numpy(x).to(dev) for x in (p.W, p.a, p.b))
    lr, shift = 0.02, 0.1            # (0.05, 0.01) overshoots from the near-uniform start and diverges: the optimiser's business
    energies = []
    for it in range(300):
        nk.metropolis_sample(sigma, W, a, b, rule=nk.NK_RULE_EXCHANGE, clusters=p.bonds, n_steps=2 * L, seed=5,
                             step_offset=it * 2 * L)
        eloc, _, stats = nk.local_energy(op, sigma, W, a, b)
        ga, gb, gW = nk.energy_gradient(sigma, W, b, eloc, stats)
        (da, db, dW), iters, res = nk.sr_solve(sigma, W, b, ga, gb, gW, diag_shift=shift, tol=1e-4, max_iter=100)
        W.sub_(lr * dW); a.sub_(lr * da); b.sub_(lr * db)
        energies.append(stats[0].item())
        assert np.isfinite(energies[-1]) and 0 < iters <= 100
    start, end = energies[0], np.mean(energies[-20:])
    print(f"E0 = {e0:.4f}; variational energy {start:.3f} -> {end:.4f} (relative error {abs(end - e0) / abs(e0):.2e})")
    assert start > -13.0                                       # a near-uniform state to begin with (E ~ -12.3)
    assert end >= e0 - 0.15                                    # variational bound, up to the Monte Carlo error
    assert abs(end - e0) / abs(e0) < 5e-3                      # an alpha = 2 RBM gets the ring to a few 1e-4
    op.close()

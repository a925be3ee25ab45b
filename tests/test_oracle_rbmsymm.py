"""Pins of the symmetric-RBM part of the oracle (Eq. (41) L1292 with the embedding of Eq. (56)) — CPU only.

* psi(g s) = psi(s) for every translation g: the defining property, checked on random configurations.
* |G| = 1 reduces to the plain RBM of `rbm_logpsi`; a direct product-of-cosh evaluation with explicit loops.
* Born identity (Eq. (11)) with the dense Kronecker Hamiltonian: sum |psi|^2 E_loc / sum |psi|^2 = <H>.
* Tied-parameter gradient against central finite differences of the exact <H> over the full Born distribution.
"""
import numpy as np
import pytest

import dense_ref as dr
from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp


def _params(F, N, scale, seed, cplx):
    rng = np.random.default_rng(seed)
    def d(*sh):
        x = rng.normal(size=sh) * scale
        return x + 1j * rng.normal(size=sh) * scale if cplx else x
    return d(F, N), d(F)


@pytest.mark.parametrize("lattice,L,cplx", [("chain", 8, False), ("square", 3, True), ("square", 4, False)])
def test_translation_invariance_and_direct_product(lattice, L, cplx):
    perms = inp.translation_perms(lattice, L)
    N = perms.shape[1]
    assert sorted(perms[3].tolist()) == list(range(N)) and np.array_equal(perms[0], np.arange(N))
    W, b = _params(3, N, 0.3, 1, cplx)
    rng = np.random.default_rng(2)
    sigma = (1 - 2 * rng.integers(0, 2, size=(20, N))).astype(np.int8)
    lp = orc.rbmsymm_logpsi(sigma, W, b, perms)
    for g in (1, len(perms) // 2, len(perms) - 1):
        moved = sigma[:, perms[g]]                          # (g^-1 s)_r = s_{g r}: another element of the orbit
        np.testing.assert_allclose(np.exp(orc.rbmsymm_logpsi(moved, W, b, perms)), np.exp(lp), rtol=1e-11)
    # explicit loops over features and group elements, cosh evaluated directly
    s0 = sigma[0].astype(np.float64)
    psi = 1.0
    for i in range(3):
        for g in range(len(perms)):
            psi = psi * np.cosh(sum(W[i, r] * s0[perms[g][r]] for r in range(N)) + b[i])
    np.testing.assert_allclose(np.exp(lp[0]), psi, rtol=1e-11)


def test_trivial_group_is_the_plain_rbm():
    N, F = 7, 5
    W, b = _params(F, N, 0.4, 3, True)
    sigma = (1 - 2 * np.random.default_rng(4).integers(0, 2, size=(9, N))).astype(np.int8)
    ident = np.arange(N)[None, :]
    np.testing.assert_allclose(orc.rbmsymm_logpsi(sigma, W, b, ident), orc.rbm_logpsi(sigma, W, None, b), atol=1e-12)


def _exact_energy(H, states, W, b, perms):
    psi = np.exp(orc.rbmsymm_logpsi(states, W, b, perms))
    return np.real(np.vdot(psi, H @ psi) / np.vdot(psi, psi))


@pytest.mark.parametrize("cplx", [False, True])
def test_born_identity_and_tied_gradient(cplx):
    L = 6
    bonds, colors = inp.chain_bonds(L)
    J = np.array([1.0])
    perms = inp.translation_perms("chain", L)
    H = dr.heisenberg(L, bonds, colors, J)
    states = dr.all_states(L)
    W, b = _params(2, L, 0.3, 7, cplx)
    eloc, lp = orc.rbmsymm_local_energy(orc.KIND_HEISENBERG, states, bonds, colors, J, 0.0, W, b, perms)
    w = np.exp(2 * lp.real)
    w /= w.sum()
    order = np.argsort(dr.state_index(states))
    E = _exact_energy(H, states[order], W, b, perms)
    assert abs(np.sum(w * eloc).real - E) < 1e-10
    # gradient over the exact distribution = derivative of the exact energy (weights in place of the sample mean)
    T = np.tanh(orc.rbmsymm_features(states, W, b, perms))
    s = states.astype(T.dtype)[:, perms]
    gW = orc.force(np.einsum("sig,sgr->sir", T, s), eloc, w)
    gb = orc.force(T.sum(axis=2), eloc, w)
    eps = 1e-5
    for (i, r) in ((0, 0), (1, 3)):
        for part in (1.0,) + ((1j,) if cplx else ()):
            dW = np.zeros_like(W); dW[i, r] = eps * part
            dE = (_exact_energy(H, states[order], W + dW, b, perms) - _exact_energy(H, states[order], W - dW, b, perms)) / (2 * eps)
            want = 2 * np.real(gW[i, r] * np.conj(part))      # f~ = d<H>/d conj(theta): d<H> = 2 Re(f~ conj(d theta))
            assert abs(dE - want) < 1e-6, (i, r, part, dE, want)
    db = np.zeros_like(b); db[1] = eps
    dE = (_exact_energy(H, states[order], W, b + db, perms) - _exact_energy(H, states[order], W, b - db, perms)) / (2 * eps)
    assert abs(dE - 2 * np.real(gb[1])) < 1e-6
    # the sample-mean routine agrees with `force` on the same terms
    rng = np.random.default_rng(5)
    pick = rng.integers(0, len(states), size=50)
    g_b, g_W = orc.rbmsymm_energy_gradient(states[pick], W, b, perms, eloc[pick])
    fW = orc.force(np.einsum("sig,sgr->sir", T[pick], s[pick]), eloc[pick])
    np.testing.assert_allclose(g_W, fW if cplx else 2 * fW.real, atol=1e-12)

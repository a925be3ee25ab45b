"""Pins of the oracle's gradient functions against things other than themselves."""
import numpy as np
import pytest

import dense_ref as dr
from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp

H, I = orc.KIND_HEISENBERG, orc.KIND_ISING


@pytest.mark.parametrize("cplx", [False, True])
def test_log_derivatives_match_finite_differences(cplx):
    # Eq. (13): O_i = d ln psi / d theta_i, checked by central differences of rbm_logpsi in float64
    rng = np.random.default_rng(4)
    N, M = 5, 3
    dt = np.complex128 if cplx else np.float64
    draw = lambda *sh: (rng.normal(size=sh) + (1j * rng.normal(size=sh) if cplx else 0)) * 0.4
    W, a, b = draw(M, N).astype(dt), draw(N).astype(dt), draw(M).astype(dt)
    sigma = inp.draw_samples(rng, 4, N, False)
    O_a, O_b, O_W = orc.rbm_log_derivatives(sigma, W, b)
    h = 1e-6
    for k in range(N):
        d = np.zeros(N, dt); d[k] = h
        fd = (orc.rbm_logpsi(sigma, W, a + d, b) - orc.rbm_logpsi(sigma, W, a - d, b)) / (2 * h)
        np.testing.assert_allclose(O_a[:, k], fd, rtol=1e-7, atol=1e-8)
    for j in range(M):
        d = np.zeros(M, dt); d[j] = h
        fd = (orc.rbm_logpsi(sigma, W, a, b + d) - orc.rbm_logpsi(sigma, W, a, b - d)) / (2 * h)
        np.testing.assert_allclose(O_b[:, j], fd, rtol=1e-7, atol=1e-8)
        for k in range(N):
            D = np.zeros((M, N), dt); D[j, k] = h
            fd = (orc.rbm_logpsi(sigma, W + D, a, b) - orc.rbm_logpsi(sigma, W - D, a, b)) / (2 * h)
            np.testing.assert_allclose(O_W[:, j, k], fd, rtol=1e-7, atol=1e-8)
    if cplx:   # holomorphic: the derivative along the imaginary direction is i times the real one (Eq. (9)-(10) L440-450)
        D = np.zeros((M, N), dt); D[1, 2] = 1j * h
        fd = (orc.rbm_logpsi(sigma, W + D, a, b) - orc.rbm_logpsi(sigma, W - D, a, b)) / (2 * h)
        np.testing.assert_allclose(fd, 1j * O_W[:, 1, 2], rtol=1e-7, atol=1e-8)


def _exact_energy(kind, N, bonds, colors, J, h, W, a, b):
    Hd = dr.heisenberg(N, bonds, colors, J) if kind == H else dr.ising(N, bonds, colors, J, h)
    psi = np.exp(orc.rbm_logpsi(dr.all_states(N), W, a, b))
    return float(np.real(psi.conj() @ (Hd @ psi)) / np.real(psi.conj() @ psi))


@pytest.mark.parametrize("kind,cplx", [(H, False), (I, False), (H, True), (I, True)])
def test_gradient_over_exact_born_distribution_equals_derivative_of_energy(kind, cplx):
    # Eq. (15)/(16) L664-668 and (27)/(28) L918-922: with E[.] taken over the exact p(s) ~ |psi(s)|^2 (all 2^N states)
    # the estimator IS the gradient of <H> = psi^+ H psi / psi^+ psi, which is differentiated numerically here from
    # the dense Kronecker Hamiltonian.
    N, M = 6, 4
    bonds, colors = inp.chain_bonds(N)
    J, h = [1.0], 0.9
    rng = np.random.default_rng(7)
    dt = np.complex128 if cplx else np.float64
    draw = lambda *sh: (rng.normal(size=sh) + (1j * rng.normal(size=sh) if cplx else 0)) * 0.3
    W, a, b = draw(M, N).astype(dt), draw(N).astype(dt), draw(M).astype(dt)
    states = dr.all_states(N)
    eloc, logpsi = orc.local_energy(kind, states, bonds, colors, J, h, W, a, b)
    p = np.abs(np.exp(logpsi)) ** 2
    p /= p.sum()
    g_a, g_b, g_W = orc.energy_gradient(states, W, b, eloc, weights=p)
    E = lambda W_, a_, b_: _exact_energy(kind, N, bonds, colors, J, h, W_, a_, b_)
    eps = 1e-6

    def check(g, make):
        for idx in np.ndindex(g.shape):
            d_re = (E(*make(idx, eps)) - E(*make(idx, -eps))) / (2 * eps)
            if not cplx:
                assert abs(g[idx] - d_re) < 2e-7 * max(1.0, abs(d_re)), (idx, g[idx], d_re)
            else:     # dE/dRe = 2 Re f~, dE/dIm = 2 Im f~ for a real E and a holomorphic psi
                d_im = (E(*make(idx, 1j * eps)) - E(*make(idx, -1j * eps))) / (2 * eps)
                assert abs(2 * g[idx].real - d_re) < 4e-7 * max(1.0, abs(d_re))
                assert abs(2 * g[idx].imag - d_im) < 4e-7 * max(1.0, abs(d_im))

    def bump(x, idx, d):
        y = x.copy(); y[idx] += d
        return y
    check(g_a, lambda idx, d: (W, bump(a, idx, d), b))
    check(g_b, lambda idx, d: (W, a, bump(b, idx, d)))
    check(g_W, lambda idx, d: (bump(W, idx, d), a, b))


@pytest.mark.parametrize("cplx", [False, True])
def test_batched_gradient_equals_definition_and_covariance_properties(cplx):
    p = inp.make_problem(H, "square", 4, 12, 64, seed=17, order=2, J=(1.0, 0.5), complex_params=cplx, scale=0.2)
    eloc, _ = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    g1 = orc.energy_gradient(p.sigma, p.W, p.b, eloc)
    g2 = orc.energy_gradient_batched(p.sigma, p.W, p.b, eloc)
    for x, y in zip(g1, g2):
        np.testing.assert_allclose(y, x, rtol=1e-11, atol=1e-13)
    # a covariance is blind to a constant shift of the local energies, and vanishes for constant local energies
    g3 = orc.energy_gradient_batched(p.sigma, p.W, p.b, eloc + 123.0)
    for x, y in zip(g2, g3):
        np.testing.assert_allclose(y, x, rtol=1e-9, atol=1e-11)
    g4 = orc.energy_gradient_batched(p.sigma, p.W, p.b, np.full_like(eloc, 3.0))
    assert all(np.abs(x).max() < 1e-14 for x in g4)
    # S^z = 0 samples: sum_k g_a[k] = Cov[sum_k s_k, E] = 0
    assert abs(np.sum(g2[0])) < 1e-12

"""Pins of the QGT part of the oracle (CPU only), against things other than itself.

* Fubini-Study (Sec. 3.5): G is the metric of the distance between normalised states, so over the
  EXACT Born distribution of a tiny system   1 - |<psi_t|psi_{t+d}>|^2 / (<psi_t|psi_t><psi_{t+d}|psi_{t+d}>)
  = d^dagger G d + O(|d|^3), with psi evaluated straight from cosh (no log-derivative code).
* G equals numpy's covariance of the columns of the Jacobian; Hermitian, positive semi-definite.
* `qgt_matvec` (Eq. (75)) equals the dense G times v (+ diagonal shift); `sr_solve` leaves no residual.
"""
import numpy as np
import pytest

from oracle import nk_oracle as orc


def _all_states(N):
    k = np.arange(2 ** N)[:, None]
    return (1 - 2 * ((k >> np.arange(N)[None, :]) & 1)).astype(np.int8)


def _params(N, M, scale, seed, cplx):
    rng = np.random.default_rng(seed)
    def d(*sh):
        x = rng.normal(size=sh) * scale
        return x + 1j * rng.normal(size=sh) * scale if cplx else x
    return d(M, N), d(N), d(M)


def _psi(states, W, a, b):
    s = states.astype(W.dtype)
    return np.exp(s @ a) * np.prod(np.cosh(s @ W.T + b[None, :]), axis=1)


@pytest.mark.parametrize("cplx", [False, True])
def test_qgt_is_the_fubini_study_metric(cplx):
    N, M = 5, 4
    W, a, b = _params(N, M, 0.3, 5, cplx)
    states = _all_states(N)
    psi0 = _psi(states, W, a, b)
    weights = np.abs(psi0) ** 2 / np.sum(np.abs(psi0) ** 2)
    # the oracle's ln-derivatives do not involve a; G's a-block is the plain spin covariance
    G = orc.qgt_dense(states, W, b, weights)
    rng = np.random.default_rng(1)
    for trial in range(3):
        dW, da, db = _params(N, M, 1.0, 100 + trial, cplx)
        d = orc.pack_params(da, db, dW)
        quad = np.real(np.conj(d) @ G @ d)
        for eps in (1e-3, 5e-4):
            psi1 = _psi(states, W + eps * dW, a + eps * da, b + eps * db)
            fid = np.abs(np.vdot(psi0, psi1)) ** 2 / (np.vdot(psi0, psi0).real * np.vdot(psi1, psi1).real)
            assert abs((1.0 - fid) / eps ** 2 - quad) < 20 * eps * max(1.0, abs(quad)), (eps, (1 - fid) / eps ** 2, quad)


@pytest.mark.parametrize("cplx", [False, True])
def test_qgt_equals_numpy_covariance_and_is_psd(cplx):
    N, M, B = 6, 5, 300
    W, a, b = _params(N, M, 0.4, 7, cplx)
    rng = np.random.default_rng(2)
    sigma = (1 - 2 * rng.integers(0, 2, size=(B, N))).astype(np.int8)
    G = orc.qgt_dense(sigma, W, b)
    J = orc.rbm_jacobian(sigma, W, b)
    # np.cov(X)[i][j] = E[dX_i conj(dX_j)]; with X = conj(J)^T this is E[conj(dO_i) dO_j] = G_ij (Eq. (23))
    np.testing.assert_allclose(G, np.cov(np.conj(J).T, bias=True), atol=1e-12)
    np.testing.assert_allclose(G, np.conj(G).T, atol=1e-13)
    assert np.linalg.eigvalsh(G).min() > -1e-12
    assert np.iscomplexobj(G) == cplx


@pytest.mark.parametrize("cplx", [False, True])
def test_matvec_and_sr_solve_against_the_dense_matrix(cplx):
    N, M, B = 5, 7, 200
    W, a, b = _params(N, M, 0.4, 9, cplx)
    rng = np.random.default_rng(3)
    sigma = (1 - 2 * rng.integers(0, 2, size=(B, N))).astype(np.int8)
    G = orc.qgt_dense(sigma, W, b)
    vW, va, vb = _params(N, M, 1.0, 11, cplx)
    out = orc.pack_params(*orc.qgt_matvec(sigma, W, b, va, vb, vW, diag_shift=0.01))
    v = orc.pack_params(va, vb, vW)
    np.testing.assert_allclose(out, (G if cplx else G.real) @ v + 0.01 * v, atol=1e-12)
    # transposed-operand guard: v_W enters as sum_jk O_W[j][k] v_W[j][k], not with v_W transposed
    if M != N:
        bad = orc.pack_params(va, vb, vW.T.copy().reshape(M, N))
        assert not np.allclose(out, G @ bad + 0.01 * bad)
    delta = orc.pack_params(*orc.sr_solve(sigma, W, b, va, vb, vW, 0.01))
    np.testing.assert_allclose((G if cplx else G.real) @ delta + 0.01 * delta, v, atol=1e-9)
    # centring: a vector along a direction whose O is constant over the samples is annihilated (eps = 0)
    const_sigma = np.tile(sigma[:1], (8, 1))
    z = orc.pack_params(*orc.qgt_matvec(const_sigma, W, b, va, vb, vW))
    assert np.abs(z).max() < 1e-12


@pytest.mark.parametrize("cplx", [False, True])
def test_batched_matvec_equals_the_dense_matrix_and_the_jacobian_route(cplx):
    """`qgt_matvec_batched` (no [B][P] Jacobian; used at full batch size) is pinned to the DEFINITION, the dense
    covariance matrix of Eq. (23) built by np.cov above, not only to `qgt_matvec`; M != N guards a transposed v_W."""
    N, M, B = 5, 7, 150
    W, a, b = _params(N, M, 0.4, 21, cplx)
    rng = np.random.default_rng(5)
    sigma = (1 - 2 * rng.integers(0, 2, size=(B, N))).astype(np.int8)
    vW, va, vb = _params(N, M, 1.0, 23, cplx)
    J = orc.rbm_jacobian(sigma, W, b)
    G = np.cov(np.conj(J).T, bias=True)
    v = orc.pack_params(va, vb, vW)
    oa, ob, oW, Jv = orc.qgt_matvec_batched(sigma, W, b, va, vb, vW, diag_shift=0.02, return_w=True)
    out = orc.pack_params(oa, ob, oW)
    np.testing.assert_allclose(out, (G if cplx else G.real) @ v + 0.02 * v, atol=1e-12)
    np.testing.assert_allclose(out, orc.pack_params(*orc.qgt_matvec(sigma, W, b, va, vb, vW, diag_shift=0.02)), atol=1e-12)
    np.testing.assert_allclose(Jv, J @ v.astype(J.dtype), atol=1e-12)
    assert np.iscomplexobj(out) == cplx

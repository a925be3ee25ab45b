"""Pins of oracle/nk_oracle.py against things other than itself (CPU only).

Each test names the passage / mathematics that fixes the expected value.
"""
import numpy as np
import pytest
import scipy.sparse.linalg as spla

import os

import dense_ref as dr
from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp

H, I = orc.KIND_HEISENBERG, orc.KIND_ISING
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


# ---------------------------------------------------------------- log cosh (Q11)
def test_log_cosh_real_matches_direct_definition():
    x = np.linspace(-300, 300, 20001)
    np.testing.assert_allclose(orc.log_cosh(x), np.log(np.cosh(x)), rtol=1e-14, atol=1e-15)
    assert orc.log_cosh(np.array([0.0]))[0] == 0.0


def test_log_cosh_large_argument_limit():
    x = np.array([-1e4, 750.0, 1e6])
    np.testing.assert_allclose(orc.log_cosh(x), np.abs(x) - np.log(2.0), rtol=1e-15)


def test_log_cosh_complex_exponentiates_to_cosh():
    rng = np.random.default_rng(1)
    z = rng.normal(size=4000) * 3 + 1j * rng.normal(size=4000) * 3
    np.testing.assert_allclose(np.exp(orc.log_cosh(z)), np.cosh(z), rtol=1e-12)
    # even function, also on the branch flip Re z < 0
    np.testing.assert_allclose(np.exp(orc.log_cosh(-z)), np.cosh(z), rtol=1e-12)


# ---------------------------------------------------------------- Pauli builder, Eq. (2)
def test_eq2_pauli_identity():
    N = 2
    O = (dr.sigmax(0, N) + dr.sigmax(1, N))
    lhs = (O @ O).toarray()
    rhs = 2 * ((dr.sigmax(0, N) @ dr.sigmax(1, N)).toarray() + np.eye(4))
    np.testing.assert_array_equal(lhs, rhs)
    golden = np.loadtxt(os.path.join(GOLD, "eq2_matrix.txt"))
    np.testing.assert_array_equal(lhs.real, golden)


# ---------------------------------------------------------------- spectra (Q5: Pauli normalisation)
def test_heisenberg_ring_spectra():
    b4, c4 = inp.chain_bonds(4)
    w = np.linalg.eigvalsh(dr.heisenberg(4, b4, c4, [1.0]).toarray())
    assert abs(w[0] + 8.0) < 1e-12 and abs(w[-1] - 4.0) < 1e-12      # L=4 ring: singlet -8, ferromagnet +n_b
    b10, c10 = inp.chain_bonds(10)
    e0 = spla.eigsh(dr.heisenberg(10, b10, c10, [1.0]), k=1, which="SA")[0][0]
    assert abs(e0 - (-18.06178542)) < 1e-6                             # = 4 * (-4.515446) Bethe/ED value for N=10


# ---------------------------------------------------------------- connected list == dense rows (Eq. (3))
def _rows_from_connected(kind, N, bonds, colors, J, h, flags=0):
    states = dr.all_states(N)
    dim = 2 ** N
    Hc = np.zeros((dim, dim))
    for idx in range(dim):
        sp_, mels, flips, n_conn = orc.connected(kind, states[idx], bonds, colors, J, h, flags)
        cols = dr.state_index(sp_)
        assert cols[0] == idx
        np.add.at(Hc[idx], cols, mels)
        assert n_conn == 1 + int(np.sum(flips[1:, 0] >= 0))
        pad = flips[1:, 0] < 0
        assert np.all(mels[1:][pad] == 0.0) and np.all(cols[1:][pad] == idx)
        act = cols[1:][~pad]
        assert len(set(act.tolist())) == len(act) and idx not in act     # no duplicate eta (Q9)
    return Hc


@pytest.mark.parametrize("case", ["chain6", "square3_j1j2", "chain5_two_colours"])
def test_connected_heisenberg_equals_dense_rows(case):
    if case == "chain6":
        bonds, colors = inp.chain_bonds(6); N = 6; J = [1.0]
    elif case == "square3_j1j2":
        bonds, colors = inp.square_bonds(3, 2); N = 9; J = [1.0, 0.5]
    else:
        bonds, colors = inp.chain_bonds(5); N = 5; J = [0.7, -1.3]
        colors = np.array([0, 1, 0, 1, 1], dtype=np.int32)
    Hd = dr.heisenberg(N, bonds, colors, J).toarray()
    Hc = _rows_from_connected(H, N, bonds, colors, J, 0.0)
    np.testing.assert_array_equal(Hc, Hd)
    np.testing.assert_array_equal(Hc, Hc.T)                              # Hermiticity of the list


def test_connected_ising_equals_dense_rows():
    bonds, colors = inp.square_bonds(3, 1)
    Hd = dr.ising(9, bonds, colors, [1.0], 3.0).toarray()
    Hc = _rows_from_connected(I, 9, bonds, colors, [1.0], 3.0)
    np.testing.assert_array_equal(Hc, Hd)
    b, c = inp.chain_bonds(7)
    np.testing.assert_array_equal(_rows_from_connected(I, 7, b, c, [-0.5], 0.25),
                                  dr.ising(7, b, c, [-0.5], 0.25).toarray())


def test_marshall_flag_is_the_sublattice_rotation():
    # On a bipartite ring, U H U with U = prod_{i in A} sz_i flips the sign of the exchange term only.
    bonds, colors = inp.chain_bonds(6)
    Hd = dr.heisenberg(6, bonds, colors, [1.0]).toarray()
    U = np.eye(64)
    for i in range(0, 6, 2):
        U = U @ dr.sigmaz(i, 6).toarray().real
    np.testing.assert_array_equal(_rows_from_connected(H, 6, bonds, colors, [1.0], 0.0, orc.FLAG_MARSHALL),
                                  U @ Hd @ U)


# ---------------------------------------------------------------- Born identity Eq. (11) L646 (brute force)
def _born_check(kind, N, bonds, colors, J, h, M, cplx, seed, sector=False):
    W, a, b = inp.draw_params(np.random.default_rng(seed), N, M, 0.3, cplx)
    states = dr.all_states(N)
    Hd = dr.heisenberg(N, bonds, colors, J) if kind == H else dr.ising(N, bonds, colors, J, h)
    if sector:
        keep = states.sum(axis=1) == 0
        states = states[keep]
        Hd = Hd[keep][:, keep]
    eloc, logpsi = orc.local_energy(kind, states, bonds, colors, J, h, W, a, b)
    psi = np.exp(logpsi)
    p = np.abs(psi) ** 2
    lhs = np.sum(p * eloc) / np.sum(p)
    rhs = (psi.conj() @ (Hd @ psi)) / (psi.conj() @ psi)
    assert abs(lhs - rhs) < 1e-11 * max(1.0, abs(rhs))
    # and pointwise: E_loc(s) psi(s) = (H psi)(s)   (Eq. (12), row = s, ratio unconjugated: Q16)
    np.testing.assert_allclose(eloc * psi, Hd @ psi, rtol=1e-10, atol=1e-12)


@pytest.mark.parametrize("cplx", [False, True])
def test_born_identity_heisenberg_chain10(cplx):
    b, c = inp.chain_bonds(10)
    _born_check(H, 10, b, c, [1.0], 0.0, 10, cplx, 11)


def test_born_identity_heisenberg_chain10_sz0_sector():
    b, c = inp.chain_bonds(10)
    _born_check(H, 10, b, c, [1.0], 0.0, 10, False, 12, sector=True)


@pytest.mark.parametrize("cplx", [False, True])
def test_born_identity_j1j2_3x3(cplx):
    b, c = inp.square_bonds(3, 2)
    _born_check(H, 9, b, c, [1.0, 0.5], 0.0, 18, cplx, 13)


@pytest.mark.parametrize("cplx", [False, True])
def test_born_identity_tfim(cplx):
    b, c = inp.square_bonds(3, 1)
    _born_check(I, 9, b, c, [1.0], 3.0, 18, cplx, 14)
    b, c = inp.chain_bonds(6)
    _born_check(I, 6, b, c, [1.0], 3.0, 5, cplx, 15)


# ---------------------------------------------------------------- closed forms (any size)
def test_uniform_psi_closed_form():
    # W = 0, a = 0, any b: psi uniform => Heisenberg E_loc = sum_c J_c n_{b,c} for every s (ferromagnetic
    # multiplet eigenvalue); TFIM E_loc = J sum_b s_i s_j - h N.
    for c_id, expect in ((1, 10.0), (2, 200.0), (4, 300.0)):
        p = inp.make_config(c_id, n_samples=6)
        e, _ = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, np.zeros_like(p.W), None, p.b)
        np.testing.assert_allclose(e, expect, rtol=1e-13)
    p = inp.make_problem(I, "square", 4, 8, 5, seed=3, J=(1.0,), h=3.0)
    e, _ = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, np.zeros_like(p.W), None, p.b)
    s = p.sigma.astype(np.float64)
    diag = (s[:, p.bonds[:, 0]] * s[:, p.bonds[:, 1]]).sum(axis=1)
    np.testing.assert_allclose(e, diag - 3.0 * 16, rtol=1e-13)


@pytest.mark.parametrize("cplx", [False, True])
def test_w_zero_visible_bias_closed_form(cplx):
    # W = 0: E_loc = diag + sum_{antiparallel b} 2 J_b exp(-2 s_i (a_i - a_j));  TFIM: diag - h sum_k exp(-2 s_k a_k)
    p = inp.make_problem(H, "square", 4, 6, 7, seed=5, order=2, J=(1.0, 0.5), complex_params=cplx, scale=0.4)
    a = p.a.astype(np.complex128 if cplx else np.float64)
    e, _ = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, np.zeros_like(p.W), p.a, p.b)
    for n, srow in enumerate(p.sigma.astype(np.float64)):
        ref = 0.0
        for (i, j), c in zip(p.bonds, p.colors):
            ref += p.J[c] * srow[i] * srow[j]
            if srow[i] != srow[j]:
                ref += 2 * p.J[c] * np.exp(-2 * srow[i] * (a[i] - a[j]))
        assert abs(e[n] - ref) < 1e-12 * max(1, abs(ref))
    q = inp.make_problem(I, "chain", 7, 3, 4, seed=6, h=1.5, complex_params=cplx, scale=0.4)
    a = q.a.astype(np.complex128 if cplx else np.float64)
    e, _ = orc.local_energy(q.kind, q.sigma, q.bonds, q.colors, q.J, q.h, np.zeros_like(q.W), q.a, None)
    s = q.sigma.astype(np.float64)
    ref = (s[:, q.bonds[:, 0]] * s[:, q.bonds[:, 1]]).sum(axis=1) - 1.5 * np.exp(-2 * s * a[None, :]).sum(axis=1)
    np.testing.assert_allclose(e, ref, rtol=1e-12)


def test_single_hidden_unit_direct_cosh():
    # M = 1: psi'/psi = exp(da) cosh(theta') / cosh(theta) with cosh evaluated directly (Q1: no factor 2, no constant)
    p = inp.make_problem(I, "chain", 6, 1, 5, seed=8, h=0.7, scale=0.5)
    W, a, b = (x.astype(np.float64) for x in (p.W, p.a, p.b))
    e, lp = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    for n, s in enumerate(p.sigma.astype(np.float64)):
        th = W[0] @ s + b[0]
        assert abs(lp[n] - (a @ s + np.log(np.cosh(th)))) < 1e-14
        ref = sum(p.J[0] * s[i] * s[j] for i, j in p.bonds)
        for k in range(6):
            ref += -0.7 * np.exp(-2 * a[k] * s[k]) * np.cosh(th - 2 * s[k] * W[0, k]) / np.cosh(th)
        assert abs(e[n] - ref) < 1e-12


def test_theta_orientation_and_logpsi_transposed_operand():
    # W is [M][N] with M != N: a transposed operand cannot even broadcast; value checked against an explicit loop
    rng = np.random.default_rng(3)
    W = rng.normal(size=(3, 5)).astype(np.float32); b = rng.normal(size=3).astype(np.float32)
    a = rng.normal(size=5).astype(np.float32)
    s = np.array([[1, -1, -1, 1, 1]], dtype=np.int8)
    ref = sum(float(a[i]) * s[0, i] for i in range(5))
    for j in range(3):
        th = float(b[j]) + sum(float(W[j, k]) * s[0, k] for k in range(5))
        ref += np.log(np.cosh(th))
    assert abs(orc.rbm_logpsi(s, W, a, b)[0] - ref) < 1e-14


# ---------------------------------------------------------------- symmetries of the estimator
def test_lattice_translation_and_hidden_permutation_invariance():
    p = inp.make_problem(H, "square", 4, 12, 6, seed=9, order=2, J=(1.0, 0.5), scale=0.3)
    e0, lp0 = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    L = 4
    perm = np.array([((x + 1) % L) * L + (y + 2) % L for x in range(L) for y in range(L)])  # translation by (1,2)
    # the translation maps the coloured bond set onto itself
    img = {(min(perm[i], perm[j]), max(perm[i], perm[j]), c) for (i, j), c in zip(p.bonds, p.colors)}
    assert img == {(min(i, j), max(i, j), c) for (i, j), c in zip(p.bonds, p.colors)}
    e1, lp1 = orc.local_energy(p.kind, p.sigma[:, perm], p.bonds, p.colors, p.J, p.h, p.W[:, perm], p.a[perm], p.b)
    np.testing.assert_allclose(e1, e0, rtol=1e-12); np.testing.assert_allclose(lp1, lp0, rtol=1e-12)
    hp = np.random.default_rng(0).permutation(12)
    e2, _ = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W[hp], p.a, p.b[hp])
    np.testing.assert_allclose(e2, e0, rtol=1e-12)
    e3, lp3 = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, -p.W, p.a, -p.b)   # cosh even
    np.testing.assert_allclose(e3, e0, rtol=1e-12); np.testing.assert_allclose(lp3, lp0, rtol=1e-12)


def test_global_spin_flip_z2():
    p = inp.make_problem(H, "chain", 8, 8, 6, seed=10, scale=0.3)
    e0, lp0 = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, None, None)
    e1, lp1 = orc.local_energy(p.kind, -p.sigma, p.bonds, p.colors, p.J, p.h, p.W, None, None)
    np.testing.assert_allclose(e1, e0, rtol=1e-12); np.testing.assert_allclose(lp1, lp0, rtol=1e-12)


def test_exact_eigenstate_gives_constant_local_energy():
    # (1,1,...,1) direction: psi uniform over the FULL space is an eigenstate of TFIM's -h sum sx part and of
    # Heisenberg; checked for Heisenberg over all 2^6 states (SU(2) multiplet S = N/2, energy J n_b).
    b, c = inp.chain_bonds(6)
    e, _ = orc.local_energy(H, dr.all_states(6), b, c, [1.0], 0.0, np.zeros((2, 6), np.float32), None, None)
    np.testing.assert_allclose(e, 6.0, rtol=1e-14)


# ---------------------------------------------------------------- statistics, Eq. (17) L675 + Q10
def test_stats_against_numpy():
    rng = np.random.default_rng(5)
    e = rng.normal(size=1000) + 1j * rng.normal(size=1000)
    mr, mi, var, cnt = orc.stats(e)
    assert abs(mr - e.real.mean()) < 1e-14 and abs(mi - e.imag.mean()) < 1e-14 and cnt == 1000
    assert abs(var - (e.real.var() + e.imag.var())) < 1e-12
    mr, mi, var, _ = orc.stats(e.real)
    assert mi == 0.0 and abs(var - np.var(e.real)) < 1e-13


def test_count_amplitudes_expected_density():
    p = inp.make_config(2, n_samples=512)
    n = orc.count_amplitudes(p.kind, p.sigma, p.bonds, p.colors, p.J)
    # uniform S^z=0 samples: expected antiparallel fraction N / (2 (N-1))
    assert abs(n / (512 * 200) - 100 / (2 * 99)) < 0.01
    by_hand = sum(int(s[i] != s[j]) for s in p.sigma for i, j in p.bonds)
    assert n == by_hand


# ---------------------------------------------------------------- stored regression values written by tests/golden/make_golden.py
def test_golden_cfg1_first_samples():
    g = np.loadtxt(os.path.join(GOLD, "cfg1_first8.txt"))
    p = inp.make_config(1, n_samples=8)
    e, lp = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    np.testing.assert_allclose(e, g[:, 0], rtol=1e-12)
    np.testing.assert_allclose(lp, g[:, 1], rtol=1e-12)

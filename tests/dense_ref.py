"""Independent pins for the oracle: Hamiltonians as explicit Kronecker products of Pauli matrices.

Nothing here uses `oracle.connected` or any bond-flip logic: an operator on site i is
I x ... x P x ... x I, and H is the operator sum of PAPER.md Eq. (50) L1556 / Eq. (54) L1881 written
out literally.  Basis convention: state index = sum_i bit_i * 2^(N-1-i) with bit 0 <-> s = +1
(sz = diag(+1, -1), the Pauli-matrix convention of L178 "local values +-1").
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp

_I = sp.identity(2, format="csr", dtype=np.complex128)
_X = sp.csr_matrix(np.array([[0, 1], [1, 0]], dtype=np.complex128))
_Y = sp.csr_matrix(np.array([[0, -1j], [1j, 0]], dtype=np.complex128))
_Z = sp.csr_matrix(np.array([[1, 0], [0, -1]], dtype=np.complex128))


def site_op(P, i, N):
    out = sp.identity(1, format="csr", dtype=np.complex128)
    for k in range(N):
        out = sp.kron(out, P if k == i else _I, format="csr")
    return out


def sigmax(i, N): return site_op(_X, i, N)
def sigmay(i, N): return site_op(_Y, i, N)
def sigmaz(i, N): return site_op(_Z, i, N)


def heisenberg(N, bonds, colors, J):
    """H = sum_b J_c(b) (sx_i sx_j + sy_i sy_j + sz_i sz_j), Eq. (50)."""
    H = sp.csr_matrix((2 ** N, 2 ** N), dtype=np.complex128)
    X = [sigmax(i, N) for i in range(N)]
    Y = [sigmay(i, N) for i in range(N)]
    Z = [sigmaz(i, N) for i in range(N)]
    for b, (i, j) in enumerate(bonds):
        H = H + J[colors[b]] * (X[i] @ X[j] + Y[i] @ Y[j] + Z[i] @ Z[j])
    assert abs(H.imag).max() < 1e-14
    return H.real.tocsr()


def ising(N, bonds, colors, J, h):
    """H = J sum_b sz_i sz_j - h sum_i sx_i, Eq. (54)."""
    H = sp.csr_matrix((2 ** N, 2 ** N), dtype=np.complex128)
    Z = [sigmaz(i, N) for i in range(N)]
    for b, (i, j) in enumerate(bonds):
        H = H + J[colors[b]] * (Z[i] @ Z[j])
    for i in range(N):
        H = H - h * sigmax(i, N)
    return H.real.tocsr()


def all_states(N):
    """int8 [2^N][N]: row `idx` is the basis state with that index (bit 0 <-> +1, site 0 = most significant)."""
    idx = np.arange(2 ** N)
    bits = (idx[:, None] >> (N - 1 - np.arange(N))[None, :]) & 1
    return (1 - 2 * bits).astype(np.int8)


def state_index(sigma):
    sigma = np.atleast_2d(sigma)
    N = sigma.shape[1]
    bits = ((1 - sigma.astype(np.int64)) // 2)
    return (bits << (N - 1 - np.arange(N))[None, :]).sum(axis=1)

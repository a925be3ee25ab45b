"""ORACLE — test infrastructure, NOT the product.

Plain, slow, float64 / complex128 CPU restatement of the batched local-energy estimator of NetKet 3
(arxiv 2112.10526) for an RBM ansatz, written from the paper's definitions.  It shares no code with the
CUDA path (`paper_2112_10526_b200/csrc`), and only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
cpu_baseline / `--impl reference` legs may import it.

What it computes, in the paper's order and notation (citations are PAPER.md lines):
  * `log_cosh(z)`            stable ln cosh z                       (Eq. (41) L1292 names ln cosh; L1298 `logcosh`)
  * `rbm_logpsi`             ln psi(s) = a.s + sum_j ln cosh(W s + b)_j   (RBM: L575; W in C^{MxN}, b in C^M: Eq. (7);
                                                                    formula and visible bias a: BASELINE.json north_star, Q1/Q2)
  * `connected`              get_conn(s) -> (eta, mels): all eta with <s|H|eta> != 0  (Eq. (3))
        Heisenberg  H = sum_b J_c(b) sigma_i . sigma_j   (Eq. (50); Pauli matrices, not S = sigma/2, cf. L1624 "/400")
        Ising       H = J sum_b sz_i sz_j - h sum_i sx_i (Eq. (54))
  * `local_energy`           A~(s) = sum_s' psi(s')/psi(s) <s|A|s'>  (Eq. (12)) — every ln psi(s') FROM SCRATCH
  * `stats`                  E[A~] ~ (1/N_s) sum A~(s_i)            (Eq. (17)) and the population variance (Q10)

  * `rbm_log_derivatives`, `force`, `energy_gradient[_batched]`   O_i = d ln psi/d theta_i (Eq. (13)),
        f~ = Cov[O, H~] (Eq. (14)/(26)), gradient 2 Re f~ | f~ (Eq. (15)/(16), (27)/(28)) — SURVEY.md §8(f) rank 1;
        pins in tests/test_oracle_gradient.py (finite differences of ln psi; finite differences of the exact
        <H> from the dense Kronecker Hamiltonian over the full Born distribution; covariance properties)

  * `rbm_jacobian`, `qgt_dense`, `qgt_matvec`, `sr_solve`   quantum geometric tensor G = Cov[O, O] (Eq. (23)), its product
        with a vector in the three steps of Eq. (75) (QGTOnTheFly), the SR system Eq. (25)/(30)/(31) — SURVEY.md §8(f)
        rank 4; pins in tests/test_oracle_qgt.py (Fubini-Study distance from exact overlaps over the full space,
        np.cov, dense solve residuals)

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): dense Kronecker-product Hamiltonians built independently in
tests/dense_ref.py (Born identity Eq. (11) L646 over the full space; row-by-row equality of the connected list),
Eq. (2), closed forms (W = 0; M = 1 with np.cosh; uniform psi), known ring spectra, symmetries.
No function here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

KIND_HEISENBERG = 0
KIND_ISING = 1
FLAG_MARSHALL = 1  # off-diagonal Heisenberg element -2J instead of +2J (Q6; default off)

LN2 = float(np.log(2.0))


def log_cosh(z):
    """ln cosh z, stable for large |Re z|; real or complex input (float64 / complex128).

    cosh is even, so flip z to Re z >= 0, then ln cosh z = z + log1p(exp(-2z)) - ln 2 (principal log1p;
    its argument has |exp(-2z)| <= 1).  DESIGN.md Q11.
    """
    z = np.asarray(z)
    if np.iscomplexobj(z):
        z = z.astype(np.complex128)
        z = np.where(z.real < 0, -z, z)
        return z + np.log1p(np.exp(-2.0 * z)) - LN2
    z = np.abs(z.astype(np.float64))
    return z + np.log1p(np.exp(-2.0 * z)) - LN2


def _up(x, cplx):
    """Exact up-cast of fp32 / complex64 stored parameters (Q12)."""
    return np.asarray(x).astype(np.complex128 if cplx else np.float64)


def rbm_logpsi(sigma, W, a=None, b=None):
    """ln psi for a batch.  sigma [B][N] (+-1), W [M][N], a [N] or None, b [M] or None -> [B]."""
    sigma = np.atleast_2d(np.asarray(sigma))
    cplx = np.iscomplexobj(W)
    W = _up(W, cplx)
    s = sigma.astype(np.complex128 if cplx else np.float64)
    theta = s @ W.T                                   # theta = W s        (Eq. (7))
    if b is not None:
        theta = theta + _up(b, cplx)[None, :]         #       + b
    out = log_cosh(theta).sum(axis=1)                 # sum_j ln cosh theta_j
    if a is not None:
        out = out + s @ _up(a, cplx)                  # + sum_i a_i s_i
    return out


def rbm_theta(sigma, W, b=None):
    """theta = W s + b for a batch, float64/complex128 [B][M]."""
    cplx = np.iscomplexobj(W)
    theta = np.atleast_2d(np.asarray(sigma)).astype(np.complex128 if cplx else np.float64) @ _up(W, cplx).T
    if b is not None:
        theta = theta + _up(b, cplx)[None, :]
    return theta


def max_conn(kind, n_sites, n_bonds):
    """Fixed width C of the connected list: slot 0 diagonal + one slot per bond (Heisenberg) / per site (Ising)."""
    return (n_bonds if kind == KIND_HEISENBERG else n_sites) + 1


def connected(kind, sigma_row, bonds, colors, J, h=0.0, flags=0):
    """get_conn for ONE basis state (Eq. (3)), fixed-width convention of DESIGN.md Q9.

    Returns (sigma_prime int8 [C][N], mels float64 [C], flips int32 [C][2], n_conn int):
      slot 0        diagonal: sigma itself, H_ss, flips (-1,-1) — always present, even if 0
      Heisenberg    slot 1+b <-> bond b=(i,j): if s_i != s_j the two spins are exchanged, element 2*J_c(b)
                    (-2*J_c(b) with FLAG_MARSHALL), flips (i,j); if s_i == s_j a PADDED slot: sigma itself,
                    element 0, flips (-1,-1)
      Ising         slot 1+k <-> site k: spin k negated, element -h, flips (k,-1)
      n_conn        number of non-padded slots (diagonal included)
    """
    s = np.asarray(sigma_row, dtype=np.int8)
    N = s.shape[0]
    bonds = np.asarray(bonds)
    J = np.asarray(J, dtype=np.float64)
    colors = np.zeros(len(bonds), dtype=np.int64) if colors is None else np.asarray(colors)
    C = max_conn(kind, N, len(bonds))
    sp = np.tile(s, (C, 1))
    mels = np.zeros(C, dtype=np.float64)
    flips = np.full((C, 2), -1, dtype=np.int32)
    diag = 0.0
    for bnd, (i, j) in enumerate(bonds):              # sz_i sz_j term of every bond (both models)
        diag += J[colors[bnd]] * float(s[i]) * float(s[j])
    mels[0] = diag
    n_conn = 1
    if kind == KIND_HEISENBERG:
        # sx sx + sy sy = 2 (s+ s- + s- s+): exchanges antiparallel spins with element 2 (Pauli convention)
        off = -2.0 if (flags & FLAG_MARSHALL) else 2.0
        for bnd, (i, j) in enumerate(bonds):
            if s[i] != s[j]:
                sp[1 + bnd, i], sp[1 + bnd, j] = s[j], s[i]
                mels[1 + bnd] = off * J[colors[bnd]]
                flips[1 + bnd] = (i, j)
                n_conn += 1
    elif kind == KIND_ISING:
        for k in range(N):                            # -h sx_k flips spin k
            sp[1 + k, k] = -s[k]
            mels[1 + k] = -h
            flips[1 + k] = (k, -1)
            n_conn += 1
    else:
        raise ValueError("unknown operator kind")
    return sp, mels, flips, n_conn


def local_energy(kind, sigma, bonds, colors, J, h, W, a=None, b=None, flags=0):
    """Local estimator Eq. (12) L652 for every row of sigma: sum over the connected list of
    mel * exp(ln psi(s') - ln psi(s)), with EVERY ln psi(s') evaluated from scratch by `rbm_logpsi`.
    Returns (eloc [B] float64|complex128, logpsi [B])."""
    sigma = np.atleast_2d(np.asarray(sigma, dtype=np.int8))
    cplx = np.iscomplexobj(W)
    B = sigma.shape[0]
    eloc = np.zeros(B, dtype=np.complex128 if cplx else np.float64)
    logpsi = rbm_logpsi(sigma, W, a, b)
    for n in range(B):
        sp, mels, _, _ = connected(kind, sigma[n], bonds, colors, J, h, flags)
        lp = rbm_logpsi(sp, W, a, b)                  # all C configurations, nothing incremental
        eloc[n] = np.sum(mels * np.exp(lp - logpsi[n]))
    return eloc, logpsi


def stats(eloc):
    """Eq. (17): mean over the batch; population variance mean |E - mean|^2 (ddof = 0).
    Returns (mean_re, mean_im, variance, count) as float64."""
    e = np.asarray(eloc).astype(np.complex128)
    m = e.sum() / e.size
    var = float(np.sum(np.abs(e - m) ** 2) / e.size)
    return float(m.real), float(m.imag), var, float(e.size)


def count_amplitudes(kind, sigma, bonds, colors, J, h=0.0):
    """Number of off-diagonal connected entries with non-zero matrix element, summed over the batch
    (the numerator of 'connected-amplitude evaluations/s')."""
    sigma = np.atleast_2d(np.asarray(sigma, dtype=np.int8))
    bonds = np.asarray(bonds)
    if kind == KIND_ISING:
        return int(sigma.shape[0] * sigma.shape[1]) if h != 0.0 else 0
    J = np.asarray(J, dtype=np.float64)
    colors = np.zeros(len(bonds), dtype=np.int64) if colors is None else np.asarray(colors)
    anti = sigma[:, bonds[:, 0]] != sigma[:, bonds[:, 1]]
    return int(anti[:, J[colors] != 0.0].sum())


# ---------------------------------------------------------------------------------------------------------
# NEXT-1: force vector / energy gradient for the RBM
# ---------------------------------------------------------------------------------------------------------
def rbm_log_derivatives(sigma, W, b=None):
    """Log-derivatives O_i(s) = d ln psi(s) / d theta_i (Eq. (13)) of the RBM, written out from
    ln psi = a.s + sum_j ln cosh(W s + b)_j:   O_{a_k} = s_k,  O_{b_j} = tanh theta_j,  O_{W_jk} = tanh theta_j s_k.
    (Pinned by central finite differences of `rbm_logpsi` in tests/test_oracle_gradient.py.)
    Returns (O_a [B][N], O_b [B][M], O_W [B][M][N])."""
    sigma = np.atleast_2d(np.asarray(sigma))
    theta = rbm_theta(sigma, W, b)
    T = np.tanh(theta)
    s = sigma.astype(T.dtype)
    return s, T, T[:, :, None] * s[:, None, :]


def force(O, eloc, weights=None):
    """Force vector f~_i = Cov[O_i, H~] = E[O_i^* (H~ - E[H~])] (Eq. (14), Eq. (26)).
    E[.] is the sample mean (Eq. (17)); `weights` (normalised probabilities) replaces it by a weighted mean —
    used only by the exact-distribution pin."""
    O = np.asarray(O)
    e = np.asarray(eloc).astype(np.complex128 if np.iscomplexobj(eloc) or np.iscomplexobj(O) else np.float64)
    if weights is None:
        weights = np.full(e.shape[0], 1.0 / e.shape[0])
    w = np.asarray(weights, dtype=np.float64)
    de = e - np.sum(w * e)
    return np.tensordot(w * de, np.conj(O), axes=(0, 0))


def energy_gradient(sigma, W, b, eloc, weights=None):
    """Gradient of <H> from samples: real parameters f = 2 Re f~ (Eq. (15) L664 / Eq. (27)); complex
    parameters of a holomorphic ansatz (the complex RBM is one) f = f~ (Eq. (16) L668 / Eq. (28)).
    Returns (g_a [N], g_b [M], g_W [M][N])."""
    cplx = np.iscomplexobj(W)
    O_a, O_b, O_W = rbm_log_derivatives(sigma, W, b)
    out = []
    for O in (O_a, O_b, O_W):
        f = force(O, eloc, weights)
        out.append(f if cplx else 2.0 * np.real(f))
    return tuple(out)


def energy_gradient_batched(sigma, W, b, eloc):
    """Same numbers as `energy_gradient` without the [B][M][N] tensor of O_W (needed at full batch size):
    g_W = sum_s conj(tanh theta_s) (dE_s / B) s_s^T as one library matmul."""
    cplx = np.iscomplexobj(W)
    sigma = np.atleast_2d(np.asarray(sigma))
    T = np.tanh(rbm_theta(sigma, W, b))
    e = np.asarray(eloc).astype(np.complex128 if cplx else np.float64)
    de = (e - e.mean()) / e.shape[0]
    s = sigma.astype(T.dtype)
    g_a = de @ s
    g_b = de @ np.conj(T)
    g_W = (np.conj(T) * de[:, None]).T @ s
    if not cplx:
        return 2.0 * g_a.real, 2.0 * g_b.real, 2.0 * g_W.real
    return g_a, g_b, g_W


# ---------------------------------------------------------------------------------------------------------
# NEXT-4: quantum geometric tensor times a vector, stochastic reconfiguration
# ---------------------------------------------------------------------------------------------------------
def rbm_jacobian(sigma, W, b=None):
    """J [B][P]: row s holds the log-derivatives O_i(s) (Eq. (13)) in the order a (N), b (M), W (M*N row-major),
    P = N + M + M N.  ("the full Jacobian matrix J_kl", App. B.2)"""
    O_a, O_b, O_W = rbm_log_derivatives(sigma, W, b)
    return np.concatenate([O_a, O_b, O_W.reshape(O_W.shape[0], -1)], axis=1)


def qgt_dense(sigma, W, b=None, weights=None):
    """G_ij = E[O_i^* O_j] - E[O_i^*] E[O_j]  (Eq. (23)) as a dense P x P matrix; E[.] the sample mean, or
    the weighted mean with normalised `weights` (exact-distribution pin only).  Real parameters: G is real."""
    J = rbm_jacobian(sigma, W, b)
    B = J.shape[0]
    w = np.full(B, 1.0 / B) if weights is None else np.asarray(weights, dtype=np.float64)
    mean = w @ J
    return (np.conj(J) * w[:, None]).T @ J - np.outer(np.conj(mean), mean)


def pack_params(v_a, v_b, v_W):
    return np.concatenate([np.ravel(v_a), np.ravel(v_b), np.ravel(v_W)])


def unpack_params(v, N, M):
    return v[:N], v[N:N + M], v[N + M:].reshape(M, N)


def qgt_matvec(sigma, W, b, v_a, v_b, v_W, diag_shift=0.0):
    """(G + eps) v without forming G, in the three steps of Eq. (75) L2219 (QGTOnTheFly):
        w = (1/N_s) J v;   dw = w - <w>;   v~ = J^dagger dw;     then  + eps v  (Eq. (25)).
    Returns (v~_a [N], v~_b [M], v~_W [M][N]).  Real parameters: Re[G] v (Eq. (30)) — G is real there."""
    sigma = np.atleast_2d(np.asarray(sigma))
    N, M = sigma.shape[1], np.shape(W)[0]
    J = rbm_jacobian(sigma, W, b)
    v = pack_params(v_a, v_b, v_W).astype(J.dtype)
    w = (J @ v) / J.shape[0]
    dw = w - w.mean()
    out = np.conj(J).T @ dw + diag_shift * v
    if not np.iscomplexobj(W):
        out = out.real
    return unpack_params(out, N, M)


def qgt_matvec_batched(sigma, W, b, v_a, v_b, v_W, diag_shift=0.0, return_w=False):
    """Same numbers as `qgt_matvec` without the [B][P] Jacobian (needed at full batch size): with O_a = s,
    O_b = tanh theta, O_W = tanh theta s^T (Eq. (13)) the three steps of Eq. (75) L2219 are
        (J v)_s = s_s . v_a + sum_j tanh(theta_sj) (v_b,j + (V_W s_s)_j),
        dw = (J v) / N_s - <(J v) / N_s>,
        v~_a = s^T dw,   v~_b = conj(tanh theta)^T dw,   v~_W = (conj(tanh theta) * dw)^T s,
    as library matmuls; + eps v (Eq. (25)).  return_w: also return J v (the tests' error scale)."""
    cplx = np.iscomplexobj(W)
    sigma = np.atleast_2d(np.asarray(sigma))
    dt = np.complex128 if cplx else np.float64
    T = np.tanh(rbm_theta(sigma, W, b))
    s = sigma.astype(dt)
    v_a, v_b, v_W = (np.asarray(x).astype(dt) for x in (v_a, v_b, v_W))
    Jv = s @ v_a + np.sum(T * (v_b[None, :] + s @ v_W.T), axis=1)
    w = Jv / sigma.shape[0]
    dw = w - w.mean()
    out_a = s.T @ dw + diag_shift * v_a
    out_b = np.conj(T).T @ dw + diag_shift * v_b
    out_W = (np.conj(T) * dw[:, None]).T @ s + diag_shift * v_W
    if not cplx:
        out_a, out_b, out_W = out_a.real, out_b.real, out_W.real
    return (out_a, out_b, out_W, Jv) if return_w else (out_a, out_b, out_W)


def sr_solve(sigma, W, b, f_a, f_b, f_W, diag_shift):
    """Stochastic reconfiguration: the solution delta of sum_j (G_ij + eps delta_ij) delta_j = f_i
    (Eq. (25) L886 with Eq. (30)/(31) L961-967), by a dense direct solve of the definition."""
    sigma = np.atleast_2d(np.asarray(sigma))
    N, M = sigma.shape[1], np.shape(W)[0]
    G = qgt_dense(sigma, W, b)
    if not np.iscomplexobj(W):
        G = G.real
    f = pack_params(f_a, f_b, f_W).astype(G.dtype)
    return unpack_params(np.linalg.solve(G + diag_shift * np.eye(G.shape[0]), f), N, M)


# ---------------------------------------------------------------------------------------------------------
# NEXT-4, second workload: the fully symmetric RBM (RBMSymm)
# ---------------------------------------------------------------------------------------------------------
def rbmsymm_features(sigma, W_sym, b_sym, perms):
    """f_g^(i)(s) = sum_r W^(i)_r s_{g r} + b^(i)   (the embedding layer, Eq. (56), with a bias per feature).
    sigma [B][N]; W_sym [F][N]; b_sym [F] or None; perms int [G][N] with perms[g][r] = the site g r.  Returns [B][F][G]."""
    sigma = np.atleast_2d(np.asarray(sigma))
    cplx = np.iscomplexobj(W_sym)
    W = _up(W_sym, cplx)
    s = sigma.astype(W.dtype)
    perms = np.asarray(perms)
    f = np.einsum("ir,sgr->sig", W, s[:, perms])         # s[:, perms][s][g][r] = s_{g r}
    if b_sym is not None:
        f = f + _up(b_sym, cplx)[None, :, None]
    return f


def rbmsymm_logpsi(sigma, W_sym, b_sym, perms):
    """ln psi = sum_{i, g in G} ln cosh f_g^(i)   (Eq. (41))."""
    f = rbmsymm_features(sigma, W_sym, b_sym, perms)
    return log_cosh(f).reshape(f.shape[0], -1).sum(axis=1)


def rbmsymm_local_energy(kind, sigma, bonds, colors, J, h, W_sym, b_sym, perms, flags=0):
    """Eq. (12) L652 for the symmetric RBM, every ln psi(s') from scratch through `rbmsymm_logpsi`."""
    sigma = np.atleast_2d(np.asarray(sigma))
    lp = rbmsymm_logpsi(sigma, W_sym, b_sym, perms)
    out = np.zeros(sigma.shape[0], dtype=np.complex128 if np.iscomplexobj(W_sym) else np.float64)
    for n in range(sigma.shape[0]):
        eta, mels, _, _ = connected(kind, sigma[n], bonds, colors, J, h, flags)
        out[n] = np.sum(mels * np.exp(rbmsymm_logpsi(eta, W_sym, b_sym, perms) - lp[n]))
    return out, lp


def rbmsymm_energy_gradient(sigma, W_sym, b_sym, perms, eloc):
    """Gradient of <H> with respect to the tied parameters: O_{b^(i)} = sum_g tanh f_g^(i),
    O_{W^(i)_r} = sum_g tanh f_g^(i) s_{g r} (Eq. (13) applied to Eq. (41)/(56)); f~ = E[O^* (H~ - E[H~])], gradient
    2 Re f~ (real) or f~ (complex), Eq. (14)-(16).  Returns (g_b [F], g_W [F][N])."""
    sigma = np.atleast_2d(np.asarray(sigma))
    cplx = np.iscomplexobj(W_sym)
    T = np.tanh(rbmsymm_features(sigma, W_sym, b_sym, perms))       # [B][F][G]
    s = sigma.astype(T.dtype)[:, np.asarray(perms)]                   # [B][G][N]: s_{g r}
    O_b = T.sum(axis=2)
    O_W = np.einsum("sig,sgr->sir", T, s)
    gb, gW = force(O_b, eloc), force(O_W, eloc)
    return (gb, gW) if cplx else (2.0 * gb.real, 2.0 * gW.real)

"""Pins of the sampler oracle (oracle/nk_sampler_oracle.py) against things other than itself — CPU only.

* Philox4x32-10: the three known-answer vectors shipped with the Random123 library (kat_vectors, "philox4x32 10").
* One transition from a fixed state: empirical frequencies over many chains against the exact transition row
  T(s -> s') = (1/n) min(1, |psi(s')|^2 / |psi(s)|^2) built here from np.cosh directly (Eq. (20)).
* Stationary distribution on a 6-site ring against |psi|^2 / Z over the enumerated space (chi-square).
* Closed forms: uniform psi accepts everything; W = 0 gives independent spins with P(+1) = e^{2a} / (e^{2a}+e^{-2a});
  the exchange rule conserves sum(sigma) and never leaves the sector.
"""
import numpy as np

from oracle import nk_sampler_oracle as smp


def test_philox_known_answer_vectors():
    kat = [
        ((0, 0, 0, 0), (0, 0), (0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8)),
        ((0xFFFFFFFF,) * 4, (0xFFFFFFFF,) * 2, (0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD)),
        ((0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344), (0xA4093822, 0x299F31D0),
         (0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1)),
    ]
    for ctr, key, want in kat:
        got = smp.philox4x32_10(*[np.uint32(c) for c in ctr], *[np.uint32(k) for k in key])
        assert tuple(int(g) for g in got) == want


def test_philox_is_vectorised_consistently():
    c = np.arange(7, dtype=np.uint32)
    out = smp.philox4x32_10(c, 1, 2, 3, 4, 5)
    for i in range(7):
        one = smp.philox4x32_10(np.uint32(i), 1, 2, 3, 4, 5)
        assert all(int(o[i]) == int(x) for o, x in zip(out, one))


def test_uniform_and_index_ranges():
    r0, u = smp.draw(12345, np.arange(100000), 7)
    assert u.min() > 0.0 and u.max() < 1.0
    assert np.all(u == u.astype(np.float32).astype(np.float64))          # exact in fp32
    assert abs(u.mean() - 0.5) < 5e-3 and abs(u.var() - 1 / 12) < 5e-3
    idx = smp.proposal_index(r0, 10)
    assert idx.min() == 0 and idx.max() == 9
    counts = np.bincount(idx, minlength=10)
    assert np.all(np.abs(counts - 1e4) < 5 * np.sqrt(1e4))
    assert smp.proposal_index(np.array([0xFFFFFFFF], dtype=np.uint32), 1024)[0] == 1023


def _psi2(states, W, a, b):
    """|psi|^2 straight from the definition with np.cosh (no log-cosh, no oracle code)."""
    s = states.astype(np.complex128 if np.iscomplexobj(W) else np.float64)
    theta = s @ W.T + b[None, :]
    psi = np.exp(s @ a) * np.prod(np.cosh(theta), axis=1)
    return np.abs(psi) ** 2


def _params(N, M, scale, seed, cplx=False):
    rng = np.random.default_rng(seed)
    def d(*sh):
        x = rng.normal(size=sh) * scale
        if cplx:
            return (x + 1j * rng.normal(size=sh) * scale).astype(np.complex64)
        return x.astype(np.float32)
    return d(M, N), d(N), d(M)


def _index(states):
    return ((states < 0).astype(np.int64) << np.arange(states.shape[1])[None, :]).sum(axis=1)


def _all_states(N):
    k = np.arange(2 ** N)[:, None]
    return (1 - 2 * ((k >> np.arange(N)[None, :]) & 1)).astype(np.int8)


def test_single_transition_frequencies_local_rule():
    N, M, B = 5, 7, 200000
    W, a, b = _params(N, M, 0.4, 11, cplx=True)
    s0 = np.array([1, -1, -1, 1, -1], dtype=np.int8)
    sig, acc, _, _ = smp.metropolis(smp.RULE_LOCAL, np.tile(s0, (B, 1)), W, a, b, 1, seed=99)
    W64, a64, b64 = (x.astype(np.complex128) for x in (W, a, b))
    p0 = _psi2(s0[None, :], W64, a64, b64)[0]
    expect_stay = 0.0
    for k in range(N):
        sp = s0.copy(); sp[k] = -sp[k]
        t = min(1.0, _psi2(sp[None, :], W64, a64, b64)[0] / p0) / N
        got = np.mean(np.all(sig == sp[None, :], axis=1))
        assert abs(got - t) < 5 * np.sqrt(t * (1 - t) / B) + 1e-9, (k, got, t)
        expect_stay += 1.0 / N - t
    got_stay = np.mean(np.all(sig == s0[None, :], axis=1))
    assert abs(got_stay - expect_stay) < 5 * np.sqrt(max(expect_stay, 1e-4) / B)
    assert abs(acc.mean() - (1 - expect_stay)) < 5 * np.sqrt(0.25 / B)


def test_single_transition_frequencies_exchange_rule():
    N, M, B = 6, 6, 200000
    W, a, b = _params(N, M, 0.5, 12)
    clusters = np.array([[i, (i + 1) % N] for i in range(N)])
    s0 = np.array([1, 1, -1, 1, -1, -1], dtype=np.int8)
    sig, acc, _, _ = smp.metropolis(smp.RULE_EXCHANGE, np.tile(s0, (B, 1)), W, a, b, 1, seed=5, clusters=clusters)
    W64, a64, b64 = (x.astype(np.float64) for x in (W, a, b))
    p0 = _psi2(s0[None, :], W64, a64, b64)[0]
    accepted = 0.0
    for i, j in clusters:
        sp = s0.copy(); sp[i], sp[j] = s0[j], s0[i]
        if np.array_equal(sp, s0):
            accepted += 1.0 / N                                   # trivial exchange: ratio 1
            continue
        t = min(1.0, _psi2(sp[None, :], W64, a64, b64)[0] / p0) / N
        accepted += t
        got = np.mean(np.all(sig == sp[None, :], axis=1))
        assert abs(got - t) < 5 * np.sqrt(t * (1 - t) / B) + 1e-9
    assert abs(acc.mean() - accepted) < 5 * np.sqrt(0.25 / B)
    assert np.all(sig.sum(axis=1) == s0.sum())


def _chi2_ok(counts, p, B):
    exp = p * B
    keep = exp > 5
    chi2 = np.sum((counts[keep] - exp[keep]) ** 2 / exp[keep])
    dof = keep.sum() - 1
    return chi2 < dof + 6 * np.sqrt(2 * dof), (chi2, dof)


def test_stationary_distribution_local_rule():
    N, M, B = 6, 8, 40000
    W, a, b = _params(N, M, 0.35, 21)
    rng = np.random.default_rng(3)
    s0 = (1 - 2 * rng.integers(0, 2, size=(B, N))).astype(np.int8)
    sig, _, _, lp = smp.metropolis(smp.RULE_LOCAL, s0, W, a, b, 20 * N, seed=2024)
    states = _all_states(N)
    p = _psi2(states, *(x.astype(np.float64) for x in (W, a, b)))
    p /= p.sum()
    ok, info = _chi2_ok(np.bincount(_index(sig), minlength=2 ** N), p, B)
    assert ok, info
    # the returned ln psi belongs to the final states
    from oracle import nk_oracle as orc
    assert np.allclose(lp, orc.rbm_logpsi(sig, W, a, b), atol=1e-12)


def test_stationary_distribution_exchange_rule_in_sector():
    N, M, B = 6, 6, 20000
    W, a, b = _params(N, M, 0.25, 22, cplx=True)
    clusters = np.array([[i, (i + 1) % N] for i in range(N)])
    base = np.array([1, -1, 1, -1, 1, -1], dtype=np.int8)
    sig, _, _, _ = smp.metropolis(smp.RULE_EXCHANGE, np.tile(base, (B, 1)), W, a, b, 150 * N, seed=77,
                                  clusters=clusters)
    assert np.all(sig.sum(axis=1) == 0)
    states = _all_states(N)
    sector = states[states.sum(axis=1) == 0]
    p = _psi2(sector, *(x.astype(np.complex128) for x in (W, a, b)))
    p /= p.sum()
    lookup = {int(k): n for n, k in enumerate(_index(sector))}
    counts = np.bincount([lookup[int(k)] for k in _index(sig)], minlength=len(sector))
    ok, info = _chi2_ok(counts, p, B)
    assert ok, info


def test_uniform_psi_accepts_every_proposal():
    N, B = 8, 64
    W = np.zeros((4, N), dtype=np.float32)
    z = np.zeros(N, dtype=np.float32)
    rng = np.random.default_rng(0)
    s0 = (1 - 2 * rng.integers(0, 2, size=(B, N))).astype(np.int8)
    sig, acc, margin, _ = smp.metropolis(smp.RULE_LOCAL, s0, W, z, np.zeros(4, dtype=np.float32), 3 * N, seed=1)
    assert np.all(acc == 3 * N)
    # replay the proposals by hand: every one of them was applied
    want = s0.copy()
    for t in range(3 * N):
        r0, _ = smp.draw(1, np.arange(B), t)
        k = smp.proposal_index(r0, N)
        want[np.arange(B), k] *= -1
    assert np.array_equal(sig, want)


def test_w_zero_gives_independent_spins():
    N, B = 4, 60000
    a = np.array([0.3, -0.2, 0.0, 0.5], dtype=np.float32)
    W = np.zeros((3, N), dtype=np.float32)
    b = np.array([0.1, -0.4, 0.2], dtype=np.float32)                 # b only rescales psi
    s0 = np.ones((B, N), dtype=np.int8)
    sig, _, _, _ = smp.metropolis(smp.RULE_LOCAL, s0, W, a, b, 30 * N, seed=8)
    a64 = a.astype(np.float64)
    p_up = np.exp(2 * a64) / (np.exp(2 * a64) + np.exp(-2 * a64))
    got = (sig > 0).mean(axis=0)
    assert np.all(np.abs(got - p_up) < 5 * np.sqrt(0.25 / B))


def test_step_and_chain_offsets_compose():
    N, M, B = 6, 5, 32
    W, a, b = _params(N, M, 0.4, 31)
    rng = np.random.default_rng(1)
    s0 = (1 - 2 * rng.integers(0, 2, size=(B, N))).astype(np.int8)
    full, acc_full, _, _ = smp.metropolis(smp.RULE_LOCAL, s0, W, a, b, 24, seed=3)
    half, acc1, _, _ = smp.metropolis(smp.RULE_LOCAL, s0, W, a, b, 10, seed=3)
    rest, acc2, _, _ = smp.metropolis(smp.RULE_LOCAL, half, W, a, b, 14, seed=3, step_offset=10)
    assert np.array_equal(full, rest) and np.array_equal(acc_full, acc1 + acc2)
    part, _, _, _ = smp.metropolis(smp.RULE_LOCAL, s0[8:], W, a, b, 24, seed=3, chain_offset=8)
    assert np.array_equal(full[8:], part)

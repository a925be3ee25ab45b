"""ORACLE (sampler part) — test infrastructure, NOT the product.

Plain float64 restatement of the Metropolis-Hastings sampler of NetKet 3 (arxiv 2112.10526, Sec. 3.4) for the RBM
ansatz, SURVEY.md §8(f) rank 2.  It shares no code with the CUDA path; only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline leg may import it.  Citations are PAPER.md lines.

  * acceptance            P_acc(s -> s') = min(1, P(s')/P(s) g(s|s')/g(s'|s)),  P(s) ∝ |psi(s)|^2      Eq. (20)
                          local flips and exchanges are symmetric kernels: the g-factor is 1               L711
  * `MetropolisLocal`     "changes one discrete local degree of freedom in each transition"                L713
  * `MetropolisExchange`  "exchanges two local degrees of freedom respecting a conserved quantity"         L713
                          the pair is an edge of the lattice graph (`graph=lattice`, L1600-1604)
  * chains                n_chains independent chains advanced together (`sigma.shape[0]`, L727); one sweep =
                          N_sites transitions ("N_sites intermediate updates", footnote 20 L1590)

Where the paper is silent (S1-S5): the random numbers.  Both sides implement the SAME counter-based
generator, Philox4x32-10 (Salmon et al., SC'11), each from the published round function:
  counter = (chain index lo, hi, transition index lo, hi), key = (seed lo, hi)  ->  four uint32 (r0, r1, r2, r3)
  proposal index  = (r0 * n) >> 32        (n = N sites, or the number of exchange pairs)   -- integer, bit-exact
  uniform         u = ((r1 >> 9) + 1/2) 2^-23   in (0, 1), exact in fp32 and fp64
  accept  iff  u < |psi(s')/psi(s)|^2    (every ln psi(s') is evaluated FROM SCRATCH here, in float64)
An exchange of two equal spins proposes s' = s: ratio 1, accepted (and counted as accepted), state unchanged.

`metropolis` also returns, per chain, the smallest |ln u - 2 Re(ln psi' - ln psi)| over its transitions: the distance
of its closest accept/reject decision from the boundary.  The fp32 GPU path may legitimately take the other branch
when that distance is below its rounding error; parity tests compare chains bit for bit where the margin is clear and
check validity (spin values, conserved magnetisation) for the rest.

Pins (tests/test_oracle_sampler.py): Philox known-answer vectors of the Random123 distribution; one-transition
frequencies from a fixed state against the exact transition row built from the dense |psi|^2 in the test; the
stationary histogram on a 6-site chain against |psi|^2 / Z (chi-square); independent-spin closed form for W = 0;
uniform psi accepts everything; exchange conserves sum(sigma).
"""
from __future__ import annotations

import numpy as np

from . import nk_oracle as _orc

RULE_LOCAL = 0
RULE_EXCHANGE = 1

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = np.uint32(0x9E3779B9)
_W1 = np.uint32(0xBB67AE85)
_MASK = np.uint64(0xFFFFFFFF)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Philox4x32 with 10 rounds.  All arguments uint32 arrays (broadcastable); returns four uint32 arrays.

    One round (Salmon et al. 2011, Sec. 3.3):  (hi0, lo0) = M0 * c0,  (hi1, lo1) = M1 * c2,
      c' = (hi1 ^ c1 ^ k0,  lo1,  hi0 ^ c3 ^ k1,  lo0);   the key is bumped by (W0, W1) between rounds.
    """
    c0, c1, c2, c3, k0, k1 = (np.asarray(x, dtype=np.uint32) for x in (c0, c1, c2, c3, k0, k1))
    c0, c1, c2, c3, k0, k1 = np.broadcast_arrays(c0, c1, c2, c3, k0, k1)
    c0, c1, c2, c3, k0, k1 = (x.copy() for x in (c0, c1, c2, c3, k0, k1))
    with np.errstate(over="ignore"):
        for r in range(10):
            p0 = _M0 * c0.astype(np.uint64)
            p1 = _M1 * c2.astype(np.uint64)
            hi0, lo0 = (p0 >> np.uint64(32)).astype(np.uint32), (p0 & _MASK).astype(np.uint32)
            hi1, lo1 = (p1 >> np.uint64(32)).astype(np.uint32), (p1 & _MASK).astype(np.uint32)
            c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
            if r < 9:
                k0 = k0 + _W0
                k1 = k1 + _W1
    return c0, c1, c2, c3


def draw(seed, chain, step):
    """(proposal word r0, uniform u in (0,1)) for chains `chain` (int array) at transition index `step` (int)."""
    seed = int(seed)
    chain = np.asarray(chain, dtype=np.uint64)
    step = np.uint64(step)
    r0, r1, _, _ = philox4x32_10((chain & _MASK).astype(np.uint32), (chain >> np.uint64(32)).astype(np.uint32),
                                 np.uint32(step & _MASK), np.uint32(step >> np.uint64(32)),
                                 np.uint32(seed & 0xFFFFFFFF), np.uint32((seed >> 32) & 0xFFFFFFFF))
    u = ((r1 >> np.uint32(9)).astype(np.float64) + 0.5) * 2.0 ** -23
    return r0, u


def proposal_index(r0, n):
    """(r0 * n) >> 32 : an index in [0, n), integer arithmetic."""
    return ((r0.astype(np.uint64) * np.uint64(n)) >> np.uint64(32)).astype(np.int64)


def propose(rule, sigma, idx, clusters=None):
    """sigma' for every chain.  Local: negate spin idx.  Exchange: swap the spins of pair clusters[idx]."""
    sp = sigma.copy()
    rows = np.arange(sigma.shape[0])
    if rule == RULE_LOCAL:
        sp[rows, idx] = -sigma[rows, idx]
    elif rule == RULE_EXCHANGE:
        i, j = clusters[idx, 0], clusters[idx, 1]
        sp[rows, i] = sigma[rows, j]
        sp[rows, j] = sigma[rows, i]
    else:
        raise ValueError("rule")
    return sp


def metropolis(rule, sigma0, W, a, b, n_steps, seed, *, clusters=None, step_offset=0, chain_offset=0):
    """Advance every row of sigma0 by n_steps Metropolis-Hastings transitions (Eq. (20)).

    Returns (sigma [B][N] int8, accepted [B] int64, min_margin [B] float64, logpsi [B] of the final states).
    """
    sigma = np.array(sigma0, dtype=np.int8, copy=True)
    B, N = sigma.shape
    n = N if rule == RULE_LOCAL else len(clusters)
    if clusters is not None:
        clusters = np.asarray(clusters, dtype=np.int64)
    chain = np.arange(B, dtype=np.uint64) + np.uint64(chain_offset)
    accepted = np.zeros(B, dtype=np.int64)
    margin = np.full(B, np.inf)
    lp = _orc.rbm_logpsi(sigma, W, a, b)
    for t in range(n_steps):
        r0, u = draw(seed, chain, step_offset + t)
        idx = proposal_index(r0, n)
        sp = propose(rule, sigma, idx, clusters)
        lp_new = _orc.rbm_logpsi(sp, W, a, b)                       # from scratch
        log_ratio = 2.0 * np.real(lp_new - lp)                      # ln |psi'/psi|^2
        moved = np.any(sp != sigma, axis=1)
        acc = np.where(moved, np.log(u) < log_ratio, True)          # s' = s: ratio 1 > u
        margin = np.where(moved, np.minimum(margin, np.abs(np.log(u) - log_ratio)), margin)
        sigma[acc] = sp[acc]
        lp = np.where(acc, lp_new, lp)
        accepted += acc
    return sigma, accepted, margin, lp

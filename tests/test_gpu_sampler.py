"""GPU parity of nk_metropolis_sample against the float64 sampler oracle (oracle/nk_sampler_oracle.py).

Both sides consume the same Philox4x32-10 stream, so a chain is reproduced BIT FOR BIT unless one of its
accept/reject decisions falls closer to the boundary than the fp32 rounding of |psi'/psi|^2: the oracle reports, per
chain, the smallest |ln u - ln|psi'/psi|^2| it met.  Chains whose margin exceeds MARGIN_TOL must agree exactly (final
configuration and accepted count); the remaining few must still be valid chains (spins +-1, magnetisation conserved
under the exchange rule).  MARGIN_TOL = 2e-4: the measured fp32 error of ln|ratio|^2 is < 2e-5 on these inputs
(incremental theta after hundreds of accepted moves included), a factor 10 below.
"""
import numpy as np
import pytest
import torch

from oracle import nk_sampler_oracle as smp
from paper_2112_10526_b200 import inputs as inp

pytestmark = pytest.mark.gpu
MARGIN_TOL = 2e-4


def dev(x):
    return None if x is None else torch.from_numpy(np.ascontiguousarray(x)).cuda()


def run_both(nk, p, rule, n_steps, *, seed=7, chunk=0, step_offset=0, chain_offset=0, a=True, b=True):
    clusters = p.bonds if rule == nk.NK_RULE_EXCHANGE else None
    sig = dev(p.sigma)
    acc = nk.metropolis_sample(sig, dev(p.W), dev(p.a) if a else None, dev(p.b) if b else None, rule=rule,
                               clusters=clusters, n_steps=n_steps, seed=seed, step_offset=step_offset,
                               chain_offset=chain_offset, chunk_size=chunk)
    torch.cuda.synchronize()
    ref, racc, margin, _ = smp.metropolis(rule, p.sigma, p.W, p.a if a else None, p.b if b else None, n_steps, seed,
                                          clusters=clusters, step_offset=step_offset, chain_offset=chain_offset)
    return sig.cpu().numpy(), acc.cpu().numpy(), ref, racc, margin


def assert_chains(p, rule, got, gacc, ref, racc, margin, min_clear=0.8):
    assert set(np.unique(got)) <= {-1, 1}
    if rule == smp.RULE_EXCHANGE:
        assert np.array_equal(got.sum(axis=1), p.sigma.sum(axis=1))
    clear = margin > MARGIN_TOL
    assert clear.mean() >= min_clear, f"only {clear.mean():.2f} of the chains have a clear margin"
    same = np.all(got == ref, axis=1) & (gacc == racc)
    bad = np.flatnonzero(clear & ~same)
    assert bad.size == 0, f"{bad.size} chains with clear margins differ, e.g. chain {bad[:5]}, margins {margin[bad[:5]]}"
    return int((~same).sum())


CASES = [  # (config, chains, rule, transitions)
    (1, 512, "local", 50), (1, 512, "exchange", 50), (2, 256, "exchange", 200), (2, 200, "local", 130),
    (3, 64, "local", 400), (4, 96, "exchange", 200), (4, 40, "local", 100), (5, 40, "exchange", 96),
]


@pytest.mark.parametrize("cfg,n,rule,steps", CASES)
def test_sampler_parity_configs(nk, cfg, n, rule, steps):
    p = inp.make_config(cfg, n_samples=n)
    r = nk.NK_RULE_LOCAL if rule == "local" else nk.NK_RULE_EXCHANGE
    got, gacc, ref, racc, margin = run_both(nk, p, r, steps)
    n_diff = assert_chains(p, r, got, gacc, ref, racc, margin)
    assert 0 < racc.mean() <= steps
    print(f"cfg {cfg} {rule}: acceptance {racc.mean() / steps:.3f}, {n_diff} of {n} chains took a borderline branch")


def test_sampler_larger_parameters(nk):
    """x5 parameters: peaked |psi|^2, low acceptance, |theta| of a trained state (Q17)."""
    p = inp.make_config(2, n_samples=128)
    p.W, p.a, p.b = (x * np.float32(5.0) for x in (p.W, p.a, p.b))
    for r in (nk.NK_RULE_LOCAL, nk.NK_RULE_EXCHANGE):
        got, gacc, ref, racc, margin = run_both(nk, p, r, 150)
        assert_chains(p, r, got, gacc, ref, racc, margin)
        assert racc.mean() < 150


def test_chunking_offsets_and_determinism(nk):
    p = inp.make_config(2, n_samples=100)
    r = nk.NK_RULE_EXCHANGE
    W, a, b = dev(p.W), dev(p.a), dev(p.b)

    def run(sig0, **kw):
        s = dev(sig0)
        acc = nk.metropolis_sample(s, W, a, b, rule=r, clusters=p.bonds, **kw)
        torch.cuda.synchronize()
        return s.cpu().numpy(), acc.cpu().numpy()

    full, acc_full = run(p.sigma, n_steps=150, seed=11)
    again, acc_again = run(p.sigma, n_steps=150, seed=11)
    assert np.array_equal(full, again) and np.array_equal(acc_full, acc_again)          # deterministic
    for chunk in (64, 33, 1):
        c, ac = run(p.sigma, n_steps=150, seed=11, chunk_size=chunk)
        assert np.array_equal(c, full) and np.array_equal(ac, acc_full)                 # chunk-independent
    part, acc_part = run(p.sigma[37:], n_steps=150, seed=11, chain_offset=37)
    assert np.array_equal(part, full[37:]) and np.array_equal(acc_part, acc_full[37:])  # shardable
    other, _ = run(p.sigma, n_steps=150, seed=12)
    assert not np.array_equal(other, full)
    # two calls continue one stream; theta is re-contracted in between, so allow borderline chains only
    h1, a1 = run(p.sigma, n_steps=70, seed=11)
    h2, a2 = run(h1, n_steps=80, seed=11, step_offset=70)
    same = np.all(h2 == full, axis=1) & (a1 + a2 == acc_full)
    assert same.mean() > 0.9


def test_sampler_edge_cases(nk):
    p = inp.make_problem(inp.KIND_HEISENBERG, "chain", 7, 5, 3, seed=3, sz0=False)   # N = 7, M = 5, B = 3
    for r, steps in ((nk.NK_RULE_LOCAL, 1), (nk.NK_RULE_LOCAL, 33), (nk.NK_RULE_EXCHANGE, 64), (nk.NK_RULE_LOCAL, 0)):
        got, gacc, ref, racc, margin = run_both(nk, p, r, steps, a=(steps != 33), b=(steps != 64))
        assert_chains(p, r, got, gacc, ref, racc, margin, min_clear=0.0)
    # empty batch, and a uniform state (W = 0): every proposal accepted
    W, a, b = dev(p.W), dev(p.a), dev(p.b)
    acc = nk.metropolis_sample(torch.empty((0, 7), dtype=torch.int8, device="cuda"), W, a, b, n_steps=5)
    assert acc.numel() == 0
    s = dev(p.sigma)
    acc = nk.metropolis_sample(s, torch.zeros_like(W), None, b, n_steps=40, seed=5)
    assert torch.all(acc == 40)


def test_sampler_argument_errors(nk):
    p = inp.make_config(1, n_samples=4)
    s, W = dev(p.sigma), dev(p.W)
    with pytest.raises(nk.NkError):
        nk.metropolis_sample(s, W, rule=nk.NK_RULE_EXCHANGE, clusters=None)
    with pytest.raises(nk.NkError):
        nk.metropolis_sample(s, W, rule=nk.NK_RULE_EXCHANGE, clusters=np.array([[0, 10]]))
    with pytest.raises(nk.NkError):
        nk.metropolis_sample(s, W, rule=5)
    with pytest.raises(nk.NkError):
        nk.metropolis_sample(s, W, n_steps=-1)


def test_sampled_energy_matches_exact_expectation(nk):
    """End to end on a 10-site ring: chains equilibrated on the GPU give a mean local energy (GPU) equal, within
    the Monte Carlo error, to <psi|H|psi>/<psi|psi> over the enumerated S^z = 0 sector (Eq. (11), Eq. (17))."""
    from oracle import nk_oracle as orc
    p = inp.make_config(1, n_samples=16384)
    op = nk.Operator.from_problem(p)
    sig, W, a, b = dev(p.sigma), dev(p.W), dev(p.a), dev(p.b)
    nk.metropolis_sample(sig, W, a, b, rule=nk.NK_RULE_EXCHANGE, clusters=p.bonds, n_steps=40 * p.n_sites, seed=3)
    eloc, _, stats = nk.local_energy(op, sig, W, a, b)
    torch.cuda.synchronize()
    k = np.arange(2 ** p.n_sites)[:, None]
    states = (1 - 2 * ((k >> np.arange(p.n_sites)[None, :]) & 1)).astype(np.int8)
    sector = states[states.sum(axis=1) == 0]
    e_all, lp_all = orc.local_energy(p.kind, sector, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    w = np.exp(2 * lp_all.real)
    exact = float((w * e_all).sum() / w.sum())
    var = float((w * (e_all - exact) ** 2).sum() / w.sum())
    mean = stats[0].item()
    assert abs(mean - exact) < 5 * np.sqrt(var / p.n_samples), (mean, exact)
    op.close()


def test_sampler_long_chain_and_widest_rbm(nk):
    """N = 3000 (94 words of spin bits per chain in shared memory) with both rules; M = 2048 on a small lattice (8 KB
    rows: the staged-row path) with an odd number of transitions."""
    p = inp.make_problem(inp.KIND_HEISENBERG, "chain", 3000, 128, 20, seed=6, scale=0.02)
    for r in (nk.NK_RULE_LOCAL, nk.NK_RULE_EXCHANGE):
        got, gacc, ref, racc, margin = run_both(nk, p, r, 70)
        assert_chains(p, r, got, gacc, ref, racc, margin, min_clear=0.7)
    p = inp.make_problem(inp.KIND_HEISENBERG, "chain", 16, 2048, 30, seed=7, scale=0.01)
    for r in (nk.NK_RULE_LOCAL, nk.NK_RULE_EXCHANGE):
        got, gacc, ref, racc, margin = run_both(nk, p, r, 77)
        assert_chains(p, r, got, gacc, ref, racc, margin, min_clear=0.7)
    # the limits of this version: M = 4096 real, M = 2048 complex (the 8-warp variants, rows read straight from L2)
    for kw in (dict(n_hidden=4096), dict(n_hidden=2048, complex_params=True)):
        p = inp.make_problem(inp.KIND_HEISENBERG, "chain", 16, kw.pop("n_hidden"), 30, seed=8, scale=0.01, **kw)
        for r in (nk.NK_RULE_LOCAL, nk.NK_RULE_EXCHANGE):
            got, gacc, ref, racc, margin = run_both(nk, p, r, 45)
            assert_chains(p, r, got, gacc, ref, racc, margin, min_clear=0.7)

"""GPU parity of nk_energy_gradient against the float64 oracle.

Tolerance: every entry of the gradient is a sum over B samples of terms v = conj(tanh theta) (E - mean) / B;
the kernel evaluates v in fp32 (relative error ~1e-7), splits it on fixed-point grids with residual < 2^-24 V
(V = max|v| of the chunk for complex parameters, its bound max_s |2 w_s| for real ones) and accumulates exactly per chunk, so |g_gpu - g_ref| <= 4e-7 * sum_s |v_s|  (+ one fp32 ulp of the output).  The
test uses the bound 1e-6 * B * max|v| >= that, evaluated from the oracle's own terms.
"""
import numpy as np
import pytest
import torch

from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp

pytestmark = pytest.mark.gpu
DEV = "cuda"


def dev(x):
    return None if x is None else torch.from_numpy(np.ascontiguousarray(x)).to(DEV)


def oracle_inputs(p):
    """E_loc from the oracle, rounded to the fp32 the C ABI takes, and its fp64 statistics."""
    e_ref, _ = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    e32 = e_ref.astype(np.complex64 if p.complex_params else np.float32)
    return e32, np.array(orc.stats(e32.astype(np.complex128 if p.complex_params else np.float64)))


def check(nk, p, e32, st, chunk):
    ga, gb, gW = nk.energy_gradient(dev(p.sigma), dev(p.W), dev(p.b), dev(e32), dev(st), chunk_size=chunk)
    torch.cuda.synchronize()
    ra, rb, rW = orc.energy_gradient_batched(p.sigma, p.W, p.b, e32)
    B = p.n_samples
    de = np.abs(e32.astype(np.complex128) - e32.astype(np.complex128).mean()).max() / B
    bound = 1e-6 * B * de * (1 if p.complex_params else 2)          # |tanh|, |sigma| <= ~1 (|tanh z| can exceed 1 slightly)
    worst = 0.0
    for name, g, r in (("a", ga, ra), ("b", gb, rb), ("W", gW, rW)):
        g = g.cpu().numpy().astype(r.dtype)
        err = np.abs(g - r).max()
        assert err <= bound + 2e-7 * np.abs(r).max(), f"grad_{name}: err {err}, bound {bound}, scale {np.abs(r).max()}"
        worst = max(worst, err / max(np.abs(r).max(), np.finfo(np.float64).tiny))   # B = 1: the gradient is exactly 0
    return worst


@pytest.mark.parametrize("cfg,n,chunk", [(1, 1024, 0), (2, 700, 256), (3, 96, 0), (4, 300, 128), (5, 40, 0)])
def test_gradient_parity_configs(nk, cfg, n, chunk):
    p = inp.make_config(cfg, n_samples=n)
    e32, st = oracle_inputs(p)
    worst = check(nk, p, e32, st, chunk)
    print(f"cfg{cfg}: max gradient error / max|g| = {worst:.2e}")


@pytest.mark.parametrize("chunk", [0, 16384])
def test_gradient_full_batch_config5(nk, chunk):
    """All 65536 samples of config 5 in the launch configuration bench.py times (the whole batch as one chunk) and in
    four chunks, against the float64 oracle on the same inputs.  The local energies are an INPUT of this call: seeded
    normal numbers with the mean and spread of config 5's (they need not come from any local-energy routine)."""
    p = inp.make_config(5)
    rng = np.random.default_rng(77)
    e32 = (-2197.8 + 4.6 * rng.standard_normal(p.n_samples)).astype(np.float32)
    st = np.array(orc.stats(e32.astype(np.float64)))
    worst = check(nk, p, e32, st, chunk)
    print(f"cfg5 full batch, chunk {chunk}: max gradient error / max|g| = {worst:.2e}")


@pytest.mark.parametrize("case", [
    dict(kind=0, lattice="chain", L=4, M=1, B=1),
    dict(kind=1, lattice="chain", L=7, M=5, B=31, h=0.8),
    dict(kind=0, lattice="square", L=4, M=130, B=77, order=2, J=(1.0, 0.5)),
    dict(kind=1, lattice="square", L=4, M=129, B=65, h=1.1, complex_params=True),
    dict(kind=0, lattice="square", L=6, M=300, B=200, complex_params=True),
    dict(kind=0, lattice="chain", L=16, M=40, B=300, scale=1e-3),     # |tanh theta| ~ 1e-3: far below the scale bound
    dict(kind=0, lattice="chain", L=16, M=4096, B=150, scale=0.02),   # the width limit of this version, real
    dict(kind=0, lattice="chain", L=16, M=2048, B=150, scale=0.02, complex_params=True),   # ... and complex
])
def test_gradient_edge_cases(nk, case):
    case = dict(case)
    # complex tanh has poles where cosh(theta) = 0 (Re theta = 0, Im theta = pi/2): keep complex |theta| well below
    # them, as the five configs do (Q18) -- otherwise |O_b| is unbounded and so is the error bound
    scale = case.pop("scale", 0.05 if case.get("complex_params") else 0.15)
    p = inp.make_problem(case.pop("kind"), case.pop("lattice"), case.pop("L"), case.pop("M"), case.pop("B"),
                         seed=44, scale=scale, **case)
    e32, st = oracle_inputs(p)
    check(nk, p, e32, st, 0)
    if p.n_samples > 64:
        check(nk, p, e32, st, 64)                       # ragged last chunk


def test_gradient_is_reproducible_and_chunk_consistent(nk):
    p = inp.make_config(2, n_samples=1000)
    e32, st = oracle_inputs(p)
    args = (dev(p.sigma), dev(p.W), dev(p.b), dev(e32), dev(st))
    g1 = [t.cpu().numpy() for t in nk.energy_gradient(*args, chunk_size=0)]
    g2 = [t.cpu().numpy() for t in nk.energy_gradient(*args, chunk_size=0)]
    g3 = [t.cpu().numpy() for t in nk.energy_gradient(*args, chunk_size=192)]
    for x, y, z in zip(g1, g2, g3):
        assert np.array_equal(x, y)                                   # bit-reproducible
        # chunking changes the fp32 rounding order and the per-chunk fixed-point grid of the 24-bit split of v
        np.testing.assert_allclose(z, x, rtol=0, atol=1e-6 * np.abs(x).max())


def test_gradient_end_to_end_from_gpu_local_energies(nk):
    """local_energy -> energy_gradient entirely on the GPU, against the oracle run on its own E_loc."""
    p = inp.make_config(4, n_samples=512)
    op = nk.Operator.from_problem(p)
    sig, W, a, b = dev(p.sigma), dev(p.W), dev(p.a), dev(p.b)
    e, _, st = nk.local_energy(op, sig, W, a, b)
    ga, gb, gW = nk.energy_gradient(sig, W, b, e, st)
    torch.cuda.synchronize()
    e_ref, _ = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    ra, rb, rW = orc.energy_gradient_batched(p.sigma, p.W, p.b, e_ref)
    for g, r in ((ga, ra), (gb, rb), (gW, rW)):
        err = np.abs(g.cpu().numpy().astype(r.dtype) - r).max()
        assert err <= 1e-4 * np.abs(r).max(), (err, np.abs(r).max())     # E_loc itself carries 1e-4 relative


def test_gradient_argument_errors(nk):
    p = inp.make_problem(0, "chain", 6, 4, 8, seed=1)
    lib = nk.load()
    assert lib.nk_energy_gradient(None, 8, 6, 4, 0, None, None, None, None, 0, None, None, None, None, 0, None) == -1
    assert lib.nk_energy_gradient_workspace_bytes(8, 6, 4, 3, 0) == 0
    e32, st = oracle_inputs(p)
    with pytest.raises(nk.NkError):
        nk.energy_gradient(dev(p.sigma), dev(p.W), dev(p.b), dev(e32[:4]), dev(st))


@pytest.mark.parametrize("cfg,n", [(2, 700), (4, 300)])
def test_gradient_of_shards_sums_to_the_gradient_of_the_union(nk, cfg, n):
    """nk_energy_gradient_sharded: unequal shards, each with the statistics of the
    WHOLE batch and n_global = B, return shares that add up to the single-rank gradient."""
    p = inp.make_config(cfg, n_samples=n)
    e32, st = oracle_inputs(p)
    full = nk.energy_gradient(dev(p.sigma), dev(p.W), dev(p.b), dev(e32), dev(st))
    cut = n // 3
    parts = []
    for sl in (slice(0, cut), slice(cut, n)):
        parts.append(nk.energy_gradient(dev(p.sigma[sl]), dev(p.W), dev(p.b), dev(e32[sl]), dev(st), n_global=n))
    torch.cuda.synchronize()
    ra, rb, rW = orc.energy_gradient_batched(p.sigma, p.W, p.b, e32)
    for g_full, g0, g1, r in zip(full, parts[0], parts[1], (ra, rb, rW)):
        tot = (g0 + g1).cpu().numpy()
        scale = np.abs(r).max()
        assert np.abs(tot - g_full.cpu().numpy()).max() <= 2e-6 * scale     # three fp32 roundings, three scales
        assert np.abs(tot.astype(r.dtype) - r).max() <= 2e-6 * scale


def test_gradient_non_finite_local_energy_propagates(nk):
    """DESIGN.md Q14: a NaN local energy (a diverged optimisation) must not come back as silent zeros from the
    fixed-point tensor-core contraction — every block of the gradient is non-finite."""
    for cfg, n in ((2, 300), (4, 200)):
        p = inp.make_config(cfg, n_samples=n)
        e32, _ = oracle_inputs(p)
        e32 = e32.copy()
        e32[5] = np.nan
        st = np.array([np.nan, np.nan if p.complex_params else 0.0, np.nan, float(n)])
        ga, gb, gW = nk.energy_gradient(dev(p.sigma), dev(p.W), dev(p.b), dev(e32), dev(st))
        torch.cuda.synchronize()
        for g in (ga, gb, gW):
            assert not np.isfinite(torch.view_as_real(g).cpu().numpy() if g.is_complex() else g.cpu().numpy()).any()

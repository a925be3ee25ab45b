"""GPU parity of the tensor-core series form of the local energy (nk_local_energy_ex with NK_FORM_SERIES, and the
automatic choice when its gate opens; paper_2112_10526_b200/csrc/series_tc.cu) against the float64 oracles:
the from-scratch one on sample subsets and the incremental one (oracle/nk_incremental.c, pinned to the from-scratch
one in test_oracle_incremental.py) on whole batches.  Same tolerance as every other form: |dE| <= 1e-4 |E| + 1e-6
(Eq. (12); BASELINE.json north_star)."""
import numpy as np
import pytest
import torch

from oracle import nk_incremental as inc
from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp
from test_gpu_parity import assert_eloc, assert_logpsi, dev, run_oracle

pytestmark = pytest.mark.gpu


def run_form(nk, p, form, chunk=None, flags=0, a=True, b=True):
    op = nk.Operator.from_problem(p, flags)
    plan = nk.LocalEnergyPlan(op, p.sigma.shape[0], p.n_sites, p.n_hidden, nk.NK_F32,
                              p.chunk_size if chunk is None else chunk, flags=form)
    e, lp, st = plan.run(dev(p.sigma), dev(p.W), dev(p.a) if a else None, dev(p.b) if b else None)
    torch.cuda.synchronize()
    out = e.cpu().numpy(), lp.cpu().numpy(), st.cpu().numpy()
    took = plan.form() if form in (0, nk.NK_FORM_SERIES) else (form, None)
    terms = getattr(plan, "series_terms", 0)
    op.close()
    return out, took[0], terms


@pytest.mark.parametrize("cfg,n", [(5, 47), (3, 96), (5, 300)])
def test_series_form_parity_forced(nk, cfg, n):
    p = inp.make_config(cfg, n_samples=n)
    (e, lp, st), form, terms = run_form(nk, p, nk.NK_FORM_SERIES, chunk=0)
    assert form == nk.NK_FORM_SERIES and 2 <= terms <= 6
    e_ref, lp_ref = (run_oracle(p) if n <= 100 else
                     inc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b))
    worst = assert_eloc(e, e_ref)
    assert_logpsi(lp, lp_ref)
    m = orc.stats(e_ref)
    assert abs(st[0] - m[0]) <= 1e-4 * abs(m[0]) + 1e-6 and st[3] == n
    print(f"cfg{cfg} series form (K = {terms}): max rel err E_loc {worst:.2e}")


def test_series_gate_automatic_choice(nk):
    """Config 5 and config 3 meet the remainder bound (the automatic call takes the series form, and its result is
    bit-identical to the forced one); config 2 is below the size limits, and parameters x6 leave the bound unmet:
    the automatic call then takes a SIMT form and NK_FORM_SERIES is refused / still runs with K = 6."""
    for cfg, n, k_want in ((5, 64, 5), (3, 64, None)):
        p = inp.make_config(cfg, n_samples=n)
        (e_auto, _, _), form, terms = run_form(nk, p, 0)
        assert form == nk.NK_FORM_SERIES and (k_want is None or terms == k_want), (cfg, form, terms)
        (e_forced, _, _), _, terms2 = run_form(nk, p, nk.NK_FORM_SERIES)
        assert terms2 == terms and np.array_equal(e_auto, e_forced)
    p = inp.make_config(2, n_samples=64)
    _, form, terms = run_form(nk, p, 0)
    assert form != nk.NK_FORM_SERIES and terms == 0
    with pytest.raises(nk.NkError):
        run_form(nk, p, nk.NK_FORM_SERIES)
    p = inp.make_config(5, n_samples=40)
    p.W = (p.W * 6).astype(np.float32)
    (e_auto, _, _), form, terms = run_form(nk, p, 0)
    assert form != nk.NK_FORM_SERIES and terms == 0
    assert_eloc(e_auto, run_oracle(p)[0])


def test_series_ragged_sizes_chunks_and_flags(nk):
    """N = 144 (not a multiple of 128), M = 300 (M_pad = 384), 288 + 288 bonds in two colours (two column tiles, the
    second ragged), B = 333 in chunks of 100 (ragged sample tiles), Marshall sign, missing biases; TFIM 12 x 12."""
    p = inp.make_problem(inp.KIND_HEISENBERG, "square", 12, 300, 333, seed=11, order=2, J=(1.0, 0.5), scale=0.02)
    e_ref, lp_ref = inc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    outs = []
    for chunk in (0, 100, 128, 1):
        (e, lp, st), form, terms = run_form(nk, p, nk.NK_FORM_SERIES, chunk=chunk)
        assert form == nk.NK_FORM_SERIES
        assert_eloc(e, e_ref)
        assert_logpsi(lp, lp_ref)
        outs.append(e)
    for e in outs[1:]:
        assert np.array_equal(outs[0], e), "per-sample results must not depend on chunk_size"
    (e, _, _), _, _ = run_form(nk, p, nk.NK_FORM_SERIES, flags=nk.NK_FLAG_MARSHALL, a=False, b=False)
    assert_eloc(e, inc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, None, None,
                                    orc.FLAG_MARSHALL)[0])
    q = inp.make_problem(inp.KIND_ISING, "square", 12, 288, 200, seed=12, scale=0.03, h=1.3)
    (e, lp, _), form, _ = run_form(nk, q, nk.NK_FORM_SERIES, chunk=77)
    e_ref, lp_ref = inc.local_energy(q.kind, q.sigma, q.bonds, q.colors, q.J, q.h, q.W, q.a, q.b)
    assert form == nk.NK_FORM_SERIES
    assert_eloc(e, e_ref)
    assert_logpsi(lp, lp_ref)


def test_series_closed_forms(nk):
    """Uniform psi (W = 0, a = 0): E_loc = n_bonds J for every sample; W = 0, a != 0 through the oracle."""
    p = inp.make_config(5, n_samples=130)
    p.W = np.zeros_like(p.W); p.a = np.zeros_like(p.a)
    (e, _, _), form, terms = run_form(nk, p, 0)
    assert form == nk.NK_FORM_SERIES and terms == 2
    np.testing.assert_allclose(e, 2048.0, rtol=2e-6)
    p = inp.make_config(5, n_samples=40)
    p.W = np.zeros_like(p.W)
    (e, _, _), _, _ = run_form(nk, p, 0)
    assert_eloc(e, run_oracle(p)[0])


@pytest.fixture(scope="module")
def cfg5_full():
    """All 65536 samples of config 5 through the incremental float64 route (minutes of host time, once per module)."""
    p = inp.make_config(5)
    e_ref, lp_ref = inc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    return p, e_ref, lp_ref


@pytest.mark.parametrize("form_name", ["auto", "series", "product", "logcosh"])
def test_config5_full_batch_every_sample(nk, cfg5_full, form_name):
    """Every one of the 65536 local energies of config 5, in the chunked launch configuration bench.py times, against
    the incremental float64 route; all forms."""
    p, e_ref, lp_ref = cfg5_full
    form = {"auto": 0, "series": nk.NK_FORM_SERIES, "product": nk.NK_FORM_PRODUCT, "logcosh": nk.NK_FORM_LOGCOSH}[form_name]
    (e, lp, st), took, terms = run_form(nk, p, form)
    if form_name == "auto":
        assert took == nk.NK_FORM_SERIES and terms == 5
    worst = assert_eloc(e, e_ref)
    assert_logpsi(lp, lp_ref)
    m = orc.stats(e_ref)
    assert abs(st[0] - m[0]) <= 1e-4 * abs(m[0]) + 1e-6 and st[3] == p.n_samples
    assert abs(st[2] - m[2]) <= 1e-3 * m[2]
    print(f"config 5, all {p.n_samples} samples, {form_name}: max rel err E_loc {worst:.2e}")


def test_series_more_than_one_theta_window(nk):
    """theta is contracted once per WINDOW of groups (api.cu carve_eloc: as many groups as keep it under 1 GiB — 8 at
    config 5's width).  136072 samples of config 5 are nine groups of 16384 (the last one ragged) = two windows, the
    second holding one partial group; sampled rows of every region against the incremental oracle, the per-sample
    results bit-equal to those of a batch that fits one window, and the eager call bit-equal to the host-buffer call
    (which keeps one group per window)."""
    B = 8 * 16384 + 5000
    p = inp.make_config(5, n_samples=B)
    (e, lp, st), form, terms = run_form(nk, p, 0)
    assert form == nk.NK_FORM_SERIES and terms == 5 and st[3] == B
    rows = np.concatenate([np.arange(0, 24), np.arange(16384 - 12, 16384 + 12), np.arange(7 * 16384 - 8, 7 * 16384 + 8),
                           np.arange(8 * 16384 - 16, 8 * 16384 + 16), np.arange(B - 24, B)])
    e_ref, lp_ref = inc.local_energy(p.kind, p.sigma[rows], p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    assert_eloc(e[rows], e_ref)
    assert_logpsi(lp[rows], lp_ref)
    # the tail of the second window as a batch of its own (one window): per-sample results do not depend on the split
    q = inp.make_config(5, n_samples=16)
    q.sigma = p.sigma[8 * 16384: 8 * 16384 + 5000].copy()
    (e_tail, lp_tail, _), _, _ = run_form(nk, q, 0)
    assert np.array_equal(e_tail, e[8 * 16384:]) and np.array_equal(lp_tail, lp[8 * 16384:])
    m = orc.stats(e.astype(np.float64))
    assert abs(st[0] - m[0]) <= 1e-9 * abs(m[0]) and abs(st[2] - m[2]) <= 1e-9 * m[2]


@pytest.mark.parametrize("cfg,n,chunk", [(5, 700, 256), (2, 300, 128), (4, 200, 0)])
def test_plan_replay_equals_the_eager_call(nk, cfg, n, chunk):
    """nk_local_energy_plan_*: the captured graph replays the same kernels — bit-identical outputs, new CONTENTS of the
    bound buffers are picked up (the form is still chosen on the device), and the flag that synchronises is refused."""
    p = inp.make_config(cfg, n_samples=n)
    dt = nk.NK_C64 if p.complex_params else nk.NK_F32
    op = nk.Operator.from_problem(p)
    sig, W, a, b = dev(p.sigma), dev(p.W), dev(p.a), dev(p.b)
    plan = nk.LocalEnergyPlan(op, n, p.n_sites, p.n_hidden, dt, chunk)
    e0, lp0, st0 = (t.clone() for t in plan.run(sig, W, a, b))
    e1, lp1, st1 = (t.clone() for t in plan.run_graph(sig, W, a, b))
    torch.cuda.synchronize()
    assert torch.equal(e0, e1) and torch.equal(lp0, lp1) and torch.equal(st0, st1)
    scale = 6.0 if cfg == 5 else 1.5                   # same addresses, new parameters (config 5: the gate now closes)
    W.mul_(scale)
    e2, _, _ = (t.clone() for t in plan.run_graph(sig, W, a, b))
    e3, _, _ = (t.clone() for t in plan.run(sig, W, a, b))
    torch.cuda.synchronize()
    assert torch.equal(e2, e3) and not torch.equal(e2, e1)
    p.W = (p.W * scale).astype(p.W.dtype)
    rows = list(range(0, n, max(1, n // 24)))
    assert_eloc(e2.cpu().numpy()[rows], run_oracle(p, rows=rows)[0])
    bad = nk.LocalEnergyPlan(op, n, p.n_sites, p.n_hidden, dt, chunk, flags=nk.NK_CHECK_SPINS)
    with pytest.raises(nk.NkError):
        bad.run_graph(sig, W, a, b)
    plan.close_plan()
    op.close()


def test_series_wide_rbm_beyond_the_register_resident_limit(nk):
    """N = 256 (16 x 16), M = 4096 = the limit of this version (alpha = 16): the series form has no register-resident
    theta, the SIMT forms run their 8-warp variants; all three against the incremental oracle."""
    p = inp.make_problem(inp.KIND_HEISENBERG, "square", 16, 4096, 200, seed=21, scale=0.01)
    e_ref, lp_ref = inc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    for form in (0, nk.NK_FORM_SERIES, nk.NK_FORM_PRODUCT, nk.NK_FORM_LOGCOSH):
        (e, lp, st), took, terms = run_form(nk, p, form, chunk=128)
        assert_eloc(e, e_ref)
        assert_logpsi(lp, lp_ref)
        if form == 0:
            assert took == nk.NK_FORM_SERIES

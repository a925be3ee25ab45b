"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star; Q13):
    connected lists      bit-exact
    ln psi               |gpu - oracle| <= 1e-5 (fp32 output; Im compared modulo 2 pi) while |ln psi| < 128, which
                         covers the five configs (max 108); beyond that the spacing of the fp32 OUTPUT itself
                         exceeds 1e-5, so half an fp32 ulp of the reference is added (Q13)
    E_loc                |gpu - oracle| <= 1e-4 |oracle| + 1e-6
"""
import numpy as np
import pytest
import torch

from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp

pytestmark = pytest.mark.gpu
DEV = "cuda"

LOGPSI_ATOL = 1e-5
ELOC_RTOL, ELOC_ATOL = 1e-4, 1e-6


def dev(x):
    return None if x is None else torch.from_numpy(np.ascontiguousarray(x)).to(DEV)


# Every test of this module that goes through run_gpu runs twice: with flags = 0 (the automatic choice of the form of
# the amplitude ratios: the product form for these parameters when they are real, include/nkb200.h) and with the
# log-cosh form forced; tests/test_gpu_product_form.py forces the product form and checks the choice itself.
FORM = {"flags": 0}


@pytest.fixture(params=["auto", "logcosh"], autouse=True)
def _form(request, nk):
    FORM["flags"] = 0 if request.param == "auto" else nk.NK_FORM_LOGCOSH
    yield
    FORM["flags"] = 0


def run_gpu(nk, p, chunk=None, flags=0, a=True, b=True):
    op = nk.Operator.from_problem(p, flags)
    e, lp, st = nk.local_energy(op, dev(p.sigma), dev(p.W), dev(p.a) if a else None, dev(p.b) if b else None,
                                chunk_size=p.chunk_size if chunk is None else chunk, flags=FORM["flags"])
    torch.cuda.synchronize()
    out = e.cpu().numpy(), lp.cpu().numpy(), st.cpu().numpy()
    op.close()
    return out


def run_oracle(p, rows=None, flags=0, a=True, b=True):
    sig = p.sigma if rows is None else p.sigma[rows]
    return orc.local_energy(p.kind, sig, p.bonds, p.colors, p.J, p.h, p.W, p.a if a else None, p.b if b else None,
                            flags)


def assert_eloc(e_gpu, e_ref):
    e_gpu = np.asarray(e_gpu).astype(np.complex128)
    e_ref = np.asarray(e_ref).astype(np.complex128)
    err = np.abs(e_gpu - e_ref)
    tol = ELOC_RTOL * np.abs(e_ref) + ELOC_ATOL
    assert np.all(np.isfinite(e_gpu.view(np.float64)))
    worst = int(np.argmax(err - tol))
    assert np.all(err <= tol), f"E_loc mismatch at {worst}: gpu {e_gpu[worst]} oracle {e_ref[worst]}"
    return float(np.max(err / (np.abs(e_ref) + 1e-30)))


def assert_logpsi(lp_gpu, lp_ref, atol=LOGPSI_ATOL):
    lp_gpu = np.asarray(lp_gpu).astype(np.complex128)
    lp_ref = np.asarray(lp_ref).astype(np.complex128)
    dre = np.abs(lp_gpu.real - lp_ref.real)
    dim = np.abs((lp_gpu.imag - lp_ref.imag + np.pi) % (2 * np.pi) - np.pi)
    big = np.abs(lp_ref.real) >= 128.0
    tol_re = atol + np.where(big, 0.5 * np.spacing(np.abs(lp_ref.real).astype(np.float32)).astype(np.float64), 0.0)
    assert np.all(dre <= tol_re), f"Re ln psi err {dre.max()}"
    assert dim.max() <= atol, f"Im ln psi err {dim.max()} (mod 2 pi)"
    return float(max(dre.max(), dim.max()))


# ------------------------------------------------------------------ nk_connected: bit-exact
@pytest.mark.parametrize("cfg,n", [(1, 1024), (2, 96), (3, 24), (4, 64), (5, 6)])
def test_connected_bit_exact(nk, cfg, n):
    p = inp.make_config(cfg, n_samples=n)
    op = nk.Operator.from_problem(p)
    flips, mels, n_conn, sp = nk.connected(op, dev(p.sigma), materialize=True)
    torch.cuda.synchronize()
    flips, mels, n_conn, sp = (t.cpu().numpy() for t in (flips, mels, n_conn, sp))
    assert flips.shape == (n, p.max_conn, 2) and sp.shape == (n, p.max_conn, p.n_sites)
    for s in range(n):
        sp_r, mels_r, flips_r, nc_r = orc.connected(p.kind, p.sigma[s], p.bonds, p.colors, p.J, p.h)
        assert np.array_equal(sp[s], sp_r), f"sigma' differs for sample {s}"
        assert np.array_equal(flips[s], flips_r)
        assert np.array_equal(mels[s], mels_r.astype(np.float32))
        assert n_conn[s] == nc_r
    op.close()


def test_connected_marshall_and_coloured_couplings(nk):
    p = inp.make_problem(inp.KIND_HEISENBERG, "square", 4, 8, 37, seed=21, order=2, J=(0.75, -1.25))
    op = nk.Operator.from_problem(p, flags=nk.NK_FLAG_MARSHALL)
    flips, mels, n_conn, sp = nk.connected(op, dev(p.sigma), materialize=False)
    torch.cuda.synchronize()
    assert sp is None
    for s in range(37):
        _, mels_r, flips_r, nc_r = orc.connected(p.kind, p.sigma[s], p.bonds, p.colors, p.J, p.h, orc.FLAG_MARSHALL)
        assert np.array_equal(flips[s].cpu().numpy(), flips_r)
        assert np.array_equal(mels[s].cpu().numpy(), mels_r.astype(np.float32))
        assert int(n_conn[s]) == nc_r


# ------------------------------------------------------------------ nk_rbm_logpsi
@pytest.mark.parametrize("cfg,n", [(1, 1024), (2, 1024), (3, 512), (4, 1024), (5, 384)])
def test_logpsi_parity(nk, cfg, n):
    p = inp.make_config(cfg, n_samples=n)
    ref = orc.rbm_logpsi(p.sigma, p.W, p.a, p.b)
    lp32, theta = nk.rbm_logpsi(dev(p.sigma), dev(p.W), dev(p.a), dev(p.b), return_theta=True)
    lp64 = nk.rbm_logpsi(dev(p.sigma), dev(p.W), dev(p.a), dev(p.b), out_f64=True)
    torch.cuda.synchronize()
    e32 = assert_logpsi(lp32.cpu().numpy(), ref)
    e64 = assert_logpsi(lp64.cpu().numpy(), ref)
    th_ref = orc.rbm_theta(p.sigma, p.W, p.b)
    th_err = np.abs(theta.cpu().numpy().astype(th_ref.dtype) - th_ref).max()
    assert th_err < 2e-6, th_err
    print(f"cfg{cfg}: ln psi err fp32-out {e32:.2e}, f64-out {e64:.2e}, theta err {th_err:.2e}, |ln psi| max "
          f"{np.abs(ref).max():.1f}")


def test_logpsi_without_biases_and_tiny_shapes(nk):
    for (N, M, B, cplx) in [(3, 1, 1, False), (5, 7, 33, True), (17, 130, 9, False), (6, 129, 40, True)]:
        rng = np.random.default_rng(N * 100 + M)
        # complex ln cosh is ill-conditioned next to the zeros of cosh (x ~ 0, y ~ pi/2): keep |theta| moderate there
        W, a, b = inp.draw_params(rng, N, M, 0.2 if cplx else 0.5, cplx)
        sigma = inp.draw_samples(rng, B, N, False)
        lp = nk.rbm_logpsi(dev(sigma), dev(W), None, None, out_f64=True)
        torch.cuda.synchronize()
        assert_logpsi(lp.cpu().numpy(), orc.rbm_logpsi(sigma, W, None, None))
        lp = nk.rbm_logpsi(dev(sigma), dev(W), dev(a), None)
        assert_logpsi(lp.cpu().numpy(), orc.rbm_logpsi(sigma, W, a, None))


# ------------------------------------------------------------------ nk_local_energy: element-by-element
@pytest.mark.parametrize("cfg,n", [(1, 1024), (2, 512), (3, 96), (4, 160), (5, 47)])
def test_local_energy_parity(nk, cfg, n):
    p = inp.make_config(cfg, n_samples=n)
    e, lp, st = run_gpu(nk, p, chunk=0)
    e_ref, lp_ref = run_oracle(p)
    worst = assert_eloc(e, e_ref)
    lerr = assert_logpsi(lp, lp_ref)
    m = orc.stats(e_ref)
    assert abs(st[0] - m[0]) <= 1e-4 * abs(m[0]) + 1e-6 and abs(st[1] - m[1]) <= 1e-4 * abs(m[0]) + 1e-6
    assert abs(st[2] - m[2]) <= 1e-3 * m[2] + 1e-9 and st[3] == n
    # the statistics are exactly those of the returned E_loc (fp64 reduction)
    np.testing.assert_allclose(st[:3], orc.stats(e.astype(np.complex128))[:3], rtol=1e-12, atol=1e-12)
    print(f"cfg{cfg}: max rel err E_loc {worst:.2e}, ln psi {lerr:.2e}")


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_launch_configuration_sampled(nk, cfg):
    """BASELINE.json's full batch in the launch configuration bench.py times (config 5: 16 chunks of 4096);
    the oracle checks a fixed sample of outputs (first and last rows of several chunks)."""
    p = inp.make_config(cfg)
    e, lp, st = run_gpu(nk, p)
    B = p.n_samples
    chunk = p.chunk_size or B
    rows = sorted({c * chunk + o for c in range(0, B // chunk, max(1, B // chunk // 4)) for o in (0, chunk - 1)}
                  | {B - 1, B // 2 + 1})
    if cfg != 5:
        rows = sorted(set(rows) | set(range(17, B, B // 24)))
    e_ref, lp_ref = run_oracle(p, rows)
    assert_eloc(e[rows], e_ref)
    assert_logpsi(lp[rows], lp_ref)
    assert np.all(np.isfinite(e.view(np.float32))) and st[3] == B
    np.testing.assert_allclose(st[:3], orc.stats(e.astype(np.complex128))[:3], rtol=1e-11, atol=1e-11)
    # property that holds at any size: uniform psi => E_loc = sum_c J_c n_{b,c} (Heisenberg) / diag - h N (Ising)
    q = inp.make_config(cfg)
    q.W = np.zeros_like(q.W); q.a = np.zeros_like(q.a)
    e0, _, _ = run_gpu(nk, q)
    if q.kind == inp.KIND_HEISENBERG:
        expect = float(sum(q.J[c] for c in q.colors))
        np.testing.assert_allclose(e0.real, expect, rtol=2e-6)
    else:
        s = q.sigma.astype(np.float64)
        diag = (s[:, q.bonds[:, 0]] * s[:, q.bonds[:, 1]]).sum(axis=1) * q.J[0]
        np.testing.assert_allclose(e0, diag - q.h * q.n_sites, rtol=2e-6, atol=1e-3)
    if q.complex_params:
        assert np.abs(e0.imag).max() < 1e-3


def test_chunking_does_not_change_results(nk):
    p = inp.make_config(2, n_samples=1000)
    ref, lref, sref = run_gpu(nk, p, chunk=0)
    for chunk in (1000, 512, 333, 15, 1, 4096):
        e, lp, st = run_gpu(nk, p, chunk=chunk)
        assert np.array_equal(e, ref) and np.array_equal(lp, lref), f"chunk {chunk}"
        assert np.array_equal(st, sref)


# ------------------------------------------------------------------ edge and degenerate cases
@pytest.mark.parametrize("case", [
    dict(kind=0, lattice="chain", L=4, M=1, B=1),                      # smallest everything
    dict(kind=0, lattice="chain", L=6, M=3, B=16, sz0=False),          # outside the S^z=0 sector, incl. all-up rows
    dict(kind=1, lattice="chain", L=7, M=5, B=31, h=0.8),              # odd N, Ising, ragged batch
    dict(kind=1, lattice="square", L=3, M=130, B=29, h=3.0),           # M just above one 128-block
    dict(kind=0, lattice="square", L=4, M=257, B=77, order=2, J=(1.0, 0.5)),
    dict(kind=0, lattice="square", L=4, M=40, B=45, order=2, J=(0.3, -0.7), complex_params=True),
    dict(kind=1, lattice="square", L=4, M=129, B=20, h=1.1, complex_params=True),
    dict(kind=1, lattice="chain", L=5, M=4, B=8, h=0.0),               # no off-diagonal element at all
    dict(kind=0, lattice="square", L=6, M=640, B=33),                  # V = 5: one CTA per SM variant
    dict(kind=0, lattice="square", L=6, M=300, B=33, complex_params=True),
])
def test_edge_cases(nk, case):
    case = dict(case)
    p = inp.make_problem(case.pop("kind"), case.pop("lattice"), case.pop("L"), case.pop("M"), case.pop("B"),
                         seed=33, scale=0.2, **case)
    if p.name.startswith("chain6"):
        p.sigma[0] = 1; p.sigma[1] = -1                                # fully polarised rows: no active bond
    e, lp, _ = run_gpu(nk, p)
    e_ref, lp_ref = run_oracle(p)
    assert_eloc(e, e_ref)
    # real parameters: the north_star bound as it stands (the per-hidden-unit scales of the W split gave the margin
    # back).  Complex parameters keep the DESIGN.md Q18 carve-out: sigma_param = 0.2 puts theta next to the zeros of
    # cosh, where d ln cosh / d theta = tanh theta is unbounded and an fp32 theta error is amplified without limit
    assert_logpsi(lp, lp_ref, atol=3e-5 if p.complex_params else LOGPSI_ATOL)


def test_null_biases_marshall_flag_and_empty_batch(nk):
    p = inp.make_problem(inp.KIND_HEISENBERG, "square", 4, 24, 50, seed=5, scale=0.3)
    e, lp, _ = run_gpu(nk, p, a=False, b=False)
    e_ref, lp_ref = run_oracle(p, a=False, b=False)
    assert_eloc(e, e_ref); assert_logpsi(lp, lp_ref)
    e, _, _ = run_gpu(nk, p, flags=nk.NK_FLAG_MARSHALL)
    assert_eloc(e, run_oracle(p, flags=orc.FLAG_MARSHALL)[0])
    op = nk.Operator.from_problem(p)
    empty = torch.empty((0, p.n_sites), dtype=torch.int8, device=DEV)
    e, lp, st = nk.local_energy(op, empty, dev(p.W), dev(p.a), dev(p.b))
    torch.cuda.synchronize()
    assert e.numel() == 0 and st.cpu().tolist() == [0.0, 0.0, 0.0, 0.0]


def test_larger_parameters_stress(nk):
    """Trained states have larger |theta| (Q17): parameters x10, ratios spanning orders of magnitude."""
    p = inp.make_config(2, n_samples=200)
    p.W = (p.W * 10).astype(np.float32); p.a = (p.a * 10).astype(np.float32); p.b = (p.b * 10).astype(np.float32)
    e, lp, _ = run_gpu(nk, p)
    e_ref, lp_ref = run_oracle(p)
    assert_eloc(e, e_ref)
    # |theta| ~ 5 .. 8 here: theta is handed to the ln cosh pass as fp32, whose spacing there is 4.8e-7 (1e-7 at the five
    # configs), so the sum over hidden units carries ~1e-5 by itself — a limit of the fp32 theta buffer, not of the W
    # split; |ln psi| ~ 300 adds half an fp32 ulp of the output (assert_logpsi).  Measured 1.1e-5 + 1.5e-5.
    assert_logpsi(lp, lp_ref, atol=2e-5)


def test_host_entry_point_matches_device_entry_point(nk):
    p = inp.make_config(4, n_samples=300)
    e_d, lp_d, st_d = run_gpu(nk, p, chunk=128)
    op = nk.Operator.from_problem(p)
    e_h, lp_h, st_h = nk.local_energy_host(op, p.sigma, p.W, p.a, p.b, chunk_size=128)
    assert np.array_equal(e_h, e_d) and np.array_equal(lp_h, lp_d) and np.array_equal(st_h, st_d)


def test_errors_are_loud(nk):
    p = inp.make_problem(inp.KIND_HEISENBERG, "chain", 6, 4, 4, seed=1)
    op = nk.Operator.from_problem(p)
    with pytest.raises(nk.NkError, match="INVALID_ARG"):                 # N does not match the operator
        nk.local_energy(op, dev(np.ones((4, 8), np.int8)), dev(np.zeros((4, 8), np.float32)))
    big = inp.draw_params(np.random.default_rng(0), 6, 4097, 0.1, False)
    with pytest.raises(nk.NkError):                                      # M beyond the supported width
        nk.local_energy(op, dev(p.sigma), dev(big[0]), None, None)
    lib = nk.load()
    ws = torch.empty(1024, dtype=torch.uint8, device=DEV)
    out = torch.empty(4, dtype=torch.float32, device=DEV)
    rc = lib.nk_local_energy(op.handle, dev(p.sigma).data_ptr(), 4, 6, 4, 0, dev(p.W).data_ptr(), None, None, 0,
                             out.data_ptr(), None, None, ws.data_ptr() + 1, 1023, None)
    assert rc == -3                                                      # misaligned / short workspace
    bad = p.sigma.copy(); bad[2, 3] = 0                                  # opt-in spin validation
    with pytest.raises(nk.NkError, match="BAD_SPIN"):
        nk.local_energy(op, dev(bad), dev(p.W), dev(p.a), dev(p.b), flags=nk.NK_CHECK_SPINS)
    e_ok, _, _ = nk.local_energy(op, dev(p.sigma), dev(p.W), dev(p.a), dev(p.b), flags=nk.NK_CHECK_SPINS)
    e_ref, _ = run_oracle(p)
    assert_eloc(e_ok.cpu().numpy(), e_ref)


@pytest.mark.parametrize("case", [
    dict(kind=0, lattice="chain", L=3000, M=128, B=6),                       # N = 3000: 94 spin words, 3000 table rows
    dict(kind=1, lattice="chain", L=2100, M=100, B=5, h=0.9),                # long Ising chain, N + 1 = 2101 slots
    dict(kind=0, lattice="chain", L=16, M=2048, B=40),                       # widest 16-warp real RBM (V = 16) on a tiny lattice
    dict(kind=0, lattice="square", L=4, M=1024, B=40, complex_params=True),  # widest 16-warp complex RBM (V = 8)
    dict(kind=0, lattice="chain", L=16, M=4096, B=40),                       # the limit: V = 32, the 8-warp variants
    dict(kind=0, lattice="square", L=4, M=2048, B=40, complex_params=True),  # the limit, complex: V = 16
    dict(kind=0, lattice="chain", L=12, M=2900, B=33, scale=0.0),            # uniform psi at V = 23: every factor is 2
])
def test_maximum_sizes(nk, case):
    """The limits of this version (include/nkb200.h): M = 4096 real, M = 2048 complex (the 8-warp variants of the
    warp-per-sample kernels, with their running products rescaled half-way), and N well beyond the 1024 of config 5
    (several shared-memory words of spins per lane, thousands of table rows), both SIMT forms of the kernel."""
    case = dict(case)
    scale = case.pop("scale", 0.02)
    p = inp.make_problem(case.pop("kind"), case.pop("lattice"), case.pop("L"), case.pop("M"), case.pop("B"),
                         seed=44, scale=scale, **case)
    e_ref, lp_ref = run_oracle(p)
    e, lp, _ = run_gpu(nk, p)
    assert_eloc(e, e_ref)
    assert_logpsi(lp, lp_ref)
    op = nk.Operator.from_problem(p)
    for form in (nk.NK_FORM_PRODUCT, nk.NK_FORM_LOGCOSH):
        e2, _, _ = nk.local_energy(op, dev(p.sigma), dev(p.W), dev(p.a), dev(p.b), flags=form)
        assert_eloc(e2.cpu().numpy(), e_ref)
    op.close()


def test_theta_fixed_point_split_at_the_top_of_a_binade(nk):
    """max|W| just below a power of two (mantissa 0.99999): the int8 split of the contraction must step its scale up
    instead of overflowing the top digit, and theta must still carry fp32-level accuracy."""
    p = inp.make_config(2, n_samples=64)
    W = p.W.copy()
    W[3, 5] = np.nextafter(np.float32(0.25), np.float32(0))             # 0.99999994 * 2^-2, the largest entry
    W[7, 11] = -np.nextafter(np.float32(0.25), np.float32(0))
    assert np.abs(W).max() == np.abs(W[3, 5])
    lp, theta = nk.rbm_logpsi(dev(p.sigma), dev(W), dev(p.a), dev(p.b), out_f64=True, return_theta=True)
    torch.cuda.synchronize()
    th_ref = orc.rbm_theta(p.sigma, W, p.b)
    assert np.abs(theta.cpu().numpy() - th_ref).max() < 2e-6           # an overflowed digit would be an error of order 1
    assert_logpsi(lp.cpu().numpy(), orc.rbm_logpsi(p.sigma, W, p.a, p.b))


def test_cuda_graph_replay_matches_the_eager_call(nk):
    """LocalEnergyPlan.run_graph: the captured call replays bit-identically, and follows changed CONTENTS of the same
    tensors (new parameters, new samples) as a VMC loop needs."""
    p = inp.make_config(2, n_samples=512)
    op = nk.Operator.from_problem(p)
    sig, W, a, b = dev(p.sigma), dev(p.W), dev(p.a), dev(p.b)
    plan = nk.LocalEnergyPlan(op, 512, p.n_sites, p.n_hidden, nk.NK_F32, 128)
    e0 = [t.clone() for t in plan.run(sig, W, a, b)]
    e1 = [t.clone() for t in plan.run_graph(sig, W, a, b)]
    e2 = [t.clone() for t in plan.run_graph(sig, W, a, b)]
    torch.cuda.synchronize()
    assert all(torch.equal(x, y) and torch.equal(x, z) for x, y, z in zip(e0, e1, e2))
    W.mul_(1.5); sig.copy_(dev(p.sigma[::-1].copy()))
    g = [t.clone() for t in plan.run_graph(sig, W, a, b)]
    r = [t.clone() for t in plan.run(sig, W, a, b)]
    torch.cuda.synchronize()
    assert all(torch.equal(x, y) for x, y in zip(g, r)) and not torch.equal(g[0], e0[0])
    op.close()


def test_non_finite_parameters_propagate(nk):
    """DESIGN.md Q14: no clamping — a NaN or Inf in W reaches theta, ln psi and E_loc on the tensor-core path (the
    fixed-point split poisons the row's scale instead of saturating its digits)."""
    p = inp.make_config(2, n_samples=64)
    for bad in (np.nan, np.inf):
        W = p.W.copy()
        W[3, 7] = bad
        lp, theta = nk.rbm_logpsi(dev(p.sigma), dev(W), dev(p.a), dev(p.b), return_theta=True)
        torch.cuda.synchronize()
        th = theta.cpu().numpy()
        assert not np.isfinite(th[:, 3]).any() and np.isfinite(np.delete(th, 3, axis=1)).all()
        assert not np.isfinite(lp.cpu().numpy()).any()
        op = nk.Operator.from_problem(p)
        e, lp2, st = nk.local_energy(op, dev(p.sigma), dev(W), dev(p.a), dev(p.b))
        torch.cuda.synchronize()
        assert not np.isfinite(e.cpu().numpy()).any() and not np.isfinite(lp2.cpu().numpy()).any()
        assert not np.isfinite(st.cpu().numpy()[0])
        op.close()


def test_complex_large_imaginary_theta(nk):
    """Im b shifted by whole multiples of 2 pi (|Im theta| up to ~13, as in trained sign structures): the fused kernel's
    fast sincos sees range-reduced arguments (rbm_lane_state.cuh wrap_pi), so E_loc keeps its bound; ln psi mod 2 pi
    likewise.  cosh is 2 pi i-periodic, so the conditioning of the problem is that of config 4 itself."""
    p = inp.make_config(4, n_samples=96)
    rng = np.random.default_rng(5)
    shift = (2 * np.pi * rng.integers(-2, 3, size=p.b.shape)).astype(np.float32)
    p.b = (p.b + 1j * shift).astype(np.complex64)
    e, lp, _ = run_gpu(nk, p)
    e_ref, lp_ref = run_oracle(p)
    assert_eloc(e, e_ref)
    assert_logpsi(lp, lp_ref, atol=3e-5)

"""GPU parity of nk_qgt_matvec against the float64 oracle's three-step product (Eq. (75)).

Tolerance: every output entry is a sum over B samples of terms conj(O_s) (w_s - <w>) / B with |O| <= ~1; the kernel
evaluates tanh(theta), w and the terms in fp32 (relative error ~1e-7 each) and contracts them exactly, so
|out_gpu - out_ref| <= 1e-6 * max_s |w_s - <w>|  (+ 2e-7 of the output scale), the bound of tests/test_gpu_gradient.py.
"""
import numpy as np
import pytest
import torch

from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp

pytestmark = pytest.mark.gpu


def dev(x):
    return None if x is None else torch.from_numpy(np.ascontiguousarray(x)).cuda()


def draw_v(p, seed):
    rng = np.random.default_rng(seed)
    def d(*sh):
        x = rng.standard_normal(sh)
        if p.complex_params:
            return (x + 1j * rng.standard_normal(sh)).astype(np.complex64)
        return x.astype(np.float32)
    return d(p.n_sites), d(p.n_hidden), d(p.n_hidden, p.n_sites)


def check(nk, p, v, shift, chunk, use_a=True, use_b=True):
    va, vb, vW = v
    out = nk.qgt_matvec(dev(p.sigma), dev(p.W), dev(p.b), dev(va) if use_a else None, dev(vb) if use_b else None,
                        dev(vW), diag_shift=shift, chunk_size=chunk)
    torch.cuda.synchronize()
    za, zb = np.zeros_like(va), np.zeros_like(vb)
    ref = orc.qgt_matvec(p.sigma, p.W, p.b, va if use_a else za, vb if use_b else zb, vW, shift)
    J = orc.rbm_jacobian(p.sigma, p.W, p.b)
    w = J @ orc.pack_params(va if use_a else za, vb if use_b else zb, vW).astype(J.dtype)
    bound = 1e-6 * np.abs(w - w.mean()).max()
    worst = 0.0
    for name, g, r, vv, used in (("a", out[0], ref[0], va, use_a), ("b", out[1], ref[1], vb, use_b),
                                 ("W", out[2], ref[2], vW, True)):
        g = g.cpu().numpy().astype(r.dtype)
        if not used:
            r = r - 0.0                                  # shift * 0
        scale = np.abs(r).max()
        err = np.abs(g - r).max()
        assert err <= bound + 2e-7 * scale + 1e-7 * shift * np.abs(vv).max(), f"out_{name}: err {err}, bound {bound}"
        worst = max(worst, err / scale)
    return worst


@pytest.mark.parametrize("cfg,n,chunk", [(1, 1024, 0), (2, 500, 128), (3, 64, 0), (4, 160, 64), (5, 12, 0)])
def test_qgt_matvec_parity_configs(nk, cfg, n, chunk):
    p = inp.make_config(cfg, n_samples=n)
    worst = check(nk, p, draw_v(p, 40 + cfg), 0.01, chunk)
    print(f"cfg{cfg}: max QGT-vector error / max|out| = {worst:.2e}")


@pytest.mark.parametrize("chunk", [0, 16384])
def test_qgt_matvec_full_batch_config5(nk, chunk):
    """All 65536 samples of config 5 (the launch configuration bench.py times, and four chunks) against the oracle's
    Jacobian-free route `qgt_matvec_batched` (pinned to the dense covariance matrix in tests/test_oracle_qgt.py)."""
    p = inp.make_config(5)
    rng = np.random.default_rng(91)
    va = rng.standard_normal(p.n_sites).astype(np.float32)
    vb = rng.standard_normal(p.n_hidden).astype(np.float32)
    vW = rng.standard_normal((p.n_hidden, p.n_sites)).astype(np.float32)
    out = nk.qgt_matvec(dev(p.sigma), dev(p.W), dev(p.b), dev(va), dev(vb), dev(vW), diag_shift=0.01, chunk_size=chunk)
    torch.cuda.synchronize()
    ra, rb, rW, Jv = orc.qgt_matvec_batched(p.sigma, p.W, p.b, va, vb, vW, 0.01, return_w=True)
    bound = 1e-6 * np.abs(Jv - Jv.mean()).max()                         # as in check(): the scale of the sample weights
    for name, g, r, vv in (("a", out[0], ra, va), ("b", out[1], rb, vb), ("W", out[2], rW, vW)):
        err = np.abs(g.cpu().numpy().astype(np.float64) - r).max()
        assert err <= bound + 2e-7 * np.abs(r).max() + 1e-9 * np.abs(vv).max(), f"out_{name}: err {err}, bound {bound}"
        print(f"cfg5 full batch chunk {chunk} out_{name}: err / max|out| = {err / np.abs(r).max():.2e}")


def test_qgt_matvec_at_the_width_limit(nk):
    """M = 4096 real / 2048 complex (include/nkb200.h): the contractions are size-generic, only the limit moved."""
    for kw in (dict(M=4096), dict(M=2048, complex_params=True)):
        p = inp.make_problem(inp.KIND_HEISENBERG, "chain", 16, kw.pop("M"), 120, seed=9, scale=0.02, **kw)
        check(nk, p, draw_v(p, 77), 0.01, 64)


def test_qgt_matvec_properties(nk):
    p = inp.make_config(2, n_samples=256)
    v, u = draw_v(p, 1), draw_v(p, 2)
    sig, W, b = dev(p.sigma), dev(p.W), dev(p.b)
    Gv = [t.cpu().numpy().astype(np.float64) for t in nk.qgt_matvec(sig, W, b, *map(dev, v))]
    Gu = [t.cpu().numpy().astype(np.float64) for t in nk.qgt_matvec(sig, W, b, *map(dev, u))]
    dot = lambda x, y: sum(float(np.vdot(a_, b_)) for a_, b_ in zip(x, y))
    assert abs(dot(u, Gv) - dot(Gu, v)) < 1e-4 * abs(dot(u, Gv))          # symmetric
    assert dot(v, Gv) > 0                                                 # positive semi-definite
    # NULL blocks, missing outputs, zero shift; chunking is bit-reproducible per chunk size
    check(nk, p, v, 0.0, 100, use_a=False, use_b=False)
    o1 = nk.qgt_matvec(sig, W, b, *map(dev, v), diag_shift=0.1, chunk_size=64)
    o2 = nk.qgt_matvec(sig, W, b, *map(dev, v), diag_shift=0.1, chunk_size=64)
    assert all(torch.equal(x, y) for x, y in zip(o1, o2))
    # a direction with constant O over the batch is annihilated: all samples identical
    same = dev(np.tile(p.sigma[:1], (64, 1)))
    z = nk.qgt_matvec(same, W, b, *map(dev, v))
    assert max(float(t.abs().max()) for t in z) < 1e-5


def test_qgt_matvec_complex_tiny_and_errors(nk):
    p = inp.make_problem(inp.KIND_HEISENBERG, "chain", 7, 5, 33, seed=3, sz0=False, complex_params=True)
    check(nk, p, draw_v(p, 9), 0.05, 0)
    check(nk, p, draw_v(p, 9), 0.05, 10)
    s, W = dev(p.sigma), dev(p.W)
    with pytest.raises(nk.NkError):
        nk.qgt_matvec(s, W, None, None, None, None)
    with pytest.raises(nk.NkError):
        nk.qgt_matvec(s, W, None, None, None, dev(draw_v(p, 1)[2]), diag_shift=-1.0)


# ------------------------------------------------------------------ nk_sr_solve: CG against the dense direct solve
def _sr_case(nk, p, shift, tol, chunk=0):
    cplx = p.complex_params
    f = draw_v(p, 77)
    (da, db, dW), iters, res = nk.sr_solve(dev(p.sigma), dev(p.W), dev(p.b), *map(dev, f), diag_shift=shift, tol=tol,
                                           max_iter=400, chunk_size=chunk)
    delta = orc.pack_params(*(t.cpu().numpy() for t in (da, db, dW))).astype(np.complex128 if cplx else np.float64)
    G = orc.qgt_dense(p.sigma, p.W, p.b)
    if not cplx:
        G = G.real
    A = G + shift * np.eye(G.shape[0])
    fv = orc.pack_params(*f).astype(A.dtype)
    ref = orc.pack_params(*orc.sr_solve(p.sigma, p.W, p.b, *f, shift))
    true_res = np.linalg.norm(A @ delta - fv) / np.linalg.norm(fv)
    cond = np.linalg.cond(A)
    err = np.linalg.norm(delta - ref) / np.linalg.norm(ref)
    return iters, res, true_res, err, cond


@pytest.mark.parametrize("case", [
    dict(cfg=1, n=2048, shift=0.05),
    dict(kind=0, lattice="square", L=4, M=16, n=1500, shift=0.02),
    dict(kind=1, lattice="chain", L=9, M=20, n=1000, shift=0.05, h=1.0, complex_params=True),
])
def test_sr_solve_matches_dense_solve(nk, case):
    case = dict(case)
    shift, n = case.pop("shift"), case.pop("n")
    if "cfg" in case:
        p = inp.make_config(case["cfg"], n_samples=n)
    else:
        p = inp.make_problem(case.pop("kind"), case.pop("lattice"), case.pop("L"), case.pop("M"), n, seed=8,
                             scale=0.2, **case)
    tol = 1e-5
    iters, res, true_res, err, cond = _sr_case(nk, p, shift, tol)
    print(f"{p.name}: P = {p.n_sites + p.n_hidden * (1 + p.n_sites)}, cond {cond:.1f}, {iters} CG iterations, "
          f"recurrence residual {res:.1e}, true residual {true_res:.1e}, |delta - dense| / |dense| = {err:.1e}")
    assert 0 < iters < 400 and res <= tol
    assert true_res <= 5 * tol + 2e-6            # the fp32 recurrence residual tracks the fp64 true residual
    assert err <= cond * (5 * tol + 2e-6)        # |dx| / |x| <= cond * |r| / |f|


def test_sr_solve_limits_and_errors(nk):
    p = inp.make_config(1, n_samples=512)
    f = draw_v(p, 5)
    sig, W, b = dev(p.sigma), dev(p.W), dev(p.b)
    # max_iter = 0 returns zero; a huge shift makes delta = f / shift after one iteration
    (da, db, dW), iters, res = nk.sr_solve(sig, W, b, *map(dev, f), max_iter=0)
    assert iters == 0 and float(dW.abs().max()) == 0.0 and res == 1.0
    (da, db, dW), iters, res = nk.sr_solve(sig, W, b, *map(dev, f), diag_shift=1e6, tol=1e-4)
    np.testing.assert_allclose(dW.cpu().numpy() * 1e6, f[2], rtol=1e-3, atol=1e-3)
    assert iters <= 4
    # f = 0 -> delta = 0 without iterating; chunked run reproduces the unchunked solution to CG accuracy
    z = tuple(np.zeros_like(x) for x in f)
    (da, db, dW), iters, _ = nk.sr_solve(sig, W, b, *map(dev, z))
    assert iters == 0 and float(da.abs().max()) == 0.0
    x0, _, _ = nk.sr_solve(sig, W, b, *map(dev, f), diag_shift=0.05, tol=1e-6)
    x1, _, _ = nk.sr_solve(sig, W, b, *map(dev, f), diag_shift=0.05, tol=1e-6, chunk_size=100)
    assert float((x0[2] - x1[2]).abs().max()) <= 1e-4 * float(x0[2].abs().max())
    with pytest.raises(nk.NkError):
        nk.sr_solve(sig, W, b, dev(f[0]), dev(f[1]), None)
    with pytest.raises(nk.NkError):
        nk.sr_solve(sig, W, b, *map(dev, f), tol=-1.0)

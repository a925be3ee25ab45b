"""nk_rbm_logpsi_static — ln psi with the library's static 16 MiB device scratch instead of a caller workspace
(include/nkb200.h; README "No-allocation entry point").  The file sorts last on purpose: the suite runs with
`pytest -x`, so a failure here hides nothing after it.  Runs alone in a fresh process and after the other GPU tests.

Checked: the new entry point against the existing nk_rbm_logpsi path (same tolerance as tests/test_gpu_parity.py,
LOGPSI_ATOL = 1e-5 absolute; the two run the same kernels, so they are in fact bit-equal) and against the float64
oracle, on two calls in a row of DIFFERENT shapes (the second call finds the first one's contents in the shared
scratch), real and complex; that the calls change the device's free memory by nothing; that a problem beyond the
static maximum is rejected with NK_ERR_WORKSPACE before anything runs."""
import ctypes as C

import numpy as np
import pytest
import torch

from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp

pytestmark = pytest.mark.gpu

LOGPSI_ATOL = 1e-5            # tests/test_gpu_parity.py


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def close(lp_a, lp_b, atol=LOGPSI_ATOL):
    a = np.asarray(lp_a).astype(np.complex128)
    b = np.asarray(lp_b).astype(np.complex128)
    dre = np.abs(a.real - b.real)
    dim = np.abs((a.imag - b.imag + np.pi) % (2 * np.pi) - np.pi)          # Im ln psi is defined modulo 2 pi
    assert dre.max() <= atol, f"Re ln psi differs by {dre.max()}"
    assert dim.max() <= atol, f"Im ln psi differs by {dim.max()}"


def problems():
    # a larger real problem first (3.2 MiB of the scratch), then a small real one of another shape, then a complex one:
    # each later call finds stale buffers of a different layout in the array
    big = inp.make_config(2)                                                # N = M = 100, 4096 samples
    small = inp.make_config(1)                                              # N = M = 10, 1024 samples
    cplx = inp.make_problem(inp.KIND_HEISENBERG, "chain", 12, 36, 257, seed=5, complex_params=True, scale=0.1)
    ragged = inp.make_problem(inp.KIND_ISING, "square", 5, 70, 333, seed=6, scale=0.05, h=1.0)   # N = 25, M = 70
    return [big, small, cplx, ragged]


def test_static_scratch_matches_workspace_path_on_consecutive_calls(nk):
    cap = nk.load().nk_rbm_logpsi_static_max_bytes()
    assert cap == 16 << 20
    for rep in range(2):                                                    # the whole sequence twice, back to back
        for p in problems():
            sigma, W, a, b = dev(p.sigma), dev(p.W), dev(p.a), dev(p.b)
            got = nk.rbm_logpsi_static(sigma, W, a, b)
            again = nk.rbm_logpsi_static(sigma, W, a, b)                    # two calls in a row on the same inputs
            ref = nk.rbm_logpsi(sigma, W, a, b)                             # the existing path, caller workspace
            torch.cuda.synchronize()
            close(got.cpu().numpy(), ref.cpu().numpy())
            close(again.cpu().numpy(), ref.cpu().numpy())
            assert torch.equal(got, again), "two consecutive calls on the same inputs disagree"
            rows = np.arange(0, p.n_samples, max(1, p.n_samples // 64))
            lp_or = orc.rbm_logpsi(p.sigma[rows], p.W, p.a, p.b)
            close(got.cpu().numpy()[rows], lp_or, atol=3e-5 if p.complex_params else LOGPSI_ATOL)


def test_static_scratch_float64_output_and_missing_bias(nk):
    p = inp.make_config(2, n_samples=777)
    sigma, W = dev(p.sigma), dev(p.W)
    out = torch.empty(777, dtype=torch.float64, device="cuda")
    got = nk.rbm_logpsi_static(sigma, W, None, None, out=out, out_f64=True)
    ref = nk.rbm_logpsi(sigma, W, None, None, out_f64=True)
    torch.cuda.synchronize()
    assert got.data_ptr() == out.data_ptr()
    close(got.cpu().numpy(), ref.cpu().numpy())
    close(got.cpu().numpy(), orc.rbm_logpsi(p.sigma, p.W, None, None))


def test_static_scratch_calls_allocate_nothing(nk):
    p = inp.make_config(2)
    sigma, W, a, b = dev(p.sigma), dev(p.W), dev(p.a), dev(p.b)
    out = torch.empty(p.n_samples, dtype=torch.float32, device="cuda")
    nk.rbm_logpsi_static(sigma, W, a, b, out=out)                           # first call: modules load, address resolved
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    reserved0 = torch.cuda.memory_reserved()
    for _ in range(3):
        nk.rbm_logpsi_static(sigma, W, a, b, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_reserved() == reserved0                        # nothing through torch's allocator either
    assert free1 == free0, f"device free memory changed by {free0 - free1} bytes across the calls"


def test_static_scratch_rejects_problems_beyond_its_maximum(nk):
    lib = nk.load()
    cap = lib.nk_rbm_logpsi_static_max_bytes()
    p = inp.make_config(2)
    B = 40000                                                               # ~31 MiB of scratch at N = M = 100
    assert lib.nk_rbm_logpsi_workspace_bytes(B, p.n_sites, p.n_hidden, nk.NK_F32) > cap
    sigma = torch.ones((B, p.n_sites), dtype=torch.int8, device="cuda")
    W, a, b = dev(p.W), dev(p.a), dev(p.b)
    with pytest.raises(nk.NkError, match="static array holds"):
        nk.rbm_logpsi_static(sigma, W, a, b)
    out = torch.full((B,), 7.0, dtype=torch.float32, device="cuda")
    n0 = nk.launch_count()
    rc = lib.nk_rbm_logpsi_static(C.c_void_p(sigma.data_ptr()), B, p.n_sites, p.n_hidden, nk.NK_F32,
                                  C.c_void_p(W.data_ptr()), C.c_void_p(a.data_ptr()), C.c_void_p(b.data_ptr()),
                                  C.c_void_p(out.data_ptr()), None, 0, None)
    torch.cuda.synchronize()
    assert rc == -3                                                         # NK_ERR_WORKSPACE
    assert nk.launch_count() == n0 and bool((out == 7.0).all())             # nothing was launched, nothing written
    # the largest batch that fits still runs
    lo, hi = 1, B
    while hi - lo > 1:
        mid = (lo + hi) // 2
        if lib.nk_rbm_logpsi_workspace_bytes(mid, p.n_sites, p.n_hidden, nk.NK_F32) <= cap:
            lo = mid
        else:
            hi = mid
    sig = dev(inp.make_config(2, n_samples=lo).sigma)
    got = nk.rbm_logpsi_static(sig, W, a, b)
    ref = nk.rbm_logpsi(sig, W, a, b)
    torch.cuda.synchronize()
    close(got.cpu().numpy(), ref.cpu().numpy())

"""GPU parity of the fully symmetric RBM workload (nk_rbmsymm_expand -> nk_local_energy / nk_energy_gradient ->
nk_rbmsymm_reduce_gradient) against the oracle's direct evaluation of Eq. (41)/(56).  Same tolerances as the plain
RBM: ln psi 1e-5 absolute, E_loc 1e-4 relative, gradient 1e-6 * max|E - mean| (sum of |G| expanded entries:
|G| times the per-entry bound of tests/test_gpu_gradient.py)."""
import numpy as np
import pytest
import torch

from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp
from test_gpu_parity import assert_eloc, assert_logpsi

pytestmark = pytest.mark.gpu


def dev(x):
    return None if x is None else torch.from_numpy(np.ascontiguousarray(x)).cuda()


def make_case(lattice, L, F, n, cplx, kind=inp.KIND_HEISENBERG, scale=0.05, seed=0, **kw):
    """A problem on the lattice with tied parameters (W_sym [F][N], b_sym [F]) drawn by the same recipe."""
    perms = inp.translation_perms(lattice, L)
    N = perms.shape[1]
    p = inp.make_problem(kind, lattice, L, F, n, seed=seed, complex_params=cplx, scale=scale, **kw)
    return p, p.W, p.b, perms                # make_problem's (W [F][N], b [F]) serve as the tied parameters


@pytest.mark.parametrize("lattice,L,F,n,cplx", [("chain", 10, 2, 256, False), ("square", 4, 3, 200, True),
                                                ("square", 6, 2, 96, False), ("square", 10, 4, 24, False)])
def test_rbmsymm_local_energy_and_gradient(nk, lattice, L, F, n, cplx):
    p, Ws, bs, perms = make_case(lattice, L, F, n, cplx, order=1)
    G, N = perms.shape
    W, b = nk.rbmsymm_expand(dev(Ws), dev(bs), dev(perms))
    # the expansion is exactly the tied weights: row (i, g) scattered by the permutation
    Wn = W.cpu().numpy()
    for i, g in ((0, 0), (F - 1, G - 1), (F // 2, G // 3)):
        assert np.array_equal(Wn[i * G + g][perms[g]], Ws[i])
    assert np.array_equal(b.cpu().numpy().reshape(F, G), np.repeat(bs[:, None], G, axis=1))
    op = nk.Operator.from_problem(p)
    sig = dev(p.sigma)
    eloc, lp, stats = nk.local_energy(op, sig, W, None, b)
    torch.cuda.synchronize()
    e_ref, lp_ref = orc.rbmsymm_local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, Ws, bs, perms)
    assert_eloc(eloc.cpu().numpy(), e_ref)
    assert_logpsi(lp.cpu().numpy(), lp_ref)
    # gradient with respect to the tied parameters, from the oracle's E_loc rounded to fp32
    e32 = e_ref.astype(np.complex64 if cplx else np.float32)
    st = dev(np.array(orc.stats(e32.astype(e_ref.dtype))))
    ga, gb, gW = nk.energy_gradient(sig, W, b, dev(e32), st)
    gWs, gbs = nk.rbmsymm_reduce_gradient(gW, gb, dev(perms), F)
    torch.cuda.synchronize()
    rb, rW = orc.rbmsymm_energy_gradient(p.sigma, Ws, bs, perms, e32)
    de = np.abs(e32.astype(e_ref.dtype) - e32.astype(e_ref.dtype).mean()).max()
    bound = 1e-6 * de * (1 if cplx else 2) * G
    for name, g, r in (("W", gWs, rW), ("b", gbs, rb)):
        err = np.abs(g.cpu().numpy().astype(r.dtype) - r).max()
        assert err <= bound + 4e-7 * np.abs(r).max(), f"grad_{name}_sym: err {err}, bound {bound}"
    op.close()


def test_rbmsymm_invariance_on_the_gpu_and_errors(nk):
    p, Ws, bs, perms = make_case("square", 6, 2, 64, False, order=1)
    W, b = nk.rbmsymm_expand(dev(Ws), dev(bs), dev(perms))
    lp0 = nk.rbm_logpsi(dev(p.sigma), W, None, b, out_f64=True).cpu().numpy()
    lp1 = nk.rbm_logpsi(dev(np.ascontiguousarray(p.sigma[:, perms[7]])), W, None, b, out_f64=True).cpu().numpy()
    np.testing.assert_allclose(lp0, lp1, atol=2e-5)                  # psi(g s) = psi(s)
    with pytest.raises(nk.NkError):
        nk.rbmsymm_expand(dev(Ws), dev(bs), dev(perms.astype(np.int64)))
    with pytest.raises(nk.NkError):
        nk.rbmsymm_reduce_gradient(W, b, dev(perms), 5)

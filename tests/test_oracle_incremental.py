"""Pins of the second CPU route (oracle/nk_incremental.c): the float64 incremental local energy must reproduce the
from-scratch oracle (oracle/nk_oracle.py, itself pinned in test_oracle_pins.py) to 1e-12 — two independent routes to
PAPER.md Eq. (12) L652 ("from-scratch vs incremental ... must agree to 1e-12")."""
import numpy as np
import pytest

from oracle import nk_incremental as inc
from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp

RTOL = 1e-12


def _both(p, flags=0, a="keep", b="keep"):
    a_ = p.a if a == "keep" else a
    b_ = p.b if b == "keep" else b
    e0, l0 = orc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, a_, b_, flags)
    e1, l1 = inc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, p.W, a_, b_, flags)
    return e0, l0, e1, l1


def _check(e0, l0, e1, l1):
    assert e1.dtype == e0.dtype and l1.dtype == l0.dtype
    assert np.max(np.abs(e1 - e0) / np.maximum(np.abs(e0), 1.0)) < RTOL
    assert np.max(np.abs(l1 - l0) / np.maximum(np.abs(l0), 1.0)) < RTOL


@pytest.mark.parametrize("cfg,n", [(1, 1024), (2, 256), (3, 48), (4, 96)])
def test_incremental_equals_from_scratch_on_configs(cfg, n):
    p = inp.make_config(cfg, n_samples=n)
    _check(*_both(p))


def test_incremental_equals_from_scratch_on_config5_subset():
    """A fixed subset of config 5 spread over its 16 chunks of 4096: the first 8 samples of each."""
    p = inp.make_config(5)
    idx = np.concatenate([np.arange(c * 4096, c * 4096 + 8) for c in range(16)])
    e0, l0 = orc.local_energy(p.kind, p.sigma[idx], p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    e1, l1 = inc.local_energy(p.kind, p.sigma[idx], p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    _check(e0, l0, e1, l1)


@pytest.mark.parametrize("complex_params", [False, True])
@pytest.mark.parametrize("kind", [inp.KIND_HEISENBERG, inp.KIND_ISING])
def test_incremental_small_cases_with_options(kind, complex_params):
    """Odd sizes, large parameters (|theta| up to ~10: the stable branch of ln cosh), Marshall sign, missing biases,
    out-of-sector samples (parallel bonds and polarised rows included)."""
    rng = np.random.default_rng(77 + kind + 2 * complex_params)
    p = inp.make_problem(kind, "square", 3, 7, 40, seed=5, complex_params=complex_params, scale=0.8, h=1.7,
                         order=2 if kind == inp.KIND_HEISENBERG else 1, J=(1.0, -0.4), sz0=False)
    p.sigma[:] = rng.choice(np.array([-1, 1], dtype=np.int8), size=p.sigma.shape)
    p.sigma[0] = 1
    p.sigma[1] = -1
    _check(*_both(p))
    _check(*_both(p, a=None))
    _check(*_both(p, b=None))
    if kind == inp.KIND_HEISENBERG:
        _check(*_both(p, flags=orc.FLAG_MARSHALL))


def test_incremental_w_zero_closed_form():
    """W = 0, a = 0: uniform psi, E_loc = sum_c J_c n_b,c = 200 on the 10 x 10 lattice."""
    p = inp.make_config(2, n_samples=32)
    e, _ = inc.local_energy(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h, np.zeros_like(p.W), None, p.b)
    assert np.allclose(e, 200.0, rtol=0, atol=1e-10)

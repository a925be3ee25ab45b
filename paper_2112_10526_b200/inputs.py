"""Seeded synthetic inputs for the batched local-energy path (shared by tests, bench and oracle checks).

This module holds NO arithmetic of the method (no log cosh, no matrix elements, no ratios): it only
draws parameters / samples and lists lattice bonds.  Both the oracle (`oracle/`) and the CUDA path
consume the arrays produced here; neither imports the other.

Recipe (BASELINE.json `configs`):
  * parameters: numpy `default_rng(1000 + c)`, float64 normal draws in the order a, b, W
    (complex: Re a, Im a, Re b, Im b, Re W, Im W), times the config's sigma_param, cast to fp32/complex64;
  * samples: `default_rng(2000 + c)`; S^z=0 configs: every row is a uniformly random permutation of
    N/2 (+1)s and N/2 (-1)s (`Spin(1/2, total_sz=0)`); config 3: i.i.d. uniform +-1; int8;
  * lattices (`Square(L, max_neighbor_order=2)`): each undirected pair once,
    site s = x*L + y, NN bonds (colour 0) listed site by site, NNN bonds (colour 1) appended after.
"""
from __future__ import annotations

import dataclasses
import hashlib

import numpy as np

KIND_HEISENBERG = 0   # H = sum_b J_c(b) sigma_i . sigma_j            (Eq. (50))
KIND_ISING = 1        # H = J sum_b sz_i sz_j - h sum_i sx_i          (Eq. (54))


def chain_bonds(L: int):
    """Periodic chain: bonds (i, i+1 mod L), colour 0.  L >= 3 so that no bond is doubled."""
    if L < 3:
        raise ValueError("chain needs L >= 3")
    bonds = np.array([[i, (i + 1) % L] for i in range(L)], dtype=np.int32)
    return bonds, np.zeros(L, dtype=np.int32)


def square_bonds(L: int, max_neighbor_order: int = 1):
    """Periodic L x L square lattice, site s = x*L + y.

    order 1: (x,y)-(x+1,y), (x,y)-(x,y+1), colour 0, site by site;
    order 2: additionally (x,y)-(x+1,y+1), (x,y)-(x+1,y-1), colour 1, appended after all NN bonds.
    """
    if L < 3:
        raise ValueError("square lattice needs L >= 3")
    if max_neighbor_order not in (1, 2):
        raise ValueError("max_neighbor_order must be 1 or 2")
    s = lambda x, y: (x % L) * L + (y % L)
    bonds, colors = [], []
    for x in range(L):
        for y in range(L):
            bonds.append((s(x, y), s(x + 1, y))); colors.append(0)
            bonds.append((s(x, y), s(x, y + 1))); colors.append(0)
    if max_neighbor_order == 2:
        for x in range(L):
            for y in range(L):
                bonds.append((s(x, y), s(x + 1, y + 1))); colors.append(1)
                bonds.append((s(x, y), s(x + 1, y - 1))); colors.append(1)
    return np.array(bonds, dtype=np.int32), np.array(colors, dtype=np.int32)


@dataclasses.dataclass
class Problem:
    """One synthetic instance: operator description + RBM parameters + sample batch."""
    name: str
    kind: int                 # KIND_HEISENBERG | KIND_ISING
    n_sites: int
    n_hidden: int
    bonds: np.ndarray         # int32 [n_b][2]
    colors: np.ndarray        # int32 [n_b]
    J: np.ndarray             # float64 [n_colors]
    h: float                  # transverse field (Ising only)
    complex_params: bool
    W: np.ndarray             # [M][N] float32 | complex64
    a: np.ndarray             # [N]
    b: np.ndarray             # [M]
    sigma: np.ndarray         # int8 [B][N], values +1/-1
    chunk_size: int = 0       # 0 = whole batch

    @property
    def n_samples(self) -> int:
        return int(self.sigma.shape[0])

    @property
    def max_conn(self) -> int:
        return (len(self.bonds) if self.kind == KIND_HEISENBERG else self.n_sites) + 1

    def sha256(self) -> dict:
        return {k: hashlib.sha256(np.ascontiguousarray(getattr(self, k)).tobytes()).hexdigest()[:16]
                for k in ("W", "a", "b", "sigma", "bonds")}


def draw_params(rng, n_sites: int, n_hidden: int, scale: float, complex_params: bool):
    N, M = n_sites, n_hidden
    if not complex_params:
        a = rng.standard_normal(N) * scale
        b = rng.standard_normal(M) * scale
        W = rng.standard_normal((M, N)) * scale
        return W.astype(np.float32), a.astype(np.float32), b.astype(np.float32)
    ar, ai = rng.standard_normal(N) * scale, rng.standard_normal(N) * scale
    br, bi = rng.standard_normal(M) * scale, rng.standard_normal(M) * scale
    Wr, Wi = rng.standard_normal((M, N)) * scale, rng.standard_normal((M, N)) * scale
    return ((Wr + 1j * Wi).astype(np.complex64), (ar + 1j * ai).astype(np.complex64),
            (br + 1j * bi).astype(np.complex64))


def draw_samples(rng, n_samples: int, n_sites: int, total_sz_zero: bool) -> np.ndarray:
    if total_sz_zero:
        if n_sites % 2:
            raise ValueError("S^z = 0 sector needs an even number of sites")
        base = np.tile(np.array([1, -1], dtype=np.int8), n_sites // 2)
        return rng.permuted(np.tile(base, (n_samples, 1)), axis=1)
    return (2 * rng.integers(0, 2, size=(n_samples, n_sites), dtype=np.int8) - 1).astype(np.int8)


# (name, kind, lattice, L, order, alpha, complex, scale, B, sz0, J, h, chunk)
_CONFIGS = {
    1: ("heis1d_L10_real_a1", KIND_HEISENBERG, "chain", 10, 1, 1, False, 0.1, 1024, True, (1.0,), 0.0, 0),
    2: ("heis2d_10x10_real_a1", KIND_HEISENBERG, "square", 10, 1, 1, False, 0.05, 4096, True, (1.0,), 0.0, 0),
    3: ("tfim2d_20x20_real_a2", KIND_ISING, "square", 20, 1, 2, False, 0.02, 8192, False, (1.0,), 3.0, 0),
    4: ("j1j2_10x10_complex_a4", KIND_HEISENBERG, "square", 10, 2, 4, True, 0.03, 16384, True, (1.0, 0.5), 0.0, 0),
    5: ("heis2d_32x32_real_a2", KIND_HEISENBERG, "square", 32, 1, 2, False, 0.01, 65536, True, (1.0,), 0.0, 4096),
    # not a BASELINE.json config: the widest real RBM the library takes (M = alpha N = 4096), config 5's
    # lattice and recipe, for the width-limit bench line (`bench.py --config 6`) and tests
    6: ("heis2d_32x32_real_a4", KIND_HEISENBERG, "square", 32, 1, 4, False, 0.01, 16384, True, (1.0,), 0.0, 4096),
}


def make_config(c: int, n_samples: int | None = None, sample_seed_offset: int = 0) -> Problem:
    """BASELINE.json `configs[c-1]` (c = 1..5; 6 = the alpha = 4 widening of config 5).  `n_samples` overrides the batch size (bench shards,
    oracle subsets); `sample_seed_offset` gives ranks of a weak-scaling run distinct batches."""
    name, kind, lat, L, order, alpha, cplx, scale, B, sz0, J, h, chunk = _CONFIGS[c]
    bonds, colors = chain_bonds(L) if lat == "chain" else square_bonds(L, order)
    N = L if lat == "chain" else L * L
    M = alpha * N
    W, a, b = draw_params(np.random.default_rng(1000 + c), N, M, scale, cplx)
    sigma = draw_samples(np.random.default_rng(2000 + c + 7919 * sample_seed_offset),
                         B if n_samples is None else n_samples, N, sz0)
    return Problem(name, kind, N, M, bonds, colors, np.array(J, dtype=np.float64), float(h), cplx,
                   W, a, b, sigma, chunk)


def make_problem(kind: int, lattice: str, L: int, n_hidden: int, n_samples: int, *, seed: int = 0,
                 order: int = 1, complex_params: bool = False, scale: float = 0.1, sz0: bool | None = None,
                 J=(1.0,), h: float = 0.0, chunk_size: int = 0) -> Problem:
    """Free-form small instance for tests (same recipe, arbitrary sizes)."""
    bonds, colors = chain_bonds(L) if lattice == "chain" else square_bonds(L, order)
    N = L if lattice == "chain" else L * L
    if sz0 is None:
        sz0 = (kind == KIND_HEISENBERG) and N % 2 == 0
    J = np.array(J, dtype=np.float64)
    if len(J) <= int(colors.max()):
        raise ValueError("need one coupling per bond colour")
    W, a, b = draw_params(np.random.default_rng(1000 + seed), N, n_hidden, scale, complex_params)
    sigma = draw_samples(np.random.default_rng(2000 + seed), n_samples, N, sz0)
    return Problem(f"{lattice}{L}_k{kind}_M{n_hidden}_s{seed}", kind, N, n_hidden, bonds, colors, J, float(h),
                   complex_params, W, a, b, sigma, chunk_size)


def translation_perms(lattice: str, L: int) -> np.ndarray:
    """Translation group of the periodic chain (|G| = L) or L x L square lattice (|G| = L^2) as site permutations:
    perms[g][r] = the site g r, with site = x * L + y as in `square_bonds`; g = 0 is the identity."""
    if lattice == "chain":
        r = np.arange(L)
        return np.stack([(r + t) % L for t in range(L)]).astype(np.int32)
    x, y = np.divmod(np.arange(L * L), L)
    return np.stack([(((x + tx) % L) * L + (y + ty) % L) for tx in range(L) for ty in range(L)]).astype(np.int32)

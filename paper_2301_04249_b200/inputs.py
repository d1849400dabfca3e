"""Seeded synthetic inputs for the RT-EOM-CCSD hot path (BASELINE.json ``configs``).

This module holds NONE of the method's arithmetic and imports neither the CUDA binding nor the
oracle: it only draws random numbers and orders orbitals.  Both sides are handed the same arrays.

Recipe: spatial orbitals 0..n-1, 0 = core (eps = -20.0 Ha), 1..o-1 valence occupied
eps ~ U[-1.5,-0.3] sorted, o..n-1 virtual eps ~ U[v_lo,v_hi] sorted; spatial Cholesky vectors
L^Q_pq (p<=q, mirrored) = sigma * exp(-Q/d) * N(0,1).  The core orbital is ionised in alpha
("c is now included in the set of unoccupied single-particle states"), so
alpha: occ {1..o-1}, virt {0, o..n-1};   beta: occ {0..o-1}, virt {o..n-1};
each spin is delivered in its own [occupied | virtual] order; fock = diag(eps) per spin.
The paper's molecules are not available; these inputs stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

SEED_BASE = 230104249


@dataclass(frozen=True)
class Config:
    name: str
    o: int            # spatial occupied (including the core orbital)
    v: int            # spatial virtual
    K: int            # n_chol
    d: float          # decay constant of exp(-Q/d)
    v_lo: float
    v_hi: float
    dt: float
    steps: int
    sigma: float = 0.3
    index: int = 0

    @property
    def dims(self):
        """(o_alpha, o_beta, v_alpha, v_beta): alpha core-ionised."""
        return self.o - 1, self.o, self.v + 1, self.v

    @property
    def n(self):
        return self.o + self.v


# d for configs 2 and 5 is not given by BASELINE.json ("same generator"): 12 (literal) and 400.
CONFIGS = {
    "tiny": Config("tiny", 4, 12, 48, 12.0, 0.1, 3.0, 0.025, 200, index=1),
    "small": Config("small", 8, 60, 340, 12.0, 0.1, 3.0, 0.025, 2000, index=2),
    "mid": Config("mid", 24, 200, 900, 150.0, 0.05, 6.0, 0.05, 500, index=3),
    "large": Config("large", 40, 360, 1600, 300.0, 0.05, 6.0, 0.05, 100, index=4),
    "largest": Config("largest", 56, 480, 2200, 400.0, 0.05, 6.0, 0.05, 20, index=5),
}


def custom(o, v, K, d=12.0, v_lo=0.1, v_hi=3.0, dt=0.025, steps=10, sigma=0.3, index=99, name="custom"):
    return Config(name, o, v, K, d, v_lo, v_hi, dt, steps, sigma, index)


def stabilised_sigma(cfg: Config) -> float:
    """sigma_s = 0.2*sqrt(144/(v*d)): keeps the ladder operator's top eigenvalue ~3 Ha at every size
    (SURVEY.md 8(d) caveat).  A documented deviation from BASELINE.json."""
    return 0.2 * float(np.sqrt(144.0 / (cfg.v * cfg.d)))


def make_problem(cfg: Config, sigma: float | None = None, fock_offdiag: float = 0.0, dtype=np.float64):
    """Returns (oa, ob, va, vb, K, L[2,K,n,n], fock[2,n,n]).  ``fock_offdiag`` > 0 adds a seeded real
    symmetric perturbation to both Fock matrices (for tests of the general-Fock code path)."""
    rng = np.random.default_rng(SEED_BASE + cfg.index)
    o, v, n, K = cfg.o, cfg.v, cfg.n, cfg.K
    sig = cfg.sigma if sigma is None else sigma
    eps = np.empty(n)
    eps[0] = -20.0
    eps[1:o] = np.sort(rng.uniform(-1.5, -0.3, o - 1))
    eps[o:] = np.sort(rng.uniform(cfg.v_lo, cfg.v_hi, v))
    scale = sig * np.exp(-np.arange(K) / cfg.d)
    order_a = np.array(list(range(1, o)) + [0] + list(range(o, n)))
    ia = np.ix_(order_a, order_a)
    L = np.empty((2, K, n, n), dtype=dtype)
    for Q in range(K):                       # one spatial vector at a time: no third copy of L (10 GB at config 5)
        A = np.triu(rng.standard_normal((n, n)))
        S = scale[Q] * (A + np.triu(A, 1).T)
        L[1, Q] = S                          # beta: spatial order
        L[0, Q] = S[ia]                      # alpha: core orbital moved to the first virtual position
    fock = np.zeros((2, n, n))
    fock[0] = np.diag(eps[order_a])
    fock[1] = np.diag(eps)
    if fock_offdiag > 0.0:
        for s in range(2):
            A = rng.standard_normal((n, n)) * fock_offdiag
            fock[s] += 0.5 * (A + A.T)
    oa, ob, va, vb = cfg.dims
    return oa, ob, va, vb, K, L, fock


def n_amplitudes(oa, ob, va, vb):
    p = lambda x: x * (x - 1) // 2
    return oa * va + ob * vb, p(oa) * p(va) + p(ob) * p(vb) + oa * ob * va * vb


def random_amplitudes(cfg_or_dims, std=1e-3, seed_offset=1000):
    """Residual-only variant: Re, Im of every unique packed element ~ N(0, std) (BASELINE.json config 1)."""
    if isinstance(cfg_or_dims, Config):
        dims, idx = cfg_or_dims.dims, cfg_or_dims.index
    else:
        dims, idx = tuple(cfg_or_dims), 0
    n1, n2 = n_amplitudes(*dims)
    rng = np.random.default_rng(SEED_BASE + seed_offset + idx)
    t1 = std * (rng.standard_normal(n1) + 1j * rng.standard_normal(n1))
    t2 = std * (rng.standard_normal(n2) + 1j * rng.standard_normal(n2))
    return t1, t2

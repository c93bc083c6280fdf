"""Seeded synthetic inputs and the workload table for the five BASELINE.json configs.

This module is shared by the oracle-side tests, the CUDA-side tests and bench.py.  It
holds NO arithmetic of the method (no epsilon tensors, no gamma matrices, no determinants,
no term expansion): only the workload table (nucleus spec as data, lattice sizes, momenta,
seeds) and the random-number recipes of SURVEY.md section 8(d) / BASELINE.json `configs`.

Propagator recipe (BASELINE.json configs[0]): for every timeslice t and site x, U_x(t) and
D_x(t) are independent 12x12 complex128 matrices, Re and Im i.i.d. N(0,1), scaled by
exp(-0.5*t), t = 0..T-1 (scale 1 at t = 0).  Layout [T][L^3][12][12], row = sink index,
column = source index, site index s = x + L*(y + L*z).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Sequence, Tuple

import numpy as np

__all__ = [
    "WickConfig", "CONFIGS", "get_config", "make_propagators_numpy", "make_propagators_torch",
    "make_random_term_list", "sample_site_times", "site_coords",
]


@dataclass(frozen=True)
class WickConfig:
    """One workload of BASELINE.json `configs` (data only)."""
    name: str
    index: int
    nucleus: Tuple[Tuple[str, int], ...]      # (('p', gamma) | ('n', gamma), ...) in product order
    n_u: int
    n_d: int
    L: int
    T: int
    momenta: Tuple[Tuple[int, int, int], ...]  # integer units of 2*pi/L
    seed: int
    random_list: bool = False                  # cfg 4b: seed-generated term list instead of the nucleus
    n_random_terms: int = 0

    @property
    def volume(self) -> int:
        return self.L ** 3

    @property
    def site_times(self) -> int:
        return self.T * self.L ** 3


# BASELINE.json configs[0..4]; "4b" is the random list of configs[4] (same tuple sizes and term count).
CONFIGS = {
    "cfg0": WickConfig("cfg0_proton", 0, (("p", 0),), 2, 1, 4, 8, ((0, 0, 0),), 1000),
    "cfg1": WickConfig("cfg1_deuteron", 1, (("p", 0), ("n", 0)), 3, 3, 16, 32, ((0, 0, 0),), 1001),
    "cfg2": WickConfig("cfg2_helium3", 2, (("p", 0), ("p", 1), ("n", 0)), 5, 4, 24, 48,
                       ((0, 0, 0), (1, 0, 0)), 1002),
    "cfg3": WickConfig("cfg3_helium4", 3, (("p", 0), ("p", 1), ("n", 0), ("n", 1)), 6, 6, 32, 64,
                       ((0, 0, 0),), 1003),
    "cfg4": WickConfig("cfg4_lithium7", 4,
                       (("p", 0), ("p", 1), ("p", 2), ("n", 0), ("n", 1), ("n", 2), ("n", 3)),
                       10, 11, 24, 48, ((0, 0, 0),), 1004),
    "cfg4b": WickConfig("cfg4b_lithium7_random_list", 4, (), 10, 11, 24, 48, ((0, 0, 0),), 1004,
                        random_list=True, n_random_terms=441),
}


def get_config(name: str) -> WickConfig:
    return CONFIGS[name]


def make_propagators_numpy(seed: int, L: int, T: int, t0: int = 0, nt: int | None = None,
                           decay: float = 0.5):
    """U, D of shape [nt][L^3][12][12] complex128 for timeslices t0..t0+nt-1 (numpy, CPU).

    Each timeslice has its own child stream, so a slice [t0, t0+nt) equals the same slice of the
    full-T array for the same seed.
    """
    nt = T - t0 if nt is None else nt
    V = L ** 3
    U = np.empty((nt, V, 12, 12), dtype=np.complex128)
    D = np.empty((nt, V, 12, 12), dtype=np.complex128)
    for i in range(nt):
        t = t0 + i
        rng = np.random.default_rng([seed, t])
        scale = np.exp(-decay * t)
        U[i] = (rng.standard_normal((V, 12, 12)) + 1j * rng.standard_normal((V, 12, 12))) * scale
        D[i] = (rng.standard_normal((V, 12, 12)) + 1j * rng.standard_normal((V, 12, 12))) * scale
    return U, D


def make_propagators_torch(seed: int, L: int, T: int, device, t0: int = 0, nt: int | None = None,
                           decay: float = 0.5):
    """Same recipe drawn with a torch generator on `device` (different stream than numpy's; both
    sides of every comparison always consume the SAME array).  Returns complex128 tensors
    [nt][L^3][12][12]; one child seed per timeslice."""
    import torch
    nt = T - t0 if nt is None else nt
    V = L ** 3
    U = torch.empty((nt, V, 12, 12), dtype=torch.complex128, device=device)
    D = torch.empty((nt, V, 12, 12), dtype=torch.complex128, device=device)
    gen = torch.Generator(device=device)
    for i in range(nt):
        t = t0 + i
        scale = float(np.exp(-decay * t))
        for k, P in enumerate((U, D)):
            gen.manual_seed(seed * 1000003 + 2 * t + k)
            r = torch.randn((V, 12, 12, 2), dtype=torch.float64, device=device, generator=gen)
            P[i] = torch.view_as_complex(r) * scale
    return U, D


def make_random_term_list(seed: int, n_u: int, n_d: int, n_terms: int):
    """cfg 4b (SURVEY.md 8(c) reading 6): each tuple a uniformly random sorted n-subset of {0..11},
    independent for a_u, b_u, a_d, b_d; weights N(0,1) + i N(0,1).  Returns uint8 arrays
    a_u, b_u [n_terms][n_u], a_d, b_d [n_terms][n_d] and complex128 w [n_terms]."""
    rng = np.random.default_rng([seed, 4242])

    def subsets(n):
        out = np.empty((n_terms, n), dtype=np.uint8)
        for i in range(n_terms):
            out[i] = np.sort(rng.choice(12, size=n, replace=False))
        return out

    a_u, b_u, a_d, b_d = subsets(n_u), subsets(n_u), subsets(n_d), subsets(n_d)
    w = rng.standard_normal(n_terms) + 1j * rng.standard_normal(n_terms)
    return a_u, b_u, a_d, b_d, w


def sample_site_times(seed: int, L: int, T: int, n_sites: int, times: Sequence[int] | None = None):
    """Seeded sample of (t, site) pairs for per-site parity at full size: n_sites sites on each of
    the timeslices {0, T//2, T-1} (default), always including site 0 and the last site."""
    rng = np.random.default_rng([seed, 777])
    V = L ** 3
    times = [0, T // 2, T - 1] if times is None else list(times)
    out: List[Tuple[int, int]] = []
    for t in sorted(set(times)):
        sites = {0, V - 1}
        while len(sites) < min(n_sites, V):
            sites.add(int(rng.integers(V)))
        out.extend((t, s) for s in sorted(sites)[:max(n_sites, 2)])
    return out


def site_coords(L: int):
    """Integer coordinates (x, y, z) of site index s = x + L*(y + L*z); shape [L^3][3]."""
    s = np.arange(L ** 3)
    return np.stack([s % L, (s // L) % L, s // (L * L)], axis=1)

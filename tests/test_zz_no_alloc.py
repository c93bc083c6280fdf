"""wick_minor_dets_static: the entry point that allocates nothing (scratch in a static device array, include/wick.h).
Collected last on purpose (file name): the suite runs with pytest -x.

Its output must equal the existing path's (wick_minor_dets: same kernels, scratch from cudaMalloc) and match the oracle's
elimination within the tolerance of tests/test_gpu_parity.py::test_minor_dets_vs_oracle, on two calls in a row that share
the static array (the second with other sizes, so stale contents of the first would show)."""
import numpy as np
import pytest
import torch

import paper_2411_08962_b200 as wk
from oracle import wick_oracle as wo

pytestmark = pytest.mark.gpu


def _case(seed, n, n_sites, n_minors):
    rng = np.random.default_rng(seed)
    P = rng.standard_normal((n_sites, 12, 12)) + 1j * rng.standard_normal((n_sites, 12, 12))
    rows = np.array([rng.permutation(12)[:n] for _ in range(n_minors)], np.uint8).reshape(n_minors, n)
    cols = np.array([rng.permutation(12)[:n] for _ in range(n_minors)], np.uint8).reshape(n_minors, n)
    return P, rows, cols


def _check(P, rows, cols, dev):
    n_minors, n = rows.shape
    Pd = torch.from_numpy(P).to(dev)
    out = torch.full((n_minors, P.shape[0]), float("nan"), dtype=torch.complex128, device=dev)   # caller-owned output
    got = wk.minor_dets_static(Pd, rows, cols, out).cpu().numpy()
    ref_path = wk.minor_dets(Pd, rows, cols).cpu().numpy()
    assert np.array_equal(got, ref_path)                          # same kernels, same launch shape: bit for bit
    sub = P[:, rows[:, :, None], cols[:, None, :]]
    ref = wo.det_elim(sub).T
    scale = np.prod(np.linalg.norm(sub, axis=3), axis=2).T
    assert np.all(np.abs(got - ref) <= 1e-13 * max(n, 1) * scale + 1e-300)


def test_static_scratch_entry_point_two_calls_in_a_row(cuda_device):
    assert wk.static_scratch_bytes() == 16 << 20
    # call 1: 6x6 minors, ragged site count (results staged in the static array), many minors
    _check(*_case(11, 6, 70, 500), cuda_device)
    # call 2 right after it: 10x10 minors (two-word descriptors), fewer minors, site count a multiple of 32 (direct stores)
    _check(*_case(12, 10, 64, 37), cuda_device)
    # call 3: ragged again with a different shape, so the staging area holds call 1's values where this call does not write
    _check(*_case(13, 3, 33, 200), cuda_device)


def test_static_scratch_entry_point_rejects_sizes_beyond_its_maximum(cuda_device):
    P, rows, cols = _case(14, 2, 32, 4097)
    Pd = torch.from_numpy(P).to(cuda_device)
    out = torch.empty((4097, 32), dtype=torch.complex128, device=cuda_device)
    with pytest.raises(wk.WickError, match="exceeds the static limit of 4096"):
        wk.minor_dets_static(Pd, rows, cols, out)
    # at the limit, ragged: 4096 minors x 224 sites per pass still fit behind the descriptors
    P, rows, cols = _case(15, 2, 40, 4096)
    _check(P, rows, cols, cuda_device)

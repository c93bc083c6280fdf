"""GPU parity tests (-m gpu): the CUDA path, called through the C-ABI binding, against the CPU oracle on
the same seeded inputs.  Tolerance (BASELINE.json north_star): |C_gpu - C_oracle| <= 1e-10 * S_abs(t),
S_abs(t) = sum_x sum_terms |w detU detD| (oracle).  Per-site sigma uses the per-site S_abs.

What runs where: full-lattice C(t) for cfg 0 at full size and for every
other config on a shrunken lattice with the FULL term list; at BASELINE's full sizes per-site sigma on
a seeded sample of sites (cfg 1-4), the device reduction against a CPU sum of the device sigma, and
closed-form structural checks (site-scaled propagators) with a one-site oracle."""
import numpy as np
import pytest
import torch

import paper_2411_08962_b200 as wk
from oracle import wick_oracle as wo
from wick_inputs import CONFIGS, make_propagators_numpy, make_random_term_list, sample_site_times

pytestmark = pytest.mark.gpu
REL_TOL = 1e-10


def _dev(a, device):
    return torch.from_numpy(np.ascontiguousarray(a)).to(device)


def _terms_for(cfg):
    c = CONFIGS[cfg]
    if c.random_list:
        return wk.build_terms_from_list(*make_random_term_list(c.seed, c.n_u, c.n_d, c.n_random_terms))
    return wk.build_terms(c.nucleus)


_SINK_CACHE = {}


def _oracle_site(cfg, U, D):
    """sigma and S_abs of one site from the oracle's OWN expansion (never from the builder's tables)."""
    c = CONFIGS[cfg]
    if c.random_list:
        a_u, b_u, a_d, b_d, w = make_random_term_list(c.seed, c.n_u, c.n_d, c.n_random_terms)
        return wo.site_terms_value(U, D, a_u, b_u, a_d, b_d, w)
    if cfg not in _SINK_CACHE:
        _SINK_CACHE[cfg] = wo.merged_terms(c.nucleus)
    return wo.site_value_outer(U, D, _SINK_CACHE[cfg])


def _oracle_lattice(cfg, U, D, momenta, L):
    T, V = U.shape[:2]
    sigma = np.zeros((T, V), complex)
    sabs = np.zeros((T, V))
    for t in range(T):
        for s in range(V):
            sigma[t, s], sabs[t, s] = _oracle_site(cfg, U[t, s], D[t, s])
    return wo.reduce_sites(sigma, momenta, L), sigma, sabs


# ---------------------------------------------------------------------------------------------
# a4 alone: every minor size, ragged site counts, unsorted index tuples
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("n", list(range(0, 13)))
@pytest.mark.parametrize("n_sites", [70, 64])
def test_minor_dets_vs_oracle(n, n_sites, cuda_device):
    rng = np.random.default_rng(100 + n)
    P = rng.standard_normal((n_sites, 12, 12)) + 1j * rng.standard_normal((n_sites, 12, 12))
    P[3] *= 1e-3                                                # scale spread across sites
    P[5, 2, :] = 0.0                                            # an exactly zero row: singular minors
    n_minors = 37 if n_sites == 70 else 300                      # spans several warps and a ragged tail
    rows = np.array([rng.permutation(12)[:n] for _ in range(n_minors)], np.uint8).reshape(n_minors, n)
    cols = np.array([rng.permutation(12)[:n] for _ in range(n_minors)], np.uint8).reshape(n_minors, n)
    got = wk.minor_dets(_dev(P, cuda_device), rows, cols).cpu().numpy()
    assert got.shape == (n_minors, n_sites)
    if n == 0:
        assert np.all(got == 1.0)
        return
    sub = P[:, rows[:, :, None], cols[:, None, :]]              # [site][minor][n][n]
    ref = wo.det_elim(sub).T
    # Hadamard bound prod_i ||row_i|| is the natural scale of the rounding error of a determinant
    scale = np.prod(np.linalg.norm(sub, axis=3), axis=2).T
    assert np.all(np.abs(got - ref) <= 1e-13 * n * scale + 1e-300)
    zero_row = np.any(rows == 2, axis=1)
    assert np.all(got[zero_row, 5] == 0.0)                      # exact zeros, no NaN from a zero pivot
    assert np.all(np.isfinite(got.view(np.float64)))


@pytest.mark.parametrize("cfg,flags", [("cfg3", 0), ("cfg3", wk.CONTRACT_NO_REG_MINORS), ("cfg2", 0), ("cfg1", 0),
                                       ("cfg4", 0), ("cfg4b", 0)])
@pytest.mark.parametrize("n_sites", [70, 64])
def test_library_minor_tables_vs_oracle(cfg, flags, n_sites, cuda_device):
    """The kernels wick_contract launches for the library's OWN tables (register-resident instance kernel and Schur-column
    cache kernel for 6x6, cached kernels for 10x10 / 11x11, column-trie kernels below), minor by minor against the oracle's
    elimination: every minor of the first, a middle and the last row tuple plus a seeded sample, on a ragged and a full
    site count, with a tiny-scale site and a site with an exactly zero row."""
    t = _terms_for(cfg)
    rng = np.random.default_rng(300 + n_sites)
    P = rng.standard_normal((n_sites, 12, 12)) + 1j * rng.standard_normal((n_sites, 12, 12))
    P[3] *= 1e-3
    P[5, 2, :] = 0.0
    tup = t.tuples()
    mins = t.minors()
    for fl in (0, 1):
        rows, cols, mrow, mcol = tup[2 * fl], tup[2 * fl + 1], mins[2 * fl], mins[2 * fl + 1]
        n = rows.shape[1]
        got = wk.minor_table(_dev(P, cuda_device), t, fl, flags=flags).cpu().numpy()
        nm = len(mrow)
        assert got.shape == (nm, n_sites)
        pick = np.flatnonzero(np.isin(mrow, [mrow.min(), int(np.median(mrow)), mrow.max()]))
        pick = np.union1d(pick, rng.choice(nm, size=min(nm, 4000), replace=False))
        sub = P[:, rows[mrow[pick]][:, :, None], cols[mcol[pick]][:, None, :]]          # [site][minor][n][n]
        ref = wo.det_elim(sub).T
        scale = np.prod(np.linalg.norm(sub, axis=3), axis=2).T
        assert np.all(np.abs(got[pick] - ref) <= 1e-13 * n * scale + 1e-300), (cfg, fl)
        zero_row = np.any(rows[mrow[pick]] == 2, axis=1)
        assert np.all(got[pick][zero_row, 5] == 0.0)
        assert np.all(np.isfinite(got.view(np.float64)))


def test_minor_dets_repeated_index_is_zero(cuda_device):
    rng = np.random.default_rng(7)
    P = rng.standard_normal((32, 12, 12)) + 1j * rng.standard_normal((32, 12, 12))
    for n in (2, 3, 4, 6, 10):
        rows = np.array([list(range(n))], np.uint8)
        rows[0, n - 1] = rows[0, 0]                             # Pauli: repeated row index
        cols = np.array([list(range(1, n + 1))], np.uint8)
        got = wk.minor_dets(_dev(P, cuda_device), rows, cols).cpu().numpy()
        scale = np.prod(np.linalg.norm(P[:, rows[0]][:, :, cols[0]], axis=2), axis=1)
        assert np.all(np.abs(got[0]) <= 1e-13 * n * scale)


# ---------------------------------------------------------------------------------------------
# full path, full lattice
# ---------------------------------------------------------------------------------------------

def _check_C(C_gpu, C_ref, sabs_t):
    err = np.abs(C_gpu - C_ref)
    assert np.all(err <= REL_TOL * sabs_t[None, :]), (err / sabs_t[None, :]).max()


@pytest.mark.parametrize("flags", [0, wk.CONTRACT_FORCE_FLAT, wk.CONTRACT_NO_STAGED, wk.CONTRACT_COMPLEX_COEFFS])
def test_cfg0_proton_full_lattice(flags, cuda_device):
    c = CONFIGS["cfg0"]
    U, D = make_propagators_numpy(c.seed, c.L, c.T)
    mom = [(0, 0, 0), (1, 0, 0), (0, 1, 2), (-1, 3, 0)]
    t = wk.build_terms(c.nucleus)
    Cg, sg = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, mom, c.L, c.T, want_sigma=True, flags=flags)
    Cg, sg = Cg.cpu().numpy(), sg.cpu().numpy()
    Cr, sr, sabs = _oracle_lattice("cfg0", U, D, mom, c.L)
    assert np.all(np.abs(sg - sr) <= REL_TOL * sabs)
    _check_C(Cg, Cr, sabs.sum(axis=1))
    # RAW-mode oracle (no sorting, no merging) on one timeslice
    raw = wo.nucleus_raw_terms(c.nucleus)
    for s in (0, 17, 63):
        v = wo.raw_site_value(U[3, s], D[3, s], raw, raw)
        assert abs(sg[3, s] - v) <= REL_TOL * sabs[3, s]


SHRUNK = {  # cfg -> (L, T, momenta): full term list, lattice the oracle finishes in about a minute
    "cfg1": (3, 2, [(0, 0, 0), (1, 0, 0)]),
    "cfg2": (2, 2, [(0, 0, 0), (1, 0, 0)]),
    "cfg3": (2, 1, [(0, 0, 0)]),
    "cfg4": (4, 3, [(0, 0, 0), (0, 0, 1)]),
    "cfg4b": (4, 3, [(0, 0, 0), (1, 1, 1)]),
}


@pytest.mark.parametrize("cfg", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg4b"])
def test_shrunken_lattice_full_term_list(cfg, cuda_device):
    c = CONFIGS[cfg]
    L, T, mom = SHRUNK[cfg]
    U, D = make_propagators_numpy(c.seed, L, T)
    t = _terms_for(cfg)
    Cg, sg = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, mom, L, T, want_sigma=True)
    Cg, sg = Cg.cpu().numpy(), sg.cpu().numpy()
    Cr, sr, sabs = _oracle_lattice(cfg, U, D, mom, L)
    assert np.all(np.abs(sg - sr) <= REL_TOL * sabs), (np.abs(sg - sr) / sabs).max()
    _check_C(Cg, Cr, sabs.sum(axis=1))
    if cfg in ("cfg1", "cfg2", "cfg4"):                         # the unstaged factorised kernel / general complex entries
        for fl in (wk.CONTRACT_NO_STAGED, wk.CONTRACT_COMPLEX_COEFFS):
            Cn = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, mom, L, T, flags=fl)
            _check_C(Cn.cpu().numpy(), Cr, sabs.sum(axis=1))
    if cfg in ("cfg1", "cfg4"):                                 # the flat path on the same list
        Cf = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, mom, L, T, flags=wk.CONTRACT_FORCE_FLAT)
        _check_C(Cf.cpu().numpy(), Cr, sabs.sum(axis=1))


@pytest.mark.parametrize("n_u,n_d", [(9, 12), (10, 9), (11, 8), (7, 5)])
def test_generic_lists_of_large_minors(n_u, n_d, cuda_device):
    """Random term lists with 9..12-index tuples: the library walks such minors in its own order (column tuples that
    miss only small indices are processed with descending columns and a parity sign, contract.cu: build_minor_descs);
    the contraction must not depend on that."""
    L, T, mom = 2, 2, [(0, 0, 0), (1, 0, 1)]
    U, D = make_propagators_numpy(900 + n_u, L, T)
    lst = make_random_term_list(77 + n_d, n_u, n_d, 300)
    t = wk.build_terms_from_list(*lst)
    Cg, sg = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, mom, L, T, want_sigma=True)
    sg = sg.cpu().numpy()
    sr, sabs = np.zeros((T, L ** 3), complex), np.zeros((T, L ** 3))
    for tt in range(T):
        for x in range(L ** 3):
            sr[tt, x], sabs[tt, x] = wo.site_terms_value(U[tt, x], D[tt, x], *lst)
    assert np.all(np.abs(sg - sr) <= REL_TOL * sabs), (np.abs(sg - sr) / sabs).max()
    _check_C(Cg.cpu().numpy(), wo.reduce_sites(sr, mom, L), sabs.sum(axis=1))


# ---------------------------------------------------------------------------------------------
# BASELINE's full sizes: sampled sites + device reduction + structure
# ---------------------------------------------------------------------------------------------

FULL = {  # cfg -> (timeslices to run, sites sampled per timeslice)
    "cfg1": ([0, 16, 31], 6),
    "cfg2": ([0, 47], 4),
    "cfg3": ([0, 32, 63], 3),
    "cfg4": ([0, 47], 8),
    "cfg4b": ([24], 8),
}


@pytest.mark.parametrize("cfg", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg4b"])
def test_full_size_sampled_sites_and_reduction(cfg, cuda_device):
    c = CONFIGS[cfg]
    times, n_sites = FULL[cfg]
    t = _terms_for(cfg)
    for tt in times:
        U, D = make_propagators_numpy(c.seed, c.L, c.T, t0=tt, nt=1)
        Cg, sg = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, c.momenta, c.L, 1, want_sigma=True)
        Cg, sg = Cg.cpu().numpy(), sg.cpu().numpy()
        assert np.all(np.isfinite(sg.view(np.float64)))
        for (_, s) in sample_site_times(c.seed, c.L, c.T, n_sites, times=[tt]):
            ref, sabs = _oracle_site(cfg, U[0, s], D[0, s])
            assert abs(sg[0, s] - ref) <= REL_TOL * sabs, (cfg, tt, s, abs(sg[0, s] - ref) / sabs)
        # device reduction (momentum phases + fixed tree) against the oracle's sum of the device sigma
        Cr = wo.reduce_sites(sg, c.momenta, c.L)
        assert np.all(np.abs(Cg - Cr) <= 1e-13 * np.sum(np.abs(sg)))


@pytest.mark.parametrize("cfg", ["cfg2", "cfg3"])
def test_full_size_site_scaled_propagators(cfg, cuda_device):
    """U_x = s_x U0 with s_x = exp(-i p.x / n_u), D_x = D0: the projection at momentum p returns
    L^3 sigma0, at another momentum 0; sigma0 from a one-site oracle call."""
    c = CONFIGS[cfg]
    L = c.L
    rng = np.random.default_rng(c.seed)
    U0 = rng.standard_normal((12, 12)) + 1j * rng.standard_normal((12, 12))
    D0 = rng.standard_normal((12, 12)) + 1j * rng.standard_normal((12, 12))
    p = np.array([1, 0, 0])
    s = np.arange(L ** 3)
    xyz = np.stack([s % L, (s // L) % L, s // (L * L)], axis=1)
    sx = np.exp(-2j * np.pi * (xyz @ p) / L / c.n_u)
    U = (U0[None] * sx[:, None, None])[None]
    D = np.broadcast_to(D0, (1, L ** 3, 12, 12)).copy()
    t = _terms_for(cfg)
    mom = [(1, 0, 0), (0, 0, 0), (0, 1, 0)]
    Cg = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, mom, L, 1).cpu().numpy()
    sigma0, sabs0 = _oracle_site(cfg, U0, D0)
    tol = REL_TOL * sabs0 * L ** 3
    assert abs(Cg[0, 0] - L ** 3 * sigma0) <= tol
    assert abs(Cg[1, 0]) <= tol and abs(Cg[2, 0]) <= tol


# ---------------------------------------------------------------------------------------------
# edge cases, determinism, host entry point
# ---------------------------------------------------------------------------------------------

def test_ragged_lattices_small_workspace_and_determinism(cuda_device):
    c = CONFIGS["cfg1"]
    t = wk.build_terms(c.nucleus)
    for L, T in ((1, 1), (3, 3), (5, 1)):                       # V = 1, 27, 125: not multiples of 32
        U, D = make_propagators_numpy(77, L, T)
        mom = [(0, 0, 0), (1, 2, 0)]
        Ud, Dd = _dev(U, cuda_device), _dev(D, cuda_device)
        C1, s1 = wk.contract(Ud, Dd, t, mom, L, T, want_sigma=True)
        C2 = wk.contract(Ud, Dd, t, mom, L, T)
        assert torch.equal(C1, C2)                              # bit-reproducible run to run
        ws = torch.empty(wk.contract_workspace_bytes(t, L, T, 2, minimum=True), dtype=torch.uint8, device=cuda_device)
        C3, s3 = wk.contract(Ud, Dd, t, mom, L, T, workspace=ws, want_sigma=True)   # 32-site batches
        Cr, sr, sabs = _oracle_lattice("cfg1", U, D, mom, L)
        assert np.all(np.abs(s1.cpu().numpy() - sr) <= REL_TOL * sabs)
        assert np.all(np.abs(s3.cpu().numpy() - sr) <= REL_TOL * sabs)
        _check_C(C1.cpu().numpy(), Cr, sabs.sum(axis=1))
        _check_C(C3.cpu().numpy(), Cr, sabs.sum(axis=1))
    with pytest.raises(wk.WickError, match="workspace"):
        wk.contract(Ud, Dd, t, mom, L, T, workspace=torch.empty(1024, dtype=torch.uint8, device=cuda_device))


def test_empty_term_list_and_isospin_alias(cuda_device):
    U, D = make_propagators_numpy(5, 2, 2)
    Ud, Dd = _dev(U, cuda_device), _dev(D, cuda_device)
    empty = wk.build_terms([("p", 0), ("p", 0)])                # Pauli-blocked: no terms
    C = wk.contract(Ud, Dd, empty, [(0, 0, 0)], 2, 2)
    assert torch.all(C == 0)
    t = wk.build_terms(CONFIGS["cfg0"].nucleus)
    C = wk.contract(Ud, Ud, t, [(0, 0, 0)], 2, 2).cpu().numpy()  # U_dev == D_dev is legal
    Cr, _, sabs = _oracle_lattice("cfg0", U, U, [(0, 0, 0)], 2)
    _check_C(C, Cr, sabs.sum(axis=1))


def test_isospin_alias_shares_the_minor_table(cuda_device):
    """U_dev == D_dev with equal flavour tables (deuteron): the d minors are not evaluated a second time and
    the result has the same bits as the run on two separate buffers holding the same propagator."""
    c = CONFIGS["cfg1"]
    L, T, mom = 3, 2, [(0, 0, 0), (1, 0, 2)]
    U, _ = make_propagators_numpy(c.seed, L, T)
    t = wk.build_terms(c.nucleus)
    Ud, Ucopy = _dev(U, cuda_device), _dev(U.copy(), cuda_device)
    wk.launch_count(reset=True)
    C_alias, s_alias = wk.contract(Ud, Ud, t, mom, L, T, want_sigma=True)
    n_alias = wk.launch_count(reset=True)
    C_two, s_two = wk.contract(Ud, Ucopy, t, mom, L, T, want_sigma=True)
    n_two = wk.launch_count(reset=True)
    assert torch.equal(C_alias, C_two) and torch.equal(s_alias, s_two)
    assert n_alias < n_two
    Cr, sr, sabs = _oracle_lattice("cfg1", U, U, mom, L)
    assert np.all(np.abs(s_alias.cpu().numpy() - sr) <= REL_TOL * sabs)
    _check_C(C_alias.cpu().numpy(), Cr, sabs.sum(axis=1))


def test_contract_host_matches_device_call(cuda_device):
    c = CONFIGS["cfg0"]
    U, D = make_propagators_numpy(c.seed, c.L, c.T)
    t = wk.build_terms(c.nucleus)
    mom = [(0, 0, 0), (1, 1, 0)]
    Ch, sh = wk.contract_host(U, D, t, mom, c.L, c.T, want_sigma=True)
    Cd, sd = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, mom, c.L, c.T, want_sigma=True)
    assert np.array_equal(sh, sd.cpu().numpy())
    assert np.array_equal(Ch, Cd.cpu().numpy())
    n0 = wk.launch_count(reset=True)
    assert n0 > 0


def test_contract_host_multi_block_overlap(cuda_device, monkeypatch):
    """wick_contract_host over several timeslice blocks (H2D of block b+1 on the copy stream while block b computes,
    PAPER.md:663; short last block): bitwise equal to the device call, and within 1e-10 of the oracle on sampled sites."""
    c = CONFIGS["cfg1"]
    L, T = 4, 7
    U, D = make_propagators_numpy(c.seed, L, T)
    t = wk.build_terms(c.nucleus)
    mom = [(0, 0, 0), (1, 0, 3)]
    monkeypatch.setenv("WICK_HOST_BLOCK_BYTES", str(2 * L ** 3 * 144 * 16))   # 2 timeslices per block: blocks of 2, 2, 2, 1
    wk.launch_count(reset=True)
    Ch, sh = wk.contract_host(U, D, t, mom, L, T, want_sigma=True)
    n_multi = wk.launch_count(reset=True)
    monkeypatch.delenv("WICK_HOST_BLOCK_BYTES")
    Ch1 = wk.contract_host(U, D, t, mom, L, T)
    n_single = wk.launch_count(reset=True)
    assert n_multi > n_single                                   # the hook really cut the call into several blocks
    # bitwise equal to device calls on the same blocks (the order of the sums inside a site depends on the number of
    # 32-site groups of a batch, so calls of different shape agree to rounding, calls of equal shape bit for bit)
    for t0 in (0, 2, 4, 6):
        nt = min(2, T - t0)
        Cd, sd = wk.contract(_dev(U[t0:t0 + nt], cuda_device), _dev(D[t0:t0 + nt], cuda_device), t, mom, L, nt, want_sigma=True)
        assert np.array_equal(Ch[:, t0:t0 + nt], Cd.cpu().numpy()) and np.array_equal(sh[t0:t0 + nt], sd.cpu().numpy())
    Cfull, sfull = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, mom, L, T, want_sigma=True)
    assert np.array_equal(Ch1, Cfull.cpu().numpy())
    assert np.all(np.abs(sh - sfull.cpu().numpy()) <= 1e-13 * np.abs(sh).max(axis=1, keepdims=True) * 1e3)
    for (tt, x) in ((0, 0), (1, 63), (2, 17), (5, 40), (6, 5), (6, 63)):
        ref, sabs = _oracle_site("cfg1", U[tt, x], D[tt, x])
        assert abs(sh[tt, x] - ref) <= REL_TOL * sabs


@pytest.mark.parametrize("cfg,L,T", [("cfg1", 3, 2), ("cfg3", 2, 1)])
def test_isospin_lists_on_the_gpu(cfg, L, T, cuda_device):
    """U == D (the paper's m_u = m_d): the swap-symmetrised factorised list (WICK_BUILD_ISOSPIN) and, for
    the deuteron, the flat list merged by the randomised identity test (IDENTITY_TEST | ISOSPIN) against the oracle's
    full expansion evaluated with D = U; and such handles refuse U != D."""
    c = CONFIGS[cfg]
    mom = [(0, 0, 0), (1, 0, 1)]
    U, Dother = make_propagators_numpy(c.seed, L, T)
    Ud = _dev(U, cuda_device)
    if cfg == "cfg3":
        # 18 s per site with two fresh determinants per term: that oracle on two sites, and on every site the oracle's method B
        # (each distinct minor once, pinned to method A in tests/test_oracle_pins.py)
        sink = wo.merged_terms(c.nucleus)
        sr, sabs = np.zeros((T, L ** 3), complex), np.zeros((T, L ** 3))
        for tt in range(T):
            for x in range(L ** 3):
                sr[tt, x], sabs[tt, x] = wo.site_value_method_b(U[tt, x], U[tt, x], sink)
        for x in (0, L ** 3 - 1):
            ref, ref_abs = _oracle_site(cfg, U[0, x], U[0, x])
            assert abs(ref - sr[0, x]) <= 1e-13 * ref_abs
        Cr = wo.reduce_sites(sr, mom, L)
    else:
        Cr, sr, sabs = _oracle_lattice(cfg, U, U, mom, L)
    handles = [wk.build_terms(c.nucleus, flags=wk.BUILD_ISOSPIN)]
    if cfg == "cfg1":
        handles.append(wk.build_terms(c.nucleus, flags=wk.BUILD_IDENTITY_TEST | wk.BUILD_ISOSPIN, seed=9))
        assert handles[1].info.n_terms == 26721 and handles[1].info.is_outer_product == 0
    for t in handles:
        Cg, sg = wk.contract(Ud, Ud, t, mom, L, T, want_sigma=True)
        assert np.all(np.abs(sg.cpu().numpy() - sr) <= REL_TOL * sabs), (np.abs(sg.cpu().numpy() - sr) / sabs).max()
        _check_C(Cg.cpu().numpy(), Cr, sabs.sum(axis=1))
        with pytest.raises(wk.WickError, match="U_dev == D_dev"):
            wk.contract(Ud, _dev(Dother, cuda_device), t, mom, L, T)


@pytest.mark.parametrize("cfg", ["cfg4", "cfg4b"])
def test_jacobi_complementary_minor_path(cfg, cuda_device):
    """WICK_CONTRACT_JACOBI: 10x10 / 11x11 minors as det A times a 2x2 / 1x1 minor of the inverse, against the
    oracle (which eliminates every minor itself) on a small lattice with the full list, on sampled sites at full size, and
    against the LU path of the library."""
    c = CONFIGS[cfg]
    L, T, mom = SHRUNK[cfg]
    U, D = make_propagators_numpy(c.seed, L, T)
    t = _terms_for(cfg)
    Ud, Dd = _dev(U, cuda_device), _dev(D, cuda_device)
    Cg, sg = wk.contract(Ud, Dd, t, mom, L, T, want_sigma=True, flags=wk.CONTRACT_JACOBI)
    Cg, sg = Cg.cpu().numpy(), sg.cpu().numpy()
    Cr, sr, sabs = _oracle_lattice(cfg, U, D, mom, L)
    assert np.all(np.abs(sg - sr) <= REL_TOL * sabs), (np.abs(sg - sr) / sabs).max()
    _check_C(Cg, Cr, sabs.sum(axis=1))
    Clu = wk.contract(Ud, Dd, t, mom, L, T).cpu().numpy()
    _check_C(Cg, Clu, sabs.sum(axis=1))
    # the same identity through the minor tables (inverse kernel, minors of the inverse, reduction) instead of the fused per-site kernel
    Cu, su = wk.contract(Ud, Dd, t, mom, L, T, want_sigma=True, flags=wk.CONTRACT_JACOBI | wk.CONTRACT_JACOBI_UNFUSED)
    assert np.all(np.abs(su.cpu().numpy() - sr) <= REL_TOL * sabs)
    _check_C(Cu.cpu().numpy(), Cr, sabs.sum(axis=1))
    tt = 0
    U1, D1 = make_propagators_numpy(c.seed, c.L, c.T, t0=tt, nt=1)
    _, s1 = wk.contract(_dev(U1, cuda_device), _dev(D1, cuda_device), t, c.momenta, c.L, 1, want_sigma=True, flags=wk.CONTRACT_JACOBI)
    s1 = s1.cpu().numpy()
    for (_, s) in sample_site_times(c.seed, c.L, c.T, 6, times=[tt]):
        ref, sa = _oracle_site(cfg, U1[0, s], D1[0, s])
        assert abs(s1[0, s] - ref) <= REL_TOL * sa


@pytest.mark.parametrize("n_u,n_d", [(9, 10), (8, 11), (11, 7)])
def test_jacobi_path_on_generic_lists(n_u, n_d, cuda_device):
    """Complement sizes 1..4 on one side, an LU-only size (7) on the other: the two paths mix per flavour."""
    L, T, mom = 2, 2, [(0, 0, 0), (1, 0, 1)]
    U, D = make_propagators_numpy(950 + n_u, L, T)
    lst = make_random_term_list(70 + n_d, n_u, n_d, 300)
    t = wk.build_terms_from_list(*lst)
    Cg, sg = wk.contract(_dev(U, cuda_device), _dev(D, cuda_device), t, mom, L, T, want_sigma=True, flags=wk.CONTRACT_JACOBI)
    sg = sg.cpu().numpy()
    sr, sabs = np.zeros((T, L ** 3), complex), np.zeros((T, L ** 3))
    for tt in range(T):
        for x in range(L ** 3):
            sr[tt, x], sabs[tt, x] = wo.site_terms_value(U[tt, x], D[tt, x], *lst)
    assert np.all(np.abs(sg - sr) <= REL_TOL * sabs), (np.abs(sg - sr) / sabs).max()
    _check_C(Cg.cpu().numpy(), wo.reduce_sites(sr, mom, L), sabs.sum(axis=1))


def test_jacobi_fused_kernel_long_list_ragged_sites_and_one_propagator(cuda_device):
    """The fused Jacobi kernel beyond the cases above: a list longer than the 1024 term records it stages in shared memory
    (the records are then read from global memory), a site count (27) that is no multiple of its 16-site CTAs, and U == D
    (both lane groups of a site invert the same matrix).  Same launch count as a short list: the fused path was taken."""
    n_u, n_d, L, T, mom = 9, 10, 3, 1, [(0, 0, 0), (1, 2, 0)]
    U, D = make_propagators_numpy(977, L, T)
    Ud, Dd = _dev(U, cuda_device), _dev(D, cuda_device)
    counts = []
    for n_terms, same in ((300, False), (1500, False), (1500, True)):
        lst = make_random_term_list(81, n_u, n_d, n_terms)
        t = wk.build_terms_from_list(*lst)
        assert (t.info.n_terms > 1024) == (n_terms > 1024)
        wk.launch_count(reset=True)
        Cg, sg = wk.contract(Ud, Ud if same else Dd, t, mom, L, T, want_sigma=True, flags=wk.CONTRACT_JACOBI)
        sg = sg.cpu().numpy()
        counts.append(wk.launch_count())
        Dh = U if same else D
        sr, sabs = np.zeros((T, L ** 3), complex), np.zeros((T, L ** 3))
        for x in range(L ** 3):
            sr[0, x], sabs[0, x] = wo.site_terms_value(U[0, x], Dh[0, x], *lst)
        assert np.all(np.abs(sg - sr) <= REL_TOL * sabs), (np.abs(sg - sr) / sabs).max()
        _check_C(Cg.cpu().numpy(), wo.reduce_sites(sr, mom, L), sabs.sum(axis=1))
    assert counts[0] == counts[1] == counts[2] and counts[0] <= 3, counts


def test_correlation_matrix_shares_the_determinants(cuda_device):
    """wick_contract_many (GEVP, Sec. V): the 2x2 correlation matrix of {p n product operator, Eq. (20)}
    against the oracle's sink x conj(source) expansion for every entry, with the minors launched once for all four."""
    L, T, mom = 3, 2, [(0, 0, 0), (1, 0, 2)]
    U, D = make_propagators_numpy(4321, L, T)
    Ud, Dd = _dev(U, cuda_device), _dev(D, cuda_device)
    ops = [wk.operator_from_nucleons(CONFIGS["cfg1"].nucleus), wk.operator_paper(wk.OP_DEUTERON_EQ20)]
    m = wk.build_terms_matrix(ops)
    lists = [m[k][kp] for k in range(2) for kp in range(2)]
    wk.contract_many(Ud, Dd, lists, mom, L, T)                   # uploads the tables
    wk.profile_enable(True)
    Cg, sg = wk.contract_many(Ud, Dd, lists, mom, L, T, want_sigma=True)
    prof = wk.profile_read()
    wk.profile_enable(False)
    assert prof["minors_u"][1] == 1 and prof["minors_d"][1] == 1 and prof["reduce"][1] == 4   # a4 once, a5 per entry
    Cg, sg = Cg.cpu().numpy(), sg.cpu().numpy()
    osink = [wo.merged_terms(CONFIGS["cfg1"].nucleus), wo.merged_from_raw(wo.deuteron_eq20_raw_terms())]
    for k in range(2):
        for kp in range(2):
            sr, sabs = np.zeros((T, L ** 3), complex), np.zeros((T, L ** 3))
            for tt in range(T):
                for x in range(L ** 3):
                    sr[tt, x], sabs[tt, x] = wo.site_value_outer(U[tt, x], D[tt, x], osink[k], osink[kp])
            e = 2 * k + kp
            assert np.all(np.abs(sg[e] - sr) <= REL_TOL * sabs), (k, kp, (np.abs(sg[e] - sr) / sabs).max())
            _check_C(Cg[e], wo.reduce_sites(sr, mom, L), sabs.sum(axis=1))
    # hermiticity of the correlation matrix entries that are each other's conjugate transpose only holds for U, D from a
    # gauge average; what must hold exactly is that single-list calls reproduce the entries
    C01 = wk.contract(Ud, Dd, m[0][1], mom, L, T).cpu().numpy()
    assert np.allclose(C01, Cg[1], rtol=1e-12, atol=0)
    other = wk.build_terms(CONFIGS["cfg0"].nucleus)
    with pytest.raises(wk.WickError, match="share"):
        wk.contract_many(Ud, Dd, [lists[0], other], mom, L, T)


def test_two_cluster_sink_against_the_two_site_oracle(cuda_device):
    """Cluster sink (plane-wave sink of Eq. 8 for single nucleons): proton at x, neutron at y, each projected to its
    own momentum, against the oracle's explicit double sum over (x, y) with stacked determinants."""
    L, T = 2, 2
    U, D = make_propagators_numpy(8642, L, T)
    Ud, Dd = _dev(U, cuda_device), _dev(D, cuda_device)
    a, b = wk.operator_from_nucleons([("p", 0)]), wk.operator_from_nucleons([("n", 0)])
    sa, sb, src = wo.merged_terms([("p", 0)]), wo.merged_terms([("n", 0)]), wo.merged_terms([("p", 0), ("n", 0)])
    for mom_a, mom_b in (((0, 0, 0), (0, 0, 0)), ((1, 0, 0), (1, 1, 0))):
        Cg = wk.two_cluster_correlator(Ud, Dd, a, b, mom_a, mom_b, L, T)
        Cr, sabs = wo.two_cluster_correlator(U, D, sa, sb, src, mom_a, mom_b, L)
        assert np.all(np.abs(Cg - Cr) <= REL_TOL * sabs), (np.abs(Cg - Cr) / sabs).max()
    # the block tensor itself on a ragged lattice: one entry against the oracle's minors
    L3 = 3
    U3, D3 = make_propagators_numpy(8643, L3, 1)
    B = wk.block_tensor(_dev(U3, cuda_device), _dev(D3, cuda_device), wk.build_block_terms(a), (0, 1, 2), L3, 1).cpu().numpy()
    import itertools
    cu = list(itertools.combinations(range(12), 2))
    ph = wo.momentum_phases(L3, [(0, 1, 2)])[0]
    for (iu, idd) in ((0, 0), (17, 5), (65, 11)):
        ref, ref_abs = 0.0, 0.0
        for x in range(L3 ** 3):
            for (ua, da, ca) in sa:
                v = ca * wo.det_elim(U3[0, x][np.ix_(ua, cu[iu])]) * D3[0, x][da[0], idd] * ph[x]
                ref += v
                ref_abs += abs(v)
        assert abs(B[0, iu, idd] - ref) <= REL_TOL * ref_abs


def test_two_cluster_sink_with_a_two_nucleon_cluster(cuda_device):
    """Cluster sink with a multi-nucleon cluster: 3He as (a slice of) the p n cluster at x and a proton at y.
    Block tensors of 3x3 / 2x1 minors over all 220 x 220 / 66 x 12 column subsets, Laplace combination on the host, against the
    oracle's double sum over (x, y) with stacked 5x5 and 4x4 determinants."""
    L, T = 2, 1
    U, D = make_propagators_numpy(8644, L, T)
    Ud, Dd = _dev(U, cuda_device), _dev(D, cuda_device)
    sa = wo.merged_terms([("p", 0), ("n", 0)])[::12]             # 20 of the 231 sink terms: the oracle stays below a minute
    sb = wo.merged_terms([("p", 1)])
    raw = lambda lst: [(c, tuple(("u", x) for x in u) + tuple(("d", x) for x in d)) for (u, d, c) in lst]
    src = wo.merged_from_raw([(c1 * c2, q1 + q2) for (c1, q1) in raw(sa) for (c2, q2) in raw(sb)])   # the product A.B, oracle side
    fl = np.array([[0] * 3 + [1] * 3 for _ in sa], np.uint8)
    chi = np.array([list(u) + list(d) for (u, d, _) in sa], np.uint8)
    a = wk.operator_from_raw(fl, chi, np.array([c for (_, _, c) in sa], complex))
    b = wk.operator_from_nucleons([("p", 1)])
    ab = wk.operator_product(a, b)
    assert ab.n_terms == len(src) and (ab.n_u, ab.n_d) == (5, 4)
    for mom_a, mom_b in (((1, 0, 1), (0, 1, 0)),):
        Cg = wk.two_cluster_correlator(Ud, Dd, a, b, mom_a, mom_b, L, T, source=ab)
        Cr, sabs = wo.two_cluster_correlator(U, D, sa, sb, src, mom_a, mom_b, L)
        assert np.all(np.abs(Cg - Cr) <= REL_TOL * sabs), (np.abs(Cg - Cr) / sabs).max()

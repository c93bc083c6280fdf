"""Host-side tests of the C-ABI library (no GPU): the term builder (steps a1, a2, a2') against the
oracle's own, independently written expansion; error codes; exported symbols; workspace planning."""
import ctypes
import re

import numpy as np
import pytest

import paper_2411_08962_b200 as wk
from oracle import wick_oracle as wo
from wick_inputs import CONFIGS, make_random_term_list

NUCLEI = {k: CONFIGS[k].nucleus for k in ("cfg0", "cfg1", "cfg2", "cfg3", "cfg4")}
# SURVEY.md section 8 structure table (re-derived by the oracle in tests/test_oracle_pins.py)
EXPECT = {
    "cfg0": dict(n_u=2, n_d=1, n_sink=21, rows_u=21, rows_d=12, minors_u=441, minors_d=144),
    "cfg1": dict(n_u=3, n_d=3, n_sink=231, rows_u=121, rows_d=121, minors_u=14641, minors_d=14641),
    "cfg2": dict(n_u=5, n_d=4, n_sink=1311, rows_u=483, rows_d=342, minors_u=233289, minors_d=116964),
    "cfg3": dict(n_u=6, n_d=6, n_sink=2716, rows_u=655, rows_d=655, minors_u=429025, minors_d=429025),
    "cfg4": dict(n_u=10, n_d=11, n_sink=21, rows_u=21, rows_d=12, minors_u=441, minors_d=144),
}


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def test_library_exports_every_declared_symbol():
    lib = wk.load_library()
    with open("include/wick.h") as f:
        header = f.read()
    declared = set(re.findall(r"\b(wick_[a-z_0-9]+)\s*\(", header))
    assert declared == set(wk.EXPORTED_SYMBOLS)
    for name in declared:
        assert getattr(lib, name) is not None
    assert b"sm_100a" in lib.wick_version()


@pytest.mark.parametrize("cfg", ["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
def test_sink_list_matches_oracle_expansion(cfg, golden):
    t = wk.build_terms(NUCLEI[cfg])
    i, e = t.info, EXPECT[cfg]
    assert (i.n_u, i.n_d, i.n_sink, i.n_source) == (e["n_u"], e["n_d"], e["n_sink"], e["n_sink"])
    assert (i.n_rows_u, i.n_cols_u, i.n_rows_d, i.n_cols_d) == (e["rows_u"], e["rows_u"], e["rows_d"], e["rows_d"])
    assert (i.n_minors_u, i.n_minors_d) == (e["minors_u"], e["minors_d"])
    assert i.n_terms == e["n_sink"] ** 2 and i.is_outer_product == 1
    assert i.n_raw == 24 ** len(NUCLEI[cfg])
    if cfg == "cfg3":
        assert i.n_sink == int(golden["he4_terms"])
    ur, uc, dr, dc = t.tuples()
    assert np.array_equal(ur, uc) and np.array_equal(dr, dc)
    for tab in (ur, dr):                                        # ascending tuples in lexicographic order
        assert np.all(np.diff(tab.astype(int), axis=1) > 0)
        as_list = [tuple(r) for r in tab]
        assert as_list == sorted(set(as_list))
    sru, srd, sc, qcu, qcd, qc = t.factors()
    mine = {(tuple(ur[a]), tuple(dr[b])): c for a, b, c in zip(sru, srd, sc)}
    ref = {(u, d): c for u, d, c in wo.merged_terms(NUCLEI[cfg])}
    assert set(mine) == set(ref)
    # the overall sign of C gamma5 is a convention that cancels in c_i conj(c_j): compare up to one global sign
    k0 = next(iter(ref))
    g = mine[k0] / ref[k0]
    assert g in (1, -1)
    assert all(mine[k] == g * ref[k] for k in ref)
    assert np.array_equal(qcu, sru) and np.array_equal(qcd, srd) and np.array_equal(qc, np.conj(sc))


@pytest.mark.parametrize("cfg", ["cfg0", "cfg1"])
def test_flat_terms_consistent_and_site_value_matches_oracle(cfg):
    t = wk.build_terms(NUCLEI[cfg])
    i = t.info
    uid, did, w = t.terms()
    sru, srd, sc, qcu, qcd, qc = t.factors()
    assert np.array_equal(uid, (sru[:, None] * i.n_cols_u + qcu[None, :]).ravel())
    assert np.array_equal(did, (srd[:, None] * i.n_cols_d + qcd[None, :]).ravel())
    assert np.array_equal(w, (sc[:, None] * qc[None, :]).ravel())
    umr, umc, dmr, dmc = t.minors()
    assert np.array_equal(umr, np.repeat(np.arange(i.n_rows_u), i.n_cols_u))
    assert np.array_equal(umc, np.tile(np.arange(i.n_cols_u), i.n_rows_u))
    # evaluate the builder's flat list with the oracle's determinant and compare with the oracle's RAW sum
    rng = np.random.default_rng(21)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    a_u, b_u, a_d, b_d, ww = t.term_tuples()
    got, sabs = wo.site_terms_value(U, D, a_u, b_u, a_d, b_d, ww)
    if cfg == "cfg0":
        raw = wo.nucleus_raw_terms(NUCLEI[cfg])
        ref = wo.raw_site_value(U, D, raw, raw)
    else:
        ref, _ = wo.site_value_outer(U, D, wo.merged_terms(NUCLEI[cfg]))
    assert abs(got - ref) < 1e-12 * sabs


def test_from_list_canonicalisation_signs_and_merging():
    """Raw tuples in any order, with repeats and duplicates: sum_k w_k detU detD over the RAW list
    (oracle, no sorting) must equal the sum over the canonical list the builder returns."""
    rng = np.random.default_rng(22)
    n_u, n_d, n_raw = 4, 3, 300
    a_u = np.array([rng.permutation(12)[:n_u] for _ in range(n_raw)], np.uint8)
    b_u = np.array([rng.permutation(12)[:n_u] for _ in range(n_raw)], np.uint8)
    a_d = np.array([rng.permutation(12)[:n_d] for _ in range(n_raw)], np.uint8)
    b_d = np.array([rng.permutation(12)[:n_d] for _ in range(n_raw)], np.uint8)
    w = _rand(rng, n_raw)
    a_u[5, 1] = a_u[5, 0]                                        # Pauli zeros
    b_d[9, 2] = b_d[9, 0]
    for src, dst in ((20, 21), (30, 31), (30, 32)):              # duplicates, one with permuted rows (sign flips)
        a_u[dst], b_u[dst], a_d[dst], b_d[dst] = a_u[src], b_u[src], a_d[src], b_d[src]
    a_u[31] = a_u[31][[1, 0, 2, 3]]
    w[40] = 0.0
    t = wk.build_terms_from_list(a_u, b_u, a_d, b_d, w)
    i = t.info
    assert i.is_outer_product == 0 and i.n_raw == n_raw
    assert i.n_terms == n_raw - 2 - 3 - 1                        # 2 Pauli zeros, 3 merged duplicates, 1 zero weight
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    ref, sabs = wo.site_terms_value(U, D, a_u, b_u, a_d, b_d, w)
    ca_u, cb_u, ca_d, cb_d, cw = t.term_tuples()
    assert np.all(np.diff(ca_u.astype(int), axis=1) > 0) and np.all(np.diff(cb_d.astype(int), axis=1) > 0)
    got, _ = wo.site_terms_value(U, D, ca_u, cb_u, ca_d, cb_d, cw)
    assert abs(got - ref) < 1e-12 * sabs
    # unique minors: every (row tuple, col tuple) pair appears once
    ur, uc, dr, dc = t.tuples()
    umr, umc, dmr, dmc = t.minors()
    assert len({(a, b) for a, b in zip(umr, umc)}) == i.n_minors_u == len(umr)
    assert len({(a, b) for a, b in zip(dmr, dmc)}) == i.n_minors_d == len(dmr)


def test_cfg4b_random_list_roundtrip():
    c = CONFIGS["cfg4b"]
    a_u, b_u, a_d, b_d, w = make_random_term_list(c.seed, c.n_u, c.n_d, c.n_random_terms)
    t = wk.build_terms_from_list(a_u, b_u, a_d, b_d, w)
    i = t.info
    assert (i.n_u, i.n_d) == (10, 11) and i.n_terms <= 441 and i.n_terms >= 430
    assert i.n_minors_u <= 441 and i.n_minors_d <= 144
    rng = np.random.default_rng(23)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    ref, sabs = wo.site_terms_value(U, D, a_u, b_u, a_d, b_d, w)
    got, _ = wo.site_terms_value(U, D, *t.term_tuples())
    assert abs(got - ref) < 1e-11 * sabs


def test_identity_test_merges_nothing_for_distinct_flavours():
    for cfg in ("cfg0", "cfg1"):
        t = wk.build_terms(NUCLEI[cfg], flags=wk.BUILD_IDENTITY_TEST, seed=7)
        assert t.info.n_identity_merged == 0 and t.info.is_outer_product == 1
        assert t.info.n_terms == EXPECT[cfg]["n_sink"] ** 2


def test_identity_test_isospin_finds_flavour_swap_classes():
    """With U == D (m_u = m_d) products related by exchanging the u and d minors coincide.
    The expected class count is obtained independently: numerical values of all products at a random
    complex point, clustered up to sign."""
    nuc = NUCLEI["cfg1"]
    plain = wk.build_terms(nuc)
    t = wk.build_terms(nuc, flags=wk.BUILD_IDENTITY_TEST | wk.BUILD_ISOSPIN, seed=11)
    rng = np.random.default_rng(24)
    U = _rand(rng, 12, 12)
    a_u, b_u, a_d, b_d, w = plain.term_tuples()
    v = wo.det_elim(U[a_u[:, :, None], b_u[:, None, :]]) * wo.det_elim(U[a_d[:, :, None], b_d[:, None, :]])
    # canonical representative of {v, -v}: the one whose real part is positive; round relative to |v|
    s = np.where(v.real < 0, -1.0, 1.0)
    key = np.round((v * s) / np.abs(v).max() * 1e9).astype(np.complex128)
    n_classes = len(np.unique(key))
    # merged weights that cancel exactly drop out; count the classes whose summed weight is non-zero
    order = np.unique(key, return_inverse=True)[1]
    wsum = np.zeros(n_classes, complex)
    np.add.at(wsum, order, w * s)
    expected = int(np.count_nonzero(np.abs(wsum) > 1e-9))
    assert t.info.n_terms == expected
    assert t.info.n_identity_merged == plain.info.n_terms - expected
    assert expected < plain.info.n_terms and t.info.is_outer_product == 0
    # merged list evaluates to the same number at another U == D point
    U2 = _rand(rng, 12, 12)
    ref, sabs = wo.site_terms_value(U2, U2, a_u, b_u, a_d, b_d, w)
    got, _ = wo.site_terms_value(U2, U2, *t.term_tuples())
    assert abs(got - ref) < 1e-11 * sabs


def test_error_codes():
    with pytest.raises(wk.WickError, match="kind"):
        wk.build_terms([("x", 0)])
    with pytest.raises(wk.WickError, match="gamma"):
        wk.build_terms([("p", 4)])
    with pytest.raises(wk.WickError, match="12 quarks"):
        wk.build_terms([("p", g % 4) for g in range(7)])        # 14 u quarks
    with pytest.raises(wk.WickError, match="n_nucleons"):
        wk.build_terms([])
    bad = np.array([[0, 12]], np.uint8)
    ok = np.array([[0, 1]], np.uint8)
    with pytest.raises(wk.WickError, match=">= 12"):
        wk.build_terms_from_list(bad, ok, ok, ok, np.ones(1, complex))
    lib = wk.load_library()
    assert lib.wick_terms_get_info(None, None) == -1
    assert lib.wick_contract_workspace_bytes(None, 4, 4, 1) == 0
    # p0 p0 vanishes by Pauli: a legal, empty list
    t = wk.build_terms([("p", 0), ("p", 0)])
    assert t.info.n_terms == 0 and t.info.n_sink == 0


def test_workspace_planning():
    t = wk.build_terms(NUCLEI["cfg3"])
    lo = wk.contract_workspace_bytes(t, 32, 64, 1, minimum=True)
    hi = wk.contract_workspace_bytes(t, 32, 64, 1)
    per_site = (429025 * 2) * 16
    assert lo >= 32 * per_site + 64 * 32768 * 16
    assert lo < hi <= (2 << 30) + 64 * 32768 * 16 + 4096
    t0 = wk.build_terms(NUCLEI["cfg0"])
    assert wk.contract_workspace_bytes(t0, 4, 8, 1) >= 512 * 585 * 16


# ---------------------------------------------------------------------------------------------
# schedule of the staged factorised reduction (host logic of contract.cu, no GPU needed)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("cfg", ["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
@pytest.mark.parametrize("n_bins", [1, 2, 37, 74])
def test_staged_schedule_covers_every_pair_once(cfg, n_bins):
    t = wk.build_terms(CONFIGS[cfg].nucleus)
    i = t.info
    batches, pairs, max_md, max_rows = t.staged_schedule_check(n_bins)   # raises if a pair is missed / doubled / out of range
    assert pairs == i.n_rows_u * i.n_cols_d
    assert 1 <= batches and 1 <= max_md <= 184 and 1 <= max_rows <= 184


def test_staged_schedule_rejects_generic_lists():
    c = CONFIGS["cfg4b"]
    t = wk.build_terms_from_list(*make_random_term_list(c.seed, c.n_u, c.n_d, c.n_random_terms))
    with pytest.raises(wk.WickError):
        t.staged_schedule_check(4)


# ---------------------------------------------------------------------------------------------
# order in which the minors kernel walks the unique minors (host logic of contract.cu)
# ---------------------------------------------------------------------------------------------

def _perm_is_odd(p):
    p = list(p)
    return sum(1 for i in range(len(p)) for j in range(i + 1, len(p)) if p[i] > p[j]) % 2 == 1


@pytest.mark.parametrize("cfg", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg4b"])
def test_minor_order_is_a_signed_permutation(cfg):
    c = CONFIGS[cfg]
    t = (wk.build_terms_from_list(*make_random_term_list(c.seed, c.n_u, c.n_d, c.n_random_terms)) if c.random_list
         else wk.build_terms(c.nucleus))
    rows_cols = t.tuples()
    minors = t.minors()
    for fl in (0, 1):
        mid, pc, neg = t.minor_order(fl)
        cols, mcol, mrow = rows_cols[2 * fl + 1], minors[2 * fl + 1], minors[2 * fl]
        assert sorted(mid.tolist()) == list(range(len(mid)))                 # every unique minor exactly once
        asc = cols[mcol[mid]]
        assert np.array_equal(np.sort(pc, axis=1), asc)                      # same index set, some order
        assert [bool(x) for x in neg] == [_perm_is_odd(p) for p in pc.tolist()]
        assert np.all(np.diff(mrow[mid]) >= 0)                               # row tuple by row tuple
        if pc.shape[1] <= 8:                                                 # small minors: minor order, ascending columns
            assert np.array_equal(mid, np.arange(len(mid))) and not neg.any()


# ---------------------------------------------------------------------------------------------
# isospin limit U == D: factorised swap symmetrisation and the merged flat list
# ---------------------------------------------------------------------------------------------

def test_isospin_counts_of_the_deuteron():
    """with U == D the identity test collapses the deuteron's 53 361 products to 26 721 and both
    flavours share one table of 14 641 minors; the factorised symmetrisation keeps 120 of the 231 sink terms."""
    nuc = NUCLEI["cfg1"]
    merged = wk.build_terms(nuc, flags=wk.BUILD_IDENTITY_TEST | wk.BUILD_ISOSPIN, seed=3)
    assert merged.info.n_terms == 26721 and merged.info.is_outer_product == 0
    assert merged.info.n_minors_u == 14641 and merged.info.n_minors_d == 14641
    ur, uc, dr, dc = merged.tuples()
    assert np.array_equal(ur, dr) and np.array_equal(uc, dc)                 # one table serves both flavours
    half = wk.build_terms(nuc, flags=wk.BUILD_ISOSPIN)
    assert half.info.is_outer_product == 1 and half.info.n_sink == 120 and half.info.n_source == 231
    assert half.info.n_terms == 120 * 231
    # (231 + 9 self-conjugate sink terms) / 2 = 120; the minimal count differs only by the 9 x 111 products that pair a
    # self-conjugate sink term with both members of a source pair
    assert 120 * 231 - 26721 == 9 * 111


@pytest.mark.parametrize("cfg", ["cfg1", "cfg3"])
def test_isospin_symmetrised_list_equals_the_full_list_at_u_equals_d(cfg):
    nuc = NUCLEI[cfg]
    full, half = wk.build_terms(nuc), wk.build_terms(nuc, flags=wk.BUILD_ISOSPIN)
    assert half.info.n_sink < full.info.n_sink and half.info.n_source == full.info.n_source
    rng = np.random.default_rng(31)
    U = _rand(rng, 12, 12)
    ur, uc, dr, dc = full.tuples()

    def value(t):
        sru, srd, sc, qcu, qcd, qc = t.factors()
        MU = wo.det_elim(U[ur[:, None, :, None], uc[None, :, None, :]])      # [row tuple][column tuple], U == D
        MD = wo.det_elim(U[dr[:, None, :, None], dc[None, :, None, :]])
        tot, tot_abs = 0.0, 0.0
        for i in range(len(sc)):
            v = sc[i] * qc * MU[sru[i], qcu] * MD[srd[i], qcd]
            tot += v.sum()
            tot_abs += np.abs(v).sum()
        return tot, tot_abs
    a, sabs = value(full)
    b, _ = value(half)
    assert abs(a - b) <= 1e-12 * sabs
    # the symmetrisation is only valid for U == D and must not be applied silently otherwise
    assert wk.build_terms(NUCLEI["cfg2"], flags=wk.BUILD_ISOSPIN).info.n_sink == wk.build_terms(NUCLEI["cfg2"]).info.n_sink


# ---------------------------------------------------------------------------------------------
# general interpolators and correlation matrices (GEVP, Sec. V)
# ---------------------------------------------------------------------------------------------

def _as_list(op):
    u, d, c = op.terms()
    return sorted((tuple(int(x) for x in a), tuple(int(x) for x in b), complex(z)) for a, b, z in zip(u, d, c))


def test_paper_operators_match_the_oracle_and_the_printed_counts(golden):
    """Eq. (20) and Eq. (21) in the builder: the printed 356 / 1026 terms (Table II, :305-306) and,
    monomial by monomial, the oracle's independent expansion."""
    d = wk.operator_paper(wk.OP_DEUTERON_EQ20)
    assert (d.n_u, d.n_d, d.n_terms) == (3, 3, int(golden["h2_terms_eq20"]))
    assert _as_list(d) == [(u, dd, complex(c)) for u, dd, c in wo.merged_from_raw(wo.deuteron_eq20_raw_terms())]
    for J in (2, 3):
        h = wk.operator_paper(wk.OP_HELIUM3_EQ21, J)
        assert (h.n_u, h.n_d, h.n_terms) == (5, 4, int(golden["he3_terms_eq21"]))
        assert _as_list(h) == [(u, dd, complex(c)) for u, dd, c in wo.merged_from_raw(wo.helium3_eq21_raw_terms(J))]
    assert wk.operator_paper(wk.OP_HELIUM3_EQ21, 0).n_terms == 744       # J in the projector's own sector: not the paper's count
    with pytest.raises(wk.WickError):
        wk.operator_paper(7)


def test_operator_from_raw_and_from_nucleons_agree():
    nuc = NUCLEI["cfg1"]
    raw = wo.nucleus_raw_terms(nuc)
    fl = np.array([[0 if f == "u" else 1 for f, _ in q] for _, q in raw], np.uint8)
    chi = np.array([[x for _, x in q] for _, q in raw], np.uint8)
    coef = np.array([c for c, _ in raw], complex)
    a, b = wk.operator_from_raw(fl, chi, coef), wk.operator_from_nucleons(nuc)
    assert _as_list(a) == _as_list(b) == [(u, d, complex(c)) for u, d, c in wo.merged_terms(nuc)]
    with pytest.raises(wk.WickError, match="quark content"):
        wk.operator_from_raw(np.array([[0, 0], [0, 1]], np.uint8), np.array([[0, 1], [0, 1]], np.uint8), np.ones(2, complex))


def test_terms_matrix_shares_one_pair_of_minor_tables():
    ops = [wk.operator_from_nucleons(NUCLEI["cfg1"]), wk.operator_paper(wk.OP_DEUTERON_EQ20)]
    m = wk.build_terms_matrix(ops)
    tup = [m[k][kp].tuples() for k in range(2) for kp in range(2)]
    for other in tup[1:]:
        assert all(np.array_equal(x, y) for x, y in zip(tup[0], other))
    assert [[m[k][kp].info.n_terms for kp in range(2)] for k in range(2)] == [[231 * 231, 231 * 356], [356 * 231, 356 * 356]]
    assert all(m[k][kp].info.is_outer_product == 1 for k in range(2) for kp in range(2))
    # the diagonal entry of the product operator evaluates like the plain handle
    rng = np.random.default_rng(41)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    ref, sabs = wo.site_terms_value(U, D, *wk.build_terms(NUCLEI["cfg1"]).term_tuples())
    got, _ = wo.site_terms_value(U, D, *m[0][0].term_tuples())
    assert abs(got - ref) <= 1e-12 * sabs
    # an off-diagonal entry against the oracle's own sink x conj(source) expansion
    sink, src = wo.merged_terms(NUCLEI["cfg1"]), wo.merged_from_raw(wo.deuteron_eq20_raw_terms())
    ref, sabs = wo.site_value_outer(U, D, sink, src)
    got, _ = wo.site_terms_value(U, D, *m[0][1].term_tuples())
    assert abs(got - ref) <= 1e-12 * sabs


# ---------------------------------------------------------------------------------------------
# cluster sinks: host combination of block tensors (Eq. 6-8)
# ---------------------------------------------------------------------------------------------

def test_cluster_combination_on_one_site_equals_the_point_sink():
    """With one lattice site the block tensors are plain sums over sink terms of products of minors (computed here with the
    oracle's determinant), and the combination must return the point-sink value of the product operator."""
    import itertools
    rng = np.random.default_rng(52)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    a, b = wk.operator_from_nucleons([("p", 0)]), wk.operator_from_nucleons([("n", 1)])
    ab = wk.operator_product(a, b)
    assert _as_list(ab) == [(u, d, complex(c)) for u, d, c in wo.merged_terms([("p", 0), ("n", 1)])]

    def block(op):
        u, d, c = op.terms()
        cu = np.array(list(itertools.combinations(range(12), op.n_u)), np.intp)
        cd = np.array(list(itertools.combinations(range(12), op.n_d)), np.intp)
        B = np.zeros((1, len(cu), len(cd)), complex)
        for ui, di, ci in zip(u.astype(np.intp), d.astype(np.intp), c):
            mu = wo.det_elim(U[ui[None, :, None], cu[:, None, :]])
            md = wo.det_elim(D[di[None, :, None], cd[:, None, :]])
            B[0] += ci * mu[:, None] * md[None, :]
        return B
    got = wk.combine_two_clusters(a, b, ab, block(a), block(b))
    ref, sabs = wo.site_value_outer(U, D, wo.merged_terms([("p", 0), ("n", 1)]))
    assert abs(got[0] - ref) <= 1e-12 * sabs
    # a two-nucleon cluster next to a nucleon (3He as deuteron + proton): same identity
    a2 = wk.operator_from_nucleons([("p", 0), ("n", 0)])
    b2 = wk.operator_from_nucleons([("p", 1)])
    got = wk.combine_two_clusters(a2, b2, wk.operator_product(a2, b2), block(a2), block(b2))
    ref, sabs = wo.site_value_outer(U, D, wo.merged_terms([("p", 0), ("n", 0), ("p", 1)]))
    assert abs(got[0] - ref) <= 1e-12 * sabs
    with pytest.raises(wk.WickError, match="quark content"):
        wk.combine_two_clusters(a, b, a, block(a), block(b))


# ---------------------------------------------------------------------------------------------
# measurement helpers of bench.py (host logic only)
# ---------------------------------------------------------------------------------------------

def test_bench_executed_flop_model_and_traffic_key(tmp_path, monkeypatch):
    import json

    import bench
    t = wk.build_terms(NUCLEI["cfg3"])
    ur, uc, dr, dc = t.tuples()
    mu_row = t.minors()[0]
    mid, pc, _ = t.minor_order(0)
    f = bench.executed_flops_per_site(6, mu_row[mid], pc, uc)
    # per row tuple: 12 instances (two pivot steps each) + 91 Schur columns + 96 pair nodes + 296 third nodes + 655 Laplace sums
    per_row = 12 * (6 + 14 + 30 + (40 + 5 + 14 + 24 + 6)) + 91 * 72 + 96 * 108 + 296 * 88 + 655 * 30
    assert f == per_row * 655 and 95 < f / 429025 < 100
    assert f < 429025 * bench.flops_lu(6) / 6                   # far below one full LU per minor: never report that as a rate
    # the committed ncu traffic only counts for the kernel sources it was measured on
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    (tmp_path / "profiles").mkdir()
    (tmp_path / "paper_2411_08962_b200" / "csrc").mkdir(parents=True)
    (tmp_path / "paper_2411_08962_b200" / "csrc" / "k.cu").write_text("// kernel\n")
    rec = {"kernel_source_hash": bench.kernel_source_hash(), "command": "ncu", "workloads": {"x": {"minors_dram_bytes_per_launch": 5}}}
    (tmp_path / "profiles" / "r02_roofline_traffic.json.txt").write_text(json.dumps(rec))
    assert bench.read_traffic("x")[0] == {"minors_dram_bytes_per_launch": 5}
    (tmp_path / "paper_2411_08962_b200" / "csrc" / "k.cu").write_text("// kernel, edited\n")
    got, why = bench.read_traffic("x")
    assert got is None and "stale" in why

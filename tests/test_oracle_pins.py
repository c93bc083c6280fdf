"""Pins for the oracle's operator algebra and correlator (oracle.wick_oracle) against things other
than itself (tier rule: "pin it to something other than itself"):

  * brute-force Wick contraction: explicit sum over ALL pairings with permutation signs
    (Eq. 11; N_perm = n_u! n_d! non-zero ones);
  * RAW (no sorting, no merging) == MERGED (canonical order with sign, Eq. 19);
  * source-side colour rotation U,D -> U (1_4 x Omega), D (1_4 x Omega), Omega in SU(3);
  * Pauli zeros (repeated index);
  * the textbook proton direct-minus-exchange contraction written as an einsum
    (Eq. 31 PAPER.md:357 and Eq. B1);
  * identity / diagonal propagators (closed forms);
  * the paper's printed term count 2716 for 4He and N_perm;
  * site-scaled propagators and time scaling (full-pipeline closed forms incl. momentum phases).
"""
import itertools
import math

import numpy as np
import pytest

from oracle import wick_oracle as wo

P0 = (("p", 0),)
DEUT = (("p", 0), ("n", 0))
HE3 = (("p", 0), ("p", 1), ("n", 0))
HE4 = (("p", 0), ("p", 1), ("n", 0), ("n", 1))
LI7 = (("p", 0), ("p", 1), ("p", 2), ("n", 0), ("n", 1), ("n", 2), ("n", 3))


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _su3(rng):
    """Random SU(3): QR of a complex Gaussian, phases fixed, determinant normalised to 1."""
    q, r = np.linalg.qr(_rand(rng, 3, 3))
    q = q * (np.diag(r) / np.abs(np.diag(r)))[None, :]
    q = q / np.linalg.det(q) ** (1.0 / 3.0)
    assert np.allclose(q.conj().T @ q, np.eye(3)) and abs(np.linalg.det(q) - 1) < 1e-12
    return q


def _merged_site(U, D, nucleus):
    sink = wo.merged_terms(nucleus)
    return wo.site_value_outer(U, D, sink)


# ------------------------------------------------------------------------------------------
# operator algebra
# ------------------------------------------------------------------------------------------

def test_cgamma5_structure():
    """C gamma5 with C = gamma4 gamma2 is real, antisymmetric, block diagonal."""
    m = wo.c_gamma5()
    assert np.array_equal(m, -m.T)
    assert np.count_nonzero(m) == 4
    assert m[0, 1] != 0 and m[2, 3] != 0 and m[0, 1] == -m[1, 0] and m[2, 3] == -m[3, 2]
    g1, g2, g3, g4, g5 = wo.gamma_matrices()
    for a, b in itertools.combinations((g1, g2, g3, g4), 2):
        assert np.allclose(a @ b + b @ a, 0)                 # Clifford algebra
    for g in (g1, g2, g3, g4, g5):
        assert np.allclose(g @ g, np.eye(4)) and np.allclose(g, g.conj().T)
    assert np.allclose(g5, np.array([[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]]) * g5[0, 2])


def test_levi_civita():
    e = wo.levi_civita()
    assert e[0, 1, 2] == 1 and e[1, 0, 2] == -1 and e[2, 0, 1] == 1 and e[0, 0, 1] == 0
    assert np.sum(np.abs(e)) == 6
    # eps_abc eps_abd = 2 delta_cd
    assert np.allclose(np.einsum("abc,abd->cd", e, e), 2 * np.eye(3))


def test_raw_term_counts():
    assert len(wo.nucleon_raw_terms("p", 0)) == 24
    assert len(wo.nucleon_raw_terms("n", 1)) == 24
    assert len(wo.nucleus_raw_terms(DEUT)) == 576            # 24^A, SURVEY 8 table


@pytest.mark.parametrize("nucleus,n_sink,sumsq", [
    (P0, 21, 30), (DEUT, 231, 1080), (HE3, 1311, 43200), (HE4, 2716, 1814400),
])
def test_merged_term_counts(nucleus, n_sink, sumsq, golden):
    """2716 is the paper's printed 4He count (tests/golden/paper_values.txt)."""
    sink = wo.merged_terms(nucleus)
    assert len(sink) == n_sink
    if nucleus is HE4:
        assert len(sink) == int(golden["he4_terms"])
    c = np.array([t[2] for t in sink])
    assert np.all(c.imag == 0) and np.all(c.real == np.round(c.real))
    assert np.sum(c.real ** 2) == sumsq
    for u, d, _ in sink:
        assert list(u) == sorted(set(u)) and list(d) == sorted(set(d))


def test_li7_hole_dual_of_proton():
    """cfg 4: p0 p1 p2 n0 n1 n2 n3 does not cancel: 21 terms, 10 u + 11 d indices each."""
    sink = wo.merged_terms(LI7)
    assert len(sink) == 21
    assert all(len(u) == 10 and len(d) == 11 for u, d, _ in sink)
    c = np.array([t[2] for t in sink]).real
    assert np.sum(c ** 2) == 109734912000
    assert len({u for u, _, _ in sink}) == 21 and len({d for _, d, _ in sink}) == 12


def test_nperm_values(golden):
    assert math.factorial(3) * math.factorial(3) == golden["nperm_h2"]
    assert math.factorial(5) * math.factorial(4) == golden["nperm_he3"]
    assert math.factorial(6) * math.factorial(6) == golden["nperm_he4"]
    assert 6 ** 4 * 4 ** 4 == golden["nloop_h2"]


def test_paper_cost_ratio_and_identity_bound(golden):
    ratio = 2 * 1026 ** 2 * (120 + 24) / (356 ** 2 * (6 + 6))
    assert abs(ratio - golden["cost_ratio_he3_h2"]) < 1.0                      # "approx 200"
    bound = wo.identity_test_error_bound(24.0 ** 12, 18, 360.0, 40)
    assert abs(bound / golden["idtest_bound_c12"] - 1) < 0.02


# ------------------------------------------------------------------------------------------
# brute force Wick sums and RAW == MERGED
# ------------------------------------------------------------------------------------------

def test_proton_brute_force_all_pairings():
    """Eq. 11 literally: all 3! pairings of the 3x3 flavour-block matrix for every raw term pair
    (only n_u! n_d! = 2 are non-zero); compared with the determinant form and with MERGED."""
    rng = np.random.default_rng(1)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    raw = wo.nucleus_raw_terms(P0)
    brute = wo.raw_site_value(U, D, raw, raw, use_leibniz=True)
    det = wo.raw_site_value(U, D, raw, raw)
    merged, sabs = _merged_site(U, D, P0)
    assert abs(brute - det) < 1e-12 * sabs
    assert abs(brute - merged) < 1e-12 * sabs


def test_deuteron_raw_equals_merged_and_brute_force_sample():
    rng = np.random.default_rng(2)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    raw = wo.nucleus_raw_terms(DEUT)
    merged, sabs = _merged_site(U, D, DEUT)
    # RAW over all 576^2 pairs is ~3e5 6x6 determinants: vectorise through det_elim in chunks
    coef = np.array([c for c, _ in raw])
    # build the flavour-block matrices with index arithmetic (row = sink quark, col = source quark)
    fl = np.array([[0 if f == "u" else 1 for f, _ in q] for _, q in raw])          # [576][6]
    ch = np.array([[c for _, c in q] for _, q in raw])                              # [576][6]
    S = np.stack([U, D])                                                            # [2][12][12]
    total = 0.0
    for i in range(len(raw)):
        same = fl[i][None, :, None] == fl[:, None, :]                               # [576][6][6]
        M = np.where(same, S[fl[i][None, :, None], ch[i][None, :, None], ch[:, None, :]], 0.0)
        total += coef[i] * np.sum(np.conj(coef) * wo.det_elim(M))
    assert abs(total - merged) < 1e-11 * sabs
    # explicit 6! = 720 pairings (36 non-zero) on a seeded sample of raw term pairs
    pick = rng.choice(len(raw), size=(6, 2))
    for i, j in pick:
        M = wo.wick_matrix(U, D, raw[i][1], raw[j][1])
        assert abs(wo.det_leibniz(M) - wo.det_elim(M)) < 1e-11 * max(1.0, abs(wo.det_elim(M)))


def test_flavour_factorisation_sign_he3_sample():
    """Eq. 12-15: the full (n_u+n_d) x (n_u+n_d) Wick determinant of a raw term pair equals
    sign * det(U block) * det(D block) with the sign of regrouping (u..., d...) at sink and source.
    Checked on 3He raw terms (9 quarks) with LAPACK as the full determinant."""
    rng = np.random.default_rng(3)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    nuc = [wo.nucleon_raw_terms(k, g) for k, g in HE3]
    for _ in range(20):
        ti = [n[rng.integers(24)] for n in nuc]
        tj = [n[rng.integers(24)] for n in nuc]
        qi = sum((t[1] for t in ti), ())
        qj = sum((t[1] for t in tj), ())
        full = np.linalg.det(wo.wick_matrix(U, D, qi, qj))
        si, ui, di = wo.canonical_monomial(qi)
        sj, uj, dj = wo.canonical_monomial(qj)
        if si == 0 or sj == 0:
            assert abs(full) < 1e-9
            continue
        fact = si * sj * wo.det_elim(U[np.ix_(ui, uj)]) * wo.det_elim(D[np.ix_(di, dj)])
        assert abs(full - fact) < 1e-10 * max(1.0, abs(fact))


def test_he4_single_terms_brute_force_pairings():
    """A handful of 4He merged terms: det(6x6) det(6x6) against the explicit n_u! n_d! = 518400-term
    pairing sum, done as (sum over 720 u pairings) x (sum over 720 d pairings)."""
    rng = np.random.default_rng(4)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    sink = wo.merged_terms(HE4)
    for k in rng.choice(len(sink), 3, replace=False):
        (au, ad, _), (bu, bd, _) = sink[k], sink[(k * 7 + 11) % len(sink)]
        lu = wo.det_leibniz(U[np.ix_(au, bu)])
        ld = wo.det_leibniz(D[np.ix_(ad, bd)])
        eu = wo.det_elim(U[np.ix_(au, bu)])
        ed = wo.det_elim(D[np.ix_(ad, bd)])
        assert abs(lu * ld - eu * ed) < 1e-11 * abs(lu * ld)


# ------------------------------------------------------------------------------------------
# invariances and special cases
# ------------------------------------------------------------------------------------------

@pytest.mark.parametrize("nucleus", [P0, DEUT])
def test_source_colour_rotation_invariance(nucleus):
    rng = np.random.default_rng(5)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    Om = np.kron(np.eye(4), _su3(rng))                      # chi = 3*spin + colour: 1_4 (x) Omega
    base, sabs = _merged_site(U, D, nucleus)
    rot, _ = _merged_site(U @ Om, D @ Om, nucleus)
    assert abs(rot - base) < 1e-12 * sabs
    only_u, _ = _merged_site(U @ Om, D, nucleus)            # negative control: rotating one flavour breaks it
    assert abs(only_u - base) > 1e-6 * sabs
    # sink-side rotation is an invariance too
    rot2, _ = _merged_site(Om @ U, Om @ D, nucleus)
    assert abs(rot2 - base) < 1e-12 * sabs


def test_pauli_zeros():
    rng = np.random.default_rng(6)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    # repeated row index or repeated column index: determinant vanishes identically
    v, s = wo.site_terms_value(U, D, [[1, 1, 5]], [[0, 2, 3]], [[4]], [[7]], [1.0])
    assert abs(v) < 1e-13 * max(s, 1.0)
    v, s = wo.site_terms_value(U, D, [[1, 2, 5]], [[3, 2, 3]], [[4]], [[7]], [1.0])
    assert abs(v) < 1e-13 * max(s, 1.0)
    assert wo.canonical_monomial((("u", 3), ("d", 1), ("u", 3)))[0] == 0
    # p_0 p_0 = 0 (same nucleon twice is Pauli blocked at a point)
    assert wo.merged_terms((("p", 0), ("p", 0))) == []


def test_proton_direct_minus_exchange_einsum():
    """Eq. 31 / B1: N_alpha = eps_ijk C_{beta gamma} u_{i alpha} u_{j beta} d_{k gamma},
    G = eps eps' C C' [ S_u(i a; i' a') S_u(j b; j' b') - S_u(i a; j' b') S_u(j b; i' a') ] S_d(k g; k' g').
    eps, C gamma5 typed in here by hand (not taken from the oracle)."""
    rng = np.random.default_rng(7)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    eps = np.zeros((3, 3, 3))
    eps[0, 1, 2] = eps[1, 2, 0] = eps[2, 0, 1] = 1
    eps[0, 2, 1] = eps[2, 1, 0] = eps[1, 0, 2] = -1
    C = np.zeros((4, 4))
    C[0, 1], C[1, 0], C[2, 3], C[3, 2] = 1, -1, 1, -1       # C gamma5 up to the overall sign (enters twice)
    U4 = U.reshape(4, 3, 4, 3)                               # [spin, colour, spin', colour']
    D4 = D.reshape(4, 3, 4, 3)
    for alpha in (0, 1):
        direct = np.einsum("ijk,bg,lmn,de,il,bjdm,gken->", eps, C, eps, C,
                           U4[alpha, :, alpha, :], U4, D4)
        exch = np.einsum("ijk,bg,lmn,de,idm,bjl,gken->", eps, C, eps, C,
                         U4[alpha, :, :, :], U4[:, :, alpha, :], D4)
        ref = direct - exch
        got, sabs = _merged_site(U, D, (("p", alpha),))
        assert abs(got - ref) < 1e-12 * sabs


@pytest.mark.parametrize("nucleus,sumsq", [(P0, 30), (DEUT, 1080), (HE3, 43200)])
def test_identity_and_diagonal_propagators(nucleus, sumsq):
    eye = np.eye(12, dtype=complex)
    got, _ = _merged_site(eye, eye, nucleus)
    assert abs(got - sumsq) < 1e-9
    rng = np.random.default_rng(8)
    lam, mu = _rand(rng, 12), _rand(rng, 12)
    got, sabs = _merged_site(np.diag(lam), np.diag(mu), nucleus)
    ref = sum(abs(c) ** 2 * np.prod(lam[list(u)]) * np.prod(mu[list(d)]) for u, d, c in wo.merged_terms(nucleus))
    assert abs(got - ref) < 1e-12 * max(sabs, abs(ref))


def test_li7_identity_propagator_and_jacobi_site_value():
    """cfg 4 end to end without any LU of a 10x10/11x11 minor on the reference side: every minor via
    Jacobi's complementary-minor identity from one LAPACK inverse per flavour."""
    rng = np.random.default_rng(9)
    U, D = _rand(rng, 12, 12), _rand(rng, 12, 12)
    sink = wo.merged_terms(LI7)
    got, sabs = wo.site_value_outer(U, D, sink)
    Ui, Di, dU, dD = np.linalg.inv(U), np.linalg.inv(D), np.linalg.det(U), np.linalg.det(D)

    def jac(A_inv, dA, I, J):
        Ic = [k for k in range(12) if k not in I]
        Jc = [k for k in range(12) if k not in J]
        comp = A_inv[np.ix_(Jc, Ic)]
        small = comp[0, 0] if len(Ic) == 1 else comp[0, 0] * comp[1, 1] - comp[0, 1] * comp[1, 0]
        return (-1) ** (sum(I) + sum(J)) * dA * small

    ref = 0.0
    for au, ad, ci in sink:
        for bu, bd, cj in sink:
            ref += ci * np.conj(cj) * jac(Ui, dU, au, bu) * jac(Di, dD, ad, bd)
    assert abs(got - ref) < 1e-9 * sabs
    eye = np.eye(12, dtype=complex)
    got, _ = wo.site_value_outer(eye, eye, sink)
    assert abs(got - 109734912000) < 1e-3


# ------------------------------------------------------------------------------------------
# full pipeline: sites, momentum phases, timeslices
# ------------------------------------------------------------------------------------------

def test_momentum_phases_exact_points():
    ph = wo.momentum_phases(4, [(0, 0, 0), (1, 0, 0), (0, 1, 1)])
    assert np.all(ph[0] == 1)
    s = np.arange(64)
    x, y, z = s % 4, (s // 4) % 4, s // 16
    assert np.allclose(ph[1], (1j) ** x)
    assert np.allclose(ph[2], (1j) ** ((y + z) % 4))
    assert abs(np.sum(ph[1])) < 1e-12                        # plane wave sums to zero over the lattice


def test_site_scaled_propagators_and_time_scaling():
    """U_x = s_x U0, D_x = r_x D0  =>  sigma(x) = s_x^{n_u} r_x^{n_d} sigma0; with
    s_x = exp(-i p.x / n_u), r_x = 1 the projection at momentum p returns L^3 sigma0 and 0 elsewhere.
    Scaling U,D by exp(-t/2) scales C(t) by exp(-(n_u+n_d) t/2)."""
    L, T = 2, 3
    rng = np.random.default_rng(10)
    U0, D0 = _rand(rng, 12, 12), _rand(rng, 12, 12)
    sink = wo.merged_terms(P0)
    a_u, b_u, a_d, b_d, w = wo.outer_product_term_arrays(sink)
    sigma0, _ = wo.site_terms_value(U0, D0, a_u, b_u, a_d, b_d, w)
    mom = [(0, 0, 0), (1, 0, 0), (1, 1, 0)]
    p = np.array([1, 1, 0])
    s = np.arange(L ** 3)
    xyz = np.stack([s % L, (s // L) % L, s // (L * L)], axis=1)
    sx = np.exp(-2j * np.pi * (xyz @ p) / L / 2)             # n_u = 2
    U = np.stack([U0[None] * sx[:, None, None] * np.exp(-0.5 * t) for t in range(T)])
    D = np.stack([np.broadcast_to(D0, (L ** 3, 12, 12)) * np.exp(-0.5 * t) for t in range(T)])
    C, sigma, sabs = wo.correlator_from_terms(U, D, a_u, b_u, a_d, b_d, w, mom, L)
    for t in range(T):
        sc = np.exp(-1.5 * t)
        assert abs(C[2, t] - L ** 3 * sigma0 * sc) < 1e-11 * sabs[t]
        assert abs(C[0, t]) < 1e-11 * sabs[t] and abs(C[1, t]) < 1e-11 * sabs[t]
    assert np.allclose(wo.reduce_sites(sigma, mom, L), C)


def test_correlator_nucleus_matches_site_loop():
    L, T = 2, 2
    rng = np.random.default_rng(11)
    U, D = _rand(rng, T, L ** 3, 12, 12), _rand(rng, T, L ** 3, 12, 12)
    C, sigma, sabs = wo.correlator_nucleus(U, D, P0, [(0, 0, 0)], L)
    sink = wo.merged_terms(P0)
    for t in range(T):
        tot = sum(wo.site_value_outer(U[t, s], D[t, s], sink)[0] for s in range(L ** 3))
        assert abs(C[0, t] - tot) < 1e-12 * sabs[t]


def test_method_b_equals_method_a():
    """site_value_method_b (every distinct minor once per site) against site_value_outer (two fresh
    determinants per term, :279-292) and, for the proton, against the explicit pairing sum of the RAW list."""
    rng = np.random.default_rng(5)
    U = rng.standard_normal((12, 12)) + 1j * rng.standard_normal((12, 12))
    D = rng.standard_normal((12, 12)) + 1j * rng.standard_normal((12, 12))
    for nucleus in ([("p", 0)], [("p", 0), ("n", 0)], [("p", 0), ("p", 1), ("n", 0)]):
        sink = wo.merged_terms(nucleus)
        a, sabs = wo.site_value_outer(U, D, sink)
        b, sabs_b = wo.site_value_method_b(U, D, sink)
        assert abs(a - b) <= 1e-13 * sabs and abs(sabs - sabs_b) <= 1e-12 * sabs
    raw = wo.nucleus_raw_terms([("p", 0)])
    b, sabs_p = wo.site_value_method_b(U, D, wo.merged_terms([("p", 0)]))
    assert abs(b - wo.raw_site_value(U, D, raw, raw, use_leibniz=True)) <= 1e-12 * sabs_p


def test_paper_operators_reproduce_the_printed_term_counts(golden):
    """Table II: 356 terms in the 2H operator of Eq. (20), 1026 per spin component in the 3He operator
    of Eq. (21).  The Eq. (4) proton is the BASELINE proton (same monomials, same coefficients): moving u^a_alpha behind
    the diquark is an even permutation and eps is cyclic."""
    assert len(wo.merged_from_raw(wo.deuteron_eq20_raw_terms())) == int(golden["h2_terms_eq20"]) == 356
    for J in (2, 3):
        assert len(wo.merged_from_raw(wo.helium3_eq21_raw_terms(J))) == int(golden["he3_terms_eq21"]) == 1026
    for kind in ("p", "n"):
        for alpha in range(4):
            assert wo.merged_from_raw(wo.paper_nucleon_raw_terms(kind, alpha)) == wo.merged_terms([(kind, alpha)])
    # merged_from_raw is the same normal form as the nucleon-by-nucleon merge
    assert wo.merged_from_raw(wo.nucleus_raw_terms([("p", 0), ("n", 0)])) == wo.merged_terms([("p", 0), ("n", 0)])
    # projectors: P+ + P- = 1, so the projected nucleons add up to the plain one
    plus, minus = wo.paper_nucleon_raw_terms("p", 1, +1), wo.paper_nucleon_raw_terms("p", 1, -1)
    assert wo.merged_from_raw(plus + minus) == wo.merged_terms([("p", 1)])


def test_deuteron_eq20_against_the_pairing_sum():
    """Eq. (20) correlator at one site: determinant form over the merged 356-term list against the explicit sum over all
    pairings of the RAW 1152-term list on a slice (Eq. 11)."""
    rng = np.random.default_rng(12)
    U = rng.standard_normal((12, 12)) + 1j * rng.standard_normal((12, 12))
    D = rng.standard_normal((12, 12)) + 1j * rng.standard_normal((12, 12))
    raw = wo.deuteron_eq20_raw_terms()
    sink = wo.merged_from_raw(raw)
    full, sabs = wo.site_value_outer(U, D, sink)
    # raw x raw with the full flavour-block determinant (no sorting, no merging): 1152^2 6x6 determinants
    vals = 0.0
    src_q = [q for _, q in raw]
    cj = np.conj(np.array([c for c, _ in raw]))
    for ci, qi in raw[::16]:                                   # a slice of the sink side, all of the source side
        M = np.stack([wo.wick_matrix(U, D, qi, qj) for qj in src_q])
        vals += ci * np.sum(cj * wo.det_elim(M))
    part_sink = wo.merged_from_raw(raw[::16])
    part, _ = wo.site_value_outer(U, D, part_sink, sink)
    assert abs(vals - part) <= 1e-11 * sabs
    assert abs(full) > 0


def test_two_cluster_value_reduces_to_the_point_sink_and_to_the_pairing_sum():
    """Cluster sinks: with both clusters at the SAME site the two-cluster value is the point-sink value of the
    product operator (a pinned function); with different sites it equals the explicit sum over all pairings (Eq. 11,
    PAPER.md:159) in which every sink quark takes its propagator row from its own cluster's site."""
    rng = np.random.default_rng(77)
    Ux, Dx, Uy, Dy = (rng.standard_normal((12, 12)) + 1j * rng.standard_normal((12, 12)) for _ in range(4))
    p, n = wo.merged_terms([("p", 0)]), wo.merged_terms([("n", 0)])
    pn = wo.merged_terms([("p", 0), ("n", 0)])
    same, sabs = wo.two_cluster_site_pair_value(Ux, Dx, Ux, Dx, p, n, pn)
    ref, _ = wo.site_value_outer(Ux, Dx, pn)
    assert abs(same - ref) <= 1e-12 * sabs
    # different sites: RAW proton x RAW neutron at the sink, RAW product at the source, Leibniz sum with per-quark sites
    raw_p, raw_n = wo.nucleon_raw_terms("p", 0), wo.nucleon_raw_terms("n", 0)
    raw_src = wo.nucleus_raw_terms([("p", 0), ("n", 0)])
    got, sabs = wo.two_cluster_site_pair_value(Ux, Dx, Uy, Dy, p, n, pn)
    tot = 0.0
    src = raw_src[::23]                                         # slices: the sum is linear in each of the three lists
    raw_p, raw_n = raw_p[::2], raw_n[1::3]
    for ca, qa in raw_p:
        for cb, qb in raw_n:
            sink_q = qa + qb
            where = [0] * len(qa) + [1] * len(qb)
            for cj, qj in src:
                M = np.zeros((6, 6), complex)
                for i, (fi, ci) in enumerate(sink_q):
                    for j, (fj, cjx) in enumerate(qj):
                        if fi == fj:
                            P = ((Ux, Uy) if fi == "u" else (Dx, Dy))[where[i]]
                            M[i, j] = P[ci, cjx]
                tot += ca * cb * np.conj(cj) * wo.det_leibniz(M)
    part, _ = wo.two_cluster_site_pair_value(Ux, Dx, Uy, Dy, wo.merged_from_raw(raw_p), wo.merged_from_raw(raw_n), wo.merged_from_raw(src))
    assert abs(tot - part) <= 1e-11 * sabs
    assert abs(got) > 0

"""CPU oracle for the determinant-form Wick contraction of arXiv 2411.08962.

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py may import it.  It shares no code with the
CUDA path or the C++ term builder (own epsilon tensor, own gamma matrices, own expansion, own
elimination), and is written to be checked against the paper by eye: plain complex128 numpy,
no blocking, no deduplication of determinants, no minor tables.

What it computes (PAPER.md = /root/reference/PAPER.md, line numbers of that file):

  * Eq. (9)  PAPER.md:145  a nucleus interpolator is  sum_chi C^{chi_1..chi_n} q(chi_1)...q(chi_n);
  * Eq. (10) PAPER.md:149  G(t) = sum_x sum_{chi,chi'} C'^{chi'} C^{chi} <q(chi_1)..q(chi_n) qbar(chi'_1)..qbar(chi'_n)>;
  * Eq. (11) PAPER.md:159  <...> = sum_sigma sgn(sigma) prod_i S(chi_i, chi'_sigma(i))      (RAW mode, `wick_det`);
  * Eq. (12)-(15) PAPER.md:170-188  per-flavour factorisation
        G(t) = eta sum_x sum_{chi,chi'} C' C det M^u(chi^u, chi'^u) det M^d(chi^d, chi'^d),
        M^q_ij = S_q(chi_i, chi'_j)  (Eq. 13)                               (MERGED mode);
  * Eq. (A1),(A2),(A7) PAPER.md:630-661  sum over terms, then over sites; BASELINE.json adds a
        momentum phase:  C(t,p) = sum_x e^{i p.x} sigma(x,t).
  * nucleons, BASELINE.json north_star / configs (same content as Eq. (4),(5)):
        p_gamma = eps_abc (u_a^T C gamma5 d_b) u_{c,gamma},  n_gamma = eps_abc (d_a^T C gamma5 u_b) d_{c,gamma},
        C = gamma4 gamma2.

Readings where the paper is silent (all listed in DESIGN.md "Readings"): Dirac-Pauli basis,
chi = 3*spin + colour, propagator row = sink index / column = source index, source tensor
C' = conj(C) on the same quark order, eta = +1, phase e^{+2 pi i n.x / L}.

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): brute-force Wick sums over all pairings
(Leibniz form of Eq. 11), source colour rotation invariance, Pauli zeros, the textbook proton
direct-minus-exchange contraction (Eq. 31 / B1) written as an einsum,
identity/diagonal propagator closed forms, the paper's printed term count 2716,
LAPACK determinants, Leibniz determinants, Cauchy-Binet, Jacobi complementary minors (n = 10, 11),
site-scaled propagators and time scaling.  No function here is "parity unpinned" except in the
sense of DESIGN.md: the global sign/normalisation of C(t) is a convention (eta, nucleon order).
"""
from __future__ import annotations

import itertools
import math
from typing import Dict, List, Sequence, Tuple

import numpy as np

# ----------------------------------------------------------------------------------------------
# Operator algebra (own copies; nothing imported from the product)
# ----------------------------------------------------------------------------------------------

def levi_civita() -> np.ndarray:
    """eps_abc, a,b,c in {0,1,2}."""
    eps = np.zeros((3, 3, 3))
    for a, b, c in itertools.permutations(range(3)):
        # parity of the permutation (a,b,c) by counting inversions
        inv = (a > b) + (a > c) + (b > c)
        eps[a, b, c] = -1.0 if inv % 2 else 1.0
    return eps


def gamma_matrices():
    """Euclidean Dirac-Pauli basis: gamma_k = [[0, -i sigma_k], [i sigma_k, 0]], gamma_4 = diag(1,1,-1,-1),
    gamma_5 = gamma_1 gamma_2 gamma_3 gamma_4.  'Upper components' = spin index 0, 1."""
    s1 = np.array([[0, 1], [1, 0]], dtype=complex)
    s2 = np.array([[0, -1j], [1j, 0]], dtype=complex)
    s3 = np.array([[1, 0], [0, -1]], dtype=complex)
    Z = np.zeros((2, 2), dtype=complex)
    g = [np.block([[Z, -1j * s], [1j * s, Z]]) for s in (s1, s2, s3)]
    g4 = np.diag([1, 1, -1, -1]).astype(complex)
    g5 = g[0] @ g[1] @ g[2] @ g4
    return g[0], g[1], g[2], g4, g5


def c_gamma5() -> np.ndarray:
    """C gamma5 with C = gamma4 gamma2.  In this basis: blockdiag(i sigma2, i sigma2), real."""
    _, g2, _, g4, g5 = gamma_matrices()
    m = (g4 @ g2) @ g5
    assert np.allclose(m.imag, 0.0)
    return m.real.copy()


# A raw term is (coef, quarks) with quarks = tuple of (flavour, chi), flavour 'u' | 'd', chi = 3*spin + colour.
RawTerm = Tuple[complex, Tuple[Tuple[str, int], ...]]


def nucleon_raw_terms(kind: str, gamma: int) -> List[RawTerm]:
    """p_gamma = eps_abc (Cg5)_{alpha beta} u(alpha,a) d(beta,b) u(gamma,c)   (kind 'p')
       n_gamma = eps_abc (Cg5)_{alpha beta} d(alpha,a) u(beta,b) d(gamma,c)   (kind 'n')
    quark order exactly as written; 6 * 4 = 24 raw terms."""
    f1, f2, f3 = ("u", "d", "u") if kind == "p" else ("d", "u", "d")
    eps, cg5 = levi_civita(), c_gamma5()
    out: List[RawTerm] = []
    for a in range(3):
        for b in range(3):
            for c in range(3):
                if eps[a, b, c] == 0:
                    continue
                for alpha in range(4):
                    for beta in range(4):
                        if cg5[alpha, beta] == 0:
                            continue
                        coef = eps[a, b, c] * cg5[alpha, beta]
                        out.append((coef, ((f1, 3 * alpha + a), (f2, 3 * beta + b), (f3, 3 * gamma + c))))
    return out


def nucleus_raw_terms(nucleus: Sequence[Tuple[str, int]]) -> List[RawTerm]:
    """Ordered Grassmann product of the nucleons (Eq. 9 with the product operator of BASELINE.json):
    24^A raw terms, quarks in operator order.  No sorting, no merging.  Only for small A."""
    terms: List[RawTerm] = [(1.0, ())]
    for kind, gamma in nucleus:
        nuc = nucleon_raw_terms(kind, gamma)
        terms = [(c1 * c2, q1 + q2) for (c1, q1) in terms for (c2, q2) in nuc]
    return terms


# ---- the paper's own interpolators (Eq. 4, 5, 20, 21, 26, 27): used for the GEVP correlation-matrix checks ----------------

def spin_projector(sign: int) -> np.ndarray:
    """P_+- = (1 +- gamma4) / 2 (below Eq. 27): diag(1,1,0,0) / diag(0,0,1,1) in the Dirac-Pauli basis."""
    g4 = gamma_matrices()[3]
    return ((np.eye(4) + sign * g4) / 2).real


def paper_nucleon_raw_terms(kind: str, alpha: int, projector: int = 0) -> List[RawTerm]:
    """Eq. (4)/(5):  p_alpha = eps_abc u^a_alpha u^b_beta (C gamma5)_{beta eta} d^c_eta  (n: u <-> d),
    quark order as written; projector = +-1 inserts P_+- as in Eq. (26)/(27), PAPER.md:271-273:
    (p_+-)_alpha = eps_abc u^a_alpha u^b_beta (C gamma5 P_+-)_{beta delta} d^c_delta."""
    f1, f2 = ("u", "d") if kind == "p" else ("d", "u")
    eps = levi_civita()
    M = c_gamma5() if projector == 0 else c_gamma5() @ spin_projector(projector)
    out: List[RawTerm] = []
    for a in range(3):
        for b in range(3):
            for c in range(3):
                if eps[a, b, c] == 0:
                    continue
                for beta in range(4):
                    for delta in range(4):
                        if M[beta, delta] == 0:
                            continue
                        out.append((eps[a, b, c] * M[beta, delta], ((f1, 3 * alpha + a), (f1, 3 * beta + b), (f2, 3 * delta + c))))
    return out


def _raw_product(*factors: Sequence[RawTerm]) -> List[RawTerm]:
    terms: List[RawTerm] = [(1.0, ())]
    for f in factors:
        terms = [(c1 * c2, q1 + q2) for (c1, q1) in terms for (c2, q2) in f]
    return terms


def deuteron_eq20_raw_terms() -> List[RawTerm]:
    """Eq. (20):  O_2H = n^T (C gamma5 P_+) p = sum_{alpha beta} n_alpha (C gamma5 P_+)_{alpha beta} p_beta
    with the nucleons of Eq. (4)/(5)."""
    M = c_gamma5() @ spin_projector(+1)
    out: List[RawTerm] = []
    for alpha in range(4):
        for beta in range(4):
            if M[alpha, beta] != 0:
                out += [(M[alpha, beta] * c, q) for (c, q) in
                        _raw_product(paper_nucleon_raw_terms("n", alpha), paper_nucleon_raw_terms("p", beta))]
    return out


def helium3_eq21_raw_terms(J: int) -> List[RawTerm]:
    """Eq. (21):  O^J_3He = p_-^T (C gamma5) n_+ p_+^J = sum_{alpha beta} (p_-)_alpha (C gamma5)_{alpha beta}
    (n_+)_beta (p_+)_J  with the projected nucleons of Eq. (26)/(27).  The paper does not say which Dirac components the
    open index J runs over; the printed 1026 terms per spin component select J in {2, 3} (DESIGN.md reading)."""
    M = c_gamma5()
    out: List[RawTerm] = []
    for alpha in range(4):
        for beta in range(4):
            if M[alpha, beta] != 0:
                out += [(M[alpha, beta] * c, q) for (c, q) in
                        _raw_product(paper_nucleon_raw_terms("p", alpha, -1), paper_nucleon_raw_terms("n", beta, +1),
                                     paper_nucleon_raw_terms("p", J, +1))]
    return out


def merged_from_raw(raw: Sequence[RawTerm]):
    """Polynomial normal form of any raw operator: canonical monomials with their accumulated coefficients, zeros
    dropped, sorted by (u_tuple, d_tuple) -- "the number of terms in the operator" of Table II."""
    acc: Dict[Tuple[tuple, tuple], complex] = {}
    for c, q in raw:
        sign, u, d = canonical_monomial(q)
        if sign:
            acc[(u, d)] = acc.get((u, d), 0.0) + sign * c
    return [(u, d, acc[(u, d)]) for (u, d) in sorted(acc) if acc[(u, d)] != 0]


def sort_with_sign(seq: Sequence) -> Tuple[int, tuple]:
    """Sort a sequence of distinct comparable items ascending; return (sign, sorted tuple), sign =
    parity of the number of inversions (Eq. 19).  A repeated item gives sign 0
    (Grassmann: q q = 0)."""
    n = len(seq)
    inv = 0
    for i in range(n):
        for j in range(i + 1, n):
            if seq[i] == seq[j]:
                return 0, tuple(sorted(seq))
            if seq[i] > seq[j]:
                inv += 1
    return (-1 if inv % 2 else 1), tuple(sorted(seq))


def canonical_monomial(quarks: Sequence[Tuple[str, int]]):
    """Reorder q(chi_1)...q(chi_n) into (all u ascending, then all d ascending); the sign is the parity
    of that reordering of anticommuting fields.  Returns (sign, u_tuple, d_tuple)."""
    keyed = [(0 if f == "u" else 1, chi) for (f, chi) in quarks]
    sign, srt = sort_with_sign(keyed)
    u = tuple(chi for (f, chi) in srt if f == 0)
    d = tuple(chi for (f, chi) in srt if f == 1)
    return sign, u, d


def merged_terms(nucleus: Sequence[Tuple[str, int]]) -> List[Tuple[Tuple[int, ...], Tuple[int, ...], complex]]:
    """Polynomial normal form of the product operator: {(u_tuple asc, d_tuple asc): coefficient}, built
    nucleon by nucleon (canonical monomial of the partial product, times the next nucleon's raw term,
    re-sorted with its sign) so that A = 7 is feasible.  Zero coefficients (Pauli / exact
    cancellation) are dropped.  Returned sorted by (u_tuple, d_tuple)."""
    acc: Dict[Tuple[tuple, tuple], complex] = {((), ()): 1.0}
    for kind, gamma in nucleus:
        nuc = nucleon_raw_terms(kind, gamma)
        nxt: Dict[Tuple[tuple, tuple], complex] = {}
        for (u, d), c1 in acc.items():
            head = tuple(("u", x) for x in u) + tuple(("d", x) for x in d)
            for c2, q in nuc:
                sign, uu, dd = canonical_monomial(head + q)
                if sign == 0:
                    continue
                key = (uu, dd)
                nxt[key] = nxt.get(key, 0.0) + sign * c1 * c2
        acc = {k: v for k, v in nxt.items() if v != 0}
    return [(u, d, acc[(u, d)]) for (u, d) in sorted(acc)]


# ----------------------------------------------------------------------------------------------
# Determinants
# ----------------------------------------------------------------------------------------------

def det_elim(M: np.ndarray) -> np.ndarray:
    """Determinant of a batch of n x n complex matrices, shape (..., n, n), by Gaussian elimination
    with partial pivoting (pivot = entry of largest modulus in the column, first one wins), the
    'LU decomposition' of PAPER.md:203.  det = sign * product of pivots; a zero pivot column gives 0."""
    A = np.array(M, dtype=np.complex128, copy=True)
    n = A.shape[-1]
    batch = A.shape[:-2]
    A = A.reshape((-1, n, n))
    B = A.shape[0]
    idx = np.arange(B)
    det = np.ones(B, dtype=np.complex128)
    for k in range(n):
        mag = A[:, k:, k].real ** 2 + A[:, k:, k].imag ** 2
        p = k + np.argmax(mag, axis=1)                     # first maximum
        swap = p != k
        rows_k = A[idx, k, :].copy()
        rows_p = A[idx, p, :].copy()
        A[idx, k, :] = rows_p
        A[idx, p, :] = rows_k
        det = np.where(swap, -det, det)
        piv = A[:, k, k].copy()
        det = det * piv
        if k + 1 < n:
            safe = np.where(piv != 0, piv, 1.0)
            mult = np.where((piv != 0)[:, None], A[:, k + 1:, k] / safe[:, None], 0.0)
            A[:, k + 1:, k:] = A[:, k + 1:, k:] - mult[:, :, None] * A[:, None, k, k:]
    return det.reshape(batch)


def det_leibniz(M: np.ndarray) -> complex:
    """Eq. (14): det M = sum_sigma sgn(sigma) prod_i M[i, sigma(i)].  One matrix, small n."""
    n = M.shape[0]
    total = 0.0 + 0.0j
    for perm in itertools.permutations(range(n)):
        sign, _ = sort_with_sign(perm)
        prod = 1.0 + 0.0j
        for i in range(n):
            prod *= M[i, perm[i]]
        total += sign * prod
    return total


# ----------------------------------------------------------------------------------------------
# RAW mode: Eq. (10) + (11) literally, no flavour regrouping, no sorting, no merging
# ----------------------------------------------------------------------------------------------

def wick_matrix(U: np.ndarray, D: np.ndarray, sink_q, src_q) -> np.ndarray:
    """M_ij = S(chi_i, chi'_j) of Eq. (11) for mixed-flavour quark sequences: S is diagonal in flavour
    (S_u = U, S_d = D, zero between different flavours); row = sink quark, column = source quark."""
    n = len(sink_q)
    M = np.zeros((n, n), dtype=np.complex128)
    for i, (fi, ci) in enumerate(sink_q):
        for j, (fj, cj) in enumerate(src_q):
            if fi == fj:
                M[i, j] = (U if fi == "u" else D)[ci, cj]
    return M


def raw_site_value(U: np.ndarray, D: np.ndarray, raw_sink: Sequence[RawTerm], raw_src: Sequence[RawTerm],
                   use_leibniz: bool = False) -> complex:
    """sigma(x,t) of one site from Eq. (10)/(11): sum_{i,j} c_i conj(c_j) sum_sigma sgn prod S, the inner
    sum taken as det of the full flavour-block matrix (or, use_leibniz=True, as the explicit sum over
    all (n_u+n_d)! pairings -- only n_u! n_d! of them are non-zero)."""
    vals = []
    for ci, qi in raw_sink:
        for cj, qj in raw_src:
            M = wick_matrix(U, D, qi, qj)
            d = det_leibniz(M) if use_leibniz else det_elim(M)
            vals.append(ci * np.conj(cj) * d)
    return complex(_sum_ld(np.array(vals)))


# ----------------------------------------------------------------------------------------------
# MERGED mode / generic term lists: Eq. (15), two fresh determinants per term (the paper's method A)
# ----------------------------------------------------------------------------------------------

def _sum_ld(v: np.ndarray) -> complex:
    """Sum in extended precision (x87 long double where available) so the oracle's own rounding
    (~1e-19 relative to sum |v|) is far below the 1e-10 parity gate."""
    v = np.asarray(v)
    re = np.sum(v.real.astype(np.longdouble))
    im = np.sum(v.imag.astype(np.longdouble))
    return complex(float(re), float(im))


def site_terms_value(U: np.ndarray, D: np.ndarray, a_u, b_u, a_d, b_d, w, chunk: int = 200000):
    """sigma = sum_k w_k det U[a_u(k), b_u(k)] det D[a_d(k), b_d(k)] for one site (Eq. A1, PAPER.md:630,
    without the minimal-set reuse: every term evaluates its own two determinants).
    Returns (sigma, S_abs) with S_abs = sum_k |w_k det det| (tolerance denominator)."""
    a_u, b_u, a_d, b_d = (np.asarray(x, dtype=np.intp) for x in (a_u, b_u, a_d, b_d))
    w = np.asarray(w, dtype=np.complex128)
    n = len(w)
    parts, absparts = [], []
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        Mu = U[a_u[s:e, :, None], b_u[s:e, None, :]]
        Md = D[a_d[s:e, :, None], b_d[s:e, None, :]]
        v = w[s:e] * det_elim(Mu) * det_elim(Md)
        parts.append(_sum_ld(v))
        absparts.append(float(np.sum(np.abs(v).astype(np.longdouble))))
    return complex(sum(parts)), float(sum(absparts))


def outer_product_term_arrays(sink, source=None):
    """Flat arrays for all (sink term i, source term j) pairs: a = sink tuples, b = source tuples,
    w = c_i conj(c_j) (Eq. 15 with C' = conj C).  `sink`/`source` are merged_terms()-style lists."""
    source = sink if source is None else source
    au = np.array([t[0] for t in sink], dtype=np.uint8)
    ad = np.array([t[1] for t in sink], dtype=np.uint8)
    cs = np.array([t[2] for t in sink], dtype=np.complex128)
    bu = np.array([t[0] for t in source], dtype=np.uint8)
    bd = np.array([t[1] for t in source], dtype=np.uint8)
    cq = np.conj(np.array([t[2] for t in source], dtype=np.complex128))
    ns, nq = len(sink), len(source)
    a_u = np.repeat(au, nq, axis=0)
    a_d = np.repeat(ad, nq, axis=0)
    b_u = np.tile(bu, (ns, 1))
    b_d = np.tile(bd, (ns, 1))
    w = np.repeat(cs, nq) * np.tile(cq, ns)
    return a_u, b_u, a_d, b_d, w


def site_value_outer(U: np.ndarray, D: np.ndarray, sink, source=None):
    """sigma(x,t) and S_abs for one site over all (i, j) pairs of a sink list and a source list, looping
    over sink terms so that memory stays small (He-4: 2716 x 2716 pairs)."""
    source = sink if source is None else source
    bu = np.array([t[0] for t in source], dtype=np.intp)
    bd = np.array([t[1] for t in source], dtype=np.intp)
    cq = np.conj(np.array([t[2] for t in source], dtype=np.complex128))
    parts, absparts = [], []
    for (au, ad, ci) in sink:
        au = np.asarray(au, dtype=np.intp)
        ad = np.asarray(ad, dtype=np.intp)
        Mu = U[au[None, :, None], bu[:, None, :]]
        Md = D[ad[None, :, None], bd[:, None, :]]
        v = (ci * cq) * det_elim(Mu) * det_elim(Md)
        parts.append(_sum_ld(v))
        absparts.append(float(np.sum(np.abs(v))))
    return complex(_sum_ld(np.array(parts))), float(sum(absparts))


def site_value_method_b(U: np.ndarray, D: np.ndarray, sink, source=None):
    """The paper's "improved" method B (PAPER.md:294; what its SERIAL C / OPENMP C rows run, :432): every DISTINCT
    (row tuple, column tuple) minor of a flavour is evaluated once per site (the minimal sets zeta_u, zeta_d of
    Eq. A1), then sigma = sum_ij c_i conj(c_j) MU[a_u(i), b_u(j)] MD[a_d(i), b_d(j)].
    Same result as site_value_outer (method A) up to rounding; used as a timed CPU baseline row and pinned against
    method A in tests/test_oracle_pins.py.  Returns (sigma, S_abs)."""
    source = sink if source is None else source
    out = []
    for f in (0, 1):
        rows = sorted({t[f] for t in sink})
        cols = sorted({t[f] for t in source})
        P = U if f == 0 else D
        r = np.array(rows, dtype=np.intp).reshape(len(rows), -1)
        c = np.array(cols, dtype=np.intp).reshape(len(cols), -1)
        M = det_elim(P[r[:, None, :, None], c[None, :, None, :]]) if r.shape[1] else np.ones((len(rows), len(cols)), complex)
        out.append((M, {t: k for k, t in enumerate(rows)}, {t: k for k, t in enumerate(cols)}))
    (MU, ru, cu), (MD, rd, cd) = out
    ju = np.array([cu[t[0]] for t in source], dtype=np.intp)
    jd = np.array([cd[t[1]] for t in source], dtype=np.intp)
    cq = np.conj(np.array([t[2] for t in source], dtype=np.complex128))
    parts, absparts = [], []
    for (au, ad, ci) in sink:
        v = (ci * cq) * MU[ru[au], ju] * MD[rd[ad], jd]
        parts.append(_sum_ld(v))
        absparts.append(float(np.sum(np.abs(v))))
    return complex(_sum_ld(np.array(parts))), float(sum(absparts))


# ----------------------------------------------------------------------------------------------
# Cluster sinks ("a cluster sink can be employed where each cluster ... [is] projected to zero momentum
# separately"; Eq. 3 / Eq. 8, PAPER.md:100, :125 for two nucleons): cluster A sits at sink site x, cluster B at sink site y
# ----------------------------------------------------------------------------------------------

def two_cluster_site_pair_value(Ux, Dx, Uy, Dy, sink_a, sink_b, source):
    """sum over sink terms iA of cluster A (quarks at site x), iB of cluster B (quarks at site y) and source terms j of
         c_A c_B conj(c_j) <q(A; x) q(B; y)  qbar(source)>
    in determinant form (Eq. 12-15): the u Wick matrix has the rows a_u(A) taken from U_x followed by the rows
    a_u(B) taken from U_y, columns b_u(j); likewise d.  Bringing  u_A d_A u_B d_B  to  u_A u_B d_A d_B  moves |u_B| fields past
    |d_A| fields: sign (-1)^(|d_A| |u_B|).  `source` is the merged list of the product operator A.B at the source.
    Returns (value, sum of |terms|)."""
    bu = np.array([t[0] for t in source], dtype=np.intp)
    bd = np.array([t[1] for t in source], dtype=np.intp)
    cq = np.conj(np.array([t[2] for t in source], dtype=np.complex128))
    total, total_abs = [], 0.0
    for (ua, da, ca) in sink_a:
        for (ub, db, cb) in sink_b:
            sign = -1.0 if (len(da) * len(ub)) % 2 else 1.0
            ua_, ub_, da_, db_ = (np.asarray(v, dtype=np.intp) for v in (ua, ub, da, db))
            Mu = np.concatenate([Ux[ua_[None, :, None], bu[:, None, :]], Uy[ub_[None, :, None], bu[:, None, :]]], axis=1)
            Md = np.concatenate([Dx[da_[None, :, None], bd[:, None, :]], Dy[db_[None, :, None], bd[:, None, :]]], axis=1)
            v = (sign * ca * cb * cq) * det_elim(Mu) * det_elim(Md)
            total.append(_sum_ld(v))
            total_abs += float(np.sum(np.abs(v)))
    return complex(_sum_ld(np.array(total))), total_abs


def two_cluster_correlator(U, D, sink_a, sink_b, source, mom_a, mom_b, L: int):
    """C(t) = sum_{x,y} e^{i p_A.x} e^{i p_B.y} <O_A(x,t) O_B(y,t) Obar(0)>  for U, D of shape [T][L^3][12][12]: every cluster is
    projected to its own momentum (the plane-wave sink of Eq. 8 when the clusters are single nucleons).
    Returns (C [T], S_abs [T])."""
    T, V = U.shape[0], U.shape[1]
    pa, pb = momentum_phases(L, [mom_a])[0], momentum_phases(L, [mom_b])[0]
    C = np.zeros(T, dtype=np.complex128)
    sabs = np.zeros(T)
    for t in range(T):
        vals = []
        for x in range(V):
            for y in range(V):
                v, a = two_cluster_site_pair_value(U[t, x], D[t, x], U[t, y], D[t, y], sink_a, sink_b, source)
                vals.append(pa[x] * pb[y] * v)
                sabs[t] += a
        C[t] = _sum_ld(np.array(vals))
    return C, sabs


def momentum_phases(L: int, momenta: Sequence[Tuple[int, int, int]]) -> np.ndarray:
    """e^{+2 pi i (n.x)/L} for every site s = x + L*(y + L*z); shape [n_mom][L^3].  (n.x) is reduced
    mod L in integers first so the phase is exact at multiples of L/4."""
    s = np.arange(L ** 3)
    x, y, z = s % L, (s // L) % L, s // (L * L)
    out = np.empty((len(momenta), L ** 3), dtype=np.complex128)
    for k, (nx, ny, nz) in enumerate(momenta):
        m = (nx * x + ny * y + nz * z) % L
        out[k] = np.exp(2j * np.pi * m / L)
    return out


def correlator_from_terms(U: np.ndarray, D: np.ndarray, a_u, b_u, a_d, b_d, w,
                          momenta: Sequence[Tuple[int, int, int]], L: int):
    """C(t,p) = sum_x e^{ip.x} sigma(x,t) (Eq. A2/A7, plus BASELINE's momentum phase)
    for U, D of shape [T][L^3][12][12].  Returns (C [n_mom][T], sigma [T][L^3], S_abs [T])."""
    T, V = U.shape[0], U.shape[1]
    assert V == L ** 3
    sigma = np.zeros((T, V), dtype=np.complex128)
    sabs = np.zeros(T)
    for t in range(T):
        for s in range(V):
            v, a = site_terms_value(U[t, s], D[t, s], a_u, b_u, a_d, b_d, w)
            sigma[t, s] = v
            sabs[t] += a
    ph = momentum_phases(L, momenta)
    C = np.zeros((len(momenta), T), dtype=np.complex128)
    for k in range(len(momenta)):
        for t in range(T):
            C[k, t] = _sum_ld(ph[k] * sigma[t])
    return C, sigma, sabs


def correlator_nucleus(U: np.ndarray, D: np.ndarray, nucleus, momenta, L: int):
    """Full MERGED-mode correlator of a product nucleus (sink list x conj source list)."""
    sink = merged_terms(nucleus)
    a_u, b_u, a_d, b_d, w = outer_product_term_arrays(sink)
    return correlator_from_terms(U, D, a_u, b_u, a_d, b_d, w, momenta, L)


def reduce_sites(sigma: np.ndarray, momenta, L: int) -> np.ndarray:
    """C[p][t] from a per-site array sigma[T][L^3] (used to check the device reduction at full size)."""
    ph = momentum_phases(L, momenta)
    T = sigma.shape[0]
    C = np.zeros((len(momenta), T), dtype=np.complex128)
    for k in range(len(momenta)):
        for t in range(T):
            C[k, t] = _sum_ld(ph[k] * sigma[t])
    return C


def identity_test_error_bound(n_terms: float, n_f: int, card_c: float, trials: int) -> float:
    """Appendix C: worst-case probability of one wrong 'identical' verdict,
    binom(N N', 2) (n_f / |C|)^T."""
    return (n_terms * (n_terms - 1.0) / 2.0) * (n_f / card_c) ** trials

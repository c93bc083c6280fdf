// Host-side term builder: steps a1, a2, a2' of DESIGN.md.
//
//  a1  Expand the ordered Grassmann product of nucleon interpolators (Eq. 9 PAPER.md:145 with the
//      nucleons of Eq. 4/5 :105-107) in the exterior algebra Lambda(C^12) (x) Lambda(C^12): a monomial is
//      a pair of 12-bit masks (u indices, d indices) in canonical order (all u ascending, then all d
//      ascending); re-ordering anticommuting fields gives the sign (Eq. 19 PAPER.md:213-224,
//      redundancy R.1); equal monomials are merged, Pauli zeros and exact cancellations dropped.
//  a2  Term list w_ij = c_i conj(c_j) over (sink i, source j) (Eq. 15 :188) and the unique-minor
//      tables per flavour (redundancy R.2 :226; zeta_u, zeta_d, Theta of Eq. A1 :628-633).
//  a2' Optional randomised identity test (Sec. III B :234-246, App. C :704-732): every term's product
//      of minors is evaluated at random points of F_p, p = 2^61 - 1, and terms whose values agree up
//      to sign in all trials are merged (Schwartz-Zippel; error bound Theorem 1 :713).
//
// Pure CPU code: no CUDA call in this file.
#include <algorithm>
#include <cstring>
#include <map>
#include <new>
#include <unordered_map>

#include "wick_internal.h"

namespace wick {

static thread_local std::string g_error;
void set_error(const std::string& msg) { g_error = msg; }

// ---------------------------------------------------------------------------------------------
// exterior algebra on (u mask, d mask)
// ---------------------------------------------------------------------------------------------

struct Mono { uint16_t u, d; };

static inline int popc(unsigned x) { return __builtin_popcount(x); }

// Append quark (flavour f: 0 = u, 1 = d; index chi) on the right of the canonical monomial
// u_{i1}..u_{ik} d_{j1}..d_{jl}.  Returns 0 if the index is already present (q q = 0), else the sign
// (+1/-1) of moving it into canonical position.
static inline int append_quark(Mono& m, int f, int chi) {
    const unsigned bit = 1u << chi;
    if (f == 0) {
        if (m.u & bit) return 0;
        const int moves = popc(m.d) + popc(m.u >> (chi + 1));   // past every d, past the larger u's
        m.u |= bit;
        return (moves & 1) ? -1 : 1;
    }
    if (m.d & bit) return 0;
    const int moves = popc(m.d >> (chi + 1));
    m.d |= bit;
    return (moves & 1) ? -1 : 1;
}

// eps_abc for a, b, c in {0,1,2}
static inline int levi_civita(int a, int b, int c) { return (a - b) * (b - c) * (c - a) / 2; }

// C gamma5 with C = gamma4 gamma2 in the Dirac-Pauli basis: real, antisymmetric, block
// diagonal; non-zero entries (0,1) = -(1,0) and (2,3) = -(3,2).  The overall sign enters once at the
// sink and once at the source for every nucleon, so it cancels in c_i conj(c_j).
static inline int c_gamma5(int alpha, int beta) {
    if (alpha == 0 && beta == 1) return 1;
    if (alpha == 1 && beta == 0) return -1;
    if (alpha == 2 && beta == 3) return 1;
    if (alpha == 3 && beta == 2) return -1;
    return 0;
}

struct RawNucleonTerm { int coef; int f[3]; int chi[3]; };

// p_gamma = eps_abc (Cg5)_{alpha beta} u(alpha,a) d(beta,b) u(gamma,c); neutron: u <-> d.  24 raw terms.
static std::vector<RawNucleonTerm> nucleon_terms(int kind, int gamma) {
    std::vector<RawNucleonTerm> out;
    const int f1 = kind == WICK_NUCLEON_PROTON ? 0 : 1, f2 = 1 - f1, f3 = f1;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
            for (int c = 0; c < 3; ++c) {
                const int e = levi_civita(a, b, c);
                if (!e) continue;
                for (int al = 0; al < 4; ++al)
                    for (int be = 0; be < 4; ++be) {
                        const int g = c_gamma5(al, be);
                        if (!g) continue;
                        RawNucleonTerm t;
                        t.coef = e * g;
                        t.f[0] = f1; t.chi[0] = 3 * al + a;
                        t.f[1] = f2; t.chi[1] = 3 * be + b;
                        t.f[2] = f3; t.chi[2] = 3 * gamma + c;
                        out.push_back(t);
                    }
            }
    return out;
}

static inline uint32_t key_of(Mono m) { return (uint32_t(m.u) << 16) | m.d; }

// Lexicographic order of the ascending tuples encoded by two masks: the mask owning the lowest
// differing bit has the smaller element at the first position where the tuples differ.
static inline bool tuple_less(uint16_t a, uint16_t b) {
    const unsigned x = unsigned(a) ^ unsigned(b);
    if (!x) return false;
    const unsigned low = x & (~x + 1u);
    return (a & low) != 0;
}

static void mask_to_tuple(uint16_t mask, int n, uint8_t* out) {
    int k = 0;
    for (int i = 0; i < 12 && k < n; ++i)
        if (mask & (1u << i)) out[k++] = uint8_t(i);
}

// distinct masks, sorted as tuples; returns id lookup
static std::vector<uint16_t> distinct_sorted(std::vector<uint16_t> v) {
    std::sort(v.begin(), v.end(), tuple_less);
    v.erase(std::unique(v.begin(), v.end()), v.end());
    return v;
}

static std::unordered_map<uint16_t, int32_t> index_of(const std::vector<uint16_t>& v) {
    std::unordered_map<uint16_t, int32_t> m;
    for (size_t i = 0; i < v.size(); ++i) m[v[i]] = int32_t(i);
    return m;
}

// ---------------------------------------------------------------------------------------------
// arithmetic in F_p, p = 2^61 - 1 (identity test)
// ---------------------------------------------------------------------------------------------

static const uint64_t P61 = (uint64_t(1) << 61) - 1;

static inline uint64_t mulmod(uint64_t a, uint64_t b) {
    const unsigned __int128 z = (unsigned __int128)a * b;
    uint64_t r = uint64_t(z & P61) + uint64_t(z >> 61);
    r = (r & P61) + (r >> 61);
    return r >= P61 ? r - P61 : r;
}
static inline uint64_t addmod(uint64_t a, uint64_t b) { uint64_t r = a + b; return r >= P61 ? r - P61 : r; }
static inline uint64_t submod(uint64_t a, uint64_t b) { return a >= b ? a - b : a + P61 - b; }
static uint64_t powmod(uint64_t a, uint64_t e) {
    uint64_t r = 1;
    while (e) { if (e & 1) r = mulmod(r, a); a = mulmod(a, a); e >>= 1; }
    return r;
}
static inline uint64_t invmod(uint64_t a) { return powmod(a, P61 - 2); }

// splitmix64: the builder's own counter-based generator (seeded by the caller)
static inline uint64_t splitmix64(uint64_t& s) {
    uint64_t z = (s += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
static uint64_t random_nonzero_residue(uint64_t& s) {
    for (;;) {
        const uint64_t r = splitmix64(s) & P61;       // 61 random bits
        if (r != 0 && r != P61) return r;
    }
}

// determinant of the n x n minor (rows, cols as masks) of a 12x12 matrix over F_p, Gaussian elimination
static uint64_t det_mod(const uint64_t A[12][12], uint16_t rows, uint16_t cols, int n) {
    uint8_t r[12], c[12];
    mask_to_tuple(rows, n, r);
    mask_to_tuple(cols, n, c);
    uint64_t M[12][12];
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) M[i][j] = A[r[i]][c[j]];
    uint64_t det = 1;
    for (int k = 0; k < n; ++k) {
        int p = k;
        while (p < n && M[p][k] == 0) ++p;
        if (p == n) return 0;
        if (p != k) {
            for (int j = k; j < n; ++j) std::swap(M[p][j], M[k][j]);
            det = submod(0, det);
        }
        det = mulmod(det, M[k][k]);
        const uint64_t inv = invmod(M[k][k]);
        for (int i = k + 1; i < n; ++i) {
            if (M[i][k] == 0) continue;
            const uint64_t f = mulmod(M[i][k], inv);
            for (int j = k + 1; j < n; ++j) M[i][j] = submod(M[i][j], mulmod(f, M[k][j]));
        }
    }
    return det;
}

}  // namespace wick

using namespace wick;

// ---------------------------------------------------------------------------------------------
// wick_terms helpers
// ---------------------------------------------------------------------------------------------

void wick_terms::ensure_flat() const {
    std::lock_guard<std::mutex> lock(mu);
    if (flat_ready) return;
    const int64_t ns = int64_t(sink.size()), nq = int64_t(source.size());
    const int64_t ncu = int64_t(f[0].cols.size()), ncd = int64_t(f[1].cols.size());
    t_uid.resize(size_t(ns * nq));
    t_did.resize(size_t(ns * nq));
    t_w.resize(size_t(ns * nq));
    for (int64_t i = 0; i < ns; ++i)
        for (int64_t j = 0; j < nq; ++j) {
            const size_t k = size_t(i * nq + j);
            t_uid[k] = int32_t(sink[i].qu * ncu + source[j].qu);
            t_did[k] = int32_t(sink[i].qd * ncd + source[j].qd);
            t_w[k] = sink[i].c * source[j].c;
        }
    flat_ready = true;
}

// Randomised identity test on the flat list.  Returns the number of terms removed.
static int64_t identity_test(wick_terms* t, unsigned flags, uint64_t seed) {
    t->ensure_flat();
    const int trials = 2;
    const int64_t n = int64_t(t->t_w.size());
    std::vector<uint64_t> val[2];
    uint64_t s = seed ^ 0x5851F42D4C957F2Dull;
    for (int tr = 0; tr < trials; ++tr) {
        uint64_t A[2][12][12];
        for (int fl = 0; fl < 2; ++fl)
            for (int i = 0; i < 12; ++i)
                for (int j = 0; j < 12; ++j) A[fl][i][j] = random_nonzero_residue(s);
        if (flags & WICK_BUILD_ISOSPIN) std::memcpy(A[1], A[0], sizeof(A[0]));
        std::vector<uint64_t> mv[2];
        for (int fl = 0; fl < 2; ++fl) {
            const FlavourTables& ft = t->f[fl];
            mv[fl].resize(ft.minor_row.size());
            for (size_t m = 0; m < mv[fl].size(); ++m)
                mv[fl][m] = det_mod(A[fl], ft.rows[ft.minor_row[m]], ft.cols[ft.minor_col[m]], ft.n);
        }
        val[tr].resize(size_t(n));
        for (int64_t k = 0; k < n; ++k) val[tr][size_t(k)] = mulmod(mv[0][t->t_uid[k]], mv[1][t->t_did[k]]);
    }
    // canonical key: (min(v0, p - v0), v1 with the sign that made v0 canonical); sign s0 in {+1,-1}
    struct Rec { uint64_t k0, k1; int64_t idx; int sgn; };
    std::vector<Rec> recs;
    recs.reserve(size_t(n));
    int64_t removed = 0;
    for (int64_t k = 0; k < n; ++k) {
        const uint64_t v0 = val[0][size_t(k)], v1 = val[1][size_t(k)];
        if (v0 == 0 && v1 == 0) { ++removed; t->t_w[size_t(k)] = 0.0; continue; }   // identically zero product
        const uint64_t n0 = submod(0, v0);
        Rec r;
        r.idx = k;
        if (v0 <= n0) { r.k0 = v0; r.k1 = v1; r.sgn = 1; }
        else          { r.k0 = n0; r.k1 = submod(0, v1); r.sgn = -1; }
        recs.push_back(r);
    }
    std::sort(recs.begin(), recs.end(), [](const Rec& a, const Rec& b) {
        if (a.k0 != b.k0) return a.k0 < b.k0;
        if (a.k1 != b.k1) return a.k1 < b.k1;
        return a.idx < b.idx;
    });
    for (size_t a = 0; a < recs.size();) {
        size_t b = a + 1;
        while (b < recs.size() && recs[b].k0 == recs[a].k0 && recs[b].k1 == recs[a].k1) ++b;
        const Rec& rep = recs[a];                              // smallest original index of the class
        for (size_t c = a + 1; c < b; ++c) {
            const double rel = double(rep.sgn * recs[c].sgn);
            t->t_w[size_t(rep.idx)] += rel * t->t_w[size_t(recs[c].idx)];
            t->t_w[size_t(recs[c].idx)] = 0.0;
            ++removed;
        }
        a = b;
    }
    // compact (stable), dropping zero weights
    size_t o = 0;
    for (size_t k = 0; k < size_t(n); ++k) {
        if (t->t_w[k] == cplx(0.0, 0.0)) continue;
        t->t_uid[o] = t->t_uid[k];
        t->t_did[o] = t->t_did[k];
        t->t_w[o] = t->t_w[k];
        ++o;
    }
    const int64_t gone = n - int64_t(o);
    t->t_uid.resize(o); t->t_did.resize(o); t->t_w.resize(o);
    t->n_terms = int64_t(o);
    if (gone > 0) {                                            // no longer an outer product
        t->outer = false;
        t->sink.clear();
        t->source.clear();
    }
    return gone;
}

static void grid_minors(FlavourTables& ft) {
    const size_t nr = ft.rows.size(), nc = ft.cols.size();
    ft.minor_row.resize(nr * nc);
    ft.minor_col.resize(nr * nc);
    for (size_t r = 0; r < nr; ++r)
        for (size_t c = 0; c < nc; ++c) {
            ft.minor_row[r * nc + c] = int32_t(r);
            ft.minor_col[r * nc + c] = int32_t(c);
        }
}

// ---------------------------------------------------------------------------------------------
// C-ABI
// Isospin limit U == D (the paper's m_u = m_d) for an outer-product list whose flavours share their row
// tuples: with M = MU = MD the product of sink term (a_u, a_d) and source term (b_u, b_d) equals the product of the
// swapped terms (a_d, a_u), (b_d, b_u).  If the sink list is symmetric under the swap up to one global sign s
// (c(a_d, a_u) = s c(a_u, a_d); the source list is its conjugate), the sum over sink terms with a_u > a_d equals the
// sum over those with a_u < a_d, so the list   { 2 c_i : a_u < a_d } + { c_i : a_u = a_d }   x   full source list
// gives the same correlator with about half the products -- and it is still an outer product, so it runs through the
// factorised reduction.  This is the swap-class merge the randomised identity test finds (Sec. III B),
// applied in factorised form.  Returns false (list untouched) when the symmetry does not hold.
static bool symmetrise_isospin(wick_terms* t) {
    if (!t->outer || t->n_u != t->n_d || t->f[0].rows != t->f[1].rows || t->f[0].cols != t->f[1].cols) return false;
    std::map<std::pair<int32_t, int32_t>, cplx> c;
    for (const FactorTerm& f : t->sink) c[{f.qu, f.qd}] = f.c;
    double s = 0.0;
    for (const FactorTerm& f : t->sink) {
        auto it = c.find({f.qd, f.qu});
        if (it == c.end()) return false;
        if (f.qu == f.qd) continue;
        const double want = (it->second == f.c) ? 1.0 : (it->second == -f.c ? -1.0 : 0.0);
        if (want == 0.0 || (s != 0.0 && want != s)) return false;
        s = want;
    }
    if (s < 0.0)
        for (const FactorTerm& f : t->sink) if (f.qu == f.qd) return false;   // c = -c: cannot be present
    std::vector<FactorTerm> half;
    for (const FactorTerm& f : t->sink) {
        if (f.qu > f.qd) continue;
        FactorTerm g = f;
        if (f.qu < f.qd) g.c *= 2.0;
        half.push_back(g);
    }
    t->sink.swap(half);
    t->n_terms = int64_t(t->sink.size()) * int64_t(t->source.size());
    t->flat_ready = false;
    t->needs_u_equals_d = true;
    return true;
}

// ---------------------------------------------------------------------------------------------
// General interpolators (GEVP correlation matrices, Sec. V): an operator is a polynomial in the
// exterior algebra, canonical monomial (u mask, d mask) -> complex coefficient.
// ---------------------------------------------------------------------------------------------
typedef std::map<uint32_t, cplx> Poly;

// canonical monomial a times canonical monomial b: the quarks of b are appended one by one (u ascending, then d ascending)
static int mono_mul(Mono a, Mono b, Mono* out) {
    int sign = 1;
    for (int chi = 0; chi < 12 && sign; ++chi) if (b.u & (1u << chi)) sign *= append_quark(a, 0, chi);
    for (int chi = 0; chi < 12 && sign; ++chi) if (b.d & (1u << chi)) sign *= append_quark(a, 1, chi);
    *out = a;
    return sign;
}

static Poly poly_mul(const Poly& A, const Poly& B, cplx scale) {
    Poly out;
    for (const auto& a : A)
        for (const auto& b : B) {
            Mono ma = {uint16_t(a.first >> 16), uint16_t(a.first & 0xffff)}, mb = {uint16_t(b.first >> 16), uint16_t(b.first & 0xffff)}, m;
            const int sign = mono_mul(ma, mb, &m);
            if (sign) out[key_of(m)] += scale * double(sign) * a.second * b.second;
        }
    return out;
}

static void poly_add(Poly& A, const Poly& B) { for (const auto& b : B) A[b.first] += b.second; }
static void poly_prune(Poly& A) { for (auto it = A.begin(); it != A.end();) it = (it->second == cplx(0.0, 0.0)) ? A.erase(it) : std::next(it); }

// (C gamma5 P)_{beta delta}: P = 1 (proj 0), P_+ = diag(1,1,0,0) (proj +1), P_- = diag(0,0,1,1) (proj -1)
static int cg5_projected(int beta, int delta, int proj) {
    if (proj > 0 && delta >= 2) return 0;
    if (proj < 0 && delta < 2) return 0;
    return c_gamma5(beta, delta);
}

// Eq. (4)/(5) PAPER.md:105-107, with the projector of Eq. (26)/(27) :271-273:
// (N)_alpha = eps_abc q1^a_alpha q1^b_beta (C gamma5 P)_{beta delta} q2^c_delta,  q1 = u, q2 = d for the proton
static Poly paper_nucleon(int kind, int alpha, int proj) {
    const int f1 = kind == WICK_NUCLEON_PROTON ? 0 : 1, f2 = 1 - f1;
    Poly out;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
            for (int c = 0; c < 3; ++c) {
                const int e = levi_civita(a, b, c);
                if (!e) continue;
                for (int be = 0; be < 4; ++be)
                    for (int de = 0; de < 4; ++de) {
                        const int g = cg5_projected(be, de, proj);
                        if (!g) continue;
                        Mono m = {0, 0};
                        int sign = append_quark(m, f1, 3 * alpha + a);
                        if (sign) sign *= append_quark(m, f1, 3 * be + b);
                        if (sign) sign *= append_quark(m, f2, 3 * de + c);
                        if (sign) out[key_of(m)] += double(e * g * sign);
                    }
            }
    poly_prune(out);
    return out;
}

struct wick_operator { int n_u = 0, n_d = 0; Poly poly; };

static bool operator_finish(wick_operator* op) {
    poly_prune(op->poly);
    op->n_u = op->n_d = 0;
    bool first = true;
    for (const auto& kv : op->poly) {
        const int nu = popc(kv.first >> 16), nd = popc(kv.first & 0xffff);
        if (first) { op->n_u = nu; op->n_d = nd; first = false; }
        else if (nu != op->n_u || nd != op->n_d) return false;
    }
    return true;
}

// ---------------------------------------------------------------------------------------------

extern "C" const char* wick_last_error(void) { return g_error.c_str(); }
extern "C" const char* wick_version(void) { return "wick-b200 0.1 (sm_100a)"; }

extern "C" int wick_build_terms(const wick_nucleon* nucleons, int n_nucleons, unsigned flags, uint64_t seed,
                                wick_terms** out) {
    if (!nucleons || !out || n_nucleons < 1) { set_error("wick_build_terms: NULL argument or n_nucleons < 1"); return WICK_ERR_ARG; }
    *out = nullptr;
    int nu = 0, nd = 0;
    for (int k = 0; k < n_nucleons; ++k) {
        if (nucleons[k].kind != WICK_NUCLEON_PROTON && nucleons[k].kind != WICK_NUCLEON_NEUTRON) {
            set_error("wick_build_terms: nucleon kind must be 0 (p) or 1 (n)"); return WICK_ERR_ARG; }
        if (nucleons[k].gamma < 0 || nucleons[k].gamma > 3) {
            set_error("wick_build_terms: gamma must be 0..3"); return WICK_ERR_ARG; }
        if (nucleons[k].kind == WICK_NUCLEON_PROTON) { nu += 2; nd += 1; } else { nu += 1; nd += 2; }
    }
    if (nu > 12 || nd > 12) { set_error("wick_build_terms: more than 12 quarks of one flavour (Pauli: operator vanishes)"); return WICK_ERR_ARG; }
    try {
        // a1: multiply nucleon by nucleon
        std::map<uint32_t, int64_t> acc;                       // integer coefficients: eps and C g5 are +-1
        acc[0] = 1;
        int64_t n_raw = 1;
        for (int k = 0; k < n_nucleons; ++k) {
            const std::vector<RawNucleonTerm> nuc = nucleon_terms(nucleons[k].kind, nucleons[k].gamma);
            n_raw *= int64_t(nuc.size());
            std::map<uint32_t, int64_t> next;
            for (const auto& kv : acc) {
                for (const RawNucleonTerm& rt : nuc) {
                    Mono m;
                    m.u = uint16_t(kv.first >> 16);
                    m.d = uint16_t(kv.first & 0xffff);
                    int sign = 1;
                    for (int q = 0; q < 3 && sign; ++q) sign *= append_quark(m, rt.f[q], rt.chi[q]);
                    if (!sign) continue;
                    next[key_of(m)] += kv.second * rt.coef * sign;
                }
            }
            acc.clear();
            for (const auto& kv : next)
                if (kv.second != 0) acc[kv.first] = kv.second;
        }
        wick_terms* t = new wick_terms();
        t->n_u = nu; t->n_d = nd; t->n_raw = n_raw;
        t->f[0].n = nu; t->f[1].n = nd;
        std::vector<uint16_t> us, ds;
        for (const auto& kv : acc) { us.push_back(uint16_t(kv.first >> 16)); ds.push_back(uint16_t(kv.first & 0xffff)); }
        t->f[0].rows = t->f[0].cols = distinct_sorted(us);
        t->f[1].rows = t->f[1].cols = distinct_sorted(ds);
        const auto iu = index_of(t->f[0].rows), id = index_of(t->f[1].rows);
        for (const auto& kv : acc) {
            FactorTerm ft;
            ft.qu = iu.at(uint16_t(kv.first >> 16));
            ft.qd = id.at(uint16_t(kv.first & 0xffff));
            ft.c = cplx(double(kv.second), 0.0);
            t->sink.push_back(ft);
        }
        std::sort(t->sink.begin(), t->sink.end(), [](const FactorTerm& a, const FactorTerm& b) {
            return a.qu != b.qu ? a.qu < b.qu : a.qd < b.qd; });
        t->source = t->sink;                                   // C' = conj(C) on the same quark order (reading 3)
        for (FactorTerm& s : t->source) s.c = std::conj(s.c);
        t->outer = true;
        t->n_terms = int64_t(t->sink.size()) * int64_t(t->source.size());
        grid_minors(t->f[0]);
        grid_minors(t->f[1]);
        if ((flags & WICK_BUILD_ISOSPIN) && !(flags & WICK_BUILD_IDENTITY_TEST)) symmetrise_isospin(t);
        if (flags & WICK_BUILD_IDENTITY_TEST) {
            t->n_identity_merged = identity_test(t, flags, seed);
            if ((flags & WICK_BUILD_ISOSPIN) && t->n_identity_merged > 0) t->needs_u_equals_d = true;
        }
        *out = t;
        return WICK_OK;
    } catch (const std::bad_alloc&) {
        set_error("wick_build_terms: out of host memory");
        return WICK_ERR_NOMEM;
    }
}

// sort a tuple ascending; returns 0 for a repeated index, else the permutation sign
static int sort_tuple_sign(const uint8_t* in, int n, uint16_t* mask) {
    uint8_t v[12];
    for (int i = 0; i < n; ++i) v[i] = in[i];
    int inv = 0;
    uint16_t m = 0;
    for (int i = 0; i < n; ++i) {
        if (m & (1u << v[i])) return 0;
        m |= uint16_t(1u << v[i]);
        for (int j = i + 1; j < n; ++j) inv += v[i] > v[j];
    }
    *mask = m;
    return (inv & 1) ? -1 : 1;
}

extern "C" int wick_build_terms_from_list(int n_u, int n_d, int64_t n_raw, const uint8_t* a_u, const uint8_t* b_u,
                                          const uint8_t* a_d, const uint8_t* b_d, const double* w_reim,
                                          unsigned flags, uint64_t seed, wick_terms** out) {
    if (!out) { set_error("wick_build_terms_from_list: out is NULL"); return WICK_ERR_ARG; }
    *out = nullptr;
    if (n_u < 0 || n_u > 12 || n_d < 0 || n_d > 12 || n_raw < 0) { set_error("wick_build_terms_from_list: need 0 <= n_u, n_d <= 12, n_raw >= 0"); return WICK_ERR_ARG; }
    if (n_raw > 0 && (!w_reim || (n_u > 0 && (!a_u || !b_u)) || (n_d > 0 && (!a_d || !b_d)))) {
        set_error("wick_build_terms_from_list: NULL array"); return WICK_ERR_ARG; }
    for (int64_t k = 0; k < n_raw; ++k) {
        for (int i = 0; i < n_u; ++i)
            if (a_u[k * n_u + i] > 11 || b_u[k * n_u + i] > 11) { set_error("wick_build_terms_from_list: u index >= 12"); return WICK_ERR_ARG; }
        for (int i = 0; i < n_d; ++i)
            if (a_d[k * n_d + i] > 11 || b_d[k * n_d + i] > 11) { set_error("wick_build_terms_from_list: d index >= 12"); return WICK_ERR_ARG; }
    }
    try {
        struct Key { uint16_t au, bu, ad, bd; bool operator<(const Key& o) const {
            if (au != o.au) return tuple_less(au, o.au);
            if (bu != o.bu) return tuple_less(bu, o.bu);
            if (ad != o.ad) return tuple_less(ad, o.ad);
            return tuple_less(bd, o.bd); } };
        std::map<Key, cplx> acc;
        for (int64_t k = 0; k < n_raw; ++k) {
            Key key = {0, 0, 0, 0};
            int s = 1;
            s *= sort_tuple_sign(a_u + k * n_u, n_u, &key.au);
            if (s) s *= sort_tuple_sign(b_u + k * n_u, n_u, &key.bu);
            if (s) s *= sort_tuple_sign(a_d + k * n_d, n_d, &key.ad);
            if (s) s *= sort_tuple_sign(b_d + k * n_d, n_d, &key.bd);
            if (!s) continue;                                  // Pauli zero
            acc[key] += double(s) * cplx(w_reim[2 * k], w_reim[2 * k + 1]);
        }
        wick_terms* t = new wick_terms();
        t->n_u = n_u; t->n_d = n_d; t->n_raw = n_raw;
        t->f[0].n = n_u; t->f[1].n = n_d;
        std::vector<uint16_t> v[4];
        for (const auto& kv : acc) {
            if (kv.second == cplx(0.0, 0.0)) continue;
            v[0].push_back(kv.first.au); v[1].push_back(kv.first.bu);
            v[2].push_back(kv.first.ad); v[3].push_back(kv.first.bd);
        }
        t->f[0].rows = distinct_sorted(v[0]); t->f[0].cols = distinct_sorted(v[1]);
        t->f[1].rows = distinct_sorted(v[2]); t->f[1].cols = distinct_sorted(v[3]);
        const auto iau = index_of(t->f[0].rows), ibu = index_of(t->f[0].cols);
        const auto iad = index_of(t->f[1].rows), ibd = index_of(t->f[1].cols);
        // unique minors = distinct (row id, col id) pairs, numbered in sorted order
        std::map<std::pair<int32_t, int32_t>, int32_t> mu_, md_;
        for (const auto& kv : acc) {
            if (kv.second == cplx(0.0, 0.0)) continue;
            mu_[{iau.at(kv.first.au), ibu.at(kv.first.bu)}] = 0;
            md_[{iad.at(kv.first.ad), ibd.at(kv.first.bd)}] = 0;
        }
        int32_t c = 0;
        for (auto& kv : mu_) { kv.second = c++; t->f[0].minor_row.push_back(kv.first.first); t->f[0].minor_col.push_back(kv.first.second); }
        c = 0;
        for (auto& kv : md_) { kv.second = c++; t->f[1].minor_row.push_back(kv.first.first); t->f[1].minor_col.push_back(kv.first.second); }
        for (const auto& kv : acc) {
            if (kv.second == cplx(0.0, 0.0)) continue;
            t->t_uid.push_back(mu_.at({iau.at(kv.first.au), ibu.at(kv.first.bu)}));
            t->t_did.push_back(md_.at({iad.at(kv.first.ad), ibd.at(kv.first.bd)}));
            t->t_w.push_back(kv.second);
        }
        t->flat_ready = true;
        t->outer = false;
        t->n_terms = int64_t(t->t_w.size());
        if (flags & WICK_BUILD_IDENTITY_TEST) {
            t->n_identity_merged = identity_test(t, flags, seed);
            if ((flags & WICK_BUILD_ISOSPIN) && t->n_identity_merged > 0) t->needs_u_equals_d = true;
        }
        *out = t;
        return WICK_OK;
    } catch (const std::bad_alloc&) {
        set_error("wick_build_terms_from_list: out of host memory");
        return WICK_ERR_NOMEM;
    }
}

extern "C" int wick_operator_from_nucleons(const wick_nucleon* nucleons, int n_nucleons, wick_operator** out) {
    if (!nucleons || !out || n_nucleons < 1) { set_error("wick_operator_from_nucleons: NULL argument or n_nucleons < 1"); return WICK_ERR_ARG; }
    *out = nullptr;
    for (int k = 0; k < n_nucleons; ++k)
        if ((nucleons[k].kind != WICK_NUCLEON_PROTON && nucleons[k].kind != WICK_NUCLEON_NEUTRON) || nucleons[k].gamma < 0 || nucleons[k].gamma > 3) {
            set_error("wick_operator_from_nucleons: kind must be 0 / 1 and gamma 0..3"); return WICK_ERR_ARG; }
    try {
        wick_operator* op = new wick_operator();
        op->poly[0] = 1.0;
        for (int k = 0; k < n_nucleons; ++k) {
            Poly nuc;
            for (const RawNucleonTerm& rt : nucleon_terms(nucleons[k].kind, nucleons[k].gamma)) {
                Mono m = {0, 0};
                int sign = 1;
                for (int q = 0; q < 3 && sign; ++q) sign *= append_quark(m, rt.f[q], rt.chi[q]);
                if (sign) nuc[key_of(m)] += double(rt.coef * sign);
            }
            op->poly = poly_mul(op->poly, nuc, 1.0);
            poly_prune(op->poly);
        }
        operator_finish(op);
        *out = op;
        return WICK_OK;
    } catch (const std::bad_alloc&) { set_error("wick_operator_from_nucleons: out of host memory"); return WICK_ERR_NOMEM; }
}

extern "C" int wick_operator_from_raw(int n_quarks, int64_t n_raw, const uint8_t* flavour, const uint8_t* chi, const double* coef_reim,
                                      wick_operator** out) {
    if (!out || n_quarks < 0 || n_quarks > 24 || n_raw < 0 || (n_raw > 0 && (!coef_reim || (n_quarks > 0 && (!flavour || !chi))))) {
        set_error("wick_operator_from_raw: bad argument"); return WICK_ERR_ARG; }
    *out = nullptr;
    for (int64_t k = 0; k < n_raw * n_quarks; ++k)
        if (flavour[k] > 1 || chi[k] > 11) { set_error("wick_operator_from_raw: flavour must be 0 / 1 and chi < 12"); return WICK_ERR_ARG; }
    try {
        wick_operator* op = new wick_operator();
        for (int64_t k = 0; k < n_raw; ++k) {
            Mono m = {0, 0};
            int sign = 1;
            for (int q = 0; q < n_quarks && sign; ++q) sign *= append_quark(m, flavour[k * n_quarks + q], chi[k * n_quarks + q]);
            if (sign) op->poly[key_of(m)] += double(sign) * cplx(coef_reim[2 * k], coef_reim[2 * k + 1]);
        }
        if (!operator_finish(op)) { delete op; set_error("wick_operator_from_raw: terms with different quark content"); return WICK_ERR_ARG; }
        *out = op;
        return WICK_OK;
    } catch (const std::bad_alloc&) { set_error("wick_operator_from_raw: out of host memory"); return WICK_ERR_NOMEM; }
}

extern "C" int wick_operator_paper(int which, int J, wick_operator** out) {
    if (!out || (which != WICK_OP_DEUTERON_EQ20 && which != WICK_OP_HELIUM3_EQ21) || J < 0 || J > 3) {
        set_error("wick_operator_paper: which must be WICK_OP_DEUTERON_EQ20 or WICK_OP_HELIUM3_EQ21, J 0..3"); return WICK_ERR_ARG; }
    *out = nullptr;
    try {
        wick_operator* op = new wick_operator();
        for (int al = 0; al < 4; ++al)
            for (int be = 0; be < 4; ++be) {
                if (which == WICK_OP_DEUTERON_EQ20) {
                    const int g = cg5_projected(al, be, +1);           // n^T (C g5 P+) p, Eq. (20)
                    if (g) poly_add(op->poly, poly_mul(paper_nucleon(WICK_NUCLEON_NEUTRON, al, 0), paper_nucleon(WICK_NUCLEON_PROTON, be, 0), double(g)));
                } else {
                    const int g = c_gamma5(al, be);                    // p_-^T (C g5) n_+ p_+^J, Eq. (21)
                    if (g) poly_add(op->poly, poly_mul(poly_mul(paper_nucleon(WICK_NUCLEON_PROTON, al, -1), paper_nucleon(WICK_NUCLEON_NEUTRON, be, +1), double(g)),
                                                       paper_nucleon(WICK_NUCLEON_PROTON, J, +1), 1.0));
                }
            }
        operator_finish(op);
        *out = op;
        return WICK_OK;
    } catch (const std::bad_alloc&) { set_error("wick_operator_paper: out of host memory"); return WICK_ERR_NOMEM; }
}

extern "C" int wick_operator_info(const wick_operator* op, int32_t* n_u, int32_t* n_d, int64_t* n_terms) {
    if (!op) { set_error("wick_operator_info: NULL argument"); return WICK_ERR_ARG; }
    if (n_u) *n_u = op->n_u;
    if (n_d) *n_d = op->n_d;
    if (n_terms) *n_terms = int64_t(op->poly.size());
    return WICK_OK;
}

extern "C" int wick_operator_export(const wick_operator* op, uint8_t* u_tuples, uint8_t* d_tuples, double* coef_reim) {
    if (!op) { set_error("wick_operator_export: NULL argument"); return WICK_ERR_ARG; }
    size_t k = 0;
    for (const auto& kv : op->poly) {
        if (u_tuples) mask_to_tuple(uint16_t(kv.first >> 16), op->n_u, u_tuples + k * size_t(op->n_u));
        if (d_tuples) mask_to_tuple(uint16_t(kv.first & 0xffff), op->n_d, d_tuples + k * size_t(op->n_d));
        if (coef_reim) { coef_reim[2 * k] = kv.second.real(); coef_reim[2 * k + 1] = kv.second.imag(); }
        ++k;
    }
    return WICK_OK;
}

extern "C" void wick_operator_free(wick_operator* op) { delete op; }

// K interpolators with the same quark content -> K x K term lists  (sink k) x conj(source k')  over ONE pair of
// unique-minor tables (the union of all row / column tuples): the determinants are shared by the whole correlation
// matrix (Sec. V, Eq. 36-38).
extern "C" int wick_build_terms_matrix(const wick_operator* const* ops, int n_ops, unsigned flags, wick_terms** out) {
    (void)flags;
    if (!ops || !out || n_ops < 1) { set_error("wick_build_terms_matrix: bad argument"); return WICK_ERR_ARG; }
    for (int k = 0; k < n_ops * n_ops; ++k) out[k] = nullptr;
    for (int k = 0; k < n_ops; ++k)
        if (!ops[k] || ops[k]->n_u != ops[0]->n_u || ops[k]->n_d != ops[0]->n_d || ops[k]->poly.empty()) {
            set_error("wick_build_terms_matrix: operators must be non-empty and share their quark content"); return WICK_ERR_ARG; }
    try {
        std::vector<uint16_t> us, ds;
        for (int k = 0; k < n_ops; ++k)
            for (const auto& kv : ops[k]->poly) { us.push_back(uint16_t(kv.first >> 16)); ds.push_back(uint16_t(kv.first & 0xffff)); }
        const std::vector<uint16_t> ru = distinct_sorted(us), rd = distinct_sorted(ds);
        const auto iu = index_of(ru), id = index_of(rd);
        std::vector<std::vector<FactorTerm>> lists(static_cast<size_t>(n_ops));
        for (int k = 0; k < n_ops; ++k) {
            for (const auto& kv : ops[k]->poly) {
                FactorTerm ft;
                ft.qu = iu.at(uint16_t(kv.first >> 16)); ft.qd = id.at(uint16_t(kv.first & 0xffff)); ft.c = kv.second;
                lists[size_t(k)].push_back(ft);
            }
            std::sort(lists[size_t(k)].begin(), lists[size_t(k)].end(), [](const FactorTerm& a, const FactorTerm& b) {
                return a.qu != b.qu ? a.qu < b.qu : a.qd < b.qd; });
        }
        for (int k = 0; k < n_ops; ++k)
            for (int kp = 0; kp < n_ops; ++kp) {
                wick_terms* t = new wick_terms();
                out[k * n_ops + kp] = t;
                t->n_u = ops[0]->n_u; t->n_d = ops[0]->n_d;
                t->f[0].n = t->n_u; t->f[1].n = t->n_d;
                t->f[0].rows = t->f[0].cols = ru;
                t->f[1].rows = t->f[1].cols = rd;
                t->sink = lists[size_t(k)];
                t->source = lists[size_t(kp)];
                for (FactorTerm& s : t->source) s.c = std::conj(s.c);       // C' = conj(C) (reading 3)
                t->outer = true;
                t->n_terms = int64_t(t->sink.size()) * int64_t(t->source.size());
                t->n_raw = t->n_terms;
                grid_minors(t->f[0]);
                grid_minors(t->f[1]);
            }
        return WICK_OK;
    } catch (const std::bad_alloc&) {
        for (int k = 0; k < n_ops * n_ops; ++k) { delete out[k]; out[k] = nullptr; }
        set_error("wick_build_terms_matrix: out of host memory");
        return WICK_ERR_NOMEM;
    }
}

extern "C" int wick_operator_product(const wick_operator* a, const wick_operator* b, wick_operator** out) {
    if (!a || !b || !out) { set_error("wick_operator_product: NULL argument"); return WICK_ERR_ARG; }
    *out = nullptr;
    if (a->n_u + b->n_u > 12 || a->n_d + b->n_d > 12) { set_error("wick_operator_product: more than 12 quarks of one flavour"); return WICK_ERR_ARG; }
    try {
        wick_operator* op = new wick_operator();
        op->poly = poly_mul(a->poly, b->poly, 1.0);
        operator_finish(op);
        *out = op;
        return WICK_OK;
    } catch (const std::bad_alloc&) { set_error("wick_operator_product: out of host memory"); return WICK_ERR_NOMEM; }
}

// all n-subsets of {0..11} as masks, in lexicographic tuple order
static std::vector<uint16_t> all_subsets(int n) {
    std::vector<uint16_t> v;
    for (unsigned m = 0; m < 4096; ++m) if (popc(m) == n) v.push_back(uint16_t(m));
    std::sort(v.begin(), v.end(), tuple_less);
    return v;
}

// Cluster sinks (block algorithm Eq. 6-8 :110-125): block handle of ONE cluster.  Rows = the cluster's own row
// tuples, columns = EVERY n-subset of the 12 source indices, no source list: wick_block_tensor evaluates
//   B[t][S_u][S_d] = sum_x e^{ip.x} sum_i c_i det U_x[a_u(i), S_u] det D_x[a_d(i), S_d].
extern "C" int wick_build_block_terms(const wick_operator* cluster, wick_terms** out) {
    if (!cluster || !out || cluster->poly.empty()) { set_error("wick_build_block_terms: NULL or empty operator"); return WICK_ERR_ARG; }
    *out = nullptr;
    try {
        wick_terms* t = new wick_terms();
        t->n_u = cluster->n_u; t->n_d = cluster->n_d;
        t->f[0].n = t->n_u; t->f[1].n = t->n_d;
        std::vector<uint16_t> us, ds;
        for (const auto& kv : cluster->poly) { us.push_back(uint16_t(kv.first >> 16)); ds.push_back(uint16_t(kv.first & 0xffff)); }
        t->f[0].rows = distinct_sorted(us); t->f[1].rows = distinct_sorted(ds);
        t->f[0].cols = all_subsets(t->n_u); t->f[1].cols = all_subsets(t->n_d);
        const auto iu = index_of(t->f[0].rows), id = index_of(t->f[1].rows);
        for (const auto& kv : cluster->poly) {
            FactorTerm ft;
            ft.qu = iu.at(uint16_t(kv.first >> 16)); ft.qd = id.at(uint16_t(kv.first & 0xffff)); ft.c = kv.second;
            t->sink.push_back(ft);
        }
        std::sort(t->sink.begin(), t->sink.end(), [](const FactorTerm& a, const FactorTerm& b) {
            return a.qu != b.qu ? a.qu < b.qu : a.qd < b.qd; });
        t->outer = true;                                       // grid tables; the source list stays empty
        t->block_mode = true;
        t->n_terms = 0;
        grid_minors(t->f[0]);
        grid_minors(t->f[1]);
        *out = t;
        return WICK_OK;
    } catch (const std::bad_alloc&) { set_error("wick_build_block_terms: out of host memory"); return WICK_ERR_NOMEM; }
}

// rank of a 12-bit mask among the n-subsets in lexicographic tuple order
static int subset_index(const std::unordered_map<uint16_t, int32_t>& idx, uint16_t mask) { return idx.at(mask); }

// C[t] = sum_j conj(c_j) sum_{S_u in b_u(j), S_d in b_d(j)} sign B_A[t][S_u][S_d] B_B[t][b_u \ S_u][b_d \ S_d]
// (generalised Laplace expansion of the two stacked determinants along the rows of cluster A; lattice independent).
extern "C" int wick_combine_two_clusters(const wick_operator* a, const wick_operator* b, const wick_operator* source,
                                         const double* BA_reim, const double* BB_reim, int T, double* C_reim) {
    if (!a || !b || !source || !BA_reim || !BB_reim || !C_reim || T < 1) { set_error("wick_combine_two_clusters: bad argument"); return WICK_ERR_ARG; }
    if (source->n_u != a->n_u + b->n_u || source->n_d != a->n_d + b->n_d) {
        set_error("wick_combine_two_clusters: the source operator must have the quark content of A.B"); return WICK_ERR_ARG; }
    try {
        const std::vector<uint16_t> cua = all_subsets(a->n_u), cda = all_subsets(a->n_d), cub = all_subsets(b->n_u), cdb = all_subsets(b->n_d);
        const auto iua = index_of(cua), ida = index_of(cda), iub = index_of(cub), idb = index_of(cdb);
        const size_t na = cua.size() * cda.size(), nb = cub.size() * cdb.size();
        // sign of taking the columns S (a subset of the ascending tuple b) for the first k = |S| rows: (-1)^(sum of positions of S + k(k-1)/2)
        auto laplace_sign = [](uint16_t full, uint16_t sub) {
            int pos = 0, sum = 0, k = 0;
            for (int bit = 0; bit < 12; ++bit) if (full & (1u << bit)) { if (sub & (1u << bit)) { sum += pos; ++k; } ++pos; }
            return ((sum + k * (k - 1) / 2) & 1) ? -1.0 : 1.0;
        };
        const double cluster_sign = ((a->n_d * b->n_u) & 1) ? -1.0 : 1.0;      // u_A d_A u_B d_B -> u_A u_B d_A d_B
        for (int t = 0; t < T; ++t) {
            const cplx* BA = reinterpret_cast<const cplx*>(BA_reim) + size_t(t) * na;
            const cplx* BB = reinterpret_cast<const cplx*>(BB_reim) + size_t(t) * nb;
            long double re = 0.0L, im = 0.0L;
            for (const auto& kv : source->poly) {
                const uint16_t bu = uint16_t(kv.first >> 16), bd = uint16_t(kv.first & 0xffff);
                cplx acc(0.0, 0.0);
                for (uint16_t su = bu;; su = uint16_t((su - 1) & bu)) {
                    if (popc(su) == a->n_u) {
                        const double sgu = laplace_sign(bu, su);
                        for (uint16_t sd = bd;; sd = uint16_t((sd - 1) & bd)) {
                            if (popc(sd) == a->n_d)
                                acc += sgu * laplace_sign(bd, sd) *
                                       BA[size_t(subset_index(iua, su)) * cda.size() + size_t(subset_index(ida, sd))] *
                                       BB[size_t(subset_index(iub, uint16_t(bu & ~su))) * cdb.size() + size_t(subset_index(idb, uint16_t(bd & ~sd)))];
                            if (sd == 0) break;
                        }
                    }
                    if (su == 0) break;
                }
                const cplx v = cluster_sign * std::conj(kv.second) * acc;
                re += v.real(); im += v.imag();
            }
            C_reim[2 * t] = double(re); C_reim[2 * t + 1] = double(im);
        }
        return WICK_OK;
    } catch (const std::bad_alloc&) { set_error("wick_combine_two_clusters: out of host memory"); return WICK_ERR_NOMEM; }
}

extern "C" int wick_terms_get_info(const wick_terms* t, wick_terms_info* info) {
    if (!t || !info) { set_error("wick_terms_get_info: NULL argument"); return WICK_ERR_ARG; }
    info->n_u = t->n_u; info->n_d = t->n_d;
    info->n_rows_u = int32_t(t->f[0].rows.size()); info->n_cols_u = int32_t(t->f[0].cols.size());
    info->n_rows_d = int32_t(t->f[1].rows.size()); info->n_cols_d = int32_t(t->f[1].cols.size());
    info->n_minors_u = int64_t(t->f[0].minor_row.size());
    info->n_minors_d = int64_t(t->f[1].minor_row.size());
    info->n_terms = t->n_terms;
    info->is_outer_product = t->outer ? 1 : 0;
    info->n_sink = int32_t(t->sink.size()); info->n_source = int32_t(t->source.size());
    info->n_raw = t->n_raw;
    info->n_identity_merged = t->n_identity_merged;
    return WICK_OK;
}

extern "C" int wick_terms_export_tuples(const wick_terms* t, uint8_t* u_rows, uint8_t* u_cols, uint8_t* d_rows, uint8_t* d_cols) {
    if (!t) { set_error("wick_terms_export_tuples: NULL handle"); return WICK_ERR_ARG; }
    uint8_t* dst[4] = {u_rows, u_cols, d_rows, d_cols};
    const std::vector<uint16_t>* src[4] = {&t->f[0].rows, &t->f[0].cols, &t->f[1].rows, &t->f[1].cols};
    const int n[4] = {t->n_u, t->n_u, t->n_d, t->n_d};
    for (int k = 0; k < 4; ++k) {
        if (!dst[k]) continue;
        for (size_t i = 0; i < src[k]->size(); ++i) mask_to_tuple((*src[k])[i], n[k], dst[k] + i * size_t(n[k]));
    }
    return WICK_OK;
}

extern "C" int wick_terms_export_minors(const wick_terms* t, int32_t* u_minor_row, int32_t* u_minor_col,
                                        int32_t* d_minor_row, int32_t* d_minor_col) {
    if (!t) { set_error("wick_terms_export_minors: NULL handle"); return WICK_ERR_ARG; }
    if (u_minor_row) std::copy(t->f[0].minor_row.begin(), t->f[0].minor_row.end(), u_minor_row);
    if (u_minor_col) std::copy(t->f[0].minor_col.begin(), t->f[0].minor_col.end(), u_minor_col);
    if (d_minor_row) std::copy(t->f[1].minor_row.begin(), t->f[1].minor_row.end(), d_minor_row);
    if (d_minor_col) std::copy(t->f[1].minor_col.begin(), t->f[1].minor_col.end(), d_minor_col);
    return WICK_OK;
}

extern "C" int wick_terms_export_terms(const wick_terms* t, int64_t first, int64_t count, int32_t* uid, int32_t* did, double* w_reim) {
    if (!t || first < 0 || count < 0 || first + count > t->n_terms) { set_error("wick_terms_export_terms: bad handle or range"); return WICK_ERR_ARG; }
    try { t->ensure_flat(); } catch (const std::bad_alloc&) { set_error("wick_terms_export_terms: out of host memory"); return WICK_ERR_NOMEM; }
    for (int64_t k = 0; k < count; ++k) {
        if (uid) uid[k] = t->t_uid[size_t(first + k)];
        if (did) did[k] = t->t_did[size_t(first + k)];
        if (w_reim) { w_reim[2 * k] = t->t_w[size_t(first + k)].real(); w_reim[2 * k + 1] = t->t_w[size_t(first + k)].imag(); }
    }
    return WICK_OK;
}

extern "C" int wick_terms_export_factors(const wick_terms* t, int32_t* sink_ru, int32_t* sink_rd, double* sink_c,
                                         int32_t* src_cu, int32_t* src_cd, double* src_c) {
    if (!t) { set_error("wick_terms_export_factors: NULL handle"); return WICK_ERR_ARG; }
    if (!t->outer) { set_error("wick_terms_export_factors: term list is not an outer product"); return WICK_ERR_UNSUPPORTED; }
    for (size_t i = 0; i < t->sink.size(); ++i) {
        if (sink_ru) sink_ru[i] = t->sink[i].qu;
        if (sink_rd) sink_rd[i] = t->sink[i].qd;
        if (sink_c) { sink_c[2 * i] = t->sink[i].c.real(); sink_c[2 * i + 1] = t->sink[i].c.imag(); }
    }
    for (size_t j = 0; j < t->source.size(); ++j) {
        if (src_cu) src_cu[j] = t->source[j].qu;
        if (src_cd) src_cd[j] = t->source[j].qd;
        if (src_c) { src_c[2 * j] = t->source[j].c.real(); src_c[2 * j + 1] = t->source[j].c.imag(); }
    }
    return WICK_OK;
}

extern "C" void wick_terms_free(wick_terms* t) {
    if (!t) return;
    wick_terms_release_device(&t->dev);
    delete t;
}

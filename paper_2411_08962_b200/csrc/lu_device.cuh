// Device helpers shared by the minors kernels (kernels.cu, minors_reg.cu): complex arithmetic, tile staging,
// pivot rule and the hybrid left-looking LU state.
#pragma once
#include "kernels.cuh"

namespace wick {

typedef double2 c128;

__device__ __forceinline__ c128 cmul(c128 a, c128 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ c128 cfma(c128 a, c128 b, c128 c) {       // a*b + c
    return make_double2(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y)));
}
__device__ __forceinline__ c128 cfnma(c128 a, c128 b, c128 c) {      // c - a*b
    return make_double2(fma(-a.x, b.x, fma(a.y, b.y, c.x)), fma(-a.x, b.y, fma(-a.y, b.x, c.y)));
}
__device__ __forceinline__ c128 csub(c128 a, c128 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ c128 cadd(c128 a, c128 b) { return make_double2(a.x + b.x, a.y + b.y); }

// ---------------------------------------------------------------------------------------------
// a3: stage the 12x12 propagators of one 32-site group: tile[e][lane], e = 12*row + col
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void stage_tile(c128* tile, const c128* __restrict__ P, int64_t st_first,
                                           int64_t n_st_total, int nthreads) {
    // consecutive threads read consecutive 16-byte elements of one site (coalesced); sites beyond the
    // end of the lattice are filled with zeros (their lanes never store a result)
    for (int idx = threadIdx.x; idx < TILE_ELEMS; idx += nthreads) {
        const int site = idx / 144, e = idx - site * 144;
        const int64_t st = st_first + site;
        c128 v = make_double2(0.0, 0.0);
        if (st < n_st_total) v = __ldg(P + st * 144 + e);
        tile[e * GROUP + site] = v;
    }
}

// ---------------------------------------------------------------------------------------------
// a4: determinants.  `tl` points at tile[0][lane]; re[i] = 12*a_i, ce[j] = b_j (warp-uniform).
// ---------------------------------------------------------------------------------------------
template <int N> struct Idx { int re[N > 0 ? N : 1]; int ce[N > 0 ? N : 1]; };

__device__ __forceinline__ c128 ld(const c128* tl, int re, int ce) { return tl[(re + ce) * GROUP]; }

__device__ __forceinline__ c128 det2(c128 a, c128 b, c128 c, c128 d) {   // a d - b c
    return cfnma(b, c, cmul(a, d));
}

// N <= 2 (N = 3 and up keep state across minors, see minors_kernel / LuState)
template <int N>
__device__ __forceinline__ c128 det_small(const c128* tl, const Idx<N>& ix) {
    static_assert(N <= 2, "larger minors go through the column trie");
    if constexpr (N == 0) return make_double2(1.0, 0.0);
    else if constexpr (N == 1) return ld(tl, ix.re[0], ix.ce[0]);
    else return det2(ld(tl, ix.re[0], ix.ce[0]), ld(tl, ix.re[0], ix.ce[1]),
                     ld(tl, ix.re[1], ix.ce[0]), ld(tl, ix.re[1], ix.ce[1]));
}

// reciprocal of a pivot: 1/(x + i y) = (x - i y) / (x^2 + y^2).  The real reciprocal is MUFU.RCP64H
// (rcp.approx.ftz.f64, ~20 bits) plus two Newton steps (relative error ~1e-16 for normal d); an exactly
// zero pivot (singular column: every candidate was 0) gives multipliers 0, so det stays exactly 0, not NaN.
// |pivot|^2 must be a normal double (|pivot| in ~[1e-154, 1e154]); outside, det over/underflows anyway.
__device__ __forceinline__ c128 crecip(c128 p) {
    const double d = fma(p.x, p.x, p.y * p.y);
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    double e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    r = d > 0.0 ? r : 0.0;
    return make_double2(p.x * r, -p.y * r);
}

// pivot key: high word of |re| + |im| (>= 0, so the integer order is the floating-point order up to
// the 2^-20 of the dropped low word): near-maximal pivots are as good as the maximal one for stability,
// and integer compares keep the argmax chain off the FP64 pipe
__device__ __forceinline__ int pivot_key(double re, double im) { return __double2hiint(fabs(re) + fabs(im)); }

// number of multipliers in the first i columns of L (column c holds rows c+1 .. N-1)
template <int N> __host__ __device__ constexpr int lcol_base(int i) { return i * (N - 1) - i * (i - 1) / 2; }

// Hybrid elimination (N >= 4): K = N-4 steps of LEFT-LOOKING LU with partial pivoting, then the closed
// form of the 4x4 Schur complement ("up to 4x4 analytic, LU above", applied to the
// trailing block as well).  det = (+-) piv_0 ... piv_{K-1} det4(S).  Left-looking: column j of the minor
// is gathered from shared memory only after the pivots of columns < j are known, in the lane's current
// row order, so the only data ever exchanged is the active column and the multipliers.
//
// The state of the K pivot steps (row order, multipliers, pivot product) depends only on the row tuple
// and the first K columns, and the six 2x2 minors of trailing columns (K, K+1) only on those and the
// two columns.  Minors are stored row tuple by row tuple with column tuples in lexicographic order
// (term_builder.cpp), so consecutive minors of a warp share these prefixes and the state is kept in
// registers across them (minors_kernel); a minor whose prefix differs starts a fresh elimination.
// Every minor is still the pivoted LU of its own matrix: identical leading work is not repeated.
//
// The multipliers of columns < R live in shared memory (Ls: this thread's slot, entry e at Ls[e * NT],
// conflict free also for the per-lane dynamic row of the exchange), those of columns R..K-1 in registers.
// Rows are exchanged only during the K pivot steps; the 4 trailing rows keep whatever order the
// pivoting left them in (det4 is evaluated in that order, the sign is already in `detp`).
// `tb` = byte address of tile[0][lane]; row / column byte offsets are 12 * a_i * 512 and b_j * 512.
template <int N, int R, int NT>
struct LuState {
    static constexpr int K = N - 4;
    static constexpr int KR = (K - R > 0) ? K - R : 1;
    uint32_t rb[N];                    // byte offset of the row at position r (per-lane order)
    double Lr[N][KR], Li[N][KR];       // register multipliers: column i >= R at [r][i - R], r > i
    c128 detp;                         // (+-) product of the K pivots
    c128 s[6];                         // 2x2 minors of trailing columns (K, K+1), row pairs 01 02 03 12 13 23
    c128 c3[4];                        // signed 3x3 minors of trailing columns (K, K+1, K+2)

    // c[r] -= L[r][i] c[i] for r > i: the elimination of column i applied to the active column
    template <int I>
    __device__ __forceinline__ void apply_column(const c128* Ls, double (&cr)[N], double (&ci)[N]) const {
#pragma unroll
        for (int r = I + 1; r < N; ++r) {
            double lr, li;
            if constexpr (I < R) { const c128 l = Ls[(lcol_base<N>(I) + r - I - 1) * NT]; lr = l.x; li = l.y; }
            else { lr = Lr[r][I - R]; li = Li[r][I - R]; }
            cr[r] = fma(-lr, cr[I], fma(li, ci[I], cr[r]));
            ci[r] = fma(-lr, ci[I], fma(-li, cr[I], ci[r]));
        }
    }
    template <int I, int J>
    __device__ __forceinline__ void apply_columns_below(const c128* Ls, double (&cr)[N], double (&ci)[N]) const {
        if constexpr (I < J) { apply_column<I>(Ls, cr, ci); apply_columns_below<I + 1, J>(Ls, cr, ci); }
    }
    __device__ __forceinline__ void load_column(const unsigned char* tb, uint32_t cbj, double (&cr)[N], double (&ci)[N]) const {
#pragma unroll
        for (int r = 0; r < N; ++r) {
            const c128 v = *reinterpret_cast<const c128*>(tb + (rb[r] + cbj));
            cr[r] = v.x; ci[r] = v.y;
        }
    }
    // pivot step J on column offset cbj (rows in the order left by steps < J)
    template <int J>
    __device__ __forceinline__ void pivot_step(const unsigned char* tb, c128* Ls, uint32_t cbj) {
        double cr[N], ci[N];
        load_column(tb, cbj, cr, ci);
        apply_columns_below<0, J>(Ls, cr, ci);
        // pivot = candidate with the largest |re| + |im| (LAPACK izamax rule) to 2^-20, first maximum wins
        int p = J;
        int best = pivot_key(cr[J], ci[J]);
#pragma unroll
        for (int r = J + 1; r < N; ++r) {
            const int m = pivot_key(cr[r], ci[r]);
            if (m > best) { best = m; p = r; }
        }
        // exchange positions J and p: active column, row offsets, multipliers of columns < J
        double pr = cr[J], pi = ci[J];
        uint32_t po = rb[J];
#pragma unroll
        for (int r = J + 1; r < N; ++r) {
            const bool hit = (p == r);
            const double tr = cr[r], ti = ci[r];
            const uint32_t to = rb[r];
            cr[r] = hit ? cr[J] : tr; ci[r] = hit ? ci[J] : ti; rb[r] = hit ? rb[J] : to;
            pr = hit ? tr : pr; pi = hit ? ti : pi; po = hit ? to : po;
        }
        rb[J] = po;
        if (R > 0 && J > 0 && p != J) {                         // shared-memory columns: swap rows J and p
#pragma unroll
            for (int i = 0; i < (J < R ? J : R); ++i) {
                c128* ej = Ls + (lcol_base<N>(i) + J - i - 1) * NT;
                c128* ep = Ls + (lcol_base<N>(i) + p - i - 1) * NT;
                const c128 a = *ej, b = *ep;
                *ej = b; *ep = a;
            }
        }
#pragma unroll
        for (int i = R; i < J; ++i) {                           // register columns: exchange by selects
            double gr = Lr[J][i - R], gi = Li[J][i - R];
#pragma unroll
            for (int r = J + 1; r < N; ++r) {
                const bool hit = (p == r);
                const double ar = Lr[r][i - R], ai = Li[r][i - R];
                Lr[r][i - R] = hit ? Lr[J][i - R] : ar; Li[r][i - R] = hit ? Li[J][i - R] : ai;
                gr = hit ? ar : gr; gi = hit ? ai : gi;
            }
            Lr[J][i - R] = gr; Li[J][i - R] = gi;
        }
        const c128 piv = make_double2(pr, pi);
        detp = (J == 0) ? piv : cmul(detp, piv);
        if (p != J) { detp.x = -detp.x; detp.y = -detp.y; }
        const c128 inv = crecip(piv);
#pragma unroll
        for (int r = J + 1; r < N; ++r) {
            const double lr = cr[r] * inv.x - ci[r] * inv.y, li = cr[r] * inv.y + ci[r] * inv.x;
            if constexpr (J < R) Ls[(lcol_base<N>(J) + r - J - 1) * NT] = make_double2(lr, li);
            else { Lr[r][J - R] = lr; Li[r][J - R] = li; }
        }
    }
    template <int J>
    __device__ __forceinline__ void pivot_steps(const unsigned char* tb, c128* Ls, const uint32_t (&cb)[N]) {
        if constexpr (J < K) { pivot_step<J>(tb, Ls, cb[J]); pivot_steps<J + 1>(tb, Ls, cb); }
    }
    // the K pivot steps of a new (row tuple, leading K columns)
    __device__ __forceinline__ void start(const unsigned char* tb, c128* Ls, const uint32_t (&rb0)[N], const uint32_t (&cb)[N]) {
#pragma unroll
        for (int r = 0; r < N; ++r) rb[r] = rb0[r];
        detp = make_double2(1.0, 0.0);                          // N = 4: no pivot step, the minor is its own Schur complement
        pivot_steps<0>(tb, Ls, cb);
    }
    // one trailing column: apply the K eliminations, keep the last 4 entries (the column of the Schur complement)
    __device__ __forceinline__ void schur_column(const unsigned char* tb, const c128* Ls, uint32_t cbj, c128 (&t)[4]) const {
        double cr[N], ci[N];
        load_column(tb, cbj, cr, ci);
        apply_columns_below<0, K>(Ls, cr, ci);
#pragma unroll
        for (int r = 0; r < 4; ++r) t[r] = make_double2(cr[K + r], ci[K + r]);
    }
    // level 1: columns K, K+1 of the minor -> s = 2x2 minors of Schur columns 0, 1 over the row pairs
    __device__ __forceinline__ void pair_from(const c128 (&t0)[4], const c128 (&t1)[4]) {
        int k = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = a + 1; b < 4; ++b) s[k++] = det2(t0[a], t1[a], t0[b], t1[b]);
    }
    __device__ __forceinline__ void first_pair(const unsigned char* tb, const c128* Ls, uint32_t cba, uint32_t cbb) {
        c128 t0[4], t1[4];
        schur_column(tb, Ls, cba, t0);
        schur_column(tb, Ls, cbb, t1);
        pair_from(t0, t1);
    }
    // level 2: column K+2 -> signed 3x3 minors of Schur columns 0..2: c3[r] = (-1)^(r+3) det(rows != r),
    // each expanded along its last column in the 2x2 minors s
    __device__ __forceinline__ void third_from(const c128 (&t)[4]) {
        const c128 m0 = cfma(t[3], s[3], cfnma(t[2], s[4], cmul(t[1], s[5])));   // rows 1,2,3
        const c128 m1 = cfma(t[3], s[1], cfnma(t[2], s[2], cmul(t[0], s[5])));   // rows 0,2,3
        const c128 m2 = cfma(t[3], s[0], cfnma(t[1], s[2], cmul(t[0], s[4])));   // rows 0,1,3
        const c128 m3 = cfma(t[2], s[0], cfnma(t[1], s[1], cmul(t[0], s[3])));   // rows 0,1,2
        c3[0] = make_double2(-m0.x, -m0.y); c3[1] = m1; c3[2] = make_double2(-m2.x, -m2.y); c3[3] = m3;
    }
    __device__ __forceinline__ void third_column(const unsigned char* tb, const c128* Ls, uint32_t cbj) {
        c128 t[4];
        schur_column(tb, Ls, cbj, t);
        third_from(t);
    }
    // level 3: last column -> det = detp * sum_r S[r][3] c3[r]  (Laplace expansion of the 4x4 Schur
    // complement along its last column); two independent partial sums keep the dependency chain short
    __device__ __forceinline__ c128 finish_from(const c128 (&t)[4]) const {
        const c128 e0 = cfma(t[1], c3[1], cmul(t[0], c3[0]));
        const c128 e1 = cfma(t[3], c3[3], cmul(t[2], c3[2]));
        return cmul(detp, cadd(e0, e1));
    }
    __device__ __forceinline__ c128 finish(const unsigned char* tb, const c128* Ls, uint32_t cbj) const {
        c128 t[4];
        schur_column(tb, Ls, cbj, t);
        return finish_from(t);
    }
};

}  // namespace wick

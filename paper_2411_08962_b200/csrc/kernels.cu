// Device kernels of the hot path, sm_100a.  See kernels.cuh for the on-chip layout.
//
//  a3  stage_tile          : propagators of 32 site-times -> shared memory, element-major / lane-minor
//  a4  minors_kernel<N>    : one unique minor per (warp iteration, lane = site).  N <= 3: analytic
//                            expression; N >= 4: N-4 steps of LU with partial pivoting, then the analytic 4x4
//                            expression of the Schur complement.  The LU is
//                            LEFT-LOOKING: column j of the minor is gathered from shared memory only
//                            after the pivots of columns < j are known, in the lane's current row
//                            order, so the only data that ever has to be exchanged in registers is
//                            the active column and the multipliers (O(N^2) selects, not O(N^3)).
//  a5  reduce_flat / reduce_outer : sigma(x,t) = sum_k w_k MU[uid_k] MD[did_k]  (Eq. A1-A5)
//  a6  finalize_sigma, project    : fixed-order sum of the partials, momentum phases, fixed tree over sites
#include <algorithm>
#include <vector>

#include "kernels.cuh"
#include "lu_device.cuh"

namespace wick {

static thread_local int64_t g_launches = 0;
int64_t launch_counter_get() { return g_launches; }
int64_t launch_counter_reset() { const int64_t v = g_launches; g_launches = 0; return v; }

// Optional per-launch timing (bench.py's roofline): CUDA events on the launching stream around every
// kernel of a class, read back with profile_read().  Off by default; thread-local.
struct ProfRec { cudaEvent_t a, b; int cls; };
static thread_local bool g_prof_on = false;
static thread_local std::vector<ProfRec> g_prof;
void profile_enable(bool on) {
    g_prof_on = on;
    if (!on) {                                                   // records never read are dropped with their events
        for (ProfRec& r : g_prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
        g_prof.clear();
    }
}
struct ProfScope {
    ProfRec r; cudaStream_t s; bool on;
    ProfScope(int cls, cudaStream_t stream) : s(stream), on(g_prof_on) {
        if (!on) return;
        r.cls = cls;
        cudaEventCreate(&r.a); cudaEventCreate(&r.b);
        cudaEventRecord(r.a, s);
    }
    ~ProfScope() { if (on) { cudaEventRecord(r.b, s); g_prof.push_back(r); } }
};
cudaError_t profile_read(double ms[PROF_CLASSES], int64_t count[PROF_CLASSES]) {
    for (int c = 0; c < PROF_CLASSES; ++c) { ms[c] = 0.0; count[c] = 0; }
    cudaError_t err = cudaSuccess;
    for (ProfRec& r : g_prof) {
        float t = 0.f;
        cudaError_t e = cudaEventSynchronize(r.b);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, r.a, r.b);
        if (e != cudaSuccess) err = e;
        ms[r.cls] += t; count[r.cls] += 1;
        cudaEventDestroy(r.a); cudaEventDestroy(r.b);
    }
    g_prof.clear();
    return err;
}

template <int N> struct MinorCfg {
    // columns of L kept in shared memory (the rest of the N-4 columns are registers)
    static constexpr int kSmemCols = (N <= 10) ? 0 : (N == 11 ? 2 : 5);
    static constexpr int kThreads = (N <= 11) ? 256 : 128;
    static constexpr int kMinBlocks = (N <= 6) ? 2 : 1;
    static constexpr size_t kSmem = size_t(TILE_BYTES) + size_t(lcol_base<(N > 1 ? N : 2)>(kSmemCols)) * 16 * kThreads;
};

// Minor descriptor (built on the host, contract.cu: pack_minor_desc): the row and column indices as
// 4-bit fields in PROCESSING order.  n <= 8: one 64-bit word (rows in the low half, columns in the high half),
// ascending tuples, result stored at the descriptor's own position.  n >= 9: two 64-bit words
//   w0 = rows (48 bits) | output minor id, low 16 bits;   w1 = columns (48 bits) | output id, high 15 bits | sign
// where the columns may be listed descending (sign = parity of the reversal) so that tuples that differ in their
// SMALL indices share leading columns too, and the descriptors are sorted for sharing, not by minor id.
// One load per minor, no dependent second load.
template <int N> struct Desc {
    static constexpr int kWords = (N <= 8) ? 1 : 2;
    unsigned long long w[kWords];
    __device__ __forceinline__ static Desc load(const unsigned long long* tab, int m) {
        Desc d;
        if constexpr (kWords == 1) d.w[0] = __ldg(tab + m);
        else { const ulonglong2 v = __ldg(reinterpret_cast<const ulonglong2*>(tab) + m); d.w[0] = v.x; d.w[1] = v.y; }
        return d;
    }
    __device__ __forceinline__ unsigned long long rows_bits() const { return kWords == 1 ? (w[0] & (N <= 4 ? 0x7fffffffull : 0xffffffffull)) : (w[0] & 0xffffffffffffull); }
    __device__ __forceinline__ unsigned long long cols_bits() const { return kWords == 1 ? (w[0] >> 32) : (w[kWords - 1] & 0xffffffffffffull); }
    // where the determinant goes (m = position of the descriptor) and whether it is negated
    __device__ __forceinline__ int out_index(int m) const {
        if constexpr (kWords == 1) return m;
        else return int(w[0] >> 48) | (int((w[kWords - 1] >> 48) & 0x7fffull) << 16);
    }
    // n <= 4: bit 31 of the word (above the 4 row fields) flags a negated result (Jacobi complementary minors, contract.cu)
    __device__ __forceinline__ bool negate() const {
        if constexpr (kWords == 1) return N <= 4 ? ((w[0] >> 31) & 1ull) != 0 : false;
        else return (w[kWords - 1] >> 63) != 0;
    }
    __device__ __forceinline__ c128 signed_result(c128 det) const { return negate() ? make_double2(-det.x, -det.y) : det; }
    __device__ __forceinline__ uint32_t row(int i) const {
        if constexpr (kWords == 1) return (uint32_t(w[0]) >> (4 * i)) & 15u;
        else return uint32_t(w[0] >> (4 * i)) & 15u;
    }
    __device__ __forceinline__ uint32_t col(int i) const {
        if constexpr (kWords == 1) return (uint32_t(w[0] >> 32) >> (4 * i)) & 15u;
        else return uint32_t(w[1] >> (4 * i)) & 15u;
    }
};

template <int N>
__global__ void __launch_bounds__(MinorCfg<N>::kThreads, MinorCfg<N>::kMinBlocks)
minors_kernel(const c128* __restrict__ P, int64_t st0, int64_t n_st_total, int S_b,
              const unsigned long long* __restrict__ desc, int n_minors, int chunk, c128* __restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    c128* tile = reinterpret_cast<c128*>(smem_raw);
    constexpr int NT = MinorCfg<N>::kThreads;
    const int g = blockIdx.x;
    const int64_t st_first = st0 + int64_t(g) * GROUP;
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);   // shuffle: the compiler then treats everything derived from the warp index as warp uniform
    const int m_begin = blockIdx.y * chunk;
    const int m_end = min(n_minors, m_begin + chunk);
    // N <= 2: warp w takes minors m_begin + w, + NT/32, ...; N >= 3: a contiguous piece of the chunk, so
    // that consecutive minors share their row tuple and leading columns (see LuState)
    constexpr int kStride = (N <= 2) ? NT / 32 : 1;
    int m = (N <= 2) ? m_begin + warp : m_begin + warp * (chunk / (NT / 32));
    const int m_stop = (N <= 2) ? m_end : min(m_end, m + chunk / (NT / 32));
    Desc<N> dn;                                                // descriptor of the next minor, fetched one iteration ahead
    if (m < m_stop) dn = Desc<N>::load(desc, m);
    stage_tile(tile, P, st_first, n_st_total, NT);
    __syncthreads();
    const c128* tl = tile + lane;
    // every lane stores: the rows of `out` are S_b >= 32 * gridDim.x wide, lanes beyond the end of the lattice hold zero tiles
    c128* outp = out + int64_t(g) * GROUP + lane;
    if constexpr (N == 3) {
        // 3x3: the cofactors of the last column depend on (row tuple, first two columns) only and are kept
        // across consecutive minors; per minor 3 loads and 3 complex multiply-adds
        c128 cof[3];
        unsigned long long prow = ~0ull, pcol = 0;
        for (; m < m_stop; ++m) {
            const Desc<N> dc = dn;
            if (m + 1 < m_stop) dn = Desc<N>::load(desc, m + 1);
            const unsigned long long rws = dc.rows_bits(), cls = dc.cols_bits();
            int re[3];
#pragma unroll
            for (int i = 0; i < 3; ++i) re[i] = int(dc.row(i)) * 12;
            if (rws != prow || ((cls ^ pcol) & 0xffull) != 0) {
                const int c0 = int(dc.col(0)), c1 = int(dc.col(1));
                const c128 a0 = ld(tl, re[0], c0), a1 = ld(tl, re[1], c0), a2 = ld(tl, re[2], c0);
                const c128 b0 = ld(tl, re[0], c1), b1 = ld(tl, re[1], c1), b2 = ld(tl, re[2], c1);
                cof[0] = det2(a1, b1, a2, b2);                   // rows 1,2
                cof[1] = det2(a2, b2, a0, b0);                   // -(rows 0,2)
                cof[2] = det2(a0, b0, a1, b1);                   // rows 0,1
            }
            const int c2 = int(dc.col(2));
            const c128 det = cfma(ld(tl, re[2], c2), cof[2], cfma(ld(tl, re[1], c2), cof[1], cmul(ld(tl, re[0], c2), cof[0])));
            prow = rws; pcol = cls;
            outp[int64_t(m) * S_b] = dc.signed_result(det);
        }
    } else if constexpr (N <= 2) {
        for (; m < m_stop; m += kStride) {
            const Desc<N> dc = dn;
            if (m + kStride < m_stop) dn = Desc<N>::load(desc, m + kStride);
            Idx<N> ix;
#pragma unroll
            for (int i = 0; i < N; ++i) { ix.re[i] = int(dc.row(i)) * 12; ix.ce[i] = int(dc.col(i)); }
            const c128 det = det_small<N>(tl, ix);
            outp[int64_t(m) * S_b] = dc.signed_result(det);
        }
    } else {
        constexpr int K = N - 4;
        constexpr uint32_t kRowStep = 12 * GROUP * 16, kColStep = GROUP * 16;
        constexpr unsigned long long kLead = (1ull << (4 * K)) - 1, kLeadPair = (1ull << (4 * (K + 2))) - 1,
                                     kLead3 = (1ull << (4 * (K + 3))) - 1;
        const unsigned char* tb = reinterpret_cast<const unsigned char*>(tl);
        c128* Ls = tile + TILE_ELEMS + threadIdx.x;
        LuState<N, MinorCfg<N>::kSmemCols, NT> lu;
        unsigned long long prow = ~0ull, pcol = 0;              // no index set has all 64 bits set: the first minor starts fresh
        for (; m < m_stop; ++m) {
            const Desc<N> dc = dn;
            if (m + 1 < m_stop) dn = Desc<N>::load(desc, m + 1);
            const unsigned long long rws = dc.rows_bits(), diff = dc.cols_bits() ^ pcol;
            const bool fresh = (rws != prow) || (diff & kLead) != 0;
            if (fresh) {
                uint32_t rb[N], cb[N];
#pragma unroll
                for (int i = 0; i < N; ++i) { rb[i] = dc.row(i) * kRowStep; cb[i] = dc.col(i) * kColStep; }
                lu.start(tb, Ls, rb, cb);
            }
            const bool new_pair = fresh || (diff & kLeadPair) != 0;
            if (new_pair) lu.first_pair(tb, Ls, dc.col(K) * kColStep, dc.col(K + 1) * kColStep);
            if (new_pair || (diff & kLead3) != 0) lu.third_column(tb, Ls, dc.col(K + 2) * kColStep);
            const c128 det = lu.finish(tb, Ls, dc.col(K + 3) * kColStep);
            prow = rws; pcol = dc.cols_bits();
            outp[int64_t(dc.out_index(m)) * S_b] = dc.signed_result(det);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// a4 for minors of size n >= 8 through Jacobi's complementary-minor identity (optional, flag
// WICK_CONTRACT_JACOBI):  det A[I, J] = (-1)^(sum I + sum J) det A  det (A^-1)[J^c, I^c].
// inverse12_kernel: 16 lanes per site invert its 12x12 propagator in registers (Gauss-Jordan with partial pivoting, same
// pivot rule as the LU kernels, pivot row broadcast by shuffles) and return det A; the (12-n) x (12-n) minors of the
// inverse then go through minors_kernel<12-n>.
// A singular propagator has no inverse: its site gets det = 0 and a zero matrix (every minor 0); use the LU path for such data.
// ---------------------------------------------------------------------------------------------
constexpr int INV_THREADS = 128;

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const uint32_t d = static_cast<uint32_t>(__cvta_generic_to_shared(smem_dst));
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ double shfl16(double v, int src) { return __shfl_sync(0xffffffffu, v, src, 16); }

// 16 lanes per site (12 used): lane = row of the propagator, its 12 entries in registers.  Gauss-Jordan in place without
// moving rows: step k picks, among the lanes that have not been a pivot row yet, the one with the largest |re| + |im| in
// column k (compared to 2^-16, first wins); every lane then does  own[c] -= g * pivot_row[c]  with g = own[k] / piv (the pivot lane itself with
// g = 1 - 1/piv, which scales it by 1/piv), and column k is replaced by the column of the inverse.  With p_k the pivot
// lane of step k the lane p_i ends up holding (A^-1)[i][p_m] in register m.
// Result of invert12 for one lane and one matrix: row `my_step` of the inverse, entry m belongs to column p_m (4-bit fields of perm).
struct InvRow { double re[12], im[12]; int my_step; unsigned long long perm; c128 det; bool singular; };

// NM matrices can be inverted TOGETHER (independent instruction streams in one thread; inverse12_kernel, the only user
// left, takes one: the fused kernel has its own four-lanes-per-matrix routine, invert12_rows3 below).
// The pivot row of a step and the reciprocal of its pivot reach the other lanes of the site by shuffles (52 per step; the
// round-2 profile showed the LSU data pipe as the limiter, 82 % busy, and a single-lane STS.128 costs it the same four
// cycles as a full-warp one, so the earlier shared-memory broadcast, 13 stores + 13 loads, was no cheaper).
// The steps are software-pipelined ("look-ahead"): step k updates column k+1 FIRST, then starts the pivot search of step
// k+1 (one packed {key, lane} word per lane, four max-shuffles) and the reciprocal of every lane's own candidate, and only
// then updates the other ten columns, so the search, the MUFU and the Newton steps run under the 40 DFMAs of the update
// instead of in front of them.  The packed word keeps the pivot key to 2^-16 (the low four bits hold the lane, smaller
// lane wins ties).

__device__ __forceinline__ unsigned packed_pivot_key(bool used, double re, double im, int sub) {
    return used ? 0u : ((((unsigned(pivot_key(re, im)) >> 4) + 1u) << 4) | unsigned(15 - sub));
}
__device__ __forceinline__ int pivot_lane16(unsigned pk) {
#pragma unroll
    for (int off = 8; off > 0; off >>= 1) pk = max(pk, __shfl_xor_sync(0xffffffffu, pk, off, 16));
    return 15 - int(pk & 15u);
}

template <int NM>
__device__ __forceinline__ void invert12(const c128* const (&P)[NM], int64_t st, bool row_ok, int sub, InvRow (&R)[NM]) {
#pragma unroll
    for (int q = 0; q < NM; ++q) {
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            c128 v = make_double2(0.0, 0.0);
            if (row_ok) v = __ldg(P[q] + st * 144 + sub * 12 + c);
            R[q].re[c] = v.x; R[q].im[c] = v.y;
        }
        R[q].my_step = 0; R[q].perm = 0; R[q].det = make_double2(1.0, 0.0); R[q].singular = false;
    }
    bool used[NM];                                                          // idle lanes never become pivots
    int who[NM];                                                            // pivot lane of the coming step
    c128 my_ip[NM];                                                         // reciprocal of this lane's candidate
#pragma unroll
    for (int q = 0; q < NM; ++q) {
        used[q] = sub >= 12;
        who[q] = pivot_lane16(packed_pivot_key(used[q], R[q].re[0], R[q].im[0], sub));
        my_ip[q] = crecip(make_double2(R[q].re[0], R[q].im[0]));
    }
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        bool is_p[NM];
#pragma unroll
        for (int q = 0; q < NM; ++q) {
            is_p[q] = (sub == who[q]);
            R[q].perm |= (unsigned long long)who[q] << (4 * k);
            if (is_p[q]) { used[q] = true; R[q].my_step = k; }
        }
#pragma unroll
        for (int q = 0; q < NM; ++q) {
            double (&re)[12] = R[q].re;
            double (&im)[12] = R[q].im;
            double pr[12], pi[12];
#pragma unroll
            for (int c = 0; c < 12; ++c) { pr[c] = shfl16(re[c], who[q]); pi[c] = shfl16(im[c], who[q]); }
            const c128 ip = make_double2(shfl16(my_ip[q].x, who[q]), shfl16(my_ip[q].y, who[q]));
            const c128 piv = make_double2(pr[k], pi[k]);
            R[q].singular = R[q].singular || (piv.x == 0.0 && piv.y == 0.0);
            R[q].det = cmul(R[q].det, piv);
            // g = own[k] / piv for the other rows, 1 - 1/piv for the pivot row (which scales it by 1/piv)
            c128 g = cmul(make_double2(re[k], im[k]), ip);
            if (is_p[q]) g = make_double2(1.0 - ip.x, -ip.y);
            auto update = [&](int c) {
                re[c] = fma(-g.x, pr[c], fma(g.y, pi[c], re[c]));
                im[c] = fma(-g.x, pi[c], fma(-g.y, pr[c], im[c]));
            };
            if (k < 11) {                                                   // look-ahead: everything step k+1 waits for
                update(k + 1);
                who[q] = pivot_lane16(packed_pivot_key(used[q], re[k + 1], im[k + 1], sub));
                my_ip[q] = crecip(make_double2(re[k + 1], im[k + 1]));
            }
#pragma unroll
            for (int c = 0; c < 12; ++c)
                if (c != k && c != k + 1) update(c);
            re[k] = is_p[q] ? ip.x : -g.x;
            im[k] = is_p[q] ? ip.y : -g.y;
        }
    }
#pragma unroll
    for (int q = 0; q < NM; ++q) {
        // sign of the permutation k -> p_k
        int inv_count = 0;
#pragma unroll
        for (int a = 0; a < 12; ++a)
#pragma unroll
            for (int b = a + 1; b < 12; ++b) inv_count += (int(R[q].perm >> (4 * a)) & 15) > (int(R[q].perm >> (4 * b)) & 15);
        if (inv_count & 1) { R[q].det.x = -R[q].det.x; R[q].det.y = -R[q].det.y; }
        if (R[q].singular) R[q].det = make_double2(0.0, 0.0);
    }
}

// store the lane's row of the inverse into a matrix whose element (r, c) sits at dst[(12 r + c) * stride]
__device__ __forceinline__ void store_inv_row(const InvRow& R, c128* dst_matrix, int stride) {
    c128* dst = dst_matrix + R.my_step * 12 * stride;
#pragma unroll
    for (int m = 0; m < 12; ++m) {
        const int col = int(R.perm >> (4 * m)) & 15;
        dst[col * stride] = R.singular ? make_double2(0.0, 0.0) : make_double2(R.re[m], R.im[m]);
    }
}

__global__ void __launch_bounds__(INV_THREADS)
inverse12_kernel(const c128* __restrict__ P, int64_t st0, int64_t n_st_total, int64_t n_batch, c128* __restrict__ inv_out, c128* __restrict__ det_out) {
    const int sub = threadIdx.x & 15;                                       // row
    const int64_t site = (int64_t(blockIdx.x) * INV_THREADS + threadIdx.x) >> 4;   // site within the batch
    const int64_t st = st0 + site;
    const bool live = site < n_batch && st < n_st_total;
    const bool row_ok = live && sub < 12;
    InvRow R[1];
    const c128* const Pq[1] = {P};
    invert12<1>(Pq, st, row_ok, sub, R);
    if (live && sub == 0) det_out[site] = R[0].det;
    if (row_ok) store_inv_row(R[0], inv_out + site * 144, 1);
}

// Fused Jacobi path for lists whose BOTH flavours have 8 <= n <= 11 and whose term count is of the order of the number of
// unique minors (Li-7-sized lists): per site both propagators are inverted in registers, the inverses go to shared
// memory, and the threads of the CTA share the flat term list:
//   sigma = det U det D sum_k w'_k det (U^-1)[J_u^c, I_u^c] det (D^-1)[J_d^c, I_d^c],   w'_k = w_k (-1)^(sum of the index sets)
// Nothing but the propagators is read from and sigma written to global memory: 4608 B per site-time.
//
// Inversion: FOUR lanes per matrix, three rows each (all 32 lanes busy; with one row per lane 12 of 16 are).  The profile of
// the row-per-lane version showed the LSU data pipe as the limiter (82 % busy): every lane needs the whole pivot row every
// step, 52 shuffles per step whatever the number of lanes a matrix is spread over, so three rows per lane cut that
// traffic per matrix four times (8 matrices per warp instead of 2).  Same Gauss-Jordan without row moves, same look-ahead
// as invert12: step k updates column k+1 first, every lane picks its best unused row of that column (its candidate),
// starts the pivot search of step k+1 over the four lanes (two max-shuffles on a packed {key, row} word) and the reciprocal
// of its candidate, then updates the other columns; the next step's shuffles read every lane's candidate row through
// two selp.f64 per value.
constexpr int JF_THREADS = 128;
constexpr int JF_SITES = 16;                                                // 32 lane groups: 16 sites x 2 flavours

struct InvRows3 { double re[3][12], im[3][12]; int my_step[3]; unsigned long long perm; c128 det; bool singular; };

__device__ __forceinline__ double shfl4(double v, int src) { return __shfl_sync(0xffffffffu, v, src, 4); }
// x_loc by two selp.f64 (the plain ternaries compile to a divergent three-way branch full of register moves)
__device__ __forceinline__ double sel3(int loc, double x0, double x1, double x2) {
    double r;
    asm("{\n\t.reg .pred p0, p1;\n\tsetp.eq.s32 p0, %4, 0;\n\tsetp.eq.s32 p1, %4, 1;\n\tselp.f64 %0, %2, %3, p1;\n\tselp.f64 %0, %1, %0, p0;\n\t}"
        : "=&d"(r) : "d"(x0), "d"(x1), "d"(x2), "r"(loc));
    return r;
}

// this lane's best unused row of column k: packed {key to 2^-16, 15 - global row} (0 if all three are used), its position
__device__ __forceinline__ unsigned local_candidate(const InvRows3& R, const bool (&used)[3], int k, int l, int& loc) {
    unsigned best = 0u;
    loc = 0;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const unsigned pk = used[j] ? 0u : ((((unsigned(pivot_key(R.re[j][k], R.im[j][k])) >> 4) + 1u) << 4) | unsigned(15 - (3 * l + j)));
        if (pk > best) { best = pk; loc = j; }
    }
    return best;
}

__device__ __forceinline__ void invert12_rows3(const c128* __restrict__ P, bool ok, int l, InvRows3& R) {
#pragma unroll
    for (int j = 0; j < 3; ++j) {
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            c128 v = make_double2(0.0, 0.0);
            if (ok) v = __ldg(P + (3 * l + j) * 12 + c);
            R.re[j][c] = v.x; R.im[j][c] = v.y;
        }
        R.my_step[j] = 0;
    }
    R.perm = 0; R.det = make_double2(1.0, 0.0); R.singular = false;
    bool used[3] = {false, false, false};
    c128 my_ip;
    unsigned pk;
    int loc;                                                                // this lane's candidate row (the pivot row if the lane wins)
    pk = local_candidate(R, used, 0, l, loc);
    my_ip = crecip(make_double2(sel3(loc, R.re[0][0], R.re[1][0], R.re[2][0]), sel3(loc, R.im[0][0], R.im[1][0], R.im[2][0])));
    pk = max(pk, __shfl_xor_sync(0xffffffffu, pk, 1, 4));
    pk = max(pk, __shfl_xor_sync(0xffffffffu, pk, 2, 4));
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        const int p = 15 - int(pk & 15u);                                  // pivot row (global index), its lane
        const int owner = (p * 11) >> 5;                                    // p / 3 for p < 16
        double pr[12], pi[12];
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            pr[c] = shfl4(sel3(loc, R.re[0][c], R.re[1][c], R.re[2][c]), owner);
            pi[c] = shfl4(sel3(loc, R.im[0][c], R.im[1][c], R.im[2][c]), owner);
        }
        const c128 ip = make_double2(shfl4(my_ip.x, owner), shfl4(my_ip.y, owner));
        const c128 piv = make_double2(pr[k], pi[k]);
        R.singular = R.singular || (piv.x == 0.0 && piv.y == 0.0);
        R.det = cmul(R.det, piv);
        R.perm |= (unsigned long long)p << (4 * k);
        bool is_p[3];
        c128 g[3];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            is_p[j] = (p == 3 * l + j);
            if (is_p[j]) { used[j] = true; R.my_step[j] = k; }
            // g = own[k] / piv for the other rows, 1 - 1/piv for the pivot row (which scales it by 1/piv)
            g[j] = cmul(make_double2(R.re[j][k], R.im[j][k]), ip);
            if (is_p[j]) g[j] = make_double2(1.0 - ip.x, -ip.y);
        }
        auto update = [&](int c) {
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                R.re[j][c] = fma(-g[j].x, pr[c], fma(g[j].y, pi[c], R.re[j][c]));
                R.im[j][c] = fma(-g[j].x, pi[c], fma(-g[j].y, pr[c], R.im[j][c]));
            }
        };
        if (k < 11) {                                                       // look-ahead: everything step k+1 waits for
            update(k + 1);
            pk = local_candidate(R, used, k + 1, l, loc);
            my_ip = crecip(make_double2(sel3(loc, R.re[0][k + 1], R.re[1][k + 1], R.re[2][k + 1]),
                                        sel3(loc, R.im[0][k + 1], R.im[1][k + 1], R.im[2][k + 1])));
            pk = max(pk, __shfl_xor_sync(0xffffffffu, pk, 1, 4));
            pk = max(pk, __shfl_xor_sync(0xffffffffu, pk, 2, 4));
        }
#pragma unroll
        for (int c = 0; c < 12; ++c)
            if (c != k && c != k + 1) update(c);
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            R.re[j][k] = is_p[j] ? ip.x : -g[j].x;
            R.im[j][k] = is_p[j] ? ip.y : -g[j].y;
        }
    }
    // sign of the permutation k -> p_k
    int inv_count = 0;
#pragma unroll
    for (int a = 0; a < 12; ++a)
#pragma unroll
        for (int b = a + 1; b < 12; ++b) inv_count += (int(R.perm >> (4 * a)) & 15) > (int(R.perm >> (4 * b)) & 15);
    if (inv_count & 1) { R.det.x = -R.det.x; R.det.y = -R.det.y; }
    if (R.singular) R.det = make_double2(0.0, 0.0);
}

// A: element (r, c) of site ls of the CTA at A[jf_elem(r, c, ls)]: site-minor layout (the 8 sites of a quarter warp read
// one 128-byte half of a 256-byte row, conflict free) with the site position rotated by the row, so that the lanes of a
// matrix, which store different rows of one column at a time, spread over the banks as well.
__device__ __forceinline__ int jf_elem(int r, int c, int ls) { return (r * 12 + c) * JF_SITES + ((ls + r) & (JF_SITES - 1)); }

// the lane's three rows of the inverse into that layout
__device__ __forceinline__ void store_inv_rows3_shared(const InvRows3& R, c128* A, int ls) {
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int m = 0; m < 12; ++m) {
            const int col = int(R.perm >> (4 * m)) & 15;
            A[jf_elem(R.my_step[j], col, ls)] = R.singular ? make_double2(0.0, 0.0) : make_double2(R.re[j][m], R.im[j][m]);
        }
}

template <int M>
__device__ __forceinline__ c128 small_minor(const c128* A, int ls, uint32_t idx) {   // rows = nibbles 0..3, columns = nibbles 4..7 of idx
    if constexpr (M == 0) return make_double2(1.0, 0.0);
    else {
        int r[M], c[M];
#pragma unroll
        for (int i = 0; i < M; ++i) { r[i] = int(idx >> (4 * i)) & 15; c[i] = int(idx >> (16 + 4 * i)) & 15; }
        auto a = [&](int i, int j) { return A[jf_elem(r[i], c[j], ls)]; };
        if constexpr (M == 1) return a(0, 0);
        else if constexpr (M == 2) return det2(a(0, 0), a(0, 1), a(1, 0), a(1, 1));
        else if constexpr (M == 3) {
            const c128 m0 = det2(a(1, 1), a(1, 2), a(2, 1), a(2, 2)), m1 = det2(a(1, 0), a(1, 2), a(2, 0), a(2, 2)), m2 = det2(a(1, 0), a(1, 1), a(2, 0), a(2, 1));
            return cfma(a(0, 2), m2, cfnma(a(0, 1), m1, cmul(a(0, 0), m0)));
        } else {
            // Laplace expansion over the row pairs (0,1) x (2,3): six products of complementary 2x2 minors
            const c128 s01 = det2(a(0, 0), a(0, 1), a(1, 0), a(1, 1)), s02 = det2(a(0, 0), a(0, 2), a(1, 0), a(1, 2)), s03 = det2(a(0, 0), a(0, 3), a(1, 0), a(1, 3));
            const c128 s12 = det2(a(0, 1), a(0, 2), a(1, 1), a(1, 2)), s13 = det2(a(0, 1), a(0, 3), a(1, 1), a(1, 3)), s23 = det2(a(0, 2), a(0, 3), a(1, 2), a(1, 3));
            const c128 t01 = det2(a(2, 0), a(2, 1), a(3, 0), a(3, 1)), t02 = det2(a(2, 0), a(2, 2), a(3, 0), a(3, 2)), t03 = det2(a(2, 0), a(2, 3), a(3, 0), a(3, 3));
            const c128 t12 = det2(a(2, 1), a(2, 2), a(3, 1), a(3, 2)), t13 = det2(a(2, 1), a(2, 3), a(3, 1), a(3, 3)), t23 = det2(a(2, 2), a(2, 3), a(3, 2), a(3, 3));
            c128 d = cmul(s01, t23);
            d = cfnma(s02, t13, d); d = cfma(s03, t12, d); d = cfma(s12, t03, d); d = cfnma(s13, t02, d); d = cfma(s23, t01, d);
            return d;
        }
    }
}

// STAGE_TERMS: the term records (32 B each) fit the CTA's shared memory beside the inverses (JF_TERMS_CAP) and are copied
// there once per CTA instead of being read through L1 / L2 in the term loop
template <int MU_, int MD_, bool STAGE_TERMS>
__global__ void __launch_bounds__(JF_THREADS, 2)
jacobi_fused_kernel(const c128* __restrict__ U, const c128* __restrict__ D, int64_t st0, int64_t n_valid,
                    const JacobiTerm* __restrict__ terms, int n_terms, c128* __restrict__ sigma) {
    extern __shared__ __align__(16) unsigned char jf_smem[];
    c128* inv_s = reinterpret_cast<c128*>(jf_smem);                        // [flavour][element][site] (jf_elem)
    c128* psum = inv_s + 2 * 144 * JF_SITES;                                // [term slot][site]
    c128* dets_s = psum + (JF_THREADS / JF_SITES) * JF_SITES;               // [flavour][site]
    const JacobiTerm* terms_s = reinterpret_cast<const JacobiTerm*>(dets_s + 2 * JF_SITES);
    if (STAGE_TERMS) {                                                      // term records: in flight during the inversions
        for (int i = threadIdx.x; i < 2 * n_terms; i += JF_THREADS)
            cp_async16(reinterpret_cast<uint4*>(dets_s + 2 * JF_SITES) + i, reinterpret_cast<const uint4*>(terms) + i);
    }
    {   // phase 1: lane group = (flavour, site), 4 lanes x 3 rows; U == D simply inverts the same matrix twice
        const int l = threadIdx.x & 3, grp = threadIdx.x >> 2;
        const int f = grp / JF_SITES, ls = grp % JF_SITES;
        const int64_t site = int64_t(blockIdx.x) * JF_SITES + ls;
        const bool ok = site < n_valid;
        InvRows3 R;
        invert12_rows3((f ? D : U) + (st0 + site) * 144, ok, l, R);
        store_inv_rows3_shared(R, inv_s + f * 144 * JF_SITES, ls);
        if (l == 0) dets_s[f * JF_SITES + ls] = R.det;
    }
    if (STAGE_TERMS) cp_async_wait_all();
    __syncthreads();
    // phase 2: lane = (site, one of 8 term slots); a half warp = the 16 sites of one term
    const int ls = threadIdx.x & (JF_SITES - 1), slot = threadIdx.x / JF_SITES;
    const c128* Ui = inv_s;
    const c128* Di = inv_s + 144 * JF_SITES;
    c128 acc = make_double2(0.0, 0.0);
#pragma unroll 4
    for (int k = slot; k < n_terms; k += JF_THREADS / JF_SITES) {
        uint2 h;
        c128 w;
        if (STAGE_TERMS) { h = *reinterpret_cast<const uint2*>(terms_s + k); w = *(reinterpret_cast<const c128*>(terms_s + k) + 1); }
        else { h = __ldg(reinterpret_cast<const uint2*>(terms + k)); w = __ldg(reinterpret_cast<const c128*>(terms + k) + 1); }
        acc = cfma(cmul(w, small_minor<MU_>(Ui, ls, h.x)), small_minor<MD_>(Di, ls, h.y), acc);
    }
    psum[slot * JF_SITES + ls] = acc;
    __syncthreads();
    if (threadIdx.x < JF_SITES) {                                           // fixed-order sum over the term slots
        const int64_t site = int64_t(blockIdx.x) * JF_SITES + threadIdx.x;
        c128 t = psum[threadIdx.x];
#pragma unroll
        for (int j = 1; j < JF_THREADS / JF_SITES; ++j) t = cadd(t, psum[j * JF_SITES + threadIdx.x]);
        if (site < n_valid) sigma[site] = cmul(t, cmul(dets_s[threadIdx.x], dets_s[JF_SITES + threadIdx.x]));
    }
}

constexpr size_t JF_SMEM = size_t(2 * 144 * JF_SITES + (JF_THREADS / JF_SITES) * JF_SITES + 2 * JF_SITES) * 16;
constexpr int JF_TERMS_CAP = 1024;                                          // 32 KB of records; two CTAs per SM still fit
constexpr size_t JF_SMEM_STAGED = JF_SMEM + size_t(JF_TERMS_CAP) * sizeof(JacobiTerm);

template <int MU_, int MD_>
static cudaError_t launch_jf(const c128* U, const c128* D, int64_t st0, int64_t n_valid, const JacobiTerm* terms, int n_terms,
                             c128* sigma, cudaStream_t stream) {
    const unsigned grid = unsigned((n_valid + JF_SITES - 1) / JF_SITES);
    if (n_terms <= JF_TERMS_CAP)
        jacobi_fused_kernel<MU_, MD_, true><<<grid, JF_THREADS, JF_SMEM + size_t(n_terms) * sizeof(JacobiTerm), stream>>>(U, D, st0, n_valid, terms, n_terms, sigma);
    else
        jacobi_fused_kernel<MU_, MD_, false><<<grid, JF_THREADS, JF_SMEM, stream>>>(U, D, st0, n_valid, terms, n_terms, sigma);
    return cudaGetLastError();
}

template <int MU_>
static cudaError_t launch_jf_d(int md, const c128* U, const c128* D, int64_t st0, int64_t n_valid, const JacobiTerm* terms, int n_terms,
                               c128* sigma, cudaStream_t stream) {
    switch (md) {
        case 1: return launch_jf<MU_, 1>(U, D, st0, n_valid, terms, n_terms, sigma, stream);
        case 2: return launch_jf<MU_, 2>(U, D, st0, n_valid, terms, n_terms, sigma, stream);
        case 3: return launch_jf<MU_, 3>(U, D, st0, n_valid, terms, n_terms, sigma, stream);
        case 4: return launch_jf<MU_, 4>(U, D, st0, n_valid, terms, n_terms, sigma, stream);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_jacobi_fused(int n_u, int n_d, const double2* U, const double2* D, int64_t st0, int64_t n_valid,
                                const JacobiTerm* terms, int64_t n_terms, double2* sigma, cudaStream_t stream) {
    if (n_valid <= 0) return cudaSuccess;
    ProfScope prof(PROF_MINORS_U, stream);
    ++g_launches;
    switch (12 - n_u) {
        case 1: return launch_jf_d<1>(12 - n_d, U, D, st0, n_valid, terms, int(n_terms), sigma, stream);
        case 2: return launch_jf_d<2>(12 - n_d, U, D, st0, n_valid, terms, int(n_terms), sigma, stream);
        case 3: return launch_jf_d<3>(12 - n_d, U, D, st0, n_valid, terms, int(n_terms), sigma, stream);
        case 4: return launch_jf_d<4>(12 - n_d, U, D, st0, n_valid, terms, int(n_terms), sigma, stream);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_inverse12(const double2* P, int64_t st0, int64_t n_st_total, int n_groups, double2* inv_out, double2* det_out,
                             int prof_cls, cudaStream_t stream) {
    if (n_groups == 0) return cudaSuccess;
    const int64_t n_batch = int64_t(n_groups) * GROUP;
    const int sites_per_cta = INV_THREADS / 16;
    ProfScope prof(prof_cls, stream);
    inverse12_kernel<<<unsigned((n_batch + sites_per_cta - 1) / sites_per_cta), INV_THREADS, 0, stream>>>(P, st0, n_st_total, n_batch, inv_out, det_out);
    ++g_launches;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// a4, 6x6 minors with a per-thread cache of Schur columns.  After the two pivot steps of a (row tuple, b0, b1) instance
// the Schur column of column index b is the same for every minor of the instance, whatever position b takes in it; the
// trie of minors_kernel re-evaluates it once per level (1143 columns per He-4 row tuple for ~100 distinct ones).  Here
// the columns b = 3..11 of the instance are computed once (9 x 4 complex = 576 B per thread in shared memory, entry e at
// Sc[e * NT + thread]: conflict free) and the levels read them; b = 2 (only possible as b2 of the instance (0,1)) is kept
// in registers.  One 256-thread CTA per SM (147 KB cache + 74 KB tile).
// ---------------------------------------------------------------------------------------------
constexpr int M6C_THREADS = 256;
constexpr size_t M6C_SMEM = size_t(TILE_BYTES) + size_t(9 * 4) * 16 * M6C_THREADS;

__global__ void __launch_bounds__(M6C_THREADS, 1)
minors6_cached_kernel(const c128* __restrict__ P, int64_t st0, int64_t n_st_total, int S_b,
                      const unsigned long long* __restrict__ desc, int n_minors, int chunk, c128* __restrict__ out) {
    constexpr int N = 6, K = 2, NT = M6C_THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    c128* tile = reinterpret_cast<c128*>(smem_raw);
    c128* Sc = tile + TILE_ELEMS + threadIdx.x;                          // this thread's cache: entry e at Sc[e * NT]
    const int g = blockIdx.x;
    const int64_t st_first = st0 + int64_t(g) * GROUP;
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);   // shuffle: the compiler then treats everything derived from the warp index as warp uniform
    const int m_begin = blockIdx.y * chunk;
    const int m_end = min(n_minors, m_begin + chunk);
    int m = m_begin + warp * (chunk / (NT / 32));
    const int m_stop = min(m_end, m + chunk / (NT / 32));
    Desc<N> dn;
    if (m < m_stop) dn = Desc<N>::load(desc, m);
    stage_tile(tile, P, st_first, n_st_total, NT);
    __syncthreads();
    const unsigned char* tb = reinterpret_cast<const unsigned char*>(tile + lane);
    // every lane stores: the rows of `out` are S_b >= 32 * gridDim.x wide, lanes beyond the end of the lattice hold zero tiles
    c128* outp = out + int64_t(g) * GROUP + lane;
    constexpr uint32_t kRowStep = 12 * GROUP * 16, kColStep = GROUP * 16;
    LuState<N, 0, NT> lu;
    c128 col2[4];                                                        // Schur column of column index 2 (instance (0,1) only)
#pragma unroll
    for (int r = 0; r < 4; ++r) col2[r] = make_double2(0.0, 0.0);
    unsigned long long prow = ~0ull, pcol = 0;
    auto cached = [&](uint32_t b, c128 (&t)[4]) {
#pragma unroll
        for (int r = 0; r < 4; ++r) t[r] = Sc[((b - 3) * 4 + r) * NT];
    };
    for (; m < m_stop; ++m) {
        const Desc<N> dc = dn;
        if (m + 1 < m_stop) dn = Desc<N>::load(desc, m + 1);
        const unsigned long long rws = dc.rows_bits(), diff = dc.cols_bits() ^ pcol;
        const bool fresh = (rws != prow) || (diff & 0xffull) != 0;
        if (fresh) {
            uint32_t rb[N], cb[N];
#pragma unroll
            for (int i = 0; i < N; ++i) { rb[i] = dc.row(i) * kRowStep; cb[i] = dc.col(i) * kColStep; }
            lu.start(tb, nullptr, rb, cb);
            const uint32_t b1 = dc.col(1);
            if (b1 < 2) lu.schur_column(tb, nullptr, 2 * kColStep, col2);
#pragma unroll 1
            for (uint32_t b = (b1 + 1 > 3 ? b1 + 1 : 3); b < 12; ++b) {
                c128 t[4];
                lu.schur_column(tb, nullptr, b * kColStep, t);
#pragma unroll
                for (int r = 0; r < 4; ++r) Sc[((b - 3) * 4 + r) * NT] = t[r];
            }
        }
        const bool new_pair = fresh || (diff & 0xffffull) != 0;
        if (new_pair) {
            c128 t0[4], t1[4];
            const uint32_t b2 = dc.col(2);
            if (b2 == 2) {
#pragma unroll
                for (int r = 0; r < 4; ++r) t0[r] = col2[r];
            } else cached(b2, t0);
            cached(dc.col(3), t1);
            lu.pair_from(t0, t1);
        }
        if (new_pair || (diff & 0xfffffull) != 0) {
            c128 t[4];
            cached(dc.col(4), t);
            lu.third_from(t);
        }
        c128 t[4];
        cached(dc.col(5), t);
        const c128 det = lu.finish_from(t);
        prow = rws; pcol = dc.cols_bits();
        outp[int64_t(m) * S_b] = det;
    }
}

// ---------------------------------------------------------------------------------------------
// a4, 10x10 (and 11x11) minors with the same per-thread cache of Schur columns: after the 6 pivot steps of a (row tuple, leading
// columns) instance only 6 column indices remain, and every minor of the instance takes 4 of them.  The 6 Schur columns
// (156 DFMA each) are computed once per instance (6 x 4 complex = 384 B per thread) and the levels combine them.
// Column tuples come in the library's clustered order (build_minor_descs), so the slot of a column index is its rank
// among the non-leading indices, kept as a nibble map.  One 256-thread CTA per SM as before (registers).
// ---------------------------------------------------------------------------------------------
// n = 11 works the same way with 5 remaining columns; its first multiplier column lives in shared memory (R = 1).
template <int N, int R> constexpr size_t mlc_smem() { return size_t(TILE_BYTES) + size_t(lcol_base<N>(R) + (12 - (N - 4)) * 4) * 16 * 256; }

template <int N, int R>
__global__ void __launch_bounds__(256, 1)
minors_large_cached_kernel(const c128* __restrict__ P, int64_t st0, int64_t n_st_total, int S_b,
                           const unsigned long long* __restrict__ desc, int n_minors, int chunk, c128* __restrict__ out) {
    static_assert(N == 10 || N == 11, "slot map and shared-memory budget are laid out for these sizes");
    constexpr int K = N - 4, NT = 256;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    c128* tile = reinterpret_cast<c128*>(smem_raw);
    c128* Ls = tile + TILE_ELEMS + threadIdx.x;                          // multipliers of the first R columns
    c128* Sc = Ls + lcol_base<N>(R) * NT;                                // this thread's cache: entry e at Sc[e * NT]
    const int g = blockIdx.x;
    const int64_t st_first = st0 + int64_t(g) * GROUP;
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);   // shuffle: the compiler then treats everything derived from the warp index as warp uniform
    const int m_begin = blockIdx.y * chunk;
    const int m_end = min(n_minors, m_begin + chunk);
    int m = m_begin + warp * (chunk / (NT / 32));
    const int m_stop = min(m_end, m + chunk / (NT / 32));
    Desc<N> dn;
    if (m < m_stop) dn = Desc<N>::load(desc, m);
    stage_tile(tile, P, st_first, n_st_total, NT);
    __syncthreads();
    const unsigned char* tb = reinterpret_cast<const unsigned char*>(tile + lane);
    // every lane stores: the rows of `out` are S_b >= 32 * gridDim.x wide, lanes beyond the end of the lattice hold zero tiles
    c128* outp = out + int64_t(g) * GROUP + lane;
    constexpr uint32_t kRowStep = 12 * GROUP * 16, kColStep = GROUP * 16;
    constexpr unsigned long long kLead = (1ull << (4 * K)) - 1, kLeadPair = (1ull << (4 * (K + 2))) - 1,
                                 kLead3 = (1ull << (4 * (K + 3))) - 1;
    LuState<N, R, NT> lu;
    unsigned long long smap = 0;                                         // column index -> cache slot (4 bits each)
    unsigned long long prow = ~0ull, pcol = 0;
    auto cached = [&](uint32_t b, c128 (&t)[4]) {
        const uint32_t slot = uint32_t(smap >> (4 * b)) & 15u;
#pragma unroll
        for (int r = 0; r < 4; ++r) t[r] = Sc[(slot * 4 + r) * NT];
    };
    for (; m < m_stop; ++m) {
        const Desc<N> dc = dn;
        if (m + 1 < m_stop) dn = Desc<N>::load(desc, m + 1);
        const unsigned long long rws = dc.rows_bits(), diff = dc.cols_bits() ^ pcol;
        const bool fresh = (rws != prow) || (diff & kLead) != 0;
        if (fresh) {
            uint32_t rb[N], cb[N];
            uint32_t lead = 0;
#pragma unroll
            for (int i = 0; i < N; ++i) { rb[i] = dc.row(i) * kRowStep; cb[i] = dc.col(i) * kColStep; if (i < K) lead |= 1u << dc.col(i); }
            lu.start(tb, Ls, rb, cb);
            smap = 0;
            uint32_t slot = 0;
#pragma unroll 1
            for (uint32_t b = 0; b < 12; ++b) {
                if (lead & (1u << b)) continue;
                c128 t[4];
                lu.schur_column(tb, Ls, b * kColStep, t);
#pragma unroll
                for (int r = 0; r < 4; ++r) Sc[(slot * 4 + r) * NT] = t[r];
                smap |= (unsigned long long)slot << (4 * b);
                ++slot;
            }
        }
        const bool new_pair = fresh || (diff & kLeadPair) != 0;
        if (new_pair) {
            c128 t0[4], t1[4];
            cached(dc.col(K), t0);
            cached(dc.col(K + 1), t1);
            lu.pair_from(t0, t1);
        }
        if (new_pair || (diff & kLead3) != 0) {
            c128 t[4];
            cached(dc.col(K + 2), t);
            lu.third_from(t);
        }
        c128 t[4];
        cached(dc.col(K + 3), t);
        const c128 det = lu.finish_from(t);
        prow = rws; pcol = dc.cols_bits();
        outp[int64_t(dc.out_index(m)) * S_b] = dc.negate() ? make_double2(-det.x, -det.y) : det;
    }
}

template <int N>
static cudaError_t launch_minors_n(const c128* P, int64_t st0, int64_t n_st_total, int n_groups, int S_b,
                                   const void* desc, int64_t n_minors, bool ascending, c128* out, int prof_cls, cudaStream_t stream) {
    constexpr int NT = MinorCfg<N>::kThreads;
    constexpr int warps = NT / 32;
    // enough CTAs for ~4 waves on 148 SMs, but at least 2 minors per warp per CTA
    int chunks = (148 * 4 + n_groups - 1) / n_groups;
    const int64_t max_chunks = (n_minors + 2 * warps - 1) / (2 * warps);
    if (chunks > max_chunks) chunks = int(max_chunks);
    if (chunks < 1) chunks = 1;
    if (chunks > 65535) chunks = 65535;
    int chunk = int((n_minors + chunks - 1) / chunks);
    chunk = ((chunk + warps - 1) / warps) * warps;            // every warp of a CTA gets the same count
    chunks = int((n_minors + chunk - 1) / chunk);
    dim3 grid(n_groups, chunks);
    ProfScope prof(prof_cls, stream);
    if constexpr (N == 10 || N == 11) {
        if (ascending) {                                       // library tables (no repeated index); slots = ranks among the non-leading indices
            constexpr int R = (N == 10) ? 0 : 1;
            minors_large_cached_kernel<N, R><<<grid, 256, mlc_smem<N, R>(), stream>>>(P, st0, n_st_total, S_b,
                                                                                      static_cast<const unsigned long long*>(desc), int(n_minors), chunk, out);
            ++g_launches;
            return cudaGetLastError();
        }
    }
    if (N == 6 && ascending)                                   // the cache slots assume ascending column tuples (library tables)
        minors6_cached_kernel<<<grid, M6C_THREADS, M6C_SMEM, stream>>>(P, st0, n_st_total, S_b,
                                                                       static_cast<const unsigned long long*>(desc), int(n_minors), chunk, out);
    else
        minors_kernel<N><<<grid, NT, MinorCfg<N>::kSmem, stream>>>(P, st0, n_st_total, S_b,
                                                                 static_cast<const unsigned long long*>(desc), int(n_minors), chunk, out);
    ++g_launches;
    return cudaGetLastError();
}

int minor_desc_words(int n) { return n <= 8 ? 1 : 2; }

cudaError_t launch_minors_reg(int n, const double2* P, int64_t st0, int64_t n_st_total, int n_groups, int S_b,
                              const RegTables& rt, double2* out, int prof_cls, cudaStream_t stream) {
    if (n_groups == 0 || rt.n_bins == 0) return cudaSuccess;
    ProfScope prof(prof_cls, stream);
    ++g_launches;
    return launch_minors_reg_impl(n, P, st0, n_st_total, n_groups, S_b, rt, out, stream);
}

cudaError_t launch_minors(int n, const double2* P, int64_t st0, int64_t n_st_total, int n_groups, int S_b,
                          const void* desc, int64_t n_minors, bool ascending, double2* out, int prof_cls, cudaStream_t stream) {
    if (n_minors == 0 || n_groups == 0) return cudaSuccess;
#define WICK_CASE(N) case N: return launch_minors_n<N>(P, st0, n_st_total, n_groups, S_b, desc, n_minors, ascending, out, prof_cls, stream);
    switch (n) {
        WICK_CASE(0) WICK_CASE(1) WICK_CASE(2) WICK_CASE(3) WICK_CASE(4) WICK_CASE(5) WICK_CASE(6)
        WICK_CASE(7) WICK_CASE(8) WICK_CASE(9) WICK_CASE(10) WICK_CASE(11) WICK_CASE(12)
        default: return cudaErrorInvalidValue;
    }
#undef WICK_CASE
}

// ---------------------------------------------------------------------------------------------
// a5: weighted bilinear products.  Lane = site; term indices and weights are warp-uniform.
// Each CTA handles one 32-site group and one chunk of the work; its warps' partial sums are
// combined in a fixed order and written to partial[chunk][site] (no atomics).
// ---------------------------------------------------------------------------------------------
constexpr int RED_THREADS = 256;

__device__ __forceinline__ void cta_combine_store(c128 acc, c128* partial_out /* &partial[chunk*S_b + g*32] */) {
    __shared__ c128 sm[RED_THREADS];
    sm[threadIdx.x] = acc;
    __syncthreads();
    if (threadIdx.x < GROUP) {
        c128 s = sm[threadIdx.x];
#pragma unroll
        for (int w = 1; w < RED_THREADS / 32; ++w) s = cadd(s, sm[w * 32 + threadIdx.x]);
        partial_out[threadIdx.x] = s;
    }
}

__global__ void __launch_bounds__(RED_THREADS)
reduce_flat_kernel(const c128* __restrict__ MU, const c128* __restrict__ MD, int S_b,
                   const int32_t* __restrict__ uid, const int32_t* __restrict__ did, const c128* __restrict__ w,
                   int64_t n_terms, int64_t chunk, c128* __restrict__ partial) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t s = int64_t(blockIdx.x) * GROUP + lane;
    const int64_t k0 = int64_t(blockIdx.y) * chunk;
    const int64_t k1 = min(n_terms, k0 + chunk);
    c128 acc = make_double2(0.0, 0.0);
    for (int64_t k = k0 + warp; k < k1; k += RED_THREADS / 32) {
        const c128 u = MU[int64_t(__ldg(uid + k)) * S_b + s];
        const c128 d = MD[int64_t(__ldg(did + k)) * S_b + s];
        acc = cfma(cmul(__ldg(w + k), u), d, acc);
    }
    cta_combine_store(acc, partial + int64_t(blockIdx.y) * S_b + int64_t(blockIdx.x) * GROUP);
}

// Outer-product lists: terms (i, j) = sink i x source j with uid = ru_i * NBu + cu_j,
// did = rd_i * NBd + cd_j, w = c_i * cbar_j.  For a fixed u row tuple ru and d column tuple cd
//     sum_{i in sink[ru]} sum_{j in src[cd]} c_i cbar_j MU[ru, cu_j] MD[rd_i, cd]
//   = ( sum_j cbar_j MU[ru, cu_j] ) * ( sum_i c_i MD[rd_i, cd] ),
// i.e. |sink[ru]| + |src[cd]| loads for |sink[ru]| * |src[cd]| terms.  The (ru, cd) plane is walked
// block by block: an item is (sink block k, source block k') of the block-diagonal factor lists
// (contract.cu: build_reduce_schedule), whose minors are a few KB per warp and are re-read from L1;
// every minor is fetched from DRAM / L2 once.  One warp = one bin of items, fixed order.
__global__ void __launch_bounds__(RED_THREADS, 2)
reduce_outer_kernel(const c128* __restrict__ MU, const c128* __restrict__ MD, int S_b, OuterTables ot,
                    c128* __restrict__ partial) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t s = int64_t(blockIdx.x) * GROUP + lane;
    const int bin = blockIdx.y * (RED_THREADS / 32) + warp;
    c128 acc = make_double2(0.0, 0.0);
    const int it0 = __ldg(ot.bin_ptr + bin), it1 = __ldg(ot.bin_ptr + bin + 1);
    for (int it = it0; it < it1; ++it) {
        const int2 kk = __ldg(ot.items + it);
        const int a0 = __ldg(ot.ru_ptr + kk.x), a1 = __ldg(ot.ru_ptr + kk.x + 1);
        const int b0 = __ldg(ot.cd_ptr + kk.y), b1 = __ldg(ot.cd_ptr + kk.y + 1);
        for (int a = a0; a < a1; ++a) {
            const int ru = __ldg(ot.ru_list + a);
            const int i0 = __ldg(ot.sink_ptr + ru), i1 = __ldg(ot.sink_ptr + ru + 1);
            const c128* MUrow = MU + int64_t(ru) * ot.n_cols_u * S_b + s;
            for (int b = b0; b < b1; ++b) {
                const int cd = __ldg(ot.cd_list + b);
                const int j0 = __ldg(ot.src_ptr + cd), j1 = __ldg(ot.src_ptr + cd + 1);
                c128 q = make_double2(0.0, 0.0);
#pragma unroll 4
                for (int j = j0; j < j1; ++j)
                    q = cfma(__ldg(ot.src_c + j), MUrow[int64_t(__ldg(ot.src_cu + j)) * S_b], q);
                c128 p = make_double2(0.0, 0.0);
                const c128* MDcol = MD + int64_t(cd) * S_b + s;
#pragma unroll 4
                for (int i = i0; i < i1; ++i)
                    p = cfma(__ldg(ot.sink_c + i), MDcol[int64_t(__ldg(ot.sink_rdoff + i)) * S_b], p);
                acc = cfma(q, p, acc);
            }
        }
    }
    cta_combine_store(acc, partial + int64_t(blockIdx.y) * S_b + int64_t(blockIdx.x) * GROUP);
}

// ---------------------------------------------------------------------------------------------
// a5, staged factorised reduction (outer-product lists whose blocks fit the STG_* capacities).
//   sigma = sum over (sink block k, source block k') of
//           sum_{ru in k} sum_{cd in k'} ( sum_{j in src[cd]} cbar_j MU[ru, cu_j] ) ( sum_{i in sink[ru]} c_i MD[rd_i, cd] )
// A batch = (d columns cd_a..cd_b of one source block) x (sink blocks ka..kb).  Per batch the CTA copies
// into shared memory, once: the MD elements [rd in blocks][cd] (cp.async, 16 B per lane, 512-byte rows)
// and the two coefficient lists it needs (source entries of the d columns, sink entries of the u-row
// tuples), so the inner loops touch no global table.  Warp w then takes the u-row tuples ru_a + w, + W, ...:
// the row MU[ru, cu in k'] goes to its private buffer (the next row is already in flight in registers),
//   P[cd] = sum_i c_i MD[rd_i, cd]            (cd unrolled: registers, one LDS + 4 DFMA per term)
//   acc  += sum_cd P[cd] * sum_j cbar_j row[cu_j]
// Every minor is read from DRAM once per batch that needs it.  Work order is fixed by the host
// schedule: bit-reproducible.
// ---------------------------------------------------------------------------------------------

constexpr int STG_W = STG_THREADS / 32;
// shared memory map (bytes)
constexpr size_t STG_OFF_ROWS = size_t(STG_MD_CAP) * GROUP * 16;
constexpr size_t STG_OFF_SINKC = STG_OFF_ROWS + size_t(STG_W) * STG_ROW_CAP * GROUP * 16;   // c128[STG_SINK_CAP]
constexpr size_t STG_OFF_SRCC = STG_OFF_SINKC + size_t(STG_SINK_CAP) * 16;                  // c128[STG_SRC_CAP]
constexpr size_t STG_OFF_SINKO = STG_OFF_SRCC + size_t(STG_SRC_CAP) * 16;                   // int[STG_SINK_CAP] MD element offset
constexpr size_t STG_OFF_SRCO = STG_OFF_SINKO + size_t(STG_SINK_CAP) * 4;                   // int[STG_SRC_CAP]  row element offset
constexpr size_t STG_OFF_SINKP = STG_OFF_SRCO + size_t(STG_SRC_CAP) * 4;                    // int[STG_ROWS_CAP + 1] per-row entry ranges
constexpr size_t STG_OFF_ROWOFF = STG_OFF_SINKP + size_t(STG_ROWS_CAP + 2) * 4;             // int[STG_ROWS_CAP] MU row offsets
constexpr size_t STG_OFF_SRCP = STG_OFF_ROWOFF + size_t(STG_ROWS_CAP + 2) * 4;              // int[16] per-cd entry ranges, int[16] u column offsets
constexpr size_t STG_SMEM = STG_OFF_SRCP + 32 * 4;
// real coefficients: {MD block, sink records, dense B, per-row entry ranges, MU row offsets, u column offsets}
constexpr size_t STG_R_SINKC = size_t(STG_MD_CAP_REAL) * GROUP * 16;
constexpr size_t STG_R_BD = STG_R_SINKC + size_t(STG_SINK_CAP) * 16;                        // double[STG_ROW_CAP][STG_NCD_CAP]
constexpr size_t STG_R_SINKP = STG_R_BD + size_t(STG_ROW_CAP) * STG_NCD_CAP * 8 + 64;
constexpr size_t STG_R_ROWOFF = STG_R_SINKP + size_t(STG_ROWS_CAP + 2) * 4;
constexpr size_t STG_R_CUOFF = STG_R_ROWOFF + size_t(STG_ROWS_CAP + 2) * 4;
constexpr size_t STG_SMEM_REAL = STG_R_CUOFF + 16 * 4;
constexpr size_t stg_smem(bool real) { return real ? STG_SMEM_REAL : STG_SMEM; }

// All u-row tuples of a batch that belong to this warp.  NCU = compile-time bound on the u columns of the
// piece (loads / stores of the row are unrolled and predicated), NCD = its number of d columns (exact).
// REAL: every coefficient of the factor lists is real (all interpolator products of wick_build_terms): a list
// entry is one 16-byte record {coefficient, element offset} and a term costs 2 DFMA instead of 4.
template <int NCU, int NCD, bool REAL>
__device__ __forceinline__ c128 staged_rows(const c128* MUs, const c128* MDl, c128* row, int warp, int n_rows, int n_cu,
                                            const int* rowoff, const int* cuoff, const int* sinkp, const c128* sinkc,
                                            const int* sinko, const int* srcp, const c128* srcc, const int* srco) {
    c128 acc = make_double2(0.0, 0.0);
    c128 X[NCU];
#pragma unroll
    for (int c = 0; c < NCU; ++c) X[c] = make_double2(0.0, 0.0);
    int r = warp;
    if (r < n_rows) {                                                    // first row: global -> registers
        const c128* src = MUs + rowoff[r];
#pragma unroll
        for (int c = 0; c < NCU; ++c)
            if (c < n_cu) X[c] = __ldg(src + cuoff[c]);
    }
    for (; r < n_rows; r += STG_W) {
#pragma unroll
        for (int c = 0; c < NCU; ++c)
            if (c < n_cu) row[c * GROUP] = X[c];
        __syncwarp();
        if (r + STG_W < n_rows) {                                        // next row: in flight during this row's arithmetic
            const c128* src = MUs + rowoff[r + STG_W];
#pragma unroll
            for (int c = 0; c < NCU; ++c)
                if (c < n_cu) X[c] = __ldg(src + cuoff[c]);
        }
        // P[cd] = sum_i c_i MD[rd_i, cd]
        c128 P[NCD];
#pragma unroll
        for (int c = 0; c < NCD; ++c) P[c] = make_double2(0.0, 0.0);
        const int i0 = sinkp[r], i1 = sinkp[r + 1];
#pragma unroll 2
        for (int i = i0; i < i1; ++i) {
            const c128 a = sinkc[i];
            const c128* md = MDl + (REAL ? __double2loint(a.y) : sinko[i]);   // element (rd_i, first cd of the piece), this lane
#pragma unroll
            for (int c = 0; c < NCD; ++c) {
                const c128 v = md[c * GROUP];
                if (REAL) { P[c].x = fma(a.x, v.x, P[c].x); P[c].y = fma(a.x, v.y, P[c].y); }
                else P[c] = cfma(a, v, P[c]);
            }
        }
        // acc += sum_cd P[cd] * sum_j cbar_j MU[ru, cu_j]
#pragma unroll
        for (int c = 0; c < NCD; ++c) {
            const int j0 = srcp[c], j1 = srcp[c + 1];
            c128 q = make_double2(0.0, 0.0);
#pragma unroll 2
            for (int j = j0; j < j1; ++j) {
                const c128 b = srcc[j];
                const c128 x = row[REAL ? __double2loint(b.y) : srco[j]];
                if (REAL) { q.x = fma(b.x, x.x, q.x); q.y = fma(b.x, x.y, q.y); }
                else q = cfma(b, x, q);
            }
            acc = cfma(q, P[c], acc);
        }
        __syncwarp();                                                    // all lanes have read the row buffer
    }
    return acc;
}

// Dense variant for pieces whose source block is (nearly) full, real coefficients: B[cu][cd] sits in shared memory as
// a dense n_cu x n_cd matrix (row stride = n_cd rounded up to 2 doubles), and
//   Q[cd] = sum_cu B[cu][cd] MU[ru, cu]
// is accumulated straight from the row's registers: no per-entry record, offset or row-buffer traffic (a 15 x 15 block
// has 225 entries: one broadcast LDS.128 feeds 4 DFMA here, against two loads and an address per 2 DFMA there).
template <int NCU, int NCD>
__device__ __forceinline__ c128 staged_rows_dense(const c128* MUs, const c128* MDl, int warp, int n_rows, int n_cu,
                                                  const int* rowoff, const int* cuoff, const int* sinkp, const c128* sinkc,
                                                  const double* Bd) {
    constexpr int NCDP = (NCD + 1) & ~1;
    c128 acc = make_double2(0.0, 0.0);
    c128 X[NCU];
#pragma unroll
    for (int c = 0; c < NCU; ++c) X[c] = make_double2(0.0, 0.0);
    int r = warp;
    if (r < n_rows) {                                                    // first row: global -> registers
        const c128* src = MUs + rowoff[r];
#pragma unroll
        for (int c = 0; c < NCU; ++c)
            if (c < n_cu) X[c] = __ldg(src + cuoff[c]);
    }
    for (; r < n_rows; r += STG_W) {
        c128 Q[NCDP];
#pragma unroll
        for (int c = 0; c < NCDP; ++c) Q[c] = make_double2(0.0, 0.0);
#pragma unroll
        for (int c = 0; c < NCU; ++c) {
            if (c < n_cu) {
                const c128 x = X[c];
                const double2* bp = reinterpret_cast<const double2*>(Bd + c * NCDP);
#pragma unroll
                for (int h = 0; h < NCDP / 2; ++h) {
                    const double2 b = bp[h];
                    Q[2 * h].x = fma(b.x, x.x, Q[2 * h].x); Q[2 * h].y = fma(b.x, x.y, Q[2 * h].y);
                    if (2 * h + 1 < NCD) { Q[2 * h + 1].x = fma(b.y, x.x, Q[2 * h + 1].x); Q[2 * h + 1].y = fma(b.y, x.y, Q[2 * h + 1].y); }
                }
            }
        }
        if (r + STG_W < n_rows) {                                        // next row: in flight during the rest of this row
            const c128* src = MUs + rowoff[r + STG_W];
#pragma unroll
            for (int c = 0; c < NCU; ++c)
                if (c < n_cu) X[c] = __ldg(src + cuoff[c]);
        }
        c128 P[NCD];
#pragma unroll
        for (int c = 0; c < NCD; ++c) P[c] = make_double2(0.0, 0.0);
        const int i0 = sinkp[r], i1 = sinkp[r + 1];
#pragma unroll 2
        for (int i = i0; i < i1; ++i) {
            const c128 a = sinkc[i];
            const c128* md = MDl + __double2loint(a.y);
#pragma unroll
            for (int c = 0; c < NCD; ++c) {
                const c128 v = md[c * GROUP];
                P[c].x = fma(a.x, v.x, P[c].x); P[c].y = fma(a.x, v.y, P[c].y);
            }
        }
#pragma unroll
        for (int c = 0; c < NCD; ++c) acc = cfma(Q[c], P[c], acc);
    }
    return acc;
}

template <int NCU>
__device__ __forceinline__ c128 staged_rows_dense_ncd(const c128* MUs, const c128* MDl, int warp, int n_rows, int n_cu, int n_cd,
                                                      const int* rowoff, const int* cuoff, const int* sinkp, const c128* sinkc,
                                                      const double* Bd) {
#define WICK_STG_CALL(NCD) staged_rows_dense<NCU, NCD>(MUs, MDl, warp, n_rows, n_cu, rowoff, cuoff, sinkp, sinkc, Bd)
    switch (n_cd) {
        case 1: return WICK_STG_CALL(1);
        case 2: return WICK_STG_CALL(2);
        case 3: return WICK_STG_CALL(3);
        case 4: return WICK_STG_CALL(4);
        case 5: return WICK_STG_CALL(5);
        case 6: return WICK_STG_CALL(6);
        case 7: return WICK_STG_CALL(7);
        default: return WICK_STG_CALL(8);
    }
#undef WICK_STG_CALL
}

template <int NCU, bool REAL>
__device__ __forceinline__ c128 staged_rows_ncd(const c128* MUs, const c128* MDl, c128* row, int warp, int n_rows, int n_cu, int n_cd,
                                                const int* rowoff, const int* cuoff, const int* sinkp, const c128* sinkc,
                                                const int* sinko, const int* srcp, const c128* srcc, const int* srco) {
#define WICK_STG_CALL(NCD) staged_rows<NCU, NCD, REAL>(MUs, MDl, row, warp, n_rows, n_cu, rowoff, cuoff, sinkp, sinkc, sinko, srcp, srcc, srco)
    static_assert(STG_NCD_CAP == 8, "one case per d-column count");
    switch (n_cd) {
        case 1: return WICK_STG_CALL(1);
        case 2: return WICK_STG_CALL(2);
        case 3: return WICK_STG_CALL(3);
        case 4: return WICK_STG_CALL(4);
        case 5: return WICK_STG_CALL(5);
        case 6: return WICK_STG_CALL(6);
        case 7: return WICK_STG_CALL(7);
        default: return WICK_STG_CALL(8);
    }
#undef WICK_STG_CALL
}

template <bool REAL>
__global__ void __launch_bounds__(STG_THREADS, STG_CTAS_PER_SM)
reduce_staged_kernel(const c128* __restrict__ MU, const c128* __restrict__ MD, int S_b, StagedTables st,
                     c128* __restrict__ partial) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    c128* MDs = reinterpret_cast<c128*>(smem_raw);                       // [element][lane]
    // REAL: {MD block, sink records, dense B, entry ranges, row offsets, column offsets}; general: the map above
    c128* sinkc = reinterpret_cast<c128*>(smem_raw + (REAL ? STG_R_SINKC : STG_OFF_SINKC));
    c128* srcc = reinterpret_cast<c128*>(smem_raw + STG_OFF_SRCC);        // general coefficients only
    int* sinko = reinterpret_cast<int*>(smem_raw + STG_OFF_SINKO);
    int* srco = reinterpret_cast<int*>(smem_raw + STG_OFF_SRCO);
    double* Bd = reinterpret_cast<double*>(smem_raw + STG_R_BD);          // real coefficients only
    int* sinkp = reinterpret_cast<int*>(smem_raw + (REAL ? STG_R_SINKP : STG_OFF_SINKP));      // [0..rows]: sink entry ranges
    int* rowoff = reinterpret_cast<int*>(smem_raw + (REAL ? STG_R_ROWOFF : STG_OFF_ROWOFF));   // [rows]: element offset of MU[ru, 0]
    int* srcp = reinterpret_cast<int*>(smem_raw + STG_OFF_SRCP);          // [0..n_cd]: source entry ranges (general only)
    int* cuoff = REAL ? reinterpret_cast<int*>(smem_raw + STG_R_CUOFF) : srcp + 16;            // [n_cu]: element offset of u column tuple
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    c128* row = reinterpret_cast<c128*>(smem_raw + STG_OFF_ROWS) + warp * STG_ROW_CAP * GROUP + lane;   // general only
    const c128* MDl = MDs + lane;
    const int64_t s = int64_t(blockIdx.x) * GROUP + lane;
    const c128* MUs = MU + s;
    const c128* MDg = MD + s;
    c128 acc = make_double2(0.0, 0.0);
    const int b0 = __ldg(st.bin_ptr + blockIdx.y), b1 = __ldg(st.bin_ptr + blockIdx.y + 1);
    int my_id = 0;                                                       // MD element id this lane holds for its warp (see below)
    for (int b = b0; b < b1; ++b) {
        const int4 v0 = __ldg(reinterpret_cast<const int4*>(st.batches + b));
        const int4 v1 = __ldg(reinterpret_cast<const int4*>(st.batches + b) + 1);
        const int4 v2 = __ldg(reinterpret_cast<const int4*>(st.batches + b) + 2);
        const int cd_a = v0.x, n_cd = v0.y - v0.x, cu_a = v0.z, n_cu = v0.w - v0.z;
        const int rd_a = v1.x, n_rd = v1.y - v1.x, ru_a = v1.z, n_rows = v1.w - v1.z;
        __syncthreads();                                                 // every warp is done with the previous batch
        {   // MD block: the element ids were laid out on the host (no division, no dependent look-up per element).  Warp w copies
            // the elements w, w + STG_W, ...: lane l fetches the id of the l-th of them (ONE load latency per batch; a load per
            // element in front of its copy cost the prologue eight dependent L2 round trips) and the ids go round by shuffle
            static_assert(STG_MD_CAP_REAL <= 32 * STG_W && STG_MD_CAP <= 32 * STG_W, "one id per lane");
            // The id lists of a bin's batches follow one another in md_ids (padded by 32 * STG_W entries), so the ids of the NEXT
            // batch are requested here as well and arrive during this batch's arithmetic.
            const int32_t* ids = st.md_ids + v2.x;
            const int n_el = n_rd * n_cd;
            const int my_e = warp + STG_W * lane;
            if (b == b0) my_id = __ldg(ids + my_e);
            for (int j = 0, e = warp; e < n_el; ++j, e += STG_W)
                cp_async16(MDs + e * GROUP + lane, MDg + int64_t(__shfl_sync(0xffffffffu, my_id, j)) * S_b);
            my_id = __ldg(ids + n_el + my_e);
            if (b + 1 < b1) {                                            // next batch descriptor -> L1
                asm volatile("prefetch.global.L1 [%0];" ::"l"(st.batches + b + 1));
                asm volatile("prefetch.global.L1 [%0];" ::"l"(reinterpret_cast<const char*>(st.batches + b + 1) + 32));
            }
        }
        // coefficient lists of the batch -> shared memory, offsets already in elements of the staged buffers
        const int sp0 = v2.z, sp1 = v2.z + v2.w;
        for (int e = threadIdx.x; e < sp1 - sp0; e += STG_THREADS) {
            const c128 cf = __ldg(st.sink_c + sp0 + e);
            const int off = (__ldg(st.sink_rdpos + sp0 + e) - rd_a) * n_cd * GROUP;
            sinkc[e] = REAL ? make_double2(cf.x, __hiloint2double(0, off)) : cf;
            if (!REAL) sinko[e] = off;
        }
        for (int r = threadIdx.x; r <= n_rows; r += STG_THREADS) {
            sinkp[r] = __ldg(st.sink_ptr + ru_a + r) - sp0;
            if (r < n_rows) rowoff[r] = __ldg(st.ru_list + ru_a + r) * st.n_cols_u * S_b;
        }
        if constexpr (REAL) {
            // dense B[cu][cd] of the piece (row stride = n_cd rounded up to 2 doubles; zeros where there is no source term)
            const int ncdp = (n_cd + 1) & ~1;
            const double* bsrc = st.b_dense + v2.y;                      // built once per piece on the host
            for (int e = threadIdx.x; e < n_cu * ncdp; e += STG_THREADS) Bd[e] = __ldg(bsrc + e);
            if (threadIdx.x < n_cu) cuoff[threadIdx.x] = __ldg(st.cu_list + cu_a + threadIdx.x) * S_b;
        } else {
            const int q0 = __ldg(st.src_ptr + cd_a), q1 = __ldg(st.src_ptr + cd_a + n_cd);
            for (int e = threadIdx.x; e < q1 - q0; e += STG_THREADS) {
                srcc[e] = __ldg(st.src_c + q0 + e);
                srco[e] = (__ldg(st.src_cupos + q0 + e) - cu_a) * GROUP;
            }
            if (threadIdx.x <= n_cd) srcp[threadIdx.x] = __ldg(st.src_ptr + cd_a + threadIdx.x) - q0;
            if (threadIdx.x >= 32 && threadIdx.x < 32 + n_cu) cuoff[threadIdx.x - 32] = __ldg(st.cu_list + cu_a + threadIdx.x - 32) * S_b;
        }
        cp_async_wait_all();
        __syncthreads();
#define WICK_STG_CALL(NCU) staged_rows_ncd<NCU, false>(MUs, MDl, row, warp, n_rows, n_cu, n_cd, rowoff, cuoff, sinkp, sinkc, sinko, srcp, srcc, srco)
        c128 v;
        if constexpr (REAL) {
            if (n_cu <= 2) v = staged_rows_dense_ncd<2>(MUs, MDl, warp, n_rows, n_cu, n_cd, rowoff, cuoff, sinkp, sinkc, Bd);
            else if (n_cu <= 4) v = staged_rows_dense_ncd<4>(MUs, MDl, warp, n_rows, n_cu, n_cd, rowoff, cuoff, sinkp, sinkc, Bd);
            else if (n_cu <= 8) v = staged_rows_dense_ncd<8>(MUs, MDl, warp, n_rows, n_cu, n_cd, rowoff, cuoff, sinkp, sinkc, Bd);
            else v = staged_rows_dense_ncd<STG_ROW_CAP>(MUs, MDl, warp, n_rows, n_cu, n_cd, rowoff, cuoff, sinkp, sinkc, Bd);
        } else if (n_cu <= 2) v = WICK_STG_CALL(2);
        else if (n_cu <= 4) v = WICK_STG_CALL(4);
        else if (n_cu <= 8) v = WICK_STG_CALL(8);
        else v = WICK_STG_CALL(STG_ROW_CAP);
#undef WICK_STG_CALL
        acc = cadd(acc, v);
    }
    // fixed-order combination of the warps -> partial[bin][site]
    __syncthreads();
    MDs[threadIdx.x] = acc;
    __syncthreads();
    if (threadIdx.x < GROUP) {
        c128 t = MDs[threadIdx.x];
#pragma unroll
        for (int w = 1; w < STG_W; ++w) t = cadd(t, MDs[w * 32 + threadIdx.x]);
        partial[int64_t(blockIdx.y) * S_b + int64_t(blockIdx.x) * GROUP + threadIdx.x] = t;
    }
}

cudaError_t launch_reduce_staged(const double2* MU, const double2* MD, int n_groups, int S_b, const StagedTables& st,
                                 double2* partial, int* n_chunks_out, cudaStream_t stream) {
    dim3 grid(n_groups, st.n_bins);
    ProfScope prof(PROF_REDUCE, stream);
    if (st.real_coeffs) reduce_staged_kernel<true><<<grid, STG_THREADS, STG_SMEM_REAL, stream>>>(MU, MD, S_b, st, partial);
    else reduce_staged_kernel<false><<<grid, STG_THREADS, STG_SMEM, stream>>>(MU, MD, S_b, st, partial);
    ++g_launches;
    *n_chunks_out = st.n_bins;
    return cudaGetLastError();
}

cudaError_t launch_reduce_flat(const double2* MU, const double2* MD, int n_groups, int S_b,
                               const int32_t* uid, const int32_t* did, const double2* w, int64_t n_terms,
                               double2* partial, int* n_chunks_out, int max_chunks, cudaStream_t stream) {
    int chunks = (148 * 8 + n_groups - 1) / n_groups;
    const int64_t cap = (n_terms + 63) / 64;                  // at least 8 terms per warp
    if (chunks > cap) chunks = int(cap);
    if (chunks > max_chunks) chunks = max_chunks;
    if (chunks < 1) chunks = 1;
    const int64_t chunk = (n_terms + chunks - 1) / chunks;
    chunks = chunk > 0 ? int((n_terms + chunk - 1) / chunk) : 1;
    if (chunks < 1) chunks = 1;
    dim3 grid(n_groups, chunks);
    ProfScope prof(PROF_REDUCE, stream);
    reduce_flat_kernel<<<grid, RED_THREADS, 0, stream>>>(MU, MD, S_b, uid, did, w, n_terms, chunk > 0 ? chunk : 1, partial);
    ++g_launches;
    *n_chunks_out = chunks;
    return cudaGetLastError();
}

cudaError_t launch_reduce_outer(const double2* MU, const double2* MD, int n_groups, int S_b, const OuterTables& ot,
                                double2* partial, int* n_chunks_out, cudaStream_t stream) {
    const int chunks = ot.n_bins / (RED_THREADS / 32);         // n_bins is a multiple of 8 (contract.cu)
    dim3 grid(n_groups, chunks);
    ProfScope prof(PROF_REDUCE, stream);
    reduce_outer_kernel<<<grid, RED_THREADS, 0, stream>>>(MU, MD, S_b, ot, partial);
    ++g_launches;
    *n_chunks_out = chunks;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// a6: sigma = fixed-order sum of the chunk partials; C(t,p) = sum_x e^{ip.x} sigma(x,t), fixed tree
// ---------------------------------------------------------------------------------------------
// 32 sites x 8 slices of the chunk range per CTA: thread (site, k) sums the chunks k, k + 8, ... in order, then the 8 partial
// sums are added in order k = 0..7 (fixed shape: bit-reproducible)
constexpr int FIN_SLICES = 8;

__global__ void __launch_bounds__(32 * FIN_SLICES)
finalize_sigma_kernel(const c128* __restrict__ partial, int n_chunks, int S_b, int64_t n_valid,
                      c128* __restrict__ sigma_batch, const c128* __restrict__ scale_a, const c128* __restrict__ scale_b) {
    __shared__ c128 sm[FIN_SLICES][32];
    const int lane = threadIdx.x & 31, k = threadIdx.x >> 5;
    const int64_t s = int64_t(blockIdx.x) * 32 + lane;
    c128 acc = make_double2(0.0, 0.0);
    if (s < n_valid)
        for (int c = k; c < n_chunks; c += FIN_SLICES) acc = cadd(acc, partial[int64_t(c) * S_b + s]);
    sm[k][lane] = acc;
    __syncthreads();
    if (k == 0 && s < n_valid) {
#pragma unroll
        for (int j = 1; j < FIN_SLICES; ++j) acc = cadd(acc, sm[j][lane]);
        if (scale_a) acc = cmul(acc, scale_a[s]);               // Jacobi path: the common factor det U (det D) of every term of the site
        if (scale_b) acc = cmul(acc, scale_b[s]);
        sigma_batch[s] = acc;
    }
}

cudaError_t launch_finalize_sigma(const double2* partial, int n_chunks, int S_b, int64_t n_valid,
                                  double2* sigma_batch, const double2* scale_a, const double2* scale_b, cudaStream_t stream) {
    if (n_valid <= 0) return cudaSuccess;
    ProfScope prof(PROF_PROJECT, stream);
    finalize_sigma_kernel<<<unsigned((n_valid + 31) / 32), 32 * FIN_SLICES, 0, stream>>>(partial, n_chunks, S_b, n_valid, sigma_batch, scale_a, scale_b);
    ++g_launches;
    return cudaGetLastError();
}

constexpr int PROJ_THREADS = 1024;      // one CTA per (momentum, timeslice): latency bound, so as many threads as a CTA can have

// one CTA per (momentum, timeslice): each thread sums its sites in index order, then a fixed tree
__global__ void __launch_bounds__(PROJ_THREADS)
project_kernel(const c128* __restrict__ sigma, int L, int T, MomentumList mom, c128* __restrict__ C_out) {
    __shared__ c128 sm[PROJ_THREADS];
    const int t = blockIdx.x, p = blockIdx.y;
    const int V = L * L * L;
    const int nx = mom.v[p][0], ny = mom.v[p][1], nz = mom.v[p][2];
    const bool zero = (nx == 0 && ny == 0 && nz == 0);
    const c128* sg = sigma + int64_t(t) * V;
    c128 acc = make_double2(0.0, 0.0);
    for (int s = threadIdx.x; s < V; s += PROJ_THREADS) {
        const c128 v = sg[s];
        if (zero) {
            acc = cadd(acc, v);
        } else {
            const int x = s % L, y = (s / L) % L, z = s / (L * L);
            long long m = (long long)nx * x + (long long)ny * y + (long long)nz * z;
            m %= L;
            if (m < 0) m += L;
            double sn, cs;
            sincospi(2.0 * double(m) / double(L), &sn, &cs);   // exact at multiples of L/4
            acc = cfma(make_double2(cs, sn), v, acc);
        }
    }
    sm[threadIdx.x] = acc;
    __syncthreads();
    for (int h = PROJ_THREADS / 2; h > 0; h >>= 1) {
        if (threadIdx.x < h) sm[threadIdx.x] = cadd(sm[threadIdx.x], sm[threadIdx.x + h]);
        __syncthreads();
    }
    if (threadIdx.x == 0) C_out[int64_t(p) * T + t] = sm[0];
}

cudaError_t launch_project(const double2* sigma, int L, int T, const MomentumList& mom, double2* C_out,
                           cudaStream_t stream) {
    if (T <= 0 || mom.n <= 0) return cudaSuccess;
    dim3 grid(T, mom.n);
    ProfScope prof(PROF_PROJECT, stream);
    project_kernel<<<grid, PROJ_THREADS, 0, stream>>>(sigma, L, T, mom, C_out);
    ++g_launches;
    return cudaGetLastError();
}


// ---------------------------------------------------------------------------------------------
// Cluster sinks (block algorithm Eq. 6-8): block tensor of one cluster,
//   part[g][cu][cd] = sum_{site in group g} e^{ip.x} sum_i c_i MU[ru_i, cu] MD[rd_i, cd]
// lane = site, one (cu, cd) pair per warp iteration, fixed shuffle tree over the 32 sites; the groups of a timeslice are
// summed in order by block_sum_kernel.  Flat over the sink terms: meant for small clusters (nucleons, deuteron).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
block_tensor_kernel(const c128* __restrict__ MU, const c128* __restrict__ MD, int S_b, int n_valid, int n_cu, int n_cd,
                    const int32_t* __restrict__ sink_ru, const int32_t* __restrict__ sink_rd, const c128* __restrict__ sink_c, int n_sink,
                    int L, int64_t site0, int3 mom, c128* __restrict__ part /* [group][n_cu * n_cd] of this batch */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = blockIdx.x;
    const int s = g * GROUP + lane;
    const bool valid = s < n_valid;
    const int sl = valid ? s : 0;
    // e^{+2 pi i (n.x)/L}, (n.x) reduced mod L in integers
    const int64_t site = site0 + sl;
    const int x = int(site % L), y = int((site / L) % L), z = int(site / (int64_t(L) * L));
    long long m = (long long)mom.x * x + (long long)mom.y * y + (long long)mom.z * z;
    m %= L; if (m < 0) m += L;
    double sn, cs;
    sincospi(2.0 * double(m) / double(L), &sn, &cs);
    const c128 ph = valid ? make_double2(cs, sn) : make_double2(0.0, 0.0);
    const int n_pairs = n_cu * n_cd;
    for (int p = blockIdx.y * 8 + warp; p < n_pairs; p += gridDim.y * 8) {
        const int cu = p / n_cd, cd = p - cu * n_cd;
        c128 acc = make_double2(0.0, 0.0);
        for (int i = 0; i < n_sink; ++i) {
            const c128 u = MU[(int64_t(__ldg(sink_ru + i)) * n_cu + cu) * S_b + sl];
            const c128 d = MD[(int64_t(__ldg(sink_rd + i)) * n_cd + cd) * S_b + sl];
            acc = cfma(cmul(__ldg(sink_c + i), u), d, acc);
        }
        acc = cmul(acc, ph);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            acc.x += __shfl_xor_sync(0xffffffffu, acc.x, off);
            acc.y += __shfl_xor_sync(0xffffffffu, acc.y, off);
        }
        if (lane == 0) part[int64_t(g) * n_pairs + p] = acc;
    }
}

__global__ void block_sum_kernel(const c128* __restrict__ part, int n_groups, int n_pairs, c128* __restrict__ out) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs) return;
    c128 acc = make_double2(0.0, 0.0);
    for (int g = 0; g < n_groups; ++g) acc = cadd(acc, part[int64_t(g) * n_pairs + p]);
    out[p] = acc;
}

cudaError_t launch_block_tensor(const double2* MU, const double2* MD, int S_b, int n_valid, int n_cu, int n_cd,
                                const int32_t* sink_ru, const int32_t* sink_rd, const double2* sink_c, int n_sink,
                                int L, int64_t site0, const int mom[3], double2* part, cudaStream_t stream) {
    const int n_groups = (n_valid + GROUP - 1) / GROUP;
    if (n_groups == 0) return cudaSuccess;
    const int n_pairs = n_cu * n_cd;
    int chunks = std::max(1, std::min((n_pairs + 7) / 8, (148 * 8 + n_groups - 1) / n_groups));
    dim3 grid(n_groups, chunks);
    ProfScope prof(PROF_REDUCE, stream);
    block_tensor_kernel<<<grid, 256, 0, stream>>>(MU, MD, S_b, n_valid, n_cu, n_cd, sink_ru, sink_rd, sink_c, n_sink, L, site0,
                                                  make_int3(mom[0], mom[1], mom[2]), part);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_block_sum(const double2* part, int n_groups, int n_pairs, double2* out, cudaStream_t stream) {
    ProfScope prof(PROF_PROJECT, stream);
    block_sum_kernel<<<(n_pairs + 127) / 128, 128, 0, stream>>>(part, n_groups, n_pairs, out);
    ++g_launches;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// Measurement helper: register-only DFMA stream (the FP64 roofline denominator)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_probe_kernel(double* out, int iters, double a, double b) {
    double x[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) x[k] = double(threadIdx.x + k);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) x[k] = fma(x[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += x[k];
    if (s == 12345.678) out[0] = s;                              // never true: keeps the chain alive
}

cudaError_t measure_fp64_peak(double* tflops, cudaStream_t stream) {
    double* d = nullptr;
    cudaError_t e = cudaMalloc(&d, 8);
    if (e != cudaSuccess) return e;
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    const int blocks = 148 * 8, iters = 1 << 15;
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(a, stream);
        dfma_probe_kernel<<<blocks, 256, 0, stream>>>(d, iters, 0.999999, 1e-9);
        cudaEventRecord(b, stream);
        e = cudaEventSynchronize(b);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        const double tf = 2.0 * 8.0 * double(iters) * 256.0 * blocks / (double(ms) * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;                     // rep 0 is the warm-up
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(d);
    *tflops = best;
    return e;
}

template <int N> static cudaError_t set_smem_attr() {
    return cudaFuncSetAttribute(minors_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(MinorCfg<N>::kSmem));
}

template <int MU_, int MD_> static cudaError_t set_jf_attr2() {
    const cudaError_t e = cudaFuncSetAttribute(jacobi_fused_kernel<MU_, MD_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(JF_SMEM_STAGED));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(jacobi_fused_kernel<MU_, MD_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(JF_SMEM));
}
template <int MU_> static cudaError_t set_jf_attr() {
    cudaError_t e;
    if ((e = set_jf_attr2<MU_, 1>()) != cudaSuccess || (e = set_jf_attr2<MU_, 2>()) != cudaSuccess || (e = set_jf_attr2<MU_, 3>()) != cudaSuccess) return e;
    return set_jf_attr2<MU_, 4>();
}

cudaError_t configure_kernels() {
    cudaError_t e;
    if ((e = set_jf_attr<1>()) != cudaSuccess || (e = set_jf_attr<2>()) != cudaSuccess || (e = set_jf_attr<3>()) != cudaSuccess ||
        (e = set_jf_attr<4>()) != cudaSuccess) return e;
    if ((e = configure_reg_kernels()) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(minors_large_cached_kernel<10, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(mlc_smem<10, 0>()))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(minors_large_cached_kernel<11, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(mlc_smem<11, 1>()))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(minors6_cached_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(M6C_SMEM))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(reduce_staged_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(STG_SMEM_REAL))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(reduce_staged_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(STG_SMEM))) != cudaSuccess) return e;
#define WICK_ATTR(N) if ((e = set_smem_attr<N>()) != cudaSuccess) return e;
    WICK_ATTR(0) WICK_ATTR(1) WICK_ATTR(2) WICK_ATTR(3) WICK_ATTR(4) WICK_ATTR(5) WICK_ATTR(6)
    WICK_ATTR(7) WICK_ATTR(8) WICK_ATTR(9) WICK_ATTR(10) WICK_ATTR(11) WICK_ATTR(12)
#undef WICK_ATTR
    return cudaSuccess;
}

}  // namespace wick

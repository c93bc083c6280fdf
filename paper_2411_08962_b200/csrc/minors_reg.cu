// a4 for "grid" minor tables (every row tuple x every column tuple, i.e. outer-product term lists), N = 6: the instance kernel.
//
// A job = (row tuple, instance) where an instance is a set of K = N-4 leading columns shared by many column tuples.  After
// the K pivot steps of the instance (left-looking LU with partial pivoting, lu_device.cuh) every minor of the instance is
//   detp * det4(S[:, b_K], S[:, b_K+1], S[:, b_K+2], S[:, b_K+3])
// with S the 4-row Schur complement; its columns are needed for the NC <= 10 "candidate" column indices that occur behind the
// leading ones.  The thread computes all candidate Schur columns ONCE: into registers (4 complex each; the LAST level of the
// trie is fully unrolled over the candidate positions, so its register indices are static and it touches no memory but the
// result store; every lane stores, the output rows are S_b >= 32 * gridDim.x wide, so lanes beyond the end of the lattice,
// whose tiles are zero, write zeros into the padding) and into a per-thread shared-memory copy (positions 0 .. NC-2, for the pair and third levels, which fetch
// their columns by dynamic index).  The trie of the instance's column tuples over candidate POSITIONS is a word program built
// on the host (contract.cu: build_reg_host; one word per third node): it is the same for every row tuple, because an outer-product list pairs every
// row tuple with the same column tuples.  Everything that steers a job is warp uniform (the warp index is taken through a
// shuffle so that the compiler knows), so every test is a uniform branch.
//
// PAPER.md:203 ("analytic up to 4x4, LU above") and R.2 (:226, nothing is evaluated twice) one level below the
// unique-minor table: every minor is still the pivoted LU of its own matrix, identical leading work is shared.
#include "kernels.cuh"
#include "lu_device.cuh"

namespace wick {

namespace {

template <int NC>
struct Trie {
    c128 T[NC][4];                    // Schur columns of the candidate positions (registers: the static last level)
    c128 s[6];                        // 2x2 minors of (detp * T[i2], T[i3]) over the row pairs 01 02 03 12 13 23
    c128 c3[4];                       // 3x3 minors of (.., T[i4]) over the row triples that leave out row r
    c128* o;                          // where the job's first minor goes (this lane)
    uint32_t k;                       // element offset of the job's next minor (minors stored so far x S_b; a job has <= 165 minors)
    uint32_t step;                    // S_b
};

// 3x3 minors of (.., t): c3[r] = det(rows != r), expanded along the last column in the 2x2 minors s
__device__ __forceinline__ void third_from(const c128 (&s)[6], const c128 (&t)[4], c128 (&c3)[4]) {
    const c128 m0 = cfma(t[3], s[3], cfnma(t[2], s[4], cmul(t[1], s[5])));   // rows 1,2,3
    const c128 m1 = cfma(t[3], s[1], cfnma(t[2], s[2], cmul(t[0], s[5])));   // rows 0,2,3
    const c128 m2 = cfma(t[3], s[0], cfnma(t[1], s[2], cmul(t[0], s[4])));   // rows 0,1,3
    const c128 m3 = cfma(t[2], s[0], cfnma(t[1], s[1], cmul(t[0], s[3])));   // rows 0,1,2
    c3[0] = m0; c3[1] = m1; c3[2] = m2; c3[3] = m3;              // UNSIGNED: the alternating sign is taken in the Laplace sum below
}

// last level, static in the candidate position: det = sum_r T[I5][r] c3[r]
template <int NC, int I5>
__device__ __forceinline__ void finish_all(Trie<NC>& c, uint32_t mask5) {
    if constexpr (I5 < NC) {
        if ((mask5 >> I5) & 1u) {
            const c128 e0 = cfnma(c.T[I5][0], c.c3[0], cmul(c.T[I5][1], c.c3[1]));   // -t0 m0 + t1 m1
            const c128 e1 = cfnma(c.T[I5][2], c.c3[2], cmul(c.T[I5][3], c.c3[3]));   // -t2 m2 + t3 m3
            // the address is formed from a 32-bit element offset right before the store: a store holds its source registers
            // until the LSU has read them (~30 cycles here), and a pointer that is incremented after every store waits for that
            c128* const here = c.o + c.k;
            c.k += c.step;
            *here = cadd(e0, e1);                                 // lanes beyond the lattice hold zero tiles and store 0 into the padding of the row
        }
        finish_all<NC, I5 + 1>(c, mask5);
    }
}

template <int N, int NC, int J>
__device__ __forceinline__ void schur_columns(const LuState<N, 0, REG_THREADS>& lu, const unsigned char* tb, unsigned long long cand,
                                              int ncand, Trie<NC>& c, c128* Sc) {
    if constexpr (J < NC) {
        if (J < ncand) {
            lu.schur_column(tb, nullptr, (uint32_t(cand >> (4 * J)) & 15u) * uint32_t(GROUP * 16), c.T[J]);
            if constexpr (J < NC - 1) {                               // the last position can only be a last column
#pragma unroll
                for (int r = 0; r < 4; ++r) Sc[(J * 4 + r) * REG_THREADS] = c.T[J][r];
            }
        }
        schur_columns<N, NC, J + 1>(lu, tb, cand, ncand, c, Sc);
    }
}

// `sc` = shared-window address of this thread's Sc[0], held in a register (given the chance the compiler rebuilds it from
// S2R for every fetch)
__device__ __forceinline__ void cached_column(uint32_t sc, uint32_t pos, c128 (&t)[4]) {
    const uint32_t a = sc + pos * uint32_t(4 * REG_THREADS * 16);
    constexpr int kStep = REG_THREADS * 16;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(t[0].x), "=d"(t[0].y) : "r"(a) : "memory");
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(t[1].x), "=d"(t[1].y) : "r"(a), "n"(kStep) : "memory");
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(t[2].x), "=d"(t[2].y) : "r"(a), "n"(2 * kStep) : "memory");
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(t[3].x), "=d"(t[3].y) : "r"(a), "n"(3 * kStep) : "memory");
}

}  // namespace

template <int NC> constexpr size_t reg_smem() { return size_t(TILE_BYTES) + size_t(NC - 1) * 4 * 16 * REG_THREADS; }

template <int N, int NC>
__global__ void __launch_bounds__(REG_THREADS, 1)
minors_reg_kernel(const c128* __restrict__ P, int64_t st0, int64_t n_st_total, int S_b, RegTables rt, c128* __restrict__ out) {
    constexpr int K = N - 4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    c128* tile = reinterpret_cast<c128*>(smem_raw);
    c128* Sc = tile + TILE_ELEMS + threadIdx.x;                       // this thread's copy of the Schur columns: entry e at Sc[e * NT]
    uint32_t sc = uint32_t(__cvta_generic_to_shared(Sc));
    asm volatile("mov.b32 %0, %0;" : "+r"(sc));                       // opaque: stays in its register
    const int g = blockIdx.x;
    const int64_t st_first = st0 + int64_t(g) * GROUP;
    const int lane = threadIdx.x & 31;
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);        // tells the compiler that everything derived from it is warp uniform
    stage_tile(tile, P, st_first, n_st_total, REG_THREADS);
    __syncthreads();
    const unsigned char* tb = reinterpret_cast<const unsigned char*>(tile + lane);
    constexpr uint32_t kRowStep = 12 * GROUP * 16, kColStep = GROUP * 16;
    const int bin = blockIdx.y * (REG_THREADS / 32) + warp;
    const int j0 = __ldg(rt.bin_ptr + bin), j1 = __ldg(rt.bin_ptr + bin + 1);
    Trie<NC> c;
    c.step = uint32_t(S_b);
    c128* outp = out + int64_t(g) * GROUP + lane;
    for (int j = j0; j < j1; ++j) {
        const uint32_t jr = __ldg(rt.bin_jobs + j);
        const RegJob* job = rt.jobs + (jr & 255u);
        const uint32_t r = jr >> 8;
        const uint32_t rows = __ldg(rt.row_nibbles + r);
        const ulonglong2 h0 = __ldg(reinterpret_cast<const ulonglong2*>(job));            // lead, cand
        const uint4 h1 = __ldg(reinterpret_cast<const uint4*>(job) + 1);                  // ncand, prog_begin, prog_end, out_base
        c128 detp;
        {
            LuState<N, 0, REG_THREADS> lu;
            uint32_t rb[N], cb[N];
#pragma unroll
            for (int i = 0; i < N; ++i) { rb[i] = ((rows >> (4 * i)) & 15u) * kRowStep; cb[i] = (i < K) ? (uint32_t(h0.x >> (4 * i)) & 15u) * kColStep : 0u; }
            lu.start(tb, nullptr, rb, cb);
            schur_columns<N, NC, 0>(lu, tb, h0.y, int(h1.x), c, Sc);
            detp = lu.detp;
        }
        c.o = outp + (size_t(r) * size_t(rt.n_cols) + size_t(h1.w)) * size_t(S_b);
        c.k = 0;
        // the instance's trie as a flat stream of third-node words {i4, mask of i5, i2, i3, first-of-its-pair flag}
        // (contract.cu: build_reg_host); the column of the next node and the word after it are in flight during a node's last level
        const uint32_t* pw = rt.prog + h1.y;
        const uint32_t* const pend = rt.prog + h1.z;
        if (pw >= pend) continue;
        uint32_t w = __ldg(pw), wn = __ldg(pw + 1);
        c128 t[4];
        cached_column(sc, w & 15u, t);
        while (true) {
            if (w & (1u << 22)) {                                     // new pair node: 2x2 minors of (detp * T[i2], T[i3])
                c128 a[4], b[4];
                cached_column(sc, (w >> 14) & 15u, a);
                cached_column(sc, (w >> 18) & 15u, b);
#pragma unroll
                for (int q = 0; q < 4; ++q) a[q] = cmul(detp, a[q]);
                int k = 0;
#pragma unroll
                for (int x = 0; x < 4; ++x)
#pragma unroll
                    for (int y = x + 1; y < 4; ++y) c.s[k++] = det2(a[x], b[x], a[y], b[y]);
            }
            third_from(c.s, t, c.c3);
            const uint32_t mask5 = (w >> 4) & 0x3ffu;
            ++pw;
            const bool more = pw < pend;
            uint32_t w2 = 0;
            if (more) {
                cached_column(sc, wn & 15u, t);
                w2 = __ldg(pw + 1);                                   // two padding words follow the last job's program
            }
            finish_all<NC, 3>(c, mask5);
            if (!more) break;
            w = wn; wn = w2;
        }
    }
}

cudaError_t launch_minors_reg_impl(int n, const double2* P, int64_t st0, int64_t n_st_total, int n_groups, int S_b,
                                   const RegTables& rt, double2* out, cudaStream_t stream) {
    if (n_groups == 0 || rt.n_bins == 0) return cudaSuccess;
    dim3 grid(n_groups, rt.n_bins / (REG_THREADS / 32));
    if (n == 6) minors_reg_kernel<6, 10><<<grid, REG_THREADS, reg_smem<10>(), stream>>>(P, st0, n_st_total, S_b, rt, out);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

bool minors_reg_supported(int n, int max_candidates) { return n == 6 && max_candidates <= 10; }

cudaError_t configure_reg_kernels() {
    return cudaFuncSetAttribute(minors_reg_kernel<6, 10>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(reg_smem<10>()));
}

}  // namespace wick

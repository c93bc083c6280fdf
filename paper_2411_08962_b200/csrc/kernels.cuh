// Device kernels of the hot path (steps a3-a6 of DESIGN.md), sm_100a.
//
// Data layout on chip ("site per lane"): a warp works on GROUP = 32 consecutive site-times; lane l
// owns site-time st0 + 32 g + l.  The propagators of the 32 sites are staged once per CTA in shared
// memory as tile[element e = 12*row + col][lane] (complex128, 16 B): the bank of an access depends on
// the lane only, so gathers with PER-LANE row order (needed by partial pivoting) are conflict free,
// and the row / column tuples of a minor are warp-uniform.  Minors are written as M[minor][site]
// (site fastest), so every global access of the minor and reduction kernels is a coalesced 512-byte row.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace wick {

constexpr int GROUP = 32;                 // site-times per warp
constexpr int TILE_ELEMS = 144 * GROUP;   // complex128 elements of one flavour tile
constexpr int TILE_BYTES = TILE_ELEMS * 16;
constexpr int MAX_MOMENTA = 64;

struct MomentumList { int n; int v[MAX_MOMENTA][3]; };

// profiling classes (wick_profile in include/wick.h)
constexpr int PROF_MINORS_U = 0, PROF_MINORS_D = 1, PROF_REDUCE = 2, PROF_PROJECT = 3, PROF_CLASSES = 4;
void profile_enable(bool on);
cudaError_t profile_read(double ms[PROF_CLASSES], int64_t count[PROF_CLASSES]);
cudaError_t measure_fp64_peak(double* tflops, cudaStream_t stream);

// launchers (kernels.cu); all enqueue on `stream` and return the cudaGetLastError() code
// `desc`: one descriptor per minor, minor_desc_words(n) 64-bit words each (kernels.cu: struct Desc);
// `ascending`: the descriptors come from the library's own tables (distinct indices, 6x6 tuples ascending), which the cached kernels rely on
int minor_desc_words(int n);
cudaError_t launch_minors(int n, const double2* P, int64_t st0, int64_t n_st_total, int n_groups, int S_b,
                          const void* desc, int64_t n_minors, bool ascending, double2* out, int prof_cls, cudaStream_t stream);
// Instance kernel for grid tables (minors_reg.cu).  An instance-job q is the same for every row tuple: K = n-4 leading
// columns, up to REG_NC_MAX candidate columns behind them, and the trie of the instance's column tuples over candidate
// POSITIONS as a word program.  The minors of a job are stored in trie order from column position out_base of the row
// tuple's list.
constexpr int REG_THREADS = 256;
constexpr int REG_NC_MAX = 10;
struct RegJob {
    unsigned long long lead, cand;        // column indices as 4-bit fields: leading (K), candidates (ncand)
    uint32_t ncand, prog_begin, prog_end, out_base;   // the job's words in RegTables::prog; first column position of its minors
};
static_assert(sizeof(RegJob) == 32, "RegJob is read with 16-byte loads");
struct RegTables {
    int n_cols, n_bins;                   // column tuples per row tuple; warps of work per site group (multiple of 8)
    const RegJob* jobs;                   // [n_jobs <= 256]
    const uint32_t* prog;                 // one word per third node: i4 | mask(i5) << 4 | i2 << 14 | i3 << 18 | first-of-its-pair << 22
    const uint32_t* row_nibbles;          // [n_rows] row indices as 4-bit fields
    const uint32_t* bin_ptr;              // [n_bins + 1]
    const uint32_t* bin_jobs;             // (row tuple << 8) | job, grouped by bin
};
cudaError_t launch_minors_reg(int n, const double2* P, int64_t st0, int64_t n_st_total, int n_groups, int S_b,
                              const RegTables& rt, double2* out, int prof_cls, cudaStream_t stream);
cudaError_t launch_minors_reg_impl(int n, const double2* P, int64_t st0, int64_t n_st_total, int n_groups, int S_b,
                                   const RegTables& rt, double2* out, cudaStream_t stream);   // minors_reg.cu
bool minors_reg_supported(int n, int max_candidates);
cudaError_t configure_reg_kernels();
cudaError_t launch_reduce_flat(const double2* MU, const double2* MD, int n_groups, int S_b,
                               const int32_t* uid, const int32_t* did, const double2* w, int64_t n_terms,
                               double2* partial, int* n_chunks_out, int max_chunks, cudaStream_t stream);
// factor lists + block schedule of the factorised reduction (device pointers; contract.cu builds them)
struct OuterTables {
    int n_cols_u, n_cols_d, n_bins;
    const int32_t *sink_ptr, *sink_rdoff; const double2* sink_c;   // CSR over u row tuple: (rd * n_cols_d, c_i)
    const int32_t *src_ptr, *src_cu; const double2* src_c;         // CSR over d column tuple: (cu, conj c_j)
    const int32_t *ru_ptr, *ru_list, *cd_ptr, *cd_list;            // tuples grouped by sink / source block
    const int32_t* bin_ptr; const int2* items;                     // per warp: list of (sink block, source block)
};
cudaError_t launch_reduce_outer(const double2* MU, const double2* MD, int n_groups, int S_b, const OuterTables& ot,
                                double2* partial, int* n_chunks_out, cudaStream_t stream);
// Staged factorised reduction (reduce_staged_kernel): a CTA walks batches = (one source block's d-column
// range) x (a run of sink blocks); the MD elements of a batch sit in shared memory once, every warp
// streams its u-row tuples' MU rows through a private buffer.  All lists hold positions in the
// block-grouped tuple lists ru_list / rd_list / cu_list / cd_list.
constexpr int STG_THREADS = 192;          // 6 warps, two CTAs per SM (one loads while the other computes)
constexpr int STG_CTAS_PER_SM = 2;
constexpr int STG_MD_CAP = 96;            // MD elements (512 B each) of a batch, general complex coefficients
constexpr int STG_MD_CAP_REAL = 184;      // ... real coefficients: no MU row buffers, the space goes to the MD block
constexpr int STG_ROW_CAP = 15;           // MU elements of one (u-row tuple, source block) row
constexpr int STG_NCD_CAP = 8;            // d columns of a batch piece (one template instance per count)
constexpr int STG_SINK_CAP = 512;         // sink entries of a batch's u-row tuples
constexpr int STG_SRC_CAP = 256;          // source entries of a batch piece's d columns
constexpr int STG_ROWS_CAP = STG_MD_CAP_REAL;  // u-row tuples of a batch
constexpr int stg_md_cap(bool real) { return real ? STG_MD_CAP_REAL : STG_MD_CAP; }
// md_off: the batch's MD element ids ((rd, cd) pairs of its block, rd-major) in StagedTables::md_ids; b_off: the dense real
// B[cu][cd] of its piece in StagedTables::b_dense (real-coefficient schedules).  Both are laid out on the host so that the
// per-batch prologue of the kernel has no dependent look-ups.
struct StagedBatch { int32_t cd_a, cd_b, cu_a, cu_b, rd_a, rd_b, ru_a, ru_b, md_off, b_off, sink_a, sink_n; };   // sink_a, sink_n: first sink entry of the batch's rows, their number
static_assert(sizeof(StagedBatch) == 48, "StagedBatch is read with three 16-byte loads");
struct StagedTables {
    int n_cols_u, n_cols_d, n_bins;
    bool real_coeffs;                                              // all c_i, cbar_j real: 16-byte {coefficient, offset} entries, 2 DFMA per term
    const int32_t *sink_ptr, *sink_rdpos; const double2* sink_c;   // CSR over POSITION in ru_list: (position of rd in rd_list, c_i)
    const int32_t *src_ptr, *src_cupos; const double2* src_c;      // CSR over POSITION in cd_list: (position of cu in cu_list, conj c_j)
    const int32_t *ru_list, *rd_list, *cu_list, *cd_list;
    const int32_t* bin_ptr; const StagedBatch* batches;            // per CTA bin: its batches, fixed order
    const int32_t* md_ids; const double* b_dense;                  // per batch / per piece, see StagedBatch
};
cudaError_t launch_reduce_staged(const double2* MU, const double2* MD, int n_groups, int S_b, const StagedTables& st,
                                 double2* partial, int* n_chunks_out, cudaStream_t stream);
// scale_a / scale_b: NULL or per-site factors multiplied into sigma (Jacobi path: det U, det D)
cudaError_t launch_finalize_sigma(const double2* partial, int n_chunks, int S_b, int64_t n_valid,
                                  double2* sigma_batch, const double2* scale_a, const double2* scale_b, cudaStream_t stream);
// Fused Jacobi path (both flavours 8 <= n <= 11): one term = complementary index sets of both minors (rows J^c in nibbles
// 0..3, columns I^c in nibbles 4..7) and the weight with the Jacobi signs folded in; sigma[site] for sites st0 .. st0 + n_valid - 1
struct JacobiTerm { uint32_t u_idx, d_idx, pad[2]; double2 w; };
static_assert(sizeof(JacobiTerm) == 32, "JacobiTerm is read with 16-byte loads");
cudaError_t launch_jacobi_fused(int n_u, int n_d, const double2* U, const double2* D, int64_t st0, int64_t n_valid,
                                const JacobiTerm* terms, int64_t n_terms, double2* sigma, cudaStream_t stream);
// Jacobi path: inverse [site in batch][12][12] and determinant [site in batch] of the propagators st0 .. of a site batch
cudaError_t launch_inverse12(const double2* P, int64_t st0, int64_t n_st_total, int n_groups, double2* inv_out, double2* det_out,
                             int prof_cls, cudaStream_t stream);
cudaError_t launch_project(const double2* sigma, int L, int T, const MomentumList& mom, double2* C_out,
                           cudaStream_t stream);
// cluster sinks: part[group][cu][cd] of one site batch of ONE timeslice (site0 = index of the batch's first site inside the
// timeslice), then the ordered sum over the groups of the timeslice
cudaError_t launch_block_tensor(const double2* MU, const double2* MD, int S_b, int n_valid, int n_cu, int n_cd,
                                const int32_t* sink_ru, const int32_t* sink_rd, const double2* sink_c, int n_sink,
                                int L, int64_t site0, const int mom[3], double2* part, cudaStream_t stream);
cudaError_t launch_block_sum(const double2* part, int n_groups, int n_pairs, double2* out, cudaStream_t stream);
cudaError_t configure_kernels();          // cudaFuncSetAttribute for the large-shared-memory kernels (once per device)

int64_t launch_counter_get();
int64_t launch_counter_reset();

}  // namespace wick

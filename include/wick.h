/* wick.h -- C-ABI of the B200-native determinant-form Wick contraction (arXiv 2411.08962).
 *
 * PAPER.md = /root/reference/PAPER.md (text of the paper); line numbers refer to that file.
 *
 * The library computes the point-sink two-point correlator of a nucleus in the paper's
 * "optimised determinant algorithm" (Sec. III; CUDA outline App. A, :616-663):
 *
 *     C(t,p) = sum_x e^{i p.x} sum_k w_k det U_x(t)[a_u(k), b_u(k)] det D_x(t)[a_d(k), b_d(k)]
 *                                                              (Eq. 15, Eq. A1/A2 :630-635)
 *
 * U_x(t), D_x(t): 12x12 complex128 up / down propagators from the source to sink site x
 * (row = sink spin-colour index chi = 3*spin + colour, column = source index; Eq. 13 :178).
 * a, b: index tuples selecting n_u (n_d) of the 12 rows / columns.  The weighted term list comes
 * from products of nucleon interpolators eps_abc (q1_a^T C gamma5 q2_b) q3_c,gamma (Eq. 4/5 :105-107).
 *
 * Two groups of entry points:
 *   host  : wick_build_terms*, wick_terms_* -- the once-per-nucleus pre-processing (Sec. III B,
 *           PAPER.md:209-246; App. C :704-732).  Pure CPU, no CUDA call.
 *   device: wick_contract, wick_minor_dets, wick_contract_host -- the per-configuration hot path on
 *           one sm_100a GPU.  There is NO CPU fallback: without a CUDA device they return
 *           WICK_ERR_CUDA.
 *
 * Conventions: every function returns WICK_OK (0) or a negative WICK_ERR_* code and never throws;
 * wick_last_error() gives a thread-local message for the last failure.  Complex numbers are
 * interleaved (re, im) doubles.  "host" / "device" on a pointer says where the memory must live.
 */
#ifndef WICK_B200_H
#define WICK_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WICK_OK              0
#define WICK_ERR_ARG        -1   /* bad argument: NULL pointer, index >= 12, n > 12, gamma > 3, L < 1 ... */
#define WICK_ERR_UNSUPPORTED -2  /* legal but not implemented size / combination                         */
#define WICK_ERR_WORKSPACE  -3   /* workspace smaller than wick_contract_min_workspace_bytes()            */
#define WICK_ERR_CUDA       -4   /* CUDA runtime error (message holds cudaGetErrorString)                 */
#define WICK_ERR_NOMEM      -5   /* host allocation failed                                                */

/* wick_build_terms* flags */
#define WICK_BUILD_IDENTITY_TEST 1u  /* run the randomised identity test (Sec. III B PAPER.md:234-246, App. C) */
#define WICK_BUILD_ISOSPIN       2u  /* the caller promises U == D (m_u = m_d).  Alone (nucleus  */
                                     /* specs): sink terms related by the u <-> d swap are folded (factor 2),  */
                                     /* the list stays an outer product and runs through the factorised        */
                                     /* reduction with about half the products.  With IDENTITY_TEST: the test  */
                                     /* evaluates both flavours on the SAME random matrix and merges the swap  */
                                     /* classes of the flat list.  A handle changed by either can only be      */
                                     /* contracted with U_dev == D_dev (WICK_ERR_ARG otherwise).               */
/* wick_contract flags */
#define WICK_CONTRACT_FORCE_FLAT 1u  /* use the flat (uid, did, w) term list even if a factorised form exists */
#define WICK_CONTRACT_COMPLEX_COEFFS 4u /* staged reduction: do not use the cheaper entries for all-real factor coefficients */
#define WICK_CONTRACT_NO_REG_MINORS 8u /* 6x6 grid tables: use the shared-memory Schur-column cache kernel instead of the register-resident one */
#define WICK_CONTRACT_JACOBI    16u  /* flavours with 8 <= n <= 11: Jacobi's complementary-minor identity (one 12x12 inverse + determinant */
                                     /* per site, then (12-n) x (12-n) minors of the inverse) instead of an LU per minor.  Error grows  */
                                     /* with the condition number of the propagator and a singular propagator contributes 0: opt-in.   */
#define WICK_CONTRACT_JACOBI_UNFUSED 32u /* with JACOBI: keep the minor tables (inverse kernel + minors of the inverse + reduction) even  */
                                     /* where the fused per-site kernel applies (both flavours 8..11, terms <= 8 x unique minors)        */
#define WICK_CONTRACT_NO_STAGED  2u  /* factorised lists: walk the block items from L1/L2 instead of staging them in shared memory */

#define WICK_NUCLEON_PROTON  0
#define WICK_NUCLEON_NEUTRON 1

/* One nucleon of a product interpolator.  kind: 0 = proton  eps_abc (u_a^T C g5 d_b) u_{c,gamma},
 * 1 = neutron eps_abc (d_a^T C g5 u_b) d_{c,gamma} (Eq. 4/5 PAPER.md:105-107; C = gamma4 gamma2 :76,
 * Dirac-Pauli basis).  gamma = open Dirac index 0..3 (0,1 = upper components). */
typedef struct { int32_t kind; int32_t gamma; } wick_nucleon;

/* Opaque canonical term list + unique-minor tables (the paper's zeta_u, zeta_d, Theta of Eq. A1,
 * PAPER.md:628-633, and the "lookup table" of :719).  Owned by the library; free with
 * wick_terms_free.  Device copies of the tables are created lazily by the first device call and
 * are released by wick_terms_free as well. */
typedef struct wick_terms wick_terms;

typedef struct {
    int32_t n_u, n_d;                 /* minor sizes (quarks per flavour)                                   */
    int32_t n_rows_u, n_cols_u;       /* distinct canonical row / column tuples of the u minors (|A_u|,|B_u|) */
    int32_t n_rows_d, n_cols_d;
    int64_t n_minors_u, n_minors_d;   /* unique minors per site = card(zeta_u), card(zeta_d)                */
    int64_t n_terms;                  /* terms of the flat list                                             */
    int32_t is_outer_product;         /* 1: terms = sink list x conj(source list), factorised form present  */
    int32_t n_sink, n_source;         /* lengths of the factor lists (0 if not an outer product)            */
    int64_t n_raw;                    /* raw terms consumed (24^A for nucleus specs, n_raw for lists)       */
    int64_t n_identity_merged;        /* terms removed by the identity test (0 if it did not run)           */
} wick_terms_info;

/* ---------------------------------------------------------------------------------------------
 * Host: term builder (steps a1, a2, a2' of DESIGN.md)
 * ------------------------------------------------------------------------------------------- */

/* Expand the ordered Grassmann product of `n_nucleons` nucleons (Eq. 9) in the exterior
 * algebra, sort every monomial into canonical order (all u indices ascending, then all d indices
 * ascending) with its permutation sign (Eq. 19, redundancy R.1), merge equal
 * monomials, drop Pauli zeros and exact cancellations; then form the correlator term list
 * w_ij = c_i conj(c_j) over (sink i, source j) (Eq. 15) and the unique-minor tables (R.2 :226).
 * nucleons: host, [n_nucleons].  *out receives a new handle.  seed is used by the identity test only.
 * Errors: WICK_ERR_ARG (NULL, n_nucleons < 1, kind not 0/1, gamma not 0..3, more than 12 quarks
 * of one flavour), WICK_ERR_NOMEM. */
int wick_build_terms(const wick_nucleon* nucleons, int n_nucleons, unsigned flags, uint64_t seed,
                     wick_terms** out);

/* Same canonicalisation for a user-supplied flat list (e.g. the seed-generated random list of
 * BASELINE.json configs[4]).  a_u, b_u: host uint8 [n_raw][n_u]; a_d, b_d: host uint8 [n_raw][n_d];
 * entries 0..11 in ANY order; a tuple with a repeated index is legal and contributes exactly 0
 * (dropped).  w_reim: host double [n_raw][2].  Duplicate (a_u,b_u,a_d,b_d) are merged. */
int wick_build_terms_from_list(int n_u, int n_d, int64_t n_raw,
                               const uint8_t* a_u, const uint8_t* b_u,
                               const uint8_t* a_d, const uint8_t* b_d,
                               const double* w_reim, unsigned flags, uint64_t seed, wick_terms** out);

/* ---- general interpolators and correlation matrices (GEVP, Sec. V, Eq. 36-38) ----------------------
 * A wick_operator is an interpolator in canonical form: monomial (u tuple, d tuple) -> complex coefficient.
 *   _from_nucleons : the ordered product of BASELINE nucleons (the sink list wick_build_terms uses);
 *   _from_raw      : any operator given as raw monomials: n_raw products of n_quarks quark fields in operator order,
 *                    flavour[k][q] in {0 = u, 1 = d}, chi[k][q] = 3*spin + colour, coefficient coef_reim[k];
 *                    sorted with the permutation sign (Eq. 19), merged, Pauli zeros dropped;
 *   _paper         : the paper's own interpolators built from the nucleons of Eq. (4)/(5) and the
 *                    projected ones of Eq. (26)/(27) (:271-273): WICK_OP_DEUTERON_EQ20 = n^T (C g5 P+) p  (Eq. 20 :256, 356
 *                    terms, Table II :305); WICK_OP_HELIUM3_EQ21 = p_-^T (C g5) n_+ p_+^J  (Eq. 21 :258; 1026 terms per
 *                    spin component for J = 2, 3, Table II :306).
 * wick_build_terms_matrix: n_ops operators with the same quark content -> n_ops^2 handles, out[k * n_ops + k'] =
 * (operator k at the sink) x conj(operator k' at the source), all over ONE pair of unique-minor tables (union of the row /
 * column tuples), so that wick_contract_many evaluates every determinant once for the whole correlation matrix.
 * Each handle is an ordinary term-list handle: free every one with wick_terms_free. */
typedef struct wick_operator wick_operator;
#define WICK_OP_DEUTERON_EQ20 1
#define WICK_OP_HELIUM3_EQ21  2
int  wick_operator_from_nucleons(const wick_nucleon* nucleons, int n_nucleons, wick_operator** out);
int  wick_operator_from_raw(int n_quarks, int64_t n_raw, const uint8_t* flavour, const uint8_t* chi, const double* coef_reim,
                            wick_operator** out);
int  wick_operator_paper(int which, int J, wick_operator** out);
int  wick_operator_info(const wick_operator* op, int32_t* n_u, int32_t* n_d, int64_t* n_terms);
/* u_tuples uint8 [n_terms][n_u], d_tuples uint8 [n_terms][n_d] (ascending), coef_reim double [n_terms][2]; any may be NULL */
int  wick_operator_export(const wick_operator* op, uint8_t* u_tuples, uint8_t* d_tuples, double* coef_reim);
void wick_operator_free(wick_operator* op);
int  wick_build_terms_matrix(const wick_operator* const* ops, int n_ops, unsigned flags, wick_terms** out);

/* ---- cluster sinks (the block algorithm of Eq. 6-8 :110-125 when the clusters are single nucleons) -----------
 * Two clusters A (quarks at sink site x) and B (quarks at sink site y), each projected to its own momentum:
 *     C(t) = sum_{x,y} e^{i p_A.x} e^{i p_B.y} < O_A(x,t) O_B(y,t)  Obar_source(0) >.
 * The stacked determinants are expanded along the rows of cluster A (generalised Laplace expansion), so the two site sums
 * factorise into the block tensors   B_X[t][S_u][S_d] = sum_x e^{i p.x} sum_i c_i det U_x[a_u(i), S_u] det D_x[a_d(i), S_d]
 * over ALL column subsets S_u, S_d (lexicographic order of the ascending tuples), evaluated on the device by
 * wick_block_tensor from a block handle (wick_build_block_terms), and combined on the host, lattice independent, by
 * wick_combine_two_clusters:  C[t] = (-1)^(|d_A||u_B|) sum_j conj(c_j) sum_{S_u, S_d} sign B_A[t][S_u][S_d] B_B[t][b_u(j) \ S_u][b_d(j) \ S_d].
 * wick_operator_product: the ordered product A.B (the natural source operator).  The device kernel is flat over the sink
 * terms of the cluster: meant for small clusters (nucleons, deuteron); a He-4-sized cluster needs a factorised kernel (not built).
 *   out_dev   : device complex128 [T][C(12,n_u)][C(12,n_d)];  momentum: host int32 [3];  workspace >= _workspace_bytes, 256-byte aligned.
 *   BA_reim, BB_reim: host copies of the two block tensors;  C_reim: host double [T][2]. */
int  wick_operator_product(const wick_operator* a, const wick_operator* b, wick_operator** out);
int  wick_build_block_terms(const wick_operator* cluster, wick_terms** out);
size_t wick_block_tensor_workspace_bytes(const wick_terms* block_terms, int L);
int  wick_block_tensor(const void* U_dev, const void* D_dev, const wick_terms* block_terms, const int32_t* momentum, int L, int T,
                       void* out_dev, void* workspace_dev, size_t workspace_bytes, unsigned flags, void* cuda_stream);
int  wick_combine_two_clusters(const wick_operator* a, const wick_operator* b, const wick_operator* source,
                               const double* BA_reim, const double* BB_reim, int T, double* C_reim);

int  wick_terms_get_info(const wick_terms* terms, wick_terms_info* info);

/* Copy the tables out (host, caller-allocated; any pointer may be NULL to skip it).
 * u_rows [n_rows_u][n_u], u_cols [n_cols_u][n_u], d_rows [n_rows_d][n_d], d_cols [n_cols_d][n_d]:
 * ascending tuples, sorted lexicographically. */
int  wick_terms_export_tuples(const wick_terms* terms, uint8_t* u_rows, uint8_t* u_cols,
                              uint8_t* d_rows, uint8_t* d_cols);
/* Unique minor m of flavour u is det U[u_rows[u_minor_row[m]], u_cols[u_minor_col[m]]].
 * u_minor_row/col: int32 [n_minors_u]; d_*: int32 [n_minors_d]. */
int  wick_terms_export_minors(const wick_terms* terms, int32_t* u_minor_row, int32_t* u_minor_col,
                              int32_t* d_minor_row, int32_t* d_minor_col);
/* Flat terms first .. first+count-1: uid, did int32 [count] (unique-minor ids), w_reim double [count][2]. */
int  wick_terms_export_terms(const wick_terms* terms, int64_t first, int64_t count,
                             int32_t* uid, int32_t* did, double* w_reim);
/* Factor lists of an outer-product term list: sink i = (row tuple ids, c_i), source j = (column tuple
 * ids, conj c_j); term (i,j) has uid = sink_ru[i]*n_cols_u + src_cu[j], did likewise, w = sink_c*src_c.
 * Returns WICK_ERR_UNSUPPORTED if !is_outer_product. */
int  wick_terms_export_factors(const wick_terms* terms, int32_t* sink_ru, int32_t* sink_rd, double* sink_c_reim,
                               int32_t* src_cu, int32_t* src_cd, double* src_c_reim);
/* The order in which the minors kernel walks one flavour's unique minors (flavour 0 = u, 1 = d) and the order in which
 * it takes each minor's columns (consecutive minors share their row tuple and leading columns; for
 * n >= 9 the column tuples are clustered by a common set of n-4 leading columns).  minor_id int32 [n_minors]: position ->
 * unique-minor id; proc_cols uint8 [n_minors][n]; negate uint8 [n_minors]: 1 if that column order is an odd
 * permutation of the ascending tuple (the kernel negates the result).  Any pointer may be NULL. */
int  wick_terms_export_minor_order(const wick_terms* terms, int flavour, int32_t* minor_id, uint8_t* proc_cols, uint8_t* negate);
/* Host-only self-check of the schedule of the staged factorised reduction (reduce_staged_kernel) for
 * n_bins CTA bins: every (u-row tuple, d-column tuple) pair of the factorised sum (PAPER.md Eq. A1-A5 regrouped) is
 * covered by exactly one batch, every batch fits the shared-memory capacities and every coefficient entry points
 * inside its staged block.  Outputs (any may be NULL): number of batches, pairs covered, largest MD block, most
 * u-row tuples in a batch.  WICK_ERR_UNSUPPORTED: not an outer-product list, or a block too large to stage. */
int  wick_terms_staged_schedule_check(const wick_terms* terms, int n_bins, int64_t* n_batches, int64_t* n_pairs,
                                      int64_t* max_md_elements, int64_t* max_rows);
void wick_terms_free(wick_terms* terms);

/* ---------------------------------------------------------------------------------------------
 * Device: the hot path (steps a3-a6 of DESIGN.md)
 * ------------------------------------------------------------------------------------------- */

/* Workspace sizes in bytes for wick_contract on a lattice of L^3 sites and T timeslices.
 * _min: smallest legal workspace (one 32-site batch); _workspace_bytes: the recommended size
 * (site batches of up to ~2 GiB of minors).  Any size >= _min is accepted; more lets the library use
 * larger site batches.  Both return 0 on a bad argument. */
size_t wick_contract_min_workspace_bytes(const wick_terms* terms, int L, int T, int n_mom);
size_t wick_contract_workspace_bytes(const wick_terms* terms, int L, int T, int n_mom);

/* C[p][t] = sum_x e^{+2 pi i (n_p . x)/L} sum_k w_k detU detD  for t = 0..T-1 (Eq. 15 / A1 / A2 / A7).
 * U_dev, D_dev : device, complex128 [T][L^3][12][12], site s = x + L*(y + L*z), 16-byte aligned.
 *                U_dev == D_dev is legal (isospin limit); if the two flavours then also share their
 *                unique-minor table (e.g. deuteron, He-4) the minors are evaluated once and serve both flavours.
 * momenta      : host, int32 [n_mom][3], integer units of 2*pi/L (read before the call returns).
 * C_out_dev    : device, complex128 [n_mom][T].
 * sigma_out_dev: NULL or device complex128 [T][L^3]: sigma(x,t) = sum_k w_k detU detD (Eq. A5 :646).
 * workspace_dev: device, workspace_bytes >= wick_contract_min_workspace_bytes, 256-byte aligned.
 * cuda_stream  : a cudaStream_t (NULL = default stream).  All work is enqueued on it; the call does
 *                not synchronise (except for a one-time upload of the tables on first use of
 *                `terms`).  Results are bit-reproducible run to run (no floating-point atomics;
 *                fixed-shape reductions).
 * Ownership: the caller owns every buffer; the library only keeps the tables inside `terms`. */
int wick_contract(const void* U_dev, const void* D_dev, const wick_terms* terms,
                  const int32_t* momenta, int n_mom, int L, int T,
                  void* C_out_dev, void* sigma_out_dev,
                  void* workspace_dev, size_t workspace_bytes, unsigned flags, void* cuda_stream);

/* Correlation matrix (GEVP, Sec. V, Eq. 36-38): n_lists term lists that share their unique-minor tables
 * (wick_build_terms_matrix).  Per site batch every determinant is evaluated ONCE (step a4), then each list runs its own
 * weighted-product kernel (a5) and projection (a6).  C_out_dev: device complex128 [n_lists][n_mom][T]; sigma_out_dev: NULL or
 * [n_lists][T][L^3]; workspace of at least wick_contract_many_workspace_bytes (the single-list sizes plus one sigma buffer per
 * extra list).  Everything else as wick_contract.  WICK_ERR_UNSUPPORTED if the lists do not share their tables. */
size_t wick_contract_many_workspace_bytes(const wick_terms* terms0, int n_lists, int L, int T, int n_mom);
int wick_contract_many(const void* U_dev, const void* D_dev, const wick_terms* const* lists, int n_lists,
                       const int32_t* momenta, int n_mom, int L, int T, void* C_out_dev, void* sigma_out_dev,
                       void* workspace_dev, size_t workspace_bytes, unsigned flags, void* cuda_stream);

/* Same computation from HOST buffers (U_host, D_host, C_out_host, sigma_out_host: host memory,
 * pinned or pageable, same layouts).  Allocates device memory itself, streams the propagators
 * timeslice block by timeslice block (blocks of <= 256 MB per flavour; H2D of block b+1 on a second stream while block b
 * computes), copies C back and synchronises before returning; on an error both streams are drained first.
 * U_host == D_host is legal (one propagator, copied once, U_dev == D_dev on the device).  Test hook: the environment
 * variable WICK_HOST_BLOCK_BYTES overrides the block size so that the multi-block path can be exercised on small lattices. */
int wick_contract_host(const void* U_host, const void* D_host, const wick_terms* terms,
                       const int32_t* momenta, int n_mom, int L, int T,
                       void* C_out_host, void* sigma_out_host, unsigned flags);

/* Step a4 alone: unique minor determinants ("analytic up to 4x4, LU above"; device_det,
 * App. A :648-652).  out[m][s] = det P_s[rows[m], cols[m]] for n_sites matrices.
 * P_dev  : device complex128 [n_sites][12][12].
 * rows, cols: host uint8 [n_minors][n], entries 0..11 (any order; no canonicalisation is applied).
 * out_dev: device complex128 [n_minors][n_sites].  n = 0..12 (n = 0 gives 1).  Synchronises. */
int wick_minor_dets(const void* P_dev, int64_t n_sites, int n, const uint8_t* rows, const uint8_t* cols,
                    int64_t n_minors, void* out_dev, void* cuda_stream);

/* wick_minor_dets for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): same arguments, same kernels, same result, but NOTHING is allocated.  The scratch wick_minor_dets
 * allocates per call (device copy of the minor descriptors; for n_sites not a multiple of 32 the padded staging buffer of
 * the results) lives in one static device array of WICK_STATIC_SCRATCH_BYTES that every GPU which loads the library
 * holds until exit.  Limits: n_minors <= WICK_STATIC_MAX_MINORS per call; if n_sites is not a multiple of 32,
 * n_minors x 32 sites x 16 B must fit the array behind the descriptors (always true within the minor limit).  Beyond
 * them the call returns WICK_ERR_UNSUPPORTED with a message; it never falls back to allocating.  All calls on a device
 * share the array, which keeps the last call's contents (nothing in it needs to start at zero: each call rewrites the
 * part it reads), so calls that overlap on the GPU (different streams or host threads) race: serialise them.
 * Synchronises the stream before returning, like wick_minor_dets.  wick_static_scratch_bytes() returns the array size. */
#define WICK_STATIC_SCRATCH_BYTES (16u << 20)
#define WICK_STATIC_MAX_MINORS    4096
int wick_minor_dets_static(const void* P_dev, int64_t n_sites, int n, const uint8_t* rows, const uint8_t* cols,
                           int64_t n_minors, void* out_dev, void* cuda_stream);
size_t wick_static_scratch_bytes(void);

/* Step a4 for one flavour (0 = u, 1 = d) of a handle's unique-minor table, through exactly the kernels wick_contract
 * launches for it (the register-resident / cached kernels for the library's own tables; `flags` as for wick_contract).
 * P_dev: device complex128 [n_sites][12][12]; out_dev: device complex128 [n_minors][S] with S = n_sites rounded up to a
 * multiple of 32 (columns >= n_sites hold the minors of a zero propagator: 0 for n >= 1).  Enqueues on cuda_stream, does not synchronise. */
int wick_terms_minor_table(const void* P_dev, int64_t n_sites, const wick_terms* terms, int flavour, unsigned flags,
                           void* out_dev, void* cuda_stream);

/* Measurement helpers (bench.py).  wick_profile_enable(1) makes every kernel launch of this thread's
 * device calls record CUDA events on its stream; wick_profile_read synchronises them, returns the
 * summed device time and launch count per class and clears the record.  Classes: 0 = u minors,
 * 1 = d minors, 2 = weighted-product reduction, 3 = sigma finalisation + momentum projection.
 * wick_measure_fp64_peak times a register-only DFMA stream on all SMs (the FP64 roofline
 * denominator) and returns TFLOP/s; it synchronises. */
typedef struct { double ms[4]; int64_t launches[4]; } wick_profile;
int wick_profile_enable(int on);
int wick_profile_read(wick_profile* out);
int wick_measure_fp64_peak(double* tflops_out, void* cuda_stream);

/* Number of kernel launches issued by this thread's device calls since the last reset (bench.py's
 * gpu_launches); _reset returns the old value. */
int64_t wick_launch_count(void);
int64_t wick_launch_count_reset(void);

/* wick_contract_host keeps its device buffers (propagator blocks, workspace), two streams and four events per host
 * thread between calls; this frees them (call it from the thread that made the host calls, with its device current). */
void wick_release_cached_buffers(void);

/* Message of the last error on this thread (thread-local, never NULL); library version string. */
const char* wick_last_error(void);
const char* wick_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WICK_B200_H */

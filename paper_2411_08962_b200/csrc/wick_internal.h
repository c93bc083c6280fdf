// Internal structures shared by the host term builder (term_builder.cpp) and the device path
// (contract.cu).  Not part of the C-ABI (include/wick.h).  No CUDA types here so that the host
// builder compiles as plain C++.
#pragma once
#include <complex>
#include <map>
#include <cstdint>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/wick.h"

namespace wick {

typedef std::complex<double> cplx;

// One flavour's unique-minor tables (the paper's zeta_q, Eq. A1).
struct FlavourTables {
    int n = 0;                                  // minor size
    std::vector<uint16_t> rows, cols;           // distinct index sets as 12-bit masks, in lexicographic tuple order
    std::vector<int32_t> minor_row, minor_col;  // unique minor m = (rows[minor_row[m]], cols[minor_col[m]])
};

// Factor of an outer-product list.  Sink: (row-tuple ids, c_i).  Source: (column-tuple ids, conj c_j).
struct FactorTerm { int32_t qu, qd; cplx c; };

// Schedule of the staged factorised reduction for one CTA-bin count (contract.cu: ensure_staged)
struct StagedDev {
    void* blob = nullptr;
    int n_bins = 0;
    bool real = false;                          // schedule built for the real-coefficient kernel
    const int32_t *sink_ptr = nullptr, *sink_rdpos = nullptr, *src_ptr = nullptr, *src_cupos = nullptr;   // CSR by list position
    const double *sink_c = nullptr, *src_c = nullptr;
    const int32_t *ru_list = nullptr, *rd_list = nullptr, *cu_list = nullptr, *cd_list = nullptr;
    const int32_t* bin_ptr = nullptr;
    const void* batches = nullptr;
    const int32_t* md_ids = nullptr;            // MD element ids of every batch
    const double* b_dense = nullptr;            // dense B[cu][cd] of every piece (real-coefficient schedules)
};

// Job schedule of the register-resident minors kernel for one flavour and bin count (contract.cu: ensure_reg)
struct RegDev {
    void* blob = nullptr;
    int n_bins = 0;
    const void *jobs = nullptr, *prog = nullptr, *rows = nullptr, *bin_ptr = nullptr, *bin_jobs = nullptr;
};

// Device-resident copies, created by the first device call that needs them (contract.cu).
struct DeviceTables {
    int device = -1;
    void* blob = nullptr;                       // one allocation holding the minor tables + factor lists
    const void* jacobi_desc[2] = {nullptr, nullptr};    // n = 8..11: complementary-minor descriptors (contract.cu: build_jacobi_descs)
    const void* minor_desc[2] = {nullptr, nullptr};     // [n_minors] packed (row indices, column indices), kernels.cu: struct Desc
    // factorised reduction: sink CSR over u row-tuple id, source CSR over d column-tuple id
    const int32_t* sink_ptr = nullptr;          // [n_rows_u + 1]
    const int32_t* sink_rd = nullptr;           // [n_sink]   d row-tuple id
    const double* sink_c = nullptr;             // [n_sink][2]
    const int32_t* src_ptr = nullptr;           // [n_cols_d + 1]
    const int32_t* src_cu = nullptr;            // [n_source] u column-tuple id
    const double* src_c = nullptr;              // [n_source][2]
    int max_sink_per_row = 0;
    // block schedule of the factorised reduction (contract.cu: build_reduce_schedule)
    const int32_t* sink_rdoff = nullptr;        // [n_sink]   rd * n_cols_d (element offset of the MD row)
    const int32_t* ru_ptr = nullptr;            // [n_sink_comp + 1]  u row tuples grouped by sink component
    const int32_t* ru_list = nullptr;
    const int32_t* cd_ptr = nullptr;            // [n_src_comp + 1]   d column tuples grouped by source component
    const int32_t* cd_list = nullptr;
    const int32_t* red_bin_ptr = nullptr;       // [n_red_bins + 1]
    const int32_t* red_items = nullptr;         // [n_items][2]  (sink component, source component)
    int n_red_bins = 0;
    int staged_state = 0;                       // 0 = not checked, 1 = eligible, -1 = blocks too large for the staged kernel
    std::map<int, StagedDev> staged;            // by 2 * number of CTA bins + (general-coefficient schedule ? 1 : 0)
    int reg_state[2] = {0, 0};                  // per flavour: 0 = not checked, 1 = register-resident minors kernel usable, -1 = not
    std::map<int, RegDev> reg[2];               // by number of warp bins per site group
    // flat list (uploaded only when the flat path runs)
    void* block_blob = nullptr;                 // block handles: sink terms as flat arrays (contract.cu: wick_block_tensor)
    const void *block_c = nullptr, *block_ru = nullptr, *block_rd = nullptr;
    void* jf_blob = nullptr;                    // fused Jacobi path: flat terms with complementary index sets (contract.cu)
    void* flat_blob = nullptr;
    const int32_t* t_uid = nullptr;
    const int32_t* t_did = nullptr;
    const double* t_w = nullptr;                // [n_terms][2]
};

void set_error(const std::string& msg);         // thread-local message behind wick_last_error()

}  // namespace wick

struct wick_terms {
    int n_u = 0, n_d = 0;
    wick::FlavourTables f[2];                   // 0 = u, 1 = d
    bool outer = false;
    bool block_mode = false;                    // wick_build_block_terms: sink list only, columns = all subsets (wick_block_tensor)
    bool needs_u_equals_d = false;              // built with WICK_BUILD_ISOSPIN and changed by it: only valid for U == D
    std::vector<wick::FactorTerm> sink, source; // outer-product factor lists (source holds conj c_j)
    int64_t n_terms = 0, n_raw = 0, n_identity_merged = 0;
    // flat list: always present for generic lists, materialised on demand for outer-product lists
    mutable std::mutex mu;
    mutable bool flat_ready = false;
    mutable std::vector<int32_t> t_uid, t_did;
    mutable std::vector<wick::cplx> t_w;
    mutable wick::DeviceTables dev;
    void ensure_flat() const;                   // term_builder.cpp
};

extern "C" void wick_terms_release_device(wick::DeviceTables* d);   // contract.cu (cudaFree)

// C-ABI device entry points: wick_contract, wick_contract_host, wick_minor_dets (include/wick.h).
// Host logic only: table upload, workspace carving, site batching and kernel launch order.
// Every arithmetic step of the path runs in the kernels of kernels.cu.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <string>
#include <vector>

#include "kernels.cuh"
#include "wick_internal.h"

using namespace wick;

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

#define WICK_CUDA(call)                                                                      \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess) {                                                             \
            set_error(std::string(#call) + ": " + cudaGetErrorString(e_));                   \
            return WICK_ERR_CUDA;                                                            \
        }                                                                                    \
    } while (0)

int ensure_configured() {
    static thread_local int configured_device = -1;
    int dev = -1;
    WICK_CUDA(cudaGetDevice(&dev));
    if (configured_device != dev) {
        WICK_CUDA(configure_kernels());
        configured_device = dev;
    }
    return WICK_OK;
}

struct BlobBuilder {
    std::vector<unsigned char> host;
    size_t add(const void* src, size_t bytes) {
        const size_t off = align_up(host.size(), 256);
        host.resize(off + bytes);
        if (bytes) std::memcpy(host.data() + off, src, bytes);
        return off;
    }
};

// index set (12-bit mask) -> its indices as 4-bit fields, ascending
uint64_t nibbles_of_mask(uint16_t mask) {
    uint64_t w = 0;
    int k = 0;
    for (int b = 0; b < 12; ++b)
        if (mask & (1u << b)) w |= uint64_t(b) << (4 * k++);
    return w;
}

// minor descriptors for launch_minors (kernels.cu: struct Desc); out_id / negate only exist for n >= 9
void pack_minor_desc(int n, uint64_t rows, uint64_t cols, uint32_t out_id, bool negate, uint64_t* out) {
    if (minor_desc_words(n) == 1) out[0] = (rows & 0xffffffffull) | (cols << 32);
    else {
        out[0] = (rows & 0xffffffffffffull) | (uint64_t(out_id & 0xffffu) << 48);
        out[1] = (cols & 0xffffffffffffull) | (uint64_t((out_id >> 16) & 0x7fffu) << 48) | (uint64_t(negate ? 1 : 0) << 63);
    }
}

// Processing order of one flavour's minors (what minors_kernel walks, position by position).
struct MinorOrder {
    std::vector<uint32_t> minor;      // position -> unique-minor id
    std::vector<uint64_t> cols;       // position -> column indices as 4-bit fields in processing order
    std::vector<uint8_t> negate;      // position -> the processing order is an odd permutation of the ascending tuple
};

// n <= 8: minor order (row tuple by row tuple, column tuples lexicographic: consecutive minors share leading columns).
// n >= 9: the K = n-4 pivot steps dominate, so the column tuples are clustered by a shared set of K LEADING columns:
// greedily take the K-subset contained in most of the remaining tuples, put it first (ascending) and the rest of each
// tuple behind it (ascending); minors are sorted by (row tuple, cluster, rest).  The determinant with permuted columns
// is the determinant times the parity of the permutation, kept as a sign bit of the descriptor.
MinorOrder build_minor_order(const FlavourTables& ft) {
    const int n = ft.n;
    const size_t nm = ft.minor_row.size();
    MinorOrder o;
    o.minor.resize(nm); o.cols.resize(nm); o.negate.assign(nm, 0);
    if (n <= 8) {
        for (size_t m = 0; m < nm; ++m) { o.minor[m] = uint32_t(m); o.cols[m] = nibbles_of_mask(ft.cols[size_t(ft.minor_col[m])]); }
        return o;
    }
    const int K = n - 4;
    const size_t nc = ft.cols.size();
    std::vector<int> cluster(nc, -1);
    std::vector<uint64_t> proc(nc, 0);
    std::vector<uint8_t> odd(nc, 0);
    size_t left = nc;
    for (int cl = 0; left > 0; ++cl) {
        std::map<uint16_t, int> count;                                  // K-subset (mask) -> number of unassigned tuples containing it
        for (size_t c = 0; c < nc; ++c) {
            if (cluster[c] >= 0) continue;
            const uint16_t full = ft.cols[c];
            for (uint16_t sub = full;; sub = uint16_t((sub - 1) & full)) {   // all submasks of the tuple
                if (__builtin_popcount(sub) == K) count[sub]++;
                if (sub == 0) break;
            }
        }
        uint16_t best = 0; int best_n = -1;
        for (const auto& kv : count)                                    // most tuples; ties: the smallest mask value
            if (kv.second > best_n) { best = kv.first; best_n = kv.second; }
        for (size_t c = 0; c < nc; ++c) {
            if (cluster[c] >= 0 || (ft.cols[c] & best) != best) continue;
            cluster[c] = cl; --left;
            const uint64_t lead = nibbles_of_mask(best), rest = nibbles_of_mask(uint16_t(ft.cols[c] & ~best));
            proc[c] = lead | (rest << (4 * K));
            int inv = 0;                                                // inversions of the processing order
            for (int i = 0; i < n; ++i)
                for (int j = i + 1; j < n; ++j) inv += ((proc[c] >> (4 * i)) & 15u) > ((proc[c] >> (4 * j)) & 15u);
            odd[c] = uint8_t(inv & 1);
        }
    }
    auto tuple_key = [n](uint64_t w) { uint64_t k = 0; for (int i = 0; i < n; ++i) k = (k << 4) | ((w >> (4 * i)) & 15u); return k; };
    std::vector<uint32_t> idx(nm);
    for (size_t m = 0; m < nm; ++m) idx[m] = uint32_t(m);
    std::stable_sort(idx.begin(), idx.end(), [&](uint32_t a, uint32_t b) {
        if (ft.minor_row[a] != ft.minor_row[b]) return ft.minor_row[a] < ft.minor_row[b];
        const size_t ca = size_t(ft.minor_col[a]), cb = size_t(ft.minor_col[b]);
        if (cluster[ca] != cluster[cb]) return cluster[ca] < cluster[cb];
        return tuple_key(proc[ca]) < tuple_key(proc[cb]);
    });
    for (size_t k = 0; k < nm; ++k) {
        const size_t c = size_t(ft.minor_col[idx[k]]);
        o.minor[k] = idx[k]; o.cols[k] = proc[c]; o.negate[k] = odd[c];
    }
    return o;
}

std::vector<uint64_t> build_minor_descs(const FlavourTables& ft) {
    const int words = minor_desc_words(ft.n);
    const MinorOrder o = build_minor_order(ft);
    std::vector<uint64_t> desc(o.minor.size() * size_t(words));
    for (size_t k = 0; k < o.minor.size(); ++k)
        pack_minor_desc(ft.n, nibbles_of_mask(ft.rows[size_t(ft.minor_row[o.minor[k]])]), o.cols[k], o.minor[k], o.negate[k] != 0,
                        desc.data() + k * size_t(words));
    return desc;
}

// Jacobi path (flag WICK_CONTRACT_JACOBI, n >= 8): descriptors of the complementary minors.  Minor (I, J) of A equals
// (-1)^(sum I + sum J) det A det (A^-1)[J^c, I^c] (0-based index sums): rows J^c, columns I^c, the sign in bit 31.
std::vector<uint64_t> build_jacobi_descs(const FlavourTables& ft) {
    const int m = 12 - ft.n;
    std::vector<uint64_t> desc(ft.minor_row.size());
    for (size_t k = 0; k < desc.size(); ++k) {
        const uint16_t I = ft.rows[size_t(ft.minor_row[k])], J = ft.cols[size_t(ft.minor_col[k])];
        int sum = 0;
        for (int b = 0; b < 12; ++b) sum += ((I >> b) & 1) * b + ((J >> b) & 1) * b;
        const uint64_t rows = nibbles_of_mask(uint16_t(~J & 0xfff)), cols = nibbles_of_mask(uint16_t(~I & 0xfff));
        pack_minor_desc(m, rows, cols, uint32_t(k), false, &desc[k]);
        if (sum & 1) desc[k] |= uint64_t(1) << 31;
    }
    return desc;
}

// Fused Jacobi path: flat term table with complementary index sets and the signs folded into the weights.
int ensure_jacobi_fused(const wick_terms* t, cudaStream_t stream, const JacobiTerm** out) {
    try { t->ensure_flat(); } catch (const std::bad_alloc&) { set_error("flat term list: out of host memory"); return WICK_ERR_NOMEM; }
    std::lock_guard<std::mutex> lock(t->mu);
    DeviceTables& d = t->dev;
    if (d.jf_blob) { *out = static_cast<const JacobiTerm*>(d.jf_blob); return WICK_OK; }
    std::vector<JacobiTerm> tab(size_t(t->n_terms));
    auto comp = [](const FlavourTables& ft, int32_t m, int* sum) {
        const uint16_t I = ft.rows[size_t(ft.minor_row[size_t(m)])], J = ft.cols[size_t(ft.minor_col[size_t(m)])];
        for (int b = 0; b < 12; ++b) *sum += ((I >> b) & 1) * b + ((J >> b) & 1) * b;
        return uint32_t(nibbles_of_mask(uint16_t(~J & 0xfff)) & 0xffffu) | (uint32_t(nibbles_of_mask(uint16_t(~I & 0xfff)) & 0xffffu) << 16);
    };
    for (size_t k = 0; k < tab.size(); ++k) {
        int sum = 0;
        tab[k].u_idx = comp(t->f[0], t->t_uid[k], &sum);
        tab[k].d_idx = comp(t->f[1], t->t_did[k], &sum);
        tab[k].pad[0] = tab[k].pad[1] = 0;
        const double sg = (sum & 1) ? -1.0 : 1.0;
        tab[k].w = make_double2(sg * t->t_w[k].real(), sg * t->t_w[k].imag());
    }
    void* blob = nullptr;
    WICK_CUDA(cudaMalloc(&blob, std::max<size_t>(tab.size() * sizeof(JacobiTerm), 256)));
    cudaError_t e = cudaMemcpyAsync(blob, tab.data(), tab.size() * sizeof(JacobiTerm), cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) { cudaFree(blob); set_error(std::string("Jacobi term table upload: ") + cudaGetErrorString(e)); return WICK_ERR_CUDA; }
    d.jf_blob = blob;
    *out = static_cast<const JacobiTerm*>(blob);
    return WICK_OK;
}

// Connected components of the bipartite graph (qu -- qd) of a factor list.  Physical sink lists are
// block diagonal (He-4: 199 blocks of at most 15 x 15 tuples), so the factorised reduction
//   sigma = sum_{ru,cd} (sum_i c_i MD[rd_i,cd]) (sum_j cbar_j MU[ru,cu_j])
// splits into (sink block, source block) items that each touch a small, disjoint set of minors:
// every MU / MD element belongs to exactly one item, so the minor buffers are read from DRAM once.
struct Components { std::vector<int> of_u, of_d; int n = 0; };

Components factor_components(int n_u, int n_d, const std::vector<FactorTerm>& list) {
    std::vector<int> parent(size_t(n_u) + size_t(n_d));
    for (size_t i = 0; i < parent.size(); ++i) parent[i] = int(i);
    auto find = [&](int x) { while (parent[x] != x) { parent[x] = parent[parent[x]]; x = parent[x]; } return x; };
    for (const FactorTerm& f : list) {
        const int a = find(f.qu), b = find(n_u + f.qd);
        if (a != b) parent[std::max(a, b)] = std::min(a, b);
    }
    Components c;
    c.of_u.assign(n_u, -1); c.of_d.assign(n_d, -1);
    std::vector<int> label(parent.size(), -1);
    for (const FactorTerm& f : list) {                        // label in order of first appearance
        const int r = find(f.qu);
        if (label[r] < 0) label[r] = c.n++;
        c.of_u[f.qu] = label[r]; c.of_d[f.qd] = label[r];
    }
    return c;
}

constexpr int MAX_RED_BINS = 2048;               // warps of work per site group (8 per CTA -> 256 partial rows)

struct ReduceSchedule {
    std::vector<int32_t> ru_ptr, ru_list, cd_ptr, cd_list, bin_ptr, items;
    int n_bins = 0;
};

// items = (sink block k, source block k'); cost = complex FMAs of its (ru, cd) double loop.
// Longest-processing-time assignment to n_bins warps; every bin's item order is fixed, so the
// reduction stays bit-reproducible.
ReduceSchedule build_reduce_schedule(const wick_terms* t, const std::vector<int32_t>& sink_ptr,
                                     const std::vector<int32_t>& src_ptr) {
    const int nru = int(t->f[0].rows.size()), nrd = int(t->f[1].rows.size());
    const int ncu = int(t->f[0].cols.size()), ncd = int(t->f[1].cols.size());
    const Components cs = factor_components(nru, nrd, t->sink);
    const Components cq = factor_components(ncu, ncd, t->source);
    ReduceSchedule r;
    auto group = [](const std::vector<int>& comp_of, int n_comp, std::vector<int32_t>& ptr, std::vector<int32_t>& list) {
        ptr.assign(size_t(n_comp) + 1, 0);
        for (int c : comp_of) if (c >= 0) ptr[size_t(c) + 1]++;
        for (int c = 0; c < n_comp; ++c) ptr[size_t(c) + 1] += ptr[size_t(c)];
        list.resize(size_t(ptr[size_t(n_comp)]));
        std::vector<int32_t> fill(ptr.begin(), ptr.end() - 1);
        for (size_t x = 0; x < comp_of.size(); ++x) if (comp_of[x] >= 0) list[size_t(fill[size_t(comp_of[x])]++)] = int32_t(x);
    };
    group(cs.of_u, cs.n, r.ru_ptr, r.ru_list);
    group(cq.of_d, cq.n, r.cd_ptr, r.cd_list);
    std::vector<int64_t> nnz_s(size_t(cs.n), 0), nnz_q(size_t(cq.n), 0);
    for (int k = 0; k < cs.n; ++k)
        for (int a = r.ru_ptr[size_t(k)]; a < r.ru_ptr[size_t(k) + 1]; ++a) {
            const int ru = r.ru_list[size_t(a)];
            nnz_s[size_t(k)] += sink_ptr[size_t(ru) + 1] - sink_ptr[size_t(ru)];
        }
    for (int k = 0; k < cq.n; ++k)
        for (int b = r.cd_ptr[size_t(k)]; b < r.cd_ptr[size_t(k) + 1]; ++b) {
            const int cd = r.cd_list[size_t(b)];
            nnz_q[size_t(k)] += src_ptr[size_t(cd) + 1] - src_ptr[size_t(cd)];
        }
    struct Item { int64_t cost; int32_t k, kp; };
    std::vector<Item> items;
    items.reserve(size_t(cs.n) * size_t(cq.n));
    for (int k = 0; k < cs.n; ++k) {
        const int64_t na = r.ru_ptr[size_t(k) + 1] - r.ru_ptr[size_t(k)];
        for (int kp = 0; kp < cq.n; ++kp) {
            const int64_t nb = r.cd_ptr[size_t(kp) + 1] - r.cd_ptr[size_t(kp)];
            items.push_back({nb * nnz_s[size_t(k)] + na * nnz_q[size_t(kp)] + na * nb + 4, k, kp});
        }
    }
    std::stable_sort(items.begin(), items.end(), [](const Item& a, const Item& b) { return a.cost > b.cost; });
    int n_bins = int(std::min<size_t>(items.size(), size_t(MAX_RED_BINS)));
    n_bins = std::max(8, (n_bins + 7) / 8 * 8);
    std::vector<int64_t> load(size_t(n_bins), 0);
    std::vector<std::vector<int32_t>> bins(static_cast<size_t>(n_bins));
    // min-heap over (load, bin)
    std::vector<std::pair<int64_t, int>> heap;
    for (int b = 0; b < n_bins; ++b) heap.push_back({0, b});
    auto cmp = [](const std::pair<int64_t, int>& a, const std::pair<int64_t, int>& b) { return a > b; };
    std::make_heap(heap.begin(), heap.end(), cmp);
    for (const Item& it : items) {
        std::pop_heap(heap.begin(), heap.end(), cmp);
        std::pair<int64_t, int>& top = heap.back();
        bins[size_t(top.second)].push_back(it.k);
        bins[size_t(top.second)].push_back(it.kp);
        top.first += it.cost;
        std::push_heap(heap.begin(), heap.end(), cmp);
    }
    r.n_bins = n_bins;
    r.bin_ptr.assign(size_t(n_bins) + 1, 0);
    for (int b = 0; b < n_bins; ++b) {
        r.bin_ptr[size_t(b) + 1] = r.bin_ptr[size_t(b)] + int32_t(bins[size_t(b)].size() / 2);
        r.items.insert(r.items.end(), bins[size_t(b)].begin(), bins[size_t(b)].end());
    }
    return r;
}

// Upload minor tables and factor lists once per handle and device.
int upload_tables(const wick_terms* t, cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(t->mu);
    int dev = -1;
    WICK_CUDA(cudaGetDevice(&dev));
    DeviceTables& d = t->dev;
    if (d.blob && d.device == dev) return WICK_OK;
    if (d.blob) { set_error("wick_terms handle was first used on another device"); return WICK_ERR_ARG; }
    BlobBuilder bb;
    size_t o_desc[2], o_jac[2] = {0, 0};
    for (int f = 0; f < 2; ++f) {
        const FlavourTables& ft = t->f[f];
        if (ft.minor_row.size() >= (size_t(1) << 31)) { set_error("more than 2^31 unique minors"); return WICK_ERR_UNSUPPORTED; }
        const std::vector<uint64_t> desc = build_minor_descs(ft);
        o_desc[f] = bb.add(desc.data(), desc.size() * 8);
        if (ft.n >= 8 && ft.n <= 11) {
            const std::vector<uint64_t> jd = build_jacobi_descs(ft);
            o_jac[f] = bb.add(jd.data(), jd.size() * 8);
        }
    }
    size_t o_sp = 0, o_srd = 0, o_sc = 0, o_qp = 0, o_qcu = 0, o_qc = 0;
    size_t o_srdoff = 0, o_rup = 0, o_rul = 0, o_cdp = 0, o_cdl = 0, o_binp = 0, o_items = 0;
    int n_red_bins = 0;
    if (t->outer) {
        const int nru = int(t->f[0].rows.size()), ncd = int(t->f[1].cols.size());
        // sink is sorted by (ru, rd): CSR over ru
        std::vector<int32_t> sp(nru + 1, 0), srd(t->sink.size());
        std::vector<double> sc(2 * t->sink.size());
        for (size_t i = 0; i < t->sink.size(); ++i) {
            sp[t->sink[i].qu + 1]++;
            srd[i] = t->sink[i].qd;
            sc[2 * i] = t->sink[i].c.real(); sc[2 * i + 1] = t->sink[i].c.imag();
        }
        int mx = 0;
        for (int r = 0; r < nru; ++r) { mx = std::max(mx, sp[r + 1]); sp[r + 1] += sp[r]; }
        d.max_sink_per_row = mx;
        // source sorted by (cd, cu): CSR over cd
        std::vector<FactorTerm> src = t->source;
        std::stable_sort(src.begin(), src.end(), [](const FactorTerm& a, const FactorTerm& b) {
            return a.qd != b.qd ? a.qd < b.qd : a.qu < b.qu; });
        std::vector<int32_t> qp(ncd + 1, 0), qcu(src.size());
        std::vector<double> qc(2 * src.size());
        for (size_t j = 0; j < src.size(); ++j) {
            qp[src[j].qd + 1]++;
            qcu[j] = src[j].qu;
            qc[2 * j] = src[j].c.real(); qc[2 * j + 1] = src[j].c.imag();
        }
        for (int c = 0; c < ncd; ++c) qp[c + 1] += qp[c];
        o_sp = bb.add(sp.data(), sp.size() * 4); o_srd = bb.add(srd.data(), srd.size() * 4); o_sc = bb.add(sc.data(), sc.size() * 8);
        o_qp = bb.add(qp.data(), qp.size() * 4); o_qcu = bb.add(qcu.data(), qcu.size() * 4); o_qc = bb.add(qc.data(), qc.size() * 8);
        std::vector<int32_t> srdoff(srd.size());
        for (size_t i = 0; i < srd.size(); ++i) srdoff[i] = srd[i] * ncd;
        const ReduceSchedule rs = build_reduce_schedule(t, sp, qp);
        n_red_bins = rs.n_bins;
        o_srdoff = bb.add(srdoff.data(), srdoff.size() * 4);
        o_rup = bb.add(rs.ru_ptr.data(), rs.ru_ptr.size() * 4); o_rul = bb.add(rs.ru_list.data(), rs.ru_list.size() * 4);
        o_cdp = bb.add(rs.cd_ptr.data(), rs.cd_ptr.size() * 4); o_cdl = bb.add(rs.cd_list.data(), rs.cd_list.size() * 4);
        o_binp = bb.add(rs.bin_ptr.data(), rs.bin_ptr.size() * 4); o_items = bb.add(rs.items.data(), rs.items.size() * 4);
    }
    void* blob = nullptr;
    WICK_CUDA(cudaMalloc(&blob, std::max<size_t>(bb.host.size(), 256)));
    cudaError_t e = cudaMemcpyAsync(blob, bb.host.data(), bb.host.size(), cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);   // bb.host dies at scope exit
    if (e != cudaSuccess) { cudaFree(blob); set_error(std::string("table upload: ") + cudaGetErrorString(e)); return WICK_ERR_CUDA; }
    unsigned char* b = static_cast<unsigned char*>(blob);
    for (int f = 0; f < 2; ++f) {
        d.minor_desc[f] = b + o_desc[f];
        d.jacobi_desc[f] = (t->f[f].n >= 8 && t->f[f].n <= 11) ? b + o_jac[f] : nullptr;
    }
    if (t->outer) {
        d.sink_ptr = reinterpret_cast<const int32_t*>(b + o_sp);
        d.sink_rd = reinterpret_cast<const int32_t*>(b + o_srd);
        d.sink_c = reinterpret_cast<const double*>(b + o_sc);
        d.src_ptr = reinterpret_cast<const int32_t*>(b + o_qp);
        d.src_cu = reinterpret_cast<const int32_t*>(b + o_qcu);
        d.src_c = reinterpret_cast<const double*>(b + o_qc);
        d.sink_rdoff = reinterpret_cast<const int32_t*>(b + o_srdoff);
        d.ru_ptr = reinterpret_cast<const int32_t*>(b + o_rup); d.ru_list = reinterpret_cast<const int32_t*>(b + o_rul);
        d.cd_ptr = reinterpret_cast<const int32_t*>(b + o_cdp); d.cd_list = reinterpret_cast<const int32_t*>(b + o_cdl);
        d.red_bin_ptr = reinterpret_cast<const int32_t*>(b + o_binp);
        d.red_items = reinterpret_cast<const int32_t*>(b + o_items);
        d.n_red_bins = n_red_bins;
    }
    d.blob = blob;
    d.device = dev;
    return WICK_OK;
}

struct StagedHost {
    bool ok = false;                                              // false: a block exceeds the staging capacities
    bool real = false;                                            // all factor coefficients real: dense-B kernel, larger MD block
    std::vector<int32_t> sink_ptr, sink_rdpos, src_ptr, src_cupos, ru_list, rd_list, cu_list, cd_list, bin_ptr;
    std::vector<double> sink_c, src_c;
    std::vector<StagedBatch> batches;
    std::vector<int32_t> md_ids;                                  // per batch: id of MD[rd][cd], rd-major over its block
    std::vector<double> b_dense;                                  // per piece: B[cu][cd], row stride = n_cd rounded up to 2 (real schedules)
};

// Host part of the staged schedule (no CUDA call): also what wick_terms_staged_schedule_check verifies.
StagedHost build_staged_host(const wick_terms* t, int n_bins, bool force_complex) {
    StagedHost h;
    h.real = !force_complex;
    for (const FactorTerm& f : t->sink) if (f.c.imag() != 0.0) h.real = false;
    for (const FactorTerm& f : t->source) if (f.c.imag() != 0.0) h.real = false;
    const int md_cap = stg_md_cap(h.real);
    const int nru = int(t->f[0].rows.size()), nrd = int(t->f[1].rows.size());
    const int ncu = int(t->f[0].cols.size()), ncd = int(t->f[1].cols.size());
    const Components cs = factor_components(nru, nrd, t->sink);
    Components cq = factor_components(ncu, ncd, t->source);
    {   // source blocks relabelled by decreasing number of d columns, so that small blocks are neighbours and can share a piece
        std::vector<int> n_cd_of(size_t(cq.n), 0), order(size_t(cq.n)), relabel(size_t(cq.n));
        for (int c : cq.of_d) if (c >= 0) n_cd_of[size_t(c)]++;
        for (int k = 0; k < cq.n; ++k) order[size_t(k)] = k;
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return n_cd_of[size_t(a)] > n_cd_of[size_t(b)]; });
        for (int k = 0; k < cq.n; ++k) relabel[size_t(order[size_t(k)])] = k;
        for (int& c : cq.of_u) if (c >= 0) c = relabel[size_t(c)];
        for (int& c : cq.of_d) if (c >= 0) c = relabel[size_t(c)];
    }
    auto group = [](const std::vector<int>& comp_of, int n_comp, std::vector<int32_t>& ptr, std::vector<int32_t>& list, std::vector<int32_t>& pos) {
        ptr.assign(size_t(n_comp) + 1, 0);
        for (int c : comp_of) if (c >= 0) ptr[size_t(c) + 1]++;
        for (int c = 0; c < n_comp; ++c) ptr[size_t(c) + 1] += ptr[size_t(c)];
        list.resize(size_t(ptr[size_t(n_comp)]));
        pos.assign(comp_of.size(), -1);
        std::vector<int32_t> next(ptr.begin(), ptr.end() - 1);
        for (size_t x = 0; x < comp_of.size(); ++x)
            if (comp_of[x] >= 0) { pos[x] = next[size_t(comp_of[x])]++; list[size_t(pos[x])] = int32_t(x); }
    };
    std::vector<int32_t> ru_ptr, ru_list, ru_pos, rd_ptr, rd_list, rd_pos, cu_ptr, cu_list, cu_pos, cd_ptr, cd_list, cd_pos;
    group(cs.of_u, cs.n, ru_ptr, ru_list, ru_pos);
    group(cs.of_d, cs.n, rd_ptr, rd_list, rd_pos);
    group(cq.of_u, cq.n, cu_ptr, cu_list, cu_pos);
    group(cq.of_d, cq.n, cd_ptr, cd_list, cd_pos);
    int max_rd = 1, max_cu = 1;
    for (int k = 0; k < cs.n; ++k) max_rd = std::max(max_rd, rd_ptr[size_t(k) + 1] - rd_ptr[size_t(k)]);
    for (int k = 0; k < cq.n; ++k) max_cu = std::max(max_cu, cu_ptr[size_t(k) + 1] - cu_ptr[size_t(k)]);
    if (max_rd > md_cap || max_cu > STG_ROW_CAP || cs.n == 0 || cq.n == 0) return h;

    // coefficient lists regrouped by list position, so that a batch's entries are contiguous:
    // sink entries by position of ru in ru_list, source entries by position of cd in cd_list
    std::vector<int32_t> sink_ptr(size_t(nru) + 1, 0), src_ptr(size_t(ncd) + 1, 0);
    for (const FactorTerm& f : t->sink) sink_ptr[size_t(ru_pos[size_t(f.qu)]) + 1]++;
    for (const FactorTerm& f : t->source) src_ptr[size_t(cd_pos[size_t(f.qd)]) + 1]++;
    for (int r = 0; r < nru; ++r) sink_ptr[size_t(r) + 1] += sink_ptr[size_t(r)];
    for (int c = 0; c < ncd; ++c) src_ptr[size_t(c) + 1] += src_ptr[size_t(c)];
    std::vector<int32_t> sink_rdpos(t->sink.size()), src_cupos(t->source.size());
    std::vector<double> sink_c(2 * t->sink.size()), src_c(2 * t->source.size());
    {
        std::vector<int32_t> next(sink_ptr.begin(), sink_ptr.end() - 1);
        for (const FactorTerm& f : t->sink) {                  // t->sink is sorted by (ru, rd): order within a row is kept
            const size_t e = size_t(next[size_t(ru_pos[size_t(f.qu)])]++);
            sink_rdpos[e] = rd_pos[size_t(f.qd)]; sink_c[2 * e] = f.c.real(); sink_c[2 * e + 1] = f.c.imag();
        }
        std::vector<FactorTerm> src = t->source;
        std::stable_sort(src.begin(), src.end(), [](const FactorTerm& a, const FactorTerm& b) {
            return a.qd != b.qd ? a.qd < b.qd : a.qu < b.qu; });
        std::vector<int32_t> nextq(src_ptr.begin(), src_ptr.end() - 1);
        for (const FactorTerm& f : src) {
            const size_t e = size_t(nextq[size_t(cd_pos[size_t(f.qd)])]++);
            src_cupos[e] = cu_pos[size_t(f.qu)]; src_c[2 * e] = f.c.real(); src_c[2 * e + 1] = f.c.imag();
        }
    }
    // a single u-row tuple or a single d column must fit the entry buffers
    for (int r = 0; r < nru; ++r) if (sink_ptr[size_t(r) + 1] - sink_ptr[size_t(r)] > STG_SINK_CAP) return h;
    for (int c = 0; c < ncd; ++c) if (src_ptr[size_t(c) + 1] - src_ptr[size_t(c)] > STG_SRC_CAP) return h;
    for (int k = 0; k < cs.n; ++k)                              // one sink block must fit a batch on its own
        if (ru_ptr[size_t(k) + 1] - ru_ptr[size_t(k)] > STG_ROWS_CAP ||
            sink_ptr[size_t(ru_ptr[size_t(k) + 1])] - sink_ptr[size_t(ru_ptr[size_t(k)])] > STG_SINK_CAP) return h;

    struct Item { int64_t cost; StagedBatch b; };
    std::vector<Item> items;
    // pieces of the d-column list: a large source block is cut into equal pieces small enough for the largest
    // sink block; neighbouring small blocks share a piece (their union is just a block-diagonal source block)
    struct Piece { int ca, cb, cuA, cuB; };
    std::vector<Piece> pieces;
    const int piece_max = std::max(1, std::min(STG_NCD_CAP, md_cap / max_rd));
    for (int kp = 0; kp < cq.n;) {
        const int cdA = cd_ptr[size_t(kp)], cdB = cd_ptr[size_t(kp) + 1];
        const int cuA = cu_ptr[size_t(kp)];
        if (cdB - cdA >= piece_max) {
            const int n_pieces = (cdB - cdA + piece_max - 1) / piece_max;
            const int piece = (cdB - cdA + n_pieces - 1) / n_pieces;
            for (int ca = cdA; ca < cdB;) {
                int cb = std::min(cdB, ca + piece);
                while (cb > ca + 1 && src_ptr[size_t(cb)] - src_ptr[size_t(ca)] > STG_SRC_CAP) --cb;
                pieces.push_back({ca, cb, cuA, cu_ptr[size_t(kp) + 1]});
                ca = cb;
            }
            ++kp;
        } else {
            int ke = kp + 1;
            while (ke < cq.n && cd_ptr[size_t(ke) + 1] - cdA <= piece_max && cu_ptr[size_t(ke) + 1] - cuA <= STG_ROW_CAP &&
                   src_ptr[size_t(cd_ptr[size_t(ke) + 1])] - src_ptr[size_t(cdA)] <= STG_SRC_CAP) ++ke;
            pieces.push_back({cdA, cd_ptr[size_t(ke)], cuA, cu_ptr[size_t(ke)]});
            kp = ke;
        }
    }
    for (const Piece& pc : pieces) {
        {
            const int ca = pc.ca, cb = pc.cb, cuA = pc.cuA, cuB = pc.cuB;
            const int n_cd = cb - ca;
            const int64_t src_work = (src_ptr[size_t(cb)] - src_ptr[size_t(ca)]) + n_cd;
            int ka = 0;
            while (ka < cs.n) {
                int kb = ka, n_rd = 0;
                while (kb < cs.n) {
                    const int n_rd2 = n_rd + rd_ptr[size_t(kb) + 1] - rd_ptr[size_t(kb)];
                    const int rows2 = ru_ptr[size_t(kb) + 1] - ru_ptr[size_t(ka)];
                    const int ent2 = sink_ptr[size_t(ru_ptr[size_t(kb) + 1])] - sink_ptr[size_t(ru_ptr[size_t(ka)])];
                    if (kb > ka && (n_rd2 * n_cd > md_cap || rows2 > STG_ROWS_CAP || ent2 > STG_SINK_CAP)) break;
                    n_rd = n_rd2;
                    ++kb;
                }
                Item it;
                it.b = StagedBatch{ca, cb, cuA, cuB, rd_ptr[size_t(ka)], rd_ptr[size_t(kb)], ru_ptr[size_t(ka)], ru_ptr[size_t(kb)], 0, 0, 0, 0};
                const int rows = ru_ptr[size_t(kb)] - ru_ptr[size_t(ka)];
                const int ent = sink_ptr[size_t(ru_ptr[size_t(kb)])] - sink_ptr[size_t(ru_ptr[size_t(ka)])];
                it.cost = int64_t(n_rd) * n_cd + 16 + int64_t(rows) * ((cuB - cuA) + src_work + 4) + int64_t(ent) * n_cd;
                items.push_back(it);
                ka = kb;
            }
        }
    }
    std::stable_sort(items.begin(), items.end(), [](const Item& a, const Item& b) { return a.cost > b.cost; });
    std::vector<std::vector<StagedBatch>> bins(static_cast<size_t>(n_bins));
    std::vector<std::pair<int64_t, int>> heap;
    for (int b = 0; b < n_bins; ++b) heap.push_back({0, b});
    auto cmp = [](const std::pair<int64_t, int>& a, const std::pair<int64_t, int>& b) { return a > b; };
    std::make_heap(heap.begin(), heap.end(), cmp);
    for (const Item& it : items) {
        std::pop_heap(heap.begin(), heap.end(), cmp);
        bins[size_t(heap.back().second)].push_back(it.b);
        heap.back().first += it.cost;
        std::push_heap(heap.begin(), heap.end(), cmp);
    }
    std::vector<int32_t> bin_ptr(size_t(n_bins) + 1, 0);
    std::vector<StagedBatch> batches;
    for (int b = 0; b < n_bins; ++b) {
        batches.insert(batches.end(), bins[size_t(b)].begin(), bins[size_t(b)].end());
        bin_ptr[size_t(b) + 1] = int32_t(batches.size());
    }
    // flattened prologue data: MD element ids per batch, dense B per piece (shared by the batches of the piece)
    {
        std::map<std::pair<int, int>, int32_t> piece_off;           // (cd_a, cu_a) identifies a piece
        for (StagedBatch& b : batches) {
            b.sink_a = sink_ptr[size_t(b.ru_a)];                     // the batch's sink entries: no look-up of the range in the kernel
            b.sink_n = sink_ptr[size_t(b.ru_b)] - b.sink_a;
            b.md_off = int32_t(h.md_ids.size());
            for (int rdi = b.rd_a; rdi < b.rd_b; ++rdi)
                for (int cdi = b.cd_a; cdi < b.cd_b; ++cdi)
                    h.md_ids.push_back(rd_list[size_t(rdi)] * ncd + cd_list[size_t(cdi)]);
            b.b_off = 0;
            if (h.real) {
                auto it = piece_off.find({b.cd_a, b.cu_a});
                if (it == piece_off.end()) {
                    const int n_cd = b.cd_b - b.cd_a, n_cu = b.cu_b - b.cu_a, ncdp = (n_cd + 1) & ~1;
                    const int32_t off = int32_t(h.b_dense.size());
                    h.b_dense.resize(h.b_dense.size() + size_t(n_cu) * size_t(ncdp), 0.0);
                    for (int cdi = 0; cdi < n_cd; ++cdi)
                        for (int j = src_ptr[size_t(b.cd_a + cdi)]; j < src_ptr[size_t(b.cd_a + cdi) + 1]; ++j)
                            h.b_dense[size_t(off) + size_t(src_cupos[size_t(j)] - b.cu_a) * size_t(ncdp) + size_t(cdi)] += src_c[2 * size_t(j)];
                    it = piece_off.emplace(std::make_pair(b.cd_a, b.cu_a), off).first;
                }
                b.b_off = it->second;
            }
        }
        if (h.b_dense.empty()) h.b_dense.push_back(0.0);
        h.md_ids.resize(h.md_ids.size() + 32 * STG_THREADS / 32, 0);  // the kernel requests the next batch's ids one batch ahead, unguarded
    }
    h.ok = true;
    h.sink_ptr = std::move(sink_ptr); h.sink_rdpos = std::move(sink_rdpos); h.src_ptr = std::move(src_ptr); h.src_cupos = std::move(src_cupos);
    h.ru_list = std::move(ru_list); h.rd_list = std::move(rd_list); h.cu_list = std::move(cu_list); h.cd_list = std::move(cd_list);
    h.bin_ptr = std::move(bin_ptr); h.sink_c = std::move(sink_c); h.src_c = std::move(src_c); h.batches = std::move(batches);
    return h;
}

// ---- staged factorised reduction: host schedule (kernels.cu: reduce_staged_kernel) --------------
// Tuples grouped by block: ru_list / rd_list by sink block, cu_list / cd_list by source block.
// Batches = (source block k', d-column piece) x (run of sink blocks) with at most STG_MD_CAP MD elements;
// batches are assigned to n_bins CTAs by longest-processing-time, each bin keeps a fixed order.
// Returns 1 and fills `out` when the list is eligible, 0 when a block is too large (caller falls back
// to reduce_outer_kernel), negative on error.
int ensure_staged(const wick_terms* t, int n_bins, bool force_complex, cudaStream_t stream, StagedTables* out) {
    std::lock_guard<std::mutex> lock(t->mu);
    DeviceTables& d = t->dev;
    if (d.staged_state < 0) return 0;
    const int nru = int(t->f[0].rows.size()), nrd = int(t->f[1].rows.size());
    const int ncu = int(t->f[0].cols.size()), ncd = int(t->f[1].cols.size());
    auto fill = [&](const StagedDev& sd) {
        out->n_cols_u = ncu; out->n_cols_d = ncd; out->n_bins = sd.n_bins;
        out->real_coeffs = sd.real;
        out->sink_ptr = sd.sink_ptr; out->sink_rdpos = sd.sink_rdpos; out->sink_c = reinterpret_cast<const double2*>(sd.sink_c);
        out->src_ptr = sd.src_ptr; out->src_cupos = sd.src_cupos; out->src_c = reinterpret_cast<const double2*>(sd.src_c);
        out->ru_list = sd.ru_list; out->rd_list = sd.rd_list; out->cu_list = sd.cu_list; out->cd_list = sd.cd_list;
        out->bin_ptr = sd.bin_ptr; out->batches = static_cast<const StagedBatch*>(sd.batches);
        out->md_ids = sd.md_ids; out->b_dense = sd.b_dense;
    };
    const int key = 2 * n_bins + (force_complex ? 1 : 0);          // schedules differ: the real-coefficient kernel stages larger MD blocks
    auto hit = d.staged.find(key);
    if (hit != d.staged.end()) { fill(hit->second); return 1; }

    const StagedHost h = build_staged_host(t, n_bins, force_complex);
    if (!h.ok) { d.staged_state = -1; return 0; }
    d.staged_state = 1;
    const std::vector<int32_t>&sink_rdpos = h.sink_rdpos, &src_cupos = h.src_cupos, &sink_ptr = h.sink_ptr, &src_ptr = h.src_ptr;
    const std::vector<int32_t>&ru_list = h.ru_list, &rd_list = h.rd_list, &cu_list = h.cu_list, &cd_list = h.cd_list, &bin_ptr = h.bin_ptr;
    const std::vector<double>&sink_c = h.sink_c, &src_c = h.src_c;
    const std::vector<StagedBatch>& batches = h.batches;
    BlobBuilder bb;
    const size_t o_srp = bb.add(sink_rdpos.data(), sink_rdpos.size() * 4), o_scp = bb.add(src_cupos.data(), src_cupos.size() * 4);
    const size_t o_sp = bb.add(sink_ptr.data(), sink_ptr.size() * 4), o_qp = bb.add(src_ptr.data(), src_ptr.size() * 4);
    const size_t o_sc = bb.add(sink_c.data(), sink_c.size() * 8), o_qc = bb.add(src_c.data(), src_c.size() * 8);
    const size_t o_ru = bb.add(ru_list.data(), ru_list.size() * 4), o_rd = bb.add(rd_list.data(), rd_list.size() * 4);
    const size_t o_cu = bb.add(cu_list.data(), cu_list.size() * 4), o_cd = bb.add(cd_list.data(), cd_list.size() * 4);
    const size_t o_bp = bb.add(bin_ptr.data(), bin_ptr.size() * 4), o_ba = bb.add(batches.data(), batches.size() * sizeof(StagedBatch));
    const size_t o_mi = bb.add(h.md_ids.data(), h.md_ids.size() * 4), o_bd = bb.add(h.b_dense.data(), h.b_dense.size() * 8);
    void* blob = nullptr;
    WICK_CUDA(cudaMalloc(&blob, std::max<size_t>(bb.host.size(), 256)));
    cudaError_t e = cudaMemcpyAsync(blob, bb.host.data(), bb.host.size(), cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);   // bb.host dies at scope exit
    if (e != cudaSuccess) { cudaFree(blob); set_error(std::string("staged schedule upload: ") + cudaGetErrorString(e)); return WICK_ERR_CUDA; }
    unsigned char* b = static_cast<unsigned char*>(blob);
    StagedDev sd;
    sd.blob = blob; sd.n_bins = n_bins; sd.real = h.real;
    sd.sink_rdpos = reinterpret_cast<const int32_t*>(b + o_srp); sd.src_cupos = reinterpret_cast<const int32_t*>(b + o_scp);
    sd.sink_ptr = reinterpret_cast<const int32_t*>(b + o_sp); sd.src_ptr = reinterpret_cast<const int32_t*>(b + o_qp);
    sd.sink_c = reinterpret_cast<const double*>(b + o_sc); sd.src_c = reinterpret_cast<const double*>(b + o_qc);
    sd.ru_list = reinterpret_cast<const int32_t*>(b + o_ru); sd.rd_list = reinterpret_cast<const int32_t*>(b + o_rd);
    sd.cu_list = reinterpret_cast<const int32_t*>(b + o_cu); sd.cd_list = reinterpret_cast<const int32_t*>(b + o_cd);
    sd.bin_ptr = reinterpret_cast<const int32_t*>(b + o_bp); sd.batches = b + o_ba;
    sd.md_ids = reinterpret_cast<const int32_t*>(b + o_mi); sd.b_dense = reinterpret_cast<const double*>(b + o_bd);
    d.staged[key] = sd;
    fill(sd);
    return 1;
}

// ---- register-resident minors kernel: host schedule (minors_reg.cu) -----------------------------
// Grid tables only (minor (r, c) = r * n_cols + c, column tuples sorted lexicographically).  Column tuples are
// grouped by their K = n-4 leading columns (an "instance"); the candidate columns of an instance are the indices
// that occur behind the leading ones, and every column tuple of the instance is a 4-subset of candidate
// positions.  Because the tuples are sorted, the minors of an instance are contiguous in a row tuple's list and
// appear in the rank order of their 4-subsets.
struct RegHost {
    bool ok = false;
    int n = 0;
    std::vector<RegJob> jobs;
    std::vector<uint32_t> prog;                                     // trie programs of the jobs (kernels.cuh: RegTables::prog)
    std::vector<double> cost;                                       // per job, in flops (LPT weights)
    std::vector<uint32_t> rows;                                     // row tuples as 4-bit fields
};

RegHost build_reg_host(const FlavourTables& ft, bool grid) {
    RegHost h;
    h.n = ft.n;
    const int n = ft.n, K = n - 4;
    if (!grid || n < 5 || ft.cols.empty() || ft.rows.empty() || ft.rows.size() >= (size_t(1) << 24)) return h;
    const size_t nc = ft.cols.size();
    if (ft.minor_row.size() != ft.rows.size() * nc) return h;
    const uint64_t lead_bits = (uint64_t(1) << (4 * K)) - 1;
    int max_cand = 0;
    for (size_t c0 = 0; c0 < nc;) {
        const uint64_t lead = nibbles_of_mask(ft.cols[c0]) & lead_bits;
        uint16_t lead_mask = 0;
        for (int i = 0; i < K; ++i) lead_mask |= uint16_t(1u << ((lead >> (4 * i)) & 15u));
        size_t c1 = c0;
        uint16_t cand_mask = 0;
        while (c1 < nc && (nibbles_of_mask(ft.cols[c1]) & lead_bits) == lead) { cand_mask |= uint16_t(ft.cols[c1] & ~lead_mask); ++c1; }
        RegJob j;
        std::memset(&j, 0, sizeof(j));
        j.lead = lead;
        j.cand = nibbles_of_mask(cand_mask);
        j.ncand = uint32_t(__builtin_popcount(cand_mask));
        max_cand = std::max(max_cand, int(j.ncand));
        if (int(j.ncand) > REG_NC_MAX) return h;
        j.out_base = uint32_t(c0);
        j.prog_begin = uint32_t(h.prog.size());
        int pos_of[12];
        { int k = 0; for (int b = 0; b < 12; ++b) pos_of[b] = (cand_mask & (1u << b)) ? k++ : -1; }
        // the tuples are sorted, so consecutive tuples with equal (i2, i3) form a pair node and with equal (i2, i3, i4) a third node;
        // one word per THIRD node: i4 | mask(i5) << 4 | i2 << 14 | i3 << 18 | (first third node of its pair) << 22
        int n_pairs = 0, n_thirds = 0;
        int p2 = -1, p3 = -1, p4 = -1;
        for (size_t c = c0; c < c1; ++c) {
            const uint64_t w = nibbles_of_mask(ft.cols[c]) >> (4 * K);
            int x[4];
            for (int i = 0; i < 4; ++i) x[i] = pos_of[(w >> (4 * i)) & 15u];
            const bool new_pair = (x[0] != p2 || x[1] != p3);
            if (new_pair) { p2 = x[0]; p3 = x[1]; p4 = -1; ++n_pairs; }
            if (x[2] != p4) {
                h.prog.push_back(uint32_t(x[2]) | (uint32_t(x[0]) << 14) | (uint32_t(x[1]) << 18) | (new_pair ? 1u << 22 : 0u));
                p4 = x[2]; ++n_thirds;
            }
            h.prog.back() |= 1u << (4 + x[3]);
        }
        j.prog_end = uint32_t(h.prog.size());
        h.jobs.push_back(j);
        // pivot steps + one Schur column per candidate + the trie levels (flops) + per-node overhead
        h.cost.push_back(150.0 * K + 8.0 * K * (2 * n - K - 1) / 2 * j.ncand + 110.0 * n_pairs + 120.0 * n_thirds + 36.0 * double(c1 - c0) + 200.0);
        c0 = c1;
    }
    if (h.jobs.size() > 256 || !minors_reg_supported(n, max_cand)) { h.jobs.clear(); return h; }
    h.prog.push_back(0); h.prog.push_back(0);                       // the kernel reads two words ahead
    h.rows.resize(ft.rows.size());
    for (size_t r = 0; r < ft.rows.size(); ++r) h.rows[r] = uint32_t(nibbles_of_mask(ft.rows[r]));
    h.ok = true;
    return h;
}

// Returns 1 and fills `out` when flavour f's minors can go through the register-resident kernel, 0 when not.
int ensure_reg(const wick_terms* t, int f, int n_bins, cudaStream_t stream, RegTables* out) {
    std::lock_guard<std::mutex> lock(t->mu);
    DeviceTables& d = t->dev;
    if (d.reg_state[f] < 0) return 0;
    auto fill = [&](const RegDev& rd) {
        out->n_cols = int(t->f[f].cols.size()); out->n_bins = rd.n_bins;
        out->jobs = static_cast<const RegJob*>(rd.jobs); out->prog = static_cast<const uint32_t*>(rd.prog); out->row_nibbles = static_cast<const uint32_t*>(rd.rows);
        out->bin_ptr = static_cast<const uint32_t*>(rd.bin_ptr); out->bin_jobs = static_cast<const uint32_t*>(rd.bin_jobs);
    };
    auto hit = d.reg[f].find(n_bins);
    if (hit != d.reg[f].end()) { fill(hit->second); return 1; }
    const RegHost h = build_reg_host(t->f[f], t->outer);
    if (!h.ok) { d.reg_state[f] = -1; return 0; }
    d.reg_state[f] = 1;
    // longest-processing-time assignment of (row tuple, job) pairs to the warp bins; fixed order
    const size_t nr = h.rows.size(), nq = h.jobs.size();
    std::vector<uint32_t> order(nq);
    for (size_t q = 0; q < nq; ++q) order[q] = uint32_t(q);
    std::stable_sort(order.begin(), order.end(), [&](uint32_t a, uint32_t b) { return h.cost[a] > h.cost[b]; });
    std::vector<std::vector<uint32_t>> bins(static_cast<size_t>(n_bins));
    std::vector<std::pair<double, int>> heap;
    for (int b = 0; b < n_bins; ++b) heap.push_back({0.0, b});
    auto cmp = [](const std::pair<double, int>& a, const std::pair<double, int>& b) { return a > b; };
    std::make_heap(heap.begin(), heap.end(), cmp);
    for (uint32_t q : order)
        for (size_t r = 0; r < nr; ++r) {
            std::pop_heap(heap.begin(), heap.end(), cmp);
            bins[size_t(heap.back().second)].push_back((uint32_t(r) << 8) | q);
            heap.back().first += h.cost[q];
            std::push_heap(heap.begin(), heap.end(), cmp);
        }
    std::vector<uint32_t> bin_ptr(size_t(n_bins) + 1, 0), bin_jobs;
    bin_jobs.reserve(nr * nq);
    for (int b = 0; b < n_bins; ++b) {
        bin_jobs.insert(bin_jobs.end(), bins[size_t(b)].begin(), bins[size_t(b)].end());
        bin_ptr[size_t(b) + 1] = uint32_t(bin_jobs.size());
    }
    BlobBuilder bb;
    const size_t o_j = bb.add(h.jobs.data(), h.jobs.size() * sizeof(RegJob)), o_r = bb.add(h.rows.data(), h.rows.size() * 4);
    const size_t o_p = bb.add(h.prog.data(), h.prog.size() * 4);
    const size_t o_bp = bb.add(bin_ptr.data(), bin_ptr.size() * 4), o_bj = bb.add(bin_jobs.data(), bin_jobs.size() * 4);
    void* blob = nullptr;
    WICK_CUDA(cudaMalloc(&blob, std::max<size_t>(bb.host.size(), 256)));
    cudaError_t e = cudaMemcpyAsync(blob, bb.host.data(), bb.host.size(), cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) { cudaFree(blob); set_error(std::string("minor job schedule upload: ") + cudaGetErrorString(e)); return WICK_ERR_CUDA; }
    unsigned char* b = static_cast<unsigned char*>(blob);
    RegDev rd;
    rd.blob = blob; rd.n_bins = n_bins;
    rd.jobs = b + o_j; rd.prog = b + o_p; rd.rows = b + o_r; rd.bin_ptr = b + o_bp; rd.bin_jobs = b + o_bj;
    d.reg[f][n_bins] = rd;
    fill(rd);
    return 1;
}

int upload_flat(const wick_terms* t, cudaStream_t stream) {
    try { t->ensure_flat(); } catch (const std::bad_alloc&) { set_error("flat term list: out of host memory"); return WICK_ERR_NOMEM; }
    std::lock_guard<std::mutex> lock(t->mu);
    DeviceTables& d = t->dev;
    if (d.flat_blob) return WICK_OK;
    const size_t n = size_t(t->n_terms);
    const size_t o_uid = 0, o_did = align_up(n * 4, 256), o_w = o_did + align_up(n * 4, 256);
    const size_t bytes = o_w + n * 16;
    void* blob = nullptr;
    WICK_CUDA(cudaMalloc(&blob, std::max<size_t>(bytes, 256)));
    unsigned char* b = static_cast<unsigned char*>(blob);
    cudaError_t e = cudaSuccess;
    if (n) {
        e = cudaMemcpyAsync(b + o_uid, t->t_uid.data(), n * 4, cudaMemcpyHostToDevice, stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(b + o_did, t->t_did.data(), n * 4, cudaMemcpyHostToDevice, stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(b + o_w, t->t_w.data(), n * 16, cudaMemcpyHostToDevice, stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    }
    if (e != cudaSuccess) { cudaFree(blob); set_error(std::string("flat list upload: ") + cudaGetErrorString(e)); return WICK_ERR_CUDA; }
    d.flat_blob = blob;
    d.t_uid = reinterpret_cast<const int32_t*>(b + o_uid);
    d.t_did = reinterpret_cast<const int32_t*>(b + o_did);
    d.t_w = reinterpret_cast<const double*>(b + o_w);
    return WICK_OK;
}

// ---- workspace plan --------------------------------------------------------------------------
constexpr int MAX_CHUNKS = 256;                  // rows of the partial buffer
constexpr size_t TARGET_MINOR_BYTES = size_t(2) << 30;
constexpr int64_t JACOBI_BYTES_PER_ST = (144 + 1) * 16;   // inverse propagator + determinant of one flavour

struct Plan {
    int64_t n_st = 0;                            // site-times T * L^3
    int64_t per_st = 0;                          // bytes of minors + partials per site-time
    size_t sigma_bytes = 0;
    int64_t S_b = 0;                             // site-times per batch (multiple of 32)
};

bool make_plan(const wick_terms* t, int n_lists, int L, int T, int n_mom, size_t workspace_bytes, bool want_max, Plan* p) {
    if (!t || n_lists < 1 || L < 1 || T < 1 || n_mom < 0 || int64_t(L) * L * L > (int64_t(1) << 31) - 1) return false;
    p->n_st = int64_t(T) * L * L * L;
    const int64_t nm = int64_t(t->f[0].minor_row.size()) + int64_t(t->f[1].minor_row.size());
    p->per_st = (nm + MAX_CHUNKS) * 16 + 2 * JACOBI_BYTES_PER_ST;   // the Jacobi buffers are always planned for, so one size serves every flag
    p->sigma_bytes = align_up(size_t(n_lists) * size_t(p->n_st) * 16, 256);
    const int64_t n_st_pad = (p->n_st + GROUP - 1) / GROUP * GROUP;
    int64_t sb;
    if (want_max) {
        sb = int64_t(TARGET_MINOR_BYTES / size_t(p->per_st)) / GROUP * GROUP;
    } else {
        if (workspace_bytes < p->sigma_bytes + 1024) { p->S_b = 0; return true; }
        sb = int64_t((workspace_bytes - p->sigma_bytes - 1024) / size_t(p->per_st)) / GROUP * GROUP;
    }
    sb = std::min<int64_t>(sb, n_st_pad);
    sb = std::min<int64_t>(sb, int64_t(1) << 22);             // keeps grid.x and 32-bit site offsets small
    if (want_max) sb = std::max<int64_t>(sb, GROUP);
    // the staged reduction runs n_groups x floor(148 / n_groups) CTAs (or n_groups when >= 148), one per SM:
    // shrink the batch until that grid fills at least 90 % of its last wave
    auto wave_fill = [](int64_t g) {
        if (g < 148) return double(g * (148 / g)) / 148.0;
        return double(g) / double((g + 147) / 148 * 148);
    };
    int64_t g = sb / GROUP;
    while (g > 1 && wave_fill(g) < 0.9) --g;
    sb = g * GROUP;
    p->S_b = sb;
    return true;
}

size_t plan_bytes(const Plan& p, int64_t S_b) { return p.sigma_bytes + 1024 + size_t(S_b) * size_t(p.per_st); }

}  // namespace

extern "C" void wick_terms_release_device(DeviceTables* d) {
    if (d->blob) cudaFree(d->blob);
    if (d->flat_blob) cudaFree(d->flat_blob);
    if (d->jf_blob) cudaFree(d->jf_blob);
    if (d->block_blob) cudaFree(d->block_blob);
    for (auto& kv : d->staged) cudaFree(kv.second.blob);
    for (int f = 0; f < 2; ++f) for (auto& kv : d->reg[f]) cudaFree(kv.second.blob);
    *d = DeviceTables();
}

extern "C" int wick_terms_export_minor_order(const wick_terms* t, int flavour, int32_t* minor_id, uint8_t* proc_cols, uint8_t* negate) {
    if (!t || (flavour != 0 && flavour != 1)) { set_error("wick_terms_export_minor_order: bad argument"); return WICK_ERR_ARG; }
    const FlavourTables& ft = t->f[flavour];
    MinorOrder o;
    try { o = build_minor_order(ft); } catch (const std::bad_alloc&) { set_error("out of host memory"); return WICK_ERR_NOMEM; }
    for (size_t k = 0; k < o.minor.size(); ++k) {
        if (minor_id) minor_id[k] = int32_t(o.minor[k]);
        if (negate) negate[k] = o.negate[k];
        if (proc_cols) for (int i = 0; i < ft.n; ++i) proc_cols[k * size_t(ft.n) + size_t(i)] = uint8_t((o.cols[k] >> (4 * i)) & 15u);
    }
    return WICK_OK;
}

extern "C" int wick_terms_staged_schedule_check(const wick_terms* t, int n_bins, int64_t* n_batches_out, int64_t* n_pairs_out,
                                               int64_t* max_md_elements_out, int64_t* max_rows_out) {
    if (!t || n_bins < 1) { set_error("wick_terms_staged_schedule_check: bad argument"); return WICK_ERR_ARG; }
    if (!t->outer) { set_error("not an outer-product term list"); return WICK_ERR_UNSUPPORTED; }
    StagedHost h;
    try { h = build_staged_host(t, n_bins, false); } catch (const std::bad_alloc&) { set_error("out of host memory"); return WICK_ERR_NOMEM; }
    if (!h.ok) { set_error("a block of the factor lists exceeds the staging capacities (the unstaged kernel is used)"); return WICK_ERR_UNSUPPORTED; }
    const size_t nru = t->f[0].rows.size(), ncd = t->f[1].cols.size();
    std::vector<uint8_t> covered(nru * ncd, 0);
    int64_t max_md = 0, max_rows = 0;
    auto fail = [](const char* what) { set_error(std::string("staged schedule: ") + what); return WICK_ERR_ARG; };
    if (h.bin_ptr.size() != size_t(n_bins) + 1 || h.bin_ptr.front() != 0 || size_t(h.bin_ptr.back()) != h.batches.size())
        return fail("bins do not cover the batch list");
    for (const StagedBatch& b : h.batches) {
        const int n_cd = b.cd_b - b.cd_a, n_cu = b.cu_b - b.cu_a, n_rd = b.rd_b - b.rd_a, rows = b.ru_b - b.ru_a;
        if (n_cd < 1 || n_cd > STG_NCD_CAP || n_cu < 1 || n_cu > STG_ROW_CAP || rows < 1 || rows > STG_ROWS_CAP ||
            int64_t(n_rd) * n_cd > stg_md_cap(h.real)) return fail("a batch exceeds a capacity");
        if (h.sink_ptr[size_t(b.ru_b)] - h.sink_ptr[size_t(b.ru_a)] > STG_SINK_CAP ||
            h.src_ptr[size_t(b.cd_b)] - h.src_ptr[size_t(b.cd_a)] > STG_SRC_CAP) return fail("a batch exceeds an entry buffer");
        max_md = std::max<int64_t>(max_md, int64_t(n_rd) * n_cd);
        max_rows = std::max<int64_t>(max_rows, rows);
        for (int r = b.ru_a; r < b.ru_b; ++r) {
            for (int i = h.sink_ptr[size_t(r)]; i < h.sink_ptr[size_t(r) + 1]; ++i)
                if (h.sink_rdpos[size_t(i)] < b.rd_a || h.sink_rdpos[size_t(i)] >= b.rd_b) return fail("a sink entry points outside the staged MD block");
            for (int c = b.cd_a; c < b.cd_b; ++c) {
                uint8_t& cell = covered[size_t(r) * ncd + size_t(c)];
                if (cell) return fail("a (u-row tuple, d-column tuple) pair is covered twice");
                cell = 1;
            }
        }
        for (int c = b.cd_a; c < b.cd_b; ++c)
            for (int j = h.src_ptr[size_t(c)]; j < h.src_ptr[size_t(c) + 1]; ++j)
                if (h.src_cupos[size_t(j)] < b.cu_a || h.src_cupos[size_t(j)] >= b.cu_b) return fail("a source entry points outside the staged MU row");
    }
    int64_t n_pairs = 0;
    for (uint8_t c : covered) n_pairs += c;
    if (n_pairs != int64_t(nru) * int64_t(ncd)) return fail("a (u-row tuple, d-column tuple) pair is not covered");
    if (n_batches_out) *n_batches_out = int64_t(h.batches.size());
    if (n_pairs_out) *n_pairs_out = n_pairs;
    if (max_md_elements_out) *max_md_elements_out = max_md;
    if (max_rows_out) *max_rows_out = max_rows;
    return WICK_OK;
}

extern "C" int64_t wick_launch_count(void) { return launch_counter_get(); }
extern "C" int64_t wick_launch_count_reset(void) { return launch_counter_reset(); }

extern "C" int wick_profile_enable(int on) { profile_enable(on != 0); return WICK_OK; }

extern "C" int wick_profile_read(wick_profile* out) {
    if (!out) { set_error("wick_profile_read: NULL argument"); return WICK_ERR_ARG; }
    WICK_CUDA(profile_read(out->ms, out->launches));
    return WICK_OK;
}

extern "C" int wick_measure_fp64_peak(double* tflops_out, void* cuda_stream) {
    if (!tflops_out) { set_error("wick_measure_fp64_peak: NULL argument"); return WICK_ERR_ARG; }
    WICK_CUDA(measure_fp64_peak(tflops_out, static_cast<cudaStream_t>(cuda_stream)));
    return WICK_OK;
}

extern "C" size_t wick_contract_min_workspace_bytes(const wick_terms* t, int L, int T, int n_mom) {
    Plan p;
    if (!make_plan(t, 1, L, T, n_mom, 0, true, &p)) return 0;
    return plan_bytes(p, GROUP);
}

extern "C" size_t wick_contract_workspace_bytes(const wick_terms* t, int L, int T, int n_mom) {
    Plan p;
    if (!make_plan(t, 1, L, T, n_mom, 0, true, &p)) return 0;
    return plan_bytes(p, p.S_b);
}

namespace {

// The hot path for n_lists term lists over ONE pair of unique-minor tables (lists[0]'s): per site batch the minors are
// evaluated once, then every list runs its own weighted-product kernel into its own sigma; n_lists = 1 is wick_contract.
int contract_lists(const void* U_dev, const void* D_dev, const wick_terms* const* lists, int n_lists, const int32_t* momenta,
                   int n_mom, int L, int T, void* C_out_dev, void* sigma_out_dev, void* workspace_dev,
                   size_t workspace_bytes, unsigned flags, void* cuda_stream, const char* who) {
    auto fail = [&](const char* msg, int code) { set_error(std::string(who) + ": " + msg); return code; };
    if (!U_dev || !D_dev || !lists || n_lists < 1 || !C_out_dev || !workspace_dev || (n_mom > 0 && !momenta)) return fail("NULL argument", WICK_ERR_ARG);
    for (int k = 0; k < n_lists; ++k) if (!lists[k]) return fail("NULL argument", WICK_ERR_ARG);
    if ((reinterpret_cast<uintptr_t>(U_dev) | reinterpret_cast<uintptr_t>(D_dev) | reinterpret_cast<uintptr_t>(C_out_dev) |
         reinterpret_cast<uintptr_t>(sigma_out_dev)) & 15) return fail("buffers must be 16-byte aligned", WICK_ERR_ARG);
    if (reinterpret_cast<uintptr_t>(workspace_dev) & 255) return fail("workspace must be 256-byte aligned", WICK_ERR_ARG);
    const wick_terms* t = lists[0];
    for (int k = 0; k < n_lists; ++k) {
        const wick_terms* tk = lists[k];
        if (tk->needs_u_equals_d && U_dev != D_dev)
            return fail("this term list was built with WICK_BUILD_ISOSPIN (terms merged that are equal only for U == D); pass U_dev == D_dev", WICK_ERR_ARG);
        if (k > 0 && (tk->n_u != t->n_u || tk->n_d != t->n_d || tk->f[0].rows != t->f[0].rows || tk->f[0].cols != t->f[0].cols ||
                      tk->f[1].rows != t->f[1].rows || tk->f[1].cols != t->f[1].cols || tk->f[0].minor_row != t->f[0].minor_row ||
                      tk->f[0].minor_col != t->f[0].minor_col || tk->f[1].minor_row != t->f[1].minor_row || tk->f[1].minor_col != t->f[1].minor_col))
            return fail("the term lists do not share their unique-minor tables (build them with wick_build_terms_matrix)", WICK_ERR_UNSUPPORTED);
    }
    Plan p;
    if (!make_plan(t, n_lists, L, T, n_mom, workspace_bytes, false, &p)) return fail("need L >= 1, T >= 1, n_mom >= 0", WICK_ERR_ARG);
    if (p.S_b < GROUP) return fail("workspace smaller than the minimum workspace", WICK_ERR_WORKSPACE);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int rc = ensure_configured();
    if (rc != WICK_OK) return rc;
    for (int k = 0; k < n_lists; ++k) {
        if ((rc = upload_tables(lists[k], stream)) != WICK_OK) return rc;
        const bool outer_k = lists[k]->outer && !(flags & WICK_CONTRACT_FORCE_FLAT);
        if (!outer_k && (rc = upload_flat(lists[k], stream)) != WICK_OK) return rc;
    }

    const DeviceTables& d = t->dev;
    const int64_t nmu = int64_t(t->f[0].minor_row.size()), nmd = int64_t(t->f[1].minor_row.size());
    const int S_b = int(p.S_b);
    unsigned char* ws = static_cast<unsigned char*>(workspace_dev);
    double2* sigma_all = reinterpret_cast<double2*>(ws);                   // [n_lists][T * L^3]
    double2* MU = reinterpret_cast<double2*>(ws + p.sigma_bytes);          // sigma_bytes is a multiple of 256
    double2* MD = MU + nmu * S_b;
    // isospin limit (the paper's m_u = m_d): one propagator for both flavours.  When the two flavours
    // also have the same unique-minor table, every d minor IS the u minor with the same id: evaluate them once.
    const bool shared_minors = (U_dev == D_dev) && t->n_u == t->n_d && t->f[0].rows == t->f[1].rows &&
                               t->f[0].cols == t->f[1].cols && t->f[0].minor_row == t->f[1].minor_row &&
                               t->f[0].minor_col == t->f[1].minor_col;
    if (shared_minors) MD = MU;
    double2* partial = MD + nmd * S_b;
    double2* jac_inv[2], *jac_det[2];
    jac_inv[0] = partial + int64_t(MAX_CHUNKS) * S_b; jac_det[0] = jac_inv[0] + int64_t(144) * S_b;
    jac_inv[1] = jac_det[0] + S_b; jac_det[1] = jac_inv[1] + int64_t(144) * S_b;
    const double2* U = static_cast<const double2*>(U_dev);
    const double2* D = static_cast<const double2*>(D_dev);

    // staged factorised reduction: one CTA per SM, n_groups x n_bins CTAs ~ one wave of 148
    std::vector<StagedTables> stg(static_cast<size_t>(n_lists));
    std::vector<char> have_staged(size_t(n_lists), 0), use_outer(size_t(n_lists), 0);
    for (int k = 0; k < n_lists; ++k) {
        const wick_terms* tk = lists[k];
        use_outer[size_t(k)] = tk->outer && !(flags & WICK_CONTRACT_FORCE_FLAT);
        if (use_outer[size_t(k)] && tk->n_terms > 0 && !(flags & WICK_CONTRACT_NO_STAGED) &&
            std::max(nmu, nmd) * int64_t(S_b) < (int64_t(1) << 31)) {   // the staged kernel keeps 32-bit element offsets
            const int groups_full = int(std::min<int64_t>(S_b, (p.n_st + GROUP - 1) / GROUP * GROUP) / GROUP);
            const int n_bins = std::max(1, std::min(MAX_CHUNKS, 148 * STG_CTAS_PER_SM / std::max(1, groups_full)));
            rc = ensure_staged(tk, n_bins, (flags & WICK_CONTRACT_COMPLEX_COEFFS) != 0, stream, &stg[size_t(k)]);
            if (rc < 0) return rc;
            have_staged[size_t(k)] = (rc == 1);
        }
    }
    const bool try_reg = t->outer && !(flags & WICK_CONTRACT_NO_REG_MINORS);
    bool use_jacobi[2];
    for (int f = 0; f < 2; ++f) use_jacobi[f] = (flags & WICK_CONTRACT_JACOBI) && d.jacobi_desc[f] != nullptr;
    // both flavours in the Jacobi range and a term list of the order of the minor tables (Li-7-sized lists): one fused kernel
    // per list, no minor table at all
    bool fused_jacobi = use_jacobi[0] && use_jacobi[1] && !(flags & WICK_CONTRACT_JACOBI_UNFUSED);
    for (int k = 0; k < n_lists && fused_jacobi; ++k)
        if (lists[k]->n_terms > 8 * (nmu + nmd) || lists[k]->n_terms >= (int64_t(1) << 31)) fused_jacobi = false;
    if (fused_jacobi) {
        for (int k = 0; k < n_lists; ++k) {
            double2* sigma = sigma_all + int64_t(k) * p.n_st;
            if (lists[k]->n_terms == 0) { WICK_CUDA(cudaMemsetAsync(sigma, 0, size_t(p.n_st) * 16, stream)); continue; }
            const JacobiTerm* jt = nullptr;
            if ((rc = ensure_jacobi_fused(lists[k], stream, &jt)) != WICK_OK) return rc;
            WICK_CUDA(launch_jacobi_fused(t->n_u, t->n_d, U, D, 0, p.n_st, jt, lists[k]->n_terms, sigma, stream));
        }
    }
    for (int64_t st0 = 0; st0 < p.n_st && !fused_jacobi; st0 += S_b) {
        const int64_t n_valid = std::min<int64_t>(S_b, p.n_st - st0);
        const int n_groups = int((n_valid + GROUP - 1) / GROUP);
        // grid tables of 6x6 minors: register-resident instance kernel, one wave of CTAs (8 warp bins each)
        const int reg_bins = std::max(1, 148 / n_groups) * (REG_THREADS / 32);   // floor: the grid must not spill into a second wave
        for (int f = 0; f < (shared_minors ? 1 : 2); ++f) {
            const int n = f == 0 ? t->n_u : t->n_d;
            const double2* Pf = f == 0 ? U : D;
            double2* Mf = f == 0 ? MU : MD;
            const int pc = f == 0 ? PROF_MINORS_U : PROF_MINORS_D;
            if (use_jacobi[f]) {
                // one 12x12 inverse + determinant per site, then the (12-n) x (12-n) complementary minors of the inverse
                WICK_CUDA(launch_inverse12(Pf, st0, p.n_st, n_groups, jac_inv[f], jac_det[f], pc, stream));
                WICK_CUDA(launch_minors(12 - n, jac_inv[f], 0, n_valid, n_groups, S_b, d.jacobi_desc[f], f == 0 ? nmu : nmd, false, Mf, pc, stream));
                continue;
            }
            RegTables rt;
            rc = try_reg ? ensure_reg(t, f, reg_bins, stream, &rt) : 0;
            if (rc < 0) return rc;
            if (rc == 1) WICK_CUDA(launch_minors_reg(n, Pf, st0, p.n_st, n_groups, S_b, rt, Mf, pc, stream));
            else WICK_CUDA(launch_minors(n, Pf, st0, p.n_st, n_groups, S_b, d.minor_desc[f], f == 0 ? nmu : nmd, true, Mf, pc, stream));
        }
        for (int k = 0; k < n_lists; ++k) {
            const wick_terms* tk = lists[k];
            const DeviceTables& dk = tk->dev;
            double2* sigma = sigma_all + int64_t(k) * p.n_st;
            int n_chunks = 1;
            if (tk->n_terms == 0) {
                WICK_CUDA(cudaMemsetAsync(sigma + st0, 0, size_t(n_valid) * 16, stream));
                continue;
            }
            if (use_outer[size_t(k)] && have_staged[size_t(k)]) {
                WICK_CUDA(launch_reduce_staged(MU, MD, n_groups, S_b, stg[size_t(k)], partial, &n_chunks, stream));
            } else if (use_outer[size_t(k)]) {
                OuterTables ot;
                ot.n_cols_u = int(tk->f[0].cols.size()); ot.n_cols_d = int(tk->f[1].cols.size());
                ot.sink_ptr = dk.sink_ptr; ot.sink_rdoff = dk.sink_rdoff; ot.sink_c = reinterpret_cast<const double2*>(dk.sink_c);
                ot.src_ptr = dk.src_ptr; ot.src_cu = dk.src_cu; ot.src_c = reinterpret_cast<const double2*>(dk.src_c);
                ot.ru_ptr = dk.ru_ptr; ot.ru_list = dk.ru_list; ot.cd_ptr = dk.cd_ptr; ot.cd_list = dk.cd_list;
                ot.bin_ptr = dk.red_bin_ptr; ot.items = reinterpret_cast<const int2*>(dk.red_items); ot.n_bins = dk.n_red_bins;
                WICK_CUDA(launch_reduce_outer(MU, MD, n_groups, S_b, ot, partial, &n_chunks, stream));
            } else {
                WICK_CUDA(launch_reduce_flat(MU, MD, n_groups, S_b, dk.t_uid, dk.t_did, reinterpret_cast<const double2*>(dk.t_w),
                                             tk->n_terms, partial, &n_chunks, MAX_CHUNKS, stream));
            }
            const double2* sc_u = use_jacobi[0] ? jac_det[0] : nullptr;
            const double2* sc_d = use_jacobi[1] ? (shared_minors ? jac_det[0] : jac_det[1]) : nullptr;
            WICK_CUDA(launch_finalize_sigma(partial, n_chunks, S_b, n_valid, sigma + st0, sc_u, sc_d, stream));
        }
    }
    for (int k = 0; k < n_lists; ++k)
        for (int m0 = 0; m0 < n_mom; m0 += MAX_MOMENTA) {
            MomentumList ml;
            ml.n = std::min(MAX_MOMENTA, n_mom - m0);
            for (int q = 0; q < ml.n; ++q)
                for (int c = 0; c < 3; ++c) ml.v[q][c] = momenta[3 * (m0 + q) + c];
            WICK_CUDA(launch_project(sigma_all + int64_t(k) * p.n_st, L, T, ml,
                                     static_cast<double2*>(C_out_dev) + (int64_t(k) * n_mom + m0) * T, stream));
        }
    if (sigma_out_dev)
        WICK_CUDA(cudaMemcpyAsync(sigma_out_dev, sigma_all, size_t(n_lists) * size_t(p.n_st) * 16, cudaMemcpyDeviceToDevice, stream));
    return WICK_OK;
}

}  // namespace

extern "C" int wick_contract(const void* U_dev, const void* D_dev, const wick_terms* t, const int32_t* momenta,
                             int n_mom, int L, int T, void* C_out_dev, void* sigma_out_dev, void* workspace_dev,
                             size_t workspace_bytes, unsigned flags, void* cuda_stream) {
    return contract_lists(U_dev, D_dev, &t, 1, momenta, n_mom, L, T, C_out_dev, sigma_out_dev, workspace_dev, workspace_bytes,
                          flags, cuda_stream, "wick_contract");
}

extern "C" size_t wick_contract_many_workspace_bytes(const wick_terms* t, int n_lists, int L, int T, int n_mom) {
    Plan p;
    if (n_lists < 1 || !make_plan(t, n_lists, L, T, n_mom, 0, true, &p)) return 0;
    return plan_bytes(p, p.S_b);
}

extern "C" int wick_contract_many(const void* U_dev, const void* D_dev, const wick_terms* const* lists, int n_lists,
                                  const int32_t* momenta, int n_mom, int L, int T, void* C_out_dev, void* sigma_out_dev,
                                  void* workspace_dev, size_t workspace_bytes, unsigned flags, void* cuda_stream) {
    return contract_lists(U_dev, D_dev, lists, n_lists, momenta, n_mom, L, T, C_out_dev, sigma_out_dev, workspace_dev, workspace_bytes,
                          flags, cuda_stream, "wick_contract_many");
}

// Cluster sinks: block tensor B[t][S_u][S_d] of a block handle (wick_build_block_terms), one timeslice after the other so that
// a 32-site group never straddles two timeslices.  Workspace: minors of a site batch + per-group partial tensors of a timeslice.
extern "C" size_t wick_block_tensor_workspace_bytes(const wick_terms* t, int L) {
    if (!t || !t->block_mode || L < 1) return 0;
    const int64_t V = int64_t(L) * L * L;
    const int64_t nm = int64_t(t->f[0].minor_row.size()) + int64_t(t->f[1].minor_row.size());
    const int64_t n_pairs = int64_t(t->f[0].cols.size()) * int64_t(t->f[1].cols.size());
    const int64_t groups = (V + GROUP - 1) / GROUP;
    int64_t sb = std::min<int64_t>(groups * GROUP, std::max<int64_t>(GROUP, int64_t(TARGET_MINOR_BYTES / size_t(nm * 16)) / GROUP * GROUP));
    return size_t(sb * nm * 16 + groups * n_pairs * 16 + 1024);
}

extern "C" int wick_block_tensor(const void* U_dev, const void* D_dev, const wick_terms* t, const int32_t* momentum, int L, int T,
                                 void* out_dev, void* workspace_dev, size_t workspace_bytes, unsigned flags, void* cuda_stream) {
    if (!U_dev || !D_dev || !t || !momentum || !out_dev || !workspace_dev || L < 1 || T < 1) { set_error("wick_block_tensor: bad argument"); return WICK_ERR_ARG; }
    if (!t->block_mode) { set_error("wick_block_tensor: not a block handle (wick_build_block_terms)"); return WICK_ERR_ARG; }
    if ((reinterpret_cast<uintptr_t>(U_dev) | reinterpret_cast<uintptr_t>(D_dev) | reinterpret_cast<uintptr_t>(out_dev)) & 15 ||
        reinterpret_cast<uintptr_t>(workspace_dev) & 255) { set_error("wick_block_tensor: misaligned buffer"); return WICK_ERR_ARG; }
    if (workspace_bytes < wick_block_tensor_workspace_bytes(t, L)) { set_error("wick_block_tensor: workspace smaller than wick_block_tensor_workspace_bytes()"); return WICK_ERR_WORKSPACE; }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int rc = ensure_configured();
    if (rc != WICK_OK) return rc;
    if ((rc = upload_tables(t, stream)) != WICK_OK) return rc;
    DeviceTables& d = t->dev;
    const int n_sink = int(t->sink.size());
    {   // sink terms as flat (row tuple ids, coefficient) arrays
        std::lock_guard<std::mutex> lock(t->mu);
        if (!d.block_blob) {
            const size_t ns = size_t(n_sink);
            std::vector<int32_t> ru(ns), rd(ns);
            std::vector<double> c(2 * ns);
            for (int i = 0; i < n_sink; ++i) { ru[size_t(i)] = t->sink[size_t(i)].qu; rd[size_t(i)] = t->sink[size_t(i)].qd; c[2 * size_t(i)] = t->sink[size_t(i)].c.real(); c[2 * size_t(i) + 1] = t->sink[size_t(i)].c.imag(); }
            BlobBuilder bb;
            const size_t o_c = bb.add(c.data(), c.size() * 8), o_u = bb.add(ru.data(), ru.size() * 4), o_d = bb.add(rd.data(), rd.size() * 4);
            void* blob = nullptr;
            WICK_CUDA(cudaMalloc(&blob, std::max<size_t>(bb.host.size(), 256)));
            cudaError_t e = cudaMemcpyAsync(blob, bb.host.data(), bb.host.size(), cudaMemcpyHostToDevice, stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
            if (e != cudaSuccess) { cudaFree(blob); set_error(std::string("block table upload: ") + cudaGetErrorString(e)); return WICK_ERR_CUDA; }
            d.block_blob = blob;
            d.block_c = static_cast<unsigned char*>(blob) + o_c; d.block_ru = static_cast<unsigned char*>(blob) + o_u; d.block_rd = static_cast<unsigned char*>(blob) + o_d;
        }
    }
    const int64_t V = int64_t(L) * L * L;
    const int64_t nmu = int64_t(t->f[0].minor_row.size()), nmd = int64_t(t->f[1].minor_row.size());
    const int n_cu = int(t->f[0].cols.size()), n_cd = int(t->f[1].cols.size());
    const int64_t n_pairs = int64_t(n_cu) * n_cd;
    const int64_t groups_t = (V + GROUP - 1) / GROUP;
    const int S_b = int(std::min<int64_t>(groups_t * GROUP, std::max<int64_t>(GROUP, int64_t(TARGET_MINOR_BYTES / size_t((nmu + nmd) * 16)) / GROUP * GROUP)));
    double2* MU = static_cast<double2*>(workspace_dev);
    double2* MD = MU + nmu * S_b;
    double2* part = MD + nmd * S_b;
    const double2* U = static_cast<const double2*>(U_dev);
    const double2* D = static_cast<const double2*>(D_dev);
    const bool try_reg = !(flags & WICK_CONTRACT_NO_REG_MINORS);
    for (int tt = 0; tt < T; ++tt) {
        const int64_t t_end = int64_t(tt + 1) * V;                     // lanes beyond the timeslice are invalid
        for (int64_t s0 = 0; s0 < V; s0 += S_b) {
            const int64_t n_valid = std::min<int64_t>(S_b, V - s0);
            const int n_groups = int((n_valid + GROUP - 1) / GROUP);
            const int reg_bins = std::max(1, 148 / n_groups) * (REG_THREADS / 32);   // floor: the grid must not spill into a second wave
            for (int f = 0; f < 2; ++f) {
                RegTables rt;
                rc = try_reg ? ensure_reg(t, f, reg_bins, stream, &rt) : 0;
                if (rc < 0) return rc;
                const double2* Pf = f == 0 ? U : D;
                double2* Mf = f == 0 ? MU : MD;
                const int pc = f == 0 ? PROF_MINORS_U : PROF_MINORS_D;
                if (rc == 1) WICK_CUDA(launch_minors_reg(t->f[f].n, Pf, int64_t(tt) * V + s0, t_end, n_groups, S_b, rt, Mf, pc, stream));
                else WICK_CUDA(launch_minors(t->f[f].n, Pf, int64_t(tt) * V + s0, t_end, n_groups, S_b, d.minor_desc[f], f == 0 ? nmu : nmd, true, Mf, pc, stream));
            }
            WICK_CUDA(launch_block_tensor(MU, MD, S_b, int(n_valid), n_cu, n_cd, static_cast<const int32_t*>(d.block_ru), static_cast<const int32_t*>(d.block_rd),
                                          static_cast<const double2*>(d.block_c), n_sink, L, s0, momentum, part + (s0 / GROUP) * n_pairs, stream));
        }
        WICK_CUDA(launch_block_sum(part, int(groups_t), int(n_pairs), static_cast<double2*>(out_dev) + int64_t(tt) * n_pairs, stream));
    }
    return WICK_OK;
}

// Step a4 for one flavour of a handle, through exactly the kernels wick_contract launches for it (tests: every minor of
// the library's own tables against the oracle's elimination).
extern "C" int wick_terms_minor_table(const void* P_dev, int64_t n_sites, const wick_terms* t, int flavour, unsigned flags,
                                      void* out_dev, void* cuda_stream) {
    if (!P_dev || !t || !out_dev || n_sites < 1 || n_sites > (int64_t(1) << 22) || (flavour != 0 && flavour != 1)) {
        set_error("wick_terms_minor_table: bad argument"); return WICK_ERR_ARG; }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int rc = ensure_configured();
    if (rc != WICK_OK) return rc;
    if ((rc = upload_tables(t, stream)) != WICK_OK) return rc;
    const FlavourTables& ft = t->f[flavour];
    const int n_groups = int((n_sites + GROUP - 1) / GROUP);
    const int S_b = n_groups * GROUP;
    const int reg_bins = std::max(1, 148 / n_groups) * (REG_THREADS / 32);   // floor: the grid must not spill into a second wave
    RegTables rt;
    rc = (t->outer && !(flags & WICK_CONTRACT_NO_REG_MINORS)) ? ensure_reg(t, flavour, reg_bins, stream, &rt) : 0;
    if (rc < 0) return rc;
    if (rc == 1) WICK_CUDA(launch_minors_reg(ft.n, static_cast<const double2*>(P_dev), 0, n_sites, n_groups, S_b, rt,
                                             static_cast<double2*>(out_dev), PROF_MINORS_U, stream));
    else WICK_CUDA(launch_minors(ft.n, static_cast<const double2*>(P_dev), 0, n_sites, n_groups, S_b, t->dev.minor_desc[flavour],
                                 int64_t(ft.minor_row.size()), true, static_cast<double2*>(out_dev), PROF_MINORS_U, stream));
    return WICK_OK;
}

namespace {
struct HostPathCache {
    enum Slot { U0 = 0, U1, D0, D1, WS, C, S, N_SLOTS };
    int device = -1;
    void* buf[N_SLOTS] = {};
    size_t cap[N_SLOTS] = {};
    cudaStream_t sc = nullptr, sx = nullptr;
    cudaEvent_t copied[2] = {nullptr, nullptr}, consumed[2] = {nullptr, nullptr};
    void release() {
        for (int k = 0; k < N_SLOTS; ++k) { if (buf[k]) cudaFree(buf[k]); buf[k] = nullptr; cap[k] = 0; }
        for (int k = 0; k < 2; ++k) {
            if (copied[k]) cudaEventDestroy(copied[k]);
            if (consumed[k]) cudaEventDestroy(consumed[k]);
            copied[k] = consumed[k] = nullptr;
        }
        if (sc) cudaStreamDestroy(sc);
        if (sx) cudaStreamDestroy(sx);
        sc = sx = nullptr;
        device = -1;
    }
    cudaError_t prepare() {                                     // streams and events for the current device
        int dev = -1;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        if (dev != device) release();
        device = dev;
        if (!sc && (e = cudaStreamCreate(&sc)) != cudaSuccess) return e;
        if (!sx && (e = cudaStreamCreate(&sx)) != cudaSuccess) return e;
        for (int k = 0; k < 2; ++k) {
            if (!copied[k] && (e = cudaEventCreateWithFlags(&copied[k], cudaEventDisableTiming)) != cudaSuccess) return e;
            if (!consumed[k] && (e = cudaEventCreateWithFlags(&consumed[k], cudaEventDisableTiming)) != cudaSuccess) return e;
        }
        return cudaSuccess;
    }
    cudaError_t acquire(int slot, size_t bytes, void** out) {   // grow-only
        if (cap[slot] < bytes) {
            if (buf[slot]) { cudaFree(buf[slot]); buf[slot] = nullptr; cap[slot] = 0; }
            const cudaError_t e = cudaMalloc(&buf[slot], bytes);
            if (e != cudaSuccess) return e;
            cap[slot] = bytes;
        }
        *out = buf[slot];
        return cudaSuccess;
    }
    ~HostPathCache() {}                                         // process exit: the driver reclaims; no CUDA calls in static destructors
};
HostPathCache& host_path_cache() { static thread_local HostPathCache c; return c; }
}  // namespace

extern "C" void wick_release_cached_buffers(void) { host_path_cache().release(); }

extern "C" int wick_contract_host(const void* U_host, const void* D_host, const wick_terms* t, const int32_t* momenta,
                                  int n_mom, int L, int T, void* C_out_host, void* sigma_out_host, unsigned flags) {
    if (!U_host || !D_host || !t || !C_out_host || (n_mom > 0 && !momenta) || L < 1 || T < 1 || n_mom < 0) {
        set_error("wick_contract_host: bad argument"); return WICK_ERR_ARG; }
    const int64_t V = int64_t(L) * L * L;
    // Timeslice blocks: propagators of block b+1 are copied on a second stream while block b computes.
    // Each block is an independent wick_contract over Tb timeslices.  The sum over the sites of a timeslice always has the
    // same shape; the order of the partial sums inside a site follows the number of 32-site groups per site batch, so
    // blockings with different batch shapes agree to rounding and equal shapes bit for bit.
    const size_t slice_bytes = size_t(V) * 144 * 16;
    size_t block_bytes = size_t(256) << 20;
    if (const char* ev = std::getenv("WICK_HOST_BLOCK_BYTES")) {   // test hook: small blocks exercise the double-buffered path
        const long long v = std::atoll(ev);
        if (v > 0) block_bytes = size_t(v);
    }
    int Tb = int(std::max<size_t>(1, block_bytes / slice_bytes));
    Tb = std::min(Tb, T);
    const size_t ws_bytes = wick_contract_workspace_bytes(t, L, Tb, n_mom);
    if (!ws_bytes) { set_error("wick_contract_host: bad sizes"); return WICK_ERR_ARG; }
    // device buffers, streams and events of the host path are kept per host thread between calls
    // (wick_release_cached_buffers frees them): a cudaMalloc of the multi-GB workspace per call costs
    // more than the contraction of a small lattice
    HostPathCache& hc = host_path_cache();
    int rc = WICK_OK;
    // on any exit both streams are drained: no copy from the caller's host buffers may still be pending
    auto cleanup = [&]() { if (hc.sc) cudaStreamSynchronize(hc.sc); if (hc.sx) cudaStreamSynchronize(hc.sx); };
#define WICK_CUDA_H(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { set_error(std::string(#call) + ": " + cudaGetErrorString(e_)); cleanup(); return WICK_ERR_CUDA; } } while (0)
    WICK_CUDA_H(hc.prepare());
    void *dU[2], *dD[2], *ws = nullptr, *dC = nullptr, *dS = nullptr;
    cudaStream_t sc = hc.sc, sx = hc.sx;
    cudaEvent_t* copied = hc.copied;
    cudaEvent_t* consumed = hc.consumed;
    for (int k = 0; k < 2; ++k) {
        WICK_CUDA_H(hc.acquire(HostPathCache::U0 + k, slice_bytes * Tb, &dU[k]));
        WICK_CUDA_H(hc.acquire(HostPathCache::D0 + k, slice_bytes * Tb, &dD[k]));
    }
    WICK_CUDA_H(hc.acquire(HostPathCache::WS, ws_bytes, &ws));
    WICK_CUDA_H(hc.acquire(HostPathCache::C, std::max<size_t>(size_t(n_mom) * Tb * 16, 16), &dC));
    if (sigma_out_host) WICK_CUDA_H(hc.acquire(HostPathCache::S, size_t(V) * Tb * 16, &dS));
    const unsigned char* Uh = static_cast<const unsigned char*>(U_host);
    const unsigned char* Dh = static_cast<const unsigned char*>(D_host);
    const bool alias = (U_host == D_host);                     // isospin limit: one propagator, copied once, U_dev == D_dev
    std::vector<double> Cblk(size_t(std::max(n_mom, 1)) * Tb * 2);
    const int n_blocks = (T + Tb - 1) / Tb;
    auto issue_copy = [&](int b) -> cudaError_t {
        const int k = b & 1, t0 = b * Tb, nt = std::min(Tb, T - t0);
        cudaError_t e = cudaStreamWaitEvent(sx, consumed[k], 0);
        if (e == cudaSuccess) e = cudaMemcpyAsync(dU[k], Uh + size_t(t0) * slice_bytes, slice_bytes * nt, cudaMemcpyHostToDevice, sx);
        if (e == cudaSuccess && !alias) e = cudaMemcpyAsync(dD[k], Dh + size_t(t0) * slice_bytes, slice_bytes * nt, cudaMemcpyHostToDevice, sx);
        if (e == cudaSuccess) e = cudaEventRecord(copied[k], sx);
        return e;
    };
    WICK_CUDA_H(issue_copy(0));
    for (int b = 0; b < n_blocks && rc == WICK_OK; ++b) {
        const int k = b & 1, t0 = b * Tb, nt = std::min(Tb, T - t0);
        if (b + 1 < n_blocks) WICK_CUDA_H(issue_copy(b + 1));
        WICK_CUDA_H(cudaStreamWaitEvent(sc, copied[k], 0));
        rc = wick_contract(dU[k], alias ? dU[k] : dD[k], t, momenta, n_mom, L, nt, dC, dS, ws, ws_bytes, flags, sc);
        if (rc != WICK_OK) break;
        WICK_CUDA_H(cudaEventRecord(consumed[k], sc));
        WICK_CUDA_H(cudaMemcpyAsync(Cblk.data(), dC, size_t(n_mom) * nt * 16, cudaMemcpyDeviceToHost, sc));
        if (sigma_out_host)
            WICK_CUDA_H(cudaMemcpyAsync(static_cast<unsigned char*>(sigma_out_host) + size_t(t0) * V * 16, dS, size_t(V) * nt * 16, cudaMemcpyDeviceToHost, sc));
        WICK_CUDA_H(cudaStreamSynchronize(sc));
        double* Co = static_cast<double*>(C_out_host);
        for (int m = 0; m < n_mom; ++m)
            std::memcpy(Co + (size_t(m) * T + t0) * 2, Cblk.data() + size_t(m) * nt * 2, size_t(nt) * 16);
    }
    cleanup();
#undef WICK_CUDA_H
    return rc;
}

extern "C" int wick_minor_dets(const void* P_dev, int64_t n_sites, int n, const uint8_t* rows, const uint8_t* cols,
                               int64_t n_minors, void* out_dev, void* cuda_stream) {
    if (!P_dev || !out_dev || n < 0 || n > 12 || n_sites < 0 || n_minors < 0 || (n > 0 && n_minors > 0 && (!rows || !cols))) {
        set_error("wick_minor_dets: bad argument"); return WICK_ERR_ARG; }
    for (int64_t k = 0; k < n_minors * n; ++k)
        if (rows[k] > 11 || cols[k] > 11) { set_error("wick_minor_dets: index >= 12"); return WICK_ERR_ARG; }
    if (n_sites == 0 || n_minors == 0) return WICK_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int rc = ensure_configured();
    if (rc != WICK_OK) return rc;
    const int64_t n_pad = (n_sites + GROUP - 1) / GROUP * GROUP;
    const bool direct = (n_pad == n_sites);                   // out[m][s] has row length n_sites: usable as S_b only if padded
    // descriptors built from the caller's tuples (any order, repeats allowed), in slabs of 32768 minors
    const int64_t slab = 32768;
    const int words = minor_desc_words(n);
    std::vector<uint64_t> desc(size_t(std::min(slab, n_minors)) * size_t(words));
    void *d_desc = nullptr, *d_tmp = nullptr;
    auto cleanup = [&]() { cudaFree(d_desc); cudaFree(d_tmp); };
#define WICK_CUDA_M(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { set_error(std::string(#call) + ": " + cudaGetErrorString(e_)); cleanup(); return WICK_ERR_CUDA; } } while (0)
    WICK_CUDA_M(cudaMalloc(&d_desc, desc.size() * 8));
    // site batches so that the padded staging buffer stays small when n_sites is not a multiple of 32
    const int64_t S_b = direct ? n_sites : std::min<int64_t>(n_pad, 4096);
    if (!direct) WICK_CUDA_M(cudaMalloc(&d_tmp, size_t(std::min(slab, n_minors)) * size_t(S_b) * 16));
    if (S_b > (int64_t(1) << 22) && direct) {                 // keep 32-bit S_b
        cleanup(); set_error("wick_minor_dets: n_sites too large for one call (max 2^22)"); return WICK_ERR_UNSUPPORTED; }
    for (int64_t m0 = 0; m0 < n_minors; m0 += slab) {
        const int64_t nm = std::min(slab, n_minors - m0);
        for (int64_t m = 0; m < nm; ++m) {
            uint64_t rw = 0, cw = 0;
            for (int i = 0; i < n; ++i) {
                rw |= uint64_t(rows[(m0 + m) * n + i]) << (4 * i);
                cw |= uint64_t(cols[(m0 + m) * n + i]) << (4 * i);
            }
            pack_minor_desc(n, rw, cw, uint32_t(m), false, desc.data() + size_t(m) * size_t(words));
        }
        WICK_CUDA_M(cudaMemcpyAsync(d_desc, desc.data(), size_t(nm) * size_t(words) * 8, cudaMemcpyHostToDevice, stream));
        double2* out = static_cast<double2*>(out_dev) + m0 * n_sites;
        if (direct) {
            WICK_CUDA_M(launch_minors(n, static_cast<const double2*>(P_dev), 0, n_sites, int(n_sites / GROUP), int(S_b),
                                      d_desc, nm, false, out, PROF_MINORS_U, stream));
        } else {
            for (int64_t s0 = 0; s0 < n_sites; s0 += S_b) {
                const int64_t nv = std::min(S_b, n_sites - s0);
                WICK_CUDA_M(launch_minors(n, static_cast<const double2*>(P_dev), s0, n_sites, int((nv + GROUP - 1) / GROUP), int(S_b),
                                          d_desc, nm, false, static_cast<double2*>(d_tmp), PROF_MINORS_U, stream));
                WICK_CUDA_M(cudaMemcpy2DAsync(out + s0, size_t(n_sites) * 16, d_tmp, size_t(S_b) * 16, size_t(nv) * 16, size_t(nm),
                                              cudaMemcpyDeviceToDevice, stream));
            }
        }
        WICK_CUDA_M(cudaStreamSynchronize(stream));           // the host descriptor slab is reused by the next one
    }
    cleanup();
#undef WICK_CUDA_M
    return WICK_OK;
}

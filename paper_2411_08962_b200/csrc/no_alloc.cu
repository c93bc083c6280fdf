// wick_minor_dets_static: step a4 alone (device_det App. A :648-652) for callers that cannot call cudaMalloc
// (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  Same kernels and same result as
// wick_minor_dets, but the scratch that call allocates per invocation -- the device copy of the minor descriptors and, for a
// site count that is not a multiple of 32, the padded staging buffer of the results -- lives in ONE file-scope device array
// of WICK_STATIC_SCRATCH_BYTES that every GPU which loads the library holds until exit.
//
// This entry point calls no cudaMalloc / cudaFree and no allocating library routine (the descriptors are packed into a
// fixed thread-local host array).  Every call on a device shares the array and finds the previous call's contents in it:
// nothing in it has to start at zero (descriptors are rewritten for the minors of the call, the staging buffer is only read
// back where this call's kernel wrote it), and calls that overlap on the GPU (two streams, two host threads) RACE on it.
#include <algorithm>
#include <cstring>
#include <mutex>
#include <string>

#include "kernels.cuh"
#include "wick_internal.h"

using namespace wick;

namespace {

constexpr size_t kScratchBytes = WICK_STATIC_SCRATCH_BYTES;
constexpr int64_t kMaxMinors = WICK_STATIC_MAX_MINORS;
constexpr size_t kDescBytes = size_t(kMaxMinors) * 2 * 8;            // two 64-bit words per minor for n >= 9
static_assert(kDescBytes % 256 == 0 && kDescBytes < kScratchBytes, "descriptor area must leave room for the staging buffer");

// In HOST code this name is only a stand-in for the device array (not a device address): the address a kernel may use is
// taken with cudaGetSymbolAddress below, once per device, with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_ptr[kMaxDevices] = {};                                 // per device: device address of g_static_scratch

int scratch_for_current_device(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { set_error(std::string("cudaGetDevice: ") + cudaGetErrorString(e)); return WICK_ERR_CUDA; }
    if (dev < 0 || dev >= kMaxDevices) { set_error("wick_minor_dets_static: device index out of range"); return WICK_ERR_UNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) { set_error(std::string("cudaGetSymbolAddress(static scratch): ") + cudaGetErrorString(e)); return WICK_ERR_CUDA; }
        e = configure_kernels();                                       // cudaFuncSetAttribute only: allocates nothing
        if (e != cudaSuccess) { set_error(std::string("configure_kernels(): ") + cudaGetErrorString(e)); return WICK_ERR_CUDA; }
        g_scratch_ptr[dev] = p;
    }
    *out = static_cast<unsigned char*>(g_scratch_ptr[dev]);
    return WICK_OK;
}

// same descriptor format as contract.cu: pack_minor_desc (kernels.cu: struct Desc), out id = position, no sign
void pack_desc(int n, uint64_t rows, uint64_t cols, uint32_t out_id, uint64_t* out) {
    if (minor_desc_words(n) == 1) out[0] = (rows & 0xffffffffull) | (cols << 32);
    else {
        out[0] = (rows & 0xffffffffffffull) | (uint64_t(out_id & 0xffffu) << 48);
        out[1] = (cols & 0xffffffffffffull) | (uint64_t((out_id >> 16) & 0x7fffu) << 48);
    }
}

}  // namespace

extern "C" size_t wick_static_scratch_bytes(void) { return kScratchBytes; }

extern "C" int wick_minor_dets_static(const void* P_dev, int64_t n_sites, int n, const uint8_t* rows, const uint8_t* cols,
                                      int64_t n_minors, void* out_dev, void* cuda_stream) {
    if (!P_dev || !out_dev || n < 0 || n > 12 || n_sites < 0 || n_minors < 0 || (n > 0 && n_minors > 0 && (!rows || !cols))) {
        set_error("wick_minor_dets_static: bad argument"); return WICK_ERR_ARG; }
    if (n_minors > kMaxMinors) {
        set_error("wick_minor_dets_static: n_minors = " + std::to_string(n_minors) + " exceeds the static limit of " +
                  std::to_string(kMaxMinors) + " minors per call (use wick_minor_dets, or split the call)");
        return WICK_ERR_UNSUPPORTED; }
    if (n_sites > (int64_t(1) << 22)) { set_error("wick_minor_dets_static: n_sites too large for one call (max 2^22)"); return WICK_ERR_UNSUPPORTED; }
    for (int64_t k = 0; k < n_minors * n; ++k)
        if (rows[k] > 11 || cols[k] > 11) { set_error("wick_minor_dets_static: index >= 12"); return WICK_ERR_ARG; }
    if (n_sites == 0 || n_minors == 0) return WICK_OK;
    const int64_t n_pad = (n_sites + GROUP - 1) / GROUP * GROUP;
    const bool direct = (n_pad == n_sites);                       // out[m][s] has row length n_sites: usable as S_b only if padded
    // ragged site count: results go through the staging area [minor][S_b] behind the descriptors, S_b sites at a time
    int64_t S_b = n_sites;
    if (!direct) {
        S_b = std::min<int64_t>(n_pad, int64_t((kScratchBytes - kDescBytes) / (size_t(n_minors) * 16)) / GROUP * GROUP);
        if (S_b < GROUP) {
            set_error("wick_minor_dets_static: " + std::to_string(n_minors) + " minors x 32 sites do not fit the static scratch of " +
                      std::to_string(kScratchBytes) + " bytes (n_sites is not a multiple of 32: results are staged)");
            return WICK_ERR_UNSUPPORTED; }
    }
    unsigned char* scratch = nullptr;
    int rc = scratch_for_current_device(&scratch);
    if (rc != WICK_OK) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    static thread_local uint64_t desc_host[size_t(kMaxMinors) * 2];   // fixed size: no host allocation either
    const int words = minor_desc_words(n);
    for (int64_t m = 0; m < n_minors; ++m) {
        uint64_t rw = 0, cw = 0;
        for (int i = 0; i < n; ++i) {
            rw |= uint64_t(rows[m * n + i]) << (4 * i);
            cw |= uint64_t(cols[m * n + i]) << (4 * i);
        }
        pack_desc(n, rw, cw, uint32_t(m), desc_host + size_t(m) * size_t(words));
    }
#define WICK_CUDA_S(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { set_error(std::string(#call) + ": " + cudaGetErrorString(e_)); cudaStreamSynchronize(stream); return WICK_ERR_CUDA; } } while (0)
    void* d_desc = scratch;
    double2* d_tmp = reinterpret_cast<double2*>(scratch + kDescBytes);
    WICK_CUDA_S(cudaMemcpyAsync(d_desc, desc_host, size_t(n_minors) * size_t(words) * 8, cudaMemcpyHostToDevice, stream));
    double2* out = static_cast<double2*>(out_dev);
    const double2* P = static_cast<const double2*>(P_dev);
    if (direct) {
        WICK_CUDA_S(launch_minors(n, P, 0, n_sites, int(n_sites / GROUP), int(S_b), d_desc, n_minors, false, out, PROF_MINORS_U, stream));
    } else {
        for (int64_t s0 = 0; s0 < n_sites; s0 += S_b) {
            const int64_t nv = std::min(S_b, n_sites - s0);
            WICK_CUDA_S(launch_minors(n, P, s0, n_sites, int((nv + GROUP - 1) / GROUP), int(S_b), d_desc, n_minors, false, d_tmp, PROF_MINORS_U, stream));
            WICK_CUDA_S(cudaMemcpy2DAsync(out + s0, size_t(n_sites) * 16, d_tmp, size_t(S_b) * 16, size_t(nv) * 16, size_t(n_minors),
                                          cudaMemcpyDeviceToDevice, stream));
        }
    }
    WICK_CUDA_S(cudaStreamSynchronize(stream));                  // desc_host is reused by this thread's next call
#undef WICK_CUDA_S
    return WICK_OK;
}

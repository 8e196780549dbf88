// fdas_plan_priv.h -- the plan object behind fdas_plan_t and the status macros (internal to
// fdas_api.cu and fdas_batch.cu).
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>

#include <complex>
#include <string>
#include <vector>

#include "../../include/fdas.h"
#include "fdas_host.h"
#include "fdas_kernels.h"

namespace fdas {
struct BatchState;   // fdas_batch.cu
void free_batch_state(BatchState*);
}

extern thread_local std::string g_detail;

static inline bool fdas_is_tc(int precision) { return precision == FDAS_BF16_TC || precision == FDAS_BF16_TC_PLANE16; }
static inline bool fdas_plane16(int precision) { return precision == FDAS_BF16_PLANE16 || precision == FDAS_BF16_TC_PLANE16; }

struct fdas_plan_s {
    fdas_info_t info;
    std::vector<fdas::cd> bank_time;  // nz x (2h+1), kept for diagnostics
    void* d_bank = nullptr;
    float2* d_tw1 = nullptr;
    float2* d_tw2 = nullptr;
    cufftHandle fft = 0;
    bool fft_made = false;
    void* d_fft_work = nullptr;
    float2* d_X = nullptr;  // nfft/2 + 1
    int32_t* d_blk_start = nullptr;
    int32_t* d_blk_len = nullptr;
    float* d_blk_med = nullptr;
    int nblk = 0;
    int nsplit = 1;
    fdas::TcGeom tc;                          // K2-TC operand geometry (FDAS_BF16_TC*)
    fdas::TcMapCache tc_maps;                 // K2-TC tensor maps of the output buffers seen so far
    int nsm = 148;
    int64_t launches = 0;
    unsigned short* d_maxplane = nullptr;    // block-max plane M (nz x nbins/8 codes of fdas_maxcode.h), written by K2
    const void* max_valid_for = nullptr;     // the plane M currently describes (nullptr: none)
    int hsum_mode = 0;                       // FDAS_HSUM_PLAIN | FDAS_HSUM_NEIGHBOUR_MAX
    unsigned short* d_maxplane_nbr = nullptr;   // dilated side plane (allocated when the mode is first set)
    cudaEvent_t ev_last = nullptr;           // end of the last public per-trial call (cross-stream ordering)
    cudaStream_t last_stream = nullptr;
    bool have_last = false;
    unsigned short* d_max2 = nullptr;        // K3 coarse side plane M2 (nz x nbins/64 codes), rebuilt from M by every call
    uint2* d_maybe = nullptr;                // K3 maybe list (maybe_capacity records)
    int64_t maybe_capacity = 0;
    int fail_prepare_in = -1;                // diagnostic (fdas_plan_debug_fail_prepare): >= 0 counts prepares down to an injected failure
    unsigned long long* d_maybe_count = nullptr;
    // workspace of fdas_search_host (lazy)
    float* ws_series = nullptr;
    void* ws_spec = nullptr;
    void* ws_plane = nullptr;
    fdas_cand_t* ws_cands = nullptr;
    int64_t ws_cap = 0;
    unsigned long long* ws_count = nullptr;
    unsigned long long* h_count = nullptr;  // pinned
    fdas::BatchState* batch = nullptr;      // workspace of fdas_search_batch (lazy)
};

#define CU(call)                                                                        \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess) {                                                        \
            g_detail = std::string(#call) + ": " + cudaGetErrorString(e_);              \
            return (e_ == cudaErrorMemoryAllocation) ? FDAS_EALLOC : FDAS_ECUDA;        \
        }                                                                               \
    } while (0)

#define CF(call)                                                                        \
    do {                                                                                \
        cufftResult r_ = (call);                                                        \
        if (r_ != CUFFT_SUCCESS) {                                                      \
            g_detail = std::string(#call) + ": cufft status " + std::to_string((int)r_); \
            return (r_ == CUFFT_ALLOC_FAILED) ? FDAS_EALLOC : FDAS_ECUFFT;              \
        }                                                                               \
    } while (0)


// Enqueue-only forms of the three per-trial calls with the block-max plane given explicitly
// (fdas_search_batch double-buffers it); arguments already validated.
int fdas_enqueue_prepare(fdas_plan_s* plan, const float* d_series, void* d_spec, cudaStream_t st);
int fdas_enqueue_convolve(fdas_plan_s* plan, const void* d_spec, void* d_plane,
                          unsigned short* d_maxplane, cudaStream_t st);
int fdas_enqueue_harmonic(fdas_plan_s* plan, const void* d_plane, unsigned short* d_maxplane,
                          bool build_max, int H, const float* h_thresholds, int64_t r_lo,
                          fdas_cand_t* d_cands, int64_t capacity, unsigned long long* d_count,
                          cudaStream_t st);

// fdas_kernels.h -- launchers of the three sm_100a kernels behind the C ABI (internal).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "../../include/fdas.h"

namespace fdas {

struct ConvParams {
    const void* spec;    // nbins complex: float2 (FDAS_FP32) or packed bf16x2 (re low, im high)
    void* plane;         // nz x pitch: float or bf16
    const void* bank;    // packed Khat, register order (fdas_host.h)
    const float2* tw1;   // [128][15]
    const float2* tw2;   // [16][7]
    int64_t nbins;
    int64_t pitch;
    int nz, h, V;
    unsigned short* maxplane;  // nz x mpitch bf16 bit patterns: max of every aligned block of 8 plane
                               // columns (as stored), rounded toward +inf (an upper bound)
    int64_t mpitch;      // nbins / 8
};

// K2: one CTA of 128 threads per (segment, template chunk); grid = (nseg, nsplit).
cudaError_t launch_convolve(int precision, const ConvParams& p, int64_t nseg, int nsplit,
                            cudaStream_t st);
int convolve_ctas_per_sm();  // resident CTAs per SM K2 is launched for (sizes the template split)

// K2-TC: the convolution stage as a dense contraction on the tensor cores (fdas_convolve_tc.cu).
// Direct correlation y_j(r) = sum_m w[r+m] conj(T_j[m]) written as D[r][n] = sum_k A[r][k] B[n][k]
// with A the sliding-window (Hankel) matrix of the bf16 spectrum and B the bf16 tap-domain bank.
struct ConvTcParams {
    const unsigned* spec;      // nbins packed bf16x2 (re low, im high)
    void* plane;               // nz x pitch: float or bf16
    const void* bimg;          // B operand image in UMMA K-major no-swizzle order (fdas_host.h)
    int bimg_bytes;
    int64_t nbins, pitch;
    int nz, h;
    int kp;                    // taps 2h+1 padded to a multiple of 16
    int ngroups, gch;          // template-pair groups per tile, chunks of 8 pairs per group (<= 6)
    unsigned short* maxplane;  // as ConvParams
    int64_t mpitch;
    __host__ __device__ int ng_cols() const { return 16 * gch; }
};
// One persistent CTA per SM; `nsm` CTAs are launched.  plane16 != 0 stores the plane as bf16.
cudaError_t launch_convolve_tc(int plane16, const ConvTcParams& p, int nsm, cudaStream_t st);
int convolve_tc_smem_bytes(const ConvTcParams& p);

struct WhitenParams {
    const float2* X;         // nfft/2 + 1 complex from cuFFT R2C
    void* spec;              // nbins complex fp32 or bf16x2
    const int32_t* blk_start;
    const int32_t* blk_len;
    float* blk_med;          // nblk (scratch)
    int nblk;
    int64_t nbins;
};
// K1a (block medians) + K1b (interpolate, scale, cast).  Two launches.
cudaError_t launch_whiten(int precision, const WhitenParams& p, cudaStream_t st);

struct HarmParams {
    const void* plane;
    int64_t nbins, pitch;
    int nz, H;
    int64_t r_lo;
    float thr[32];
    fdas_cand_t* cands;
    int64_t capacity;
    unsigned long long* count;        // caller's: true number of candidates
    unsigned short* maxplane;         // plan-owned block-max plane (bf16 bits, rounded up), nz x mpitch
    int64_t mpitch;                   // nbins / 8
    uint2* maybe;                     // plan-owned list of (r, j): fundamentals that failed the prefilter
    int64_t maybe_capacity;
    unsigned long long* maybe_count;  // plan-owned; followed by the overflow flag
    unsigned* overflow;               // plan-owned: set if the maybe list was too small
};
// K3: [build_max] + prefilter (pass A) + exact (pass B) + flags (pass C); `launches` receives the
// number of kernels launched.
cudaError_t launch_harmonic(int plane_is_bf16, bool build_max, const HarmParams& p, cudaStream_t st,
                            int* launches);

}  // namespace fdas

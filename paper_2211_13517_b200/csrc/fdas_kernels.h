// fdas_kernels.h -- launchers of the three sm_100a kernels behind the C ABI (internal).
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>

#include "../../include/fdas.h"

namespace fdas {

// A function attribute (cudaFuncSetAttribute) belongs to one device: this remembers, per device ordinal, where
// it has been set already (one bit per device, safe across host threads; ordinals >= 64 are set every time).
struct PerDeviceOnce {
    std::atomic<unsigned long long> mask{0ULL};
    template <class F>
    cudaError_t run(F&& set_attribute) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        const bool tracked = dev >= 0 && dev < 64;
        if (tracked && ((mask.load(std::memory_order_acquire) >> dev) & 1ULL)) return cudaSuccess;
        e = set_attribute();
        if (e == cudaSuccess && tracked) mask.fetch_or(1ULL << dev, std::memory_order_release);
        return e;
    }
};

struct ConvParams {
    const void* spec;    // nbins complex: float2 (FDAS_FP32) or packed bf16x2 (re low, im high)
    void* plane;         // nz x pitch: float or bf16
    const void* bank;    // packed Khat, register order (fdas_host.h)
    const float2* tw1;   // [T][15], T = seg_len / 16 (fdas_host.h build_twiddles)
    const float2* tw2;   // [Rb][Ra - 1]
    int64_t nbins;
    int64_t pitch;
    int nz, h, V;
    unsigned short* maxplane;  // nz x mpitch codes (fdas_maxcode.h): an upper bound of the max of every
                               // aligned block of 8 plane columns (as stored)
    int64_t mpitch;      // nbins / 8
};

// K2: one CTA of seg_len / 16 threads per (segment, template chunk); grid = (nseg, nsplit);
// seg_len = 1024, 2048 or 4096.
cudaError_t launch_convolve(int precision, int seg_len, const ConvParams& p, int64_t nseg, int nsplit,
                            cudaStream_t st);
int convolve_ctas_per_sm(int seg_len);  // resident CTAs per SM K2 is launched for (sizes the template split)

// K2-TC: the convolution stage as a dense contraction on the tensor cores (fdas_convolve_tc.cu).
// Direct correlation y_j(r) = sum_m w[r+m] conj(T_j[m]) written as D[p][n] = sum_k A[p][k] B[n][k]
// with A the bf16 tap-domain bank (one row per conjugate pair of templates, kept in tensor memory) and
// B the sliding-window (Hankel) matrix of the bf16 spectrum.
struct ConvTcParams {
    const unsigned* spec;      // nbins packed bf16x2 (re low, im high)
    void* plane;               // nz x pitch: float or bf16
    const uint32_t* bimg;      // bank image [2 parts][128 rows][kp/2 words] (fdas_host.h pack_bank_tc)
    int64_t nbins, pitch;
    int nz, h;
    int kp;                    // taps 2h+1 padded to a multiple of 16
    int npair;                 // conjugate template pairs handled by THIS launch, 1..128 (one TMEM lane each)
    int npair_total;           // nz / 2: pair p is rows j+ = nz - npair_total + p, j- = npair_total - 1 - p
    int pair0;                 // first pair of this launch (a bank of more than 128 pairs takes several)
    unsigned short* maxplane;  // as ConvParams
    int64_t mpitch;
};
// Tensor maps of the plane buffers seen so far (encoded on the host once per buffer).
struct TcMapCache {
    static constexpr int kEntries = 4;
    struct Entry {
        alignas(64) unsigned char pmap[128];        // CUtensorMap of the plane (boxes of 32 rows x 64 bins)
        alignas(64) unsigned char pmap_tail[128];   // the same with boxes of npair % 32 rows (ragged banks)
        const void* plane = nullptr;
        bool valid = false;
    } e[kEntries];
    int next = 0;
};
// One persistent CTA per SM; `nsm` CTAs are launched.  plane16 != 0 stores the plane as bf16.
cudaError_t launch_convolve_tc(int plane16, const ConvTcParams& p, TcMapCache* cache, int nsm, cudaStream_t st);
int convolve_tc_smem_bytes(int kp, int npair, int plane16);

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
    int tq[32];                       // pass A's integer thresholds (filled by launch_harmonic)
    fdas_cand_t* cands;
    int64_t capacity;
    unsigned long long* count;        // caller's: true number of candidates
    unsigned short* maxplane;         // plan-owned block-max plane (codes of fdas_maxcode.h), nz x mpitch
    int64_t mpitch;                   // nbins / 8
    uint2* maybe;                     // plan-owned list of (r, j): fundamentals that failed the prefilter
    int64_t maybe_capacity;
    unsigned long long* maybe_count;  // plan-owned; followed by the overflow flag
    unsigned* overflow;               // plan-owned: set if the maybe list was too small
    unsigned short* max2;             // plan-owned coarse side plane: nz x nbins / 64 codes, max of 8 codes of M
    int nbr;                          // 1: neighbour-maximised sums (reading A24)
    unsigned short* maxplane_nbr;     // plan-owned dilated side plane the prefilter scans when nbr = 1
};
// K3: [build_max] + prefilter (pass A) + exact (pass B) + flags (pass C); `launches` receives the
// number of kernels launched.
cudaError_t launch_harmonic(int plane_is_bf16, bool build_max, const HarmParams& p, cudaStream_t st,
                            int* launches);

}  // namespace fdas

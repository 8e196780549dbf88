// fdas_whiten.cu -- K1, running-median power whitening (BASELINE.json north_star; DESIGN.md step a2,
// reading A3).
//   K1a  one CTA per block of the A3 schedule: |X|^2 in registers, exact median by radix selection
//        (even count: mean of the two middle values)
//   K1b  per bin: linear interpolation of the block medians between block centres (constant outside
//        the first/last centre), w[k] = X[k] sqrt(ln2 / m(k)), w[0] = 0, stored fp32 or bf16 (RNE)
#include <cuda_bf16.h>

#include "fdas_kernels.h"

namespace fdas {

constexpr int kMedThreads = 256;
constexpr int kMedMax = 4096;
constexpr int kMedPer = kMedMax / kMedThreads;  // powers held in registers per thread

// Exact order statistics by radix selection on the bit patterns of the (non-negative) powers:
// four 8-bit passes, each a shared-memory histogram of the keys that still match the selected
// prefix, then the bin holding rank k.  The second middle value (even count) is either the same
// key (duplicates) or the smallest key above it.
__global__ void __launch_bounds__(kMedThreads) block_median_kernel(const WhitenParams p) {
    __shared__ unsigned hist[256];
    __shared__ unsigned sel_bin, sel_below, s_cnt_le, s_min_gt;
    const int b = blockIdx.x;
    const int start = p.blk_start[b], n = p.blk_len[b];
    unsigned key[kMedPer];
#pragma unroll
    for (int q = 0; q < kMedPer; ++q) {
        const int i = threadIdx.x + q * kMedThreads;
        key[q] = 0xffffffffu;
        if (i < n) {
            const float2 x = __ldg(p.X + start + i);
            key[q] = __float_as_uint(x.x * x.x + x.y * x.y);
        }
    }
    unsigned k = (unsigned)((n - 1) / 2);  // 0-based rank of the lower middle value
    unsigned prefix = 0u, mask = 0u;
    for (int shift = 24; shift >= 0; shift -= 8) {
        hist[threadIdx.x] = 0u;  // kMedThreads == 256 bins
        __syncthreads();
#pragma unroll
        for (int q = 0; q < kMedPer; ++q) {
            const int i = threadIdx.x + q * kMedThreads;
            if (i < n && (key[q] & mask) == prefix) atomicAdd(&hist[(key[q] >> shift) & 255u], 1u);
        }
        __syncthreads();
        if (threadIdx.x < 32) {
            unsigned c[8], local = 0u;
#pragma unroll
            for (int t = 0; t < 8; ++t) { c[t] = hist[threadIdx.x * 8 + t]; local += c[t]; }
            unsigned incl = local;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned v = __shfl_up_sync(0xffffffffu, incl, d);
                if (threadIdx.x >= d) incl += v;
            }
            unsigned below = incl - local;  // keys in lower bins
            if (k >= below && k < incl) {   // exactly one lane
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    if (k < below + c[t]) { sel_bin = threadIdx.x * 8 + t; sel_below = below; break; }
                    below += c[t];
                }
            }
        }
        __syncthreads();
        k -= sel_below;
        prefix |= sel_bin << shift;
        mask |= 255u << shift;
    }
    // prefix = key of rank (n-1)/2.  Rank n/2: same key if enough keys <= prefix, else the next key up.
    if (threadIdx.x == 0) { s_cnt_le = 0u; s_min_gt = 0xffffffffu; }
    __syncthreads();
    unsigned cnt = 0u, mn = 0xffffffffu;
#pragma unroll
    for (int q = 0; q < kMedPer; ++q) {
        const int i = threadIdx.x + q * kMedThreads;
        if (i < n) {
            if (key[q] <= prefix) ++cnt; else mn = min(mn, key[q]);
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        cnt += __shfl_xor_sync(0xffffffffu, cnt, d);
        mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, d));
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&s_cnt_le, cnt); atomicMin(&s_min_gt, mn); }
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned hi_rank = (unsigned)(n / 2);
        const unsigned hi_key = (s_cnt_le > hi_rank) ? prefix : s_min_gt;
        p.blk_med[b] = 0.5f * (__uint_as_float(prefix) + __uint_as_float(hi_key));
    }
}

// Twice the centre of block b (an integer): 2 c_b = 2 s_b + l_b - 1.
__device__ __forceinline__ int64_t centre2(const WhitenParams& p, int b) {
    return 2 * (int64_t)__ldg(p.blk_start + b) + __ldg(p.blk_len + b) - 1;
}

constexpr int kScaleThreads = 256;
constexpr int kScalePer = 8;   // bins per thread, strided by the CTA width (coalesced)

// One CTA scales kScaleThreads * kScalePer consecutive bins.  The bracketing pair of block centres is
// found once per CTA by binary search for its first bin; every bin then walks forward from there (the
// blocks are >= 32 bins long, usually 4096: a handful of steps at most).
template <bool BF16>
__global__ void __launch_bounds__(kScaleThreads) whiten_scale_kernel(const WhitenParams p) {
    __shared__ int s_lo;
    const int64_t k0 = (int64_t)blockIdx.x * (kScaleThreads * kScalePer);
    const int last = p.nblk - 1;
    if (threadIdx.x == 0) {
        int lo = 0, hi = last;   // largest lo with c2[lo] <= 2 k0 (0 if none)
        const int64_t k2 = 2 * k0;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (centre2(p, mid) <= k2) lo = mid; else hi = mid;
        }
        s_lo = lo;
    }
    __syncthreads();
    const int64_t c2_first = centre2(p, 0), c2_last = centre2(p, last);
    const float m_first = p.blk_med[0], m_last = p.blk_med[last];
    // the bracketing pair of centres and its medians stay in registers while the bins remain between them
    int lo = min(s_lo, max(last - 1, 0));
    int64_t c2lo = centre2(p, lo), c2hi = centre2(p, min(lo + 1, last));
    float mlo = p.blk_med[lo], mhi = p.blk_med[min(lo + 1, last)];
    float slope = (mhi - mlo) / (float)(int)max(c2hi - c2lo, (int64_t)1);       // per half bin (centres are in half bins)
#pragma unroll
    for (int q = 0; q < kScalePer; ++q) {
        const int64_t k = k0 + threadIdx.x + q * kScaleThreads;
        if (k >= p.nbins) break;
        float2 w = make_float2(0.f, 0.f);
        if (k > 0) {
            const int64_t k2 = 2 * k;
            float m;
            if (k2 <= c2_first) m = m_first;
            else if (k2 >= c2_last) m = m_last;
            else {
                if (k2 >= c2hi) {                                       // c2[lo] <= k2 < c2[lo+1]
                    while (lo + 1 < last && centre2(p, lo + 1) <= k2) ++lo;
                    c2lo = centre2(p, lo); c2hi = centre2(p, lo + 1);
                    mlo = p.blk_med[lo]; mhi = p.blk_med[lo + 1];
                    slope = (mhi - mlo) / (float)(int)(c2hi - c2lo);
                }
                m = fmaf((float)(int)(k2 - c2lo), slope, mlo);         // the distances fit 32 bits (blocks <= 4096 bins)
            }
            const float sc = 0.83255461115769775635f * rsqrtf(m);       // sqrt(ln 2 / m)
            const float2 x = __ldg(p.X + k);
            w = make_float2(x.x * sc, x.y * sc);
        }
        if (BF16) {
            const __nv_bfloat162 pk = __floats2bfloat162_rn(w.x, w.y);  // .x (re) in the low half
            reinterpret_cast<unsigned int*>(p.spec)[k] = *reinterpret_cast<const unsigned int*>(&pk);
        } else {
            reinterpret_cast<float2*>(p.spec)[k] = w;
        }
    }
}

cudaError_t launch_whiten(int precision, const WhitenParams& p, cudaStream_t st) {
    block_median_kernel<<<p.nblk, kMedThreads, 0, st>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int per_cta = kScaleThreads * kScalePer;
    const unsigned grid = (unsigned)((p.nbins + per_cta - 1) / per_cta);
    if (precision == FDAS_FP32) whiten_scale_kernel<false><<<grid, kScaleThreads, 0, st>>>(p);
    else whiten_scale_kernel<true><<<grid, kScaleThreads, 0, st>>>(p);
    return cudaGetLastError();
}

}  // namespace fdas

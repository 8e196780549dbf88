// fdas_whiten.cu -- K1, running-median power whitening (BASELINE.json north_star; DESIGN.md step a2,
// reading A3).
//   K1a  one CTA per block of the A3 schedule: |X|^2 into shared memory, bitonic sort, exact median
//        (even count: mean of the two middle values)
//   K1b  per bin: linear interpolation of the block medians between block centres (constant outside
//        the first/last centre), w[k] = X[k] sqrt(ln2 / m(k)), w[0] = 0, stored fp32 or bf16 (RNE)
#include <cuda_bf16.h>

#include "fdas_kernels.h"

namespace fdas {

constexpr int kMedThreads = 1024;
constexpr int kMedMax = 4096;

__global__ void __launch_bounds__(kMedThreads) block_median_kernel(const WhitenParams p) {
    __shared__ float v[kMedMax];
    const int b = blockIdx.x;
    const int start = p.blk_start[b], n = p.blk_len[b];
    int npad = 1;
    while (npad < n) npad <<= 1;
    for (int i = threadIdx.x; i < npad; i += kMedThreads) {
        float pw = __int_as_float(0x7f800000);  // +inf padding sorts to the end
        if (i < n) {
            const float2 x = __ldg(p.X + start + i);
            pw = x.x * x.x + x.y * x.y;
        }
        v[i] = pw;
    }
    __syncthreads();
    for (int k = 2; k <= npad; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = threadIdx.x; i < npad; i += kMedThreads) {
                const int ixj = i ^ j;
                if (ixj > i) {
                    const float a = v[i], c = v[ixj];
                    const bool up = ((i & k) == 0);
                    if ((a > c) == up) { v[i] = c; v[ixj] = a; }
                }
            }
            __syncthreads();
        }
    }
    if (threadIdx.x == 0) p.blk_med[b] = 0.5f * (v[(n - 1) / 2] + v[n / 2]);
}

template <bool BF16>
__global__ void __launch_bounds__(256) whiten_scale_kernel(const WhitenParams p) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= p.nbins) return;
    float2 w = make_float2(0.f, 0.f);
    if (k > 0) {
        // twice the block centres are integers: 2 c_b = 2 s_b + l_b - 1
        const int64_t k2 = 2 * k;
        const int last = p.nblk - 1;
        const int64_t c2_first = 2 * (int64_t)p.blk_start[0] + p.blk_len[0] - 1;
        const int64_t c2_last = 2 * (int64_t)p.blk_start[last] + p.blk_len[last] - 1;
        float m;
        if (k2 <= c2_first) m = p.blk_med[0];
        else if (k2 >= c2_last) m = p.blk_med[last];
        else {
            int lo = 0, hi = last;  // c2[lo] <= k2 < c2[hi]
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                const int64_t c2m = 2 * (int64_t)__ldg(p.blk_start + mid) + __ldg(p.blk_len + mid) - 1;
                if (c2m <= k2) lo = mid; else hi = mid;
            }
            const int64_t c2lo = 2 * (int64_t)__ldg(p.blk_start + lo) + __ldg(p.blk_len + lo) - 1;
            const int64_t c2hi = 2 * (int64_t)__ldg(p.blk_start + hi) + __ldg(p.blk_len + hi) - 1;
            const float t = (float)(k2 - c2lo) / (float)(c2hi - c2lo);
            const float mlo = p.blk_med[lo], mhi = p.blk_med[hi];
            m = mlo + t * (mhi - mlo);
        }
        const float sc = sqrtf(0.69314718055994530942f / m);
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

cudaError_t launch_whiten(int precision, const WhitenParams& p, cudaStream_t st) {
    block_median_kernel<<<p.nblk, kMedThreads, 0, st>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)((p.nbins + 255) / 256);
    if (precision == FDAS_FP32) whiten_scale_kernel<false><<<grid, 256, 0, st>>>(p);
    else whiten_scale_kernel<true><<<grid, 256, 0, st>>>(p);
    return cudaGetLastError();
}

}  // namespace fdas

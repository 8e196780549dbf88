// fdas_harmonic.cu -- K3, harmonic summing, thresholding and candidate compaction (BASELINE.json
// north_star "harmonic summing and thresholding"; DESIGN.md step a6, readings A12, A13, A14).
//   S_h(r,j) = sum_{k=1..h} P[row_k(j)][k r]  while k r <= Nb-1 and 0 <= v2 <= 2 c2,
//   v2 = 2 k j - (k-1) c2 (twice the row of harmonic k), c2 = nz-1, row_k = (v2+1)/2
//   (half-integers round away from zero).  A candidate (r, j, h) is emitted for every S_h > T_h.
// One thread per fundamental (r, j): lanes of a warp hold consecutive r, so harmonic k is a
// stride-k gather along one plane row; hits are compacted with one atomic per warp.
#include <cuda_bf16.h>

#include "fdas_kernels.h"

namespace fdas {

template <typename T> __device__ __forceinline__ float ldp(const T* p);
template <> __device__ __forceinline__ float ldp<float>(const float* p) { return __ldg(p); }
template <> __device__ __forceinline__ float ldp<__nv_bfloat16>(const __nv_bfloat16* p) {
    return __bfloat162float(*p);
}

// S_h at (r, j) if defined (r in [r_lo, Nb), all h harmonics inside the plane).
template <typename T>
__device__ bool harmonic_sum_at(const T* P, const HarmParams& p, int64_t r, int j, int h, float* out) {
    if (j < 0 || j >= p.nz || r < p.r_lo || r >= p.nbins) return false;
    const int c2 = p.nz - 1;
    float S = 0.f;
    for (int k = 1; k <= h; ++k) {
        const int v2 = 2 * k * j - (k - 1) * c2;
        if (v2 < 0 || v2 > 2 * c2 || (int64_t)k * r > p.nbins - 1) return false;
        const int row = min((v2 + 1) >> 1, c2);
        S += ldp(P + (size_t)row * p.pitch + (size_t)k * r);
    }
    *out = S;
    return true;
}

template <typename T>
__global__ void __launch_bounds__(256) harmonic_kernel(const HarmParams p) {
    const T* P = reinterpret_cast<const T*>(p.plane);
    const int j = blockIdx.y;
    const int64_t r = p.r_lo + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool inb = r < p.nbins;
    const int c2 = p.nz - 1;
    const unsigned lane = threadIdx.x & 31;
    float S = 0.f;
    for (int k = 1; k <= p.H; ++k) {
        const int v2 = 2 * k * j - (k - 1) * c2;
        const bool valid = inb && v2 >= 0 && v2 <= 2 * c2 && (int64_t)k * r <= p.nbins - 1;
        if (!__any_sync(0xffffffffu, valid)) break;
        if (valid) {
            const int row = min((v2 + 1) >> 1, c2);
            S += ldp(P + (size_t)row * p.pitch + (size_t)k * r);
        }
        const bool hit = valid && (S > p.thr[k - 1]);
        const unsigned hits = __ballot_sync(0xffffffffu, hit);
        if (hits) {
            unsigned long long base = 0;
            if (lane == (unsigned)(__ffs(hits) - 1))
                base = atomicAdd(p.count, (unsigned long long)__popc(hits));
            base = __shfl_sync(0xffffffffu, base, __ffs(hits) - 1);
            if (hit) {
                const unsigned long long slot = base + __popc(hits & ((1u << lane) - 1u));
                if ((int64_t)slot < p.capacity) {
                    // local-maximum attribute over the 8 neighbours for which S_k is defined;
                    // strict against neighbours that precede (j, r) lexicographically
                    unsigned flag = 1;
                    for (int dj = -1; dj <= 1 && flag; ++dj)
                        for (int dr = -1; dr <= 1 && flag; ++dr) {
                            if (dj == 0 && dr == 0) continue;
                            float nv;
                            if (!harmonic_sum_at(P, p, r + dr, j + dj, k, &nv)) continue;
                            const bool precedes = (dj < 0) || (dj == 0 && dr < 0);
                            if (precedes ? !(S > nv) : !(S >= nv)) flag = 0;
                        }
                    fdas_cand_t c;
                    c.r = (uint32_t)r;
                    c.zidx = (int16_t)j;
                    c.h = (uint16_t)k;
                    c.power = S;
                    c.flags = flag;
                    p.cands[slot] = c;
                }
            }
        }
    }
}

cudaError_t launch_harmonic(int plane_is_bf16, const HarmParams& p, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(p.count, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    if (p.r_lo >= p.nbins) return cudaSuccess;
    dim3 grid((unsigned)((p.nbins - p.r_lo + 255) / 256), (unsigned)p.nz), block(256);
    if (plane_is_bf16) harmonic_kernel<__nv_bfloat16><<<grid, block, 0, st>>>(p);
    else harmonic_kernel<float><<<grid, block, 0, st>>>(p);
    return cudaGetLastError();
}

}  // namespace fdas

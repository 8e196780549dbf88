// fdas_harmonic.cu -- K3, harmonic summing, thresholding and candidate compaction (BASELINE.json
// north_star "harmonic summing and thresholding"; DESIGN.md step a6, readings A12, A13, A14).
//   S_h(r,j) = sum_{k=1..h} P[row_k(j)][k r]  while k r <= Nb-1 and 0 <= v2 <= 2 c2,
//   v2 = 2 k j - (k-1) c2 (twice the row of harmonic k), c2 = nz-1, row_k = (v2+1)/2
//   (half-integers round away from zero).  A candidate (r, j, h) is emitted for every S_h > T_h.
//
// HBM-bound: every harmonic k is a stride-k gather along one plane row.  A CTA owns one row j and a
// tile of kTile fundamentals; thread t handles r = tile + t + 256 i (i < kRpt), so each load
// instruction of a warp touches a contiguous run of k*32 elements (min(32, 4k) sectors) and the row
// index arithmetic is CTA-uniform.  Threshold hits only set a bit; the rare emission path recomputes
// S_h in the same summation order, adds the local-maximum attribute and claims a slot atomically.
#include <cuda_bf16.h>

#include "fdas_kernels.h"

namespace fdas {

constexpr int kHarmThreads = 256;
constexpr int kRpt = 4;
constexpr int kTile = kHarmThreads * kRpt;

template <typename T> __device__ __forceinline__ float ldp(const T* p);
template <> __device__ __forceinline__ float ldp<float>(const float* p) { return __ldg(p); }
template <> __device__ __forceinline__ float ldp<__nv_bfloat16>(const __nv_bfloat16* p) {
    return __bfloat162float(__ldg(p));
}

// Geometry handed BY VALUE to the rare emission path (a reference to the kernel parameter struct
// would force every thread to spill all of it to local memory at kernel entry).
struct HarmGeom {
    int64_t nbins, pitch, r_lo, capacity;
    fdas_cand_t* cands;
    unsigned long long* count;
    int nz;
};

// S_h at (r, j) if defined (r in [r_lo, Nb), all h harmonics inside the plane); summed k = 1..h.
template <typename T>
__device__ bool harmonic_sum_at(const T* P, const HarmGeom p, int64_t r, int j, int h, float* out) {
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
__device__ __noinline__ void emit_candidate(const T* P, const HarmGeom p, int64_t r, int j, int h) {
    float S;
    if (!harmonic_sum_at(P, p, r, j, h, &S)) return;
    const unsigned long long slot = atomicAdd(p.count, 1ULL);
    if ((int64_t)slot >= p.capacity) return;
    // local-maximum attribute over the 8 neighbours for which S_h is defined; strict against the
    // neighbours that precede (j, r) lexicographically
    unsigned flag = 1;
    for (int dj = -1; dj <= 1 && flag; ++dj)
        for (int dr = -1; dr <= 1 && flag; ++dr) {
            if (dj == 0 && dr == 0) continue;
            float nv;
            if (!harmonic_sum_at(P, p, r + dr, j + dj, h, &nv)) continue;
            const bool precedes = (dj < 0) || (dj == 0 && dr < 0);
            if (precedes ? !(S > nv) : !(S >= nv)) flag = 0;
        }
    fdas_cand_t c;
    c.r = (uint32_t)r;
    c.zidx = (int16_t)j;
    c.h = (uint16_t)h;
    c.power = S;
    c.flags = flag;
    p.cands[slot] = c;
}

template <typename T>
__global__ void __launch_bounds__(kHarmThreads) harmonic_kernel(const HarmParams p) {
    const T* __restrict__ P = reinterpret_cast<const T*>(p.plane);
    const int j = blockIdx.y;
    const int c2 = p.nz - 1;
    // r of element i: rb + 256 i.  The tile grid starts at 0; r < r_lo is masked.
    const int64_t rb = (int64_t)blockIdx.x * kTile + threadIdx.x;
    const int64_t last = p.nbins - 1;
    float S[kRpt];
    unsigned hits[kRpt];
#pragma unroll
    for (int i = 0; i < kRpt; ++i) { S[i] = 0.f; hits[i] = 0u; }

    for (int k = 1; k <= p.H; ++k) {
        const int v2 = 2 * k * j - (k - 1) * c2;          // CTA-uniform
        if (v2 < 0 || v2 > 2 * c2) break;
        if ((int64_t)k * ((int64_t)blockIdx.x * kTile) > last) break;   // whole tile beyond Nb/k
        const int row = min((v2 + 1) >> 1, c2);
        const T* __restrict__ rowp = P + (size_t)row * p.pitch;
        const float thr = p.thr[k - 1];
        float v[kRpt];
#pragma unroll
        for (int i = 0; i < kRpt; ++i) {
            const int64_t c = (int64_t)k * (rb + 256 * i);
            // beyond the plane: +0 keeps S finite, the hit bit is masked below
            v[i] = (c <= last) ? ldp(rowp + c) : 0.f;
        }
#pragma unroll
        for (int i = 0; i < kRpt; ++i) {
            const int64_t c = (int64_t)k * (rb + 256 * i);
            S[i] += v[i];
            if (c <= last && S[i] > thr) hits[i] |= 1u << (k - 1);
        }
    }
    unsigned any = 0;
#pragma unroll
    for (int i = 0; i < kRpt; ++i) {
        if (rb + 256 * i < p.r_lo) hits[i] = 0u;
        any |= hits[i];
    }
    if (any) {
        HarmGeom g;
        g.nbins = p.nbins; g.pitch = p.pitch; g.r_lo = p.r_lo; g.capacity = p.capacity;
        g.cands = p.cands; g.count = p.count; g.nz = p.nz;
#pragma unroll 1
        for (int i = 0; i < kRpt; ++i) {
            unsigned m = hits[i];
            while (m) {
                const int k = __ffs(m);
                m &= m - 1;
                emit_candidate(P, g, rb + 256 * i, j, k);
            }
        }
    }
}

cudaError_t launch_harmonic(int plane_is_bf16, const HarmParams& p, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(p.count, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    if (p.r_lo >= p.nbins) return cudaSuccess;
    dim3 grid((unsigned)((p.nbins + kTile - 1) / kTile), (unsigned)p.nz), block(kHarmThreads);
    if (plane_is_bf16) harmonic_kernel<__nv_bfloat16><<<grid, block, 0, st>>>(p);
    else harmonic_kernel<float><<<grid, block, 0, st>>>(p);
    return cudaGetLastError();
}

}  // namespace fdas

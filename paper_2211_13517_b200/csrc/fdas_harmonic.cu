// fdas_harmonic.cu -- K3, harmonic summing, thresholding and candidate compaction (BASELINE.json
// north_star "harmonic summing and thresholding"; DESIGN.md step a6, readings A12, A13, A14).
//   S_h(r,j) = sum_{k=1..h} P[row_k(j)][k r]  while k r <= Nb-1 and 0 <= v2 <= 2 c2,
//   v2 = 2 k j - (k-1) c2 (twice the row of harmonic k), c2 = nz-1, row_k = (v2+1)/2
//   (half-integers round away from zero).  A candidate (r, j, h) is emitted for every S_h > T_h.
//
// The direct evaluation is HBM-bound: the stride-k gathers touch 3.2x the plane in 32-byte sectors.
// K3 therefore works branch-and-bound on the block-max plane M[j][b] = max P[j][8b..8b+7] that K2
// writes beside the plane (1/8 of its size):
//   pass A (prefilter)  U_h(r,j) = sum_{k<=h} M[row_k][(k r) >> 3] >= S_h(r,j) term by term, in the
//                       same summation order, and fp32 addition is monotone -- so U_h <= T_h for all
//                       h proves that (r, j) has no candidate without touching the plane.  The few
//                       fundamentals that fail the test go to a "maybe" list.
//   pass B (exact)      one thread per maybe entry: the plain definition above on the real plane,
//                       thresholds, local-maximum attribute, atomic slot claim.
// Results are identical to evaluating every fundamental exactly.  When the plane was not produced by
// fdas_convolve_plane of this plan (hand-made planes), M is first rebuilt from it (build_max_kernel).
#include <cuda_bf16.h>

#include "fdas_kernels.h"

namespace fdas {

constexpr int kHarmThreads = 256;
constexpr int kRpt = 4;
constexpr int kTile = kHarmThreads * kRpt;
constexpr int kExactBlocks = 592;

template <typename T> __device__ __forceinline__ float ldp(const T* p);
template <> __device__ __forceinline__ float ldp<float>(const float* p) { return __ldg(p); }
template <> __device__ __forceinline__ float ldp<__nv_bfloat16>(const __nv_bfloat16* p) {
    return __bfloat162float(__ldg(p));
}

// Geometry handed BY VALUE to the out-of-line exact path (a reference to the kernel parameter
// struct would make every thread spill all of it to local memory at kernel entry).
struct HarmGeom {
    int64_t nbins, pitch, r_lo, capacity;
    fdas_cand_t* cands;
    unsigned long long* count;
    int nz, H;
};

__device__ __forceinline__ HarmGeom geom_of(const HarmParams& p) {
    HarmGeom g;
    g.nbins = p.nbins; g.pitch = p.pitch; g.r_lo = p.r_lo; g.capacity = p.capacity;
    g.cands = p.cands; g.count = p.count; g.nz = p.nz; g.H = p.H;
    return g;
}

// S_h at (r, j) if defined (r in [r_lo, Nb), all h harmonics inside the plane); summed k = 1..h.
template <typename T>
__device__ bool harmonic_sum_at(const T* P, const HarmGeom& g, int64_t r, int j, int h, float* out) {
    if (j < 0 || j >= g.nz || r < g.r_lo || r >= g.nbins) return false;
    const int c2 = g.nz - 1;
    float S = 0.f;
    for (int k = 1; k <= h; ++k) {
        const int v2 = 2 * k * j - (k - 1) * c2;
        if (v2 < 0 || v2 > 2 * c2 || (int64_t)k * r > g.nbins - 1) return false;
        const int row = min((v2 + 1) >> 1, c2);
        S += ldp(P + (size_t)row * g.pitch + (size_t)k * r);
    }
    *out = S;
    return true;
}

// The plain definition for one fundamental: all h, thresholds, local-maximum attribute (8 neighbours
// for which S_h is defined; strict against those preceding (j, r) lexicographically), slot claim.
template <typename T>
__device__ __noinline__ void exact_fundamental(const T* P, const HarmGeom g, const float* thr,
                                               int64_t r, int j) {
    if (r < g.r_lo || r >= g.nbins) return;
    const int c2 = g.nz - 1;
    float S = 0.f;
    for (int h = 1; h <= g.H; ++h) {
        const int v2 = 2 * h * j - (h - 1) * c2;
        if (v2 < 0 || v2 > 2 * c2 || (int64_t)h * r > g.nbins - 1) break;
        const int row = min((v2 + 1) >> 1, c2);
        S += ldp(P + (size_t)row * g.pitch + (size_t)h * r);
        if (!(S > thr[h - 1])) continue;
        const unsigned long long slot = atomicAdd(g.count, 1ULL);   // the true count
        if ((int64_t)slot >= g.capacity) continue;
        unsigned flag = 1;
        for (int dj = -1; dj <= 1 && flag; ++dj)
            for (int dr = -1; dr <= 1 && flag; ++dr) {
                if (dj == 0 && dr == 0) continue;
                float nv;
                if (!harmonic_sum_at(P, g, r + dr, j + dj, h, &nv)) continue;
                const bool precedes = (dj < 0) || (dj == 0 && dr < 0);
                if (precedes ? !(S > nv) : !(S >= nv)) flag = 0;
            }
        fdas_cand_t c;
        c.r = (uint32_t)r;
        c.zidx = (int16_t)j;
        c.h = (uint16_t)h;
        c.power = S;
        c.flags = flag;
        g.cands[slot] = c;
    }
}

// ---- M from an arbitrary plane (only when K2 did not just write it): one thread per block of 8.
template <typename T>
__global__ void __launch_bounds__(256) build_max_kernel(const HarmParams p) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y;
    if (b >= p.mpitch) return;
    const T* src = reinterpret_cast<const T*>(p.plane) + (size_t)j * p.pitch + 8 * b;
    float m = ldp(src);
#pragma unroll
    for (int i = 1; i < 8; ++i) m = fmaxf(m, ldp(src + i));
    p.maxplane[(size_t)j * p.mpitch + b] = m;
}

// ---- pass A: upper bounds from the block-max plane.  A CTA owns one row j and a tile of kTile
// fundamentals; thread t handles r = tile + t + 256 i, so the row arithmetic is CTA-uniform and the
// lanes of a warp read runs of (32 k)/8 consecutive elements of M.
template <typename T>
__global__ void __launch_bounds__(kHarmThreads) prefilter_kernel(const HarmParams p) {
    __shared__ float sthr[32];   // thresholds for the (rare) out-of-line exact path
    if (threadIdx.x < 32) sthr[threadIdx.x] = p.thr[threadIdx.x];
    __syncthreads();
    const int j = blockIdx.y;
    const int c2 = p.nz - 1;
    const int64_t rb = (int64_t)blockIdx.x * kTile + threadIdx.x;
    const int64_t last = p.nbins - 1;
    float U[kRpt];
    bool flagged[kRpt];
#pragma unroll
    for (int i = 0; i < kRpt; ++i) { U[i] = 0.f; flagged[i] = false; }

    for (int k = 1; k <= p.H; ++k) {
        const int v2 = 2 * k * j - (k - 1) * c2;          // CTA-uniform
        if (v2 < 0 || v2 > 2 * c2) break;
        if ((int64_t)k * ((int64_t)blockIdx.x * kTile) > last) break;   // whole tile beyond Nb/k
        const int row = min((v2 + 1) >> 1, c2);
        const float* __restrict__ mrow = p.maxplane + (size_t)row * p.mpitch;
        const float thr = p.thr[k - 1];
        float v[kRpt];
#pragma unroll
        for (int i = 0; i < kRpt; ++i) {
            const int64_t c = (int64_t)k * (rb + 256 * i);
            v[i] = (c <= last) ? __ldg(mrow + (c >> 3)) : 0.f;
        }
#pragma unroll
        for (int i = 0; i < kRpt; ++i) {
            const int64_t c = (int64_t)k * (rb + 256 * i);
            U[i] += v[i];
            flagged[i] = flagged[i] || (c <= last && U[i] > thr);
        }
    }
#pragma unroll
    for (int i = 0; i < kRpt; ++i) {
        const int64_t r = rb + 256 * i;
        if (flagged[i] && r >= p.r_lo) {
            const unsigned long long slot = atomicAdd(p.maybe_count, 1ULL);
            if (slot < (unsigned long long)p.maybe_capacity) {
                p.maybe[slot] = make_uint2((unsigned)r, (unsigned)j);
            } else {   // list full: evaluate here so that nothing is ever dropped
                exact_fundamental(reinterpret_cast<const T*>(p.plane), geom_of(p), sthr, r, j);
            }
        }
    }
}

// ---- pass B: one thread per maybe entry.
template <typename T>
__global__ void __launch_bounds__(128) exact_kernel(const HarmParams p) {
    __shared__ float sthr[32];
    if (threadIdx.x < 32) sthr[threadIdx.x] = p.thr[threadIdx.x];
    __syncthreads();
    const T* P = reinterpret_cast<const T*>(p.plane);
    const unsigned long long n = min(*p.maybe_count, (unsigned long long)p.maybe_capacity);
    const HarmGeom g = geom_of(p);
    for (unsigned long long q = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; q < n;
         q += (unsigned long long)gridDim.x * blockDim.x) {
        const uint2 rec = p.maybe[q];
        exact_fundamental(P, g, sthr, (int64_t)rec.x, (int)rec.y);
    }
}

cudaError_t launch_harmonic(int plane_is_bf16, bool build_max, const HarmParams& p, cudaStream_t st,
                            int* launches) {
    *launches = 0;
    cudaError_t e = cudaMemsetAsync(p.count, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(p.maybe_count, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    if (p.r_lo >= p.nbins) return cudaSuccess;
    if (build_max) {
        dim3 grid((unsigned)((p.mpitch + 255) / 256), (unsigned)p.nz);
        if (plane_is_bf16) build_max_kernel<__nv_bfloat16><<<grid, 256, 0, st>>>(p);
        else build_max_kernel<float><<<grid, 256, 0, st>>>(p);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        ++*launches;
    }
    dim3 grid((unsigned)((p.nbins + kTile - 1) / kTile), (unsigned)p.nz), block(kHarmThreads);
    if (plane_is_bf16) prefilter_kernel<__nv_bfloat16><<<grid, block, 0, st>>>(p);
    else prefilter_kernel<float><<<grid, block, 0, st>>>(p);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ++*launches;
    if (plane_is_bf16) exact_kernel<__nv_bfloat16><<<kExactBlocks, 128, 0, st>>>(p);
    else exact_kernel<float><<<kExactBlocks, 128, 0, st>>>(p);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ++*launches;
    return cudaSuccess;
}

}  // namespace fdas

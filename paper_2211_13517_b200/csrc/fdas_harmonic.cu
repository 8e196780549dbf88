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
//                       h proves that (r, j) has no candidate without touching the plane.  Blocks of
//                       8 fundamentals in which some bound fails go to a "maybe" list.
//   pass B (exact)      one thread per listed fundamental: the plain definition above on the real
//                       plane, thresholds, local-maximum attribute, atomic slot claim.
// Results are identical to evaluating every fundamental exactly.  When the plane was not produced by
// fdas_convolve_plane of this plan (hand-made planes), M is first rebuilt from it (build_max_kernel).
#include <cuda_bf16.h>

#include "fdas_kernels.h"

namespace fdas {

constexpr int kHarmThreads = 256;
constexpr int kExactBlocks = 148 * 16;

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

// ---- pass A: upper bounds from the block-max plane.  Thread <-> one block B of 8 consecutive
// fundamentals r = 8B + i of row j (CTA = 256 blocks of one row), so harmonic k needs the min(k, 8)
// elements M[row_k][kB + ((k i) >> 3)]: with k unrolled every index is a compile-time offset and the
// whole test costs one FADD + one FSETP per (fundamental, harmonic).  A block with any U_h > T_h is
// appended to the maybe list as (B, j).
template <int K>
__device__ __forceinline__ void prefilter_step(const float* __restrict__ mrow, const unsigned B,
                                               const float thr, const int nv, float (&U)[8], bool& any) {
    const float* src = mrow + (size_t)K * B;
    constexpr int NL = K < 8 ? K : 8;
    float m[NL];
    if (nv == 8) {
#pragma unroll
        for (int q = 0; q < NL; ++q) m[q] = __ldg(src + (K <= 8 ? q : ((K * q) >> 3)));
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            U[i] += m[K <= 8 ? ((K * i) >> 3) : i];
            any = any || (U[i] > thr);
        }
    } else {   // the one block per row that straddles r = (Nb-1)/K
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (i < nv) {
                U[i] += __ldg(src + ((K * i) >> 3));
                any = any || (U[i] > thr);
            }
        }
    }
}

template <int K>
__device__ __forceinline__ void prefilter_from(const HarmParams& p, const int j, const int c2,
                                               const unsigned B, float (&U)[8], bool& any) {
    if constexpr (K <= 32) {
        if (K > p.H) return;
        const int v2 = 2 * K * j - (K - 1) * c2;          // CTA-uniform
        if (v2 < 0 || v2 > 2 * c2) return;
        const unsigned rmax = (unsigned)((p.nbins - 1) / K);   // last fundamental with harmonic K inside
        if (8u * (blockIdx.x * (unsigned)kHarmThreads) > rmax) return;   // whole CTA beyond Nb/K
        const int row = min((v2 + 1) >> 1, c2);
        const int nv = (8u * B > rmax) ? 0 : (int)min(8u, rmax - 8u * B + 1u);
        if (nv > 0) prefilter_step<K>(p.maxplane + (size_t)row * p.mpitch, B, p.thr[K - 1], nv, U, any);
        prefilter_from<K + 1>(p, j, c2, B, U, any);
    }
}

__global__ void __launch_bounds__(kHarmThreads) prefilter_kernel(const HarmParams p) {
    const int j = blockIdx.y;
    const unsigned B = blockIdx.x * (unsigned)kHarmThreads + threadIdx.x;
    if ((int64_t)B >= p.mpitch) return;
    float U[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) U[i] = 0.f;
    bool any = false;
    prefilter_from<1>(p, j, p.nz - 1, B, U, any);
    if (any && (int64_t)(8u * B + 7u) >= p.r_lo) {
        const unsigned long long slot = atomicAdd(p.maybe_count, 1ULL);
        if (slot < (unsigned long long)p.maybe_capacity) p.maybe[slot] = make_uint2(B, (unsigned)j);
        else atomicExch(p.overflow, 1u);   // handled by pass B (falls back to the full scan)
    }
}

// ---- pass B: 8 lanes per maybe record (B, j), lane i evaluates r = 8B + i by the plain definition.
// If the maybe list overflowed (pathological thresholds), every fundamental is evaluated instead.
template <typename T>
__global__ void __launch_bounds__(128) exact_kernel(const HarmParams p) {
    __shared__ float sthr[32];
    if (threadIdx.x < 32) sthr[threadIdx.x] = p.thr[threadIdx.x];
    __syncthreads();
    const T* P = reinterpret_cast<const T*>(p.plane);
    const HarmGeom g = geom_of(p);
    const unsigned long long tid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned long long nthr = (unsigned long long)gridDim.x * blockDim.x;
    if (*p.overflow == 0u) {
        const unsigned long long n = *p.maybe_count * 8ULL;
        for (unsigned long long q = tid; q < n; q += nthr) {
            const uint2 rec = p.maybe[q >> 3];
            exact_fundamental(P, g, sthr, (int64_t)rec.x * 8 + (int64_t)(q & 7), (int)rec.y);
        }
    } else {
        const unsigned long long n = (unsigned long long)p.nbins * (unsigned long long)p.nz;
        for (unsigned long long q = tid; q < n; q += nthr)
            exact_fundamental(P, g, sthr, (int64_t)(q % (unsigned long long)p.nbins),
                              (int)(q / (unsigned long long)p.nbins));
    }
}

cudaError_t launch_harmonic(int plane_is_bf16, bool build_max, const HarmParams& p, cudaStream_t st,
                            int* launches) {
    *launches = 0;
    cudaError_t e = cudaMemsetAsync(p.count, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(p.maybe_count, 0, 2 * sizeof(unsigned long long), st);   // + overflow flag
    if (e != cudaSuccess) return e;
    if (p.r_lo >= p.nbins) return cudaSuccess;
    if (build_max) {
        dim3 grid((unsigned)((p.mpitch + 255) / 256), (unsigned)p.nz);
        if (plane_is_bf16) build_max_kernel<__nv_bfloat16><<<grid, 256, 0, st>>>(p);
        else build_max_kernel<float><<<grid, 256, 0, st>>>(p);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        ++*launches;
    }
    dim3 grid((unsigned)((p.mpitch + kHarmThreads - 1) / kHarmThreads), (unsigned)p.nz), block(kHarmThreads);
    prefilter_kernel<<<grid, block, 0, st>>>(p);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ++*launches;
    if (plane_is_bf16) exact_kernel<__nv_bfloat16><<<kExactBlocks, 128, 0, st>>>(p);
    else exact_kernel<float><<<kExactBlocks, 128, 0, st>>>(p);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ++*launches;
    return cudaSuccess;
}

}  // namespace fdas

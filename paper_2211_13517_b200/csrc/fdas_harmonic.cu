// fdas_harmonic.cu -- K3, harmonic summing, thresholding and candidate compaction (BASELINE.json
// north_star "harmonic summing and thresholding"; DESIGN.md step a6, readings A12, A13, A14).
//   S_h(r,j) = sum_{k=1..h} P[row_k(j)][k r]  while k r <= Nb-1 and 0 <= v2 <= 2 c2,
//   v2 = 2 k j - (k-1) c2 (twice the row of harmonic k), c2 = nz-1, row_k = (v2+1)/2
//   (half-integers round away from zero).  A candidate (r, j, h) is emitted for every S_h > T_h.
//
// The direct evaluation is HBM-bound: the stride-k gathers touch 3.2x the plane in 32-byte sectors.
// K3 therefore works branch-and-bound on the block-max plane M[j][b] >= max P[j][8b..8b+7] (bf16, rounded
// toward +inf) that K2 writes beside the plane (1/16 of its bytes):
//   pass A (prefilter)  U_h(r,j) = sum_{k<=h} M[row_k][(k r) >> 3] >= S_h(r,j) term by term, in the
//                       same summation order, and fp32 addition is monotone -- so U_h <= T_h for all
//                       h proves that (r, j) has no candidate without touching the plane.  The few
//                       fundamentals for which some bound fails go to a "maybe" list.
//   pass B (exact)      one thread per listed fundamental: the plain definition above on the real
//                       plane, thresholds, atomic slot claim.
//   pass C (flags)      one thread per (stored candidate, neighbour): local-maximum attribute.
// Results are identical to evaluating every fundamental exactly.  When the plane was not produced by
// fdas_convolve_plane of this plan (hand-made planes), M is first rebuilt from it (build_max_kernel).
//
// Neighbour-maximised sums (FDAS_HSUM_NEIGHBOUR_MAX, reading A24):
//   S'_h(r,j) = sum_{k<=h} max_{|d| <= floor(k/2)} P[row_k(j)][k r + d]   (bins clipped to [0, Nb))
// so that a fundamental between two bins does not lose its harmonics.  The same branch-and-bound
// runs on a DILATED side plane M'[j][b] = max_{|e| <= D} M[j][b+e], D = ceil(floor(H/2) / 8) blocks: the
// window of harmonic k lies inside blocks (k r >> 3) - D .. + D, so M'[row_k][(k r) >> 3] bounds its
// maximum and pass A is unchanged; passes B and C evaluate the windowed maxima on the real plane.
#include <cuda_bf16.h>

#include <algorithm>

#include "fdas_kernels.h"

namespace fdas {

constexpr int kExactBlocks = 148 * 16;
constexpr int kFlagBlocks = 148 * 4;

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
    const unsigned short* maxplane;   // block-max side plane (bf16 bits, upper bounds), nz x mpitch
    int64_t mpitch;
    int nz, H;
};

__device__ __forceinline__ HarmGeom geom_of(const HarmParams& p) {
    HarmGeom g;
    g.nbins = p.nbins; g.pitch = p.pitch; g.r_lo = p.r_lo; g.capacity = p.capacity;
    g.cands = p.cands; g.count = p.count; g.nz = p.nz; g.H = p.H;
    g.maxplane = p.maxplane; g.mpitch = p.mpitch;
    return g;
}

// S_h at (r, j) if defined (r in [r_lo, Nb), all h harmonics inside the plane); summed k = 1..h,
// the gathers issued eight at a time.
template <typename T>
__device__ bool harmonic_sum_at(const T* P, const HarmGeom& g, int64_t r, int j, int h, float* out) {
    if (j < 0 || j >= g.nz || r < g.r_lo || r >= g.nbins) return false;
    const int c2 = g.nz - 1;
    {   // validity is monotone in k: test the deepest harmonic only
        const int v2 = 2 * h * j - (h - 1) * c2;
        if (v2 < 0 || v2 > 2 * c2 || (int64_t)h * r > g.nbins - 1) return false;
    }
    float S = 0.f;
    for (int k0 = 1; k0 <= h; k0 += 8) {
        float v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int k = k0 + q;
            v[q] = 0.f;
            if (k <= h) {
                const int row = min((2 * k * j - (k - 1) * c2 + 1) >> 1, c2);
                v[q] = ldp(P + (size_t)row * g.pitch + (size_t)k * r);
            }
        }
#pragma unroll
        for (int q = 0; q < 8; ++q)
            if (k0 + q <= h) S += v[q];
    }
    *out = S;
    return true;
}

__device__ __forceinline__ void emit_candidate(const HarmGeom& g, int64_t r, int j, int h, float S) {
    const unsigned long long slot = atomicAdd(g.count, 1ULL);   // the true count
    if ((int64_t)slot >= g.capacity) return;
    fdas_cand_t c;
    c.r = (uint32_t)r;
    c.zidx = (int16_t)j;
    c.h = (uint16_t)h;
    c.power = S;
    c.flags = 1u;   // local-maximum attribute: cleared by flag_kernel if a neighbour beats it
    g.cands[slot] = c;
}

// The plain definition for one fundamental: all h, thresholds, slot claim; sums stay in k order.
// Harmonics 1..4 are gathered first (4 DRAM sectors); the deeper sums are then bounded from above by
// continuing the same running sum with the block maxima M (an L2-resident side plane) in place of the
// plane values -- term by term M >= P and fp32 addition is monotone -- and only if such a bound exceeds
// its threshold are harmonics 5.. gathered from the plane, 8 at a time (independent addresses).  Most
// fundamentals the prefilter lets through are settled by the first four gathers.
template <typename T>
__device__ __noinline__ void exact_fundamental(const T* P, const HarmGeom g, const float* thr,
                                               int64_t r, int j) {
    if (r < g.r_lo || r >= g.nbins) return;
    const int c2 = g.nz - 1;
    int hmax = 0;   // number of defined harmonics
    for (int h = 1; h <= g.H; ++h) {
        const int v2 = 2 * h * j - (h - 1) * c2;
        if (v2 < 0 || v2 > 2 * c2 || (int64_t)h * r > g.nbins - 1) break;
        hmax = h;
    }
    auto row_of = [&](int h) { return min((2 * h * j - (h - 1) * c2 + 1) >> 1, c2); };
    float S = 0.f;
    {
        float v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int h = 1 + q;
            v[q] = (h <= hmax) ? ldp(P + (size_t)row_of(h) * g.pitch + (size_t)h * r) : 0.f;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int h = 1 + q;
            if (h > hmax) break;
            S += v[q];
            if (S > thr[h - 1]) emit_candidate(g, r, j, h, S);
        }
    }
    if (hmax <= 4) return;
    {   // can any deeper sum still exceed its threshold?
        float U = S;
        bool deeper = false;
        for (int h0 = 5; h0 <= hmax && !deeper; h0 += 8) {
            unsigned short m[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int h = h0 + q;
                m[q] = (h <= hmax) ? __ldg(g.maxplane + (size_t)row_of(h) * g.mpitch + (size_t)(((int64_t)h * r) >> 3)) : 0;
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int h = h0 + q;
                if (h > hmax) break;
                U += __uint_as_float((unsigned)m[q] << 16);
                if (U > thr[h - 1]) deeper = true;
            }
        }
        if (!deeper) return;
    }
    for (int h0 = 5; h0 <= hmax; h0 += 8) {
        float v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int h = h0 + q;
            v[q] = (h <= hmax) ? ldp(P + (size_t)row_of(h) * g.pitch + (size_t)h * r) : 0.f;
        }
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int h = h0 + q;
            if (h > hmax) break;
            S += v[q];
            if (S > thr[h - 1]) emit_candidate(g, r, j, h, S);
        }
    }
}

// Neighbour-maximised variant of the plain definition (reading A24): harmonic h is the largest plane
// value within floor(h/2) bins of h r (clipped to the plane); sums stay in k order.
template <typename T>
__device__ __forceinline__ float window_max(const T* prow, int64_t c, int w, int64_t nbins) {
    const int64_t lo = max((int64_t)0, c - w), hi = min(nbins - 1, c + w);
    float best = ldp(prow + lo);
    for (int64_t x = lo + 1; x <= hi; ++x) best = fmaxf(best, ldp(prow + x));
    return best;
}
template <typename T>
__device__ bool harmonic_sum_nbr_at(const T* P, const HarmGeom& g, int64_t r, int j, int h, float* out) {
    if (j < 0 || j >= g.nz || r < g.r_lo || r >= g.nbins) return false;
    const int c2 = g.nz - 1;
    {
        const int v2 = 2 * h * j - (h - 1) * c2;
        if (v2 < 0 || v2 > 2 * c2 || (int64_t)h * r > g.nbins - 1) return false;
    }
    float S = 0.f;
    for (int k = 1; k <= h; ++k) {
        const int row = min((2 * k * j - (k - 1) * c2 + 1) >> 1, c2);
        S += window_max(P + (size_t)row * g.pitch, (int64_t)k * r, k >> 1, g.nbins);
    }
    *out = S;
    return true;
}
template <typename T>
__device__ __noinline__ void exact_fundamental_nbr(const T* P, const HarmGeom g, const float* thr, int64_t r,
                                                   int j) {
    if (r < g.r_lo || r >= g.nbins) return;
    const int c2 = g.nz - 1;
    float S = 0.f;
    for (int h = 1; h <= g.H; ++h) {
        const int v2 = 2 * h * j - (h - 1) * c2;
        if (v2 < 0 || v2 > 2 * c2 || (int64_t)h * r > g.nbins - 1) break;
        const int row = min((v2 + 1) >> 1, c2);
        S += window_max(P + (size_t)row * g.pitch, (int64_t)h * r, h >> 1, g.nbins);
        if (S > thr[h - 1]) emit_candidate(g, r, j, h, S);
    }
}

// bf16 bit pattern of a non-negative power rounded toward +inf, and back.
__device__ __forceinline__ unsigned short bf16_up(float v) {
    return (unsigned short)((__float_as_uint(v) + 0xffffu) >> 16);
}
__device__ __forceinline__ float bf16_lo(unsigned w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(unsigned w) { return __uint_as_float(w & 0xffff0000u); }

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
    p.maxplane[(size_t)j * p.mpitch + b] = bf16_up(m);
}

// ---- M' = M dilated by D blocks on either side (neighbour-maximised sums): one thread per block.
__global__ void __launch_bounds__(256) dilate_max_kernel(const unsigned short* __restrict__ src,
                                                         unsigned short* __restrict__ dst, int64_t mpitch, int D) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= mpitch) return;
    const unsigned short* row = src + (size_t)blockIdx.y * mpitch;
    unsigned m = 0;     // bf16 patterns of non-negative values order like the values
    for (int64_t e = max((int64_t)0, b - D); e <= min(mpitch - 1, b + D); ++e) m = max(m, (unsigned)__ldg(row + e));
    dst[(size_t)blockIdx.y * mpitch + b] = (unsigned short)m;
}

// ---- pass A: upper bounds from the block-max plane.
// Thread <-> 4 consecutive blocks of M = 32 consecutive fundamentals r = 32 Q + i of row j, so that
// harmonic k <= 8 is k contiguous 128-bit loads (M[row_k][4kQ .. 4kQ+4k-1]) and every fundamental
// picks element (k i) >> 3 of them -- a compile-time register choice once k and i are unrolled.  The
// loads of harmonics 1..4 (then 5-6, 7-8, then one harmonic at a time) are all issued before the
// first add: the kernel moves < 1 GB and would otherwise be bound by DRAM latency, not bandwidth.
// One FADD, one FSETP and one predicated OR per (fundamental, harmonic) for h >= 3 (h = 1, 2 are
// evaluated once per block / half block); fundamentals with any U_h > T_h go to the maybe list as (r, j).
constexpr int kPfThreads = 128;

// Harmonic K for the 32 fundamentals of quad-block Q, all of them valid (K (32Q+31) <= Nb-1).
template <int K, int NV>
__device__ __forceinline__ void pf_load(const unsigned short* __restrict__ mrow, const unsigned Q,
                                        const bool on, float (&m)[NV]) {
    if constexpr (K <= 8) {
        static_assert(NV == 4 * K, "k <= 8 loads 4k contiguous elements");
        const uint2* src = reinterpret_cast<const uint2*>(mrow + (size_t)4 * K * Q);   // 8K bytes, 8-byte aligned
#pragma unroll
        for (int q = 0; q < K; ++q) {
            uint2 v = make_uint2(0u, 0u);
            if (on) v = __ldg(src + q);
            m[4 * q] = bf16_lo(v.x); m[4 * q + 1] = bf16_hi(v.x);
            m[4 * q + 2] = bf16_lo(v.y); m[4 * q + 3] = bf16_hi(v.y);
        }
    } else {
        static_assert(NV == 32, "k > 8 gathers one element per fundamental");
        const unsigned short* src = mrow + (size_t)4 * K * Q;
#pragma unroll
        for (int i = 0; i < 32; ++i) m[i] = on ? bf16_lo(__ldg(src + ((K * i) >> 3))) : 0.f;
    }
}

template <int K, int NV>
__device__ __forceinline__ void pf_add(const float (&m)[NV], const float thr, const bool on,
                                       float (&U)[32], unsigned& flagged) {
    if (on) {
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            U[i] += m[K <= 8 ? ((K * i) >> 3) : i];
            if (U[i] > thr) flagged |= 1u << i;
        }
    }
}

struct PfRow { const unsigned short* mrow; float thr; };

__device__ __forceinline__ PfRow pf_row(const HarmParams& p, const int j, const int k) {
    const int c2 = p.nz - 1;
    const int v2 = 2 * k * j - (k - 1) * c2;   // only called for k <= hz: v2 is in range
    PfRow r;
    r.mrow = p.maxplane + (size_t)min((v2 + 1) >> 1, c2) * p.mpitch;
    r.thr = p.thr[k - 1];
    return r;
}

// Harmonic K > 8 of the 32 fundamentals of quad-block Q: the thread's slice M[row_K][4KQ .. 4KQ+4K-1]
// (8K bytes) is read with 64-bit loads in two halves -- fundamentals 0..15 pick elements
// (K i) >> 3 < 2K (words 0..K-1), fundamentals 16..31 elements >= 2K (words K..2K-1) -- instead of one
// 16-bit gather per fundamental: half the load instructions, K + 2 live registers instead of 32.
template <int K>
__device__ __forceinline__ void pf_deep(const unsigned short* __restrict__ mrow, const unsigned Q,
                                        const float thr, float (&U)[32], unsigned& flagged) {
    const unsigned* words = reinterpret_cast<const unsigned*>(mrow + (size_t)4 * K * Q);   // 8-byte aligned
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        constexpr int kPairs = K / 2 + 1;                 // 64-bit loads covering the half's K words
        const int w0 = half ? (K & ~1) : 0;               // first word loaded (even: aligned)
        unsigned wv[2 * kPairs];
#pragma unroll
        for (int c = 0; c < kPairs; ++c) {
            // the last pair of the second half may reach one word past the slice when K is even
            if (w0 + 2 * c + 1 < 2 * K) {
                const uint2 v = __ldg(reinterpret_cast<const uint2*>(words + w0) + c);
                wv[2 * c] = v.x;
                wv[2 * c + 1] = v.y;
            } else if (w0 + 2 * c < 2 * K) {
                wv[2 * c] = __ldg(words + w0 + 2 * c);
                wv[2 * c + 1] = 0u;
            } else {
                wv[2 * c] = wv[2 * c + 1] = 0u;
            }
        }
#pragma unroll
        for (int ii = 0; ii < 16; ++ii) {
            const int i = 16 * half + ii;
            const int e = (K * i) >> 3;                   // element of the slice (compile time)
            const unsigned w = wv[(e >> 1) - w0];
            U[i] += (e & 1) ? bf16_hi(w) : bf16_lo(w);
            if (U[i] > thr) flagged |= 1u << i;
        }
    }
}

template <int K>
__device__ __forceinline__ void pf_single_from(const HarmParams& p, const int j, const unsigned Q,
                                               const int he_max, const int he, float (&U)[32],
                                               unsigned& flagged) {
    if constexpr (K <= 32) {
        if (K > he_max) return;                 // CTA-uniform: no thread of this CTA goes deeper
        const PfRow r = pf_row(p, j, K);
        if constexpr (K <= 8) {
            float m[4 * K];
            pf_load<K>(r.mrow, Q, he >= K, m);
            pf_add<K>(m, r.thr, he >= K, U, flagged);
        } else {
            if (he >= K) pf_deep<K>(r.mrow, Q, r.thr, U, flagged);
        }
        pf_single_from<K + 1>(p, j, Q, he_max, he, U, flagged);
    }
}

// Fundamentals of quad-block Q flagged by pass A go to the maybe list as (r, j).
__device__ __forceinline__ void pf_emit(const HarmParams& p, const unsigned Q, const int j, unsigned flagged) {
    // r < r_lo never yields candidates
    if (32 * (int64_t)Q < p.r_lo) {
        const int64_t cut = p.r_lo - 32 * (int64_t)Q;
        flagged = (cut >= 32) ? 0u : (flagged & ~((1u << (int)cut) - 1u));
    }
    if (flagged) {
        const int n = __popc(flagged);
        const unsigned long long base = atomicAdd(p.maybe_count, (unsigned long long)n);
        if (base + (unsigned long long)n <= (unsigned long long)p.maybe_capacity) {
            unsigned long long slot = base;
            while (flagged) {
                const int i = __ffs(flagged) - 1;
                flagged &= flagged - 1;
                p.maybe[slot++] = make_uint2(32u * Q + (unsigned)i, (unsigned)j);
            }
        } else {
            atomicExch(p.overflow, 1u);   // pass B then falls back to the full scan
        }
    }
}

// Rows with at most kShallowDepth = 4 harmonics inside the plane (|z| > zmax/5: the nlow first and the
// nlow last rows, four fifths of the plane).  Harmonic k picks block (k i) >> 3 for fundamental i of a
// block of 8, so U_1 is the same for all 8 fundamentals, U_2 for halves, U_3 takes 4 and U_4 5 distinct
// values per block: 12 sums and compares stand for 32.  A thread streams 8 blocks (64 fundamentals) of
// M[j] and the 8k blocks of M[row_k] they map to; few registers, every load issued up front.
constexpr int kPfShallowThreads = 256;
constexpr int kShallowDepth = 4;

__device__ __forceinline__ float bf16_at(const uint4 (&w)[4], const int e) {   // element e of up to 32 (static e)
    const uint4 v = w[e >> 3];
    const unsigned x = ((e >> 1) & 3) == 0 ? v.x : ((e >> 1) & 3) == 1 ? v.y : ((e >> 1) & 3) == 2 ? v.z : v.w;
    return (e & 1) ? bf16_hi(x) : bf16_lo(x);
}

// DMAX = 2 | 4: deepest harmonic of the rows this instance scans, rows [ja, jb) and their mirror images
// [nz - jb, nz - ja) (the two-harmonic instance needs a third of the registers of the four-harmonic one).
template <int DMAX>
__global__ void __launch_bounds__(kPfShallowThreads) prefilter_shallow_kernel(const HarmParams p, const int ja,
                                                                              const int jb) {
    const int y = blockIdx.y;
    const int j = y < jb - ja ? ja + y : p.nz - jb + (y - (jb - ja));
    const int c2 = p.nz - 1;
    const unsigned O = blockIdx.x * (unsigned)kPfShallowThreads + threadIdx.x;   // octet of blocks
    if (O >= (unsigned)(p.mpitch >> 3)) return;
    const unsigned last = (unsigned)(p.nbins - 1);
    const int d = abs(2 * j - c2);
    const int hz = min(DMAX, d == 0 ? p.H : min(p.H, c2 / d));   // 1 .. DMAX here (CTA-uniform)
    const PfRow r1 = pf_row(p, j, 1);
    uint4 m1[4], m2[4], m3[4], m4[4];   // (only the first DMAX arrays are live)
    m1[0] = __ldg(reinterpret_cast<const uint4*>(r1.mrow) + O);
    if (hz <= 1 && r1.thr >= 0.f) {
        // one harmonic only (half of the plane's rows): M > T_1 on the bf16 bit patterns.  For
        // non-negative values the order of the patterns is the order of the values, and with
        // tb = pattern of T_1 truncated to bf16, M > T_1 <=> pattern(M) > tb (M is a bf16 value).
        // (A negative T_1 passes every point, M = 0 included: no early exit then.)
        const unsigned tb = __float_as_uint(r1.thr) >> 16;
        const unsigned tb2 = tb | (tb << 16);
        if ((__vcmpgtu2(m1[0].x, tb2) | __vcmpgtu2(m1[0].y, tb2) | __vcmpgtu2(m1[0].z, tb2) |
             __vcmpgtu2(m1[0].w, tb2)) == 0u)
            return;                                   // nothing above threshold: almost every thread
    }
    // dep: harmonics inside the plane for all 64 fundamentals of this thread
    const int dep = (int)min((unsigned)hz, last / (64u * O + 63u));
    PfRow r2 = r1, r3 = r1, r4 = r1;
    if (hz >= 2) r2 = pf_row(p, j, 2);
    if (DMAX >= 3 && hz >= 3) r3 = pf_row(p, j, 3);
    if (DMAX >= 4 && hz >= 4) r4 = pf_row(p, j, 4);
    if (dep >= 2) {
#pragma unroll
        for (int c = 0; c < 2; ++c) m2[c] = __ldg(reinterpret_cast<const uint4*>(r2.mrow) + 2 * O + c);
    }
    if (DMAX >= 3 && dep >= 3) {
#pragma unroll
        for (int c = 0; c < 3; ++c) m3[c] = __ldg(reinterpret_cast<const uint4*>(r3.mrow) + 3 * O + c);
    }
    if (DMAX >= 4 && dep >= 4) {
#pragma unroll
        for (int c = 0; c < 4; ++c) m4[c] = __ldg(reinterpret_cast<const uint4*>(r4.mrow) + 4 * O + c);
    }
    unsigned f[2] = {0u, 0u};   // flags of fundamentals 64 O + 32 t + i
#pragma unroll
    for (int q = 0; q < 8; ++q) {          // block q: fundamentals 8q..8q+7
        const int sh = 8 * (q & 3);
        unsigned fl = 0u;
        const float u1 = bf16_at(m1, q);
        if (u1 > r1.thr) fl |= 0xffu;
        if (dep >= 2) {
            // U_2: fundamentals 0..3 -> block 2q, 4..7 -> block 2q+1 of row_2
            const float u2[2] = {u1 + bf16_at(m2, 2 * q), u1 + bf16_at(m2, 2 * q + 1)};
            if (u2[0] > r2.thr) fl |= 0x0fu;
            if (u2[1] > r2.thr) fl |= 0xf0u;
            if (DMAX >= 3 && dep >= 3) {
                // U_3: (i >> 2, (3 i) >> 3) = (0,0) for i = 0,1,2; (0,1) for 3; (1,1) for 4,5; (1,2) for 6,7
                const float u3[4] = {u2[0] + bf16_at(m3, 3 * q), u2[0] + bf16_at(m3, 3 * q + 1),
                                     u2[1] + bf16_at(m3, 3 * q + 1), u2[1] + bf16_at(m3, 3 * q + 2)};
                if (u3[0] > r3.thr) fl |= 0x07u;
                if (u3[1] > r3.thr) fl |= 0x08u;
                if (u3[2] > r3.thr) fl |= 0x30u;
                if (u3[3] > r3.thr) fl |= 0xc0u;
                if (DMAX >= 4 && dep >= 4) {
                    // U_4 adds block i >> 1 of row_4: i = 0,1 | 2 | 3 | 4,5 | 6,7
                    if (u3[0] + bf16_at(m4, 4 * q) > r4.thr) fl |= 0x03u;
                    if (u3[0] + bf16_at(m4, 4 * q + 1) > r4.thr) fl |= 0x04u;
                    if (u3[1] + bf16_at(m4, 4 * q + 1) > r4.thr) fl |= 0x08u;
                    if (u3[2] + bf16_at(m4, 4 * q + 2) > r4.thr) fl |= 0x30u;
                    if (u3[3] + bf16_at(m4, 4 * q + 3) > r4.thr) fl |= 0xc0u;
                }
            }
        }
        f[q >> 2] |= fl << sh;
    }
    if (dep < hz) {
        // the thread that straddles r = (Nb-1)/(dep+1): harmonic dep+1 exists for its first
        // fundamentals only (no deeper one can: see DESIGN.md K3); U_dep is rebuilt in k order
        const int k = dep + 1;
        const unsigned rmax = last / (unsigned)k;
        if (64u * O <= rmax) {
            const int nv = (int)min(64u, rmax - 64u * O + 1u);
            const float thr_k = p.thr[k - 1];
            for (int i = 0; i < nv; ++i) {
                float u = 0.f;
                for (int kk = 1; kk <= k; ++kk) {
                    const PfRow rk = pf_row(p, j, kk);
                    u += bf16_lo(__ldg(rk.mrow + (size_t)8 * kk * O + ((kk * i) >> 3)));
                }
                if (u > thr_k) f[i >> 5] |= 1u << (i & 31);
            }
        }
    }
    pf_emit(p, 2u * O, j, f[0]);
    pf_emit(p, 2u * O + 1u, j, f[1]);
}

__global__ void __launch_bounds__(kPfThreads, 8) prefilter_kernel(const HarmParams p, const int nlow) {
    const int j = nlow + blockIdx.y;   // the rows with more than kShallowDepth harmonics (|z| <= zmax/5)
    const int c2 = p.nz - 1;
    const unsigned Q0 = blockIdx.x * (unsigned)kPfThreads;
    const unsigned Q = Q0 + threadIdx.x;
    const unsigned nquad = (unsigned)(p.mpitch >> 2);   // nbins / 32
    if (Q >= nquad) return;
    const unsigned last = (unsigned)(p.nbins - 1);
    // hz: harmonics inside the plane in z for this row (CTA-uniform): twice the row of harmonic k is
    // v2 = k d + c2 with d = 2 j - c2, and 0 <= v2 <= 2 c2  <=>  k |d| <= c2
    const int d = abs(2 * j - c2);
    const int hz = d == 0 ? p.H : min(p.H, c2 / d);
    // he: harmonics for which all 32 fundamentals of this thread are inside the plane in r
    const int he = (int)min((unsigned)hz, last / (32u * Q + 31u));
    const int he_max = (int)min((unsigned)hz, last / (32u * Q0 + 31u));   // deepest in this CTA
    float U[32];
    unsigned flagged = 0u;   // bit i: some U_h of fundamental 32 Q + i exceeds T_h

    {   // harmonics 1..4: ten 128-bit loads in flight
        const PfRow r1 = pf_row(p, j, 1);
        float m1[4], m2[8], m3[12], m4[16];
        pf_load<1>(r1.mrow, Q, true, m1);
        PfRow r2 = r1, r3 = r1, r4 = r1;
        if (he_max >= 2) { r2 = pf_row(p, j, 2); pf_load<2>(r2.mrow, Q, he >= 2, m2); }
        if (he_max >= 3) { r3 = pf_row(p, j, 3); pf_load<3>(r3.mrow, Q, he >= 3, m3); }
        if (he_max >= 4) { r4 = pf_row(p, j, 4); pf_load<4>(r4.mrow, Q, he >= 4, m4); }
        // harmonic k picks block (k i) >> 3 for fundamental i of a block of 8: U_1 is the same for all
        // 8, U_2 for the 4 of a half block, U_3 takes 4 and U_4 5 distinct values per block -- 12 sums
        // and compares per block stand for 32 (h <= 4 are 90 % of all (r, j, h) triples of the plane)
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (m1[q] > r1.thr) flagged |= 0xffu << (8 * q);
        float u2[8];
#pragma unroll
        for (int gq = 0; gq < 8; ++gq) u2[gq] = m1[gq >> 1];
        if (he >= 2) {
#pragma unroll
            for (int gq = 0; gq < 8; ++gq) {
                u2[gq] += m2[gq];
                if (u2[gq] > r2.thr) flagged |= 0xfu << (4 * gq);
            }
        }
        if (he >= 3) {
            float u3[16];
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                // (i >> 2, (3 i) >> 3) = (0,0) for i = 0,1,2; (0,1) for 3; (1,1) for 4,5; (1,2) for 6,7
                u3[4 * b + 0] = u2[2 * b] + m3[3 * b];
                u3[4 * b + 1] = u2[2 * b] + m3[3 * b + 1];
                u3[4 * b + 2] = u2[2 * b + 1] + m3[3 * b + 1];
                u3[4 * b + 3] = u2[2 * b + 1] + m3[3 * b + 2];
                if (u3[4 * b + 0] > r3.thr) flagged |= 0x07u << (8 * b);
                if (u3[4 * b + 1] > r3.thr) flagged |= 0x08u << (8 * b);
                if (u3[4 * b + 2] > r3.thr) flagged |= 0x30u << (8 * b);
                if (u3[4 * b + 3] > r3.thr) flagged |= 0xc0u << (8 * b);
            }
            if (he >= 4) {
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    // U_4 adds block i >> 1 of row_4: i = 0,1 | 2 | 3 | 4,5 | 6,7
                    const float v0 = u3[4 * b + 0] + m4[4 * b], v1 = u3[4 * b + 0] + m4[4 * b + 1];
                    const float v2 = u3[4 * b + 1] + m4[4 * b + 1], v3 = u3[4 * b + 2] + m4[4 * b + 2];
                    const float v4 = u3[4 * b + 3] + m4[4 * b + 3];
                    if (v0 > r4.thr) flagged |= 0x03u << (8 * b);
                    if (v1 > r4.thr) flagged |= 0x04u << (8 * b);
                    if (v2 > r4.thr) flagged |= 0x08u << (8 * b);
                    if (v3 > r4.thr) flagged |= 0x30u << (8 * b);
                    if (v4 > r4.thr) flagged |= 0xc0u << (8 * b);
                    U[8 * b + 0] = v0; U[8 * b + 1] = v0; U[8 * b + 2] = v1; U[8 * b + 3] = v2;
                    U[8 * b + 4] = v3; U[8 * b + 5] = v3; U[8 * b + 6] = v4; U[8 * b + 7] = v4;
                }
            } else {
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    U[8 * b + 0] = u3[4 * b]; U[8 * b + 1] = u3[4 * b]; U[8 * b + 2] = u3[4 * b];
                    U[8 * b + 3] = u3[4 * b + 1];
                    U[8 * b + 4] = u3[4 * b + 2]; U[8 * b + 5] = u3[4 * b + 2];
                    U[8 * b + 6] = u3[4 * b + 3]; U[8 * b + 7] = u3[4 * b + 3];
                }
            }
        } else {
#pragma unroll
            for (int i = 0; i < 32; ++i) U[i] = u2[i >> 2];
        }
    }
    if (he_max >= 5) {   // harmonics 5, 6: eleven loads in flight
        const PfRow r5 = pf_row(p, j, 5);
        float m5[20], m6[24];
        pf_load<5>(r5.mrow, Q, he >= 5, m5);
        PfRow r6 = r5;
        if (he_max >= 6) { r6 = pf_row(p, j, 6); pf_load<6>(r6.mrow, Q, he >= 6, m6); }
        pf_add<5>(m5, r5.thr, he >= 5, U, flagged);
        if (he_max >= 6) pf_add<6>(m6, r6.thr, he >= 6, U, flagged);
    }
    pf_single_from<7>(p, j, Q, he_max, he, U, flagged);

    // the (at most a few) harmonics for which only some of the 32 fundamentals are inside the plane
    for (int k = he + 1; k <= hz; ++k) {
        const unsigned rmax = last / (unsigned)k;
        if (32u * Q > rmax) break;
        const int nv = (int)min(32u, rmax - 32u * Q + 1u);
        const PfRow r = pf_row(p, j, k);
        const unsigned short* src = r.mrow + (size_t)k * 4 * Q;
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            if (i < nv) {
                U[i] += bf16_lo(__ldg(src + ((k * i) >> 3)));
                if (U[i] > r.thr) flagged |= 1u << i;
            }
        }
    }

    pf_emit(p, Q, j, flagged);
}

// ---- pass B: one thread per maybe record (r, j): the plain definition on the real plane.
// If the maybe list overflowed (pathological thresholds), every fundamental is evaluated instead.
template <typename T, int NBR>
__global__ void __launch_bounds__(128) exact_kernel(const HarmParams p) {
    __shared__ float sthr[32];
    if (threadIdx.x < 32) sthr[threadIdx.x] = p.thr[threadIdx.x];
    __syncthreads();
    const T* P = reinterpret_cast<const T*>(p.plane);
    const HarmGeom g = geom_of(p);
    const unsigned long long tid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned long long nthr = (unsigned long long)gridDim.x * blockDim.x;
    if (*p.overflow == 0u) {
        const unsigned long long n = *p.maybe_count;
        for (unsigned long long q = tid; q < n; q += nthr) {
            const uint2 rec = p.maybe[q];
            if (NBR) exact_fundamental_nbr(P, g, sthr, (int64_t)rec.x, (int)rec.y);
            else exact_fundamental(P, g, sthr, (int64_t)rec.x, (int)rec.y);
        }
    } else {
        const unsigned long long n = (unsigned long long)p.nbins * (unsigned long long)p.nz;
        for (unsigned long long q = tid; q < n; q += nthr) {
            const int64_t r = (int64_t)(q % (unsigned long long)p.nbins);
            const int j = (int)(q / (unsigned long long)p.nbins);
            if (NBR) exact_fundamental_nbr(P, g, sthr, r, j);
            else exact_fundamental(P, g, sthr, r, j);
        }
    }
}

// ---- pass C: local-maximum attribute, one thread per (stored candidate, neighbour): the flag is
// cleared unless S_h(r,j) >= S_h at the neighbour (r+dr, j+dj) where that is defined, strictly >
// for the neighbours that precede (j, r) lexicographically (reading A14).
template <typename T, int NBR>
__global__ void __launch_bounds__(128) flag_kernel(const HarmParams p) {
    const T* P = reinterpret_cast<const T*>(p.plane);
    const HarmGeom g = geom_of(p);
    const unsigned long long stored = min(*p.count, (unsigned long long)p.capacity);
    const unsigned long long n = stored * 8ULL;
    for (unsigned long long q = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; q < n;
         q += (unsigned long long)gridDim.x * blockDim.x) {
        const fdas_cand_t c = p.cands[q >> 3];
        const int nb = (int)(q & 7);
        const int idx = nb < 4 ? nb : nb + 1;          // skip the centre of the 3 x 3 stencil
        const int dj = idx / 3 - 1, dr = idx % 3 - 1;
        float nv;
        if (!(NBR ? harmonic_sum_nbr_at(P, g, (int64_t)c.r + dr, (int)c.zidx + dj, (int)c.h, &nv)
                  : harmonic_sum_at(P, g, (int64_t)c.r + dr, (int)c.zidx + dj, (int)c.h, &nv)))
            continue;
        const bool precedes = (dj < 0) || (dj == 0 && dr < 0);
        if (precedes ? !(c.power > nv) : !(c.power >= nv)) atomicAnd(&p.cands[q >> 3].flags, ~1u);
    }
}

cudaError_t launch_harmonic(int plane_is_bf16, bool build_max, const HarmParams& p_in, cudaStream_t st,
                            int* launches) {
    *launches = 0;
    HarmParams p = p_in;
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
    if (p.nbr) {
        // the prefilter (and nothing else) scans the dilated side plane from here on
        if (!p.maxplane_nbr) return cudaErrorInvalidValue;
        const int D = ((p.H >> 1) + 7) >> 3;
        dim3 grid((unsigned)((p.mpitch + 255) / 256), (unsigned)p.nz);
        dilate_max_kernel<<<grid, 256, 0, st>>>(p.maxplane, p.maxplane_nbr, p.mpitch, D);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        ++*launches;
        p.maxplane = p.maxplane_nbr;
    }
    // rows j < nlow and j >= nz - nlow have at most kShallowDepth harmonics inside the plane (reading
    // A12), rows j < nlow2 and j >= nz - nlow2 at most two
    int nlow = 0, nlow2 = 0;
    if ((p.mpitch & 7) == 0) {   // the shallow passes stream octets of blocks
        const int c2 = p.nz - 1;
        auto hz_of = [&](int j) { const int d = c2 - 2 * j; return d == 0 ? p.H : std::min(p.H, c2 / d); };
        while (2 * nlow2 < p.nz - 1 && hz_of(nlow2) <= 2) ++nlow2;
        nlow = nlow2;
        while (2 * nlow < p.nz - 1 && hz_of(nlow) <= kShallowDepth) ++nlow;
    }
    const unsigned sgx = (unsigned)((p.mpitch / 8 + kPfShallowThreads - 1) / kPfShallowThreads);
    if (nlow2 > 0) {
        prefilter_shallow_kernel<2><<<dim3(sgx, (unsigned)(2 * nlow2)), kPfShallowThreads, 0, st>>>(p, 0, nlow2);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        ++*launches;
    }
    if (nlow > nlow2) {
        prefilter_shallow_kernel<4><<<dim3(sgx, (unsigned)(2 * (nlow - nlow2))), kPfShallowThreads, 0, st>>>(p, nlow2, nlow);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        ++*launches;
    }
    if (p.nz - 2 * nlow > 0) {
        dim3 grid((unsigned)((p.mpitch / 4 + kPfThreads - 1) / kPfThreads), (unsigned)(p.nz - 2 * nlow)), block(kPfThreads);
        prefilter_kernel<<<grid, block, 0, st>>>(p, nlow);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        ++*launches;
    }
    if (p.nbr) {
        if (plane_is_bf16) exact_kernel<__nv_bfloat16, 1><<<kExactBlocks, 128, 0, st>>>(p);
        else exact_kernel<float, 1><<<kExactBlocks, 128, 0, st>>>(p);
    } else {
        if (plane_is_bf16) exact_kernel<__nv_bfloat16, 0><<<kExactBlocks, 128, 0, st>>>(p);
        else exact_kernel<float, 0><<<kExactBlocks, 128, 0, st>>>(p);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ++*launches;
    if (p.capacity > 0) {
        if (p.nbr) {
            if (plane_is_bf16) flag_kernel<__nv_bfloat16, 1><<<kFlagBlocks, 128, 0, st>>>(p);
            else flag_kernel<float, 1><<<kFlagBlocks, 128, 0, st>>>(p);
        } else {
            if (plane_is_bf16) flag_kernel<__nv_bfloat16, 0><<<kFlagBlocks, 128, 0, st>>>(p);
            else flag_kernel<float, 0><<<kFlagBlocks, 128, 0, st>>>(p);
        }
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        ++*launches;
    }
    return cudaSuccess;
}

}  // namespace fdas

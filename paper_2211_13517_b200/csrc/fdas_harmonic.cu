// fdas_harmonic.cu -- K3, harmonic summing, thresholding and candidate compaction (BASELINE.json
// north_star "harmonic summing and thresholding"; DESIGN.md step a6, readings A12, A13, A14).
//   S_h(r,j) = sum_{k=1..h} P[row_k(j)][k r]  while k r <= Nb-1 and 0 <= v2 <= 2 c2,
//   v2 = 2 k j - (k-1) c2 (twice the row of harmonic k), c2 = nz-1, row_k = (v2+1)/2
//   (half-integers round away from zero).  A candidate (r, j, h) is emitted for every S_h > T_h.
//
// The direct evaluation is HBM-bound: the stride-k gathers touch 3.2x the plane in 32-byte sectors.
// K3 therefore works branch-and-bound on the block-max plane M[j][b] >= max P[j][8b..8b+7] (16-bit codes in
// units of 1/8, rounded up, fdas_maxcode.h) that K2 writes beside the plane (1/16 of its bytes):
//   pass A (prefilter)  U_h(r,j) = sum_{k<=h} M[row_k][(k r) >> 3] >= S_h(r,j) term by term (exact integer
//                       sums of the codes, two fundamentals per 32-bit add) -- so U_h <= T_h for all
//                       h proves that (r, j) has no candidate without touching the plane.  The few
//                       fundamentals for which some bound fails go to a "maybe" list.  Where a fundamental
//                       has at most four harmonics (most of the plane) the same bound is first taken on
//                       coarse blocks of 64 columns (M2 = max of 8 codes of M, level 0), and only the coarse
//                       blocks that fail are looked at block by block (level 1, by the same thread); the rest -- the first fifth
//                       of the 39 rows with |z| <= zmax/5 at the SKA size -- is prefilter_kernel's.
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
#include <cmath>

#include "fdas_kernels.h"
#include "fdas_maxcode.h"

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
    const unsigned short* maxplane;   // block-max side plane (codes of fdas_maxcode.h), nz x mpitch
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
                                               int64_t r, int j, unsigned hint) {
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
    if (hint != 0xffffu) {
        // the prefilter's hint (pf_emit_warp): 8 S_h <= 8 S_4 + (U_h - U_4) <= ceil(8 S_4 (1 + 2^-20)) + E + tq_h
        const float s8 = S * (8.0f * (1.0f + 9.5367431640625e-7f));
        if (s8 < 60000.f && (int)ceilf(s8) + ((int)hint - 8192) <= 0) return;
        // (not ruled out: the bound below would say the same -- straight to the gathers)
    } else {   // no hint (block level, straddling threads, full scan): can any deeper sum still exceed its threshold?
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
                U += (float)m[q] * (1.0f / kMaxCodeScale);
                if (U > thr[h - 1] || m[q] >= kMaxCodeSat) deeper = true;   // a saturated code bounds nothing
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
    p.maxplane[(size_t)j * p.mpitch + b] = (unsigned short)max_code(m);
}

// ---- M' = M dilated by D <= 8 blocks on either side (D > 2 is served by the D = 8 instance: a larger window is still a bound) (neighbour-maximised sums): one thread per octet of
// blocks (a 128-bit word and its two neighbours; codes order like the values, missing neighbours count 0).
template <int D>
__global__ void __launch_bounds__(256) dilate_max_kernel(const unsigned short* __restrict__ src,
                                                         unsigned short* __restrict__ dst, int64_t mpitch) {
    const int64_t nO = mpitch >> 3;                       // mpitch is a multiple of 8
    const int64_t O = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (O >= nO) return;
    const uint4* row = reinterpret_cast<const uint4*>(src + (size_t)blockIdx.y * mpitch);
    const uint4 z = make_uint4(0u, 0u, 0u, 0u);
    const uint4 w[3] = {O > 0 ? __ldg(row + O - 1) : z, __ldg(row + O), O + 1 < nO ? __ldg(row + O + 1) : z};
    unsigned c[24];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        c[8 * q + 0] = w[q].x & 0xffffu; c[8 * q + 1] = w[q].x >> 16;
        c[8 * q + 2] = w[q].y & 0xffffu; c[8 * q + 3] = w[q].y >> 16;
        c[8 * q + 4] = w[q].z & 0xffffu; c[8 * q + 5] = w[q].z >> 16;
        c[8 * q + 6] = w[q].w & 0xffffu; c[8 * q + 7] = w[q].w >> 16;
    }
    unsigned o[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        unsigned m = c[8 + e];
#pragma unroll
        for (int x = 1; x <= D; ++x) m = max(m, max(c[8 + e - x], c[8 + e + x]));
        o[e] = m;
    }
    reinterpret_cast<uint4*>(dst + (size_t)blockIdx.y * mpitch)[O] =
        make_uint4(o[0] | (o[1] << 16), o[2] | (o[3] << 16), o[4] | (o[5] << 16), o[6] | (o[7] << 16));
}

// ---- pass A: upper bounds from the block-max plane, in integer arithmetic on the codes of fdas_maxcode.h.
// U_h(r,j) = sum_{k<=h} M[row_k][(k r) >> 3] (codes) >= 8 S_h(r,j), and with the integer thresholds
// tq_h <= 8 T_h (1 - 2^-18) of launch_harmonic, U_h <= tq_h for all h proves that (r, j) has no candidate.
// Two fundamentals share one 32-bit register: X = U_h + (0x7fff - tq_h) per half-word, so that bit 15 of
// a half-word is set exactly when U_h > tq_h.  All quantities stay within 16 bits (32 x 1023 + 0x7fff <
// 2^16; tq_h in [-1, 1022], so a saturated code trips its flag alone): no carry ever crosses the
// half-words, and one IADD3 (sum + next code pair + threshold step) and one LOP3 (flag accumulation) serve
// two (fundamental, harmonic) pairs.
//
// Thread <-> 4 consecutive blocks of M = 32 consecutive fundamentals r = 32 Q + i of row j, so that
// harmonic k is the 4k codes M[row_k][4kQ .. 4kQ+4k-1] (k contiguous 64-bit loads) and fundamental i picks
// code (k i) >> 3 of them -- a compile-time choice once k and i are unrolled (one PRMT per pair of
// fundamentals, none where the pair is an aligned word).
constexpr int kPfThreads = 128;   // (coarsen_items assumes 128)

struct PfRow { const unsigned short* mrow; int tq; };

template <class P>
__device__ __forceinline__ PfRow pf_row(const P& p, const int j, const int k) {
    const int c2 = p.nz - 1;
    const int v2 = 2 * k * j - (k - 1) * c2;   // only called for k <= hz: v2 is in range
    PfRow r;
    r.mrow = p.maxplane + (size_t)min((v2 + 1) >> 1, c2) * p.mpitch;
    r.tq = p.tq[k - 1];
    return r;
}

// Harmonic K <= 4 for the 32 fundamentals of quad-block Q: the 4K codes M[row_K][4KQ .. 4KQ+4K-1].
template <int K>
__device__ __forceinline__ void pf_load(const unsigned short* __restrict__ mrow, const unsigned Q, const bool on,
                                        int (&m)[4 * K]) {
    const uint2* src = reinterpret_cast<const uint2*>(mrow + (size_t)4 * K * Q);   // 8K bytes, 8-byte aligned
#pragma unroll
    for (int q = 0; q < K; ++q) {
        uint2 v = make_uint2(0u, 0u);
        if (on) v = __ldg(src + q);
        m[4 * q] = (int)(v.x & 0xffffu); m[4 * q + 1] = (int)(v.x >> 16);
        m[4 * q + 2] = (int)(v.y & 0xffffu); m[4 * q + 3] = (int)(v.y >> 16);
    }
}

// The pair (code e0, code e1) of a slice held as 32-bit words (two codes per word), e0 and e1 static.
template <int E0, int E1, int W0, int NW>
__device__ __forceinline__ unsigned pf_pair(const unsigned (&w)[NW]) {
    constexpr int a = (E0 >> 1) - W0, b = (E1 >> 1) - W0;
    static_assert(a >= 0 && a < NW && b >= 0 && b < NW, "code outside the loaded words");
    if constexpr (a == b && (E0 & 1) == 0 && (E1 & 1) == 1) {
        return w[a];
    } else {
        constexpr unsigned sel = ((E0 & 1) ? 0x32u : 0x10u) | ((E1 & 1) ? 0x7600u : 0x5400u);
        return __byte_perm(w[a], w[b], sel);
    }
}

// One harmonic K for the pairs P0 .. P0 + NP - 1 of fundamentals (2p, 2p+1) from the words w (first word W0
// of the slice): X += codes + step, F = max(F, X) on each half-word (bit 15 of F: some U_h exceeded tq_h).
template <int K, int P0, int NP, int W0, int NW, int PI = 0>
__device__ __forceinline__ void pf_pairs(const unsigned (&w)[NW], const unsigned step, unsigned (&X)[16],
                                         unsigned (&F)[16]) {
    if constexpr (PI < NP) {
        constexpr int p = P0 + PI;
        const unsigned m2 = pf_pair<((K * (2 * p)) >> 3), ((K * (2 * p + 1)) >> 3), W0, NW>(w);
        X[p] = X[p] + m2 + step;
        F[p] = __vmaxu2(F[p], X[p]);
        pf_pairs<K, P0, NP, W0, NW, PI + 1>(w, step, X, F);
    }
}

// The words of harmonic K that one HALF of the thread's fundamentals pick: fundamentals 0..15 pick codes
// (K i) >> 3 < 2K (words 0 .. K-1), fundamentals 16..31 codes 2K .. 4K-1 (words from K rounded down to even,
// so that the 64-bit loads stay aligned).
template <int K, int HALF> struct PfHalf {
    static constexpr int W0 = HALF ? (K & ~1) : 0;
    static constexpr int kLoads = HALF ? (2 * K - W0) / 2 : (K + 1) / 2;     // 64-bit loads
    static constexpr int NW = 2 * kLoads;
};
template <int K, int HALF>
__device__ __forceinline__ void pf_half_load(const unsigned short* __restrict__ mrow, const unsigned Q,
                                             unsigned (&w)[PfHalf<K, HALF>::NW]) {
    const uint2* src = reinterpret_cast<const uint2*>(mrow + (size_t)4 * K * Q + 2 * PfHalf<K, HALF>::W0);
#pragma unroll
    for (int c = 0; c < PfHalf<K, HALF>::kLoads; ++c) {
        const uint2 v = __ldg(src + c);
        w[2 * c] = v.x;
        w[2 * c + 1] = v.y;
    }
}

// Harmonic K alone (all 32 fundamentals inside the plane), half by half: at most K + 2 words live.
template <int K>
__device__ __forceinline__ void pf_harmonic(const unsigned short* __restrict__ mrow, const unsigned Q,
                                            const unsigned step, unsigned (&X)[16], unsigned (&F)[16]) {
    {
        unsigned w[PfHalf<K, 0>::NW];
        pf_half_load<K, 0>(mrow, Q, w);
        pf_pairs<K, 0, 8, PfHalf<K, 0>::W0, PfHalf<K, 0>::NW>(w, step, X, F);
    }
    {
        unsigned w[PfHalf<K, 1>::NW];
        pf_half_load<K, 1>(mrow, Q, w);
        pf_pairs<K, 8, 8, PfHalf<K, 1>::W0, PfHalf<K, 1>::NW>(w, step, X, F);
    }
}

// Harmonics K and K + 1 together: the loads of both are in flight before the first add of either -- the
// kernel is bound by the latency of its dependent loads (L2 / DRAM), so every step that carries two harmonics
// shortens the chain of a thread that has sixteen.
template <int K>
__device__ __forceinline__ void pf_harmonic2(const unsigned short* __restrict__ mrowa,
                                             const unsigned short* __restrict__ mrowb, const unsigned Q,
                                             const unsigned stepa, const unsigned stepb, unsigned (&X)[16],
                                             unsigned (&F)[16]) {
    {
        unsigned wa[PfHalf<K, 0>::NW], wb[PfHalf<K + 1, 0>::NW];
        pf_half_load<K, 0>(mrowa, Q, wa);
        pf_half_load<K + 1, 0>(mrowb, Q, wb);
        pf_pairs<K, 0, 8, PfHalf<K, 0>::W0, PfHalf<K, 0>::NW>(wa, stepa, X, F);
        pf_pairs<K + 1, 0, 8, PfHalf<K + 1, 0>::W0, PfHalf<K + 1, 0>::NW>(wb, stepb, X, F);
    }
    {
        unsigned wa[PfHalf<K, 1>::NW], wb[PfHalf<K + 1, 1>::NW];
        pf_half_load<K, 1>(mrowa, Q, wa);
        pf_half_load<K + 1, 1>(mrowb, Q, wb);
        pf_pairs<K, 8, 8, PfHalf<K, 1>::W0, PfHalf<K, 1>::NW>(wa, stepa, X, F);
        pf_pairs<K + 1, 8, 8, PfHalf<K + 1, 1>::W0, PfHalf<K + 1, 1>::NW>(wb, stepb, X, F);
    }
}

// Harmonics K, K+1, .. while every fundamental of the thread has them (k <= he; he_max is the CTA's deepest),
// two per step.
template <int K>
__device__ __forceinline__ void pf_from(const HarmParams& p, const int j, const unsigned Q, const int he_max,
                                        const int he, unsigned (&X)[16], unsigned (&F)[16]) {
    if constexpr (K <= 32) {
        if (K > he_max) return;                 // CTA-uniform: no thread of this CTA goes deeper
        if (he >= K) {
            const PfRow ra = pf_row(p, j, K);
            // threshold step of a harmonic on both half-words: -(tq_K - tq_{K-1}) as one 32-bit integer
            const unsigned stepa = (unsigned)(p.tq[K - 2] - ra.tq) * 0x10001u;
            if constexpr (K + 1 <= 32) {
                if (he >= K + 1) {
                    const PfRow rb = pf_row(p, j, K + 1);
                    pf_harmonic2<K>(ra.mrow, rb.mrow, Q, stepa, (unsigned)(ra.tq - rb.tq) * 0x10001u, X, F);
                } else {
                    pf_harmonic<K>(ra.mrow, Q, stepa, X, F);
                }
            } else {
                pf_harmonic<K>(ra.mrow, Q, stepa, X, F);
            }
        }
        pf_from<K + 2>(p, j, Q, he_max, he, X, F);
    }
}

// Fundamentals of quad-block Q flagged by pass A go to the maybe list as (r, j).
template <class P>
__device__ __forceinline__ void pf_emit(const P& p, const unsigned Q, const int j, unsigned flagged) {
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
                p.maybe[slot++] = make_uint2(32u * Q + (unsigned)i, (unsigned)j | (0xffffu << 16));   // no hint
            }
        } else {
            atomicExch(p.overflow, 1u);   // pass B then falls back to the full scan
        }
    }
}

// The same for a whole (converged) warp: one atomic slot claim per warp instead of one per thread -- with
// 16-harmonic rows most threads of the general kernel have a flagged fundamental, and their claims would all
// queue at the one L2 slice that holds the counter.
// A record is (r, j | hint << 16).  hint = kHintNone, or E + kHintBias with
//   E = max_{h >= 5} (U_h - tq_h) - U_4   (codes; the thread's `hint` words hold it for its 16 pairs):
// once the exact pass knows S_4, ceil(8 S_4) + E <= 0 proves that no deeper sum can exceed its threshold
// (8 S_h <= 8 S_4 + (U_h - U_4)), without gathering the twelve block-max codes again.
constexpr int kHintBias = 8192;
constexpr unsigned kHintNone = 0xffffu;
__device__ __forceinline__ void pf_emit_warp(const HarmParams& p, const unsigned Q, const int j, unsigned flagged,
                                             const unsigned* hint) {
    if (32 * (int64_t)Q < p.r_lo) {
        const int64_t cut = p.r_lo - 32 * (int64_t)Q;
        flagged = (cut >= 32) ? 0u : (flagged & ~((1u << (int)cut) - 1u));
    }
    const unsigned lane = threadIdx.x & 31u;
    const int n = __popc(flagged);
    int incl = n;                                   // inclusive prefix sum over the lanes
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, d);
        if ((int)lane >= d) incl += v;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    if (total == 0) return;
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(p.maybe_count, (unsigned long long)total);
    base = __shfl_sync(0xffffffffu, base, 0);
    if (base + (unsigned long long)total <= (unsigned long long)p.maybe_capacity) {
        unsigned long long slot = base + (unsigned long long)(incl - n);
        while (flagged) {
            const int i = __ffs(flagged) - 1;
            flagged &= flagged - 1;
            unsigned hi = kHintNone;
            if (hint) hi = (i & 1) ? (hint[i >> 1] >> 16) : (hint[i >> 1] & 0xffffu);
            p.maybe[slot++] = make_uint2(32u * Q + (unsigned)i, (unsigned)j | (hi << 16));
        }
    } else if (lane == 0) {
        atomicExch(p.overflow, 1u);   // pass B then falls back to the full scan
    }
}

// ---- level 1 of pass A for the parts of the plane with at most kShallowDepth = 4 harmonics: the block-level
// bound for the 64 fundamentals of an octet of blocks (= one coarse block) that failed the coarse bound below
// (called from prefilter_coarse_kernel for those blocks only).
// Harmonic k picks block (k i) >> 3 for fundamental i of a block of 8, so U_1 is the same for all 8
// fundamentals, U_2 for halves, U_3 takes 4 and U_4 5 distinct values per block: 12 sums and compares stand for
// 32.  A thread reads 8 blocks of M[j] and the 8k blocks of M[row_k] they map to, every load issued up front.
constexpr int kShallowDepth = 4;

__device__ __forceinline__ int code_at(const uint4 (&w)[4], const int e) {   // code e of up to 32 (static e)
    const uint4 v = w[e >> 3];
    const unsigned x = ((e >> 1) & 3) == 0 ? v.x : ((e >> 1) & 3) == 1 ? v.y : ((e >> 1) & 3) == 2 ? v.z : v.w;
    return (int)((e & 1) ? (x >> 16) : (x & 0xffffu));
}

// The 64 fundamentals of octet O (8 blocks of M) of row j, for at most DMAX harmonics: the caller guarantees
// that no fundamental of the octet has a harmonic DMAX + 1 inside the plane (in z or in r).
template <int DMAX, class P>
__device__ __forceinline__ void pf_shallow_octet(const P& p, const unsigned O, const int j) {
    const int c2 = p.nz - 1;
    const unsigned last = (unsigned)(p.nbins - 1);
    const int d = abs(2 * j - c2);
    const int hz = min(DMAX, d == 0 ? p.H : min(p.H, c2 / d));   // 1 .. DMAX here
    const PfRow r1 = pf_row(p, j, 1);
    uint4 m1[4], m2[4], m3[4], m4[4];   // (only the first DMAX arrays are live)
    m1[0] = __ldg(reinterpret_cast<const uint4*>(r1.mrow) + O);
    if (hz <= 1 && r1.tq >= 0) {
        // one harmonic only (half of the plane's rows): code > tq_1 on the packed half-words.
        // (tq_1 = -1 passes every point, code 0 included: no early exit then.)
        const unsigned tb2 = (unsigned)r1.tq * 0x10001u;
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
        const int u1 = code_at(m1, q);
        if (u1 > r1.tq) fl |= 0xffu;
        if (dep >= 2) {
            // U_2: fundamentals 0..3 -> block 2q, 4..7 -> block 2q+1 of row_2
            const int u2[2] = {u1 + code_at(m2, 2 * q), u1 + code_at(m2, 2 * q + 1)};
            if (u2[0] > r2.tq) fl |= 0x0fu;
            if (u2[1] > r2.tq) fl |= 0xf0u;
            if (DMAX >= 3 && dep >= 3) {
                // U_3: (i >> 2, (3 i) >> 3) = (0,0) for i = 0,1,2; (0,1) for 3; (1,1) for 4,5; (1,2) for 6,7
                const int u3[4] = {u2[0] + code_at(m3, 3 * q), u2[0] + code_at(m3, 3 * q + 1),
                                   u2[1] + code_at(m3, 3 * q + 1), u2[1] + code_at(m3, 3 * q + 2)};
                if (u3[0] > r3.tq) fl |= 0x07u;
                if (u3[1] > r3.tq) fl |= 0x08u;
                if (u3[2] > r3.tq) fl |= 0x30u;
                if (u3[3] > r3.tq) fl |= 0xc0u;
                if (DMAX >= 4 && dep >= 4) {
                    // U_4 adds block i >> 1 of row_4: i = 0,1 | 2 | 3 | 4,5 | 6,7
                    if (u3[0] + code_at(m4, 4 * q) > r4.tq) fl |= 0x03u;
                    if (u3[0] + code_at(m4, 4 * q + 1) > r4.tq) fl |= 0x04u;
                    if (u3[1] + code_at(m4, 4 * q + 1) > r4.tq) fl |= 0x08u;
                    if (u3[2] + code_at(m4, 4 * q + 2) > r4.tq) fl |= 0x30u;
                    if (u3[3] + code_at(m4, 4 * q + 3) > r4.tq) fl |= 0xc0u;
                }
            }
        }
        f[q >> 2] |= fl << sh;
    }
    if (dep < hz && 64u * O <= last / (unsigned)(dep + 1)) {
        // the thread that straddles the end of harmonic dep+1's range (one per harmonic and row): harmonic
        // dep+1 exists for its first fundamentals only -- all 64 go to the exact pass, which knows
        f[0] = f[1] = 0xffffffffu;
    }
    pf_emit(p, 2u * O, j, f[0]);
    pf_emit(p, 2u * O + 1u, j, f[1]);
}

// What pf_shallow_octet reads of the kernel parameters, BY VALUE for the out-of-line call from the coarse
// kernel (a reference to the parameter struct would make every thread copy all of it to local memory).
struct PfArgs {
    const unsigned short* maxplane;
    int64_t mpitch, nbins, r_lo, maybe_capacity;
    uint2* maybe;
    unsigned long long* maybe_count;
    unsigned* overflow;
    int nz, H;
    int tq[kShallowDepth];
};
__device__ __noinline__ void pf_shallow_octet_call(const PfArgs a, const unsigned O, const int j) {
    pf_shallow_octet<kShallowDepth>(a, O, j);
}

// ---- level 0 of pass A: the same bound on COARSE blocks of 64 plane columns.
// M2[j][B] = max of the 8 codes M[j][8B .. 8B+7] (row-major, 1/8 of M: 25 MB at the SKA size, L2-resident).
// For a fundamental r of coarse block B harmonic k lies in the coarse blocks kB .. kB + k - 1 of row_k, so
//     U0_h(B,j) = sum_{k<=h} max_{i<k} M2[row_k][kB + i]  >=  U_h(r,j)  >=  8 S_h(r,j)   for all r in B:
// U0_h <= tq_h for all h settles 64 fundamentals at once.  It serves the parts of the plane with at most
// kShallowDepth harmonics -- the shallow rows, and of the deep rows the fundamentals r >= 64 b_deep -- where
// the sum of a few maxima of Exp(1) noise stays far below the thresholds; for the (B, j) that fail the same thread
// goes on to the block level (pf_shallow_octet).  (With 16 harmonics the coarse bound is useless: the deep part of the deep rows is
// prefilter_kernel's.)
// M2[i] = max of the 8 codes M[8 i .. 8 i + 7] over the items [begin, end) (M's rows are contiguous, so both
// planes are linear arrays); a CTA of kPfThreads threads, four 128-bit loads in flight per thread.
__device__ __forceinline__ void coarsen_items(const unsigned short* __restrict__ M, unsigned short* __restrict__ M2,
                                              const int64_t begin, const int64_t end) {
    const uint4* src = reinterpret_cast<const uint4*>(M);
    for (int64_t i0 = begin + threadIdx.x; i0 < end; i0 += 4 * 128) {
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            v[u] = (i0 + 128 * u < end) ? __ldg(src + i0 + 128 * u) : make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            unsigned m = __vmaxu2(__vmaxu2(v[u].x, v[u].y), __vmaxu2(v[u].z, v[u].w));
            m = max(m & 0xffffu, m >> 16);
            if (i0 + 128 * u < end) M2[i0 + 128 * u] = (unsigned short)m;
        }
    }
}


// Thread <-> 8 consecutive coarse blocks B = 8 G + q of row j (one 128-bit word of M2[j]); harmonic k needs
// the 8k coarse blocks 8kG .. 8kG + 8k - 1 of row_k (k words); all loads are issued up front.
__global__ void __launch_bounds__(256) prefilter_coarse_kernel(const HarmParams p, const unsigned b_deep) {
    const unsigned nB = (unsigned)(p.mpitch >> 3), nG = nB >> 3;      // nB is a multiple of 8 here
    const unsigned G = blockIdx.x * 256u + threadIdx.x;
    const int j = blockIdx.y;
    if (G >= nG) return;
    const unsigned last = (unsigned)(p.nbins - 1);
    const int c2 = p.nz - 1;
    const int d = abs(2 * j - c2);
    const int hzr = d == 0 ? p.H : min(p.H, c2 / d);
    const bool deep = hzr > kShallowDepth;
    if (deep && 8u * G + 7u < b_deep) return;                          // the deep part of a deep row
    const int hz = min(hzr, kShallowDepth);                            // CTA-uniform
    const unsigned short* const M2 = p.max2;
    const uint4 m1 = __ldg(reinterpret_cast<const uint4*>(M2 + (size_t)j * nB) + G);
    if (hz <= 1 && p.tq[0] >= 0 && !deep) {
        const unsigned tb2 = (unsigned)p.tq[0] * 0x10001u;
        if ((__vcmpgtu2(m1.x, tb2) | __vcmpgtu2(m1.y, tb2) | __vcmpgtu2(m1.z, tb2) | __vcmpgtu2(m1.w, tb2)) == 0u)
            return;                                                    // almost every thread of a one-harmonic row
    }
    // harmonic k of coarse block B exists iff some fundamental of the block has it: 64 k B <= Nb - 1, i.e.
    // B <= bmax_k; the codes of harmonic k as 4k words (two codes each), zeros where not loaded
    unsigned w2[8], w3[12], w4[16];
    {
        auto load = [&](const int k, unsigned* w) {
            const int row = min((2 * k * j - (k - 1) * c2 + 1) >> 1, c2);     // (unused when k > hz)
            const uint4* src = reinterpret_cast<const uint4*>(M2 + (size_t)row * nB);
#pragma unroll 4
            for (int c = 0; c < 4; ++c) {
                if (c < k) {
                    const unsigned g = (unsigned)k * G + (unsigned)c;
                    const uint4 v = (k <= hz && g < nG) ? __ldg(src + g) : make_uint4(0u, 0u, 0u, 0u);
                    w[4 * c] = v.x; w[4 * c + 1] = v.y; w[4 * c + 2] = v.z; w[4 * c + 3] = v.w;
                }
            }
        };
        load(2, w2); load(3, w3); load(4, w4);
    }
    const unsigned w1[4] = {m1.x, m1.y, m1.z, m1.w};
    auto lo = [](unsigned x) { return (int)(x & 0xffffu); };
    auto hi = [](unsigned x) { return (int)(x >> 16); };
    auto max2 = [&](unsigned x) { return max(lo(x), hi(x)); };
    {   // the whole thread at once: V_h = sum_{k<=h} (largest code of harmonic k among all its blocks) >= U0_h(B)
        // for each of the 8 coarse blocks; V_h <= tq_h for all h settles them together
        unsigned a1 = __vmaxu2(__vmaxu2(w1[0], w1[1]), __vmaxu2(w1[2], w1[3]));
        unsigned a2 = 0u, a3 = 0u, a4 = 0u;
#pragma unroll
        for (int c = 0; c < 8; ++c) a2 = __vmaxu2(a2, w2[c]);
#pragma unroll
        for (int c = 0; c < 12; ++c) a3 = __vmaxu2(a3, w3[c]);
#pragma unroll
        for (int c = 0; c < 16; ++c) a4 = __vmaxu2(a4, w4[c]);
        int V = max2(a1);
        bool any = V > p.tq[0];
        V += max2(a2); any = any || (hz >= 2 && V > p.tq[1]);
        V += max2(a3); any = any || (hz >= 3 && V > p.tq[2]);
        V += max2(a4); any = any || (hz >= 4 && V > p.tq[3]);
        if (!any) return;
    }
    const unsigned bmax2 = last / 128u, bmax3 = last / 192u, bmax4 = last / 256u;
    unsigned fl = 0u;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const unsigned B = 8u * G + (unsigned)q;
        int U = (q & 1) ? hi(w1[q >> 1]) : lo(w1[q >> 1]);
        bool f = U > p.tq[0];
        if (hz >= 2 && B <= bmax2) {                                     // codes 2q, 2q+1: word q
            U += max2(w2[q]);
            f = f || U > p.tq[1];
            if (hz >= 3 && B <= bmax3) {                                 // codes 3q .. 3q+2
                const int e = 3 * q;
                const int m3 = (e & 1) ? max(hi(w3[e >> 1]), max2(w3[(e >> 1) + 1]))
                                       : max(max2(w3[e >> 1]), lo(w3[(e >> 1) + 1]));
                U += m3;
                f = f || U > p.tq[2];
                if (hz >= 4 && B <= bmax4) {                             // codes 4q .. 4q+3: words 2q, 2q+1
                    U += max2(__vmaxu2(w4[2 * q], w4[2 * q + 1]));
                    f = f || U > p.tq[3];
                }
            }
        }
        if (f && !(deep && B < b_deep)) fl |= 1u << q;
    }
    if (fl) {   // (rare) level 1 right here: the block-level bound for the 64 fundamentals of each failing coarse block
        PfArgs a;
        a.maxplane = p.maxplane; a.mpitch = p.mpitch; a.nbins = p.nbins; a.r_lo = p.r_lo;
        a.maybe_capacity = p.maybe_capacity; a.maybe = p.maybe; a.maybe_count = p.maybe_count; a.overflow = p.overflow;
        a.nz = p.nz; a.H = p.H;
#pragma unroll
        for (int k = 0; k < kShallowDepth; ++k) a.tq[k] = p.tq[k];
        while (fl) {
            const int q = __ffs(fl) - 1;
            fl &= fl - 1;
            pf_shallow_octet_call(a, 8u * G + (unsigned)q, j);
        }
    }
}

// The launch also carries the CTAs that build the coarse plane M2 from M (coarsen_items), interleaved with the
// prefilter's own (odd / even block index): that stream is bound by DRAM bandwidth, the prefilter by the
// latency of its dependent loads, and neither needs the other's result -- side by side they take the time
// of the longer one.  gx x gy = the prefilter's grid; per > 0: coarsen items per CTA.
__global__ void __launch_bounds__(kPfThreads, 8) prefilter_kernel(const HarmParams p, const int nlow,
                                                                  const unsigned q_end, const unsigned gx,
                                                                  const unsigned gy, const int64_t per) {
    unsigned bid = blockIdx.x;
    if (per > 0) {
        if (bid & 1u) {
            const int64_t total = (int64_t)p.nz * (p.mpitch >> 3), begin = (int64_t)(bid >> 1) * per;
            coarsen_items(p.maxplane, p.max2, begin, min(total, begin + per));
            return;
        }
        bid >>= 1;
    }
    if (bid >= gx * gy) return;
    const int j = nlow + (int)(bid / gx);   // the rows with more than kShallowDepth harmonics (|z| <= zmax/5)
    const int c2 = p.nz - 1;
    const unsigned Q0 = (bid % gx) * (unsigned)kPfThreads;
    // q_end <= nbins / 32: the quad-blocks beyond it belong to the coarse level.  The threads beyond stay (with
    // nothing to do) for the warp-wide slot claim at the end; they redo the last quad-block's loads.
    const bool mine = Q0 + threadIdx.x < q_end;
    const unsigned Q = mine ? Q0 + threadIdx.x : q_end - 1u;
    const unsigned last = (unsigned)(p.nbins - 1);
    // hz: harmonics inside the plane in z for this row (CTA-uniform): twice the row of harmonic k is
    // v2 = k d + c2 with d = 2 j - c2, and 0 <= v2 <= 2 c2  <=>  k |d| <= c2
    const int d = abs(2 * j - c2);
    const int hz = d == 0 ? p.H : min(p.H, c2 / d);
    // he: harmonics for which all 32 fundamentals of this thread are inside the plane in r
    const int he = (int)min((unsigned)hz, last / (32u * Q + 31u));
    const int he_max = (int)min((unsigned)hz, last / (32u * Q0 + 31u));   // deepest in this CTA
    unsigned flagged = 0u;   // bit i: some U_h of fundamental 32 Q + i exceeds tq_h
    int U4[20];              // U_4 of block b: [5b] i = 0,1  [5b+1] i = 2  [5b+2] i = 3  [5b+3] i = 4,5  [5b+4] i = 6,7
    {   // harmonics 1..4: ten 64-bit loads in flight; harmonic k picks block (k i) >> 3 for fundamental i of a
        // block of 8: U_1 is the same for all 8, U_2 for the 4 of a half block, U_3 takes 4 and U_4 5 distinct
        // values per block -- 12 sums and compares per block stand for 32 (h <= 4 are 90 % of all (r, j, h)
        // triples of the plane)
        const PfRow r1 = pf_row(p, j, 1);
        int m1[4], m2[8], m3[12], m4[16];
        pf_load<1>(r1.mrow, Q, true, m1);
        PfRow r2 = r1, r3 = r1, r4 = r1;
        if (he_max >= 2) { r2 = pf_row(p, j, 2); pf_load<2>(r2.mrow, Q, he >= 2, m2); }
        if (he_max >= 3) { r3 = pf_row(p, j, 3); pf_load<3>(r3.mrow, Q, he >= 3, m3); }
        if (he_max >= 4) { r4 = pf_row(p, j, 4); pf_load<4>(r4.mrow, Q, he >= 4, m4); }
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (m1[q] > r1.tq) flagged |= 0xffu << (8 * q);
        if (he >= 2) {
            int u2[8];
#pragma unroll
            for (int gq = 0; gq < 8; ++gq) {
                u2[gq] = m1[gq >> 1] + m2[gq];
                if (u2[gq] > r2.tq) flagged |= 0xfu << (4 * gq);
            }
            if (he >= 3) {
                int u3[16];
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    // (i >> 2, (3 i) >> 3) = (0,0) for i = 0,1,2; (0,1) for 3; (1,1) for 4,5; (1,2) for 6,7
                    u3[4 * b + 0] = u2[2 * b] + m3[3 * b];
                    u3[4 * b + 1] = u2[2 * b] + m3[3 * b + 1];
                    u3[4 * b + 2] = u2[2 * b + 1] + m3[3 * b + 1];
                    u3[4 * b + 3] = u2[2 * b + 1] + m3[3 * b + 2];
                    if (u3[4 * b + 0] > r3.tq) flagged |= 0x07u << (8 * b);
                    if (u3[4 * b + 1] > r3.tq) flagged |= 0x08u << (8 * b);
                    if (u3[4 * b + 2] > r3.tq) flagged |= 0x30u << (8 * b);
                    if (u3[4 * b + 3] > r3.tq) flagged |= 0xc0u << (8 * b);
                }
                if (he >= 4) {
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        // U_4 adds block i >> 1 of row_4: i = 0,1 | 2 | 3 | 4,5 | 6,7
                        U4[5 * b + 0] = u3[4 * b + 0] + m4[4 * b];
                        U4[5 * b + 1] = u3[4 * b + 0] + m4[4 * b + 1];
                        U4[5 * b + 2] = u3[4 * b + 1] + m4[4 * b + 1];
                        U4[5 * b + 3] = u3[4 * b + 2] + m4[4 * b + 2];
                        U4[5 * b + 4] = u3[4 * b + 3] + m4[4 * b + 3];
                        if (U4[5 * b + 0] > r4.tq) flagged |= 0x03u << (8 * b);
                        if (U4[5 * b + 1] > r4.tq) flagged |= 0x04u << (8 * b);
                        if (U4[5 * b + 2] > r4.tq) flagged |= 0x08u << (8 * b);
                        if (U4[5 * b + 3] > r4.tq) flagged |= 0x30u << (8 * b);
                        if (U4[5 * b + 4] > r4.tq) flagged |= 0xc0u << (8 * b);
                    }
                }
            }
        }
    }
    // Per thread: U_4 of its 16 pairs while the deep harmonics run, then the exact pass's hint (see pf_emit_warp).
    __shared__ __align__(16) unsigned stash[kPfThreads * 20];   // rows of 16 words, pitch 20: conflict-free 128-bit accesses
    unsigned* const my = stash + threadIdx.x * 20;
    bool hinted = false;
    if (he_max >= 5) {       // CTA-uniform
        // harmonics 5..: two fundamentals per register, X = U + (0x7fff - tq) on each half-word
        unsigned X[16], F[16];   // pair p: fundamentals 2p (low half-word) and 2p + 1 (high)
        if (he >= 5) {
            const unsigned base = (unsigned)(0x7fff - p.tq[3]) * 0x10001u;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const unsigned u0 = (unsigned)U4[5 * b + 0] * 0x10001u;
                const unsigned u1 = (unsigned)U4[5 * b + 1] | ((unsigned)U4[5 * b + 2] << 16);
                const unsigned u2 = (unsigned)U4[5 * b + 3] * 0x10001u, u3 = (unsigned)U4[5 * b + 4] * 0x10001u;
                *reinterpret_cast<uint4*>(my + 4 * b) = make_uint4(u0, u1, u2, u3);
                X[4 * b + 0] = u0 + base; X[4 * b + 1] = u1 + base; X[4 * b + 2] = u2 + base; X[4 * b + 3] = u3 + base;
            }
#pragma unroll
            for (int pp = 0; pp < 16; ++pp) F[pp] = 0u;
        }
        pf_from<5>(p, j, Q, he_max, he, X, F);
        if (he >= 5) {
            // F = max_{h >= 5} X_h on each half-word.  bit 15 - p <- fundamental 2p, bit 31 - p <- fundamental 2p + 1
            unsigned acc = 0u;
#pragma unroll
            for (int pp = 0; pp < 16; ++pp) acc |= (F[pp] & 0x80008000u) >> pp;
            if (acc) {
#pragma unroll
                for (int pp = 0; pp < 16; ++pp) {
                    if (acc & (0x8000u >> pp)) flagged |= 1u << (2 * pp);
                    if (acc & (0x80000000u >> pp)) flagged |= 1u << (2 * pp + 1);
                }
            }
            if (flagged) {
                // hint for the exact pass: E = max_{h >= 5} (U_h - tq_h) - U_4 = max X - U_4 - 0x7fff, biased by
                // kHintBias (every half-word of F - U_4 is >= 0x7fff - 1022, so nothing borrows)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const uint4 u = *reinterpret_cast<const uint4*>(my + 4 * b);
                    constexpr unsigned kSub = (unsigned)(0x7fff - kHintBias) * 0x10001u;
                    *reinterpret_cast<uint4*>(my + 4 * b) = make_uint4(F[4 * b] - u.x - kSub, F[4 * b + 1] - u.y - kSub,
                                                                       F[4 * b + 2] - u.z - kSub, F[4 * b + 3] - u.w - kSub);
                }
                hinted = true;
            }
        }
    }
    if (he < hz && 32u * Q <= last / (unsigned)(he + 1)) {
        // the thread that straddles the end of harmonic he+1's range (one per harmonic and row): that
        // harmonic exists for its first fundamentals only -- all 32 go to the exact pass, which knows
        flagged = 0xffffffffu;
        hinted = false;
    }
    pf_emit_warp(p, Q, j, mine ? flagged : 0u, hinted ? my : nullptr);
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
            if (NBR) exact_fundamental_nbr(P, g, sthr, (int64_t)rec.x, (int)(rec.y & 0xffffu));
            else exact_fundamental(P, g, sthr, (int64_t)rec.x, (int)(rec.y & 0xffffu), rec.y >> 16);
        }
    } else {
        const unsigned long long n = (unsigned long long)p.nbins * (unsigned long long)p.nz;
        for (unsigned long long q = tid; q < n; q += nthr) {
            const int64_t r = (int64_t)(q % (unsigned long long)p.nbins);
            const int j = (int)(q / (unsigned long long)p.nbins);
            if (NBR) exact_fundamental_nbr(P, g, sthr, r, j);
            else exact_fundamental(P, g, sthr, r, j, 0xffffu);
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
    // integer thresholds of pass A: tq_h <= 8 T_h (1 - 2^-18) -- the slack covers the rounding of the exact
    // pass's fp32 sums (S_h^fp32 <= (1 + 2^-19) sum P for h <= 32) -- clamped below the saturated code, so
    // that a block without a bound trips every flag; a negative T_h passes every point (tq = -1)
    for (int h = 0; h < 32; ++h) {
        const float T = p.thr[h];
        if (!(T >= 0.f)) {
            p.tq[h] = -1;
        } else {
            const double v = std::floor((double)kMaxCodeScale * (double)T * (1.0 - 1.0 / 262144.0));
            p.tq[h] = v > (double)(kMaxCodeSat - 1) ? (int)(kMaxCodeSat - 1) : (int)v;
        }
    }
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
        if (D > 8 || (p.mpitch & 7)) return cudaErrorInvalidValue;     // H <= 32 gives D <= 2; mpitch = nbins / 8
        dim3 grid((unsigned)((p.mpitch / 8 + 255) / 256), (unsigned)p.nz);
        switch (D) {   // D = 1 for H <= 17, 2 up to H = 32 (compile-time window: the loop unrolls to 2 D maxima per block)
            case 0: dilate_max_kernel<0><<<grid, 256, 0, st>>>(p.maxplane, p.maxplane_nbr, p.mpitch); break;
            case 1: dilate_max_kernel<1><<<grid, 256, 0, st>>>(p.maxplane, p.maxplane_nbr, p.mpitch); break;
            case 2: dilate_max_kernel<2><<<grid, 256, 0, st>>>(p.maxplane, p.maxplane_nbr, p.mpitch); break;
            default: dilate_max_kernel<8><<<grid, 256, 0, st>>>(p.maxplane, p.maxplane_nbr, p.mpitch); break;
        }
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        ++*launches;
        p.maxplane = p.maxplane_nbr;
    }
    // rows j < nlow and j >= nz - nlow have at most kShallowDepth harmonics inside the plane (reading A12)
    int nlow = 0;
    const bool coarse = (p.mpitch & 63) == 0 && p.max2 != nullptr;  // the coarse level reads 8 coarse blocks per word
    if (coarse) {
        const int c2 = p.nz - 1;
        auto hz_of = [&](int j) { const int d = c2 - 2 * j; return d == 0 ? p.H : std::min(p.H, c2 / d); };
        // (the centre row of an odd bank is classified like every other row: with H <= kShallowDepth it is
        // shallow too, nlow reaches (nz + 1) / 2 and no row is left for the general prefilter -- the same
        // partition as prefilter_coarse_kernel's `deep`, so that no fundamental is listed twice)
        while (2 * nlow < p.nz && hz_of(nlow) <= kShallowDepth) ++nlow;
    }
    const int ndeep = std::max(0, p.nz - 2 * nlow);   // rows with more than kShallowDepth harmonics
    // of a deep row the general kernel takes the fundamentals r < 64 b_deep only (those that can have a fifth
    // harmonic inside the plane); the rest goes through the coarse level like the shallow rows
    unsigned b_deep = 0, q_end = (unsigned)(p.mpitch / 4);
    if (coarse) {
        const unsigned nB = (unsigned)(p.mpitch / 8);
        b_deep = std::min(nB, (unsigned)((p.nbins - 1) / (64 * (kShallowDepth + 1))) + 1u);
        q_end = 2u * b_deep;
    }
    {   // the general prefilter (deep rows, r < 64 b_deep) and, interleaved with it, the CTAs that build M2
        // (p.maxplane is the dilated plane in the neighbour-maximised mode)
        const unsigned gx = ndeep > 0 ? (q_end + kPfThreads - 1) / kPfThreads : 0u, gy = (unsigned)std::max(ndeep, 0);
        unsigned nblk = gx * gy;
        int64_t per = 0;
        if (coarse) {
            const int64_t total = (int64_t)p.nz * (p.mpitch >> 3);
            nblk = std::max(nblk, 148u * 8u);
            per = ((total + nblk - 1) / nblk + 511) / 512 * 512;
            nblk *= 2;
        }
        if (nblk > 0) {
            prefilter_kernel<<<nblk, kPfThreads, 0, st>>>(p, nlow, q_end, gx, gy, per);
            if ((e = cudaGetLastError()) != cudaSuccess) return e;
            ++*launches;
        }
    }
    if (coarse) {
        const unsigned nB = (unsigned)(p.mpitch / 8);
        prefilter_coarse_kernel<<<dim3((nB / 8 + 255) / 256, (unsigned)p.nz), 256, 0, st>>>(p, b_deep);
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

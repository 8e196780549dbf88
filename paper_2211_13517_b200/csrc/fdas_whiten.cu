// fdas_whiten.cu -- K1, running-median power whitening (BASELINE.json north_star; DESIGN.md step a2,
// reading A3).
//   K1a  one CTA per block of the A3 schedule: |X|^2 in registers, exact median by radix selection
//        (even count: mean of the two middle values)
//   K1b  per bin: linear interpolation of the block medians between block centres (constant outside
//        the first/last centre), w[k] = X[k] sqrt(ln2 / m(k)), w[0] = 0, stored fp32 or bf16 (RNE)
#include <cuda_bf16.h>

#include <mutex>
#include <string>

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

// ---------------------------------------------------------------------------------------------------
// fdas_whiten_static (include/fdas.h) -- K1 for callers that may not allocate device memory.
//
// The plan-based path keeps K1's scratch (block schedule + median table) in cudaMalloc'd buffers that
// fdas_plan creates.  A caller that cannot create a plan -- a stage of a real-time backend whose HBM was
// all handed to its own pool at start-up (a later cudaMalloc can fail there, and it synchronises the
// whole device, stalling the ingest streams), or a plug-in that may only touch the buffers it is given --
// gets the same two kernels with the scratch in the fixed array below.  The array is part of the
// library image: every GPU that loads libfdas.so holds its 51 KB until the process exits.
//
// g_whiten_static_scratch is a DEVICE symbol.  In host code its name is only a host-side stand-in (the
// address of a shadow variable), never a device address: the address the kernels receive comes from
// cudaGetSymbolAddress, looked up once per device with that device current.
// ---------------------------------------------------------------------------------------------------
extern thread_local std::string g_detail;   // fdas_api.cu: text behind fdas_last_error_detail()

namespace {

constexpr int64_t kStaticMinBins = 1024;                 // smallest spectrum a plan can have (N >= 2 * 1024)
constexpr int64_t kStaticMaxBins = (int64_t)1 << 24;     // stated maximum of the entry point
constexpr int kStaticMaxBlocks = 4352;                   // the A3 schedule of 2^24 bins has 4124 blocks
constexpr size_t kStaticSection = (size_t)kStaticMaxBlocks * 4;   // 17408 bytes = 68 x 256
// three sections of kStaticSection bytes: blk_start (int32), blk_len (int32), blk_med (float)
static __device__ __align__(256) unsigned char g_whiten_static_scratch[3 * kStaticSection];

// Block schedule of reading A3 (the same rule as fdas::whitening_blocks on the host), written on the
// device so that nothing is copied from pageable host memory: thread 0 walks the short blocks at the
// low-frequency end (a few dozen), from the first 4096-bin block on the starts are an arithmetic series.
__global__ void __launch_bounds__(256) static_schedule_kernel(int32_t* blk_start, int32_t* blk_len,
                                                              long long nb, int nblk) {
    __shared__ int s_i0;
    __shared__ long long s_s0;
    if (threadIdx.x == 0) {
        long long s = 1;
        int i = 0;
        while (s < nb) {
            const int lg = 63 - __clzll(s);
            long long l = (lg >= 2) ? (1ll << (lg - 2)) : 1ll;
            if (l < 32) l = 32;
            if (l >= 4096) break;
            if (s + l > nb) l = nb - s;
            blk_start[i] = (int32_t)s;
            blk_len[i] = (int32_t)l;
            ++i;
            s += l;
        }
        s_i0 = i;
        s_s0 = s;
    }
    __syncthreads();
    for (int i = s_i0 + (int)threadIdx.x; i < nblk; i += (int)blockDim.x) {
        const long long s = s_s0 + (long long)(i - s_i0) * 4096;
        blk_start[i] = (int32_t)s;
        blk_len[i] = (int32_t)((nb - s < 4096) ? (nb - s) : 4096);
    }
}

int static_block_count(int64_t nb) {   // host: number of blocks of the A3 schedule (no tables needed)
    int64_t s = 1;
    int n = 0;
    while (s < nb) {
        const int lg = 63 - __builtin_clzll((unsigned long long)s);
        int64_t l = (lg >= 2) ? ((int64_t)1 << (lg - 2)) : 1;
        if (l < 32) l = 32;
        if (l > 4096) l = 4096;
        if (s + l > nb) l = nb - s;
        s += l;
        ++n;
    }
    return n;
}

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
unsigned char* g_static_ptr[kStaticMaxDevices] = {};   // device address of the scratch, per device ordinal

}  // namespace

extern "C" int fdas_whiten_static(const float* d_X, int64_t nbins, void* d_spec, int spec_bf16,
                                  void* cuda_stream) {
    if (!d_X || !d_spec || (spec_bf16 != 0 && spec_bf16 != 1)) return FDAS_EARG;
    if (nbins < kStaticMinBins) {
        g_detail = "fdas_whiten_static: nbins " + std::to_string(nbins) + " is below the minimum " +
                   std::to_string(kStaticMinBins);
        return FDAS_EARG;
    }
    if (nbins > kStaticMaxBins) {
        g_detail = "fdas_whiten_static: nbins " + std::to_string(nbins) +
                   " exceeds the fixed scratch array's maximum of " + std::to_string(kStaticMaxBins) +
                   " bins (use a plan and fdas_prepare_spectrum for longer spectra)";
        return FDAS_EUNSUPPORTED;
    }
    const int nblk = static_block_count(nbins);
    if (nblk < 1 || nblk > kStaticMaxBlocks) {
        g_detail = "fdas_whiten_static: block schedule does not fit the fixed scratch array";
        return FDAS_EUNSUPPORTED;
    }
    // set-up, once per device: the device address of the scratch array on the CURRENT device
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kStaticMaxDevices) {
        g_detail = std::string("fdas_whiten_static: cudaGetDevice: ") +
                   (e != cudaSuccess ? cudaGetErrorString(e) : "device ordinal out of range");
        return FDAS_ECUDA;
    }
    unsigned char* base = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_static_mutex);
        if (!g_static_ptr[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_whiten_static_scratch);
            if (e != cudaSuccess || !p) {
                g_detail = std::string("fdas_whiten_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e);
                return FDAS_ECUDA;
            }
            g_static_ptr[dev] = static_cast<unsigned char*>(p);
        }
        base = g_static_ptr[dev];
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    fdas::WhitenParams w;
    w.X = reinterpret_cast<const float2*>(d_X);
    w.spec = d_spec;
    int32_t* blk_start = reinterpret_cast<int32_t*>(base);
    int32_t* blk_len = reinterpret_cast<int32_t*>(base + kStaticSection);
    w.blk_start = blk_start;
    w.blk_len = blk_len;
    w.blk_med = reinterpret_cast<float*>(base + 2 * kStaticSection);
    w.nblk = nblk;
    w.nbins = nbins;
    // Nothing in the scratch has to start at zero: the schedule kernel rewrites entries 0..nblk-1 of both
    // tables and K1a rewrites medians 0..nblk-1 before K1b reads them; entries beyond nblk left by a
    // longer earlier call are never read.
    static_schedule_kernel<<<1, 256, 0, st>>>(blk_start, blk_len, (long long)nbins, nblk);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = fdas::launch_whiten(spec_bf16 ? FDAS_BF16 : FDAS_FP32, w, st);
    if (e != cudaSuccess) {
        g_detail = std::string("fdas_whiten_static: launch: ") + cudaGetErrorString(e);
        return FDAS_ECUDA;
    }
    return FDAS_OK;
}

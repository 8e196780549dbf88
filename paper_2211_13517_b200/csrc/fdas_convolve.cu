// fdas_convolve.cu -- K2, the fused convolution stage ("the most computationally
// demanding section (the convolution stage)"; DESIGN.md step a4 + a5).
//
// One CTA (T = L/16 threads, 16 points per thread; L = seg_len = 1024, 2048 or 4096) owns one
// overlap-save segment s and a contiguous chunk of templates:
//   stage-in   g_s[i] = w[sV - h + i] (zero outside [0,Nb)), read once
//   forward    S = FFT_L(g_s) in registers/shared memory, kept in 32 registers per thread
//   loop j     x = S . Khat_j (Khat_j streamed from L2 with 128-bit loads, prefetched one template
//              ahead), y = IFFT_L(x) (three register passes, two shared-memory exchanges),
//              P[j][sV + t] = |y[t]|^2 for the V valid samples only, written once, streaming stores
// so the spectrum is read once and the plane written once.  fp32 arithmetic throughout; the bf16
// variants only change the storage format of w, Khat (and optionally P) -- reading A10.
#include <cuda_bf16.h>

#include "fdas_fft_core.cuh"
#include "fdas_kernels.h"
#include "fdas_maxcode.h"

namespace fdas {

// Resident CTAs per SM each instance is compiled for: 12 warps per SM at L = 1024 and 2048 (3 CTAs of 128
// threads beat 4 at L = 2048: profiles/r01c); L = 4096 keeps 15 pass-3 twiddles in registers as well and
// runs one CTA of 256 threads.
template <int L> struct CtasPerSm { static constexpr int value = L == 1024 ? 6 : L == 2048 ? 3 : 1; };

// First half of the inverse FFT: up to the write of exchange 2 (x is dead afterwards).
template <int L>
__device__ __forceinline__ void ifft_head(float2 (&x)[16], float2* X1, float2* X2, const int tid,
                                          const float2 (&tw1)[15]) {
    pass1(x, tw1);
    x1_store<L>(X1, tid, x);
    __syncthreads();
    xrow_load(X1, tid, x);
    pass2<L>(x);
    x2_store<L>(X2, tid, x);
}
// Second half: barrier, read of exchange 2, last pass.
template <int L>
__device__ __forceinline__ void ifft_tail(float2 (&x)[16], const float2* X2, const int tid,
                                          const float2 (&tw2)[SegGeom<L>::NTw2]) {
    __syncthreads();
    xrow_load(X2, tid, x);
    pass3<L>(x, tw2);
}

// 128-bit read-only loads of the next template, issued as volatile asm after pass 3: the compiler can
// neither sink them to the point of use nor hoist them into the register-heavy passes, so the L2 latency
// is hidden by the epilogue (powers, stores, block maxima) at the cost of 16 (bf16) / 32 (fp32) registers
// over that span only.
__device__ __forceinline__ uint4 ldg_v4(const void* ptr) {
    uint4 v;
    // plain ld.global (not .nc): a non-coherent load may legally be moved across bar.sync
    asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(ptr) : "memory");
    return v;
}


// S K for a stored template value (fp32 pair, or bf16 re in the low half and im in the high half).
__device__ __forceinline__ float2 cmul_k32(float2 s, unsigned kx, unsigned ky) {
    return cmul(s, make_float2(__uint_as_float(kx), __uint_as_float(ky)));
}
__device__ __forceinline__ float2 cmul_k16(float2 s, unsigned v) {
    return cmul(s, make_float2(__uint_as_float(v << 16), __uint_as_float(v & 0xffff0000u)));
}

// Epilogue of one (segment, template).  Ra = 8 (L = 1024, 2048): thread t holds y[2t + e + OutStride q] in
// x[e*8 + q]; Ra = 16 (L = 4096): y[t + 256 q] in x[q].  Writes the powers of the valid samples with
// streaming stores and, for K3's prefilter, an upper bound of the maximum of every aligned block of 8
// plane columns (= 4 or 8 consecutive lanes) of the values AS STORED, as the 16-bit code of
// fdas_maxcode.h (units of 1/8, rounded up; codes order like the values).  Two blocks (q, q+1) share one
// 32-bit word through the shuffles.  `prow` / `mrow` already point at this thread's first column of row j, so every store has an
// immediate offset; q < qmax <=> the sample is valid (r < Nb and t < V), q < qmax_m <=> this lane also
// writes the block maximum.
template <int PREC, int L>
__device__ __forceinline__ void store_powers(const float2 (&x)[16], void* prow, unsigned short* mrow,
                                             const int qmax, const int qmax_m) {
    typedef SegGeom<L> G;
    constexpr int kStride = G::OutStride;
    constexpr int NQ = G::Ra == 16 ? 16 : 8;
#pragma unroll
    for (int q2 = 0; q2 < NQ; q2 += 2) {
        float mx[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int q = q2 + u;
            if constexpr (G::Ra == 16) {
                float p0 = fmaf(x[q].x, x[q].x, x[q].y * x[q].y);
                if (PREC == FDAS_BF16_PLANE16) {
                    const __nv_bfloat16 pk = __float2bfloat16_rn(p0);
                    if (q < qmax)
                        __stcs(reinterpret_cast<unsigned short*>(prow) + kStride * q, __bfloat16_as_ushort(pk));
                    p0 = __bfloat162float(pk);
                } else {
                    if (q < qmax) __stcs(reinterpret_cast<float*>(prow) + kStride * q, p0);
                }
                mx[u] = p0;
            } else {
                float p0 = fmaf(x[q].x, x[q].x, x[q].y * x[q].y);
                float p1 = fmaf(x[8 + q].x, x[8 + q].x, x[8 + q].y * x[8 + q].y);
                if (PREC == FDAS_BF16_PLANE16) {
                    const __nv_bfloat162 pk = __floats2bfloat162_rn(p0, p1);
                    if (q < qmax)
                        __stcs(reinterpret_cast<unsigned int*>(reinterpret_cast<__nv_bfloat16*>(prow) + kStride * q),
                               *reinterpret_cast<const unsigned int*>(&pk));
                    p0 = __low2float(pk);
                    p1 = __high2float(pk);
                } else {
                    if (q < qmax)
                        __stcs(reinterpret_cast<float2*>(reinterpret_cast<float*>(prow) + kStride * q), make_float2(p0, p1));
                }
                mx[u] = fmaxf(p0, p1);
            }
        }
        // block-max codes (fdas_maxcode.h): low half = block q2, high half = block q2 + 1
        unsigned w = max_code2(mx[0], mx[1]);
        w = __vmaxu2(w, __shfl_xor_sync(0xffffffffu, w, 1));
        w = __vmaxu2(w, __shfl_xor_sync(0xffffffffu, w, 2));
        if constexpr (G::Ra == 16) w = __vmaxu2(w, __shfl_xor_sync(0xffffffffu, w, 4));
        if (q2 < qmax_m) mrow[(kStride / 8) * q2] = (unsigned short)w;
        if (q2 + 1 < qmax_m) mrow[(kStride / 8) * (q2 + 1)] = (unsigned short)(w >> 16);
    }
}

template <int PREC, int L>
__global__ void __launch_bounds__(SegGeom<L>::T, CtasPerSm<L>::value) convolve_kernel(const ConvParams p) {
    typedef SegGeom<L> G;
    constexpr int T = G::T;
    extern __shared__ __align__(16) float2 xbuf[];
    float2* const X1 = xbuf;
    float2* const X2 = xbuf + G::XbufElems;
    const int tid = threadIdx.x;
    const int64_t s = blockIdx.x;
    const int per = (p.nz + (int)gridDim.y - 1) / (int)gridDim.y;
    const int jbeg = (int)blockIdx.y * per;
    const int jend = min(p.nz, jbeg + per);
    if (jbeg >= jend) return;

    float2 tw1[15], tw2[G::NTw2];
#pragma unroll
    for (int i = 0; i < 15; ++i) tw1[i] = __ldg(p.tw1 + tid * 15 + i);
#pragma unroll
    for (int i = 0; i < G::NTw2; ++i) tw2[i] = __ldg(p.tw2 + (tid / G::Ra) * G::NTw2 + i);

    // ---- stage-in (conjugated: forward FFT = conj(IFFT(conj g))); thread tid holds bins k0_of(tid) + T k1
    float2 x[16];
    const int64_t g0 = s * p.V - p.h + G::k0_of(tid);
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        const int64_t k = g0 + T * k1;
        float2 v = make_float2(0.f, 0.f);
        if (k >= 0 && k < p.nbins) {
            if (PREC == FDAS_FP32) v = __ldg(reinterpret_cast<const float2*>(p.spec) + k);
            else v = unpack_bf16x2(__ldg(reinterpret_cast<const unsigned int*>(p.spec) + k));
        }
        x[k1] = make_float2(v.x, -v.y);
    }
    ifft_head<L>(x, X1, X2, tid, tw1);
    ifft_tail<L>(x, X2, tid, tw2);
    // x holds conj(S) in output order: to natural order through X1, then to (k0, k1) order
    if constexpr (G::Ra == 16) {
#pragma unroll
        for (int q = 0; q < 16; ++q) X1[tid + G::OutStride * q] = make_float2(x[q].x, -x[q].y);
    } else {
        float4* lin = reinterpret_cast<float4*>(X1);
#pragma unroll
        for (int q = 0; q < 8; ++q)
            lin[tid + (G::OutStride / 2) * q] = make_float4(x[q].x, -x[q].y, x[8 + q].x, -x[8 + q].y);
    }
    __syncthreads();
    float2 S[16];
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) S[k1] = X1[G::k0_of(tid) + T * k1];
    __syncthreads();

    // ---- template loop
    const int64_t sV = s * p.V;
    const int nvalid = (int)min((int64_t)p.V, p.nbins - sV);
    constexpr int NQ = G::Ra == 16 ? 16 : 8;
    const int col0 = G::Ra == 16 ? tid : 2 * tid;          // this thread's first output column of the segment
    const int qmax = max(0, min(NQ, (nvalid - col0 + G::OutStride - 1) / G::OutStride));
    const int qmax_m = (tid & (G::Ra == 16 ? 7 : 3)) == 0 ? qmax : 0;
    constexpr int kPlaneElem = (PREC == FDAS_BF16_PLANE16) ? 2 : 4;
    char* prow = reinterpret_cast<char*>(p.plane) + ((size_t)jbeg * p.pitch + sV + col0) * kPlaneElem;
    const size_t prow_step = (size_t)p.pitch * kPlaneElem;
    unsigned short* mrow = p.maxplane + (size_t)jbeg * p.mpitch + ((sV + col0) >> 3);
    constexpr int NK = (PREC == FDAS_FP32) ? 8 : 4;    // 128-bit words of one template per thread
    const uint4* bank = reinterpret_cast<const uint4*>(p.bank) + (size_t)jbeg * NK * T + tid;
    uint4 K[NK];
#pragma unroll
    for (int c = 0; c < NK; ++c) K[c] = ldg_v4(bank + c * T);
    for (int j = jbeg; j < jend; ++j) {
        if (PREC == FDAS_FP32) {
#pragma unroll
            for (int c = 0; c < NK; ++c) {
                x[2 * c] = cmul_k32(S[2 * c], K[c].x, K[c].y);
                x[2 * c + 1] = cmul_k32(S[2 * c + 1], K[c].z, K[c].w);
            }
        } else {
#pragma unroll
            for (int c = 0; c < NK; ++c) {
                x[4 * c + 0] = cmul_k16(S[4 * c + 0], K[c].x);
                x[4 * c + 1] = cmul_k16(S[4 * c + 1], K[c].y);
                x[4 * c + 2] = cmul_k16(S[4 * c + 2], K[c].z);
                x[4 * c + 3] = cmul_k16(S[4 * c + 3], K[c].w);
            }
        }
        ifft_head<L>(x, X1, X2, tid, tw1);
        bank += NK * T;
        ifft_tail<L>(x, X2, tid, tw2);
        if (j + 1 < jend) {   // the next template, fetched after pass 3 (keeps its registers out of the passes)
#pragma unroll
            for (int c = 0; c < NK; ++c) K[c] = ldg_v4(bank + c * T);
        }
        store_powers<PREC, L>(x, prow, mrow, qmax, qmax_m);
        prow += prow_step;
        mrow += p.mpitch;
    }
}

int convolve_ctas_per_sm(int seg_len) {
    return seg_len == 1024 ? CtasPerSm<1024>::value : seg_len == 4096 ? CtasPerSm<4096>::value : CtasPerSm<2048>::value;
}

template <int PREC, int L>
static cudaError_t launch_one(const ConvParams& p, int64_t nseg, int nsplit, cudaStream_t st) {
    typedef SegGeom<L> G;
    constexpr int smem = 2 * G::XbufElems * (int)sizeof(float2);
    auto kern = convolve_kernel<PREC, L>;
    if (smem > 48 * 1024) {
        static PerDeviceOnce attr;      // per template instance, per device
        const cudaError_t ea = attr.run([&] {
            return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        });
        if (ea != cudaSuccess) return ea;
    }
    kern<<<dim3((unsigned)nseg, (unsigned)nsplit), G::T, smem, st>>>(p);
    return cudaGetLastError();
}

template <int L>
static cudaError_t launch_prec(int precision, const ConvParams& p, int64_t nseg, int nsplit, cudaStream_t st) {
    switch (precision) {
        case FDAS_FP32: return launch_one<FDAS_FP32, L>(p, nseg, nsplit, st);
        case FDAS_BF16: return launch_one<FDAS_BF16, L>(p, nseg, nsplit, st);
        case FDAS_BF16_PLANE16: return launch_one<FDAS_BF16_PLANE16, L>(p, nseg, nsplit, st);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_convolve(int precision, int seg_len, const ConvParams& p, int64_t nseg, int nsplit,
                            cudaStream_t st) {
    switch (seg_len) {
        case 1024: return launch_prec<1024>(precision, p, nseg, nsplit, st);
        case 2048: return launch_prec<2048>(precision, p, nseg, nsplit, st);
        case 4096: return launch_prec<4096>(precision, p, nseg, nsplit, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace fdas

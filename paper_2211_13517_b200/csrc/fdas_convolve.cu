// fdas_convolve.cu -- K2, the fused convolution stage ("the most computationally
// demanding section (the convolution stage)"; DESIGN.md step a4 + a5).
//
// One CTA (128 threads, 16 points per thread) owns one overlap-save segment s and a contiguous
// chunk of templates:
//   stage-in   g_s[i] = w[sV - h + i] (zero outside [0,Nb)), read once, coalesced
//   forward    S = FFT_2048(g_s) in registers/shared memory, kept in 32 registers per thread
//   loop j     x = S . Khat_j (Khat_j streamed from L2 with 128-bit loads, prefetched one template
//              ahead), y = IFFT_2048(x) (three register passes, two shared-memory exchanges),
//              P[j][sV + t] = |y[t]|^2 for the V valid samples only, written once, streaming stores
// so the spectrum is read once and the plane written once.  fp32 arithmetic throughout; the bf16
// variants only change the storage format of w, Khat (and optionally P) -- reading A10.
#include <cuda_bf16.h>

#include "fdas_fft_core.cuh"
#include "fdas_kernels.h"

namespace fdas {

constexpr int kCtasPerSm = 3;   // resident CTAs per SM the kernel is compiled for (3 beat 4: profiles/r01c)

// First half of the inverse FFT: up to the write of exchange 2 (x is dead afterwards).
__device__ __forceinline__ void ifft2048_head(float2 (&x)[16], float2* X1, float2* X2, const int tid,
                                              const float2 (&tw1)[15]) {
    pass1(x, tw1);
    x1_store(X1, tid, x);
    __syncthreads();
    xrow_load(X1, tid, x);
    pass2(x);
    x2_store(X2, tid, x);
}
// Second half: barrier, read of exchange 2, last pass.
__device__ __forceinline__ void ifft2048_tail(float2 (&x)[16], const float2* X2, const int tid,
                                              const float2 (&tw2)[7]) {
    __syncthreads();
    xrow_load(X2, tid, x);
    pass3(x, tw2);
}
__device__ __forceinline__ void ifft2048(float2 (&x)[16], float2* X1, float2* X2, const int tid,
                                         const float2 (&tw1)[15], const float2 (&tw2)[7]) {
    ifft2048_head(x, X1, X2, tid, tw1);
    ifft2048_tail(x, X2, tid, tw2);
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

// Epilogue of one (segment, template): thread t holds y[2t + e + 256 q] in x[e*8 + q].  Writes the
// powers of the valid samples with streaming stores and, for K3's prefilter, an upper bound of the
// maximum of every aligned block of 8 plane columns (= 4 consecutive lanes) of the values AS STORED:
// bf16 rounded toward +inf (powers are >= 0, so adding 0xffff to the bit pattern and truncating
// rounds up; for non-negative values the bf16 order is the order of the bit patterns).  Two blocks
// (q, q+1) share one 32-bit word through the two shuffles.  `prow` / `mrow` already point at this
// thread's first column of row j, so every store has an immediate offset; q < qmax <=> the sample is
// valid (r < Nb and t < V), q < qmax_m <=> this lane also writes the block maximum.
template <int PREC>
__device__ __forceinline__ void store_powers(const float2 (&x)[16], void* prow, unsigned short* mrow,
                                             const int qmax, const int qmax_m) {
#pragma unroll
    for (int q2 = 0; q2 < 8; q2 += 2) {
        float mx[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int q = q2 + u;
            float p0 = fmaf(x[q].x, x[q].x, x[q].y * x[q].y);
            float p1 = fmaf(x[8 + q].x, x[8 + q].x, x[8 + q].y * x[8 + q].y);
            if (PREC == FDAS_BF16_PLANE16) {
                const __nv_bfloat162 pk = __floats2bfloat162_rn(p0, p1);
                if (q < qmax)
                    __stcs(reinterpret_cast<unsigned int*>(reinterpret_cast<__nv_bfloat16*>(prow) + 256 * q),
                           *reinterpret_cast<const unsigned int*>(&pk));
                p0 = __low2float(pk);
                p1 = __high2float(pk);
            } else {
                if (q < qmax)
                    __stcs(reinterpret_cast<float2*>(reinterpret_cast<float*>(prow) + 256 * q), make_float2(p0, p1));
            }
            mx[u] = fmaxf(p0, p1);
        }
        // bytes 2,3 of each rounded-up pattern: low half = block q2, high half = block q2 + 1
        unsigned w = __byte_perm(__float_as_uint(mx[0]) + 0xffffu, __float_as_uint(mx[1]) + 0xffffu, 0x7632);
        w = __vmaxu2(w, __shfl_xor_sync(0xffffffffu, w, 1));
        w = __vmaxu2(w, __shfl_xor_sync(0xffffffffu, w, 2));
        if (q2 < qmax_m) mrow[32 * q2] = (unsigned short)w;
        if (q2 + 1 < qmax_m) mrow[32 * (q2 + 1)] = (unsigned short)(w >> 16);
    }
}

template <int PREC, int MINB>
__global__ void __launch_bounds__(kThreads, MINB) convolve_kernel(const ConvParams p) {
    __shared__ __align__(16) float2 X1[kXbufElems];
    __shared__ __align__(16) float2 X2[kXbufElems];
    const int tid = threadIdx.x;
    const int64_t s = blockIdx.x;
    const int per = (p.nz + (int)gridDim.y - 1) / (int)gridDim.y;
    const int jbeg = (int)blockIdx.y * per;
    const int jend = min(p.nz, jbeg + per);
    if (jbeg >= jend) return;

    float2 tw1[15], tw2[7];
#pragma unroll
    for (int i = 0; i < 15; ++i) tw1[i] = __ldg(p.tw1 + tid * 15 + i);
#pragma unroll
    for (int i = 0; i < 7; ++i) tw2[i] = __ldg(p.tw2 + (tid >> 3) * 7 + i);

    // ---- stage-in (conjugated: forward FFT = conj(IFFT(conj g)))
    float2 x[16];
    const int64_t g0 = s * p.V - p.h + tid;
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        const int64_t k = g0 + 128 * k1;
        float2 v = make_float2(0.f, 0.f);
        if (k >= 0 && k < p.nbins) {
            if (PREC == FDAS_FP32) v = __ldg(reinterpret_cast<const float2*>(p.spec) + k);
            else v = unpack_bf16x2(__ldg(reinterpret_cast<const unsigned int*>(p.spec) + k));
        }
        x[k1] = make_float2(v.x, -v.y);
    }
    ifft2048(x, X1, X2, tid, tw1, tw2);
    // x[e*8 + n2b] = conj(S[2 tid + e + 256 n2b]): to natural order through X1, then to (k0, k1) order
    {
        float4* lin = reinterpret_cast<float4*>(X1);
#pragma unroll
        for (int q = 0; q < 8; ++q)
            lin[tid + 128 * q] = make_float4(x[q].x, -x[q].y, x[8 + q].x, -x[8 + q].y);
    }
    __syncthreads();
    float2 S[16];
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) S[k1] = X1[tid + 128 * k1];
    __syncthreads();

    // ---- template loop
    const int64_t sV = s * p.V;
    const int nvalid = (int)min((int64_t)p.V, p.nbins - sV);
    const int qmax = max(0, min(8, (nvalid - 2 * tid + 255) >> 8));
    const int qmax_m = (tid & 3) == 0 ? qmax : 0;
    constexpr int kPlaneElem = (PREC == FDAS_BF16_PLANE16) ? 2 : 4;
    char* prow = reinterpret_cast<char*>(p.plane) + ((size_t)jbeg * p.pitch + sV + 2 * tid) * kPlaneElem;
    const size_t prow_step = (size_t)p.pitch * kPlaneElem;
    unsigned short* mrow = p.maxplane + (size_t)jbeg * p.mpitch + ((sV + 2 * tid) >> 3);
    constexpr int NK = (PREC == FDAS_FP32) ? 8 : 4;    // 128-bit words of one template per thread
    const uint4* bank = reinterpret_cast<const uint4*>(p.bank) + (size_t)jbeg * NK * 128 + tid;
    uint4 K[NK];
#pragma unroll
    for (int c = 0; c < NK; ++c) K[c] = ldg_v4(bank + c * 128);
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
        ifft2048_head(x, X1, X2, tid, tw1);
        bank += NK * 128;
        ifft2048_tail(x, X2, tid, tw2);
        if (j + 1 < jend) {   // the next template, fetched after pass 3 (keeps its registers out of the passes)
#pragma unroll
            for (int c = 0; c < NK; ++c) K[c] = ldg_v4(bank + c * 128);
        }
        store_powers<PREC>(x, prow, mrow, qmax, qmax_m);
        prow += prow_step;
        mrow += p.mpitch;
    }
}

int convolve_ctas_per_sm() { return kCtasPerSm; }

cudaError_t launch_convolve(int precision, const ConvParams& p, int64_t nseg, int nsplit,
                            cudaStream_t st) {
    const dim3 grid((unsigned)nseg, (unsigned)nsplit), block(kThreads);
    switch (precision) {
        case FDAS_FP32: convolve_kernel<FDAS_FP32, kCtasPerSm><<<grid, block, 0, st>>>(p); break;
        case FDAS_BF16: convolve_kernel<FDAS_BF16, kCtasPerSm><<<grid, block, 0, st>>>(p); break;
        case FDAS_BF16_PLANE16: convolve_kernel<FDAS_BF16_PLANE16, kCtasPerSm><<<grid, block, 0, st>>>(p); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace fdas

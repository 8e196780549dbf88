// fdas_fft_core.cuh -- per-thread building blocks of the L-point segment FFT (L = 1024, 2048, 4096) used by
// the fused convolution kernel (fdas_convolve.cu).  Every function is __host__ __device__ so that the exact
// index arithmetic and exchange-buffer layouts can also be stepped on the CPU, thread by thread, by
// the test-only emulator (tests/emu/fdas_emu.cu) -- there is no GPU on the development box.
//
// Inverse transform y[n] = sum_p Y[p] exp(+2 pi i n p / L) (unnormalised), T = L/16 threads x 16 points,
// three register passes (16 x Rb x Ra, L = 16 Ra Rb) with two shared-memory exchanges:
//   p = k0 + T k1               k0 = kA + Ra kB in [0,T), kA in [0,Ra), kB in [0,Rb), k1 in [0,16)
//   n = n1 + 16 (nB + Rb nA)    n1 in [0,16), nB in [0,Rb), nA in [0,Ra)
//   pass 1 (thread tid = kB + Rb kA)   A[n1]  = wL^(n1 k0) * sum_k1 Y[k0 + T k1] w16^(n1 k1)
//   pass 2 (row (n1, kA))              C[nB]  = sum_kB A[n1][kA + Ra kB] wRb^(nB kB)
//   pass 3 (row (n1, nB))              y[n1 + 16 nB + 16 Rb nA] = sum_kA wT^(nB kA) C[kA][nB] wRa^(nA kA)
// with wN^(x) = exp(+2 pi i x / N).  A pass of radix 16 is one 16-point DFT per thread, a pass of radix 8
// two 8-point DFTs per thread (rows of 16 = two groups of 8).  L = 1024: Rb = Ra = 8; 2048: Rb = 16,
// Ra = 8; 4096: Rb = Ra = 16.  Convolution stage of PAPER.md:23 (section 2.2).
#pragma once
#include <cuda_runtime.h>

#define FDAS_HD __host__ __device__ __forceinline__

namespace fdas {

constexpr int kPts = 16;        // points per thread
constexpr int kRowStride = 18;  // float2 per exchange-buffer row: 16 data + 2 pad (144 B: LDS.128 conflict-free)

// Geometry of the L-point segment transform.
template <int L>
struct SegGeom {
    static_assert(L == 1024 || L == 2048 || L == 4096, "segment lengths built: 1024, 2048, 4096");
    static constexpr int kL = L;
    static constexpr int T = L / 16;                   // threads per segment
    static constexpr int Rb = (L == 1024) ? 8 : 16;    // radix of pass 2 (over kB)
    static constexpr int Ra = T / Rb;                  // radix of pass 3 (over kA): 8, 8, 16
    static constexpr int RowsPerN1 = T / 16;           // exchange-1 rows that share one n1
    static constexpr int NTw2 = Ra - 1;                // pass-3 twiddles per thread
    static constexpr int OutStride = 16 * Rb;          // thread v holds y[m + OutStride nA]
    static constexpr int XbufElems = T * kRowStride;   // float2 elements per exchange buffer
    // The input bin k0 of thread tid (tid = kB + Rb kA holds Y[k0 + T k1], k0 = kA + Ra kB): with this
    // assignment the 16 (8) threads that feed one pass-2 row are consecutive, so a half-warp writes one
    // contiguous 128-byte row segment in both exchanges.
    static __host__ __device__ constexpr int k0_of(int tid) { return tid / Rb + Ra * (tid % Rb); }
};

// ---- complex arithmetic on (re, im) register pairs.
// On sm_100a every operation below is ONE packed instruction (FADD2 / FMUL2 / FFMA2, PTX *.f32x2):
// two IEEE fp32 results per issue slot, rounding identical to the scalar forms.  ptxas folds the
// mov.b64 pack/unpack of the operands into SASS operand modifiers (.F32 broadcast, .LO_HI swap,
// per-half negation on FADD2), so multiplying by +-i never costs an instruction.  The host forms
// (test-only emulator) spell out the same arithmetic.
#ifdef __CUDA_ARCH__
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk2(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float2 up2(u64 v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
#endif

FDAS_HD float2 cconj(float2 a) { return make_float2(a.x, -a.y); }
FDAS_HD float2 cadd(float2 a, float2 b) {   // a + b
#ifdef __CUDA_ARCH__
    return up2(add2(pk2(a.x, a.y), pk2(b.x, b.y)));
#else
    return make_float2(a.x + b.x, a.y + b.y);
#endif
}
FDAS_HD float2 csub(float2 a, float2 b) {   // a - b
#ifdef __CUDA_ARCH__
    return up2(add2(pk2(a.x, a.y), pk2(-b.x, -b.y)));
#else
    return make_float2(a.x - b.x, a.y - b.y);
#endif
}
FDAS_HD float2 cadd_i(float2 a, float2 b) {  // a + i b
#ifdef __CUDA_ARCH__
    return up2(add2(pk2(a.x, a.y), pk2(-b.y, b.x)));
#else
    return make_float2(a.x - b.y, a.y + b.x);
#endif
}
FDAS_HD float2 csub_i(float2 a, float2 b) {  // a - i b
#ifdef __CUDA_ARCH__
    return up2(add2(pk2(a.x, a.y), pk2(b.y, -b.x)));
#else
    return make_float2(a.x + b.y, a.y - b.x);
#endif
}
FDAS_HD float2 rot45(float2 a) { return cadd_i(a, a); }     // a (1 + i):  sqrt2 w8^1 a
FDAS_HD float2 rot135(float2 a) {                           // a (-1 + i): sqrt2 w8^3 a
#ifdef __CUDA_ARCH__
    return up2(add2(pk2(-a.x, -a.y), pk2(-a.y, a.x)));
#else
    return make_float2(-a.x - a.y, a.x - a.y);
#endif
}
FDAS_HD float2 cscale(float2 a, const float r) {            // r a, r real
#ifdef __CUDA_ARCH__
    return up2(mul2(pk2(a.x, a.y), pk2(r, r)));
#else
    return make_float2(a.x * r, a.y * r);
#endif
}
FDAS_HD float2 caxpy(const float r, float2 a, float2 c) {   // c + r a, r real
#ifdef __CUDA_ARCH__
    return up2(fma2(pk2(a.x, a.y), pk2(r, r), pk2(c.x, c.y)));
#else
    return make_float2(fmaf(r, a.x, c.x), fmaf(r, a.y, c.y));
#endif
}
FDAS_HD float2 caxpy_i(const float r, float2 a, float2 c) {  // c + r (i a), r real
#ifdef __CUDA_ARCH__
    return up2(fma2(pk2(-a.y, a.x), pk2(r, r), pk2(c.x, c.y)));
#else
    return make_float2(fmaf(r, -a.y, c.x), fmaf(r, a.x, c.y));
#endif
}
// a w = w.x a + w.y (i a): FMUL2 + FFMA2.  The swapped, half-negated pair (-a.y, a.x) must be the
// FIRST multiplicand: only operands A and C of FFMA2 take the per-half sign, B takes the broadcast.
FDAS_HD float2 cmul(float2 a, float2 w) {
#ifdef __CUDA_ARCH__
    return up2(fma2(pk2(-a.y, a.x), pk2(w.y, w.y), mul2(pk2(a.x, a.y), pk2(w.x, w.x))));
#else
    return make_float2(fmaf(-a.y, w.y, a.x * w.x), fmaf(a.x, w.y, a.y * w.x));
#endif
}

// y_d = sum_a x_a (+i)^(a d), in place.
FDAS_HD void bfly4_inv(float2& x0, float2& x1, float2& x2, float2& x3) {
    const float2 t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), d = csub(x1, x3);
    x0 = cadd(t0, t2);
    x1 = cadd_i(t1, d);
    x2 = csub(t0, t2);
    x3 = csub_i(t1, d);
}
// Same butterfly with x2 = R u2 still unscaled (the 1/sqrt2 of a w8-type twiddle folded into FMAs).
FDAS_HD void bfly4_inv_s2(float2& x0, float2& x1, float2& u2, float2& x3, const float R) {
    const float2 t0 = caxpy(R, u2, x0), t1 = caxpy(-R, u2, x0), t2 = cadd(x1, x3), d = csub(x1, x3);
    x0 = cadd(t0, t2);
    x1 = cadd_i(t1, d);
    u2 = csub(t0, t2);
    x3 = csub_i(t1, d);
}
// ... with x1 = R u1, x3 = R u3 unscaled and x2 = i v2 (v2 not yet rotated).
FDAS_HD void bfly4_inv_s13_i2(float2& x0, float2& u1, float2& v2, float2& u3, const float R) {
    const float2 t0 = cadd_i(x0, v2), t1 = csub_i(x0, v2), w = cadd(u1, u3), d = csub(u1, u3);
    x0 = caxpy(R, w, t0);
    u1 = caxpy_i(R, d, t1);
    v2 = caxpy(-R, w, t0);
    u3 = caxpy_i(-R, d, t1);
}

// 16-point inverse DFT, natural order in and out: x[n] <- sum_k x[k] exp(+2 pi i n k / 16).
// k = b + 4a, n = d + 4c: radix-4 over a, twiddle w16^(b d), radix-4 over b.  76 packed instructions.
FDAS_HD void dft16_inv(float2 (&x)[16]) {
    const float C1 = 0.92387953251128673848f;  // cos(pi/8)
    const float S1 = 0.38268343236508978178f;  // sin(pi/8)
    const float R = 0.70710678118654752440f;   // sqrt(1/2)
#pragma unroll
    for (int b = 0; b < 4; ++b) bfly4_inv(x[b], x[b + 4], x[b + 8], x[b + 12]);  // -> E_b[d] at x[b+4d]
    // twiddles w16^(b d); the w8-type ones (b d = 2 or 6) keep their 1/sqrt2 for the next stage and
    // w16^4 = i is absorbed by the butterfly of d = 2
    x[1 + 4] = cmul(x[1 + 4], make_float2(C1, S1));      // b=1 d=1: w16^1
    x[1 + 8] = rot45(x[1 + 8]);                          // b=1 d=2: w16^2 (x R later)
    x[1 + 12] = cmul(x[1 + 12], make_float2(S1, C1));    // b=1 d=3: w16^3
    x[2 + 4] = rot45(x[2 + 4]);                          // b=2 d=1: w16^2 (x R later)
    x[2 + 12] = rot135(x[2 + 12]);                       // b=2 d=3: w16^6 (x R later)
    x[3 + 4] = cmul(x[3 + 4], make_float2(S1, C1));      // b=3 d=1: w16^3
    x[3 + 8] = rot135(x[3 + 8]);                         // b=3 d=2: w16^6 (x R later)
    x[3 + 12] = cmul(x[3 + 12], make_float2(-C1, -S1));  // b=3 d=3: w16^9 = -w16^1
    bfly4_inv(x[0], x[1], x[2], x[3]);                   // d = 0: F_0[c] at x[c]
    bfly4_inv_s2(x[4], x[5], x[6], x[7], R);             // d = 1: b = 2 unscaled
    bfly4_inv_s13_i2(x[8], x[9], x[10], x[11], R);       // d = 2: b = 1, 3 unscaled, b = 2 times i
    bfly4_inv_s2(x[12], x[13], x[14], x[15], R);         // d = 3: b = 2 unscaled
    float2 y[16];
#pragma unroll
    for (int d = 0; d < 4; ++d)
#pragma unroll
        for (int c = 0; c < 4; ++c) y[d + 4 * c] = x[c + 4 * d];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = y[i];
}

// 8-point inverse DFT on x[o..o+7], natural order in and out.  k = b + 4a, n = d + 2c.
FDAS_HD void dft8_inv(float2 (&x)[16], const int o) {
    const float R = 0.70710678118654752440f;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const float2 s = cadd(x[o + b], x[o + b + 4]), t = csub(x[o + b], x[o + b + 4]);
        x[o + b] = s;        // E_b[0]
        x[o + b + 4] = t;    // E_b[1]
    }
    // twiddle w8^(b) on E_b[1]: b = 1 -> (1+i)/sqrt2, b = 2 -> i, b = 3 -> (-1+i)/sqrt2 (R and i folded below)
    x[o + 5] = rot45(x[o + 5]);
    x[o + 7] = rot135(x[o + 7]);
    bfly4_inv(x[o + 0], x[o + 1], x[o + 2], x[o + 3]);             // d = 0: F_0[c] at x[o+c]
    bfly4_inv_s13_i2(x[o + 4], x[o + 5], x[o + 6], x[o + 7], R);   // d = 1: F_1[c] at x[o+4+c]
    float2 y[8];
#pragma unroll
    for (int d = 0; d < 2; ++d)
#pragma unroll
        for (int c = 0; c < 4; ++c) y[d + 2 * c] = x[o + c + 4 * d];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[o + i] = y[i];
}

// ---- pass 1: thread tid holds x[k1] = Y[k0_of(tid) + T k1];  tw1[n1-1] = wL^(n1 * k0_of(tid))
FDAS_HD void pass1(float2 (&x)[16], const float2 (&tw1)[15]) {
    dft16_inv(x);
#pragma unroll
    for (int n1 = 1; n1 < 16; ++n1) x[n1] = cmul(x[n1], tw1[n1 - 1]);
}

// Exchange 1 write: element (n1, kA, kB) of thread tid = kB + Rb kA goes to row n1 (T/16) + tid/16,
// column tid % 16 -- for Rb = 16 that is row (n1, kA), column kB; for Rb = 8 row (n1, kA/2), column
// 8 (kA % 2) + kB.  16 x 64-bit stores; a half-warp writes one contiguous 128-byte row segment.
template <int L>
FDAS_HD void x1_store(float2* X1, const int tid, const float2 (&x)[16]) {
    const int base = (tid >> 4) * kRowStride + (tid & 15);
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) X1[base + n1 * SegGeom<L>::RowsPerN1 * kRowStride] = x[n1];
}

// Row read used after both exchanges: thread tid reads its own 16-element row with 8 x 128-bit
// loads (row pitch 144 B rotates consecutive threads over the eight 16-byte bank groups).
FDAS_HD void xrow_load(const float2* X, const int tid, float2 (&x)[16]) {
    const float4* p = reinterpret_cast<const float4*>(X + tid * kRowStride);
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        float4 v = p[c];
        x[2 * c] = make_float2(v.x, v.y);
        x[2 * c + 1] = make_float2(v.z, v.w);
    }
}

// ---- pass 2: thread u = n1 (T/16) + w holds row (n1, w).  Rb = 16: x[kB] of kA = w -> x[nB];
// Rb = 8: x[8 e + kB] of kA = 2 w + e -> x[8 e + nB].
template <int L>
FDAS_HD void pass2(float2 (&x)[16]) {
    if constexpr (SegGeom<L>::Rb == 16) {
        dft16_inv(x);
    } else {
        dft8_inv(x, 0);
        dft8_inv(x, 8);
    }
}

// Exchange 2 write by thread u = n1 (T/16) + w: element (n1, kA, nB) goes to the pass-3 row of (n1, nB),
// column kA (Ra = 16: row n1 + 16 nB) or column 8 (n1 % 2) + kA (Ra = 8: row n1/2 + 8 nB, shared by
// n1 = 2a, 2a+1).  A half-warp (a quarter-warp of the 128-bit stores of L = 1024) writes one contiguous
// 128-byte row segment.
template <int L>
FDAS_HD void x2_store(float2* X2, const int u, const float2 (&x)[16]) {
    typedef SegGeom<L> G;
    const int n1 = u / G::RowsPerN1, w = u % G::RowsPerN1;
    if constexpr (G::Ra == 16) {
        const int base = n1 * kRowStride + w;
#pragma unroll
        for (int nB = 0; nB < 16; ++nB) X2[base + nB * 16 * kRowStride] = x[nB];
    } else if constexpr (G::Rb == 16) {
        const int base = (n1 >> 1) * kRowStride + (n1 & 1) * 8 + w;
#pragma unroll
        for (int nB = 0; nB < 16; ++nB) X2[base + nB * 8 * kRowStride] = x[nB];
    } else {
        const int base = (n1 >> 1) * kRowStride + (n1 & 1) * 8 + 2 * w;     // kA = 2 w, 2 w + 1: one 16-byte store
#pragma unroll
        for (int nB = 0; nB < 8; ++nB)
            *reinterpret_cast<float4*>(X2 + base + nB * 8 * kRowStride) = make_float4(x[nB].x, x[nB].y, x[8 + nB].x, x[8 + nB].y);
    }
}

// ---- pass 3: thread v holds its row of kA values; tw2[kA-1] = wT^(nB kA), nB = v / 16 (Ra = 16) or v / 8.
// Ra = 16: x[kA] of (n1, nB) = (v % 16, v / 16) -> x[nA] = y[v + 256 nA].
// Ra = 8:  x[8 e + kA] of n1 = 2 (v % 8) + e, nB = v / 8 -> x[8 e + nA] = y[2 v + e + 16 Rb nA].
template <int L>
FDAS_HD void pass3(float2 (&x)[16], const float2 (&tw2)[SegGeom<L>::NTw2]) {
    if constexpr (SegGeom<L>::Ra == 16) {
#pragma unroll
        for (int k = 1; k < 16; ++k) x[k] = cmul(x[k], tw2[k - 1]);
        dft16_inv(x);
    } else {
#pragma unroll
        for (int k = 1; k < 8; ++k) {
            x[k] = cmul(x[k], tw2[k - 1]);
            x[8 + k] = cmul(x[8 + k], tw2[k - 1]);
        }
        dft8_inv(x, 0);
        dft8_inv(x, 8);
    }
}
// Output index of x[i] after pass 3 in thread v.
template <int L>
FDAS_HD int out_index(const int v, const int i) {
    typedef SegGeom<L> G;
    return G::Ra == 16 ? v + G::OutStride * i : 2 * v + (i >> 3) + G::OutStride * (i & 7);
}

// Round-to-nearest-even float -> bfloat16 bits and back (storage format of the bf16 path,
// PAPER.md:23; reading A10).
FDAS_HD unsigned short f32_to_bf16_rne(float f) {
    union { float f; unsigned int u; } v;
    v.f = f;
    unsigned int u = v.u;
    u += 0x7fffu + ((u >> 16) & 1u);
    return (unsigned short)(u >> 16);
}
FDAS_HD float bf16_bits_to_f32(unsigned int hi16) {
    union { float f; unsigned int u; } v;
    v.u = hi16 << 16;
    return v.f;
}
FDAS_HD unsigned int pack_bf16x2(float re, float im) {  // low half = re, high half = im
    return (unsigned int)f32_to_bf16_rne(re) | ((unsigned int)f32_to_bf16_rne(im) << 16);
}
FDAS_HD float2 unpack_bf16x2(unsigned int v) {
    union { float f; unsigned int u; } lo, hi;
    lo.u = v << 16;
    hi.u = v & 0xffff0000u;
    return make_float2(lo.f, hi.f);
}

}  // namespace fdas

// fdas_maxcode.h -- the block-max side plane M that K2 / K2-TC write beside the plane and K3's
// branch-and-bound prefilter scans (K3).  One 16-bit CODE per aligned block of 8 plane columns:
//     c = min(kMaxCodeSat, ceil(kMaxCodeScale * max of the 8 values AS STORED))
// so that c / kMaxCodeScale >= every value of the block (an upper bound, exact in fp32: the scale is a
// power of two), and c = kMaxCodeSat says "no bound" (a block holding a value >= 127.875).  Integer codes
// let the prefilter sum two fundamentals per 32-bit add: 32 harmonics x 1023 < 2^15, so the packed sums
// never carry from one half-word into the other.  NaN and negative maxima give code 0.
#pragma once
#include <cuda_runtime.h>

namespace fdas {

constexpr unsigned kMaxCodeSat = 1023u;
constexpr float kMaxCodeScale = 8.0f;

__host__ __device__ inline unsigned max_code(float m) {
#ifdef __CUDA_ARCH__
    // ceil(8 t) without a float-to-integer conversion (a quarter-rate instruction): 8 t + 2^23 rounded toward
    // +inf is the integer ceil(8 t) + 2^23 (floats are spaced by 1 there), whose low bits are the code.
    // t is clamped to [0, 1023/8] first (fmaxf drops a NaN: code 0).
    const float t = fminf(fmaxf(m, 0.f), (float)kMaxCodeSat / kMaxCodeScale);
    return __float_as_uint(__fmaf_ru(t, kMaxCodeScale, 8388608.0f)) & 0xffffu;
#else
    const float t = m * kMaxCodeScale;
    if (!(t > 0.f)) return 0u;
    if (t >= (float)kMaxCodeSat) return kMaxCodeSat;
    const unsigned f = (unsigned)t;
    return (float)f < t ? f + 1u : f;
#endif
}

#ifdef __CUDACC__
// The codes of two maxima in one word (a in the low half): the low half-words of the two sums above.
__device__ __forceinline__ unsigned max_code2(float a, float b) {
    const float lim = (float)kMaxCodeSat / kMaxCodeScale;
    const float ta = fminf(fmaxf(a, 0.f), lim), tb = fminf(fmaxf(b, 0.f), lim);
    return __byte_perm(__float_as_uint(__fmaf_ru(ta, kMaxCodeScale, 8388608.0f)),
                       __float_as_uint(__fmaf_ru(tb, kMaxCodeScale, 8388608.0f)), 0x5410);
}
#endif

}  // namespace fdas

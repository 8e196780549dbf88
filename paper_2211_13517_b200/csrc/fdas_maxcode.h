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
    return min(__float2uint_ru(m * kMaxCodeScale), kMaxCodeSat);   // NaN -> 0, +inf -> saturated
#else
    const float t = m * kMaxCodeScale;
    if (!(t > 0.f)) return 0u;
    if (t >= (float)kMaxCodeSat) return kMaxCodeSat;
    const unsigned f = (unsigned)t;
    return (float)f < t ? f + 1u : f;
#endif
}

}  // namespace fdas

// fdas_host.h -- host-side (plan-time) mathematics of libfdas: template bank, twiddle tables,
// whitening block schedule, thresholds.  Pure C++ (no CUDA calls) so it also links into the
// test-only emulator.  Shares nothing with oracle/.
#pragma once
#include <complex>
#include <cstdint>
#include <vector>

namespace fdas {

typedef std::complex<double> cd;

// Fresnel integrals C(t) = int_0^t cos(pi s^2/2) ds, S(t) = int_0^t sin(pi s^2/2) ds.
void fresnel_cs(double t, double* C, double* S);

// Half-width rule (reading A5): h = round-up-to-multiple-of-32(ceil(zmax/2) + 16).
int template_halfwidth(double zmax);

// Closed-form response of a constant-fdot signal (Ransom et al. 2002; reading A4):
// T_z[m], m = -h..h, truncated and scaled to unit L2 norm.  out has 2h+1 entries.
void template_response(double z, int h, cd* out);

struct Bank {
    int nz = 0, h = 0, L = 0;
    std::vector<cd> time;      // nz x (2h+1): unit-norm T_j[m]
    std::vector<cd> freq;      // nz x L: Khat_j[p] = conj(FFT_L(c_j))[p] / L, c_j[i] = T_j[i-h]
};
void build_bank(double zmax, double zstep, int nz, int h, int L, Bank* bank);

// In-place iterative radix-2 FFT (sign = -1 forward, +1 inverse, unnormalised).
void host_fft(cd* a, int n, int sign);

// Segment lengths the FFT kernel is built for, and the input bin k0 of thread tid of its CTA
// (fdas_fft_core.cuh SegGeom: T = L/16 threads, tid = kB + Rb kA holds bins k0 + T k1, k0 = kA + Ra kB).
bool seg_len_supported(int L);
int seg_k0_of(int L, int tid);

// Kernel register order: thread tid holds Khat[k0_of(tid) + T k1], k1 = 0..15.
// fp32: float4 words [nz][8][T] = {K[k0+T(2c)], K[k0+T(2c+1)]}  (re, im, re, im)
// bf16: uint4  words [nz][4][T] = 4 complex k1 = 4c..4c+3, each (bf16 im << 16) | bf16 re
void pack_bank_fp32(const Bank& bank, std::vector<float>* out);
void pack_bank_bf16(const Bank& bank, std::vector<uint32_t>* out);

// K2-TC operand geometry (fdas_convolve_tc.cu).  The nz templates are npair = nz/2 conjugate pairs
// (T_{-z} = conj(T_z)) plus, for odd nz, the z = 0 row; pair p is rows j+ = nz - npair + p and
// j- = npair - 1 - p.
struct TcGeom {
    int npair = 0;    // nz / 2 conjugate pairs
    int kp = 0;       // taps 2h+1 padded to a multiple of 16
    int nchunk = 0;   // kernel launches: the kernel holds up to 128 pairs (one TMEM lane each)
    int chunk = 0;    // pairs per launch (a multiple of 32; the last launch takes the remainder)
};
// false when the bank does not fit the kernel (no pair at all, or too many taps for the tensor-memory
// columns left beside the accumulators).
bool tc_geometry(int nz, int h, TcGeom* g);
// Bank images for tensor memory, one per launch c: word [((c*2 + part)*128 + l)*(kp/2) + w] =
// bf16(X[2w]) | bf16(X[2w+1]) << 16 (RNE), X[k] = Re (part 0) or Im (part 1) of T_{j+(p)}[k - h] for pair
// p = c*chunk + l, zero for k > 2h and for lanes beyond the launch's pairs.
// *asym receives max |T_{j-}[m] - conj(T_{j+}[m])| over the bank (must be ~1e-16 for the pairing).
void pack_bank_tc(const Bank& bank, const TcGeom& g, std::vector<uint32_t>* out, double* asym);

// tw1[tid][n1-1] = exp(+2 pi i n1 k0_of(tid) / L), n1 = 1..15 (T x 15 complex fp32)
// tw2[nB][kA-1]  = exp(+2 pi i nB kA / T), nB = 0..Rb-1, kA = 1..Ra-1 (Rb x (Ra-1) complex fp32)
void build_twiddles(int L, std::vector<float>* tw1, std::vector<float>* tw2);

// Whitening block schedule (reading A3): s_0 = 1, len = clamp(2^(floor(log2 s) - 2), 32, 4096),
// truncated at nb.
void whitening_blocks(int64_t nb, std::vector<int32_t>* start, std::vector<int32_t>* len);

// T_h with Q(h, T_h) = erfc(nsigma/sqrt 2)/2 (reading A13).
int thresholds_from_sigma(int H, double nsigma, float* out);

}  // namespace fdas

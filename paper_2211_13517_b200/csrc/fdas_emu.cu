// fdas_emu.cu -- TEST-ONLY host emulator of the K2 CTA (libfdas_emu.so).  NOT part of the product:
// libfdas.so does not contain it and the Python binding never loads it.  It steps the exact
// __host__ __device__ building blocks of fdas_fft_core.cuh thread by thread, phase by phase (one
// loop over the 128 "threads" per barrier interval), with the same packed template bank, twiddle
// tables and index arithmetic as fdas_convolve.cu, so that layout or indexing mistakes show up in
// the CPU test-suite (tests/test_host_logic.py) on a box without a GPU.  It also exposes the
// plan-time host mathematics (templates, Fresnel integrals, thresholds, whitening blocks) for the
// same purpose.
#include <cstring>
#include <vector>

#include "../../include/fdas.h"
#include "fdas_fft_core.cuh"
#include "fdas_host.h"

using namespace fdas;

namespace {

struct Cta {
    float2 x[kThreads][16];
    float2 S[kThreads][16];
    float2 tw1[kThreads][15];
    float2 tw2[kThreads][7];
    std::vector<float2> X1, X2;
    Cta() : X1(kXbufElems), X2(kXbufElems) {}
};

void emu_ifft2048(Cta& c) {
    for (int t = 0; t < kThreads; ++t) { pass1(c.x[t], c.tw1[t]); x1_store(c.X1.data(), t, c.x[t]); }
    for (int t = 0; t < kThreads; ++t) { xrow_load(c.X1.data(), t, c.x[t]); pass2(c.x[t]); x2_store(c.X2.data(), t, c.x[t]); }
    for (int t = 0; t < kThreads; ++t) { xrow_load(c.X2.data(), t, c.x[t]); pass3(c.x[t], c.tw2[t]); }
}

}  // namespace

extern "C" {

int fdas_emu_fresnel(double t, double* C, double* S) { fresnel_cs(t, C, S); return 0; }

int fdas_emu_halfwidth(double zmax) { return template_halfwidth(zmax); }

// out: nz x (2h+1) complex doubles (interleaved)
int fdas_emu_templates(double zmax, double zstep, int nz, int h, double* out) {
    std::vector<cd> T(2 * h + 1);
    for (int j = 0; j < nz; ++j) {
        template_response(-zmax + j * zstep, h, T.data());
        std::memcpy(out + (size_t)j * 2 * (2 * h + 1), T.data(), sizeof(cd) * (2 * h + 1));
    }
    return 0;
}

int fdas_emu_thresholds(int H, double nsigma, float* out) { return thresholds_from_sigma(H, nsigma, out); }

int64_t fdas_emu_whitening_blocks(int64_t nb, int32_t* start, int32_t* len, int64_t cap) {
    std::vector<int32_t> s, l;
    whitening_blocks(nb, &s, &l);
    for (size_t i = 0; i < s.size() && (int64_t)i < cap; ++i) { start[i] = s[i]; len[i] = l[i]; }
    return (int64_t)s.size();
}

// 2048-point inverse FFT of one vector through the emulated CTA (natural order in and out).
int fdas_emu_ifft2048(const float* in, float* out) {
    std::vector<float> t1, t2;
    build_twiddles(&t1, &t2);
    Cta* c = new Cta();
    for (int t = 0; t < kThreads; ++t) {
        for (int i = 0; i < 15; ++i) c->tw1[t][i] = make_float2(t1[(t * 15 + i) * 2], t1[(t * 15 + i) * 2 + 1]);
        for (int i = 0; i < 7; ++i) c->tw2[t][i] = make_float2(t2[((t >> 3) * 7 + i) * 2], t2[((t >> 3) * 7 + i) * 2 + 1]);
        for (int k1 = 0; k1 < 16; ++k1) c->x[t][k1] = make_float2(in[2 * (t + 128 * k1)], in[2 * (t + 128 * k1) + 1]);
    }
    emu_ifft2048(*c);
    for (int t = 0; t < kThreads; ++t)
        for (int e = 0; e < 2; ++e)
            for (int q = 0; q < 8; ++q) {
                const int n = 2 * t + e + 256 * q;
                out[2 * n] = c->x[t][e * 8 + q].x;
                out[2 * n + 1] = c->x[t][e * 8 + q].y;
            }
    delete c;
    return 0;
}

// Emulated fdas_convolve_plane: spec = nb complex fp32 (interleaved); plane = nz x nb floats.
// precision FDAS_BF16*: spec and bank are first rounded to bf16 exactly as the device path stores
// them; FDAS_BF16_PLANE16 additionally rounds the stored powers to bf16 (returned as float).
int fdas_emu_convolve(const float* spec, int64_t nb, double zmax, double zstep, int precision,
                      float* plane) {
    const int L = kL;
    const int nz = (int)(2.0 * zmax / zstep + 0.5) + 1;
    const int h = template_halfwidth(zmax);
    const int V = L - 2 * h;
    if (V <= 0) return FDAS_EARG;
    const int64_t nseg = (nb + V - 1) / V;
    Bank bank;
    build_bank(zmax, zstep, nz, h, L, &bank);
    std::vector<float> bank32;
    std::vector<uint32_t> bank16;
    if (precision == FDAS_FP32) pack_bank_fp32(bank, &bank32); else pack_bank_bf16(bank, &bank16);
    std::vector<float> t1, t2;
    build_twiddles(&t1, &t2);
    Cta* c = new Cta();
    for (int t = 0; t < kThreads; ++t) {
        for (int i = 0; i < 15; ++i) c->tw1[t][i] = make_float2(t1[(t * 15 + i) * 2], t1[(t * 15 + i) * 2 + 1]);
        for (int i = 0; i < 7; ++i) c->tw2[t][i] = make_float2(t2[((t >> 3) * 7 + i) * 2], t2[((t >> 3) * 7 + i) * 2 + 1]);
    }
    for (int64_t s = 0; s < nseg; ++s) {
        // stage-in, conjugated
        for (int t = 0; t < kThreads; ++t) {
            const int64_t g0 = s * V - h + t;
            for (int k1 = 0; k1 < 16; ++k1) {
                const int64_t k = g0 + 128 * k1;
                float2 v = make_float2(0.f, 0.f);
                if (k >= 0 && k < nb) {
                    v = make_float2(spec[2 * k], spec[2 * k + 1]);
                    if (precision != FDAS_FP32) v = unpack_bf16x2(pack_bf16x2(v.x, v.y));
                }
                c->x[t][k1] = make_float2(v.x, -v.y);
            }
        }
        emu_ifft2048(*c);
        float4* lin = reinterpret_cast<float4*>(c->X1.data());
        for (int t = 0; t < kThreads; ++t)
            for (int q = 0; q < 8; ++q)
                lin[t + 128 * q] = make_float4(c->x[t][q].x, -c->x[t][q].y, c->x[t][8 + q].x, -c->x[t][8 + q].y);
        for (int t = 0; t < kThreads; ++t)
            for (int k1 = 0; k1 < 16; ++k1) c->S[t][k1] = c->X1[t + 128 * k1];
        const int64_t sV = s * V;
        const int nvalid = (int)((nb - sV) < V ? (nb - sV) : V);
        for (int j = 0; j < nz; ++j) {
            for (int t = 0; t < kThreads; ++t) {
                if (precision == FDAS_FP32) {
                    const float* b = bank32.data() + ((size_t)j * 8 * 128 + t) * 4;
                    for (int q = 0; q < 8; ++q) {
                        const float* K = b + (size_t)q * 128 * 4;
                        c->x[t][2 * q] = cmul(c->S[t][2 * q], make_float2(K[0], K[1]));
                        c->x[t][2 * q + 1] = cmul(c->S[t][2 * q + 1], make_float2(K[2], K[3]));
                    }
                } else {
                    const uint32_t* b = bank16.data() + ((size_t)j * 4 * 128 + t) * 4;
                    for (int q = 0; q < 4; ++q) {
                        const uint32_t* K = b + (size_t)q * 128 * 4;
                        for (int u = 0; u < 4; ++u)
                            c->x[t][4 * q + u] = cmul(c->S[t][4 * q + u], unpack_bf16x2(K[u]));
                    }
                }
            }
            emu_ifft2048(*c);
            float* row = plane + (size_t)j * nb + sV;
            for (int t = 0; t < kThreads; ++t)
                for (int q = 0; q < 8; ++q)
                    if (2 * t + 256 * q < nvalid) {
                        float p0 = c->x[t][q].x * c->x[t][q].x + c->x[t][q].y * c->x[t][q].y;
                        float p1 = c->x[t][8 + q].x * c->x[t][8 + q].x + c->x[t][8 + q].y * c->x[t][8 + q].y;
                        if (precision == FDAS_BF16_PLANE16) {
                            p0 = bf16_bits_to_f32(f32_to_bf16_rne(p0));
                            p1 = bf16_bits_to_f32(f32_to_bf16_rne(p1));
                        }
                        row[2 * t + 256 * q] = p0;
                        row[2 * t + 256 * q + 1] = p1;
                    }
        }
    }
    delete c;
    return FDAS_OK;
}

}  // extern "C"

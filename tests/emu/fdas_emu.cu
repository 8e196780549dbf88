// fdas_emu.cu -- TEST-ONLY host emulator of the K2 CTA (tests/emu/libfdas_emu.so).  NOT part of the
// product: it lives under tests/, libfdas.so does not contain it and the Python binding never loads it.  It steps the exact
// __host__ __device__ building blocks of fdas_fft_core.cuh thread by thread, phase by phase (one
// loop over the 128 "threads" per barrier interval), with the same packed template bank, twiddle
// tables and index arithmetic as fdas_convolve.cu, so that layout or indexing mistakes show up in
// the CPU test-suite (tests/test_host_logic.py) on a box without a GPU.  It also exposes the
// plan-time host mathematics (templates, Fresnel integrals, thresholds, whitening blocks) for the
// same purpose.
#include <algorithm>
#include <cstring>
#include <vector>

#include "../../include/fdas.h"
#include "../../paper_2211_13517_b200/csrc/fdas_fft_core.cuh"
#include "../../paper_2211_13517_b200/csrc/fdas_host.h"
#include "../../paper_2211_13517_b200/csrc/fdas_maxcode.h"
#include "../../paper_2211_13517_b200/csrc/fdas_tc_common.h"

using namespace fdas;

namespace {

template <int L>
struct Cta {
    typedef SegGeom<L> G;
    float2 x[G::T][16];
    float2 S[G::T][16];
    float2 tw1[G::T][15];
    float2 tw2[G::T][G::NTw2];
    std::vector<float2> X1, X2;
    Cta() : X1(G::XbufElems), X2(G::XbufElems) {
        std::vector<float> t1, t2;
        build_twiddles(L, &t1, &t2);
        for (int t = 0; t < G::T; ++t) {
            for (int i = 0; i < 15; ++i) tw1[t][i] = make_float2(t1[(t * 15 + i) * 2], t1[(t * 15 + i) * 2 + 1]);
            const int nB = t / G::Ra;
            for (int i = 0; i < G::NTw2; ++i)
                tw2[t][i] = make_float2(t2[(nB * G::NTw2 + i) * 2], t2[(nB * G::NTw2 + i) * 2 + 1]);
        }
    }
};

// one loop over the T "threads" per barrier interval
template <int L>
void emu_ifft(Cta<L>& c) {
    constexpr int T = SegGeom<L>::T;
    for (int t = 0; t < T; ++t) { pass1(c.x[t], c.tw1[t]); x1_store<L>(c.X1.data(), t, c.x[t]); }
    for (int t = 0; t < T; ++t) { xrow_load(c.X1.data(), t, c.x[t]); pass2<L>(c.x[t]); x2_store<L>(c.X2.data(), t, c.x[t]); }
    for (int t = 0; t < T; ++t) { xrow_load(c.X2.data(), t, c.x[t]); pass3<L>(c.x[t], c.tw2[t]); }
}

template <int L>
int emu_ifft_vec(const float* in, float* out) {
    typedef SegGeom<L> G;
    Cta<L>* c = new Cta<L>();
    for (int t = 0; t < G::T; ++t)
        for (int k1 = 0; k1 < 16; ++k1) {
            const int p = G::k0_of(t) + G::T * k1;
            c->x[t][k1] = make_float2(in[2 * p], in[2 * p + 1]);
        }
    emu_ifft(*c);
    for (int t = 0; t < G::T; ++t)
        for (int i = 0; i < 16; ++i) {
            const int n = out_index<L>(t, i);
            out[2 * n] = c->x[t][i].x;
            out[2 * n + 1] = c->x[t][i].y;
        }
    delete c;
    return 0;
}

template <int L>
int emu_convolve(const float* spec, int64_t nb, double zmax, double zstep, int precision, float* plane) {
    typedef SegGeom<L> G;
    constexpr int T = G::T;
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
    Cta<L>* c = new Cta<L>();
    for (int64_t s = 0; s < nseg; ++s) {
        // stage-in, conjugated
        for (int t = 0; t < T; ++t) {
            const int64_t g0 = s * V - h + G::k0_of(t);
            for (int k1 = 0; k1 < 16; ++k1) {
                const int64_t k = g0 + T * k1;
                float2 v = make_float2(0.f, 0.f);
                if (k >= 0 && k < nb) {
                    v = make_float2(spec[2 * k], spec[2 * k + 1]);
                    if (precision != FDAS_FP32) v = unpack_bf16x2(pack_bf16x2(v.x, v.y));
                }
                c->x[t][k1] = make_float2(v.x, -v.y);
            }
        }
        emu_ifft(*c);
        // conj(S) in output order -> natural order through X1 -> (k0, k1) order
        for (int t = 0; t < T; ++t)
            for (int i = 0; i < 16; ++i) c->X1[out_index<L>(t, i)] = make_float2(c->x[t][i].x, -c->x[t][i].y);
        for (int t = 0; t < T; ++t)
            for (int k1 = 0; k1 < 16; ++k1) c->S[t][k1] = c->X1[G::k0_of(t) + T * k1];
        const int64_t sV = s * V;
        const int nvalid = (int)((nb - sV) < V ? (nb - sV) : V);
        for (int j = 0; j < nz; ++j) {
            for (int t = 0; t < T; ++t) {
                if (precision == FDAS_FP32) {
                    const float* b = bank32.data() + ((size_t)j * 8 * T + t) * 4;
                    for (int q = 0; q < 8; ++q) {
                        const float* K = b + (size_t)q * T * 4;
                        c->x[t][2 * q] = cmul(c->S[t][2 * q], make_float2(K[0], K[1]));
                        c->x[t][2 * q + 1] = cmul(c->S[t][2 * q + 1], make_float2(K[2], K[3]));
                    }
                } else {
                    const uint32_t* b = bank16.data() + ((size_t)j * 4 * T + t) * 4;
                    for (int q = 0; q < 4; ++q) {
                        const uint32_t* K = b + (size_t)q * T * 4;
                        for (int u = 0; u < 4; ++u)
                            c->x[t][4 * q + u] = cmul(c->S[t][4 * q + u], unpack_bf16x2(K[u]));
                    }
                }
            }
            emu_ifft(*c);
            float* row = plane + (size_t)j * nb + sV;
            for (int t = 0; t < T; ++t)
                for (int i = 0; i < 16; ++i) {
                    const int n = out_index<L>(t, i);
                    if (n >= nvalid) continue;
                    float p0 = c->x[t][i].x * c->x[t][i].x + c->x[t][i].y * c->x[t][i].y;
                    if (precision == FDAS_BF16_PLANE16) p0 = bf16_bits_to_f32(f32_to_bf16_rne(p0));
                    row[n] = p0;
                }
        }
    }
    delete c;
    return FDAS_OK;
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

// L-point inverse FFT of one vector through the emulated CTA (natural order in and out).
int fdas_emu_ifft(int L, const float* in, float* out) {
    switch (L) {
        case 1024: return emu_ifft_vec<1024>(in, out);
        case 2048: return emu_ifft_vec<2048>(in, out);
        case 4096: return emu_ifft_vec<4096>(in, out);
        default: return FDAS_EUNSUPPORTED;
    }
}

// Emulated fdas_convolve_plane: spec = nb complex fp32 (interleaved); plane = nz x nb floats.
// precision FDAS_BF16*: spec and bank are first rounded to bf16 exactly as the device path stores
// them; FDAS_BF16_PLANE16 additionally rounds the stored powers to bf16 (returned as float).
int fdas_emu_convolve(const float* spec, int64_t nb, double zmax, double zstep, int seg_len, int precision,
                      float* plane) {
    switch (seg_len) {
        case 1024: return emu_convolve<1024>(spec, nb, zmax, zstep, precision, plane);
        case 2048: return emu_convolve<2048>(spec, nb, zmax, zstep, precision, plane);
        case 4096: return emu_convolve<4096>(spec, nb, zmax, zstep, precision, plane);
        default: return FDAS_EUNSUPPORTED;
    }
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// K2-TC stepped on the host: the same bank image (as the kernel writes it to tensor memory), window
// image in shared memory, descriptor encodings, MMA issue order, TMEM column map and epilogue as
// fdas_convolve_tc.cu; only tcgen05.mma is replaced by `emu_umma_ts`, which reads the A operand from
// the emulated tensor memory (lane = row, two bf16 per 32-bit column) and decodes the shared-memory
// descriptor of the B operand as the hardware is documented to (K-major, no swizzle, K = 16).
namespace {

inline float bf16_to_f(uint16_t b) { return bf16_bits_to_f32(b); }

// D[lane][dcol + n] (+)= sum_k A[lane][acol*2 + k] B[n][k]; A words are TMEM columns of packed pairs.
void emu_umma_ts(const std::vector<unsigned char>& smem, std::vector<uint32_t>& tmem /*128 x 512*/, int dcol,
                 int acol, uint64_t bdesc, uint32_t idesc, bool accumulate) {
    const uint32_t b0 = (uint32_t)(bdesc & 0x3fff) << 4, blb = (uint32_t)((bdesc >> 16) & 0x3fff) << 4,
                   bsb = (uint32_t)((bdesc >> 32) & 0x3fff) << 4;
    const int N = (int)((idesc >> 17) & 0x3f) << 3, M = (int)((idesc >> 24) & 0x1f) << 4;
    for (int i = 0; i < M; ++i)
        for (int n = 0; n < N; ++n) {
            float acc = 0.0f;
            if (accumulate) std::memcpy(&acc, &tmem[(size_t)i * 512 + dcol + n], 4);
            for (int k = 0; k < 16; ++k) {
                const uint32_t aw = tmem[(size_t)i * 512 + acol + k / 2];
                const uint16_t av = (uint16_t)(aw >> (16 * (k & 1)));
                const uint32_t bo = b0 + (n % 8) * 16 + (n / 8) * bsb + (k / 8) * blb + (k % 8) * 2;
                uint16_t bv;
                std::memcpy(&bv, &smem[bo], 2);
                acc += bf16_to_f(av) * bf16_to_f(bv);
            }
            std::memcpy(&tmem[(size_t)i * 512 + dcol + n], &acc, 4);
        }
}

}  // namespace

extern "C" {
// spec: nb complex fp32 (rounded here to bf16 as K1b stores it); plane: nz x nb float (plane16: the
// bf16-rounded value as float); maxplane: nz x nb/8 block-max codes.  nb must be a multiple of 128.
int fdas_emu_convolve_tc(const float* spec, int64_t nb, double zmax, double zstep, int plane16,
                         float* plane, uint16_t* maxplane) {
    using namespace fdas::tc;
    const int nz = (int)(2.0 * zmax / zstep + 0.5) + 1;
    const int h = template_halfwidth(zmax);
    if (nb % kTileR != 0) return FDAS_EARG;
    Bank bank;
    build_bank(zmax, zstep, nz, h, 2048, &bank);   // only the tap-domain templates are used
    TcGeom g;
    if (!tc_geometry(nz, h, &g)) return FDAS_EUNSUPPORTED;
    std::vector<uint32_t> img;
    double asym = 0.0;
    pack_bank_tc(bank, g, &img, &asym);
    if (asym > 1e-12) return FDAS_EUNSUPPORTED;
    const int kw = g.kp / 2, ksteps = g.kp / 16;
    std::vector<uint32_t> specq((size_t)nb);
    for (int64_t k = 0; k < nb; ++k) specq[k] = pack_bf16x2(spec[2 * k], spec[2 * k + 1]);
    const int64_t mpitch = nb / 8, ntiles = nb / kTileR;
    auto store = [&](int j, int64_t r, float P) {
        if (j < 0 || j >= nz) return;                         // lanes beyond the launch's pairs: no row
        if (plane16) P = bf16_bits_to_f32(f32_to_bf16_rne(P));
        plane[(size_t)j * nb + r] = P;
    };
    for (int c = 0; c < g.nchunk; ++c) {                       // one kernel launch per chunk of pairs
    const int pair0 = c * g.chunk, npair = std::min(g.chunk, g.npair - pair0);
    const int jplus0 = nz - g.npair + pair0, jminus0 = g.npair - 1 - pair0;
    const Layout L = make_layout(g.kp, 2 * ((npair + 31) / 32), 1, plane16);
    std::vector<unsigned char> smem((size_t)L.total, 0xff);   // 0xff: unwritten bf16 reads as NaN
    std::vector<uint32_t> tmem((size_t)128 * 512, 0x7fc00000u);
    for (int part = 0; part < 2; ++part)                      // the kernel's tcgen05.st of the bank
        for (int lane = 0; lane < 128; ++lane)
            for (int w = 0; w < kw; ++w)
                tmem[(size_t)lane * 512 + kBankCol0 + part * kw + w] = img[(((size_t)c * 2 + part) * 128 + lane) * kw + w];
    uint32_t item = 0;
    int it = 0;
    for (int64_t tile = 0; tile < ntiles; ++tile, ++it) {
        // producer
        const int hs = it % kHStages;
        uint16_t* sre = reinterpret_cast<uint16_t*>(&smem[L.st_off]);
        uint16_t* sim = reinterpret_cast<uint16_t*>(&smem[L.st_off + L.st_part]);
        const int nrows = window_rows(g.kp), nsrc = nrows + 24;
        const int64_t base = tile * kTileR - h;
        for (int i = 0; i < nsrc; ++i) {
            const int64_t idx = base + i;
            const uint32_t v = (idx >= 0 && idx < nb) ? specq[idx] : 0u;
            sre[i] = (uint16_t)v;
            sim[i] = (uint16_t)(v >> 16);
        }
        unsigned char* hst = &smem[L.h_off + hs * L.h_stage];
        for (int rho = 0; rho < nrows; ++rho)
            for (int part = 0; part < 2; ++part) {
                const uint32_t* w32 = reinterpret_cast<const uint32_t*>(part ? sim : sre) + (rho >> 1);
                const uint4 o = window_row(w32, rho);
                std::memcpy(hst + window_row_offset(rho, part), &o, 16);
            }
        if ((nz & 1) && pair0 == 0)
            for (int b = 0; b < kTileR; ++b) {
                const float2 w = unpack_bf16x2(specq[tile * kTileR + b]);
                store(g.npair, tile * kTileR + b, fmaf(w.x, w.x, w.y * w.y));
            }
        // MMA issuer (sub-tiles in the order 0, 2, 1, 3; accumulator stage = s >> 1) + epilogue
        const uint32_t idesc = instr_desc(2 * kSubR);
        const uint32_t hbase = (uint32_t)(L.h_off + hs * L.h_stage);
        for (int pos = 0; pos < kSubTiles; ++pos, ++item) {
            const int s = 2 * (pos & 1) + (pos >> 1);
            const int st = pos & 1;
            const int d_r = st * kAccCols, d_i = d_r + 2 * kSubR;
            for (int ks = 0; ks < ksteps; ++ks) {
                const uint64_t bd = smem_desc(hbase + window_desc_offset(s, ks), kWinLbo, kWinSbo);
                emu_umma_ts(smem, tmem, d_r, kBankCol0 + 8 * ks, bd, idesc, ks > 0);
                emu_umma_ts(smem, tmem, d_i, kBankCol0 + kw + 8 * ks, bd, idesc, ks > 0);
            }
            for (int p = 0; p < npair; ++p)
                for (int bg = 0; bg < kSubR / 8; ++bg)
                    for (int e = 0; e < 8; ++e) {
                        float Ar, Ai, Br, Bi, Pp, Pm;
                        std::memcpy(&Ar, &tmem[(size_t)p * 512 + d_r + 16 * bg + e], 4);
                        std::memcpy(&Ai, &tmem[(size_t)p * 512 + d_r + 16 * bg + 8 + e], 4);
                        std::memcpy(&Br, &tmem[(size_t)p * 512 + d_i + 16 * bg + e], 4);
                        std::memcpy(&Bi, &tmem[(size_t)p * 512 + d_i + 16 * bg + 8 + e], 4);
                        pair_powers(Ar, Br, Ai, Bi, &Pp, &Pm);
                        const int64_t r = tile * kTileR + kSubR * s + 8 * bg + e;
                        store(jplus0 + p, r, Pp);
                        store(jminus0 - p, r, Pm);
                    }
        }
    }
    }
    // block maxima of the values as stored, as the codes of fdas_maxcode.h
    for (int j = 0; j < nz; ++j)
        for (int64_t b = 0; b < mpitch; ++b) {
            float m = plane[(size_t)j * nb + 8 * b];
            for (int e = 1; e < 8; ++e) m = std::max(m, plane[(size_t)j * nb + 8 * b + e]);
            maxplane[(size_t)j * mpitch + b] = (uint16_t)max_code(m);
        }
    return FDAS_OK;
}

}  // extern "C"

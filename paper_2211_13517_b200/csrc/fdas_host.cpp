// fdas_host.cpp -- plan-time host mathematics of libfdas (see fdas_host.h).  No CUDA calls.
#include "fdas_host.h"

#include <algorithm>
#include <cmath>
#include <cstring>

namespace fdas {

static const double kPi = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------------------------------------
// Fresnel integrals.  |t| <= 1.6: Maclaurin series.  Otherwise through the complementary error
// function of complex argument, C + iS = (1+i)/2 * (1 - erfc(zc)), zc = (sqrt(pi)/2)(1-i) t, with
// erfc(zc) = exp(-zc^2)/sqrt(pi) / (zc + (1/2)/(zc + 1/(zc + (3/2)/(zc + ...)))) evaluated by the
// modified Lentz recurrence (Re zc > 0 for t > 0); odd symmetry for t < 0.
// ---------------------------------------------------------------------------------------------
void fresnel_cs(double t, double* C, double* S) {
    const double x = std::fabs(t);
    double c, s;
    if (x <= 1.6) {
        const double a = 0.5 * kPi * x * x;
        double u = 1.0;  // a^m / m!
        double sc = 0.0, ss = 0.0;
        for (int m = 0; m < 200; ++m) {
            const double term = u / (2.0 * m + 1.0);
            if (m % 2 == 0) sc += ((m / 2) % 2 == 0) ? term : -term;
            else ss += (((m - 1) / 2) % 2 == 0) ? term : -term;
            u *= a / (m + 1.0);
            if (u < 1e-20 && m > 4) break;
        }
        c = x * sc;
        s = x * ss;
    } else {
        const cd zc = 0.5 * std::sqrt(kPi) * cd(1.0, -1.0) * x;
        const double tiny = 1e-300;
        cd f = zc, Cn = zc, Dn = 0.0;
        for (int k = 1; k < 20000; ++k) {
            const double ak = 0.5 * k;
            Dn = zc + ak * Dn;
            if (std::abs(Dn) == 0.0) Dn = tiny;
            Cn = zc + ak / Cn;
            if (std::abs(Cn) == 0.0) Cn = tiny;
            Dn = 1.0 / Dn;
            const cd delta = Cn * Dn;
            f *= delta;
            if (std::abs(delta - 1.0) < 1e-16) break;
        }
        const double ph = 0.5 * kPi * x * x;  // exp(-zc^2) = exp(+i pi x^2 / 2)
        const cd erfc_z = cd(std::cos(ph), std::sin(ph)) / std::sqrt(kPi) / f;
        const cd E = 0.5 * cd(1.0, 1.0) * (1.0 - erfc_z);
        c = E.real();
        s = E.imag();
    }
    *C = (t < 0) ? -c : c;
    *S = (t < 0) ? -s : s;
}

int template_halfwidth(double zmax) {
    const int base = (int)std::ceil(zmax / 2.0) + 16;
    return ((base + 31) / 32) * 32;
}

// R_z(q) = exp(-i pi q^2 / z) / sqrt(2z) * [ (C(t2)-C(t1)) + i (S(t2)-S(t1)) ],
// t1 = sqrt(2z)(-1/2 - q/z), t2 = sqrt(2z)(1/2 - q/z), z > 0;  R_{-z} = conj(R_z);  R_0 = sinc.
static cd response_R(double z, double q) {
    if (z == 0.0) {
        if (q == 0.0) return 1.0;
        const double a = kPi * q;
        return std::sin(a) / a;
    }
    const double az = std::fabs(z);
    const double rt = std::sqrt(2.0 * az);
    const double t1 = rt * (-0.5 - q / az), t2 = rt * (0.5 - q / az);
    double c1, s1, c2, s2;
    fresnel_cs(t1, &c1, &s1);
    fresnel_cs(t2, &c2, &s2);
    const double ph = -kPi * q * q / az;
    cd R = cd(std::cos(ph), std::sin(ph)) / rt * cd(c2 - c1, s2 - s1);
    return (z > 0) ? R : std::conj(R);
}

void template_response(double z, int h, cd* out) {
    const cd g = cd(std::cos(-kPi * z / 4.0), std::sin(-kPi * z / 4.0));
    double n2 = 0.0;
    for (int m = -h; m <= h; ++m) {
        cd v = g * response_R(z, (double)m);
        if (m & 1) v = -v;  // (-1)^m: r is the mid-observation frequency (reading A4)
        out[m + h] = v;
        n2 += std::norm(v);
    }
    const double sc = 1.0 / std::sqrt(n2);
    for (int i = 0; i <= 2 * h; ++i) out[i] *= sc;
}

void host_fft(cd* a, int n, int sign) {
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(a[i], a[j]);
    }
    for (int len = 2; len <= n; len <<= 1) {
        for (int k = 0; k < len / 2; ++k) {
            const double ang = sign * 2.0 * kPi * k / len;
            const cd w(std::cos(ang), std::sin(ang));
            for (int i = k; i < n; i += len) {
                const cd u = a[i], v = a[i + len / 2] * w;
                a[i] = u + v;
                a[i + len / 2] = u - v;
            }
        }
    }
}

void build_bank(double zmax, double zstep, int nz, int h, int L, Bank* bank) {
    bank->nz = nz;
    bank->h = h;
    bank->L = L;
    const int taps = 2 * h + 1;
    bank->time.assign((size_t)nz * taps, cd(0.0));
    bank->freq.assign((size_t)nz * L, cd(0.0));
    std::vector<cd> c(L);
    for (int j = 0; j < nz; ++j) {
        const double z = -zmax + j * zstep;
        cd* T = &bank->time[(size_t)j * taps];
        template_response(z, h, T);
        for (int i = 0; i < L; ++i) c[i] = (i < taps) ? T[i] : cd(0.0);
        host_fft(c.data(), L, -1);
        cd* K = &bank->freq[(size_t)j * L];
        for (int p = 0; p < L; ++p) K[p] = std::conj(c[p]) / (double)L;
    }
}

bool seg_len_supported(int L) { return L == 1024 || L == 2048 || L == 4096; }

// (Rb, Ra) of fdas_fft_core.cuh SegGeom<L>: L = 16 Ra Rb.
static void seg_radices(int L, int* Rb, int* Ra) {
    *Rb = (L == 1024) ? 8 : 16;
    *Ra = (L / 16) / *Rb;
}

int seg_k0_of(int L, int tid) {
    int Rb, Ra;
    seg_radices(L, &Rb, &Ra);
    return tid / Rb + Ra * (tid % Rb);
}

void pack_bank_fp32(const Bank& bank, std::vector<float>* out) {
    const int L = bank.L, T = L / 16;
    out->assign((size_t)bank.nz * L * 2, 0.0f);
    for (int j = 0; j < bank.nz; ++j)
        for (int c = 0; c < 8; ++c)
            for (int tid = 0; tid < T; ++tid) {
                const int k0 = seg_k0_of(L, tid);
                float* w = &(*out)[(((size_t)j * 8 + c) * T + tid) * 4];
                const cd a = bank.freq[(size_t)j * L + k0 + T * (2 * c)];
                const cd b = bank.freq[(size_t)j * L + k0 + T * (2 * c + 1)];
                w[0] = (float)a.real(); w[1] = (float)a.imag();
                w[2] = (float)b.real(); w[3] = (float)b.imag();
            }
}

static uint32_t bf16_rne(float f) {
    uint32_t u;
    std::memcpy(&u, &f, 4);
    u += 0x7fffu + ((u >> 16) & 1u);
    return u >> 16;
}

void pack_bank_bf16(const Bank& bank, std::vector<uint32_t>* out) {
    const int L = bank.L, T = L / 16;
    out->assign((size_t)bank.nz * L, 0u);
    for (int j = 0; j < bank.nz; ++j)
        for (int c = 0; c < 4; ++c)
            for (int tid = 0; tid < T; ++tid) {
                const int k0 = seg_k0_of(L, tid);
                for (int q = 0; q < 4; ++q) {
                    const cd a = bank.freq[(size_t)j * L + k0 + T * (4 * c + q)];
                    (*out)[(((size_t)j * 4 + c) * T + tid) * 4 + q] =
                        bf16_rne((float)a.real()) | (bf16_rne((float)a.imag()) << 16);
                }
            }
}

bool tc_geometry(int nz, int h, TcGeom* g) {
    if (nz < 2 || h < 1) return false;
    g->npair = nz / 2;
    g->kp = ((2 * h + 1) + 15) / 16 * 16;
    g->nchunk = (g->npair + 127) / 128;
    g->chunk = (((g->npair + g->nchunk - 1) / g->nchunk) + 31) / 32 * 32;     // balanced, whole lane quarters
    // 256 tensor-memory columns hold the two accumulator stages, the rest the two bank images
    return 256 + g->kp <= 512;
}

void pack_bank_tc(const Bank& bank, const TcGeom& g, std::vector<uint32_t>* out, double* asym) {
    const int taps = 2 * bank.h + 1, kw = g.kp / 2;
    out->assign((size_t)g.nchunk * 2 * 128 * kw, 0u);
    double worst = 0.0;
    for (int p = 0; p < g.npair; ++p) {
        const cd* tp = &bank.time[(size_t)(bank.nz - g.npair + p) * taps];
        const cd* tm = &bank.time[(size_t)(g.npair - 1 - p) * taps];
        const int c = p / g.chunk, l = p % g.chunk;
        for (int k = 0; k < taps; ++k) {
            worst = std::max(worst, std::abs(tm[k] - std::conj(tp[k])));
            for (int part = 0; part < 2; ++part) {
                const uint32_t b = bf16_rne((float)(part ? tp[k].imag() : tp[k].real()));
                (*out)[(((size_t)c * 2 + part) * 128 + l) * kw + k / 2] |= b << (16 * (k & 1));
            }
        }
    }
    if (asym) *asym = worst;
}

void build_twiddles(int L, std::vector<float>* tw1, std::vector<float>* tw2) {
    const int T = L / 16;
    int Rb, Ra;
    seg_radices(L, &Rb, &Ra);
    tw1->assign((size_t)T * 15 * 2, 0.0f);
    for (int tid = 0; tid < T; ++tid)
        for (int n1 = 1; n1 < 16; ++n1) {
            const double ang = 2.0 * kPi * (double)((n1 * seg_k0_of(L, tid)) % L) / (double)L;
            (*tw1)[(tid * 15 + n1 - 1) * 2 + 0] = (float)std::cos(ang);
            (*tw1)[(tid * 15 + n1 - 1) * 2 + 1] = (float)std::sin(ang);
        }
    tw2->assign((size_t)Rb * (Ra - 1) * 2, 0.0f);
    for (int q = 0; q < Rb; ++q)
        for (int k = 1; k < Ra; ++k) {
            const double ang = 2.0 * kPi * (double)((q * k) % T) / (double)T;
            (*tw2)[(q * (Ra - 1) + k - 1) * 2 + 0] = (float)std::cos(ang);
            (*tw2)[(q * (Ra - 1) + k - 1) * 2 + 1] = (float)std::sin(ang);
        }
}

void whitening_blocks(int64_t nb, std::vector<int32_t>* start, std::vector<int32_t>* len) {
    start->clear();
    len->clear();
    int64_t s = 1;
    while (s < nb) {
        int lg = 63 - __builtin_clzll((unsigned long long)s);
        int64_t l = (lg >= 2) ? ((int64_t)1 << (lg - 2)) : 1;
        if (l < 32) l = 32;
        if (l > 4096) l = 4096;
        if (s + l > nb) l = nb - s;
        start->push_back((int32_t)s);
        len->push_back((int32_t)l);
        s += l;
    }
}

// Newton iteration on ln Q(h,T) = -T + ln sum_{i<h} T^i/i!, d/dT = -(T^{h-1}/(h-1)!) / sum.
int thresholds_from_sigma(int H, double nsigma, float* out) {
    if (H < 1 || H > 64 || !out || !(nsigma > 0.0)) return 1;
    const double lp = std::log(0.5 * std::erfc(nsigma / std::sqrt(2.0)));
    for (int h = 1; h <= H; ++h) {
        double T = h + nsigma * std::sqrt((double)h) + 0.5 * nsigma * nsigma;  // start above the root
        for (int it = 0; it < 100; ++it) {
            double term = 1.0, sum = 1.0;
            for (int i = 1; i < h; ++i) { term *= T / i; sum += term; }
            const double lq = -T + std::log(sum);
            const double dlq = -term / sum;  // term = T^{h-1}/(h-1)!
            const double step = (lq - lp) / dlq;
            T -= step;
            if (T < 0) T = 0.5 * (T + step);
            if (std::fabs(step) < 1e-13 * (1.0 + T)) break;
        }
        out[h - 1] = (float)T;
    }
    return 0;
}

}  // namespace fdas

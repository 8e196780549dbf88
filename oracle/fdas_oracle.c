/*
 * fdas_oracle.c -- CPU ORACLE for the FDAS hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or constant with the CUDA
 * library under paper_2211_13517_b200/csrc/ and neither includes the other.
 *
 * Everything is double precision, written as the plain definition of each step so it can be
 * checked against the text by eye.  The paper contains no formula for any step; each
 * function cites the passage it serves and the DESIGN.md reading (A1..A19, taken from
 * SURVEY.md 8(c)) that fixes what the paper leaves open.
 *
 *   O1 orc_spectrum      PAPER.md:9 "Fourier Domain", "FFT"          pinned: P1
 *   O2 orc_whiten        BASELINE.json north_star "running-median power whitening" (A3) pinned: P2
 *   O3 orc_template      PAPER.md:19 "matched filtering", PAPER.md:75 (Ransom 2002) (A4,A5) pinned: P3
 *   O4 orc_plane         PAPER.md:19, "convolutions"  (A7,A8)        pinned: P4-P8
 *   O4' orc_plane_ols_dft  same result through naive-DFT overlap-save            pinned: P6(iv)
 *   O5 orc_harmonic_sums_at / O6 orc_candidates  north_star "harmonic summing and thresholding"
 *                                                 (A12,A13,A14)                  pinned: P9,P10
 *   orc_thresholds       north_star "threshold 6 sigma" (A13)                    pinned: P10
 *   O5n orc_harmonic_sums_nbr_at / orc_candidates_nbr  harmonic sums that do not lose power when the
 *                        fundamental lies between two bins (reading A24)  pinned: P13
 * No function here is "parity unpinned"; the pins live in tests/test_oracle_pins.py.
 *
 * Complex arrays are interleaved (re, im) doubles.  OpenMP is used only to spread independent
 * output elements over host cores (so the oracle can be timed on all of them); no blocking,
 * fusion or reordering of the arithmetic beyond the definitions below.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * O1 -- discrete Fourier transform.
 * ------------------------------------------------------------------------------------------- */

/* Plain O(n^2) DFT: out[k] = sum_n in[n] exp(sign * 2 pi i k n / n). */
int orc_dft(const double* in_, double* out_, int64_t n, int sign) {
    const cplx* in = (const cplx*)in_;
    cplx* out = (cplx*)out_;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) {
        cplx acc = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            int64_t kj = (k * j) % n; /* reduce the angle exactly before the trig call */
            double ang = (double)sign * 2.0 * M_PI * (double)kj / (double)n;
            acc += in[j] * (cos(ang) + I * sin(ang));
        }
        out[k] = acc;
    }
    return 0;
}

/* Textbook iterative radix-2 decimation-in-time FFT, in place, n a power of two.
 * a[k] <- sum_j a[j] exp(sign * 2 pi i j k / n); no normalisation. */
int orc_fft(double* a_, int64_t n, int sign) {
    cplx* a = (cplx*)a_;
    if (n < 1 || (n & (n - 1)) != 0) return 1;
    /* bit-reversal permutation */
    for (int64_t i = 1, j = 0; i < n; ++i) {
        int64_t bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = a[i]; a[i] = a[j]; a[j] = t; }
    }
    /* table of exp(sign 2 pi i q / n), q = 0..n/2-1, each from its own cos/sin call */
    int64_t half = n / 2;
    cplx* tw = (cplx*)malloc(sizeof(cplx) * (size_t)(half > 0 ? half : 1));
    if (!tw) return 2;
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < half; ++q) {
        double ang = (double)sign * 2.0 * M_PI * (double)q / (double)n;
        tw[q] = cos(ang) + I * sin(ang);
    }
    for (int64_t len = 2; len <= n; len <<= 1) {
        int64_t step = n / len;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; i += len) {
            for (int64_t k = 0; k < len / 2; ++k) {
                cplx u = a[i + k];
                cplx v = a[i + k + len / 2] * tw[k * step];
                a[i + k] = u + v;
                a[i + k + len / 2] = u - v;
            }
        }
    }
    free(tw);
    return 0;
}

/* O1: X[k] = sum_{n<nfft} x[n] exp(-2 pi i k n / nfft), k = 0..nfft/2-1 (Nyquist dropped, A2).
 * x: the first nfft float32 samples of the series, promoted to double. */
int orc_spectrum(const float* x, int64_t nfft, double* X_) {
    cplx* buf = (cplx*)malloc(sizeof(cplx) * (size_t)nfft);
    if (!buf) return 2;
    for (int64_t n = 0; n < nfft; ++n) buf[n] = (double)x[n];
    int rc = orc_fft((double*)buf, nfft, -1);
    if (rc == 0) memcpy(X_, buf, sizeof(cplx) * (size_t)(nfft / 2));
    free(buf);
    return rc;
}

/* ---------------------------------------------------------------------------------------------
 * O2 -- block-median power whitening (reading A3).
 *   blocks: s_0 = 1, l_b = clamp(2^(floor(log2 s_b) - 2), 32, 4096) truncated at nb,
 *           s_{b+1} = s_b + l_b
 *   m_b = median of |X|^2 over the block (even count: mean of the two middle values)
 *   c_b = s_b + (l_b - 1)/2;  m(k) = linear interpolation of (c_b, m_b), constant outside
 *   w[k] = X[k] sqrt(ln 2 / m(k)),  w[0] = 0
 * ------------------------------------------------------------------------------------------- */
static int64_t block_len(int64_t s, int64_t nb) {
    int lg = 0;
    while (((int64_t)1 << (lg + 1)) <= s) ++lg; /* floor(log2 s) */
    int64_t l = (lg >= 2) ? ((int64_t)1 << (lg - 2)) : 1;
    if (l < 32) l = 32;
    if (l > 4096) l = 4096;
    if (s + l > nb) l = nb - s;
    return l;
}

int64_t orc_whiten_nblocks(int64_t nb) {
    int64_t cnt = 0;
    for (int64_t s = 1; s < nb; s += block_len(s, nb)) ++cnt;
    return cnt;
}

static int cmp_double(const void* a, const void* b) {
    double x = *(const double*)a, y = *(const double*)b;
    return (x > y) - (x < y);
}

/* med_out / ctr_out (each orc_whiten_nblocks(nb) doubles) may be NULL. */
int orc_whiten(const double* X_, int64_t nb, double* w_, double* med_out, double* ctr_out) {
    const cplx* X = (const cplx*)X_;
    cplx* w = (cplx*)w_;
    int64_t nblk = orc_whiten_nblocks(nb);
    if (nblk < 1) return 1;
    double* med = (double*)malloc(sizeof(double) * (size_t)nblk);
    double* ctr = (double*)malloc(sizeof(double) * (size_t)nblk);
    double* tmp = (double*)malloc(sizeof(double) * 4096);
    if (!med || !ctr || !tmp) return 2;
    int64_t b = 0;
    for (int64_t s = 1; s < nb; ++b) {
        int64_t l = block_len(s, nb);
        for (int64_t i = 0; i < l; ++i) {
            cplx v = X[s + i];
            tmp[i] = creal(v) * creal(v) + cimag(v) * cimag(v);
        }
        qsort(tmp, (size_t)l, sizeof(double), cmp_double);
        med[b] = 0.5 * (tmp[(l - 1) / 2] + tmp[l / 2]);
        ctr[b] = (double)s + 0.5 * (double)(l - 1);
        s += l;
    }
    w[0] = 0.0;
    for (int64_t k = 1; k < nb; ++k) {
        double m;
        if ((double)k <= ctr[0]) m = med[0];
        else if ((double)k >= ctr[nblk - 1]) m = med[nblk - 1];
        else {
            int64_t lo = 0, hi = nblk - 1; /* ctr[lo] <= k < ctr[hi] */
            while (hi - lo > 1) {
                int64_t mid = (lo + hi) / 2;
                if (ctr[mid] <= (double)k) lo = mid; else hi = mid;
            }
            double t = ((double)k - ctr[lo]) / (ctr[hi] - ctr[lo]);
            m = med[lo] + t * (med[hi] - med[lo]);
        }
        w[k] = X[k] * sqrt(log(2.0) / m);
    }
    if (med_out) memcpy(med_out, med, sizeof(double) * (size_t)nblk);
    if (ctr_out) memcpy(ctr_out, ctr, sizeof(double) * (size_t)nblk);
    free(med); free(ctr); free(tmp);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * O3 -- constant-acceleration response templates by numerical quadrature (readings A4, A5).
 *   T_z[m] = integral_0^1 exp( 2 pi i [ -(m + z/2) u + (z/2) u^2 ] ) du,   m = -h..h
 *   then T_z <- T_z / sqrt(sum_m |T_z[m]|^2)
 * Quadrature: composite Gauss-Legendre, ORC_GL_ORDER nodes on each of
 * ORC_GL_PANELS + (|m| + |z|)/2 equal panels (the phase turns by at most ~2 pi (|m| + |z|) over
 * [0,1], so every panel sees only a few radians).
 * ------------------------------------------------------------------------------------------- */
#define ORC_GL_ORDER 32
#define ORC_GL_PANELS 64

/* Nodes/weights of the n-point Gauss-Legendre rule on [-1,1]: roots of P_n by Newton's method
 * on the three-term recurrence, w_i = 2 / ((1 - x_i^2) P_n'(x_i)^2). */
int orc_gauss_legendre(int n, double* x, double* wgt) {
    for (int i = 0; i < n; ++i) {
        double t = cos(M_PI * ((double)i + 0.75) / ((double)n + 0.5));
        double dp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p0 = 1.0, p1 = t;
            for (int k = 2; k <= n; ++k) {
                double p2 = ((2.0 * k - 1.0) * t * p1 - (k - 1.0) * p0) / (double)k;
                p0 = p1; p1 = p2;
            }
            dp = (double)n * (t * p1 - p0) / (t * t - 1.0);
            double dt = p1 / dp;
            t -= dt;
            if (fabs(dt) < 1e-16) break;
        }
        /* recompute derivative at the converged root */
        double p0 = 1.0, p1 = t;
        for (int k = 2; k <= n; ++k) {
            double p2 = ((2.0 * k - 1.0) * t * p1 - (k - 1.0) * p0) / (double)k;
            p0 = p1; p1 = p2;
        }
        dp = (double)n * (t * p1 - p0) / (t * t - 1.0);
        x[i] = t;
        wgt[i] = 2.0 / ((1.0 - t * t) * dp * dp);
    }
    return 0;
}

/* Half-width rule (A5): h = round-up-to-multiple-of-32( ceil(zmax/2) + 16 ). */
int orc_halfwidth(double zmax) {
    int base = (int)ceil(zmax / 2.0) + 16;
    return ((base + 31) / 32) * 32;
}

/* T[0..2h] holds m = -h..h.  normalise != 0 -> unit L2 norm after truncation. */
int orc_template(double z, int h, double* T_, int normalise) {
    cplx* T = (cplx*)T_;
    double gx[ORC_GL_ORDER], gw[ORC_GL_ORDER];
    orc_gauss_legendre(ORC_GL_ORDER, gx, gw);
    double norm2 = 0.0;
    for (int m = -h; m <= h; ++m) {
        cplx acc = 0.0;
        int panels = ORC_GL_PANELS + (int)((fabs((double)m) + fabs(z)) / 2.0);
        for (int p = 0; p < panels; ++p) {
            double a = (double)p / panels, b = (double)(p + 1) / panels;
            for (int i = 0; i < ORC_GL_ORDER; ++i) {
                double u = 0.5 * (a + b) + 0.5 * (b - a) * gx[i];
                double phase = 2.0 * M_PI * (-((double)m + 0.5 * z) * u + 0.5 * z * u * u);
                acc += 0.5 * (b - a) * gw[i] * (cos(phase) + I * sin(phase));
            }
        }
        T[m + h] = acc;
        norm2 += creal(acc) * creal(acc) + cimag(acc) * cimag(acc);
    }
    if (normalise) {
        double s = 1.0 / sqrt(norm2);
        for (int i = 0; i <= 2 * h; ++i) T[i] *= s;
    }
    return 0;
}

/* Bank: rows j = 0..nz-1, z_j = -zmax + j zstep (A6); bank is nz x (2h+1) complex. */
int orc_template_bank(double zmax, double zstep, int nz, int h, double* bank) {
#pragma omp parallel for schedule(dynamic)
    for (int j = 0; j < nz; ++j)
        orc_template(-zmax + (double)j * zstep, h, bank + (size_t)j * 2 * (2 * h + 1), 1);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * O4 -- the f-fdot power plane by direct correlation (readings A7, A8, A9).
 *   y_j(r) = sum_{m=-h}^{h} w[r+m] conj(T_j[m]),  w = 0 outside [0, nb);  P[j][r] = |y_j(r)|^2
 * ------------------------------------------------------------------------------------------- */
static inline double plane_point(const cplx* w, int64_t nb, const cplx* T, int h, int64_t r) {
    cplx y = 0.0;
    for (int m = -h; m <= h; ++m) {
        int64_t k = r + m;
        if (k < 0 || k >= nb) continue;
        y += w[k] * conj(T[m + h]);
    }
    return creal(y) * creal(y) + cimag(y) * cimag(y);
}

/* P is nz x (r1 - r0), row-major: P[j*(r1-r0) + (r - r0)] for r in [r0, r1). */
int orc_plane(const double* w_, int64_t nb, const double* bank_, int nz, int h,
              int64_t r0, int64_t r1, double* P) {
    const cplx* w = (const cplx*)w_;
    const cplx* bank = (const cplx*)bank_;
    int64_t width = r1 - r0;
    if (r0 < 0 || r1 > nb || width < 0) return 1;
#pragma omp parallel for collapse(2) schedule(static)
    for (int j = 0; j < nz; ++j)
        for (int64_t r = r0; r < r1; ++r)
            P[(size_t)j * (size_t)width + (size_t)(r - r0)] =
                plane_point(w, nb, bank + (size_t)j * (2 * h + 1), h, r);
    return 0;
}

/* Sampled outputs: out[i] = P[jj[i]][rr[i]]. */
int orc_plane_points(const double* w_, int64_t nb, const double* bank_, int nz, int h,
                     const int64_t* rr, const int32_t* jj, int64_t npts, double* out) {
    const cplx* w = (const cplx*)w_;
    const cplx* bank = (const cplx*)bank_;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < npts; ++i) {
        if (jj[i] < 0 || jj[i] >= nz || rr[i] < 0 || rr[i] >= nb) { out[i] = NAN; continue; }
        out[i] = plane_point(w, nb, bank + (size_t)jj[i] * (2 * h + 1), h, rr[i]);
    }
    return 0;
}

/* O4' -- the same plane through overlap-save with naive O(L^2) DFTs (second, independent mode):
 *   V = L - 2h;  g_s[i] = w[sV - h + i], i = 0..L-1 (zero outside [0,nb))
 *   c_j[i] = T_j[i - h] for i = 0..2h, else 0;  K_j = conj(DFT_L(c_j))
 *   y = IDFT_L( DFT_L(g_s) . K_j ) / L ;  P[j][sV + t] = |y[t]|^2 for t = 0..V-1, sV + t < nb */
int orc_plane_ols_dft(const double* w_, int64_t nb, const double* bank_, int nz, int h, int L,
                      double* P) {
    const cplx* w = (const cplx*)w_;
    const cplx* bank = (const cplx*)bank_;
    int V = L - 2 * h;
    if (V <= 0) return 1;
    int64_t nseg = (nb + V - 1) / V;
    cplx* K = (cplx*)malloc(sizeof(cplx) * (size_t)nz * L);
    cplx* c = (cplx*)malloc(sizeof(cplx) * (size_t)L);
    cplx* G = (cplx*)malloc(sizeof(cplx) * (size_t)L);
    cplx* g = (cplx*)malloc(sizeof(cplx) * (size_t)L);
    cplx* prod = (cplx*)malloc(sizeof(cplx) * (size_t)L);
    cplx* y = (cplx*)malloc(sizeof(cplx) * (size_t)L);
    if (!K || !c || !G || !g || !prod || !y) return 2;
    for (int j = 0; j < nz; ++j) {
        for (int i = 0; i < L; ++i) c[i] = (i <= 2 * h) ? bank[(size_t)j * (2 * h + 1) + i] : 0.0;
        orc_dft((double*)c, (double*)(K + (size_t)j * L), L, -1);
        for (int i = 0; i < L; ++i) K[(size_t)j * L + i] = conj(K[(size_t)j * L + i]);
    }
    for (int64_t s = 0; s < nseg; ++s) {
        for (int i = 0; i < L; ++i) {
            int64_t k = s * V - h + i;
            g[i] = (k >= 0 && k < nb) ? w[k] : 0.0;
        }
        orc_dft((double*)g, (double*)G, L, -1);
        for (int j = 0; j < nz; ++j) {
            for (int i = 0; i < L; ++i) prod[i] = G[i] * K[(size_t)j * L + i];
            orc_dft((double*)prod, (double*)y, L, +1);
            for (int t = 0; t < V; ++t) {
                int64_t r = s * V + t;
                if (r >= nb) break;
                cplx v = y[t] / (double)L;
                P[(size_t)j * (size_t)nb + (size_t)r] = creal(v) * creal(v) + cimag(v) * cimag(v);
            }
        }
    }
    free(K); free(c); free(G); free(g); free(prod); free(y);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * O5 / O6 -- harmonic sums, thresholds, candidates (readings A12, A13, A14).
 *   S_h(r,j) = sum_{k=1..h} P[idx(k z_j)][k r],  defined iff h r <= nb-1 and |h z_j| <= zmax
 *   idx(z') = (z' + zmax)/zstep; with c2 = nz-1 = 2 zmax/zstep the row of harmonic k of row j is
 *   (2 k j - (k-1) c2)/2, rounded half away from zero when it is a half-integer.
 * ------------------------------------------------------------------------------------------- */
static int harmonic_row(int j, int k, int nz, int* row) {
    int64_t c2 = nz - 1;
    int64_t v2 = 2 * (int64_t)k * j - (int64_t)(k - 1) * c2; /* twice the row index */
    if (v2 < 0 || v2 > 2 * c2) return 0;                     /* |k z_j| > zmax */
    *row = (int)((v2 + 1) / 2);                              /* v2 >= 0: half rounds up = away from 0 */
    if (*row > nz - 1) *row = nz - 1;
    return 1;
}

/* S[0..H-1] <- S_1..S_H at (r, j); returns hmax = number of defined sums (S_h defined for h <= hmax). */
int orc_harmonic_sums_at(const double* P, int64_t nb, int nz, int H, int64_t r, int j, double* S) {
    double acc = 0.0;
    int hmax = 0;
    for (int k = 1; k <= H; ++k) {
        int row;
        if ((int64_t)k * r > nb - 1) break;
        if (!harmonic_row(j, k, nz, &row)) break;
        acc += P[(size_t)row * (size_t)nb + (size_t)((int64_t)k * r)];
        S[k - 1] = acc;
        hmax = k;
    }
    return hmax;
}

/* O5 at sampled fundamentals straight from the whitened spectrum (for sizes where the full plane
 * is too large): S[i*H + (k-1)] = S_k(rr[i], jj[i]) for k <= hmax[i], every needed plane point
 * computed one by one by the O4 definition. */
int orc_harmonic_sums_sampled(const double* w_, int64_t nb, const double* bank_, int nz, int h, int H,
                              const int64_t* rr, const int32_t* jj, int64_t npts, double* S,
                              int32_t* hmax) {
    const cplx* w = (const cplx*)w_;
    const cplx* bank = (const cplx*)bank_;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < npts; ++i) {
        double acc = 0.0;
        int hm = 0;
        for (int k = 1; k <= H; ++k) {
            int row;
            if ((int64_t)k * rr[i] > nb - 1) break;
            if (!harmonic_row(jj[i], k, nz, &row)) break;
            acc += plane_point(w, nb, bank + (size_t)row * (2 * h + 1), h, (int64_t)k * rr[i]);
            S[i * H + (k - 1)] = acc;
            hm = k;
        }
        hmax[i] = hm;
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * O5n -- neighbour-maximised harmonic sums (reading A24; serves PAPER.md:9
 * "sacrificing less than 3 % in numerical sensitivity").  A signal whose fundamental lies at
 * r_c = r + delta, |delta| <= 1/2, has its k-th harmonic at k r_c = k r + k delta, up to k/2 bins from
 * k r, so harmonic k is taken where it is largest within that reach:
 *   S'_h(r,j) = sum_{k=1..h} max_{|d| <= floor(k/2), 0 <= k r + d <= nb-1} P[row_k(j)][k r + d]
 * defined exactly when S_h is (h r <= nb-1 and |h z_j| <= zmax).  S'_1 = S_1; S'_h >= S_h.
 * ------------------------------------------------------------------------------------------- */
int orc_harmonic_sums_nbr_at(const double* P, int64_t nb, int nz, int H, int64_t r, int j, double* S) {
    double acc = 0.0;
    int hmax = 0;
    for (int k = 1; k <= H; ++k) {
        int row;
        if ((int64_t)k * r > nb - 1) break;
        if (!harmonic_row(j, k, nz, &row)) break;
        double best = -1.0;
        for (int64_t d = -(k / 2); d <= k / 2; ++d) {
            int64_t c = (int64_t)k * r + d;
            if (c < 0 || c > nb - 1) continue;
            double v = P[(size_t)row * (size_t)nb + (size_t)c];
            if (v > best) best = v;
        }
        acc += best;
        S[k - 1] = acc;
        hmax = k;
    }
    return hmax;
}

static int sum_defined_nbr(const double* P, int64_t nb, int nz, int64_t r_lo, int64_t r, int j, int h,
                           double* val) {
    if (j < 0 || j >= nz || r < r_lo || r >= nb) return 0;
    double S[64];
    int hmax = orc_harmonic_sums_nbr_at(P, nb, nz, h, r, j, S);
    if (hmax < h) return 0;
    *val = S[h - 1];
    return 1;
}

/* Candidates of the neighbour-maximised sums: the rule of orc_candidates (O6) applied to S'. */
int64_t orc_candidates_nbr(const double* P, int64_t nb, int nz, int H, const double* thr, int64_t r_lo,
                           int64_t* c_r, int32_t* c_j, int32_t* c_h, double* c_pow, int32_t* c_flag,
                           int64_t capacity) {
    int64_t count = 0;
    if (H < 1 || H > 64) return -1;
    for (int j = 0; j < nz; ++j) {
        for (int64_t r = r_lo; r < nb; ++r) {
            double S[64];
            int hmax = orc_harmonic_sums_nbr_at(P, nb, nz, H, r, j, S);
            for (int h = 1; h <= hmax; ++h) {
                if (!(S[h - 1] > thr[h - 1])) continue;
                int flag = 1;
                for (int dj = -1; dj <= 1 && flag; ++dj)
                    for (int dr = -1; dr <= 1 && flag; ++dr) {
                        if (dj == 0 && dr == 0) continue;
                        double nv;
                        if (!sum_defined_nbr(P, nb, nz, r_lo, r + dr, j + dj, h, &nv)) continue;
                        int precedes = (dj < 0) || (dj == 0 && dr < 0);
                        if (precedes ? !(S[h - 1] > nv) : !(S[h - 1] >= nv)) flag = 0;
                    }
                if (count < capacity) {
                    c_r[count] = r; c_j[count] = j; c_h[count] = h;
                    c_pow[count] = S[h - 1]; c_flag[count] = flag;
                }
                ++count;
            }
        }
    }
    return count;
}

static int sum_defined(const double* P, int64_t nb, int nz, int64_t r_lo, int64_t r, int j, int h,
                       double* val) {
    if (j < 0 || j >= nz || r < r_lo || r >= nb) return 0;
    double S[64];
    int hmax = orc_harmonic_sums_at(P, nb, nz, h, r, j, S);
    if (hmax < h) return 0;
    *val = S[h - 1];
    return 1;
}

/* Candidates: all (r, j, h), r in [r_lo, nb), with S_h(r,j) > thr[h-1] (strict).
 * flag bit 0 = 1 iff S_h(r,j) >= S_h at all existing 8 neighbours (r+-1, j+-1) for which S_h is
 * defined, and strictly > those neighbours that precede it in (j, r) lexicographic order.
 * Returns the true count; stores the first `capacity` in (j, r, h) loop order. */
int64_t orc_candidates(const double* P, int64_t nb, int nz, int H, const double* thr, int64_t r_lo,
                       int64_t* c_r, int32_t* c_j, int32_t* c_h, double* c_pow, int32_t* c_flag,
                       int64_t capacity) {
    int64_t count = 0;
    if (H < 1 || H > 64) return -1;
    for (int j = 0; j < nz; ++j) {
        for (int64_t r = r_lo; r < nb; ++r) {
            double S[64];
            int hmax = orc_harmonic_sums_at(P, nb, nz, H, r, j, S);
            for (int h = 1; h <= hmax; ++h) {
                if (!(S[h - 1] > thr[h - 1])) continue;
                int flag = 1;
                for (int dj = -1; dj <= 1 && flag; ++dj)
                    for (int dr = -1; dr <= 1 && flag; ++dr) {
                        if (dj == 0 && dr == 0) continue;
                        double nv;
                        if (!sum_defined(P, nb, nz, r_lo, r + dr, j + dj, h, &nv)) continue;
                        int precedes = (dj < 0) || (dj == 0 && dr < 0);
                        if (precedes ? !(S[h - 1] > nv) : !(S[h - 1] >= nv)) flag = 0;
                    }
                if (count < capacity) {
                    c_r[count] = r; c_j[count] = j; c_h[count] = h;
                    c_pow[count] = S[h - 1]; c_flag[count] = flag;
                }
                ++count;
            }
        }
    }
    return count;
}

/* Thresholds (A13): T_h solves Q(h, T_h) = p, p = erfc(nsigma/sqrt 2)/2 (one-sided Gaussian tail),
 * Q(h, T) = exp(-T) sum_{i<h} T^i / i!  (survival function of a sum of h unit exponentials).
 * Solved by bisection. */
static double erlang_sf(int h, double T) {
    double term = 1.0, sum = 1.0;
    for (int i = 1; i < h; ++i) { term *= T / (double)i; sum += term; }
    return exp(-T) * sum;
}

int orc_thresholds(int H, double nsigma, double* T) {
    double p = 0.5 * erfc(nsigma / sqrt(2.0));
    for (int h = 1; h <= H; ++h) {
        double lo = 0.0, hi = 1.0;
        while (erlang_sf(h, hi) > p) hi *= 2.0;
        for (int it = 0; it < 200; ++it) {
            double mid = 0.5 * (lo + hi);
            if (erlang_sf(h, mid) > p) lo = mid; else hi = mid;
        }
        T[h - 1] = 0.5 * (lo + hi);
    }
    return 0;
}

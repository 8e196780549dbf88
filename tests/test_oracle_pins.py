"""Pins for the CPU oracle (oracle/fdas_oracle.c): every oracle step is checked against something
other than itself -- closed forms, library routines, brute force, invariants (SURVEY.md 8(c)
P1..P12).  CPU only.
"""
import os

import numpy as np
import pytest
from scipy import integrate, special, stats

from paper_2211_13517_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden", "survey_spot_values.txt")


def golden():
    out = {"R": [], "E": [], "M": [], "T": None, "TINY": None}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, *v = line.split()
        v = [float(t) for t in v]
        if k in ("R", "E", "M"):
            out[k].append(v)
        elif k == "T":
            out["T"] = np.array(v)
        else:
            out[k] = v[0]
    return out


def fresnel_R(z, q):
    """Closed-form response (Ransom et al. 2002 form) via scipy's Fresnel integrals."""
    q = np.asarray(q, dtype=np.float64)
    if z == 0:
        return np.sinc(q).astype(np.complex128)
    az = abs(z)
    t1 = np.sqrt(2 * az) * (-0.5 - q / az)
    t2 = np.sqrt(2 * az) * (0.5 - q / az)
    S2, C2 = special.fresnel(t2)
    S1, C1 = special.fresnel(t1)
    R = np.exp(-1j * np.pi * q * q / az) / np.sqrt(2 * az) * ((C2 - C1) + 1j * (S2 - S1))
    return R if z > 0 else np.conj(R)


def closed_form_T(z, h):
    m = np.arange(-h, h + 1)
    return (-1.0) ** m * np.exp(-1j * np.pi * z / 4) * fresnel_R(z, m.astype(float))


# ------------------------------------------------------------------------------------------ P1
def test_p1_fft_vs_dft_vs_numpy_and_parseval(oracle):
    rng = np.random.default_rng(11)
    for n in (1, 2, 8, 64, 1024, 4096):
        x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
        F = oracle.fft(x, -1)
        assert np.abs(F - oracle.dft(x, -1)).max() <= 1e-9 * max(1.0, np.abs(F).max())
        assert np.abs(F - np.fft.fft(x)).max() <= 1e-10 * max(1.0, np.abs(F).max())
        assert np.abs(oracle.fft(F, +1) / n - x).max() <= 1e-12 * max(1.0, np.abs(x).max())
        assert np.isclose(np.sum(np.abs(x) ** 2), np.sum(np.abs(F) ** 2) / n, rtol=1e-12)
    # a single complex exponential lands in exactly one bin with the forward sign convention
    n = 256
    x = np.exp(2j * np.pi * 37 * np.arange(n) / n)
    F = oracle.fft(x, -1)
    assert abs(F[37] - n) < 1e-9 and np.abs(np.delete(F, 37)).max() < 1e-9


def test_p1_spectrum_is_the_positive_half_of_the_real_dft(oracle):
    x = np.random.default_rng(5).standard_normal(1 << 14).astype(np.float32)
    X = oracle.spectrum(x, 1 << 14)
    ref = np.fft.rfft(x.astype(np.float64))[: 1 << 13]
    assert X.shape == (1 << 13,)
    assert np.abs(X - ref).max() <= 1e-10 * np.abs(ref).max()


# ------------------------------------------------------------------------------------------ P2
def test_p2_whitening_closed_form_linear_power(oracle):
    """|X[k]|^2 = k: every block median equals its centre, so m(k) = k between the first and last
    centres and |w|^2 = ln 2 there; outside it is clamped to the end medians."""
    nb = 50000
    k = np.arange(nb, dtype=np.float64)
    X = np.sqrt(k) * np.exp(1j * 0.37 * k)
    w, med, ctr = oracle.whiten(X, want_blocks=True)
    assert w[0] == 0
    assert np.allclose(med, ctr, rtol=1e-12)
    inside = (k >= ctr[0]) & (k <= ctr[-1])
    assert np.allclose(np.abs(w[inside]) ** 2, np.log(2.0), rtol=1e-12)
    lo = (k >= 1) & (k < ctr[0])
    assert np.allclose(np.abs(w[lo]) ** 2, np.log(2.0) * k[lo] / ctr[0], rtol=1e-12)
    hi = k > ctr[-1]
    assert np.allclose(np.abs(w[hi]) ** 2, np.log(2.0) * k[hi] / ctr[-1], rtol=1e-12)
    assert np.allclose(np.angle(w[1:] / X[1:]), 0.0, atol=1e-12)  # phases untouched


def test_p2_block_schedule(oracle):
    """First block starts at 1; lengths 32 until s >= 256, double with every octave, cap 4096; the
    blocks tile [1, nb) exactly."""
    nb = 1 << 20
    X = np.ones(nb, dtype=np.complex128)
    _, med, ctr = oracle.whiten(X, want_blocks=True)
    # recover starts/lengths from consecutive centres: c_b = s_b + (l_b-1)/2, s_{b+1} = s_b + l_b
    s, lens = 1, []
    for c in ctr:
        l = int(round(2 * (c - s) + 1))
        lens.append(l)
        s += l
    assert s == nb
    lens = np.array(lens)
    assert lens[0] == 32 and lens.max() == 4096 and np.all(lens[:8] == 32)
    starts = 1 + np.concatenate([[0], np.cumsum(lens)[:-1]])
    big = starts >= 16384
    assert np.all(lens[big][:-1] == 4096)
    mid = (starts >= 1024) & (starts < 2048)
    assert np.all(lens[mid] == 256)


def test_p2_white_noise_statistics_and_scale_invariance(oracle):
    nfft = 1 << 20
    x = np.random.default_rng(3).standard_normal(nfft).astype(np.float32)
    X = oracle.spectrum(x, nfft)
    w = oracle.whiten(X)
    nb = nfft // 2
    p = np.abs(w[128:]) ** 2
    assert abs(p.mean() - 1.0) < 3.0 / np.sqrt(nb) + 0.01   # Exp(mu): median = mu ln 2
    w2 = oracle.whiten(7.5 * X)
    assert np.abs(w2 - w).max() < 1e-12 * np.abs(w).max()


# ------------------------------------------------------------------------------------------ P3
def test_p3_gauss_legendre_rule(oracle):
    x, wgt = oracle.gauss_legendre(32)
    assert np.isclose(wgt.sum(), 2.0, rtol=1e-14)
    for deg in (2, 10, 40, 62):   # exact for polynomials up to degree 63
        assert np.isclose(np.sum(wgt * x ** deg), 2.0 / (deg + 1), rtol=1e-12)
    assert abs(np.sum(wgt * x ** 63)) < 1e-13


def test_p3_template_quadrature_vs_closed_form_vs_spot_values(oracle):
    g = golden()
    for z in (0.0, 0.5, 1.0, 7.0, -20.0, 37.5, 96.0, -96.0):
        T = oracle.template(z, 64, normalise=False)
        assert np.abs(T - closed_form_T(z, 64)).max() < 5e-13, z
    for z, q, re, im in g["R"]:
        T = oracle.template(z, 64, normalise=False)[64 + int(q)]
        Rq = T / ((-1.0) ** int(q) * np.exp(-1j * np.pi * z / 4))
        assert abs(Rq - (re + 1j * im)) < 2e-6


def test_p3_template_vs_dft_of_a_synthesised_chirp(oracle):
    """Third route: X[k] of a real unit chirp ~ (n/2) e^{i phi} T_z[k - r_c] (reading A4)."""
    n = 1 << 14
    for z, r_c in ((12.0, 3000), (-31.0, 5000)):
        x = inputs.chirp(n, n, inputs.Signal(r_c=float(r_c), z=z, amp=1.0, phase=0.0))
        X = np.fft.fft(x)
        h = 40
        T = oracle.template(z, h, normalise=False)
        seg = X[r_c - h: r_c + h + 1] / (n / 2)
        # remove the global phase e^{i phi}: phi = 2 pi (-(r_c - z/2)/2 + z/8) from v = u - 1/2
        phi = 2 * np.pi * (-(r_c) * 0.5 + z / 8.0)
        assert np.abs(seg * np.exp(-1j * phi) - T).max() < 2e-4


def test_p3_template_symmetries_and_energy(oracle):
    g = golden()
    T0 = oracle.template(0.0, 32)
    assert abs(T0[32] - 1) < 1e-14 and np.abs(np.delete(T0, 32)).max() < 1e-14   # z=0 -> delta
    for z in (3.0, 40.0, 96.0):
        Tp = oracle.template(z, 64, normalise=False)
        Tm = oracle.template(-z, 64, normalise=False)
        assert np.abs(Tm - np.conj(Tp)).max() < 1e-13            # T_{-z} = conj(T_z)
        assert np.abs(np.abs(Tp) - np.abs(Tp[::-1])).max() < 1e-13  # |T_z[-m]| = |T_z[m]|
    for z, E in g["E"]:
        T = oracle.template(z, 64, normalise=False)
        assert abs(np.sum(np.abs(T) ** 2) - E) < 2e-5
    # Parseval: the full response has unit energy (|exp(i phase)|^2 integrates to 1 over u in [0,1])
    T = oracle.template(8.0, 2000, normalise=False)
    assert abs(np.sum(np.abs(T) ** 2) - 1.0) < 2e-4
    Tn = oracle.template(57.0, 64)
    assert np.isclose(np.sum(np.abs(Tn) ** 2), 1.0, rtol=1e-13)
    assert oracle.halfwidth(96) == 64 and oracle.halfwidth(16) == 32 and oracle.halfwidth(97) == 96


# ------------------------------------------------------------------------------------- P4 .. P8
def _noise_w(nb, seed):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal(nb) + 1j * rng.standard_normal(nb)) / np.sqrt(2.0)


def test_p4_z0_row_is_the_power_spectrum(oracle):
    w = _noise_w(5000, 1)
    bank = oracle.template_bank(16.0, 1.0)
    P = oracle.plane(w, bank)
    assert np.abs(P[16] - np.abs(w) ** 2).max() < 1e-13


def test_p5_brute_force_time_domain_correlation(oracle):
    """y_brute(r,z) = N^-1/2 sum_n x[n] exp(-2 pi i [(r - z/2) u + (z/2) u^2]), u = n/N: fixes every
    sign convention (z sign, conj, mid-observation reference).  The truncated template converges
    to it as the guard h grows."""
    N = 4096
    rng = np.random.default_rng(7)
    x = rng.standard_normal(N) + inputs.chirp(N, N, inputs.Signal(r_c=700.0, z=12.0, amp=0.3, phase=0.4))
    X = np.fft.fft(x)[: N // 2]
    w = X / np.sqrt(N)
    u = np.arange(N) / N
    pts = [(700, 12.0), (700, -12.0), (701, 12.0), (650, 5.0), (900, -20.0), (700, 0.0)]
    errs = []
    for h in (16, 64, 256):
        err = 0.0
        for r, z in pts:
            T = oracle.template(z, h, normalise=False)[None, :]
            P = oracle.plane_points(w, T, [r], [0])[0]
            yb = np.sum(x * np.exp(-2j * np.pi * ((r - z / 2) * u + (z / 2) * u * u))) / np.sqrt(N)
            err = max(err, abs(np.sqrt(P) - abs(yb)))
        errs.append(err)
    assert errs[2] < 3e-3 and errs[2] < errs[0]
    # the matched point carries the signal; the sign-flipped template does not
    T = oracle.template(12.0, 256, normalise=False)[None, :]
    Tm = oracle.template(-12.0, 256, normalise=False)[None, :]
    Pm = oracle.plane_points(w, T, [700], [0])[0]
    Pw = oracle.plane_points(w, Tm, [700], [0])[0]
    assert Pm > 0.8 * (0.3 ** 2 * N / 4) and Pw < 0.2 * Pm


def test_p6_invariants(oracle):
    nb = 6000
    w1, w2 = _noise_w(nb, 2), _noise_w(nb, 3)
    bank = oracle.template_bank(16.0, 1.0)
    h = (bank.shape[1] - 1) // 2
    P1, P2 = oracle.plane(w1, bank), oracle.plane(w2, bank)
    # (i) linearity of y before |.|^2: parallelogram law
    lhs = oracle.plane(w1 + w2, bank) + oracle.plane(w1 - w2, bank)
    assert np.abs(lhs - 2 * (P1 + P2)).max() < 1e-11
    assert np.abs(oracle.plane(3.0 * w1, bank) - 9.0 * P1).max() < 1e-10
    # (ii) shift by d bins (not a multiple of V = 1984) shifts every row by d
    d = 777
    ws = np.concatenate([np.zeros(d), w1[:-d]])
    Ps = oracle.plane(ws, bank)
    assert np.abs(Ps[:, d + h: nb - h] - P1[:, h: nb - d - h]).max() < 1e-12
    # (iii) w -> conj(w) maps row z to row -z (T_{-z} = conj(T_z))
    Pc = oracle.plane(np.conj(w1), bank)
    assert np.abs(Pc - P1[::-1]).max() < 1e-12
    # partial range and sampled points agree with the full plane
    Pr = oracle.plane(w1, bank, 1000, 1300)
    assert np.array_equal(Pr, P1[:, 1000:1300])
    rr = np.array([0, 5, 1984, 5999]); jj = np.array([0, 32, 16, 7], dtype=np.int32)
    assert np.array_equal(oracle.plane_points(w1, bank, rr, jj), P1[jj, rr])


def test_p6_direct_equals_naive_dft_overlap_save(oracle):
    nb = 1000
    w = _noise_w(nb, 4)
    bank = oracle.template_bank(8.0, 2.0, h=32)
    P = oracle.plane(w, bank)
    for L in (128, 256):   # V = 64, 192: several segments and a ragged tail
        Po = oracle.plane_ols_dft(w, bank, L)
        assert np.abs(Po - P).max() < 1e-11 * P.max()


def test_p7_noise_free_chirp_closed_forms(oracle):
    g = golden()
    nfft = 1 << 16
    a, r_c, z0 = 0.05, 9000, 20.0
    x = inputs.chirp(nfft, nfft, inputs.Signal(r_c=float(r_c), z=z0, amp=a, phase=1.0))
    w = np.fft.fft(x)[: nfft // 2] / np.sqrt(nfft)
    bank = oracle.template_bank(32.0, 1.0)       # h = 32
    h = (bank.shape[1] - 1) // 2
    P = oracle.plane(w, bank, r_c - 8, r_c + 9)
    jz = 32 + int(z0)
    E = np.sum(np.abs(closed_form_T(z0, h)) ** 2)
    peak = a * a * nfft / 4 * E
    assert np.isclose(P[jz, 8], peak, rtol=2e-3)
    assert np.unravel_index(np.argmax(P), P.shape) == (jz, 8)
    # matched row at integer offsets: sinc^2 -> 0
    assert P[jz, 7] < 1e-3 * peak and P[jz, 9] < 1e-3 * peak
    # z mismatch at r = r_c: |int_0^1 exp(i pi dz (u^2 - u)) du|^2 (time-domain closed form)
    for dz, fac in g["M"]:
        if dz != int(dz):
            continue
        re = integrate.quad(lambda u: np.cos(np.pi * dz * (u * u - u)), 0, 1)[0]
        im = integrate.quad(lambda u: np.sin(np.pi * dz * (u * u - u)), 0, 1)[0]
        f = re * re + im * im
        assert abs(f - fac) < 2e-3
        for sgn in (-1, 1):
            assert np.isclose(P[jz + sgn * int(dz), 8] / peak, f, atol=0.01)


def test_p7_tiny_config_noise_free_tie(oracle):
    """configs[0]: z0 = 7.5 sits between templates 7 and 8: equal noise-free powers."""
    g = golden()
    wl = inputs.tiny()
    x = inputs.chirp(wl.nfft, wl.nfft, wl.signals[0])
    w = np.fft.fft(x)[: wl.nfft // 2] / np.sqrt(wl.nfft)
    bank = oracle.template_bank(wl.zmax, wl.zstep)
    P = oracle.plane(w, bank, 19990, 20011)
    p7, p8 = P[16 + 7, 10], P[16 + 8, 10]
    assert np.isclose(p7, p8, rtol=1e-3)
    assert np.isclose(p7, g["TINY"], rtol=5e-3)


def test_p8_noise_rows_are_unit_exponential(oracle):
    w = _noise_w(40000, 9)
    bank = oracle.template_bank(16.0, 1.0)
    P = oracle.plane(w, bank)[:, 100:-100]
    assert abs(P.mean() - 1.0) < 0.02
    assert abs(P.var() - 1.0) < 0.06
    assert stats.kstest(P[5, ::70], "expon").pvalue > 1e-3


# ------------------------------------------------------------------------------------ P9, P10
def test_p9_harmonic_sums_on_hand_made_planes(oracle):
    nz, nb, H, r_lo = 33, 600, 16, 5       # zmax = 16, zstep = 1
    P = np.ones((nz, nb))
    for r, j in ((5, 16), (37, 16), (37, 20), (599, 0), (20, 8)):
        S = oracle.harmonic_sums_at(P, H, r, j)
        z = j - 16
        hmax = min(H, (nb - 1) // r, 16 // abs(z) if z else H)
        assert len(S) == hmax and np.allclose(S, np.arange(1, hmax + 1))
    # everything passes a negative threshold: count = number of defined (r, j, h) triples
    c = oracle.candidates(P, H, -np.ones(H), r_lo)
    expect = sum(((nb - 1) // h - r_lo + 1) * (2 * (16 // h) + 1) for h in range(1, H + 1))
    assert c.count == expect
    # a single spike at (r', z') contributes to S_h(r'/k, z'/k) for every k dividing both, h >= k
    P = np.zeros((nz, nb))
    rp, zp = 360, 12
    P[16 + zp, rp] = 5.0
    c = oracle.candidates(P, H, np.full(H, 1.0), r_lo)
    got = c.triples()
    want = set()
    for k in range(1, H + 1):
        if rp % k == 0 and zp % k == 0 and rp // k >= r_lo:
            r, z = rp // k, zp // k
            for h in range(k, H + 1):
                if h * r <= nb - 1 and abs(h * z) <= 16:
                    want.add((r, 16 + z, h))
    assert got == want and len(want) > 5
    assert all(p == 5.0 and f == 1 for p, f in c.as_dict().values())


def test_p9_local_max_flag_tie_rule(oracle):
    nz, nb = 9, 100
    P = np.zeros((nz, nb))
    P[4, 50] = 3.0; P[4, 51] = 3.0; P[5, 49] = 3.0   # three equal neighbours
    c = oracle.candidates(P, 1, np.array([1.0]), 1).as_dict()
    # the first in (j, r) order keeps the flag; later equal neighbours lose it
    assert c[(50, 4, 1)][1] == 1 and c[(51, 4, 1)][1] == 0 and c[(49, 5, 1)][1] == 0


def test_p9_half_integer_rows_round_away_from_zero(oracle):
    """nz even (zmax/zstep half-integer): row of harmonic k is round-half-away((2kj-(k-1)(nz-1))/2)."""
    nz, nb = 6, 50           # zmax = 1, zstep = 0.4: z = -1, -.6, -.2, .2, .6, 1
    P = np.arange(nz * nb, dtype=np.float64).reshape(nz, nb)
    S = oracle.harmonic_sums_at(P, 4, 3, 3)      # z = 0.2: 2z = .4 -> idx 3.5 -> row 4; 3z = .6 -> row 4
    assert np.allclose(S, np.cumsum([P[3, 3], P[4, 6], P[4, 9], P[5, 12]]))
    S = oracle.harmonic_sums_at(P, 4, 3, 4)      # z = 0.6: 2z = 1.2 > zmax -> only h = 1
    assert len(S) == 1


def test_p10_thresholds(oracle):
    g = golden()
    T = oracle.thresholds(16, 6.0)
    p = stats.norm.sf(6.0)
    assert np.isclose(T[0], -np.log(p), rtol=1e-12)                       # closed form for h = 1
    assert np.allclose(T, special.gammainccinv(np.arange(1, 17), p), rtol=1e-9)
    assert np.abs(T - g["T"]).max() < 6e-4
    T3 = oracle.thresholds(4, 3.0)
    assert np.allclose(special.gammaincc(np.arange(1, 5), T3), stats.norm.sf(3.0), rtol=1e-9)


def test_p10_noise_only_false_alarm_count(oracle):
    w = _noise_w(60000, 21)
    bank = oracle.template_bank(16.0, 1.0)
    P = oracle.plane(w, bank)
    thr = oracle.thresholds(1, 3.5)
    c = oracle.candidates(P, 1, thr, 64)
    expect = stats.norm.sf(3.5) * P.shape[0] * (60000 - 64)
    assert 0.6 * expect < c.count < 1.5 * expect     # neighbouring points are correlated


# ----------------------------------------------------------------------------------------- P12
def test_p12_tiny_config_recovers_the_injected_signal(oracle):
    wl = inputs.tiny()
    x = inputs.series_for(wl)
    res = oracle.run(x, wl.nfft, wl.zmax, wl.zstep, wl.nharm, wl.nsigma, wl.r_lo)
    assert res.P.shape == (33, 65536)
    jmax, rmax = np.unravel_index(np.argmax(res.P), res.P.shape)
    assert rmax == 20000 and jmax in (16 + 7, 16 + 8)       # half-integer z0: either neighbour
    trip = res.cands.triples()
    assert (20000, 23, 1) in trip or (20000, 24, 1) in trip
    assert 1 <= res.cands.count < 200
    # noise part of the plane has unit mean
    assert abs(res.P[:, 30000:60000].mean() - 1.0) < 0.02


def test_p9_sampled_harmonic_sums_equal_the_full_plane_route(oracle):
    nb = 3000
    w = _noise_w(nb, 31)
    bank = oracle.template_bank(16.0, 1.0)
    P = oracle.plane(w, bank)
    rng = np.random.default_rng(2)
    rr = rng.integers(1, nb, 200); jj = rng.integers(0, 33, 200).astype(np.int32)
    S, hmax = oracle.harmonic_sums_sampled(w, bank, 16, rr, jj)
    for i in range(200):
        ref = oracle.harmonic_sums_at(P, 16, rr[i], jj[i])
        assert hmax[i] == len(ref)
        assert np.allclose(S[i, :hmax[i]], ref, rtol=1e-13)
        assert np.all(np.isnan(S[i, hmax[i]:]))


# ----------------------------------------------------------------------------------------- P13
def test_p13_neighbour_maximised_sums_on_hand_made_planes(oracle):
    """O5n (reading A24): harmonic k is taken at its largest value within floor(k/2) bins of k r.
    Pinned by closed forms on constructed planes: a constant plane, the first sum, monotonicity,
    the harmonics of a fundamental at r0 + 0.37 (all recovered, the plain sum loses 7 of 8), the exact
    reach of the window and its clipping at the ends of the plane."""
    nz, nb, H = 33, 4000, 8
    mid = 16
    # constant plane: S'_h = h, defined exactly where S_h is
    P = np.ones((nz, nb))
    for r, j in ((5, 16), (37, 18), (499, 0), (3999, 16), (2000, 16)):
        S, Sn = oracle.harmonic_sums_at(P, H, r, j), oracle.harmonic_sums_nbr_at(P, H, r, j)
        assert len(S) == len(Sn) and np.allclose(Sn, np.arange(1, len(Sn) + 1))
    # S'_1 = S_1 and S'_h >= S_h on a random plane
    rng = np.random.default_rng(131)
    P = rng.exponential(1.0, size=(nz, nb))
    for r, j in ((7, 16), (123, 14), (400, 17), (1999, 16), (64, 20)):
        S, Sn = oracle.harmonic_sums_at(P, H, r, j), oracle.harmonic_sums_nbr_at(P, H, r, j)
        assert len(S) == len(Sn) and Sn[0] == S[0] and np.all(Sn >= S - 1e-15)
        assert np.all(np.diff(Sn) <= P.max() + 1e-12) and np.all(np.diff(Sn) > 0)
    # a pulsar whose fundamental sits at r_c = r0 + 0.37 (z = 2): harmonic k peaks at round(k r_c)
    r0, z, A = 300, 2, 10.0
    P = np.zeros((nz, nb))
    shifts = [int(np.floor(0.37 * k + 0.5)) for k in range(1, H + 1)]         # 0 1 1 1 2 2 3 3
    assert shifts == [0, 1, 1, 1, 2, 2, 3, 3] and all(s <= (k + 1) // 2 for k, s in enumerate(shifts))
    for k, s in zip(range(1, H + 1), shifts):
        P[mid + k * z, k * r0 + s] = A
    assert np.allclose(oracle.harmonic_sums_nbr_at(P, H, r0, mid + z), A * np.arange(1, H + 1))
    assert np.allclose(oracle.harmonic_sums_at(P, H, r0, mid + z), A)          # only k = 1 lies on k r0
    # the reach is exactly floor(k/2): a spike one bin further is not picked up
    for k in (2, 3, 4, 7, 8):
        w = k // 2
        for d, seen in ((w, True), (-w, True), (w + 1, False), (-w - 1, False)):
            P = np.zeros((nz, nb))
            P[mid, k * 100 + d] = 3.0
            Sn = oracle.harmonic_sums_nbr_at(P, H, 100, mid)
            assert (Sn[k - 1] == 3.0) == seen and (k == 1 or Sn[k - 2] == 0.0)
    # clipping: the window of the last defined harmonic stops at bin nb - 1, that of r = 0 at bin 0
    P = np.zeros((nz, nb))
    P[mid, nb - 1] = 2.0
    Sn = oracle.harmonic_sums_nbr_at(P, H, (nb - 1) // 4, mid)       # 4 r = 3996: window 3994..3998 -> no
    assert len(Sn) == 4 and Sn[3] == 0.0
    Sn = oracle.harmonic_sums_nbr_at(P, H, 1333, mid)                # 3 r = 3999 = nb - 1, window 3998..3999
    assert len(Sn) == 3 and Sn[2] == 2.0
    P = np.zeros((nz, nb)); P[mid, 0] = 4.0; P[mid, 1] = 1.0
    assert np.allclose(oracle.harmonic_sums_nbr_at(P, 4, 0, mid), [4, 8, 12, 16])   # every window contains bin 0


def test_p13_neighbour_maximised_candidates(oracle):
    """orc_candidates_nbr = the O6 rule on S': the triples of a constructed plane, the count of defined
    triples under a negative threshold (identical to the plain sums'), powers and the tie rule."""
    nz, nb, H, r_lo = 33, 600, 16, 5
    mid = 16
    P = np.ones((nz, nb))
    c = oracle.candidates(P, H, -np.ones(H), r_lo, nbr=True)
    expect = sum(((nb - 1) // h - r_lo + 1) * (2 * (16 // h) + 1) for h in range(1, H + 1))
    assert c.count == expect == oracle.candidates(P, H, -np.ones(H), r_lo).count
    # one off-bin second harmonic: (r0, z = 3) fundamental 5.0 at r0, second harmonic 5.0 at 2 r0 + 1
    P = np.zeros((nz, nb))
    r0 = 100
    P[mid + 3, r0] = 5.0
    P[mid + 6, 2 * r0 + 1] = 5.0
    plain = oracle.candidates(P, 2, np.array([4.0, 9.0]), r_lo).as_dict()
    nbr = oracle.candidates(P, 2, np.array([4.0, 9.0]), r_lo, nbr=True).as_dict()
    assert (r0, mid + 3, 2) not in plain and nbr[(r0, mid + 3, 2)][0] == 10.0
    # the spike at 2 r0 + 1 is also the k = 2 neighbour of fundamentals r0 + 1 (2 r0 + 2 - 1): S'_2 = 5 < 9
    assert (r0 + 1, mid + 3, 2) not in nbr
    assert set(k for k in nbr if k[2] == 1) == set(k for k in plain if k[2] == 1)    # h = 1 is unchanged
    assert nbr[(r0, mid + 3, 2)][1] == 1                                            # isolated: local maximum
    # tie rule on S': two equal neighbouring fundamentals, the first in (j, r) order keeps the flag
    P = np.zeros((nz, nb)); P[mid, 50] = 3.0; P[mid, 51] = 3.0
    d = oracle.candidates(P, 1, np.array([1.0]), 1, nbr=True).as_dict()
    assert d[(50, mid, 1)][1] == 1 and d[(51, mid, 1)][1] == 0

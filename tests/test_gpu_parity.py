"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle on the same seeded
inputs.  Tolerances are BASELINE.json north_star's:
    fp32 path   |GPU - oracle| <= 1e-4 x plane maximum
    bf16 path   <= 2e-2 x plane maximum, candidate powers within 3 %
    candidate (r, z, h) lists identical except entries within that tolerance of the threshold.
Run with `pytest -m gpu` on the B200 box.
"""
import numpy as np
import pytest

from paper_2211_13517_b200 import inputs
from helpers import (REL_POW, STRICT_REL, TOL, PlaneStats, compare_candidates, gpu_cand_dict,
                     local_amplitude, membership_window, oracle_margin_fn, record_stats)

pytestmark = pytest.mark.gpu

ALL_PREC = ["fp32", "bf16", "bf16_plane16", "bf16_tc", "bf16_tc_plane16"]


@pytest.fixture(scope="module")
def fdas():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2211_13517_b200 import fdas as F   # raises if libfdas.so is missing (no fallback)
    return F


@pytest.fixture(scope="module")
def torch_():
    import torch
    return torch


def spec_to_complex(torch, d_spec):
    a = d_spec.float().cpu().numpy().astype(np.float64)
    return a[:, 0] + 1j * a[:, 1]


def spec_from_complex(torch, w, precision):
    a = np.stack([w.real, w.imag], axis=1).astype(np.float32)
    t = torch.from_numpy(a).cuda()
    return t if precision == "fp32" else t.to(torch.bfloat16)


def run_gpu(fdas, torch, wl, x, precision, capacity=1 << 16, thr=None):
    plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, precision)
    d_x = torch.from_numpy(x).cuda()
    d_spec, d_plane = plan.alloc_spec(), plan.alloc_plane()
    d_plane.fill_(float("nan"))
    d_c, d_n = plan.alloc_cands(capacity)
    if thr is None:
        thr = fdas.thresholds_from_sigma(wl.nharm, wl.nsigma)
    plan.prepare_spectrum(d_x, d_spec)
    plan.convolve_plane(d_spec, d_plane)
    plan.harmonic_sum_peaks(d_plane, wl.nharm, thr, wl.r_lo, d_c, d_n)
    torch.cuda.synchronize()
    res = plan.read_cands(d_c, d_n)
    return plan, d_spec, d_plane, res, thr


# ------------------------------------------------------------------------------------ configs[0]
def test_tiny_fp32_full_parity(fdas, torch_, oracle):
    torch = torch_
    wl = inputs.tiny()
    x = inputs.series_for(wl)
    plan, d_spec, d_plane, res, thr = run_gpu(fdas, torch, wl, x, "fp32")
    info = plan.info
    assert (info.nfft, info.nbins, info.nz, info.halfwidth, info.valid, info.nseg) == \
        (1 << 17, 1 << 16, 33, 32, 1984, 34)
    orc = oracle.run(x, wl.nfft, wl.zmax, wl.zstep, wl.nharm, wl.nsigma, wl.r_lo, want_candidates=False)
    # library templates = oracle templates (closed form vs quadrature)
    assert np.abs(plan.templates_host() - orc.bank).max() < 1e-12
    # whitened spectrum
    w_gpu = spec_to_complex(torch, d_spec)
    assert w_gpu[0] == 0
    assert np.abs(w_gpu - orc.w).max() <= 2e-5 * np.abs(orc.w).max()
    # plane: every element, fp32 tolerance
    P_gpu = d_plane.cpu().numpy().astype(np.float64)
    assert not np.isnan(P_gpu).any()
    ps = PlaneStats("fp32")
    ps.add(P_gpu, orc.P, local_amplitude(orc.w))
    ps.check(orc.P.max())
    # candidates (oracle gets the same float32 thresholds)
    oc = oracle.candidates(orc.P, wl.nharm, thr.astype(np.float64), wl.r_lo)
    s_at, margin = oracle_margin_fn(oracle, orc.P, wl.nharm, wl.r_lo)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, TOL["fp32"] * orc.P.max(),
                               None, s_at, margin, strict_rel=STRICT_REL["fp32"])
    assert res.count == len(res.cands) and stats["common"] >= 1
    assert stats["only_gpu"] + stats["only_orc"] == 0, stats
    record_stats("tiny_fp32", {**ps.summary(orc.P.max()), **stats})
    keys = set(gpu_cand_dict(res.cands))
    assert (20000, 23, 1) in keys or (20000, 24, 1) in keys     # the injected signal (z0 = 7.5)
    assert plan.launch_count() == 7      # K1a, K1b, K2, K3: general prefilter (+ coarsen), coarse + block level, exact, flags (cuFFT not counted)


# ------------------------------------------------------------------------------------ configs[1]
@pytest.fixture(scope="module")
def medium_oracle(oracle):
    wl = inputs.medium()
    x = inputs.series_for(wl)
    orc = oracle.run(x, wl.nfft, wl.zmax, wl.zstep, wl.nharm, wl.nsigma, wl.r_lo, want_candidates=False)
    return wl, x, orc


@pytest.mark.parametrize("precision", ALL_PREC)
def test_medium_full_parity(fdas, torch_, oracle, medium_oracle, precision):
    torch = torch_
    wl, x, orc = medium_oracle
    plan, d_spec, d_plane, res, thr = run_gpu(fdas, torch, wl, x, precision)
    assert (plan.info.nbins, plan.info.nz, plan.info.halfwidth, plan.info.nseg) == (1 << 20, 193, 64, 547)
    pmax = orc.P.max()
    tol = TOL[precision] * pmax
    # plane, element by element, in row chunks to bound host memory
    ps = PlaneStats(precision)
    W = local_amplitude(orc.w)
    for j0 in range(0, plan.info.nz, 16):
        Pg = d_plane[j0:j0 + 16].float().cpu().numpy().astype(np.float64)
        assert not np.isnan(Pg).any()
        ps.add(Pg, orc.P[j0:j0 + 16], W)
    ps.check(pmax)
    worst = ps.worst_abs
    oc = oracle.candidates(orc.P, wl.nharm, thr.astype(np.float64), wl.r_lo)
    s_at, margin = oracle_margin_fn(oracle, orc.P, wl.nharm, wl.r_lo)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, tol, REL_POW[precision],
                               s_at, margin, strict_rel=STRICT_REL[precision])
    if precision == "fp32":
        assert stats["only_gpu"] + stats["only_orc"] == 0, stats
    else:       # bf16 storage moves ~0.3 % of the 4e4 triples across their threshold, all within 3 % of it
        assert stats["only_gpu"] + stats["only_orc"] <= 0.01 * stats["common"], stats
    assert stats["flags_checked"] > 1000
    record_stats("medium_" + precision, {**ps.summary(pmax), **stats})
    # the four injected chirps are recovered at (round(r_c), nearest z)
    keys = set(gpu_cand_dict(res.cands))
    for s in wl.signals:
        if s.amp ** 2 * wl.nfft / 4 < 60:
            continue
        r0, j0 = int(round(s.r_c)), int(round(s.z + wl.zmax))
        assert any((r0 + dr, j0 + dj, 1) in keys for dr in (-1, 0, 1) for dj in (-1, 0, 1)), s
    assert stats["common"] >= 4
    print(precision, ps.summary(pmax), stats)


# --------------------------------------------------------------- K2 alone, fed a chosen spectrum
@pytest.mark.parametrize("precision", ALL_PREC)
def test_convolve_alone_seams_tail_and_invariants(fdas, torch_, oracle, precision):
    torch = torch_
    n = 1 << 15                      # nbins = 16384: 9 segments of V = 1984 + ragged tail
    plan = fdas.Plan(n, 64e-6, 16.0, 1.0, 2048, precision)
    nb, nz = plan.info.nbins, plan.info.nz
    rng = np.random.default_rng(8)
    w = (rng.standard_normal(nb) + 1j * rng.standard_normal(nb)) / np.sqrt(2)
    for k in (0, 1, 1983, 1984, 1985, 3968, nb - 1):      # lines on and around segment seams
        w[k] += 12.0
    d_spec = spec_from_complex(torch, w, precision)
    wq = spec_to_complex(torch, d_spec)                   # what the kernel actually reads
    d_plane = plan.alloc_plane(); d_plane.fill_(float("nan"))
    plan.convolve_plane(d_spec, d_plane)
    torch.cuda.synchronize()
    Pg = d_plane.float().cpu().numpy().astype(np.float64)
    assert not np.isnan(Pg).any()
    bank = oracle.template_bank(16.0, 1.0)
    P = oracle.plane(w, bank)
    ps = PlaneStats(precision)
    ps.add(Pg, P, local_amplitude(w))
    ps.check(P.max())
    if precision == "fp32":
        # z = 0 row is the power spectrum; conj(w) flips the z axis; a shift by d bins (not a
        # multiple of V) shifts every row
        assert np.abs(Pg[16] - np.abs(wq) ** 2).max() <= 1e-5 * P.max()
        d_spec_c = spec_from_complex(torch, np.conj(w), precision)
        d_plane_c = plan.alloc_plane()
        plan.convolve_plane(d_spec_c, d_plane_c)
        Pc = d_plane_c.cpu().numpy()
        assert np.abs(Pc - Pg[::-1]).max() <= 1e-5 * P.max()
        d = 777
        ws = np.concatenate([np.zeros(d), w[:-d]])
        d_plane_s = plan.alloc_plane()
        plan.convolve_plane(spec_from_complex(torch, ws, precision), d_plane_s)
        Ps = d_plane_s.cpu().numpy()
        assert np.abs(Ps[:, d + 32: nb - 32] - Pg[:, 32: nb - d - 32]).max() <= 1e-5 * P.max()
    else:
        # quantised oracle (reading A11): bf16-rounded spectrum, double arithmetic -- the kernel's
        # remaining error is template quantisation + fp32 arithmetic (+ plane rounding)
        Pq = oracle.plane(wq, bank)
        assert np.abs(Pg - Pq).max() <= 1e-2 * P.max()
    if precision.startswith("bf16_tc"):
        # tensor-core contraction: the z = 0 row is |w|^2 of the stored spectrum (T_0 = delta), and
        # conj(w) negates Im-part accumulators only, so the z axis flips bit-exactly
        rel = 2.0 ** -8 if precision.endswith("plane16") else 1e-6
        assert np.abs(Pg[16] - np.abs(wq) ** 2).max() <= rel * P.max()
        d_plane_c = plan.alloc_plane()
        plan.convolve_plane(spec_from_complex(torch, np.conj(w), precision), d_plane_c)
        assert torch.equal(d_plane_c, torch.flip(d_plane, dims=[0]))


def test_smallest_plan_and_zmax0(fdas, torch_, oracle):
    torch = torch_
    plan = fdas.Plan(4096, 64e-6, 0.0, 1.0, 2048, "fp32")   # N = 2 * seg_len, one template (delta)
    assert (plan.info.nbins, plan.info.nz, plan.info.halfwidth, plan.info.nseg) == (2048, 1, 32, 2)
    x = np.random.default_rng(1).standard_normal(4096).astype(np.float32)
    d_spec, d_plane = plan.alloc_spec(), plan.alloc_plane()
    plan.prepare_spectrum(torch.from_numpy(x).cuda(), d_spec)
    plan.convolve_plane(d_spec, d_plane)
    torch.cuda.synchronize()
    w = spec_to_complex(torch, d_spec)
    worc = oracle.whiten(oracle.spectrum(x, 4096))
    assert np.abs(w - worc).max() <= 2e-5 * np.abs(worc).max()
    assert np.abs(d_plane.cpu().numpy()[0] - np.abs(w) ** 2).max() <= 1e-5 * (np.abs(w) ** 2).max()


def test_non_power_of_two_series_uses_largest_pow2(fdas, torch_, oracle):
    torch = torch_
    n = 100_000                                # nfft = 65536 (reading A1); the tail is ignored
    plan = fdas.Plan(n, 64e-6, 16.0, 1.0, 2048, "fp32")
    assert plan.info.n_in == n and plan.info.nfft == 65536
    x = np.random.default_rng(12).standard_normal(n).astype(np.float32)
    d_spec = plan.alloc_spec()
    plan.prepare_spectrum(torch.from_numpy(x).cuda(), d_spec)
    torch.cuda.synchronize()
    worc = oracle.whiten(oracle.spectrum(x, 65536))
    assert np.abs(spec_to_complex(torch, d_spec) - worc).max() <= 2e-5 * np.abs(worc).max()


# ----------------------------------------------------------------- K3 alone on hand-made planes
@pytest.mark.parametrize("precision", ["fp32", "bf16_plane16"])
def test_harmonic_sum_alone_many_candidates(fdas, torch_, oracle, precision):
    torch = torch_
    plan = fdas.Plan(1 << 15, 64e-6, 16.0, 1.0, 2048, precision)
    nb, nz = plan.info.nbins, plan.info.nz
    rng = np.random.default_rng(17)
    P32 = rng.exponential(1.0, size=(nz, nb)).astype(np.float32)
    d_plane = torch.from_numpy(P32).cuda()
    if precision == "bf16_plane16":
        d_plane = d_plane.to(torch.bfloat16)
    P = d_plane.float().cpu().numpy().astype(np.float64)     # the values the kernel reads
    H = 16
    thr = fdas.thresholds_from_sigma(H, 3.0)                 # ~1e-3 of the points pass
    d_c, d_n = plan.alloc_cands(1 << 18)
    plan.harmonic_sum_peaks(d_plane, H, thr, 5, d_c, d_n)
    torch.cuda.synchronize()
    res = plan.read_cands(d_c, d_n)
    oc = oracle.candidates(P, H, thr.astype(np.float64), 5)
    assert oc.count > 500
    s_at, margin = oracle_margin_fn(oracle, P, H, 5)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, 2e-6 * P.max(), None, s_at, margin,
                               strict_rel=1e-5)
    assert stats["only_gpu"] + stats["only_orc"] <= 3 and stats["flags_checked"] > 100
    # H = 1, r_lo beyond the plane, capacity overflow
    plan.harmonic_sum_peaks(d_plane, 1, thr, nb, d_c, d_n)
    assert plan.read_cands(d_c, d_n).count == 0
    d_small, _ = plan.alloc_cands(10)
    plan.harmonic_sum_peaks(d_plane, H, thr, 5, d_small, d_n)
    small = plan.read_cands(d_small, d_n)
    assert small.count == res.count and len(small.cands) == 10
    assert set(gpu_cand_dict(small.cands)) <= set(gpu_cand_dict(res.cands))


@pytest.mark.parametrize("H", [1, 2, 3, 4, 5, 32])
def test_harmonic_sum_small_h_exact_sets(fdas, torch_, oracle, H):
    """K3 on a hand-made plane for small harmonic counts: with H <= 2 every row but z = 0 goes
    through the streaming shallow pass, H = 3, 5 mix both passes; the threads that straddle
    r = (Nb-1)/k (harmonic k defined for their first fundamentals only) and an r_lo inside a block
    are exercised.  fp32 plane, so the candidate set must be the oracle's exactly (up to rounding
    at the threshold)."""
    torch = torch_
    plan = fdas.Plan(1 << 13, 64e-6, 16.0, 1.0, 2048, "fp32")      # nbins = 4096: few CTAs per row
    nb, nz = plan.info.nbins, plan.info.nz
    rng = np.random.default_rng(23 + H)
    P32 = rng.exponential(1.0, size=(nz, nb)).astype(np.float32)
    # spikes around the harmonic cut-offs r = (Nb-1)/k and at the plane's corners
    for k in (1, 2, 3):
        rc = (nb - 1) // k
        for dr in (-33, -2, -1, 0):
            P32[:, min(nb - 1, max(0, rc + dr))] += 9.0
    P32[0, 0] += 50.0; P32[nz - 1, nb - 1] += 50.0; P32[nz // 2, 77] += 50.0
    d_plane = torch.from_numpy(P32).cuda()
    P = P32.astype(np.float64)
    thr = fdas.thresholds_from_sigma(H, 2.5)
    r_lo = 37
    d_c, d_n = plan.alloc_cands(1 << 18)
    plan.harmonic_sum_peaks(d_plane, H, thr, r_lo, d_c, d_n)
    torch.cuda.synchronize()
    res = plan.read_cands(d_c, d_n)
    oc = oracle.candidates(P, H, thr.astype(np.float64), r_lo)
    assert oc.count > 200 and res.count == len(res.cands)
    s_at, margin = oracle_margin_fn(oracle, P, H, r_lo)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, 2e-6 * P.max(), None, s_at, margin,
                               strict_rel=1e-5)
    assert stats["only_gpu"] + stats["only_orc"] <= 2, stats
    assert min(k[0] for k in gpu_cand_dict(res.cands)) >= r_lo
    # the count is the oracle's (gpu_cand_dict has already refused duplicated records: with H <= 4 the z = 0
    # row of an odd bank once went through both prefilter levels and was listed twice)
    assert res.count == oc.count + stats["only_gpu"] - stats["only_orc"]


@pytest.mark.parametrize("H", [1, 2, 4, 5])
@pytest.mark.parametrize("zmax", [0.0, 1.0])
def test_harmonic_sum_counts_on_the_smallest_banks(fdas, torch_, oracle, H, zmax):
    """nz = 1 and nz = 3 (odd banks, the centre row is the whole or a third of the plane), no list overflow:
    count and set equal the oracle's, no record twice."""
    torch = torch_
    plan = fdas.Plan(1 << 15, 64e-6, zmax, 1.0, 2048, "fp32")
    nb, nz = plan.info.nbins, plan.info.nz
    assert nz == 2 * int(zmax) + 1
    rng = np.random.default_rng(101 + H + int(zmax))
    P32 = rng.exponential(1.0, size=(nz, nb)).astype(np.float32)
    d_plane = torch.from_numpy(P32).cuda()
    P = P32.astype(np.float64)
    thr = fdas.thresholds_from_sigma(H, 2.5)
    d_c, d_n = plan.alloc_cands(1 << 16)
    plan.harmonic_sum_peaks(d_plane, H, thr, 1, d_c, d_n)
    torch.cuda.synchronize()
    res = plan.read_cands(d_c, d_n)
    oc = oracle.candidates(P, H, thr.astype(np.float64), 1)
    assert oc.count > 50 and res.count == len(res.cands)
    s_at, margin = oracle_margin_fn(oracle, P, H, 1)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, 2e-6 * P.max(), None, s_at, margin,
                               strict_rel=1e-5)
    assert stats["only_gpu"] + stats["only_orc"] <= 2, stats
    assert res.count == oc.count + stats["only_gpu"] - stats["only_orc"]


@pytest.mark.parametrize("case", range(8))
def test_harmonic_sum_hand_made_planes_against_the_oracle(fdas, torch_, oracle, case):
    """K3 alone on seeded hand-made planes that stress the integer bounds of the prefilter: values far above the
    saturation of the block-max codes (127.875), exact multiples of the code unit (1/8), zeros, thresholds that are
    not monotone in h, a negative threshold (every point passes), thresholds above the saturation, r_lo inside a
    block, odd and even template counts, plane widths of 1024 .. 32768 bins -- and in the neighbour-maximised mode
    as well.  fp32 planes: the candidate set is the oracle's (up to rounding at a threshold)."""
    torch = torch_
    rng = np.random.default_rng(900 + case)
    zmax = [16.0, 7.5, 32.0, 16.0, 96.0, 3.0, 16.0, 7.5][case]
    n = [1 << 13, 1 << 14, 1 << 15, 1 << 16, 1 << 13, 1 << 14, 1 << 11, 1 << 13][case]
    H = [16, 8, 5, 32, 16, 12, 4, 16][case]
    nbr = case in (3, 6)
    plan = fdas.Plan(n, 64e-6, zmax, 1.0, 1024 if n == (1 << 11) else 2048, "fp32")
    nb, nz = plan.info.nbins, plan.info.nz
    P32 = rng.exponential(1.0, size=(nz, nb)).astype(np.float32)
    P32 = np.ceil(P32 * 8.0).astype(np.float32) / 8.0 if case % 2 else P32          # exact code boundaries
    P32[rng.random((nz, nb)) < 0.05] = 0.0
    for _ in range(40):                                                             # lines with harmonics
        j, r = int(rng.integers(0, nz)), int(rng.integers(1, nb // 4))
        a = float(rng.choice([6.0, 30.0, 127.875, 128.0, 500.0, 4000.0]))
        c = (nz - 1) // 2
        for k in range(1, 9):
            rk, jk = k * r, k * (j - c) + c                  # row of harmonic k (odd template counts)
            if nz % 2 and rk < nb and 0 <= jk < nz:
                P32[jk, rk] += a / k
    thr = fdas.thresholds_from_sigma(H, [3.0, 2.5, 3.5, 2.0, 3.0, 2.5, 2.5, 3.0][case]).copy()
    if case == 1:
        thr[2] = 0.6 * thr[1]; thr[5] = 400.0               # not monotone; one above the saturation
    if case == 2:
        thr[0] = -1.0                                       # every point passes h = 1
    if case == 5:
        thr[:] = thr * 6.0 + 130.0                          # all above the saturation: only strong lines
    r_lo = [37, 1, 64, 9, 200, 5, 3, 0][case]
    if nbr:
        plan.set_harmonic_mode("neighbour_max")
    d_plane = torch.from_numpy(P32).cuda()
    cap = 1 << 22
    d_c, d_n = plan.alloc_cands(cap)
    plan.harmonic_sum_peaks(d_plane, H, thr, r_lo, d_c, d_n)
    torch.cuda.synchronize()
    res = plan.read_cands(d_c, d_n)
    P = P32.astype(np.float64)
    oc = oracle.candidates(P, H, thr.astype(np.float64), r_lo, capacity=cap, nbr=nbr)
    assert res.count <= cap and oc.count > 50
    got, want = gpu_cand_dict(res.cands), oc.as_dict()
    sums = oracle.harmonic_sums_nbr_at if nbr else oracle.harmonic_sums_at
    for key in set(got) ^ set(want):                        # one-sided: the oracle's sum sits on its threshold
        so = want[key][0] if key in want else float(sums(P, key[2], key[0], key[1])[key[2] - 1])
        assert abs(so - thr[key[2] - 1]) <= 2e-6 * max(abs(so), 1.0), (case, key, so, thr[key[2] - 1])
    assert len(set(got) ^ set(want)) <= 4
    for key in set(got) & set(want):
        assert abs(got[key][0] - want[key][0]) <= 2e-6 * max(want[key][0], 1.0), (case, key)
    assert min(k[0] for k in got) >= r_lo
    plan.close()


def test_abi_errors_on_device(fdas, torch_):
    import ctypes as C
    torch = torch_
    plan = fdas.Plan(1 << 15, 64e-6, 16.0, 1.0, 2048, "fp32")
    lib = fdas.lib()
    d_plane = plan.alloc_plane()
    thr = np.ones(32, dtype=np.float32)
    thr_c = thr.ctypes.data_as(C.POINTER(C.c_float))
    d_c, d_n = plan.alloc_cands(16)
    assert lib.fdas_harmonic_sum_peaks(plan._h, d_plane.data_ptr(), 0, thr_c, 0, d_c.data_ptr(), 16, d_n.data_ptr(), None) == fdas.FDAS_EARG
    assert lib.fdas_harmonic_sum_peaks(plan._h, d_plane.data_ptr(), 33, thr_c, 0, d_c.data_ptr(), 16, d_n.data_ptr(), None) == fdas.FDAS_EARG
    assert lib.fdas_harmonic_sum_peaks(plan._h, d_plane.data_ptr(), 4, thr_c, -1, d_c.data_ptr(), 16, d_n.data_ptr(), None) == fdas.FDAS_EARG
    assert lib.fdas_harmonic_sum_peaks(plan._h, None, 4, thr_c, 0, d_c.data_ptr(), 16, d_n.data_ptr(), None) == fdas.FDAS_EARG
    assert lib.fdas_convolve_plane(plan._h, None, d_plane.data_ptr(), None) == fdas.FDAS_EARG
    assert lib.fdas_prepare_spectrum(plan._h, None, None, None) == fdas.FDAS_EARG


# ------------------------------------------------------------------ end-to-end host entry point
def test_search_host_equals_device_calls(fdas, torch_):
    torch = torch_
    wl = inputs.tiny()
    x = inputs.series_for(wl)
    plan, _, _, res, thr = run_gpu(fdas, torch, wl, x, "fp32")
    out = plan.search_host(x, wl.nharm, thr, wl.r_lo, capacity=4096)
    assert out.count == res.count
    assert gpu_cand_dict(out.cands) == gpu_cand_dict(res.cands)
    tiny_cap = plan.search_host(x, wl.nharm, thr, wl.r_lo, capacity=1)
    assert tiny_cap.count == res.count and len(tiny_cap.cands) == 1


# ------------------------------------------------------- configs[2] at full size: sampled parity
@pytest.mark.parametrize("precision", ["bf16", "fp32", "bf16_tc", "bf16_tc_plane16", "bf16_plane16"])
def test_ska_full_size_sampled_parity(fdas, torch_, oracle, precision):
    """SKA-like single DM trial in the launch configuration bench.py times.  The oracle computes
    sampled plane points and sampled harmonic sums one by one from its own whitened spectrum."""
    torch = torch_
    wl = inputs.ska()
    x = inputs.series_for(wl)
    plan, d_spec, d_plane, res, thr = run_gpu(fdas, torch, wl, x, precision)
    info = plan.info
    assert (info.n_in, info.nfft, info.nbins, info.nz, info.nseg) == (9_375_000, 1 << 23, 1 << 22, 193, 2185)
    w = oracle.whiten(oracle.spectrum(x, wl.nfft))
    w_gpu = spec_to_complex(torch, d_spec)
    stol = 2e-5 if precision == "fp32" else 1e-2
    assert np.abs(w_gpu - w).max() <= stol * np.abs(w).max()
    bank = oracle.template_bank(wl.zmax, wl.zstep)
    nb, nz, V = info.nbins, info.nz, info.valid
    rng = np.random.default_rng(99)
    rr = [rng.integers(0, nb, 30000)]
    jj = [rng.integers(0, nz, 30000)]
    # segment seams, the first bins, the ragged tail, and the injected signals' neighbourhoods
    seams = np.array([s * V + d for s in (1, 2, 1000, 2184) for d in (-2, -1, 0, 1, 2)])
    tiles = np.array([t * 128 + d for t in (1, 147, 148, 149, 32767) for d in (-1, 0, 1)])   # K2-TC tile seams
    for cols in (seams, tiles, np.arange(0, 70), np.arange(nb - 70, nb)):
        for j in (0, 56, 96, 136, 192):
            rr.append(cols); jj.append(np.full(cols.size, j))
    for s in wl.signals:
        for k in (1, 2):
            r0, j0 = int(round(k * s.r_c)), int(round(k * s.z + wl.zmax))
            g_r, g_j = np.meshgrid(np.arange(r0 - 6, r0 + 7), np.arange(j0 - 3, j0 + 4))
            rr.append(g_r.ravel()); jj.append(g_j.ravel())
    rr = np.concatenate(rr).astype(np.int64); jj = np.concatenate(jj).astype(np.int32)
    Po = oracle.plane_points(w, bank, rr, jj)
    Pg = d_plane[torch.from_numpy(jj.astype(np.int64)).cuda(), torch.from_numpy(rr).cuda()].float().cpu().numpy()
    # plane maximum: taken from the GPU plane, cross-checked against the oracle at that point
    flat = int(torch.argmax(d_plane.float()).item())
    jm, rm = flat // info.plane_pitch, flat % info.plane_pitch
    pmax = float(oracle.plane_points(w, bank, [rm], [jm])[0])
    assert abs(float(d_plane[jm, rm]) - pmax) <= TOL[precision] * pmax and pmax > 100
    worst = np.abs(Pg - Po).max()
    assert worst <= TOL[precision] * pmax, worst / pmax
    assert not torch.isnan(d_plane.float().sum()).item()      # every element was written
    # candidates: every GPU candidate is valid in the oracle; sampled fundamentals agree both ways
    gd = gpu_cand_dict(res.cands)
    assert res.count == len(gd) and res.count < 20000
    tol = TOL[precision] * pmax
    if gd:
        keys = sorted(gd)
        kr = np.array([k[0] for k in keys]); kj = np.array([k[1] for k in keys], dtype=np.int32)
        S, hmax = oracle.harmonic_sums_sampled(w, bank, wl.nharm, kr, kj)
        for i, (r, j, h) in enumerate(keys):
            assert h <= hmax[i]
            so = S[i, h - 1]
            assert so > thr[h - 1] - membership_window(thr, h, tol, precision), ((r, j, h), so)
            assert abs(gd[(r, j, h)][0] - so) <= h * tol
            if REL_POW[precision] is not None:
                assert abs(gd[(r, j, h)][0] - so) <= REL_POW[precision] * so
    sr = np.concatenate([rng.integers(wl.r_lo, nb, 4000)] +
                        [np.arange(int(round(s.r_c)) - 3, int(round(s.r_c)) + 4) for s in wl.signals])
    sj = np.concatenate([rng.integers(0, nz, 4000)] +
                        [np.full(7, int(round(s.z + wl.zmax))) for s in wl.signals]).astype(np.int32)
    S, hmax = oracle.harmonic_sums_sampled(w, bank, wl.nharm, sr, sj)
    found = 0
    for i in range(sr.size):
        for h in range(1, hmax[i] + 1):
            key = (int(sr[i]), int(sj[i]), h)
            win = membership_window(thr, h, tol, precision)
            if S[i, h - 1] > thr[h - 1] + win:
                assert key in gd, key
                found += 1
            elif S[i, h - 1] < thr[h - 1] - win:
                assert key not in gd, key
    assert found >= 2          # both injected fundamentals
    print(precision, "sampled worst/max", worst / pmax, "pmax", pmax, "cands", res.count, "found", found)


# ---------------------------------------------- K2's block-max side plane and the K3 prefilter
@pytest.mark.parametrize("precision", ["fp32", "bf16_plane16", "bf16_tc", "bf16_tc_plane16"])
def test_blockmax_plane_and_prefilter_equivalence(fdas, torch_, precision):
    """M[j][b] written by K2 equals the maximum of the 8 stored plane values of block b rounded up to
    bfloat16 (bit-exact), and
    the branch-and-bound search gives the same candidates whether M comes from K2 or is rebuilt from
    a copy of the plane."""
    torch = torch_
    wl = inputs.medium()
    x = inputs.series_for(wl)
    plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, precision)
    d_spec, d_plane = plan.alloc_spec(), plan.alloc_plane()
    plan.prepare_spectrum(torch.from_numpy(x).cuda(), d_spec)
    plan.convolve_plane(d_spec, d_plane)
    torch.cuda.synchronize()
    ptr, pitch = plan.debug_maxplane()
    nz, nb = plan.info.nz, plan.info.nbins
    assert pitch == nb // 8
    M = _device_view(torch, ptr, nz * pitch).view(nz, pitch).clone()
    ref = d_plane.float().view(nz, pitch, 8).amax(dim=2)
    assert torch.equal(M, max_codes(torch, ref))
    up = M.float() / 8.0          # the bound a code stands for (1023: none)
    assert bool(((up >= ref) | (M == 1023)).all()) and bool(((up <= ref + 0.125) | (M == 1023)).all())
    H = wl.nharm
    thr = fdas.thresholds_from_sigma(H, 4.0)      # lower threshold: more work for the exact pass
    d_c, d_n = plan.alloc_cands(1 << 18)
    plan.harmonic_sum_peaks(d_plane, H, thr, wl.r_lo, d_c, d_n)
    a = plan.read_cands(d_c, d_n)
    clone = d_plane.clone()
    plan.harmonic_sum_peaks(clone, H, thr, wl.r_lo, d_c, d_n)
    b = plan.read_cands(d_c, d_n)
    assert a.count == b.count and a.count > 1000
    assert gpu_cand_dict(a.cands) == gpu_cand_dict(b.cands)


@pytest.mark.parametrize("precision", ["bf16_tc", "bf16_tc_plane16"])
@pytest.mark.parametrize("zmax", [4.0, 10.0, 20.0, 52.0, 7.5, 110.0, 140.0])
def test_tensor_core_path_odd_banks(fdas, torch_, oracle, precision, zmax):
    """K2-TC with banks whose pair count is not a multiple of 32 (4, 10, 20, 52 pairs: a ragged last
    lane quarter, stored through the tail tensor map), an even bank without a z = 0 row (zmax 7.5: 8
    pairs), 110 pairs (all four lane quarters, single-buffered staging) and 140 pairs (two launches of 96
    and 44): no row outside the plane may be touched (canaries), every real row must be written, the
    block-max side plane must be exact and the candidates must match."""
    torch = torch_
    n = 1 << 14                                   # nbins = 8192: 64 tiles over <= 148 CTAs
    plan = fdas.Plan(n, 64e-6, zmax, 1.0, 2048, precision)
    nb, nz = plan.info.nbins, plan.info.nz
    assert nz == int(2 * zmax) + 1
    rng = np.random.default_rng(int(zmax))
    w = (rng.standard_normal(nb) + 1j * rng.standard_normal(nb)) / np.sqrt(2)
    for k in (0, 127, 128, 129, 5000, nb - 1):
        w[k] += 10.0
    d_spec = spec_from_complex(torch, w, precision)
    wq = spec_to_complex(torch, d_spec)
    # canaries around the plane: the rows before and after it must stay untouched
    elem = torch.bfloat16 if precision.endswith("plane16") else torch.float32
    big = torch.full((nz + 16, nb), -7.0, dtype=elem, device="cuda")
    d_plane = big[8:8 + nz]
    plan.convolve_plane(d_spec, d_plane)
    torch.cuda.synchronize()
    assert bool((big[:8] == -7.0).all()) and bool((big[8 + nz:] == -7.0).all())
    Pg = d_plane.float().cpu().numpy().astype(np.float64)
    assert (Pg >= 0).all()                        # every element written (canary is negative)
    bank = oracle.template_bank(zmax, 1.0)
    P = oracle.plane(w, bank)
    assert np.abs(Pg - P).max() <= TOL[precision] * P.max()
    assert np.abs(Pg - oracle.plane(wq, bank)).max() <= 1e-2 * P.max()
    # block-max side plane: bit-exact upper bound of the stored values
    ptr, pitch = plan.debug_maxplane()
    M = _device_view(torch, ptr, nz * pitch).view(nz, pitch).clone()
    ref = d_plane.float().contiguous().view(nz, pitch, 8).amax(dim=2)
    assert torch.equal(M, max_codes(torch, ref))
    # harmonic sums on that plane
    H = 8
    thr = fdas.thresholds_from_sigma(H, 3.0)
    d_c, d_n = plan.alloc_cands(1 << 16)
    plan.harmonic_sum_peaks(d_plane, H, thr, 16, d_c, d_n)
    res = plan.read_cands(d_c, d_n)
    oc = oracle.candidates(Pg, H, thr.astype(np.float64), 16)
    s_at, margin = oracle_margin_fn(oracle, Pg, H, 16)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, 2e-6 * Pg.max(), None, s_at, margin,
                               strict_rel=1e-5)
    assert stats["only_gpu"] + stats["only_orc"] <= 2 and stats["common"] > 10, stats


def test_tensor_core_path_unsupported_banks(fdas, torch_):
    """Banks the tensor-core kernel cannot hold are refused at plan time (no silent fallback):
    nz = 1 (no conjugate pairs) and templates of more than 255 taps (zmax 260: h = 160; the bank images
    would not fit the tensor-memory columns beside the accumulators); the FFT path takes the same plans."""
    for zmax, zstep in ((0.0, 1.0), (260.0, 1.0)):
        with pytest.raises(fdas.FdasError) as ei:
            fdas.Plan(1 << 14, 64e-6, zmax, zstep, 2048, "bf16_tc")
        assert ei.value.status == fdas.FDAS_EUNSUPPORTED
        fdas.Plan(1 << 14, 64e-6, zmax, zstep, 2048, "bf16").close()


def max_codes(torch, ref):
    """Expected block-max codes (csrc/fdas_maxcode.h): min(1023, ceil(8 x max of the 8 stored values)) as int16."""
    return torch.clamp(torch.ceil(ref * 8.0), min=0.0, max=1023.0).to(torch.int16)


def _device_view(torch, ptr, numel):
    """int16 tensor aliasing `numel` 16-bit words of device memory at `ptr` (no copy)."""
    class _Iface:
        __cuda_array_interface__ = {"shape": (numel,), "typestr": "<i2", "data": (ptr, False), "version": 3}
    return torch.as_tensor(_Iface(), device="cuda")


@pytest.mark.parametrize("precision", ["bf16_tc", "bf16"])
def test_ska_zero_padded_2p24_sampled_parity(fdas, torch_, oracle, precision):
    """Reading A1-B of configs[2]: all 9,375,000 samples, mean-subtracted and zero-padded to 2^24 by
    the caller (Nb = 2^23, 1.6e9 plane points, a 6.5 GB fp32 plane, 65536 K2-TC tiles), both bf16
    formulations: sampled plane parity against the oracle's own spectrum, candidates valid in the oracle."""
    torch = torch_
    wl = inputs.ska_padded()
    x = inputs.series_for(wl)
    assert x.size == 1 << 24 and not x[9_375_000:].any() and abs(float(x[:9_375_000].mean())) < 1e-6
    plan, d_spec, d_plane, res, thr = run_gpu(fdas, torch, wl, x, precision)
    info = plan.info
    assert (info.nfft, info.nbins, info.nz) == (1 << 24, 1 << 23, 193)
    w = oracle.whiten(oracle.spectrum(x, wl.nfft))
    assert np.abs(spec_to_complex(torch, d_spec) - w).max() <= 1e-2 * np.abs(w).max()
    bank = oracle.template_bank(wl.zmax, wl.zstep)
    nb, nz = info.nbins, info.nz
    rng = np.random.default_rng(5)
    rr = [rng.integers(0, nb, 20000)]; jj = [rng.integers(0, nz, 20000)]
    edge = np.concatenate([np.arange(0, 70), np.arange(nb - 70, nb),
                           np.array([t * 128 + d for t in (1, 148, 32768, 65535) for d in (-1, 0, 1)])])
    for j in (0, 96, 192):
        rr.append(edge); jj.append(np.full(edge.size, j))
    for s in wl.signals:
        r0, j0 = int(round(s.r_c)), int(round(s.z + wl.zmax))
        g_r, g_j = np.meshgrid(np.arange(r0 - 6, r0 + 7), np.arange(j0 - 3, j0 + 4))
        rr.append(g_r.ravel()); jj.append(g_j.ravel())
    rr = np.concatenate(rr).astype(np.int64); jj = np.concatenate(jj).astype(np.int32)
    Po = oracle.plane_points(w, bank, rr, jj)
    Pg = d_plane[torch.from_numpy(jj.astype(np.int64)).cuda(), torch.from_numpy(rr).cuda()].float().cpu().numpy()
    flat = int(torch.argmax(d_plane).item())
    jm, rm = flat // info.plane_pitch, flat % info.plane_pitch
    pmax = float(oracle.plane_points(w, bank, [rm], [jm])[0])
    assert abs(float(d_plane[jm, rm]) - pmax) <= TOL[precision] * pmax and pmax > 30
    assert np.abs(Pg - Po).max() <= TOL[precision] * pmax
    assert not torch.isnan(d_plane.sum()).item()
    gd = gpu_cand_dict(res.cands)
    assert res.count == len(gd) and 0 < res.count < 50000
    keys = sorted(gd)
    S, hmax = oracle.harmonic_sums_sampled(w, bank, wl.nharm, np.array([k[0] for k in keys]),
                                           np.array([k[1] for k in keys], dtype=np.int32))
    tol = TOL[precision] * pmax
    for i, (r, j, h) in enumerate(keys):
        so = S[i, h - 1]
        assert h <= hmax[i] and so > thr[h - 1] - membership_window(thr, h, tol, precision)
        assert abs(gd[(r, j, h)][0] - so) <= min(h * tol, REL_POW[precision] * so)


def test_ska_zero_padded_2p24_every_point(fdas, torch_, oracle):
    """The padded reading in full: all 1.6e9 plane points of the tensor-core path and of the FFT path against
    the oracle, whose plane is computed in chunks of 2^19 columns (0.8 GB each; the 13 GB plane is never
    resident), max-norm and the noise-floor statistic of reading A23."""
    torch = torch_
    wl = inputs.ska_padded()
    x = inputs.series_for(wl)
    w = oracle.whiten(oracle.spectrum(x, wl.nfft))
    bank = oracle.template_bank(wl.zmax, wl.zstep)
    W = local_amplitude(w)
    planes, stats = {}, {}
    for precision in ("bf16_tc", "bf16"):
        plan, d_spec, d_plane, res, thr = run_gpu(fdas, torch, wl, x, precision)
        planes[precision] = d_plane
        stats[precision] = PlaneStats(precision)
        plan.close()
        del d_spec
    nb = w.size
    pmax, step = 0.0, 1 << 19
    for r0 in range(0, nb, step):
        Po = oracle.plane(w, bank, r0, r0 + step)
        pmax = max(pmax, float(Po.max()))
        for precision, d_plane in planes.items():
            Pg = d_plane[:, r0:r0 + step].float().cpu().numpy().astype(np.float64)
            assert not np.isnan(Pg).any()
            stats[precision].add(Pg, Po, W[r0:r0 + step])
        del Po
    for precision, ps in stats.items():
        assert ps.npoints == 193 * nb
        ps.check(pmax)
        record_stats("ska_padded_full_" + precision, {**ps.summary(pmax), "pmax": pmax})
        print(precision, ps.summary(pmax))


# ------------------------------------- configs[3] / configs[4]: pipelined batch of DM trials
def _sequential(fdas, torch, plan, x, wl, thr, capacity=1 << 16):
    d_x = torch.from_numpy(x).cuda()
    d_spec, d_plane = plan.alloc_spec(), plan.alloc_plane()
    d_c, d_n = plan.alloc_cands(capacity)
    plan.prepare_spectrum(d_x, d_spec)
    plan.convolve_plane(d_spec, d_plane)
    plan.harmonic_sum_peaks(d_plane, wl.nharm, thr, wl.r_lo, d_c, d_n)
    torch.cuda.synchronize()
    return plan.read_cands(d_c, d_n), d_spec, d_plane


def test_batch_small_trial_counts_and_overflow(fdas, torch_):
    """fdas_search_batch == the three calls per trial, for 0, 1, 2 and 5 trials (slot reuse), device
    and host inputs, and with a capacity that overflows."""
    torch = torch_
    wl = inputs.tiny()
    plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, "fp32")
    thr = fdas.thresholds_from_sigma(wl.nharm, 4.5)        # lower threshold: tens of candidates per trial
    xs = [inputs.make_series(wl.n, 500 + i, wl.signals if i % 2 == 0 else ()) for i in range(5)]
    want = [gpu_cand_dict(_sequential(fdas, torch, plan, x, wl, thr)[0].cands) for x in xs]
    assert all(len(w) > 3 for w in want) and len(want[0]) != len(want[1])
    counts, _, st = plan.search_batch([], wl.nharm, thr, wl.r_lo, capacity=16)
    assert st == fdas.FDAS_OK and counts.size == 0
    for n in (1, 2, 5):
        for on_host in (False, True):
            series = xs[:n] if on_host else [torch.from_numpy(x).cuda() for x in xs[:n]]
            counts, cands, st = plan.search_batch(series, wl.nharm, thr, wl.r_lo, capacity=4096)
            assert st == fdas.FDAS_OK
            for t in range(n):
                assert counts[t] == len(want[t])
                assert gpu_cand_dict(cands[t, :counts[t]]) == want[t], (n, on_host, t)
    counts, cands, st = plan.search_batch(xs, wl.nharm, thr, wl.r_lo, capacity=2)
    assert st == fdas.FDAS_EOVERFLOW
    for t in range(5):
        assert counts[t] == len(want[t])
        assert set(gpu_cand_dict(cands[t, :2])) <= set(want[t])
    # the plan still serves single calls afterwards (its own block-max plane is rebuilt or rewritten)
    again = gpu_cand_dict(_sequential(fdas, torch, plan, xs[3], wl, thr)[0].cands)
    assert again == want[3]


def test_batch_failure_in_the_middle_leaves_the_plan_usable(fdas, torch_):
    """A host batch of five trials whose fourth prepare step fails (fault injection: a CUDA call the runtime
    refuses, while earlier trials are already in flight).  The call reports FDAS_ECUDA after draining its three
    streams, and the plan then serves a correct batch and correct single calls."""
    import ctypes as C
    torch = torch_
    wl = inputs.tiny()
    plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, "fp32")
    thr = fdas.thresholds_from_sigma(wl.nharm, 4.5)
    xs = [inputs.make_series(wl.n, 700 + i, wl.signals if i % 2 == 0 else ()) for i in range(5)]
    want = [gpu_cand_dict(_sequential(fdas, torch, plan, x, wl, thr)[0].cands) for x in xs]
    pinned = [torch.from_numpy(x).pin_memory() for x in xs]
    cap = 4096
    out = np.zeros((5, cap), dtype=fdas.CAND_DTYPE)
    thr_c = thr.ctypes.data_as(C.POINTER(C.c_float))
    plan.debug_fail_prepare(3)
    with pytest.raises(fdas.FdasError) as ei:
        plan.search_batch(pinned, wl.nharm, thr, wl.r_lo, capacity=cap)
    assert ei.value.status == fdas.FDAS_ECUDA and "injected" in str(ei.value)
    torch.cuda.synchronize()                        # nothing is left in flight, no sticky error
    counts, cands, st = plan.search_batch(pinned, wl.nharm, thr, wl.r_lo, capacity=cap)
    assert st == fdas.FDAS_OK
    for t in range(5):
        assert counts[t] == len(want[t]) and gpu_cand_dict(cands[t, :counts[t]]) == want[t], t
    assert gpu_cand_dict(_sequential(fdas, torch, plan, xs[2], wl, thr)[0].cands) == want[2]
    # fdas_search_host refuses a bad H before queueing anything
    cnt = C.c_int64(-1)
    assert fdas.lib().fdas_search_host(plan._h, pinned[0].data_ptr(), 0, thr_c, wl.r_lo, out.ctypes.data, cap,
                                       C.byref(cnt), None) == fdas.FDAS_EARG
    assert fdas.lib().fdas_search_host(plan._h, pinned[0].data_ptr(), 33, thr_c, wl.r_lo, out.ctypes.data, cap,
                                       C.byref(cnt), None) == fdas.FDAS_EARG
    assert fdas.lib().fdas_search_host(plan._h, pinned[0].data_ptr(), wl.nharm, thr_c, -1, out.ctypes.data, cap,
                                       C.byref(cnt), None) == fdas.FDAS_EARG
    res = plan.search_host(xs[1], wl.nharm, thr, wl.r_lo, capacity=cap)
    assert gpu_cand_dict(res.cands) == want[1]
    plan.close()


@pytest.mark.parametrize("precision", ["bf16_tc", "bf16"])
@pytest.mark.parametrize("half_res", [False, True])
def test_batch_ska_members_full_size(fdas, torch_, oracle, half_res, precision):
    """Members 5, 6, 7 of configs[3] (6 carries an injected accelerated signal), and the 128 us shape
    of configs[4], through the pipelined batch in the configuration bench.py times: equal to the
    per-trial calls, signal recovered at its (r, z), sampled oracle parity on the signal's trial."""
    torch = torch_
    members = [inputs.batched_member(i, half_res=half_res) for i in (5, 6, 7)]
    wl = members[1]
    assert len(wl.signals) == 1 and not members[0].signals
    plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, precision)
    assert plan.info.nfft == (1 << 22 if half_res else 1 << 23)
    thr = fdas.thresholds_from_sigma(wl.nharm, wl.nsigma)
    xs = [inputs.series_for(m) for m in members]
    pinned = [torch.from_numpy(x).pin_memory() for x in xs]
    counts, cands, st = plan.search_batch(pinned, wl.nharm, thr, wl.r_lo, capacity=1 << 14)
    assert st == fdas.FDAS_OK
    dev = [torch.from_numpy(x).cuda() for x in xs]
    counts_d, cands_d, st = plan.search_batch(dev, wl.nharm, thr, wl.r_lo, capacity=1 << 14)
    assert st == fdas.FDAS_OK and list(counts_d) == list(counts)
    seq = None
    for t in range(3):
        res, d_spec, d_plane = _sequential(fdas, torch, plan, xs[t], wl, thr)
        got = gpu_cand_dict(cands[t, :counts[t]])
        assert got == gpu_cand_dict(res.cands) == gpu_cand_dict(cands_d[t, :counts_d[t]])
        if t == 1:
            seq = (got, d_spec, d_plane)
        else:
            del d_spec, d_plane
    got, d_spec, d_plane = seq
    s = wl.signals[0]
    r0, j0 = int(round(s.r_c)), int(round(s.z + wl.zmax))
    assert any(abs(k[0] - r0) <= 1 and abs(k[1] - j0) <= 1 and k[2] == 1 for k in got), (r0, j0)
    # sampled oracle parity on the signal's trial
    w = oracle.whiten(oracle.spectrum(xs[1], wl.nfft))
    bank = oracle.template_bank(wl.zmax, wl.zstep)
    g_r, g_j = np.meshgrid(np.arange(r0 - 8, r0 + 9), np.arange(max(0, j0 - 4), min(plan.info.nz, j0 + 5)))
    rng = np.random.default_rng(7)
    rr = np.concatenate([g_r.ravel(), rng.integers(0, plan.info.nbins, 5000)]).astype(np.int64)
    jj = np.concatenate([g_j.ravel(), rng.integers(0, plan.info.nz, 5000)]).astype(np.int32)
    Po = oracle.plane_points(w, bank, rr, jj)
    Pg = d_plane[torch.from_numpy(jj.astype(np.int64)).cuda(), torch.from_numpy(rr).cuda()].float().cpu().numpy()
    pmax = float(Po.max())
    assert pmax > 50 and np.abs(Pg - Po).max() <= TOL["bf16"] * pmax
    keys = sorted(got)
    S, hmax = oracle.harmonic_sums_sampled(w, bank, wl.nharm, np.array([k[0] for k in keys]),
                                           np.array([k[1] for k in keys], dtype=np.int32))
    for i, (r, j, h) in enumerate(keys):
        so = S[i, h - 1]
        assert h <= hmax[i] and so > thr[h - 1] - membership_window(thr, h, TOL["bf16"] * pmax, "bf16")
        assert abs(got[(r, j, h)][0] - so) <= min(h * TOL["bf16"] * pmax, REL_POW["bf16"] * so)


# ------------------------------------------ configs[2] at full size: EVERY plane point and candidate
@pytest.fixture(scope="module")
def ska_oracle_full(oracle):
    """The oracle's whole SKA-like plane (193 x 2^22 doubles, 6.5 GB) and its candidate list."""
    wl = inputs.ska()
    x = inputs.series_for(wl)
    w = oracle.whiten(oracle.spectrum(x, wl.nfft))
    bank = oracle.template_bank(wl.zmax, wl.zstep)
    P = oracle.plane(w, bank)
    return wl, x, w, P, local_amplitude(w)


@pytest.mark.parametrize("precision", ["bf16_tc", "bf16", "fp32", "bf16_plane16", "bf16_tc_plane16"])
def test_ska_full_plane_parity(fdas, torch_, oracle, ska_oracle_full, precision):
    """The benched configuration, compared in full (not sampled): all 8.1e8 plane points against the
    oracle (max-norm and the noise-floor statistic), and the complete candidate list under the literal
    north_star window plus the strict 3 % window."""
    torch = torch_
    wl, x, w, P, W = ska_oracle_full
    plan, d_spec, d_plane, res, thr = run_gpu(fdas, torch, wl, x, precision)
    nz, nb = plan.info.nz, plan.info.nbins
    assert P.shape == (nz, nb)
    pmax = float(P.max())
    ps = PlaneStats(precision)
    for j0 in range(0, nz, 8):
        Pg = d_plane[j0:j0 + 8].float().cpu().numpy().astype(np.float64)
        assert not np.isnan(Pg).any()
        ps.add(Pg, P[j0:j0 + 8], W)
    ps.check(pmax)
    oc = oracle.candidates(P, wl.nharm, thr.astype(np.float64), wl.r_lo)
    s_at, margin = oracle_margin_fn(oracle, P, wl.nharm, wl.r_lo)
    gd = gpu_cand_dict(res.cands)
    assert res.count == len(gd)
    stats = compare_candidates(gd, oc.as_dict(), thr, TOL[precision] * pmax, REL_POW[precision], s_at, margin,
                               strict_rel=STRICT_REL[precision])
    if precision == "fp32":
        assert stats["only_gpu"] + stats["only_orc"] == 0, stats
    else:   # each one-sided triple is inside the window (compare_candidates); their NUMBER is bounded too
        assert stats["only_gpu"] + stats["only_orc"] <= max(2, 0.01 * stats["common"]), stats
    for s in wl.signals:                       # both injected pulsars: fundamental and second harmonic sum
        r0, j0 = int(round(s.r_c)), int(round(s.z + wl.zmax))
        assert (r0, j0, 1) in gd and (r0, j0, 2) in gd, s
    record_stats("ska_full_" + precision, {**ps.summary(pmax), **stats, "pmax": pmax})
    print(precision, ps.summary(pmax), stats)


# ---------------------------------------------------------------- K3: paths no other test reaches
def test_harmonic_maybe_list_overflow_falls_back_to_full_scan(fdas, torch_, oracle):
    """Thresholds so low that the prefilter flags more fundamentals than its list holds (2^22): pass B
    must fall back to scanning every fundamental.  The true count and a capped list are compared with
    the oracle."""
    torch = torch_
    plan = fdas.Plan(1 << 19, 64e-6, 16.0, 1.0, 2048, "fp32")       # 33 x 2^18 points
    nb, nz = plan.info.nbins, plan.info.nz
    rng = np.random.default_rng(41)
    P32 = rng.exponential(1.0, size=(nz, nb)).astype(np.float32)
    d_plane = torch.from_numpy(P32).cuda()
    H = 2
    thr = np.array([0.1, 0.25], dtype=np.float32)
    d_c, d_n = plan.alloc_cands(1 << 16)
    plan.harmonic_sum_peaks(d_plane, H, thr, 3, d_c, d_n)
    torch.cuda.synchronize()
    res = plan.read_cands(d_c, d_n)
    oc = oracle.candidates(P32.astype(np.float64), H, thr.astype(np.float64), 3, capacity=1 << 24)
    assert oc.count > (1 << 22) + (1 << 20)                        # far more than the list holds
    assert abs(res.count - oc.count) <= 8, (res.count, oc.count)   # fp32 vs double sums at the threshold
    # membership of the 65536 stored records in the oracle's ~1e7 triples, by sorted integer keys
    okey = (oc.r.astype(np.int64) * 64 + oc.j) * 64 + oc.h
    order = np.argsort(okey)
    okey, opow = okey[order], oc.power[order]
    c = res.cands
    assert len(c) == 1 << 16
    gkey = (c["r"].astype(np.int64) * 64 + c["zidx"]) * 64 + c["h"]
    assert np.unique(gkey).size == gkey.size
    pos = np.minimum(np.searchsorted(okey, gkey), okey.size - 1)
    hit = okey[pos] == gkey
    assert np.all(np.abs(c["power"][hit] - opow[pos[hit]]) <= 1e-5 * opow[pos[hit]])
    assert (~hit).sum() <= 8
    s_at, _ = oracle_margin_fn(oracle, P32.astype(np.float64), H, 3)
    for rec in c[~hit]:
        key = (int(rec["r"]), int(rec["zidx"]), int(rec["h"]))
        assert abs(s_at(*key) - thr[key[2] - 1]) <= 1e-5 * thr[key[2] - 1], key


def test_harmonic_every_coarse_block_fails_on_a_large_plane(fdas, torch_):
    """Every one of the 10^6 coarse blocks (64 fundamentals each) fails the coarse bound, every thread of the coarse
    level goes on to the block level, the maybe list overflows and pass B scans every fundamental.  H = 1, so the
    expected set is the definition itself: every P > T_1, r >= r_lo."""
    torch = torch_
    plan = fdas.Plan(1 << 21, 64e-6, 32.0, 1.0, 2048, "fp32")       # 65 x 2^20 points, 65 x 16384 coarse blocks
    nb, nz = plan.info.nbins, plan.info.nz
    assert nz * (nb // 64) > (1 << 20)
    rng = np.random.default_rng(43)
    P32 = rng.exponential(1.0, size=(nz, nb)).astype(np.float32)
    d_plane = torch.from_numpy(P32).cuda()
    thr = np.array([0.05], dtype=np.float32)
    r_lo = 5
    d_c, d_n = plan.alloc_cands(1 << 16)
    plan.harmonic_sum_peaks(d_plane, 1, thr, r_lo, d_c, d_n)
    torch.cuda.synchronize()
    res = plan.read_cands(d_c, d_n)
    assert res.count == int((P32[:, r_lo:] > thr[0]).sum())          # bit-exact: S_1 is the stored value
    c = res.cands
    assert len(c) == 1 << 16 and np.all(c["h"] == 1) and np.all(c["r"] >= r_lo)
    key = c["zidx"].astype(np.int64) * nb + c["r"]
    assert np.unique(key).size == key.size
    assert np.array_equal(c["power"], P32[c["zidx"], c["r"]]) and np.all(c["power"] > thr[0])
    # and the same call on a quiet plane with one line finds exactly that line through both levels
    d_plane.zero_()
    d_plane[40, 123457] = 3.0
    plan.harmonic_sum_peaks(d_plane, 1, thr, r_lo, d_c, d_n)
    res = plan.read_cands(d_c, d_n)
    assert res.count == 1 and (int(res.cands[0]["r"]), int(res.cands[0]["zidx"]), int(res.cands[0]["h"])) == (123457, 40, 1)


def test_harmonic_even_nz_half_integer_rows(fdas, torch_, oracle):
    """Reading A20 on the GPU: with an even number of templates (z = -7.5 .. 7.5) the odd harmonics
    of a row fall between two rows and round half away from zero, on both sides."""
    torch = torch_
    plan = fdas.Plan(1 << 14, 64e-6, 7.5, 1.0, 2048, "fp32")
    nb, nz = plan.info.nbins, plan.info.nz
    assert nz == 16
    rng = np.random.default_rng(43)
    P32 = rng.exponential(1.0, size=(nz, nb)).astype(np.float32)
    for j in range(nz):                       # a spike per row at harmonics of r = 500 + 7 j
        for k in (1, 2, 3):
            P32[j, k * (500 + 7 * j)] += 15.0
    d_plane = torch.from_numpy(P32).cuda()
    H = 8
    thr = fdas.thresholds_from_sigma(H, 3.0)
    d_c, d_n = plan.alloc_cands(1 << 18)
    plan.harmonic_sum_peaks(d_plane, H, thr, 10, d_c, d_n)
    torch.cuda.synchronize()
    res = plan.read_cands(d_c, d_n)
    P = P32.astype(np.float64)
    oc = oracle.candidates(P, H, thr.astype(np.float64), 10)
    s_at, margin = oracle_margin_fn(oracle, P, H, 10)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, 2e-6 * P.max(), None, s_at, margin,
                               strict_rel=1e-5)
    assert stats["only_gpu"] + stats["only_orc"] <= 2 and stats["common"] > 100, stats
    assert any(k[2] >= 3 for k in gpu_cand_dict(res.cands))        # sums that use a half-integer row


def test_plane_refilled_in_place_and_invalidate(fdas, torch_, oracle):
    """The block-max side plane is never trusted for a plane this plan did not write (it is rebuilt on
    every call), and fdas_plan_invalidate_plane covers a convolve-written plane modified in place."""
    torch = torch_
    plan = fdas.Plan(1 << 14, 64e-6, 16.0, 1.0, 2048, "fp32")
    nb, nz = plan.info.nbins, plan.info.nz
    H = 4
    thr = fdas.thresholds_from_sigma(H, 3.5)
    d_c, d_n = plan.alloc_cands(1 << 16)
    rng = np.random.default_rng(47)
    d_plane = torch.empty((nz, nb), dtype=torch.float32, device="cuda")
    for it in range(3):                                  # same tensor, new contents every time
        P32 = rng.exponential(1.0 + it, size=(nz, nb)).astype(np.float32)
        d_plane.copy_(torch.from_numpy(P32))
        plan.harmonic_sum_peaks(d_plane, H, thr, 8, d_c, d_n)
        torch.cuda.synchronize()
        got = set(gpu_cand_dict(plan.read_cands(d_c, d_n).cands))
        want = oracle.candidates(P32.astype(np.float64), H, thr.astype(np.float64), 8).triples()
        assert len(got ^ want) <= 2 and len(want) > 20 * (it + 1), (it, len(got), len(want))
    # a plane written by fdas_convolve_plane, then changed by the caller
    w = (rng.standard_normal(nb) + 1j * rng.standard_normal(nb)) / np.sqrt(2)
    d_spec = spec_from_complex(torch, w, "fp32")
    plan.convolve_plane(d_spec, d_plane)
    plan.harmonic_sum_peaks(d_plane, H, thr, 8, d_c, d_n)
    before = set(gpu_cand_dict(plan.read_cands(d_c, d_n).cands))
    d_plane[5, 4000] = 99.0
    d_plane[20, 7001] = 77.0
    plan.invalidate_plane()
    plan.harmonic_sum_peaks(d_plane, H, thr, 8, d_c, d_n)
    after = set(gpu_cand_dict(plan.read_cands(d_c, d_n).cands))
    assert (4000, 5, 1) in after and (7001, 20, 1) in after and before <= after
    want = oracle.candidates(d_plane.cpu().numpy().astype(np.float64), H, thr.astype(np.float64), 8).triples()
    assert len(after ^ want) <= 2


def test_two_streams_share_one_plan(fdas, torch_):
    """Calls of one plan issued on two streams without host synchronisation are ordered on the device
    (plan scratch is shared): both trials give what they give alone."""
    torch = torch_
    wl = inputs.tiny()
    plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, "fp32")
    thr = fdas.thresholds_from_sigma(wl.nharm, 4.5)
    xs = [inputs.make_series(wl.n, 700 + i, wl.signals if i == 0 else ()) for i in range(2)]
    want = [gpu_cand_dict(_sequential(fdas, torch, plan, x, wl, thr)[0].cands) for x in xs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    bufs = []
    for x in xs:
        d_c, d_n = plan.alloc_cands(1 << 14)
        bufs.append((torch.from_numpy(x).cuda(), plan.alloc_spec(), plan.alloc_plane(), d_c, d_n))
    torch.cuda.synchronize()
    for rep in range(4):
        for (d_x, d_spec, d_plane, d_c, d_n), st in zip(bufs, streams):
            plan.prepare_spectrum(d_x, d_spec, stream=st)
            plan.convolve_plane(d_spec, d_plane, stream=st)
            plan.harmonic_sum_peaks(d_plane, wl.nharm, thr, wl.r_lo, d_c, d_n, stream=st)
    torch.cuda.synchronize()
    for (d_x, d_spec, d_plane, d_c, d_n), w_ in zip(bufs, want):
        assert gpu_cand_dict(plan.read_cands(d_c, d_n).cands) == w_


# ----------------------------------------------------- other template banks
@pytest.mark.parametrize("precision", ALL_PREC)
@pytest.mark.parametrize("zmax,zstep", [(16.0, 0.5), (16.0, 2.0), (96.0, 0.5)])
def test_other_z_spacings_full_parity(fdas, torch_, oracle, precision, zmax, zstep):
    """Half-bin and coarse banks (zmax 16, zstep 0.5 -> 65 templates, zstep 2 -> 17; the paper's zmax 96
    at half-bin spacing -> 385 templates = 192 conjugate pairs, two K2-TC launches): the plane element by
    element against the oracle's bank of the same spacing, and the harmonic sums (whose rows are
    idx(k z_j) = (k z_j + zmax)/zstep) against the oracle's candidates on the GPU's plane."""
    torch = torch_
    n = 1 << 16
    plan = fdas.Plan(n, 64e-6, zmax, zstep, 2048, precision)
    nb, nz = plan.info.nbins, plan.info.nz
    assert nz == int(round(2 * zmax / zstep)) + 1
    rng = np.random.default_rng(int(10 * zstep))
    w = (rng.standard_normal(nb) + 1j * rng.standard_normal(nb)) / np.sqrt(2)
    for k, a in ((3000, 9.0), (6000, 9.0), (9000, 6.0), (12000, 6.0), (nb - 1, 8.0), (0, 8.0)):
        w[k] += a
    d_spec = spec_from_complex(torch, w, precision)
    d_plane = plan.alloc_plane(); d_plane.fill_(float("nan"))
    plan.convolve_plane(d_spec, d_plane)
    H = 8
    thr = fdas.thresholds_from_sigma(H, 3.5)
    d_c, d_n = plan.alloc_cands(1 << 17)
    plan.harmonic_sum_peaks(d_plane, H, thr, 16, d_c, d_n)
    torch.cuda.synchronize()
    Pg = d_plane.float().cpu().numpy().astype(np.float64)
    assert not np.isnan(Pg).any()
    bank = oracle.template_bank(zmax, zstep)
    assert bank.shape[0] == nz and np.abs(plan.templates_host() - bank).max() < 1e-12
    P = oracle.plane(w, bank)
    ps = PlaneStats(precision)
    ps.add(Pg, P, local_amplitude(w))
    ps.check(P.max())
    res = plan.read_cands(d_c, d_n)
    oc = oracle.candidates(Pg, H, thr.astype(np.float64), 16)
    s_at, margin = oracle_margin_fn(oracle, Pg, H, 16)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, 2e-6 * Pg.max(), None, s_at, margin,
                               strict_rel=1e-5)
    assert stats["only_gpu"] + stats["only_orc"] <= 2 and stats["common"] > 50, stats
    record_stats(f"zmax{zmax:g}_zstep{zstep}_{precision}", {**ps.summary(P.max()), **stats})


# ------------------------------------------- other segment lengths (seg_len 1024 / 4096)
FFT_PREC = ["fp32", "bf16", "bf16_plane16"]


@pytest.mark.parametrize("precision", FFT_PREC)
@pytest.mark.parametrize("zmax,seg_len", [(16.0, 1024), (96.0, 1024), (16.0, 4096), (96.0, 4096), (96.0, 2048)])
def test_other_segment_lengths_full_parity(fdas, torch_, oracle, precision, zmax, seg_len):
    """The FFT kernel at L = 1024 (16 x 8 x 8, 64 threads) and L = 4096 (16 x 16 x 16, 256 threads): plane
    element by element against the oracle with lines on and around the seams of THIS segmentation
    (V = L - 2h), a ragged last segment, the side plane through the harmonic sums on the GPU's own plane."""
    torch = torch_
    n = 1 << 16
    plan = fdas.Plan(n, 64e-6, zmax, 1.0, seg_len, precision)
    nb, nz, V = plan.info.nbins, plan.info.nz, plan.info.valid
    assert plan.info.seg_len == seg_len and V == seg_len - 2 * plan.info.halfwidth
    assert plan.info.nseg == -(-nb // V) and nb % V != 0
    rng = np.random.default_rng(seg_len + int(zmax))
    w = (rng.standard_normal(nb) + 1j * rng.standard_normal(nb)) / np.sqrt(2)
    for k in (0, 1, V - 1, V, V + 1, 2 * V, 5 * V - 3, nb - 1):
        w[k] += 12.0
    d_spec = spec_from_complex(torch, w, precision)
    d_plane = plan.alloc_plane(); d_plane.fill_(float("nan"))
    plan.convolve_plane(d_spec, d_plane)
    H = 8
    thr = fdas.thresholds_from_sigma(H, 3.5)
    d_c, d_n = plan.alloc_cands(1 << 17)
    plan.harmonic_sum_peaks(d_plane, H, thr, 16, d_c, d_n)
    torch.cuda.synchronize()
    Pg = d_plane.float().cpu().numpy().astype(np.float64)
    assert not np.isnan(Pg).any()
    bank = oracle.template_bank(zmax, 1.0)
    P = oracle.plane(w, bank)
    ps = PlaneStats(precision)
    ps.add(Pg, P, local_amplitude(w))
    ps.check(P.max())
    # block-max side plane of this segmentation: bit-exact upper bounds of the stored plane
    ptr, pitch = plan.debug_maxplane()
    M = _device_view(torch, ptr, nz * pitch).view(nz, pitch).clone()
    ref = d_plane.float().view(nz, pitch, 8).amax(dim=2)
    assert torch.equal(M, max_codes(torch, ref))
    res = plan.read_cands(d_c, d_n)
    oc = oracle.candidates(Pg, H, thr.astype(np.float64), 16)
    s_at, margin = oracle_margin_fn(oracle, Pg, H, 16)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, 2e-6 * Pg.max(), None, s_at, margin,
                               strict_rel=1e-5)
    assert stats["only_gpu"] + stats["only_orc"] <= 2 and stats["common"] > 50, stats
    record_stats(f"seg{seg_len}_zmax{zmax:g}_{precision}", {**ps.summary(P.max()), **stats})


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
@pytest.mark.parametrize("seg_len", [1024, 4096])
def test_medium_other_segment_lengths(fdas, torch_, oracle, medium_oracle, precision, seg_len):
    """configs[1] end to end (547 -> 1171 / 265 segments) at the other two segment lengths: every plane
    point and the candidate list against the oracle."""
    import dataclasses
    torch = torch_
    wl0, x, orc = medium_oracle
    wl = dataclasses.replace(wl0, seg_len=seg_len)
    plan, d_spec, d_plane, res, thr = run_gpu(fdas, torch, wl, x, precision)
    assert plan.info.seg_len == seg_len and plan.info.nseg == -(-plan.info.nbins // (seg_len - 128))
    pmax = orc.P.max()
    ps = PlaneStats(precision)
    W = local_amplitude(orc.w)
    for j0 in range(0, plan.info.nz, 16):
        Pg = d_plane[j0:j0 + 16].float().cpu().numpy().astype(np.float64)
        assert not np.isnan(Pg).any()
        ps.add(Pg, orc.P[j0:j0 + 16], W)
    ps.check(pmax)
    oc = oracle.candidates(orc.P, wl.nharm, thr.astype(np.float64), wl.r_lo)
    s_at, margin = oracle_margin_fn(oracle, orc.P, wl.nharm, wl.r_lo)
    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, TOL[precision] * pmax, REL_POW[precision],
                               s_at, margin, strict_rel=STRICT_REL[precision])
    if precision == "fp32":
        assert stats["only_gpu"] + stats["only_orc"] == 0, stats
    else:
        assert stats["only_gpu"] + stats["only_orc"] <= 0.01 * stats["common"], stats
    record_stats(f"medium_seg{seg_len}_{precision}", {**ps.summary(pmax), **stats})


# ------------------------------------- neighbour-maximised harmonic sums
def nbr_thresholds(thr):
    """A caller's choice of thresholds for S': the plain T_h raised by the growth of the noise mean,
    sum_k (H_{2 floor(k/2) + 1} - 1), H_m = mean of the maximum of m unit exponentials."""
    out, shift = [], 0.0
    for k, t in enumerate(thr, start=1):
        m = 2 * (k // 2) + 1
        shift += sum(1.0 / i for i in range(1, m + 1)) - 1.0
        out.append(t + shift)
    return np.array(out, dtype=np.float32)


@pytest.mark.parametrize("precision,H", [("fp32", 16), ("bf16_plane16", 16), ("fp32", 32), ("fp32", 3)])
def test_neighbour_max_mode_alone_on_hand_made_planes(fdas, torch_, oracle, precision, H):
    """K3 in FDAS_HSUM_NEIGHBOUR_MAX mode on a hand-made plane against the oracle's O5n candidates:
    the dilated side plane (1 block either side for H <= 17, 2 for H = 32) must not lose a candidate,
    the windowed maxima, the clipping at the ends of the plane and the flags must agree."""
    torch = torch_
    plan = fdas.Plan(1 << 14, 64e-6, 16.0, 1.0, 2048, precision)
    nb, nz = plan.info.nbins, plan.info.nz
    rng = np.random.default_rng(61 + H)
    P32 = rng.exponential(1.0, size=(nz, nb)).astype(np.float32)
    for k in (1, 2, 3, 5):                       # spikes next to the harmonic cut-offs and the plane's ends
        P32[:, min(nb - 1, (nb - 1) // k + 1)] += 8.0
    P32[:, 0] += 20.0; P32[:, nb - 1] += 20.0
    d_plane = torch.from_numpy(P32).cuda()
    if precision == "bf16_plane16":
        d_plane = d_plane.to(torch.bfloat16)
    P = d_plane.float().cpu().numpy().astype(np.float64)
    thr = nbr_thresholds(fdas.thresholds_from_sigma(H, 2.5))
    r_lo = 3
    d_c, d_n = plan.alloc_cands(1 << 19)
    plan.set_harmonic_mode("neighbour_max")
    plan.harmonic_sum_peaks(d_plane, H, thr, r_lo, d_c, d_n)
    torch.cuda.synchronize()
    res = plan.read_cands(d_c, d_n)
    oc = oracle.candidates(P, H, thr.astype(np.float64), r_lo, nbr=True)
    assert oc.count > 300 and res.count == len(res.cands)

    def s_at(r, j, h):
        if j < 0 or j >= nz or r < r_lo or r >= nb:
            return None
        S = oracle.harmonic_sums_nbr_at(P, h, r, j)
        return float(S[h - 1]) if len(S) >= h else None

    def margin(r, j, h):
        vals = [s_at(r + dr, j + dj, h) for dj in (-1, 0, 1) for dr in (-1, 0, 1) if (dj, dr) != (0, 0)]
        vals = [abs(s_at(r, j, h) - v) for v in vals if v is not None]
        return min(vals) if vals else None

    stats = compare_candidates(gpu_cand_dict(res.cands), oc.as_dict(), thr, 2e-6 * P.max(), None, s_at, margin,
                               strict_rel=1e-5)
    assert stats["only_gpu"] + stats["only_orc"] <= 3 and stats["flags_checked"] > 50, stats
    assert any(k[2] == H for k in gpu_cand_dict(res.cands)) or H == 32
    # back to the plain sums on the same plan: the plain candidate set again
    plan.set_harmonic_mode("plain")
    thr_p = fdas.thresholds_from_sigma(H, 3.0)
    plan.harmonic_sum_peaks(d_plane, H, thr_p, r_lo, d_c, d_n)
    got = set(gpu_cand_dict(plan.read_cands(d_c, d_n).cands))
    want = oracle.candidates(P, H, thr_p.astype(np.float64), r_lo).triples()
    assert len(got ^ want) <= 3


@pytest.mark.parametrize("precision", ["fp32", "bf16_tc"])
def test_neighbour_max_mode_recovers_an_off_bin_pulsar(fdas, torch_, oracle, precision):
    """End to end on a pulsar at r_c = 40000.37 with 8 equal harmonics: candidate-set parity of the
    neighbour-maximised mode against the oracle (O1..O4, O5n), and the recovered S_8 of both modes."""
    torch = torch_
    wl = inputs.offbin()
    x = inputs.series_for(wl)
    orc = oracle.run(x, wl.nfft, wl.zmax, wl.zstep, wl.nharm, wl.nsigma, wl.r_lo, want_candidates=False)
    plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, precision)
    d_spec, d_plane = plan.alloc_spec(), plan.alloc_plane()
    d_c, d_n = plan.alloc_cands(1 << 16)
    thr_p = fdas.thresholds_from_sigma(wl.nharm, wl.nsigma)
    thr_n = nbr_thresholds(thr_p)
    plan.prepare_spectrum(torch.from_numpy(x).cuda(), d_spec)
    plan.convolve_plane(d_spec, d_plane)
    plan.harmonic_sum_peaks(d_plane, wl.nharm, thr_p, wl.r_lo, d_c, d_n)
    plain = gpu_cand_dict(plan.read_cands(d_c, d_n).cands)
    plan.set_harmonic_mode("neighbour_max")
    plan.harmonic_sum_peaks(d_plane, wl.nharm, thr_n, wl.r_lo, d_c, d_n)
    nbr = gpu_cand_dict(plan.read_cands(d_c, d_n).cands)
    s = wl.signals[0]
    r0, j0 = int(round(s.r_c)), int(round(s.z + wl.zmax))
    S_plain = oracle.harmonic_sums_at(orc.P, wl.nharm, r0, j0)
    S_nbr = oracle.harmonic_sums_nbr_at(orc.P, wl.nharm, r0, j0)
    assert len(S_nbr) == 8 and S_nbr[7] > 1.5 * S_plain[7] and S_nbr[7] > thr_n[7] + 20
    assert (r0, j0, 8) in nbr and (r0, j0, 8) not in plain            # the deep sum is found by S' only
    tol = TOL[precision] * orc.P.max()
    oc = oracle.candidates(orc.P, wl.nharm, thr_n.astype(np.float64), wl.r_lo, nbr=True)

    nz_, nb_ = orc.P.shape

    def s_at(r, j, h):
        if j < 0 or j >= nz_ or r < wl.r_lo or r >= nb_:
            return None
        S = oracle.harmonic_sums_nbr_at(orc.P, h, r, j)
        return float(S[h - 1]) if len(S) >= h else None

    def margin(r, j, h):     # the local-maximum flag of this mode is compared too (where the oracle's margin allows)
        vals = [s_at(r + dr, j + dj, h) for dj in (-1, 0, 1) for dr in (-1, 0, 1) if (dj, dr) != (0, 0)]
        vals = [abs(s_at(r, j, h) - v) for v in vals if v is not None]
        return min(vals) if vals else None

    stats = compare_candidates(nbr, oc.as_dict(), thr_n, tol, REL_POW[precision], s_at, margin,
                               strict_rel=STRICT_REL[precision])
    assert stats["common"] >= 8 and stats["flags_checked"] >= 4, stats
    if precision == "fp32":
        assert stats["only_gpu"] + stats["only_orc"] == 0, stats
    record_stats("offbin_nbr_" + precision, {**stats, "S8_plain": float(S_plain[7]), "S8_nbr": float(S_nbr[7]),
                                             "gpu_S8_nbr": nbr[(r0, j0, 8)][0], "T8_plain": float(thr_p[7]),
                                             "T8_nbr": float(thr_n[7])})

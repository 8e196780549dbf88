"""Seeded synthetic inputs shaped like the paper's SKA-like FDAS workload.

This module is the ONE piece shared by the CPU oracle tests and the CUDA path: it only
synthesises float32 time series (noise + injected signals) and names the five workload
configurations of BASELINE.json.  It holds none of the method's arithmetic (no FFT-based
filtering, no templates, no whitening, no harmonic sums) and imports neither ``oracle`` nor
the CUDA binding.

Workload shape: PAPER.md:35 (§3) "600 second T_obs, 64 us resolution, 5925 DM trials with 3050 at
full time resolution, 193 acceleration trials".  Signal convention (reading A4):
``x[n] = a*cos(2*pi*(r_c*v + z*v^2/2) + phi)``, ``v = n/nfft - 1/2`` so that ``r_c`` is the
mid-observation frequency in Fourier bins and ``z`` the drift in bins over the nfft samples used.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

TSAMP_FULL = 64e-6
TSAMP_HALF = 128e-6     # BASELINE.json configs[4]
N_SKA_FULL = 9_375_000  # 600 s / 64 us
N_SKA_HALF = 4_687_500  # 600 s / 128 us


@dataclass(frozen=True)
class Signal:
    """One injected constant-fdot sinusoid (harmonic k has frequency k*r_c and drift k*z)."""
    r_c: float
    z: float
    amp: float
    phase: float = 0.0
    nharm: int = 1
    harm_decay: float = 0.8


@dataclass(frozen=True)
class Workload:
    name: str
    n: int                 # samples in the time series handed to fdas_plan
    tsamp: float
    zmax: float
    zstep: float
    seg_len: int
    nharm: int             # H of the harmonic sum
    nsigma: float
    r_lo: int
    precisions: Tuple[str, ...]
    seed: int
    signals: Tuple[Signal, ...] = field(default_factory=tuple)
    red_knee: float = 0.0  # 0 = white noise only

    @property
    def nfft(self) -> int:
        """Largest power of two <= n (reading A1)."""
        return 1 << (int(self.n).bit_length() - 1)

    @property
    def nz(self) -> int:
        return int(round(2 * self.zmax / self.zstep)) + 1


def largest_pow2_le(n: int) -> int:
    return 1 << (int(n).bit_length() - 1)


def chirp(n: int, nfft: int, sig: Signal) -> np.ndarray:
    """float64 samples of one injected signal over n samples (v referenced to nfft)."""
    v = np.arange(n, dtype=np.float64) / float(nfft) - 0.5
    base = 2.0 * np.pi * (sig.r_c * v + 0.5 * sig.z * v * v)
    out = np.zeros(n, dtype=np.float64)
    for k in range(1, sig.nharm + 1):
        a_k = sig.amp * sig.harm_decay ** (k - 1)
        ph_k = sig.phase if k == 1 else sig.phase + 0.7 * (k - 1)
        out += a_k * np.cos(k * base + ph_k)
    return out


def red_noise(n: int, knee: float, rng: np.random.Generator) -> np.ndarray:
    """Unit-white-level 1/f component: PSD_red(k) = PSD_white * (knee / k), random phases.

    Built in the Fourier domain over the n samples and brought back with an inverse real FFT
    (input synthesis only; not part of the method).
    """
    nb = n // 2 + 1
    k = np.arange(nb, dtype=np.float64)
    amp = np.zeros(nb)
    amp[1:] = np.sqrt(knee / k[1:])
    # white noise of unit variance has E|X_k|^2 = n; a random-phase line of that power
    spec = amp * np.sqrt(n / 2.0) * (rng.standard_normal(nb) + 1j * rng.standard_normal(nb))
    spec[0] = 0.0
    return np.fft.irfft(spec, n=n)


def make_series(n: int, seed: int, signals=(), red_knee: float = 0.0, nfft_ref: int = 0) -> np.ndarray:
    """float32 time series: N(0,1) noise (+ optional red noise) + injected signals.  The signals'
    (r_c, z) refer to a transform of nfft_ref samples (default: the largest power of two <= n)."""
    rng = np.random.default_rng(seed)
    nfft = nfft_ref if nfft_ref > 0 else largest_pow2_le(n)
    x = rng.standard_normal(n)
    if red_knee > 0.0:
        x = x + red_noise(n, red_knee, rng)
    for s in signals:
        x = x + chirp(n, nfft, s)
    return np.ascontiguousarray(x, dtype=np.float32)


def _medium_signals(seed: int) -> Tuple[Signal, ...]:
    rng = np.random.default_rng(seed + 1000)
    sigs = []
    for _ in range(4):
        amp = float(rng.uniform(0.02, 0.1))
        z0 = float(rng.uniform(-80.0, 80.0))
        r_c = float(rng.uniform(5.0e3, 1.0e6))
        ph = float(rng.uniform(0.0, 2.0 * np.pi))
        sigs.append(Signal(r_c=r_c, z=z0, amp=amp, phase=ph))
    return tuple(sigs)


def tiny() -> Workload:
    """BASELINE.json configs[0]."""
    return Workload("tiny", 1 << 17, TSAMP_FULL, 16.0, 1.0, 2048, 16, 6.0, 64, ("fp32",), 1,
                    (Signal(r_c=20000.3, z=7.5, amp=0.05),))


def medium() -> Workload:
    """BASELINE.json configs[1]."""
    return Workload("medium", 1 << 21, TSAMP_FULL, 96.0, 1.0, 2048, 8, 6.0, 64,
                    ("fp32", "bf16"), 2, _medium_signals(2))


def offbin() -> Workload:
    """A pulsar whose fundamental lies BETWEEN two Fourier bins (r_c = integer + 0.37, 8 harmonics of equal
    amplitude, z = 2): harmonic k sits at k r_c, up to k/2 bins from k round(r_c), so the plain harmonic
    sum loses it and the neighbour-maximised sum (reading A24) does not.  Medium-sized."""
    return Workload("offbin", 1 << 21, TSAMP_FULL, 96.0, 1.0, 2048, 8, 6.0, 64, ("fp32", "bf16"), 7,
                    (Signal(r_c=40000.37, z=2.0, amp=0.006, phase=0.7, nharm=8, harm_decay=1.0),))


def ska(seed: int = 3, half_res: bool = False, signals=None) -> Workload:
    """BASELINE.json configs[2] (and the 128 us series of configs[4] with half_res=True)."""
    n = N_SKA_HALF if half_res else N_SKA_FULL
    if signals is None:
        signals = (Signal(r_c=123456.01, z=40.0, amp=0.012, phase=0.3, nharm=5),
                   Signal(r_c=654321.01, z=-40.0, amp=0.012, phase=1.1, nharm=5))
        if half_res:
            signals = tuple(Signal(s.r_c / 2 + 0.005, s.z, s.amp * 1.4142, s.phase, s.nharm)
                            for s in signals)
    return Workload("ska_half" if half_res else "ska", n, TSAMP_HALF if half_res else TSAMP_FULL,
                    96.0, 1.0, 2048, 16, 6.0, 64, ("bf16",), seed, tuple(signals), red_knee=600.0)


N_SKA_PADDED = 1 << 24


def ska_padded(seed: int = 3) -> Workload:
    """The secondary reading A1-B of configs[2] ("zero-padded ... for the real FFT"): all 9,375,000
    samples, mean-subtracted and zero-padded to 2^24 by the caller -- for the library it is simply a
    series of N = 2^24 samples (nfft 2^24, Nb 2^23, a 6.5 GB fp32 plane).  (r_c, z) of the injected
    signals are in bins of the padded transform."""
    signals = (Signal(r_c=246912.02, z=40.0, amp=0.012, phase=0.3, nharm=5),
               Signal(r_c=1308642.02, z=-40.0, amp=0.012, phase=1.1, nharm=5))
    return Workload("ska_padded", N_SKA_PADDED, TSAMP_FULL, 96.0, 1.0, 2048, 16, 6.0, 64, ("bf16",), seed,
                    signals, red_knee=600.0)


BATCH_SIGNAL_SERIES = (6, 17, 23, 38, 49, 60)   # ~10 % of 64 carry one injected signal


def batched_member(i: int, half_res: bool = False) -> Workload:
    """Series i (0..63) of BASELINE.json configs[3]: seeds 100..163."""
    seed = 100 + i
    sigs: Tuple[Signal, ...] = ()
    if i in BATCH_SIGNAL_SERIES:
        rng = np.random.default_rng(seed + 5000)
        sigs = (Signal(r_c=float(rng.integers(20000, 2_000_000)) + 0.01,
                       z=float(rng.uniform(-90.0, 90.0)), amp=0.01,
                       phase=float(rng.uniform(0, 2 * np.pi))),)
    return ska(seed=seed, half_res=half_res, signals=sigs)


SURVEY_TRIALS_FULL = 3050
SURVEY_TRIALS_HALF = 2875   # BASELINE.json configs[4]


def series_for(w: Workload) -> np.ndarray:
    if w.name == "ska_padded":
        x = make_series(N_SKA_FULL, w.seed, w.signals, w.red_knee, nfft_ref=w.n).astype(np.float64)
        out = np.zeros(w.n, dtype=np.float32)
        out[:N_SKA_FULL] = (x - x.mean()).astype(np.float32)
        return out
    return make_series(w.n, w.seed, w.signals, w.red_knee)


def shard_trials(n_trials: int, rank: int, world: int) -> List[int]:
    """DM trials are independent: rank r takes trials r, r+world, ... (no collective)."""
    return list(range(rank, n_trials, world))

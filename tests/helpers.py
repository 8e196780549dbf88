"""Comparison rules shared by the parity tests (readings A11, A14, A23)."""
from __future__ import annotations

import numpy as np

# BASELINE.json north_star: plane tolerance as a fraction of the plane maximum, candidate powers within
# 3 % on the bf16 paths.
TOL = {"fp32": 1e-4, "bf16": 2e-2, "bf16_plane16": 2e-2, "bf16_tc": 2e-2, "bf16_tc_plane16": 2e-2}
REL_POW = {"fp32": None, "bf16": 0.03, "bf16_plane16": 0.03, "bf16_tc": 0.03, "bf16_tc_plane16": 0.03}
# Strict window for candidate-set differences (reading A14): a triple present on one side only must
# have its oracle sum within this FRACTION of its threshold (besides north_star's absolute window).
STRICT_REL = {"fp32": 1e-5, "bf16": 0.03, "bf16_plane16": 0.03, "bf16_tc": 0.03, "bf16_tc_plane16": 0.03}
# Noise-floor statistic (reading A23): |dy| <= C_AMP * W(r), W = largest |w| within +-NOISE_WINDOW
# bins, i.e. |dP| <= 2 sqrt(P) E + E^2 (+ the rounding of a bf16-stored plane), E = C_AMP W.
C_AMP = {"fp32": 5e-6, "bf16": 1e-2, "bf16_plane16": 1e-2, "bf16_tc": 1e-2, "bf16_tc_plane16": 1e-2}
NOISE_WINDOW = 2048


def membership_window(thr, h, tol_abs, precision):
    """How far from its threshold the oracle sum of a one-sided candidate may lie (reading A14):
    north_star's absolute tolerance AND the strict relative window."""
    return min(tol_abs, STRICT_REL[precision] * float(thr[h - 1]))


def gpu_cand_dict(cands):
    """structured CAND_DTYPE array -> {(r, j, h): (power, flag)}; a triple listed twice is an error
    (the list is a set: fdas.h, "identical to evaluating every fundamental")."""
    out = {(int(c["r"]), int(c["zidx"]), int(c["h"])): (float(c["power"]), int(c["flags"]) & 1)
           for c in cands}
    assert len(out) == len(cands), f"{len(cands) - len(out)} duplicated candidate records"
    return out


def local_amplitude(w, window=NOISE_WINDOW):
    """W(r) = max |w[r']| over |r' - r| <= window (the scale a point's rounding error follows: the
    products of a matched filter, and of an overlap-save segment, involve only nearby bins)."""
    from scipy.ndimage import maximum_filter1d
    return maximum_filter1d(np.abs(w), size=2 * window + 1, mode="constant", cval=0.0)


class PlaneStats:
    """Accumulates the plane statistics over row/column chunks:
    worst |dP| (for north_star's max-norm), the noise-floor ratio of reading A23 over every point, and
    the plain figure |dP| / (0.03 P + 1e-3) over points with oracle P < 30 (reported)."""

    def __init__(self, precision):
        self.precision = precision
        self.worst_abs = 0.0
        self.worst_noise_ratio = 0.0
        self.worst_plain_ratio = 0.0
        self.npoints = 0

    def add(self, Pg, Po, W):
        """Pg, Po: (rows, cols) GPU / oracle powers; W: (cols,) local amplitude of those columns."""
        D = np.abs(Pg - Po)
        self.worst_abs = max(self.worst_abs, float(D.max()))
        E = C_AMP[self.precision] * W[None, :]
        bound = 2.0 * np.sqrt(Po) * E + E * E
        if self.precision.endswith("plane16"):
            bound = bound + 2.0 ** -8 * Po
        bound = bound + 1e-12
        self.worst_noise_ratio = max(self.worst_noise_ratio, float((D / bound).max()))
        lo = Po < 30.0
        if lo.any():
            self.worst_plain_ratio = max(self.worst_plain_ratio, float((D[lo] / (0.03 * Po[lo] + 1e-3)).max()))
        self.npoints += D.size

    def check(self, pmax):
        assert self.worst_abs <= TOL[self.precision] * pmax, (self.precision, self.worst_abs / pmax)
        assert self.worst_noise_ratio <= 1.0, (self.precision, "noise-floor ratio", self.worst_noise_ratio)

    def summary(self, pmax):
        return dict(precision=self.precision, points=self.npoints, worst_over_max=self.worst_abs / pmax,
                    noise_floor_ratio=self.worst_noise_ratio, plain_ratio_P_lt_30=self.worst_plain_ratio)


def compare_candidates(gpu: dict, orc: dict, thr, tol_abs, rel_pow, sum_lookup, neighbour_margin=None,
                       strict_rel=0.03, max_outside_strict=0):
    """Candidate-list rule of BASELINE.json north_star / reading A14.

    gpu, orc      {(r, j, h): (power, flag)}
    thr           thresholds T_1..T_H (the float32 values handed to the GPU)
    tol_abs       north_star's tolerance (1e-4 or 2e-2 times the plane maximum): a triple found on one
                  side only must have |S_h - T_h| <= tol_abs, S_h the ORACLE's sum (literal reading)
    strict_rel    ... and |S_h - T_h| <= strict_rel * T_h as well (the stricter window; the number of
                  triples outside it may not exceed max_outside_strict)
    rel_pow       relative bound on the powers of common candidates (None: absolute bound only);
                  a sum of h plane points may be off by h * tol_abs
    sum_lookup    f(r, j, h) -> oracle S_h (float) or None if undefined; used for GPU-only triples
    neighbour_margin  f(r, j, h) -> min |S_h - neighbour S_h| in the oracle, for the flag rule
    Returns a dict of statistics; raises AssertionError on a violation.
    """
    only_gpu = set(gpu) - set(orc)
    only_orc = set(orc) - set(gpu)
    outside_strict, worst_window = 0, 0.0

    def excused(key, p):
        nonlocal outside_strict, worst_window
        t = float(thr[key[2] - 1])
        assert abs(p - t) <= tol_abs, f"one-sided candidate {key}: oracle power {p}, threshold {t}"
        worst_window = max(worst_window, abs(p - t) / t)
        if abs(p - t) > strict_rel * t:
            outside_strict += 1

    for key in only_orc:
        excused(key, orc[key][0])
    for key in only_gpu:
        p = sum_lookup(*key)
        assert p is not None, f"GPU candidate {key} is not defined in the oracle"
        excused(key, p)
    assert outside_strict <= max_outside_strict, \
        f"{outside_strict} one-sided candidates further than {strict_rel:.1e} x T_h from their threshold"
    worst_abs, worst_rel, flags_checked, flag_mismatch = 0.0, 0.0, 0, 0
    for key in set(gpu) & set(orc):
        pg, fg = gpu[key]
        po, fo = orc[key]
        h = key[2]
        worst_abs = max(worst_abs, abs(pg - po))
        worst_rel = max(worst_rel, abs(pg - po) / po)
        assert abs(pg - po) <= h * tol_abs, f"{key}: gpu {pg} oracle {po}"
        if rel_pow is not None:
            assert abs(pg - po) <= rel_pow * po, f"{key}: gpu {pg} oracle {po} (> {rel_pow:.0%})"
        if neighbour_margin is not None:
            m = neighbour_margin(*key)
            # non-fragile: the margin to every neighbour exceeds what the two sums may differ by
            if m is not None and m > 2 * min(h * tol_abs, max(strict_rel, 1e-5) * po):
                flags_checked += 1
                if fg != fo:
                    flag_mismatch += 1
    assert flag_mismatch == 0, f"{flag_mismatch} non-fragile local-max flags differ"
    return dict(common=len(set(gpu) & set(orc)), only_gpu=len(only_gpu), only_orc=len(only_orc),
                outside_strict=outside_strict, worst_window=worst_window,
                worst_abs=worst_abs, worst_rel=worst_rel, flags_checked=flags_checked)


def oracle_margin_fn(oracle, P, H, r_lo):
    """min |S_h(r,j) - S_h(neighbour)| over the defined 8 neighbours, from a full oracle plane."""
    nz, nb = P.shape

    def s_at(r, j, h):
        if j < 0 or j >= nz or r < r_lo or r >= nb:
            return None
        S = oracle.harmonic_sums_at(P, h, r, j)
        return float(S[h - 1]) if len(S) >= h else None

    def margin(r, j, h):
        s0 = s_at(r, j, h)
        best = None
        for dj in (-1, 0, 1):
            for dr in (-1, 0, 1):
                if dj == 0 and dr == 0:
                    continue
                v = s_at(r + dr, j + dj, h)
                if v is None:
                    continue
                d = abs(s0 - v)
                best = d if best is None else min(best, d)
        return best

    return s_at, margin


def record_stats(name, stats):
    """Append one line of measured statistics to the file the environment variable FDAS_PARITY_STATS names
    (nothing is written without it: a plain test run has no side effect).  `python tests/helpers.py FILE`
    turns such a file into the markdown table kept under profiles/.  Best effort, never fails a test."""
    import json
    import os
    path = os.environ.get("FDAS_PARITY_STATS")
    if not path:
        return
    try:
        os.makedirs(os.path.dirname(os.path.abspath(path)), exist_ok=True)
        with open(path, "a") as f:
            f.write(json.dumps({"test": name, **stats}) + "\n")
    except OSError:
        pass


def stats_table(lines):
    """Markdown table of the records record_stats wrote (the last record of each test wins)."""
    import json
    seen = {}
    for line in lines:
        if line.strip():
            r = json.loads(line)
            seen[r["test"]] = r

    def f(r, k, fmt):
        return fmt % r[k] if k in r else ""

    out = ["| test | plane points | worst abs err / max | noise-floor ratio (A23) | plain ratio, P<30 | common | only GPU | "
           "only oracle | outside strict window | widest window / T_h | worst rel power | flags checked |",
           "|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for k, r in seen.items():
        out.append(" ".join(str(c) for c in (
            "|", k, "|", r.get("points", ""), "|", f(r, "worst_over_max", "%.2e"), "|", f(r, "noise_floor_ratio", "%.3f"),
            "|", f(r, "plain_ratio_P_lt_30", "%.3g"), "|", r.get("common", ""), "|", r.get("only_gpu", ""), "|",
            r.get("only_orc", ""), "|", r.get("outside_strict", ""), "|", f(r, "worst_window", "%.2e"), "|",
            f(r, "worst_rel", "%.2e"), "|", r.get("flags_checked", ""), "|")))
    return "\n".join(out)


if __name__ == "__main__":
    import sys
    print(stats_table(open(sys.argv[1])))

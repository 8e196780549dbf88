"""Comparison rules shared by the parity tests (readings A11, A14)."""
from __future__ import annotations

import numpy as np


def gpu_cand_dict(cands):
    """structured CAND_DTYPE array -> {(r, j, h): (power, flag)}"""
    return {(int(c["r"]), int(c["zidx"]), int(c["h"])): (float(c["power"]), int(c["flags"]) & 1)
            for c in cands}


def compare_candidates(gpu: dict, orc: dict, thr, tol_abs, rel_pow, sum_lookup, neighbour_margin=None):
    """Candidate-list rule of BASELINE.json north_star / reading A14.

    gpu, orc      {(r, j, h): (power, flag)}
    thr           thresholds T_1..T_H (the float32 values handed to the GPU)
    tol_abs       plane tolerance (1e-4 or 2e-2 times the plane maximum); a sum of h points may be
                  off by h * tol_abs
    rel_pow       relative bound on candidate powers (None: absolute bound only)
    sum_lookup    f(r, j, h) -> oracle S_h (float) or None if undefined; used for GPU-only triples
    neighbour_margin  f(r, j, h) -> min |S_h - neighbour S_h| in the oracle, for the flag rule
    Returns a dict of statistics; raises AssertionError on a violation.
    """
    only_gpu = set(gpu) - set(orc)
    only_orc = set(orc) - set(gpu)
    for (r, j, h) in only_orc:
        p = orc[(r, j, h)][0]
        assert abs(p - thr[h - 1]) <= h * tol_abs, f"oracle-only candidate {(r, j, h)} power {p} thr {thr[h-1]}"
    for (r, j, h) in only_gpu:
        p = sum_lookup(r, j, h)
        assert p is not None, f"GPU candidate {(r, j, h)} is not defined in the oracle"
        assert abs(p - thr[h - 1]) <= h * tol_abs, f"GPU-only candidate {(r, j, h)} oracle power {p} thr {thr[h-1]}"
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
            if m is not None and m > 2 * h * tol_abs:
                flags_checked += 1
                if fg != fo:
                    flag_mismatch += 1
    assert flag_mismatch == 0, f"{flag_mismatch} non-fragile local-max flags differ"
    return dict(common=len(set(gpu) & set(orc)), only_gpu=len(only_gpu), only_orc=len(only_orc),
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

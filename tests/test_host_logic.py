"""CPU tests of the library's host logic and boundary (no GPU compute):
  - libfdas.so loads and exports every symbol include/fdas.h declares; argument validation
  - plan-time mathematics (closed-form templates, thresholds, whitening blocks) against the oracle
  - the K2 CTA stepped on the CPU by the test-only emulator against the oracle plane
  - trial sharding over ranks with a world_size-2 gloo group
"""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2211_13517_b200 import build, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def emu():
    sys.path.insert(0, os.path.join(ROOT, "tests", "emu"))
    import build_emu
    L = C.CDLL(build_emu.build_emu())
    L.fdas_emu_convolve.argtypes = [C.c_void_p, C.c_int64, C.c_double, C.c_double, C.c_int, C.c_int, C.c_void_p]
    L.fdas_emu_templates.argtypes = [C.c_double, C.c_double, C.c_int, C.c_int, C.c_void_p]
    L.fdas_emu_ifft.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
    L.fdas_emu_fresnel.argtypes = [C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.fdas_emu_thresholds.argtypes = [C.c_int, C.c_double, C.c_void_p]
    L.fdas_emu_whitening_blocks.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_int64]
    L.fdas_emu_whitening_blocks.restype = C.c_int64
    L.fdas_emu_halfwidth.argtypes = [C.c_double]
    L.fdas_emu_convolve_tc.argtypes = [C.c_void_p, C.c_int64, C.c_double, C.c_double, C.c_int, C.c_void_p, C.c_void_p]
    return L


@pytest.fixture(scope="module")
def fdaslib():
    build.build_lib()
    from paper_2211_13517_b200 import fdas
    return fdas


def test_abi_exports_every_declared_symbol(fdaslib):
    hdr = open(os.path.join(ROOT, "include", "fdas.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(fdas_[a-z_0-9]+)\s*\(", hdr))
    assert {"fdas_plan", "fdas_prepare_spectrum", "fdas_convolve_plane", "fdas_harmonic_sum_peaks"} <= declared
    lib = fdaslib.lib()
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in fdas.h but not exported"
    assert declared == set(fdaslib.EXPORTS)
    assert C.sizeof(fdaslib.FdasInfo) == 104 and fdaslib.CAND_DTYPE.itemsize == 16


def test_argument_validation_needs_no_device(fdaslib):
    lib = fdaslib.lib()
    h = C.c_void_p()
    E = fdaslib
    bad = [
        (0, 64e-6, 16.0, 1.0, 2048, 0),          # N too small
        (4095, 64e-6, 16.0, 1.0, 2048, 0),       # N < 2 * seg_len
        (1 << 17, 0.0, 16.0, 1.0, 2048, 0),      # tsamp
        (1 << 17, 64e-6, -1.0, 1.0, 2048, 0),    # zmax
        (1 << 17, 64e-6, 16.0, 0.0, 2048, 0),    # zstep
        (1 << 17, 64e-6, 16.0, 0.7, 2048, 0),    # 2 zmax / zstep not an integer
        (1 << 17, 64e-6, 16.0, 1.0, 2000, 0),    # seg_len not a power of two
        (1 << 17, 64e-6, 16.0, 1.0, 2048, 7),    # precision
        (1 << 17, 64e-6, 4000.0, 1.0, 2048, 0),  # V = L - 2h <= 0
    ]
    for args in bad:
        assert lib.fdas_plan(C.byref(h), *args) == E.FDAS_EARG, args
        assert not h.value
    for seg in (256, 512, 8192):                 # powers of two the FFT kernel is not built for
        assert lib.fdas_plan(C.byref(h), 1 << 17, 64e-6, 16.0, 1.0, seg, 0) == E.FDAS_EUNSUPPORTED
    assert lib.fdas_plan(None, 1 << 17, 64e-6, 16.0, 1.0, 2048, 0) == E.FDAS_EARG
    assert lib.fdas_plan_info(None, None) == E.FDAS_EARG
    assert lib.fdas_destroy(None) == E.FDAS_EARG
    assert lib.fdas_strerror(E.FDAS_EUNSUPPORTED).decode().startswith("unsupported")
    thr = np.empty(4, dtype=np.float32)
    assert lib.fdas_thresholds_from_sigma(0, 6.0, thr.ctypes.data_as(C.POINTER(C.c_float))) == E.FDAS_EARG
    assert lib.fdas_thresholds_from_sigma(33, 6.0, thr.ctypes.data_as(C.POINTER(C.c_float))) == E.FDAS_EARG


def test_plan_fails_loudly_without_a_device(fdaslib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(fdaslib.FdasError) as ei:
        fdaslib.Plan(1 << 17, 64e-6, 16.0, 1.0)
    assert ei.value.status in (fdaslib.FDAS_ECUDA, fdaslib.FDAS_EALLOC)


def test_library_templates_match_the_oracle_quadrature(emu, oracle):
    for zmax, zstep in ((16.0, 1.0), (96.0, 1.0), (4.0, 0.5)):
        nz = int(round(2 * zmax / zstep)) + 1
        h = oracle.halfwidth(zmax)
        assert emu.fdas_emu_halfwidth(zmax) == h
        T = np.empty((nz, 2 * h + 1), dtype=np.complex128)
        emu.fdas_emu_templates(zmax, zstep, nz, h, T.ctypes.data)
        assert np.abs(T - oracle.template_bank(zmax, zstep)).max() < 1e-12


def test_library_thresholds_and_blocks_match_the_oracle(emu, oracle, fdaslib):
    for H, ns in ((16, 6.0), (8, 6.0), (32, 3.0), (1, 10.0)):
        out = np.empty(H, dtype=np.float32)
        assert emu.fdas_emu_thresholds(H, ns, out.ctypes.data) == 0
        assert np.allclose(out, oracle.thresholds(H, ns), rtol=3e-7)
        assert np.array_equal(out, fdaslib.thresholds_from_sigma(H, ns))
    for nb in (2048, 65536, 1 << 22, 100000):
        s = np.empty(4096, dtype=np.int32); l = np.empty(4096, dtype=np.int32)
        n = emu.fdas_emu_whitening_blocks(nb, s.ctypes.data, l.ctypes.data, 4096)
        _, _, ctr = oracle.whiten(np.ones(nb, dtype=np.complex128), want_blocks=True)
        assert n == len(ctr)
        assert np.allclose(s[:n] + 0.5 * (l[:n] - 1), ctr)
        assert s[0] == 1 and s[n - 1] + l[n - 1] == nb


@pytest.mark.parametrize("L", [1024, 2048, 4096])
def test_emulated_segment_fft(emu, L):
    """The three register passes and two exchanges of the segment transform (fdas_fft_core.cuh), stepped
    thread by thread, against numpy for every segment length the kernel is built for."""
    rng = np.random.default_rng(0)
    x = (rng.standard_normal(L) + 1j * rng.standard_normal(L)).astype(np.complex64)
    out = np.full(L, np.nan, dtype=np.complex64)
    assert emu.fdas_emu_ifft(L, x.ctypes.data, out.ctypes.data) == 0
    ref = np.fft.ifft(x.astype(np.complex128)) * L
    assert np.abs(out - ref).max() < 1e-6 * np.abs(ref).max()
    # a single tone lands in exactly one output sample (index maps of both exchanges)
    for p0 in (1, 17, L // 16 + 3, L - 1):
        x = np.zeros(L, dtype=np.complex64)
        x[p0] = 1.0
        assert emu.fdas_emu_ifft(L, x.ctypes.data, out.ctypes.data) == 0
        assert np.abs(out - np.exp(2j * np.pi * p0 * np.arange(L) / L)).max() < 2e-6
    assert emu.fdas_emu_ifft(512, x.ctypes.data, out.ctypes.data) != 0


@pytest.mark.parametrize("zmax,nb,seg_len", [(16.0, 7000, 2048), (96.0, 4500, 2048), (0.0, 4096, 2048),
                                             (16.0, 7000, 1024), (96.0, 4500, 1024), (16.0, 9000, 4096),
                                             (96.0, 8200, 4096)])
def test_emulated_k2_matches_the_oracle_plane(emu, oracle, zmax, nb, seg_len):
    """Same index arithmetic, packed bank and exchange layouts as the CUDA kernel, stepped on the
    CPU: several segments, a ragged tail, a strong line, all three storage precisions, every seg_len."""
    rng = np.random.default_rng(4)
    w = ((rng.standard_normal(nb) + 1j * rng.standard_normal(nb)) / np.sqrt(2)).astype(np.complex64)
    w[nb // 3] += 15.0
    w[1] += 9.0
    w[nb - 1] += 7.0
    nz = int(2 * zmax) + 1
    bank = oracle.template_bank(zmax, 1.0)
    P = oracle.plane(w.astype(np.complex128), bank)
    for prec, tol in ((0, 1e-6), (1, 2e-2), (2, 2e-2)):
        out = np.full((nz, nb), np.nan, dtype=np.float32)
        assert emu.fdas_emu_convolve(w.ctypes.data, nb, zmax, 1.0, seg_len, prec, out.ctypes.data) == 0
        assert not np.isnan(out).any()                      # every r < nb written, nothing else
        assert np.abs(out - P).max() <= tol * P.max(), (prec, np.abs(out - P).max() / P.max())


@pytest.mark.parametrize("zmax,nb", [(16.0, 1152), (96.0, 640), (10.0, 384), (52.0, 256), (140.0, 256)])
def test_emulated_k2_tc_matches_the_oracle_plane(emu, oracle, zmax, nb):
    """K2-TC (tensor-core contraction) stepped on the CPU: same bank image in (emulated) tensor memory,
    interleaved re/im sliding-window image in shared memory with its UMMA descriptor (SBO = 128 B,
    LBO = 256 B), issue order, TMEM column map and pair epilogue as fdas_convolve_tc.cu; tcgen05.mma
    replaced by an operand walker.  Several tiles, both edges (zero fill below bin 0 and above nb), strong
    lines at the edges; zmax = 140 (140 pairs) takes two launches of 96 and 44 pairs."""
    rng = np.random.default_rng(5)
    w = ((rng.standard_normal(nb) + 1j * rng.standard_normal(nb)) / np.sqrt(2)).astype(np.complex64)
    w[nb // 3] += 15.0
    w[1] += 9.0
    w[nb - 1] += 7.0
    nz = int(2 * zmax) + 1
    bank = oracle.template_bank(zmax, 1.0)
    P = oracle.plane(w.astype(np.complex128), bank)

    def bf16(a):   # round-to-nearest-even to bfloat16, returned as float32
        u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)
        return ((u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000).astype(np.uint32).view(np.float32)

    Pq = oracle.plane(bf16(w.real).astype(np.float64) + 1j * bf16(w.imag).astype(np.float64), bank)
    for plane16 in (0, 1):
        out = np.full((nz, nb), np.nan, dtype=np.float32)
        mx = np.zeros((nz, nb // 8), dtype=np.uint16)
        assert emu.fdas_emu_convolve_tc(w.ctypes.data, nb, zmax, 1.0, plane16, out.ctypes.data, mx.ctypes.data) == 0
        assert not np.isnan(out).any()
        assert np.abs(out - P).max() <= 2e-2 * P.max()
        # against the oracle on the bf16-rounded spectrum (reading A11) only the bf16 rounding of the
        # taps (2^-9 relative per tap) and, for plane16, of the stored power remains
        assert np.abs(out - Pq).max() <= (5e-3 if not plane16 else 9e-3) * Pq.max(), np.abs(out - Pq).max() / Pq.max()
        # block-max codes (units of 1/8, rounded up, 1023 = no bound) bound the stored values from above
        blk = out.reshape(nz, nb // 8, 8).max(axis=2)
        assert np.array_equal(mx, np.minimum(np.ceil(blk * np.float32(8.0)), 1023).astype(np.uint16))
        assert ((mx / 8.0 >= blk) | (mx == 1023)).all()


# --------------------------------------------------------------------------- sharding over ranks
def test_shard_trials_partition():
    for n, world in ((64, 1), (64, 2), (5925, 8), (3, 4)):
        parts = [inputs.shard_trials(n, r, world) for r in range(world)]
        flat = sorted(t for p in parts for t in p)
        assert flat == list(range(n))
        assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1


_GLOO_WORKER = r"""
import os, sys, json
sys.path.insert(0, sys.argv[1])
import torch, torch.distributed as dist
from paper_2211_13517_b200 import dist as fd, inputs
ctx = fd.init_from_env(backend="gloo")
mine = inputs.shard_trials(7, ctx.rank, ctx.world)
# stand-in for per-trial work: deterministic candidate count and points per trial
counts = {t: (t * 3) % 5 for t in mine}
pts = 1000 * len(mine)
total_pts = fd.sum_over_ranks(ctx, pts)
t_max = fd.max_over_ranks(ctx, 1.0 + ctx.rank)
allc = fd.gather_dicts(ctx, counts)
fd.barrier(ctx)
if ctx.rank == 0:
    print(json.dumps({"total_pts": total_pts, "t_max": t_max, "allc": sorted(allc.items())}))
fd.finalize(ctx)
"""


def test_gloo_world2_sharding(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER)
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script), ROOT]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    res = json.loads(line)
    assert res["total_pts"] == 7000
    assert res["t_max"] == 2.0
    assert res["allc"] == [[str(t), (t * 3) % 5] for t in sorted(range(7), key=str)] or \
        dict((int(k), v) for k, v in res["allc"]) == {t: (t * 3) % 5 for t in range(7)}


def test_bench_starts_its_own_ranks_and_shares_one_workload_string():
    """`bench.py --gpus N` launched plainly re-executes itself under torch.distributed.run with N ranks;
    both arms describe the workload with the same string; the DRAM traffic comes from profiles/."""
    sys.path.insert(0, ROOT)
    import bench
    cmd = bench.spawn_command(4, ["--gpus", "4", "--steps", "7"])
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node=4" in cmd and "127.0.0.1" in cmd
    assert cmd[-4:] == ["--gpus", "4", "--steps", "7"] and cmd[-5].endswith("bench.py")
    wl = inputs.ska()
    assert "N=9375000" in bench.workload_string(wl) and "nz=193" in bench.workload_string(wl)
    t = bench.ncu_traffic("ska", "bf16_tc")
    assert t is not None and t["file"].startswith("profiles/") and 3.2e9 < t["traffic"] < 3.6e9
    assert "convolve_tc_kernel" in t["kernel"] and t["commit"]
    assert bench.ncu_traffic("tiny", "bf16_tc") is None


def test_parity_stats_are_written_only_on_request_and_tabulated(tmp_path, monkeypatch):
    import helpers
    monkeypatch.delenv("FDAS_PARITY_STATS", raising=False)
    helpers.record_stats("nowhere", {"points": 1})                       # no variable: no file anywhere
    assert not os.path.exists(os.path.join(str(tmp_path), "stats.jsonl"))
    path = os.path.join(str(tmp_path), "sub", "stats.jsonl")
    monkeypatch.setenv("FDAS_PARITY_STATS", path)
    helpers.record_stats("a", {"points": 10, "worst_over_max": 1e-3, "common": 5})
    helpers.record_stats("a", {"points": 12, "worst_over_max": 2e-3, "common": 6})
    helpers.record_stats("b", {"only_gpu": 1})
    table = helpers.stats_table(open(path)).splitlines()
    assert len(table) == 4 and table[2].startswith("| a | 12 | 2.00e-03") and "| b |" in table[3]

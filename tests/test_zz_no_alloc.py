"""fdas_whiten_static: whitening for callers that are not allowed to allocate device memory.

Some users of this library cannot call cudaMalloc: a stage of a real-time backend that gave all of its
HBM to its own pool at start-up (a later cudaMalloc may fail, and it stalls every stream of the device
while it runs), or a plug-in that may only touch the buffers it is handed.  They cannot create an
fdas_plan (which allocates the whitening tables), so the library offers them one plan-free call whose
tables live in a fixed 51 KB array inside libfdas.so (limit: 2^24 bins).

This file checks that call against the existing path (fdas_plan + fdas_prepare_spectrum) on the same raw
spectrum X, on calls made one after another that share the fixed array: a long spectrum, then a short
one (the array still holds the long call's tables beyond the short schedule), then the long one again.
The tolerance is the one the parity tests apply to the whitened spectrum (2e-5 of its largest modulus
for fp32; one bf16 rounding step for bf16); because both paths run the same two kernels the outputs
are also required to be bit-identical.

The file is named so that pytest collects it last (`pytest --collect-only`): under `pytest -x` a
failure here cannot hide the other tests.  It passes alone in a fresh process and after the others.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2211_13517_b200 import inputs

pytestmark = pytest.mark.gpu

MAX_BINS = 1 << 24    # the stated limit of the fixed scratch array


@pytest.fixture(scope="module")
def fdas():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2211_13517_b200 import fdas as F   # raises if libfdas.so is missing (no fallback)
    return F


def _existing_path(fdas, torch, wl, precision):
    """fdas_prepare_spectrum through a plan; returns (plan, whitened spectrum, pointer to the raw X)."""
    plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, precision)
    d_x = torch.from_numpy(inputs.series_for(wl)).cuda()
    d_ref = plan.alloc_spec()
    plan.prepare_spectrum(d_x, d_ref)
    torch.cuda.synchronize()
    x_ptr, ncomplex = plan.debug_rawspectrum()
    assert ncomplex == plan.info.nbins + 1
    return plan, d_ref, x_ptr


def _compare(torch, d_new, d_ref, precision):
    new = d_new.float().cpu().numpy().astype(np.float64)
    ref = d_ref.float().cpu().numpy().astype(np.float64)
    assert not np.isnan(new).any()
    wmax = np.hypot(ref[:, 0], ref[:, 1]).max()
    tol = 2e-5 * wmax if precision == "fp32" else 2.0 ** -8 * wmax
    assert np.abs(new - ref).max() <= tol
    assert torch.equal(d_new.view(torch.uint8), d_ref.view(torch.uint8))   # same kernels, same X: same bits
    assert new[0, 0] == 0.0 and new[0, 1] == 0.0                           # w[0] = 0 (reading A2)


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_whiten_static_matches_prepare_spectrum_on_calls_in_a_row(fdas, precision):
    import torch
    long_wl, short_wl = inputs.medium(), inputs.tiny()     # 2^20 bins (284 blocks), 2^16 bins (44 blocks)
    plan_l, ref_l, x_l = _existing_path(fdas, torch, long_wl, precision)
    plan_s, ref_s, x_s = _existing_path(fdas, torch, short_wl, precision)
    nb_l, nb_s = plan_l.info.nbins, plan_s.info.nbins
    outs = []
    for x_ptr, nb in ((x_l, nb_l), (x_s, nb_s), (x_l, nb_l)):
        out = torch.full((nb, 2), float("nan"), dtype=ref_l.dtype, device="cuda")
        fdas.whiten_static(x_ptr, nb, out)          # same stream every time: the calls do not overlap
        outs.append(out)
    torch.cuda.synchronize()
    _compare(torch, outs[0], ref_l, precision)
    _compare(torch, outs[1], ref_s, precision)
    _compare(torch, outs[2], ref_l, precision)
    # a further call, after every kernel of the entry point has run once: the device's free memory is
    # the same before and after (nothing was allocated on the device)
    out = torch.empty((nb_s, 2), dtype=ref_s.dtype, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    fdas.whiten_static(x_s, nb_s, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    _compare(torch, out, ref_s, precision)
    plan_l.close()
    plan_s.close()


def test_whiten_static_at_its_maximum_size(fdas):
    """2^24 bins, the most the fixed array holds (4124 blocks of its 4352 entries)."""
    import torch
    g = torch.Generator(device="cuda")
    g.manual_seed(20221113)
    d_x = torch.randn(1 << 25, generator=g, device="cuda", dtype=torch.float32)
    plan = fdas.Plan(1 << 25, 64e-6, 4.0, 1.0, 2048, "fp32")
    assert plan.info.nbins == MAX_BINS
    d_ref = plan.alloc_spec()
    plan.prepare_spectrum(d_x, d_ref)
    torch.cuda.synchronize()
    x_ptr, _ = plan.debug_rawspectrum()
    out = torch.full((MAX_BINS, 2), float("nan"), dtype=torch.float32, device="cuda")
    fdas.whiten_static(x_ptr, MAX_BINS, out)
    torch.cuda.synchronize()
    _compare(torch, out, d_ref, "fp32")
    plan.close()


@pytest.mark.parametrize("spec_dtype", ["float32", "bfloat16"])
@pytest.mark.parametrize("nbins", [1024, 100_003, 1_000_001])
def test_whiten_static_against_the_oracle_on_lengths_a_plan_cannot_have(fdas, oracle, nbins, spec_dtype):
    """A plan always has a power-of-two number of bins; this call takes any length from 1024 to 2^24, so the
    lengths whose last block is cut short are compared with the CPU oracle's whitening (O2) directly, at the
    tolerances of the parity tests (2e-5 of the largest modulus for fp32, 1e-2 for bf16 storage), with guard
    rows behind the output that must stay untouched."""
    import torch
    rng = np.random.default_rng(nbins)
    red = 1.0 + 30.0 / (1.0 + np.arange(nbins + 1) / 500.0)                     # a red-noise-like slope to whiten
    X32 = np.stack([rng.standard_normal(nbins + 1) * red, rng.standard_normal(nbins + 1) * red], axis=1).astype(np.float32)
    d_X = torch.from_numpy(X32).cuda()
    w = oracle.whiten(X32[:nbins, 0].astype(np.float64) + 1j * X32[:nbins, 1].astype(np.float64))
    dt = getattr(torch, spec_dtype)
    buf = torch.full((nbins + 64, 2), float("nan"), dtype=dt, device="cuda")
    fdas.whiten_static(d_X, nbins, buf[:nbins])
    torch.cuda.synchronize()
    got = buf[:nbins].float().cpu().numpy().astype(np.float64)
    assert torch.isnan(buf[nbins:].float()).all().item()                        # nothing written past the end
    assert not np.isnan(got).any() and got[0, 0] == 0.0 and got[0, 1] == 0.0
    tol = (2e-5 if spec_dtype == "float32" else 1e-2) * np.abs(w).max()
    assert np.abs(got[:, 0] + 1j * got[:, 1] - w).max() <= tol


def test_whiten_static_refuses_sizes_beyond_the_fixed_array(fdas):
    import torch
    lib = fdas.lib()
    buf = torch.zeros(4096, dtype=torch.float32, device="cuda")
    p = C.c_void_p(buf.data_ptr())
    # refused before anything is launched, so the small buffers are never touched
    assert lib.fdas_whiten_static(p, MAX_BINS + 1, p, 0, None) == fdas.FDAS_EUNSUPPORTED
    detail = lib.fdas_last_error_detail().decode()
    assert "16777216" in detail and "exceeds" in detail
    assert lib.fdas_whiten_static(p, 1023, p, 0, None) == fdas.FDAS_EARG
    assert lib.fdas_whiten_static(None, 4096, p, 0, None) == fdas.FDAS_EARG
    assert lib.fdas_whiten_static(p, 4096, None, 0, None) == fdas.FDAS_EARG
    assert lib.fdas_whiten_static(p, 4096, p, 2, None) == fdas.FDAS_EARG
    torch.cuda.synchronize()
    assert float(buf.abs().max()) == 0.0

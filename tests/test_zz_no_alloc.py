"""hk_opacity_noalloc: the opacity function for callers that may not allocate GPU memory.

Some users of this library cannot let it take memory from the CUDA driver at call time: their process handed the whole
GPU to an allocator of its own at start-up, or the call sits in a latency-bound loop next to other running streams, or
their deployment forbids allocation once it is up.  For them hk_opacity_noalloc runs the kernels of hk_opacity with the
library's work space (per-line records, line-range tables, tile counters) in a fixed ~11 MiB array inside libhk.so.

What is checked here: the new entry point gives bit-for-bit the kappa of hk_opacity (the bar the repo's determinism tests
use; both run the same kernels in the same order) on calls made back to back on the same stream, where each call finds in
the shared array whatever the previous one left — a longer list before a shorter one, FP32 records before an FP64 call,
a different grid; that the free device memory does not move across such calls; and that requests beyond the stated
limits are refused with a message that names the limit.

This file is collected last on purpose (pytest -x stops at the first failure): a failure here hides no other test.  It
passes alone in a fresh process (the first call then does the one-time set-up) and after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import workloads
import paper_1503_03806_b200 as hk


def _case(seed, n_lines, nu_max, cutoff, T, P):
    wl = workloads.small(seed=seed, n_lines=n_lines, nu_max=nu_max, cutoff=cutoff, T=T, P_atm=P)
    return wl, hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0), T, P


def _both(wl, lines, T, P, out, **kw):
    """(kappa of the existing path, kappa of the no-alloc entry point written into `out`)"""
    ref = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, mass_amu=wl.mass_amu, **kw)
    got = hk.hk_opacity_noalloc(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out, mass_amu=wl.mass_amu, **kw)
    assert got is out
    return ref, got


def test_same_kappa_as_hk_opacity_on_calls_in_a_row():
    import torch
    # each call inherits the array as the one before left it: many lines then few, a wide grid then a ragged narrow one
    # (N = 3333), FP32-variant records then FP64 only, a Doppler-dominated list (series region) then a Lorentz-dominated one
    cases = [
        (_case(11, 3000, 400.0, 100.0, 1000.0, 1e-5), dict()),
        (_case(12, 50, 33.33, 7.0, 300.0, 1e-3), dict()),
        (_case(13, 2000, 250.0, 25.0, 1500.0, 1.0), dict(precision=hk.HK_FP32)),
        (_case(14, 300, 60.0, 25.0, 800.0, 100.0), dict(cutoff_widths=200.0)),
        (_case(12, 50, 33.33, 7.0, 300.0, 1e-3), dict()),
    ]
    outs = [torch.full((c[0][0].n_points,), float("nan"), dtype=torch.float64, device="cuda") for c in cases]
    for rounds in range(2):                                   # the whole sequence twice, back to back
        for ((wl, lines, T, P), kw), out in zip(cases, outs):
            ref, got = _both(wl, lines, T, P, out, **kw)
            torch.cuda.synchronize()
            assert torch.isfinite(got).all() and float(got.max()) > 0.0
            assert torch.equal(got, ref), (wl.name, kw, float((got - ref).abs().max()))
    # a mixture: the second species is added to the running sum, as with hk_opacity
    (wl, lines, T, P), _ = cases[0]
    half = hk.Lines.from_numpy(wl.nu0[::2], wl.S[::2], wl.gamma0[::2]), hk.Lines.from_numpy(wl.nu0[1::2], wl.S[1::2], wl.gamma0[1::2])
    acc_ref = torch.empty_like(outs[0])
    acc_got = torch.empty_like(outs[0])
    for k, part in enumerate(half):
        hk.hk_opacity(part, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out=acc_ref, accumulate=k > 0, abundance=0.5)
        hk.hk_opacity_noalloc(part, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, acc_got, accumulate=k > 0, abundance=0.5)
    torch.cuda.synchronize()
    assert torch.equal(acc_got, acc_ref)


def test_free_device_memory_does_not_move():
    import torch
    (wl, lines, T, P) = _case(21, 4000, 500.0, 100.0, 1200.0, 0.1)
    out = torch.empty(wl.n_points, dtype=torch.float64, device="cuda")
    ref, got = _both(wl, lines, T, P, out)                    # first call on this device, if the file runs alone: set-up
    out32 = torch.empty_like(out)
    ref32, _ = _both(wl, lines, T, P, out32, precision=hk.HK_FP32)
    torch.cuda.synchronize()
    assert torch.equal(got, ref)
    out.fill_(float("nan"))
    out32.fill_(float("nan"))
    hk.hk_trim()                                              # the library's pool is now empty: any use of it must grow it
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(2):
        hk.hk_opacity_noalloc(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out)
        hk.hk_opacity_noalloc(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, out32, precision=hk.HK_FP32)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    assert free1 == free0, (free0, free1)
    assert torch.equal(out, ref) and torch.equal(out32, ref32)


def test_requests_beyond_the_fixed_work_space_are_refused():
    import torch
    assert hk.HK_NOALLOC_MAX_LINES == 65536 and hk.HK_NOALLOC_MAX_POINTS == 4194304
    n = hk.HK_NOALLOC_MAX_LINES + 1
    nu0 = torch.linspace(1.0, 99.0, n, dtype=torch.float64, device="cuda")
    big = hk.Lines(nu0, torch.full_like(nu0, 1e-22), torch.full_like(nu0, 0.05))
    out = torch.zeros(10000, dtype=torch.float64, device="cuda")
    with pytest.raises(hk.HKError) as e:
        hk.hk_opacity_noalloc(big, 1000.0, 1.0, 0.0, 100.0, 0.01, 25.0, out)
    assert e.value.code == -5 and "HK_NOALLOC_MAX_LINES = 65536" in str(e.value) and str(n) in str(e.value)
    few = hk.Lines(nu0[:100].contiguous(), big.S[:100].contiguous(), big.gamma0[:100].contiguous())
    wide = torch.zeros(hk.HK_NOALLOC_MAX_POINTS + 256, dtype=torch.float64, device="cuda")
    with pytest.raises(hk.HKError) as e:
        hk.hk_opacity_noalloc(few, 1000.0, 1.0, 0.0, 0.01 * wide.numel(), 0.01, 25.0, wide)
    assert e.value.code == -5 and "HK_NOALLOC_MAX_POINTS = 4194304" in str(e.value)
    shifted = hk.Lines(few.nu0, few.S, few.gamma0, delta=torch.zeros_like(few.nu0))
    with pytest.raises(hk.HKError) as e:
        hk.hk_opacity_noalloc(shifted, 1000.0, 1.0, 0.0, 100.0, 0.01, 25.0, out)
    assert e.value.code == -5 and "delta" in str(e.value)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0 and float(wide.abs().max()) == 0.0      # a refused call writes nothing
    # the largest admitted sizes run (the whole array in use) and agree with hk_opacity
    full = hk.Lines(nu0[:-1].contiguous(), big.S[:-1].contiguous(), big.gamma0[:-1].contiguous())
    edge = torch.empty(hk.HK_NOALLOC_MAX_POINTS, dtype=torch.float64, device="cuda")
    nu_max = 100.0
    dnu = nu_max / hk.HK_NOALLOC_MAX_POINTS
    assert hk.hk_grid_size(0.0, nu_max, dnu) == hk.HK_NOALLOC_MAX_POINTS
    hk.hk_opacity_noalloc(full, 1000.0, 1.0, 0.0, nu_max, dnu, 0.05, edge)
    ref = hk.hk_opacity(full, 1000.0, 1.0, 0.0, nu_max, dnu, 0.05)
    torch.cuda.synchronize()
    assert torch.equal(edge, ref) and float(edge.max()) > 0.0

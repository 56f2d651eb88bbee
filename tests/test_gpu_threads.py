"""Two host threads drive the library at once (include/hk.h: "calls may come from several host threads").

PAPER.md:215 (section 2.5): the calculation is "repeat[ed] ... for multiple combinations of temperature and pressure"; the
natural way to drive that from a host is one thread per stream.  Each thread has a torch stream and an hk.Context of its
own and mixes context calls with the one-shot entry points (hk_opacity, hk_kdist, hk_opacity_host); one thread alone
switches hk_set_timing on (the switch, its events and the last-error text are per thread).  What the library shares between
them — the per-device memory pool, the once-per-device kernel attributes and launch grids — is taken under locks.  Every
result must be the bits of the same call made serially.
"""
import threading

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import workloads
import paper_1503_03806_b200 as hk

N_CALLS = 50


def _work(tid, wl, lines, pairs, results, errors, timing, barrier):
    import torch
    try:
        torch.cuda.set_device(0)
        stream = torch.cuda.Stream()
        with torch.cuda.stream(stream):
            ctx = hk.Context(lines, stream=stream)
            if timing:
                hk.hk_set_timing(True)
            barrier.wait()
            out = []
            for n in range(N_CALLS):
                T, P = pairs[(n + 7 * tid) % len(pairs)]
                kind = n % 4
                if kind == 0:
                    k = ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
                    if timing:
                        ms = hk.hk_last_stage_ms()
                        assert len(ms) == 3 and all(v >= 0.0 for v in ms) and ms[1] > 0.0
                    out.append((n, k))
                elif kind == 1:
                    k = hk.hk_opacity(lines, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff, stream=stream,
                                      precision=hk.HK_FP32 if n % 8 == 1 else hk.HK_FP64)
                    out.append((n, k))
                elif kind == 2:
                    k = ctx.opacity(T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
                    out.append((n, hk.hk_kdist(k, wl.dnu, wl.bin_width, wl.n_g, stream=stream)))
                else:
                    kap, kt = hk.hk_opacity_host(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff,
                                                 bin_width=wl.bin_width, n_g=wl.n_g, stream=stream)
                    out.append((n, torch.cat((kap, kt.ravel()))))
            stream.synchronize()
            if timing:
                hk.hk_set_timing(False)
            ctx.close()
            results[tid] = [(n, t.cpu().numpy().copy()) for n, t in out]
    except Exception as e:                                      # surfaces in the main thread
        errors.append((tid, repr(e)))
        try:
            barrier.abort()
        except Exception:
            pass


def test_two_threads_interleaved_equal_the_serial_run():
    import torch
    wl = workloads.small(seed=61, n_lines=3000, nu_max=600.0, cutoff=25.0)          # 60 000 points: the ranged host path too
    lines = hk.Lines.from_numpy(wl.nu0, wl.S, wl.gamma0)
    pairs = [(1500.0, 1.0), (800.0, 10.0), (2500.0, 1e-3), (300.0, 0.1), (1000.0, 100.0)]
    torch.cuda.synchronize()

    def run(threads):
        results, errors = {}, []
        barrier = threading.Barrier(len(threads))
        ts = [threading.Thread(target=_work, args=(tid, wl, lines, pairs, results, errors, tid == 0, barrier)) for tid in threads]
        for t in ts:
            t.start()
        for t in ts:
            t.join(timeout=300)
        assert not errors, errors
        assert all(not t.is_alive() for t in ts)
        return results

    serial = {}
    for tid in (0, 1):
        serial.update(run([tid]))
    both = run([0, 1])
    for tid in (0, 1):
        assert len(both[tid]) == len(serial[tid]) == N_CALLS
        for (n, a), (m, b) in zip(both[tid], serial[tid]):
            assert n == m and a.shape == b.shape
            assert np.array_equal(a, b), (tid, n, float(np.abs(a - b).max()))

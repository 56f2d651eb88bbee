"""Host logic of the N > 1 path (paper_1503_03806_b200/shard.py) on CPU: world_size 2 over gloo.

Each rank computes ITS shard with the oracle standing in for the device call (same arguments it would hand to hk_opacity:
its own nu_min/nu_max and its slice of the line list), the shards are gathered, and the concatenation must equal the
unsharded oracle result: proves the bin-aligned ranges, the line halo and the pair partition are right.  No collective is
on the data path; gloo carries only the gather that the test itself needs.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import workloads
from paper_1503_03806_b200 import shard


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = workloads.small(seed=11, n_lines=600, nu_max=80.0, cutoff=7.0)
        # ramp the density so that equal widths would NOT balance
        wl.nu0 = np.sort(80.0 * (1.0 - np.sqrt(1.0 - wl.nu0 / 80.0)))
        N = wl.n_points
        ppb = int(round(wl.bin_width / wl.dnu))
        shards = shard.shard_grid(wl.nu0, wl.nu_min, N, wl.dnu, wl.cutoff, ppb, world)
        me = shards[rank]
        sl = slice(me.line_lo, me.line_hi)
        T, P = wl.T[0], wl.P_atm[0]
        kap = oracle.opacity(wl.nu0[sl], wl.S[sl], wl.gamma0[sl], T, P, me.nu_min, me.nu_max, wl.dnu, wl.cutoff)
        assert kap.shape[0] == me.j_hi - me.j_lo
        ktab = oracle.kdist(kap, ppb, wl.n_g)
        gathered = [None] * world
        dist.all_gather_object(gathered, (me.j_lo, kap, ktab, me.evals))
        # T-P pairs: every pair owned exactly once, in order
        owned = [None] * world
        dist.all_gather_object(owned, list(shard.shard_pairs(7, rank, world)))
        if rank == 0:
            full = oracle.opacity(wl.nu0, wl.S, wl.gamma0, T, P, wl.nu_min, wl.nu_max, wl.dnu, wl.cutoff)
            got = np.concatenate([g[1] for g in sorted(gathered, key=lambda g: g[0])])
            kgot = np.concatenate([g[2] for g in sorted(gathered, key=lambda g: g[0])])
            kfull = oracle.kdist(full, ppb, wl.n_g)
            ev = [g[3] for g in gathered]
            q.put(dict(err=float(np.abs(got / full - 1.0).max()), kerr=float(np.abs(kgot / kfull - 1.0).max()),
                       n=int(got.shape[0]), N=N, evals=ev, total=int(oracle.count_evals(wl.nu0, wl.nu_min, N, wl.dnu, wl.cutoff)),
                       pairs=sum(owned, []), widths=[s.j_hi - s.j_lo for s in shards]))
    finally:
        dist.destroy_process_group()


def test_grid_and_pair_sharding_world2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res["n"] == res["N"]
    # each rank's grid nu_min' + j*dnu may differ from nu_min + (j_lo+j)*dnu by one rounding: far below the 1e-6 bar
    assert res["err"] < 1e-9 and res["kerr"] < 1e-9
    assert sum(res["evals"]) == res["total"]
    assert max(res["evals"]) < 0.62 * res["total"]               # balanced by work ...
    assert res["widths"][0] < res["widths"][1]                  # ... not by width (density ramps down)
    assert res["pairs"] == list(range(7))


def test_shard_pairs_and_grid_edges():
    for n, w in ((200, 8), (7, 2), (3, 3), (0, 2), (5, 8)):
        parts = [list(shard.shard_pairs(n, r, w)) for r in range(w)]
        assert sum(parts, []) == list(range(n))
        assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    wl = workloads.config(0)
    sh = shard.shard_grid(wl.nu0, wl.nu_min, wl.n_points, wl.dnu, wl.cutoff, 1000, 8)
    assert sh[0].j_lo == 0 and sh[-1].j_hi == wl.n_points
    assert all(a.j_hi == b.j_lo for a, b in zip(sh, sh[1:]))
    assert all(s.j_lo % 1000 == 0 for s in sh)
    for s in sh:     # the halo holds every line that can reach the range, and only a contiguous slice
        reach = (wl.nu0 + wl.cutoff >= s.nu_min - 1e-9) & (wl.nu0 - wl.cutoff <= s.nu_max + 1e-9)
        idx = np.flatnonzero(reach)
        assert s.line_lo <= idx[0] + 1 and s.line_hi >= idx[-1]
    with pytest.raises(ValueError):
        shard.shard_grid(wl.nu0, 0.0, 1001, 0.01, 25.0, 1000, 2)

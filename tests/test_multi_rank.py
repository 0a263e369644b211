"""N > 1 host logic on CPU: two gloo ranks shard the DM list as the paper does (every
GPU gets the same input and a slice of the DM list), build their plans through the C ABI and agree
with the oracle's full table; timing is aggregated as max over ranks."""
import os
import socket
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import paper_1107_2516_b200 as dd
    from paper_1107_2516_b200 import shard, synth
    from oracle import dedisp_oracle as orc

    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        # brute force: cfg-1 geometry, 67 trials (not a multiple of the world size)
        cf = synth.scaled(synth.configs()[1], ndm=67)
        lo, hi = shard.dm_slice(cf.ndm, world, rank)
        plan = dd.Plan(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list[lo:hi])
        full = shard.gather_rows(plan.shifts(), dist)
        ref = orc.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
        ok_tab = bool((full == ref).all())
        md = shard.max_over_ranks(plan.max_delay, dist)
        # subband: whole coarse groups per rank
        cs = synth.scaled(synth.configs()[4], nchans=256, nsub=4, ndm=5 * 32, n_out=1024)
        slo, shi = shard.dm_slice(cs.ndm, world, rank, multiple=cs.nfine)
        sp = dd.Plan(cs.nchans, cs.f_top_mhz, cs.df_mhz, cs.t_samp_ms, cs.dm_list[slo:shi], cs.nsub, cs.nfine)
        s1, s2, nom, m2 = sp.subband_shifts()
        t = orc.subband_tables(cs.nchans, cs.f_top_mhz, cs.df_mhz, cs.t_samp_ms, cs.dm_list, cs.nsub, cs.nfine)
        ok_sub = bool((shard.gather_rows(s2, dist) == t.s2).all() and (shard.gather_rows(s1, dist) == t.s1).all())
        # timing rule: whole-job units / max over ranks of the device time
        v, ms = shard.job_throughput(float(hi - lo), 10.0 * (rank + 1), dist)
        q.put((rank, lo, hi, slo, shi, ok_tab, md, int(ref.max()), ok_sub, v, ms))
    finally:
        dist.destroy_process_group()


def test_dm_slices_cover_the_list():
    sys.path.insert(0, ROOT)
    from paper_1107_2516_b200 import shard
    for ndm, world, mult in [(67, 2, 1), (4096, 8, 32), (5, 8, 1), (160, 3, 32), (0, 2, 1)]:
        edges = [shard.dm_slice(ndm, world, r, mult) for r in range(world)]
        assert edges[0][0] == 0 and edges[-1][1] == ndm
        assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
        lens = [hi - lo for lo, hi in edges]
        assert all(n % mult == 0 for n in lens) and max(lens) - min(lens) <= mult
    with pytest.raises(ValueError):
        shard.dm_slice(10, 2, 2)
    with pytest.raises(ValueError):
        shard.dm_slice(33, 2, 0, multiple=32)
    assert shard.beam_of(3, 4, 1) == 13
    assert shard.max_over_ranks(2.5) == 2.5 and shard.job_throughput(10.0, 5.0)[0] == 2000.0


@pytest.mark.timeout(300)
def test_two_gloo_ranks_shard_the_dm_list():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=240) for _ in range(world))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (r0, lo0, hi0, slo0, shi0, *rest0), (r1, lo1, hi1, slo1, shi1, *rest1) = res
    assert (lo0, hi0, lo1, hi1) == (0, 34, 34, 67)
    assert (slo0, shi0, slo1, shi1) == (0, 96, 96, 160)
    for ok_tab, md, refmax, ok_sub, v, ms in (rest0, rest1):
        assert ok_tab and ok_sub
        assert md == refmax                       # max over ranks of the shards' max_delay
        assert ms == 20.0 and np.isclose(v, 67.0 / 0.020)

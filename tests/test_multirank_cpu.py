"""World-size-2 gloo tests of the multi-GPU host logic: time shards with a
max_shift halo and DM shards reproduce the single-device result with no data-path collective;
whole-job throughput is sum(units) / max(time).  The per-shard transform here is the ORACLE
(tests may use it; there is no GPU in this container) -- what is under test is the sharding."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2311_05341_b200 import shard  # noqa: E402


def test_time_shards_cover_output_exactly():
    for nsamps, mx, world in [(4096, 130, 2), (1000, 999, 4), (70001, 333, 8), (50, 3, 3)]:
        sh = shard.time_shards(nsamps, mx, world)
        assert sh[0].out_start == 0 and sh[-1].out_stop == nsamps - mx
        for a, b in zip(sh, sh[1:]):
            assert a.out_stop == b.out_start
        assert max(s.out_len for s in sh) - min(s.out_len for s in sh) <= 1
        for s in sh:
            if s.out_len:
                assert s.in_start == s.out_start and s.in_stop == s.out_stop + mx <= nsamps
    with pytest.raises(ValueError):
        shard.time_shards(10, 10, 2)


def test_dm_shards_cover_list():
    for ndm, world in [(1000, 8), (5, 8), (32, 2)]:
        sl = shard.dm_shards(ndm, world)
        assert sl[0][0] == 0 and sl[-1][1] == ndm
        assert all(a[1] == b[0] for a, b in zip(sl, sl[1:]))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, mode, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    from oracle import oracle
    from paper_2311_05341_b200 import workloads as W
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = W.CONFIGS["tiny"]
        table, mx = oracle.shift_table(cfg.nchans, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list)
        x = W.make_input_numpy(cfg, table, cfg.nsamps - mx)
        full = oracle.dedisperse(x, table, cfg.nsamps - mx)
        if mode == "time":
            s = shard.time_shards(cfg.nsamps, mx, world)[rank]
            part = oracle.dedisperse(np.ascontiguousarray(x[:, s.in_start:s.in_stop]), table, s.out_len)
            ok = np.array_equal(part, full[:, s.out_start:s.out_stop])
        else:
            d0, d1 = shard.dm_shards(cfg.ndm, world)[rank]
            part = oracle.dedisperse(x, table[d0:d1], cfg.nsamps - mx)
            ok = np.array_equal(part, full[d0:d1])
        # reporting collective: sum(units) / max(time)
        value, ms = shard.job_throughput(100.0 * (rank + 1), 10.0 * (rank + 1), dist)
        agree = torch.tensor([1 if ok else 0])
        dist.all_reduce(agree, op=dist.ReduceOp.MIN)
        q.put((rank, bool(agree.item()), value, ms))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("mode", ["time", "dm"])
def test_two_rank_shards_reproduce_single_device_result(mode, oracle):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q, port, world = ctx.Queue(), _free_port(), 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, mode, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ok, value, ms in res:
        assert ok, "rank %d: shard output differs from the single-device result" % rank
        assert ms == 20.0 and abs(value - 300.0 / 0.020) < 1e-9

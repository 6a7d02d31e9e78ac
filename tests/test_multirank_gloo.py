"""N > 1 host logic on CPU: two gloo ranks (127.0.0.1).  bench.py's max-over-ranks timing / whole-job aggregate, and the
z-slab shard ownership of the C ABI (vol_shard_layers needs no GPU): the shards partition the volume exactly."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    import bench
    import paper_1602_06645_b200 as vf

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # timing: every rank reports its own device time, all must agree on the maximum
        mine = [10.0 + 5.0 * rank, 3.0 - rank]
        got = bench.max_over_ranks(mine, world, "cpu")
        # sharding: gather every rank's owned layers
        nz = 44
        layers = torch.from_numpy(vf.shard_layers(nz, rank, world).astype(np.int64))
        pad = torch.full((nz,), -1, dtype=torch.int64)
        pad[: layers.numel()] = layers
        allp = [torch.empty_like(pad) for _ in range(world)]
        dist.all_gather(allp, pad)
        q.put((rank, got, [a[a >= 0].tolist() for a in allp]))
    finally:
        dist.destroy_process_group()


def test_two_ranks_timing_and_shards():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=180) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, owned in res:
        assert got == [15.0, 3.0]                                    # max over ranks of each entry
        flat = sorted(k for o in owned for k in o)
        assert flat == list(range(44))                               # every layer owned exactly once
        for r, o in enumerate(owned):
            assert all((k // 8) % world == r for k in o)             # VOL_SLAB = 8 layers dealt round-robin
    sys.path.insert(0, ROOT)
    import bench
    assert bench.whole_job_value(1000, 10, 2, 5.0) == 2 * 1000 * 10 / 5e-3      # replicas: every rank fuses a scan of its own
    assert bench.whole_job_value(1000, 10, 1, 5.0) == 1000 * 10 / 5e-3          # --shard: ONE scan, whatever the number of ranks
    args = bench.parse(["--gpus", "2", "--shard"])
    assert args.shard and args.shard_of is None and bench.parse(["--shard-of", "1,4"]).shard_of == "1,4"


def test_shard_layers_rejects_bad_arguments():
    import paper_1602_06645_b200 as vf
    L = vf.lib()
    assert L.vol_shard_layers(0, 0, 1, None, 0) == vf.VOL_E_ARG
    assert L.vol_shard_layers(8, 2, 2, None, 0) == vf.VOL_E_ARG
    assert list(vf.shard_layers(20, 0, 1)) == list(range(20))
    assert list(vf.shard_layers(20, 1, 2)) == [8, 9, 10, 11, 12, 13, 14, 15]

"""Multi-GPU path: windows are independent (Eq. 2), so the op shards by
contiguous window ranges with NO collective.  Host-side logic tested here with 2 gloo ranks on CPU:
each rank takes its shard (workloads.shard_windows), the shards tile the scene exactly, are balanced by
voxel count, and the oracle evaluated per shard reproduces the unsharded result bit for bit (which is what
makes the no-collective design correct)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2401_00912_b200 import workloads as wl
from oracle import sla_oracle


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
    sc = wl.make_scene(wl.lengths_config0(), 2, 16, "f32", seed=31)
    shards = wl.shard_windows(sc.lengths, world)
    w0, w1 = shards[rank]
    off = sc.offsets
    r0, r1 = int(off[w0]), int(off[w1])
    qq, kk, vv = sc.tensor("q"), sc.tensor("k"), sc.tensor("v")
    local_off = (off[w0:w1 + 1] - off[w0]).astype(np.int32)
    out_local = sla_oracle.forward(qq[r0:r1], kk[r0:r1], vv[r0:r1], local_off)
    # only bookkeeping crosses ranks (row counts), never tensor data of the op
    rows = torch.tensor([r1 - r0], dtype=torch.int64)
    allrows = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(allrows, rows)
    q.put((rank, w0, w1, r0, r1, out_local, [int(t.item()) for t in allrows]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_window_sharding_needs_no_collective():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    sc = wl.make_scene(wl.lengths_config0(), 2, 16, "f32", seed=31)
    full = sla_oracle.forward(sc.tensor("q"), sc.tensor("k"), sc.tensor("v"), sc.offsets)
    assert res[0][1] == 0 and res[-1][2] == sc.W and res[0][2] == res[1][1]       # shards tile the windows
    assert sum(res[0][6]) == sc.N
    assert abs(res[0][6][0] - res[0][6][1]) <= 2 * int(sc.lengths.max())             # balanced by voxels
    for _, w0, w1, r0, r1, out_local, _ in res:
        assert np.array_equal(out_local, full[r0:r1])                              # bit-identical


def test_shard_windows_properties():
    for c in (1, 3):
        ln = wl.make_config(c).lengths
        for world in (1, 2, 4, 8):
            sh = wl.shard_windows(ln, world)
            assert sh[0][0] == 0 and sh[-1][1] == len(ln)
            assert all(sh[i][1] == sh[i + 1][0] for i in range(world - 1))
            off = np.concatenate([[0], np.cumsum(ln)])
            rows = [int(off[b] - off[a]) for a, b in sh]
            assert sum(rows) == int(ln.sum())
            assert max(rows) - min(rows) <= 2 * int(ln.max())

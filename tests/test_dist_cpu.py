"""N > 1 host logic on CPU: world_size 2, gloo backend, 127.0.0.1 rendezvous.

The path shards by (sequence, KV-head group) with no data-path collective: each rank runs the
whole decode step on its own KV heads; the only exchange a tensor-parallel deployment needs is an all-gather of the
[B][Hq][D] outputs.  Here each rank computes its shard with the CPU oracle (no GPU in this tier), the shards are
all-gathered with torch.distributed and must reproduce the unsharded result exactly; the timing reduction used by
bench.py (max over ranks) is checked on the same process group.
"""
import math
import os
import socket

import numpy as np
import pytest

from paper_2606_31519_b200 import dist as rdist
from paper_2606_31519_b200 import synth


def test_shard_ranges_cover_without_overlap():
    for n in (0, 1, 7, 8, 13):
        for world in (1, 2, 3, 8):
            got = [rdist.shard_range(n, r, world) for r in range(world)]
            assert got[0][0] == 0 and got[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(got, got[1:]))
            sizes = [hi - lo for lo, hi in got]
            assert max(sizes) - min(sizes) <= 1
    (g0, g1), (h0, h1) = rdist.kv_head_shard(8, 32, 1, 2)
    assert (g0, g1, h0, h1) == (4, 8, 16, 32)
    with pytest.raises(ValueError):
        rdist.shard_range(4, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, ret):
    import torch
    import torch.distributed as dist
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from oracle import rbq_oracle as orc
    orc.build()
    r, _, w_ = rdist.init_process_group("gloo")
    assert (r, w_) == (rank, world)
    w = synth.make_workload(1, L=1200)
    rot, _ = orc.rotation_from_gaussian(w.rot_gauss)
    sm = 1.0 / math.sqrt(w.D)
    (g0, g1), (h0, h1) = rdist.kv_head_shard(w.Hkv, w.Hq, rank, world)
    K, V, q = (np.ascontiguousarray(w.K[:, g0:g1]), np.ascontiguousarray(w.V[:, g0:g1]), np.ascontiguousarray(w.q[:, h0:h1]))
    c_k = orc.centroid(K, w.seq_lens)
    codes, f_scale, _ = orc.encode(K, np.zeros_like(w.seq_lens), w.seq_lens, orc.ROT_DENSE, rot, c_k)
    ref = orc.decode_step(q, K, V, codes, f_scale, None, c_k, None, w.seq_lens, w.seq_lens, orc.ROT_DENSE, rot, w.p, sm)
    mine = torch.from_numpy(np.ascontiguousarray(ref["out"], dtype=np.float32))
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)                                    # the one exchange of the sharded path
    full = torch.cat(parts, dim=1).numpy()
    t = rdist.max_over_ranks(10.0 + rank)                           # bench.py's timing reduction
    s = rdist.sum_over_ranks(1.0)
    rdist.barrier()
    if rank == 0:
        ret["full"], ret["t"], ret["s"] = full, t, s
    dist.destroy_process_group()


def test_kv_head_sharding_world2_gloo(orc):
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, port, ret), nprocs=world, join=True)
    assert ret["t"] == 11.0 and ret["s"] == 2.0
    w = synth.make_workload(1, L=1200)
    rot, _ = orc.rotation_from_gaussian(w.rot_gauss)
    c_k = orc.centroid(w.K, w.seq_lens)
    codes, f_scale, _ = orc.encode(w.K, np.zeros_like(w.seq_lens), w.seq_lens, orc.ROT_DENSE, rot, c_k)
    ref = orc.decode_step(w.q, w.K, w.V, codes, f_scale, None, c_k, None, w.seq_lens, w.seq_lens, orc.ROT_DENSE, rot,
                          w.p, 1.0 / math.sqrt(w.D))
    assert np.array_equal(ret["full"], ref["out"].astype(np.float32)), "sharded + all-gathered output != unsharded"

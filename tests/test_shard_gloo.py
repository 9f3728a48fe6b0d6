"""The multi-GPU host logic on CPU: frame-range sharding over two ranks and the one exchange step
(all-reduce SUM of counts, all-reduce MIN of witness keys) with the gloo backend.  Per-rank partial
results come from the oracle here (no GPU in this test); the combination must equal the oracle's
result on the whole range."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as W
from paper_2606_15437_b200 import shard as sh

NONE_KEY = (1 << 63) - 1


def pack_keys(res, kn):
    """Test-side restatement of kripke_witness_to_keys (include/kripke.h)."""
    out = np.empty(len(res["wit_f"]), np.int64)
    for i, (f, v, w) in enumerate(zip(res["wit_f"].tolist(), res["wit_v"].tolist(), res["wit_w"].tolist())):
        out[i] = NONE_KEY if f == (1 << 64) - 1 else (((f << kn) | v) << 3) | w
    return out


def _worker(rank, world, port, n, k, cls, total, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import volume as V
    progs = W.corpus_c2(64)
    code, offs = W.pack_programs(progs)
    begin, count = sh.shard_range(total, rank, world)
    res = V.census(code, offs, n, k, cls, begin, count, threads=1)
    counts = torch.from_numpy(np.stack([res["models"], res["frames"]], 1).astype(np.int64))
    keys = torch.from_numpy(pack_keys(res, k * n))
    sh.combine(counts, keys)
    if rank == 0:
        out.put((counts.numpy().copy(), keys.numpy().copy()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("n,cls,total", [(3, 0, 512), (3, 1, 64), (4, 2, 355), (3, 3, 5)])
def test_two_rank_shards_combine_to_the_full_scan(vol, n, cls, total):
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n, 2, cls, total, out)) for r in range(2)]
    for p in procs:
        p.start()
    counts, keys = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    progs = W.corpus_c2(64)
    code, offs = W.pack_programs(progs)
    want = vol.census(code, offs, n, 2, cls)
    assert (counts[:, 0] == want["models"].astype(np.int64)).all()
    assert (counts[:, 1] == want["frames"].astype(np.int64)).all()
    assert (keys == pack_keys(want, 2 * n)).all()


def test_shard_ranges_tile_the_range():
    for total in (0, 1, 7, 52, 6942, 1 << 25):
        for world in (1, 2, 3, 8):
            pieces = [sh.shard_range(total, r, world) for r in range(world)]
            assert pieces[0][0] == 0 and sum(c for _, c in pieces) == total
            for (b0, c0), (b1, _) in zip(pieces, pieces[1:]):
                assert b0 + c0 == b1

"""N > 1 host logic on CPU: shard plan + the 24-byte exchange over gloo (world size 2), checked
against the oracle's global winner.  The per-shard partials are built from the oracle's
per-candidate outputs, so this test needs no GPU; the kernels' side of the same path is covered by
test_device_and_shard_paths_match_host_path (-m gpu)."""
import os
import struct
import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as W
from oracle.oracle import Oracle
from paper_1906_02318_b200.shard import shard_plan, gather_partials, decode_key


def _pack(safe, dist_f32, H, steps, index):
    primary = struct.unpack("<I", struct.pack("<f", dist_f32 * dist_f32))[0] if safe else H - steps
    return ((0 if safe else 1) << 62) | (primary << 30) | index


def test_shard_plan_partitions_the_index_space():
    for N, inc, world in [(10, 1, 3), (1 << 20, 1, 8), (7, 0, 2), (5, 1, 5), (3, 1, 4)]:
        seen = []
        for r in range(world):
            b, c = shard_plan(N, inc, world, r)
            seen += list(range(b, b + c))
        assert seen == list(range(N + inc))


def _worker(rank, world, port, ref, H, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    N = len(ref["steps_all"]) - 1
    b, c = shard_plan(N, 1, world, rank)
    keys = [_pack(ref["steps_all"][i] == H, np.float32(ref["dist_all"][i]), H, int(ref["steps_all"][i]), i)
            for i in range(b, b + c)]
    part = torch.tensor([min(keys), int((ref["steps_all"][b:b + c] == H).sum()),
                         int(np.minimum(ref["steps_all"][b:b + c] + 1, H).sum())], dtype=torch.int64)
    allp = gather_partials(part, world).view(world, 3)
    key = int(allp[:, 0].min()); n_safe = int(allp[:, 1].sum()); n_exec = int(allp[:, 2].sum())
    out[rank] = (decode_key(key), n_safe, n_exec)
    dist.destroy_process_group()


def test_two_rank_exchange_matches_global_winner():
    w = W.make("C2", N=777)
    o = Oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 2)
    for x0, uu, t in zip(x0s, uus, ticks):
        ref = o.step(x0, uu, int(t), detail=True)
        small = {k: ref[k] for k in ("steps_all", "dist_all")}
        mgr = mp.Manager(); out = mgr.dict()
        port = 29500 + (os.getpid() % 2000) + int(t)
        mp.spawn(_worker, args=(2, port, small, w.H, out), nprocs=2, join=True)
        for r in range(2):
            (unsafe, primary, index), n_safe, n_exec = out[r]
            assert index == ref["index"] and (1 - unsafe) == ref["safe"]
            assert n_safe == ref["n_safe"] and n_exec == ref["n_exec"]

"""world_size-2 gloo test (CPU) of the N > 1 path: replicas only, no data-path collective
(DESIGN.md §8).  Each rank plans its own conversations; ranks meet only to take the max of
their step times and the sum of their work."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_01839_b200 import binding as B
from paper_2606_01839_b200 import build as libbuild
from paper_2606_01839_b200 import replicas, synth


def _worker(rank, world, port, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(replicas.rank_seed(1, rank))
    kv = synth.uniform_lengths(rng, 64, 1024, 8192)
    plan = B.Plan(B.attn_shape(32, 8, 128), [1] * 64, kv)          # host-only plan: no GPU needed
    items, wb = plan.decode_items()
    blocks = int((items[:, 3] - items[:, 2]).sum())
    local_bytes = float(kv.sum()) * 8 * 128 * 2 * 2
    assert blocks == int(sum(synth.blocks_for(t) for t in kv)) * 8  # this rank's plan covers exactly its own KV
    ms, total = replicas.aggregate(dist, 0.2 + 0.05 * rank, local_bytes)
    ret[rank] = (ms, total, local_bytes, int(kv[0]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_share_nothing_but_the_clock():
    libbuild.build_library()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.get_context("spawn").Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    (ms0, tot0, b0, k0), (ms1, tot1, b1, k1) = ret[0], ret[1]
    assert ms0 == ms1 == 0.25                       # max over ranks
    assert tot0 == tot1 == b0 + b1                  # whole-job work
    assert k0 != k1                                 # different conversations per replica


def test_placement_replay_balances_decoders():
    # lowest active occupancy wins; a full decoder is skipped
    need = [10, 10, 10, 30, 5, 5, 100, 1]
    got = replicas.bind_conversations(need, pool_blocks=60, world=2)
    assert got == [0, 1, 0, 1, 0, 0, -1, 0]
    assert replicas.aggregate(None, 1.5, 7.0) == (1.5, 7.0)

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


FAKE = 1 << 40          # a 128-byte aligned "device" address: the allocator and tickets are host-only


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
    # lowest active occupancy wins; a full decoder is skipped.  The replay goes through
    # csv_place / kv_alloc_blocks on real pool handles (host-only pools over a fake device address).
    need = [10, 10, 10, 30, 5, 5, 100, 1]
    pools = [B.KvPool(B.pool_desc(1, 60, 8, 128), FAKE, 1 << 40) for _ in range(2)]
    where, tables = replicas.bind_conversations(need, pools)
    assert where == [0, 1, 0, 1, 0, 0, -1, 0]
    assert [None if t is None else len(t) for t in tables] == [10, 10, 10, 30, 5, 5, None, 1]
    assert [p.used_blocks for p in pools] == [31, 40]
    # unequal decoders: occupancy is the RATIO used / total (S17), not the block count
    pools = [B.KvPool(B.pool_desc(1, 100, 8, 128), FAKE, 1 << 40), B.KvPool(B.pool_desc(1, 20, 8, 128), FAKE, 1 << 40)]
    where, _ = replicas.bind_conversations([10, 1, 1, 1], pools)
    assert where == [0, 1, 1, 0]            # 10/100 vs 0/20 -> 1; 10 % vs 5 % -> 1; 10 % vs 10 % tie -> 0
    assert replicas.aggregate(None, 1.5, 7.0) == (1.5, 7.0)




def _handoff_worker(rank, world, port, ret):
    """rank 0 = prefiller, ranks 1.. = decoders.  Host side of the cross-GPU handoff: the router's
    placement (csv_place), block allocation on the bound decoder, the ticket's trip to the prefiller."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    desc = B.pool_desc(2, 64, 8, 128)
    if rank == 0:
        got = [replicas.recv_ticket(dist, 1) for _ in range(3)]
        ret[0] = got
    else:
        pool = B.KvPool(desc, FAKE, B.kv_pool_bytes(desc))
        pool.set_free_order(np.arange(63, -1, -1))
        export = (bytes(range(64)), 8192)                  # stands in for csv_ipc_export (needs a GPU)
        t1 = replicas.handoff_ticket(pool, 300, export=export, decoder=1)
        t2 = replicas.handoff_ticket(pool, 5, 11, export=export, decoder=1)
        t3 = replicas.handoff_ticket(pool, 20, 300, ids=t1["ids"] + list(pool.alloc_blocks(1)), export=export, decoder=1)
        for t in (t1, t2, t3):
            replicas.send_ticket(dist, t, 0)
        try:
            replicas.handoff_ticket(pool, 16 * 64)         # more than the pool has left: all-or-nothing
            full = False
        except B.CsvError as e:
            full = e.code == B.CSV_E_NOMEM
        ret[1] = (pool.used_blocks, full)
    dist.barrier()
    dist.destroy_process_group()


def test_handoff_tickets_travel_from_decoder_to_prefiller():
    libbuild.build_library()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.get_context("spawn").Manager()
    ret = mgr.dict()
    mp.spawn(_handoff_worker, args=(2, port, ret), nprocs=2, join=True)
    t1, t2, t3 = ret[0]
    assert t1["ids"] == list(range(63, 44, -1)) and t1["tokens"] == 300 and t1["token_offset"] == 0   # 19 blocks, free order
    assert t2["ids"] == [44] and t2["token_offset"] == 11
    assert t3["ids"] == t1["ids"] + [43] and t3["token_offset"] == 300
    assert t1["shape"] == (2, 64, 8, 128) and t1["handle"] == bytes(range(64)) and t1["offset"] == 8192
    assert ret[1] == (21, True)                            # occupancy the placement rule reads; the failed ticket took nothing
    pools = replicas.PeerPools()
    try:
        pools.get({"decoder": 0, "handle": None, "offset": 0, "shape": (1, 1, 1, 64)})
        assert False
    except ValueError:
        pass


def _p2p_failure_worker(rank, world, port, ret, who_fails):
    """handoff_p2p.run on a box without a GPU: one side fails on its first CUDA call.  Both ranks must leave run()
    (the decoder with an error record) and still be in step for the collectives that follow it in bench.py."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2606_01839_b200 import handoff_p2p

    if who_fails == "prefiller":   # the decoder's offer succeeds (stand-in, no GPU); the prefiller then dies in its push
        handoff_p2p._decoder_offer = lambda st, *a: {"tickets": [], "stagings": [], "stagings2": []}
    out = handoff_p2p.run(dist, rank, tokens=64, layers=1, convs=2, iters=1)
    box = [out if rank == 1 else None]
    dist.broadcast_object_list(box, src=1)             # what bench.py does next: every rank must arrive here
    ret[rank] = box[0]
    dist.barrier()
    dist.destroy_process_group()


def test_p2p_leg_failure_on_either_side_does_not_hang_the_ranks():
    # an exception on one rank inside handoff_p2p.run left the other rank waiting in a different collective.
    libbuild.build_library()
    for who in ("decoder", "prefiller"):
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        mgr = mp.get_context("spawn").Manager()
        ret = mgr.dict()
        mp.spawn(_p2p_failure_worker, args=(2, port, ret, who), nprocs=2, join=True)
        assert ret[0] == ret[1] and "error" in ret[0], ret[0]
        assert ret[0]["error"].startswith(who), ret[0]["error"]


def test_bench_launches_its_own_ranks_when_torchrun_did_not():
    # `python bench.py --gpus 2` with no WORLD_SIZE in the environment must become two ranks on its own (a plain
    # --gpus N run measured one replica).  The reference arm runs without a GPU: rank 0 times the oracle, rank 1 exits 0.
    import json
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], cwd=root, env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, lines                      # rank 0 alone prints
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["n_gpus"] == 2 and out["value"] > 0
    assert out["cpu_baseline"]["kind"] == "oracle" and out["e2e"]["h2d_bytes_per_step"] == 0

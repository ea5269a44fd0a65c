"""The paper's one exchange step across two processes / two GPUs (§4 "the resulting KV
cache is transferred once to the bound decoder"; PAPER.md:96 / Fig. 3: the transfer is the cost disaggregation adds).

    python -m torch.distributed.run --nnodes=1 --nproc-per-node 2 --master-addr 127.0.0.1 --master-port 29611 \
        -m paper_2606_01839_b200.handoff_p2p [--tokens 8192] [--layers 32] [--convs 4]

rank 0 = prefiller (owns the turn-1 K/V, token-major), rank 1 = decoder (owns the paged pool and its allocator).
Each rank uses GPU `LOCAL_RANK % device_count`: with two GPUs the stores cross NVLink, with one GPU (this box) the two
processes share it and the same code path runs through a CUDA IPC mapping of the decoder's pool.  Two routes are timed:
  direct  kv_handoff_direct_batch on the prefiller pushes straight into the decoder's pool (one kernel, no staging);
  staged  kv_pack_batch on the prefiller writes the messages into staging buffers that live on the DECODER (peer
          mapped), then the decoder runs kv_unpack_batch locally: the NCCL-free form of "send the message, then scatter".
The decoder checks both pools bit for bit against a local kv_handoff_direct of the same seeded K/V (device RNG with
the same seed gives the same bits on both ranks).  Control messages (tickets, done flags) go through torch.distributed
object collectives (gloo: they are host data).  Prints one JSON line on rank 1.
"""
import argparse
import json
import os

import numpy as np
import torch
import torch.distributed as dist

from . import binding as B
from . import replicas, synth


def seeded_kv(seed, NL, tokens, Hkv, d):
    gen = torch.Generator(device="cuda")
    gen.manual_seed(seed)
    n = NL * tokens * Hkv * d
    k = torch.randint(-32768, 32767, (n,), dtype=torch.int16, device="cuda", generator=gen)
    v = torch.randint(-32768, 32767, (n,), dtype=torch.int16, device="cuda", generator=gen)
    return k, v


def event_ms(fn, stream=None):
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--tokens", type=int, default=8192)
    ap.add_argument("--layers", type=int, default=32)
    ap.add_argument("--convs", type=int, default=4)
    ap.add_argument("--iters", type=int, default=3)
    args = ap.parse_args()
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world != 2:
        raise SystemExit("handoff_p2p needs exactly two ranks (prefiller, decoder)")
    ngpu = torch.cuda.device_count()
    dev = int(os.environ.get("LOCAL_RANK", str(rank))) % ngpu
    torch.cuda.set_device(dev)
    dist.init_process_group("gloo")          # control plane only: tickets and flags are host objects
    NL, Hkv, d = args.layers, 8, 128
    toks = [max(16, args.tokens - 37 * i) for i in range(args.convs)]        # ragged last blocks
    desc_blocks = synth.pool_blocks_for(toks, slack=0.10)
    desc = B.pool_desc(NL, desc_blocks, Hkv, d)
    payload = sum(toks) * NL * Hkv * d * 2 * 2

    if rank == 1:
        # ---------------- decoder ----------------
        rng = np.random.default_rng(5)
        pools, mems = [], []
        for _ in range(3):                  # [0] direct target, [1] staged target, [2] local reference
            mem = torch.zeros(B.kv_pool_bytes(desc) // 2, dtype=torch.int16, device="cuda")
            pool = B.KvPool(desc, mem)
            pool.set_free_order(synth.shuffled_free_order(np.random.default_rng(5), desc_blocks))
            pools.append(pool)
            mems.append(mem)
        stagings = [torch.zeros(B.kv_staging_bytes(desc, t) // 2, dtype=torch.int16, device="cuda") for t in toks]
        tickets = [replicas.handoff_ticket(pools[0], t, export=B.csv_ipc_export(mems[0]), decoder=1) for t in toks]
        ids = [np.asarray(tk["ids"], dtype=np.int32) for tk in tickets]
        for p in pools[1:]:
            for t in toks:
                p.alloc_blocks(synth.blocks_for(t))                           # same free order -> same ids
        torch.cuda.synchronize()
        dist.broadcast_object_list([{"tickets": tickets, "stagings": [B.csv_ipc_export(s) for s in stagings]}], src=1)
        res = [None]
        dist.broadcast_object_list(res, src=0)                                # prefiller: both routes written
        d_ids = [torch.from_numpy(i).cuda() for i in ids]
        nids = [len(i) for i in ids]
        unpack_ms = event_ms(lambda: B.kv_unpack_batch(pools[1], stagings, toks, [0] * len(toks), d_ids, nids))
        ks, vs = zip(*[seeded_kv(100 + i, NL, t, Hkv, d) for i, t in enumerate(toks)])
        B.kv_handoff_direct_batch(pools[2], list(ks), list(vs), toks, [0] * len(toks), d_ids, nids)
        torch.cuda.synchronize()
        ok_direct = bool(torch.equal(mems[0], mems[2]))
        ok_staged = bool(torch.equal(mems[1], mems[2]))
        r0 = res[0]
        same_gpu = ngpu < 2
        out = {"what": "prefiller -> decoder KV handoff across two processes", "gpus": min(ngpu, 2), "same_gpu": same_gpu,
               "convs": len(toks), "tokens": toks, "layers": NL, "payload_gb": payload / 1e9,
               "direct_ms": r0["direct_ms"], "direct_payload_gbs": payload / r0["direct_ms"] / 1e6,
               "staged_pack_to_peer_ms": r0["pack_ms"], "staged_unpack_ms": unpack_ms,
               "staged_payload_gbs": payload / (r0["pack_ms"] + unpack_ms) / 1e6,
               "bit_exact_direct": ok_direct, "bit_exact_staged": ok_staged,
               "bound": "HBM (both processes on one GPU)" if same_gpu else "NVLink 5, 900 GB/s per direction"}
        print(json.dumps(out), flush=True)
        dist.barrier()
        if not (ok_direct and ok_staged):
            raise SystemExit(1)
    else:
        # ---------------- prefiller ----------------
        box = [None]
        dist.broadcast_object_list(box, src=1)
        tickets, st_exports = box[0]["tickets"], box[0]["stagings"]
        ks, vs = zip(*[seeded_kv(100 + i, NL, t, Hkv, d) for i, t in enumerate(toks)])
        ks, vs = list(ks), list(vs)
        peers = replicas.PeerPools()
        pool = peers.get(tickets[0])                                           # one mapping for the decoder's pool
        d_ids = [torch.tensor(tk["ids"], dtype=torch.int32, device="cuda") for tk in tickets]
        nids = [len(tk["ids"]) for tk in tickets]
        offs = [0] * len(toks)
        direct = lambda: B.kv_handoff_direct_batch(pool, ks, vs, toks, offs, d_ids, nids)
        direct()
        torch.cuda.synchronize()
        direct_ms = min(event_ms(direct) for _ in range(args.iters))
        peer_st = [B.csv_ipc_open(h, off) for h, off in st_exports]
        pack = lambda: B.kv_pack_batch(desc, ks, vs, toks, offs, peer_st)
        pack()
        torch.cuda.synchronize()
        pack_ms = min(event_ms(pack) for _ in range(args.iters))
        torch.cuda.synchronize()
        dist.broadcast_object_list([{"direct_ms": direct_ms, "pack_ms": pack_ms}], src=0)
        dist.barrier()                                                         # the decoder has read everything
        for p in peer_st:
            B.csv_ipc_close(p)
        peers.close()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()

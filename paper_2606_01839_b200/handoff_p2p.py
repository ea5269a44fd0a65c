"""The paper's one exchange step across two processes / two GPUs (§4 "the resulting KV
cache is transferred once to the bound decoder"; PAPER.md:96 / Fig. 3: the transfer is the cost disaggregation adds).

    python -m torch.distributed.run --nnodes=1 --nproc-per-node 2 --master-addr 127.0.0.1 --master-port 29611 \
        -m paper_2606_01839_b200.handoff_p2p [--tokens 8192] [--layers 32] [--convs 4]

rank 0 = prefiller (owns the turn-1 K/V, token-major), rank 1 = decoder (owns the paged pool and its allocator).
Each rank uses GPU `LOCAL_RANK % device_count`: with two GPUs the stores cross NVLink, with one GPU (this box) the two
processes share it and the same code path runs through a CUDA IPC mapping of the decoder's pool.  Three routes are timed
(see run()): the direct push, the staged route (pack straight into peer-mapped staging, local unpack) and the copy-engine
route (local pack, cudaMemcpyAsync of the message to the peer, local unpack: SURVEY NEXT-1's comparison arm).
The decoder checks every pool bit for bit against a local kv_handoff_direct of the same seeded K/V (device RNG with
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


def run(dist, rank, tokens=8192, layers=32, convs=4, iters=3, prefiller=0, decoder=1):
    """The two-rank handoff program under an EXISTING process group (bench.py calls it on ranks 0 and 1 when two devices
    are visible; every other rank passes through).  Three routes are timed, each bit-exact-checked on the decoder:
      direct  kv_handoff_direct_batch on the prefiller pushes straight into the decoder's pool (one kernel, no staging);
      staged  kv_pack_batch on the prefiller writes the messages into staging buffers that live on the DECODER (peer
              mapped), then the decoder runs kv_unpack_batch locally;
      copy    kv_pack_batch into LOCAL staging, csv_ipc_copy (cudaMemcpyAsync, the copy engine) of each message into the
              decoder's staging, then the local kv_unpack_batch: SURVEY NEXT-1's cudaMemcpyPeerAsync comparison.
    Returns the record on the decoder rank, None elsewhere."""
    grp = dist.new_group([prefiller, decoder]) if dist.get_world_size() > 2 else None   # collective: every rank calls it
    if rank not in (prefiller, decoder):
        return None
    # Failure safety: the two ranks always exchange the same three messages in the same order (decoder's offer, prefiller's
    # result, barrier), whatever happens in between.  A side that fails sends {"error": ...} in place of its message, so
    # the other side never waits in a collective its peer will not enter, and both return (the decoder with the error
    # record) instead of hanging the job.
    bcast = lambda box, src: dist.broadcast_object_list(box, src=src, group=grp)
    if rank == decoder:
        st = {}
        try:
            offer = _decoder_offer(st, tokens, layers, convs, decoder)
        except Exception as e:
            offer = {"error": "decoder: %r" % (e,)}
        bcast([offer], decoder)
        res = [None]
        bcast(res, prefiller)                                                 # prefiller: every route written (or its error)
        err = offer.get("error") or (res[0] or {}).get("error")
        if err:
            out = {"what": "prefiller -> decoder KV handoff across two processes", "error": err[:300]}
        else:
            try:
                out = _decoder_check(st, res[0])
            except Exception as e:
                out = {"what": "prefiller -> decoder KV handoff across two processes", "error": ("decoder: %r" % (e,))[:300]}
        dist.barrier(group=grp)
        return out
    box, opened, peers = [None], [], replicas.PeerPools()
    bcast(box, decoder)
    try:
        if "error" in box[0]:
            raise RuntimeError(box[0]["error"])
        result = _prefiller_push(box[0], peers, opened, tokens, layers, convs, iters)
    except Exception as e:
        result = {"error": str(e) if "error" in (box[0] or {}) else "prefiller: %r" % (e,)}
    bcast([result], prefiller)
    dist.barrier(group=grp)                                                    # the decoder has read everything
    try:
        for p in opened:
            B.csv_ipc_close(p)
        peers.close()
    except Exception:
        pass
    return None


def _shape(tokens, layers, convs):
    NL, Hkv, d = layers, 8, 128
    toks = [max(16, tokens - 37 * i) for i in range(convs)]        # ragged last blocks
    desc_blocks = synth.pool_blocks_for(toks, slack=0.10)
    return NL, Hkv, d, toks, desc_blocks, B.pool_desc(NL, desc_blocks, Hkv, d)


def _decoder_offer(st, tokens, layers, convs, decoder):
    """Decoder, before the push: four pools over one free order, two staging sets, the tickets.  Returns the offer message."""
    NL, Hkv, d, toks, desc_blocks, desc = _shape(tokens, layers, convs)
    pools, mems = [], []
    for _ in range(4):                  # [0] direct target, [1] staged target, [2] local reference, [3] copy target
        mem = torch.zeros(B.kv_pool_bytes(desc) // 2, dtype=torch.int16, device="cuda")
        pool = B.KvPool(desc, mem)
        pool.set_free_order(synth.shuffled_free_order(np.random.default_rng(5), desc_blocks))
        pools.append(pool)
        mems.append(mem)
    stagings = [torch.zeros(B.kv_staging_bytes(desc, t) // 2, dtype=torch.int16, device="cuda") for t in toks]
    stagings2 = [torch.zeros(B.kv_staging_bytes(desc, t) // 2, dtype=torch.int16, device="cuda") for t in toks]
    tickets = [replicas.handoff_ticket(pools[0], t, export=B.csv_ipc_export(mems[0]), decoder=decoder) for t in toks]
    for p in pools[1:]:
        for t in toks:
            p.alloc_blocks(synth.blocks_for(t))                           # same free order -> same ids
    torch.cuda.synchronize()
    st.update(pools=pools, mems=mems, stagings=stagings, stagings2=stagings2, tickets=tickets, shape=(NL, Hkv, d, toks))
    return {"tickets": tickets, "stagings": [B.csv_ipc_export(s) for s in stagings],
            "stagings2": [B.csv_ipc_export(s) for s in stagings2]}


def _decoder_check(st, r0):
    """Decoder, after the push: local unpacks of the two staged routes, a local reference push, bit-for-bit comparison."""
    NL, Hkv, d, toks = st["shape"]
    pools, mems, stagings, stagings2 = st["pools"], st["mems"], st["stagings"], st["stagings2"]
    ngpu = torch.cuda.device_count()
    payload = sum(toks) * NL * Hkv * d * 2 * 2
    ids = [np.asarray(tk["ids"], dtype=np.int32) for tk in st["tickets"]]
    d_ids = [torch.from_numpy(i).cuda() for i in ids]
    nids = [len(i) for i in ids]
    unpack_ms = event_ms(lambda: B.kv_unpack_batch(pools[1], stagings, toks, [0] * len(toks), d_ids, nids))
    B.kv_unpack_batch(pools[3], stagings2, toks, [0] * len(toks), d_ids, nids)
    ks, vs = zip(*[seeded_kv(100 + i, NL, t, Hkv, d) for i, t in enumerate(toks)])
    B.kv_handoff_direct_batch(pools[2], list(ks), list(vs), toks, [0] * len(toks), d_ids, nids)
    torch.cuda.synchronize()
    ok_direct = bool(torch.equal(mems[0], mems[2]))
    ok_staged = bool(torch.equal(mems[1], mems[2]))
    ok_copy = bool(torch.equal(mems[3], mems[2]))
    same_gpu = r0["prefiller_device"] == torch.cuda.current_device() or ngpu < 2
    out = {"what": "prefiller -> decoder KV handoff across two processes", "gpus": 1 if same_gpu else 2, "same_gpu": same_gpu,
           "convs": len(toks), "tokens": toks, "layers": NL, "payload_gb": payload / 1e9,
           "direct_ms": r0["direct_ms"], "direct_payload_gbs": payload / r0["direct_ms"] / 1e6,
           "staged_pack_to_peer_ms": r0["pack_ms"], "staged_unpack_ms": unpack_ms,
           "staged_payload_gbs": payload / (r0["pack_ms"] + unpack_ms) / 1e6,
           "copy_pack_local_ms": r0["pack_local_ms"], "copy_memcpy_peer_ms": r0["copy_ms"],
           "copy_payload_gbs": payload / (r0["pack_local_ms"] + r0["copy_ms"] + unpack_ms) / 1e6,
           "memcpy_peer_gbs": payload / r0["copy_ms"] / 1e6,
           "bit_exact_direct": ok_direct, "bit_exact_staged": ok_staged, "bit_exact_copy": ok_copy,
           "bound": "HBM (both processes on one GPU)" if same_gpu else
                    "NVLink 5: 900 GB/s per direction nominal, 770 GB/s measured peer copy (B200_PROFILING.md)"}
    if not same_gpu:
        out["direct_frac_of_measured_peer_copy_770"] = out["direct_payload_gbs"] / 770.0
    return out


def _prefiller_push(offer, peers, opened, tokens, layers, convs, iters):
    """Prefiller: the three routes, each warmed once and timed `iters` times.  Every csv_ipc_open mapping is appended to
    `opened` as soon as it exists so that the caller can close it whatever happens later."""
    NL, Hkv, d, toks, _, desc = _shape(tokens, layers, convs)
    tickets, st_exports, st2_exports = offer["tickets"], offer["stagings"], offer["stagings2"]
    ks, vs = zip(*[seeded_kv(100 + i, NL, t, Hkv, d) for i, t in enumerate(toks)])
    ks, vs = list(ks), list(vs)
    pool = peers.get(tickets[0])                                           # one mapping for the decoder's pool
    for tk in tickets:
        replicas.validate_ticket(tk)                                       # ids crossed a process boundary (conserve_kv.h)
    d_ids = [torch.tensor(tk["ids"], dtype=torch.int32, device="cuda") for tk in tickets]
    nids = [len(tk["ids"]) for tk in tickets]
    offs = [0] * len(toks)
    direct = lambda: B.kv_handoff_direct_batch(pool, ks, vs, toks, offs, d_ids, nids)
    direct()
    torch.cuda.synchronize()
    direct_ms = min(event_ms(direct) for _ in range(iters))
    peer_st = []
    for h, off in st_exports:
        peer_st.append(B.csv_ipc_open(h, off))
        opened.append(peer_st[-1])
    pack = lambda: B.kv_pack_batch(desc, ks, vs, toks, offs, peer_st)
    pack()
    torch.cuda.synchronize()
    pack_ms = min(event_ms(pack) for _ in range(iters))
    # copy-engine route: pack locally, then one cudaMemcpyAsync per message into the decoder's second staging set
    peer_st2 = []
    for h, off in st2_exports:
        peer_st2.append(B.csv_ipc_open(h, off))
        opened.append(peer_st2[-1])
    local_st = [torch.zeros(B.kv_staging_bytes(desc, t) // 2, dtype=torch.int16, device="cuda") for t in toks]
    pack_local = lambda: B.kv_pack_batch(desc, ks, vs, toks, offs, local_st)
    pack_local()
    torch.cuda.synchronize()
    pack_local_ms = min(event_ms(pack_local) for _ in range(iters))
    copy = lambda: [B.csv_ipc_copy(dst, src, src.numel() * 2) for dst, src in zip(peer_st2, local_st)]
    copy()
    torch.cuda.synchronize()
    copy_ms = min(event_ms(copy) for _ in range(iters))
    torch.cuda.synchronize()
    return {"direct_ms": direct_ms, "pack_ms": pack_ms, "pack_local_ms": pack_local_ms, "copy_ms": copy_ms,
            "prefiller_device": torch.cuda.current_device()}


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
    out = run(dist, rank, args.tokens, args.layers, args.convs, args.iters)
    if out is not None:
        print(json.dumps(out), flush=True)
    dist.destroy_process_group()
    if out is not None and ("error" in out or not (out["bit_exact_direct"] and out["bit_exact_staged"] and out["bit_exact_copy"])):
        raise SystemExit(1)


if __name__ == "__main__":
    main()

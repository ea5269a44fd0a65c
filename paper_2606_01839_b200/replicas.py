"""Replica bookkeeping for N > 1 GPUs (replicas only, no data-path collective).

Conversations are independent units bound to one decoder for life, so N GPUs
are N pools and N independent tail steps.  The only cross-rank traffic is measurement: a barrier
and two scalar reductions (max time, summed work).  Works on any torch.distributed backend
(nccl on GPUs; gloo in the CPU tests).
"""
import torch


def rank_seed(base_seed, rank):
    """Every replica serves its own conversations: same length recipe, different seed."""
    return int(base_seed) + 100 * int(rank)


def bind_conversations(need_blocks, pools):
    """Replay of an arrival sequence through the library's placement call: each arriving
    conversation is bound by csv_place to one of `pools` (binding.KvPool handles, one per decoder) and its blocks are
    allocated there, for life.  Returns (decoder index per conversation, -1 = nobody fits; block ids per conversation).
    No placement arithmetic here: the rule lives in csv_place."""
    from . import binding as B

    where, tables = [], []
    for need in need_blocks:
        try:
            k = B.csv_place(pools, int(need))
        except B.CsvError as e:
            if e.code != B.CSV_E_NOMEM:
                raise
            where.append(-1)
            tables.append(None)
            continue
        where.append(k)
        tables.append(pools[k].alloc_blocks(int(need)))
    return where, tables


def aggregate(dist, local_ms, local_units, device="cpu"):
    """(max over ranks of the step time, sum over ranks of the units) -> whole-job rate inputs."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(local_ms), float(local_units)
    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ---------------- cross-GPU one-shot handoff ("transferred once to the bound decoder") ------
# Protocol, one process per GPU:  the DECODER owns its pool and allocator; it allocates the conversation's blocks and
# sends a ticket (plain host data: shape, block ids, the IPC handle of the pool's allocation).  The PREFILLER maps the
# pool once per decoder, wraps it in a kv_pool_t and pushes the conversation with kv_handoff_direct: its stores cross
# NVLink, nothing is staged or loaded from the peer.  It then tells the decoder (any message after a stream sync).

def handoff_ticket(pool, tokens, token_offset=0, ids=None, export=None, decoder=0):
    """Decoder side.  pool: binding.KvPool.  Allocates ceil((offset + tokens) / 16) blocks unless the conversation's
    table `ids` is given (a later push into blocks it already owns).  export: (handle, offset) from
    binding.csv_ipc_export(pool memory), or None when prefiller and decoder share a process.  All-or-nothing."""
    from . import binding as B

    if tokens <= 0 or token_offset < 0:
        raise ValueError("tokens must be > 0 and token_offset >= 0")
    need = (token_offset + tokens + B.BLOCK - 1) // B.BLOCK
    if ids is None:
        ids = pool.alloc_blocks(need)                      # raises CsvError(CSV_E_NOMEM) and changes nothing if short
    if len(ids) < need:
        raise ValueError("table shorter than ceil((offset + tokens) / 16)")
    d = pool.desc
    return {"decoder": int(decoder), "tokens": int(tokens), "token_offset": int(token_offset),
            "ids": [int(i) for i in ids],
            "shape": (int(d.num_layers), int(d.num_blocks), int(d.num_kv_heads), int(d.head_dim)),
            "handle": None if export is None else bytes(export[0]), "offset": 0 if export is None else int(export[1])}


def validate_ticket(ticket):
    """Prefiller side, before any launch that uses a ticket's ids.  The ids came over a channel and the kernels do not
    range-check them (conserve_kv.h): one bad id would be a silent out-of-bounds write into another process's allocation.
    Checks the table against the ticket's own shape; PeerPools.get bounds that shape by the mapped allocation."""
    ids, nb = ticket["ids"], int(ticket["shape"][1])
    need = (ticket["token_offset"] + ticket["tokens"] + 15) // 16
    if ticket["tokens"] <= 0 or ticket["token_offset"] < 0 or len(ids) < need:
        raise ValueError("ticket: table shorter than ceil((offset + tokens) / 16)")
    if any((not isinstance(i, int)) or i < 0 or i >= nb for i in ids) or len(set(ids)) != len(ids):
        raise ValueError("ticket: block ids must be unique and inside [0, num_blocks)")


def send_ticket(dist, ticket, dst):
    dist.send_object_list([ticket], dst=dst)


def recv_ticket(dist, src):
    box = [None]
    dist.recv_object_list(box, src=src)
    return box[0]


class PeerPools:
    """Prefiller side: one mapping + kv_pool_t wrapper per decoder pool, opened on first use."""

    def __init__(self):
        self._pools = {}

    def get(self, ticket, local_pool=None):
        from . import binding as B

        key = (ticket["decoder"], ticket["handle"], ticket["offset"])
        if key not in self._pools:
            NL, nb, Hkv, d = (int(x) for x in ticket["shape"])
            if local_pool is not None:      # the ticket's shape is only trusted as far as it matches what we hold
                ld = local_pool.desc
                if (ld.num_layers, ld.num_blocks, ld.num_kv_heads, ld.head_dim) != (NL, nb, Hkv, d):
                    raise ValueError("ticket shape does not match the local pool")
            desc = B.pool_desc(NL, nb, Hkv, d)
            if ticket["handle"] is None:
                if local_pool is None:
                    raise ValueError("ticket without an IPC handle needs the local pool")
                self._pools[key] = (local_pool, None)
            else:
                ptr = B.csv_ipc_open(ticket["handle"], ticket["offset"])
                # shape and offset arrived with the handle: the pool they describe must lie inside what was really mapped,
                # else a "valid" block id of an oversized descriptor is a store outside the decoder's allocation
                need = B.kv_pool_bytes(desc)
                try:
                    have = B.csv_ipc_mapped_bytes(ptr)
                    if need == 0 or need > have:
                        raise ValueError("ticket: a pool of shape %r needs %d bytes, the mapped allocation has %d after the "
                                         "offset" % ((NL, nb, Hkv, d), need, have))
                except Exception:
                    B.csv_ipc_close(ptr)
                    raise
                self._pools[key] = (B.KvPool(desc, ptr, need), ptr)
        return self._pools[key][0]

    def push(self, ticket, d_k, d_v, d_ids=None, stream=None, local_pool=None):
        """kv_handoff_direct of one conversation into the ticket's pool.  d_k, d_v: [NL][tokens][Hkv][d] bf16 device
        tensors of THIS process.  Returns the device id tensor used (keep it alive until the stream has passed)."""
        import torch
        from . import binding as B

        pool = self.get(ticket, local_pool)
        validate_ticket(ticket)
        if d_ids is None:
            d_ids = torch.tensor(ticket["ids"], dtype=torch.int32, device="cuda")
        B.kv_handoff_direct(pool, d_k, d_v, ticket["tokens"], ticket["token_offset"], d_ids, len(ticket["ids"]), stream)
        return d_ids

    def close(self):
        from . import binding as B

        for pool, ptr in self._pools.values():
            if ptr is not None:
                pool.destroy()
                B.csv_ipc_close(ptr)
        self._pools = {}

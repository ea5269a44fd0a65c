"""Device-resident synthetic workloads of BASELINE.json's configs (bench.py and the full-size
parity tests).  Plumbing only: random pool contents, block tables from the library's own
allocator with a shuffled free list, query tensors.  No attention arithmetic, no layout formula
(a pool filled with random bf16 bits is a valid KV cache whatever the in-tile format, because
the format is a bijection inside each tile).
"""
import numpy as np
import torch

from . import binding as B
from . import synth


def randn_bf16_bits(n_elems, gen, mean=0.0, chunk=1 << 27):
    """int16 CUDA tensor holding bf16 N(mean,1) bit patterns (generated in chunks to bound fp32 scratch)."""
    out = torch.empty(n_elems, dtype=torch.bfloat16, device="cuda")
    for s in range(0, n_elems, chunk):
        e = min(n_elems, s + chunk)
        out[s:e] = (torch.randn(e - s, device="cuda", generator=gen, dtype=torch.float32) + mean).to(torch.bfloat16)
    return out.view(torch.int16)


class TailWorkload:
    """A decoder pool holding `kv_lens` conversations + one step's queries (q_lens per conversation)."""

    def __init__(self, Hq, Hkv, d, q_lens, kv_lens, NL=1, seed=0, slack=0.10, mpt=0, v_mean=0.0, device_rank=0):
        self.Hq, self.Hkv, self.d, self.NL = Hq, Hkv, d, NL
        self.q_lens = [int(x) for x in q_lens]
        self.kv_lens = [int(x) for x in kv_lens]
        rng = np.random.default_rng(seed)
        gen = torch.Generator(device="cuda")
        gen.manual_seed(1000 + seed)
        self.num_blocks = synth.pool_blocks_for(self.kv_lens, slack=slack)
        self.desc = B.pool_desc(NL, self.num_blocks, Hkv, d)
        self.pool_bytes = B.kv_pool_bytes(self.desc)
        self.d_pool = randn_bf16_bits(self.pool_bytes // 2, gen, mean=v_mean)
        self.pool = B.KvPool(self.desc, self.d_pool)
        self.pool.set_free_order(synth.shuffled_free_order(rng, self.num_blocks))   # consecutive blocks never adjacent
        self.tables = [self.pool.alloc_blocks(synth.blocks_for(t)) for t in self.kv_lens]
        self.h_tables, self.max_blocks = synth.dense_tables(self.tables, pad=0)
        self.d_tables = torch.from_numpy(self.h_tables).cuda()
        self.shape = B.attn_shape(Hq, Hkv, d)
        self.mpt = mpt
        self._gen = gen
        self._setup_queries(self.q_lens)

    def _setup_queries(self, q_lens):
        Hq, Hkv, d, NL, gen = self.Hq, self.Hkv, self.d, self.NL, self._gen
        self.q_lens = [int(x) for x in q_lens]
        self.total_q = int(sum(self.q_lens))
        self.d_q = randn_bf16_bits(self.total_q * Hq * d, gen).view(self.total_q, Hq, d)
        self.d_k_new = randn_bf16_bits(NL * self.total_q * Hkv * d, gen)
        self.d_v_new = randn_bf16_bits(NL * self.total_q * Hkv * d, gen)
        self.d_out = torch.zeros((self.total_q, Hq, d), dtype=torch.int16, device="cuda")
        self.d_lse = torch.zeros((self.total_q, Hq), dtype=torch.float32, device="cuda")
        self.ws = torch.empty(max(128, B.csv_plan_workspace_bytes(self.shape, self.q_lens, self.kv_lens, self.mpt)),
                              dtype=torch.uint8, device="cuda")
        self.plan = B.Plan(self.shape, self.q_lens, self.kv_lens, self.mpt, self.ws)
        torch.cuda.synchronize()

    def with_q_lens(self, q_lens, kv_lens=None):
        """Another step over the SAME pool and tables (e.g. config 5's append call next to its decode call).
        kv_lens (optional) may shorten the conversations: the pool simply holds more than the step looks at."""
        import copy

        other = copy.copy(self)
        if kv_lens is not None:
            assert all(int(a) <= int(b) for a, b in zip(kv_lens, self.kv_lens))
            other.kv_lens = [int(x) for x in kv_lens]
        other._setup_queries(q_lens)
        return other

    def with_extra_chunks(self, convs, m):
        """One MIXED step over the same pool: every conversation keeps its decode row, and each conversation in `convs`
        also appends an m-token chunk (BASELINE.json configs[4]: "decode for all 16 conversations plus 4 append chunks").
        A conversation has one q_len per batch entry, so the chunk is a second entry whose block table names the same
        blocks (attention only reads them: S11).  Attention-only steps (the rows are already in the pool)."""
        import copy

        other = copy.copy(self)
        convs = [int(c) for c in convs]
        other.kv_lens = self.kv_lens + [self.kv_lens[c] for c in convs]
        other.tables = self.tables + [self.tables[c] for c in convs]
        other.h_tables = np.concatenate([self.h_tables, self.h_tables[convs]], axis=0)
        other.d_tables = torch.from_numpy(other.h_tables).cuda()
        other._setup_queries(list(self.q_lens) + [int(m)] * len(convs))
        return other

    def tail_attn(self, layer=0, stream=None):
        """csv_tail_step without the KV write (d_k_new = d_v_new = NULL): decode rows + chunks, one call."""
        B.csv_tail_step(self.plan, self.pool, layer, self.d_q, None, None, self.d_tables, self.max_blocks, self.d_out,
                        self.d_lse, stream)

    # algorithmic work: KV bytes read once per call
    def decode_kv_bytes(self):
        return sum(kv for q, kv in zip(self.q_lens, self.kv_lens) if q == 1) * self.Hkv * self.d * 2 * 2

    def append_kv_bytes(self):
        return sum(kv for q, kv in zip(self.q_lens, self.kv_lens) if q > 1) * self.Hkv * self.d * 2 * 2

    def append_flops(self):
        f = 0
        for m, kv in zip(self.q_lens, self.kv_lens):
            if m > 1:
                P = kv - m
                f += 4 * self.d * self.Hq * m * (P + (m + 1) / 2.0)
        return f

    def kv_append_tokens(self, stream=None):
        B.kv_append_tokens(self.pool, self.plan, self.d_k_new, self.d_v_new, self.d_tables, self.max_blocks, stream)

    def decode(self, layer=0, stream=None):
        B.paged_decode_attn(self.plan, self.pool, layer, self.d_q, self.d_tables, self.max_blocks, self.d_out, self.d_lse,
                            stream)

    def decode_step(self, layer=0, stream=None):
        """Fused tail step: new-token K/V write + decode attention in one launch (decode rows only)."""
        per_layer = self.total_q * self.Hkv * self.d
        B.paged_decode_step(self.plan, self.pool, layer, self.d_q, self.d_k_new[layer * per_layer:],
                            self.d_v_new[layer * per_layer:], self.d_tables, self.max_blocks, self.d_out, self.d_lse, stream)

    def tail_step(self, layer=0, stream=None):
        """One mixed tail step in one call: every new row's K/V write, decode attention, append attention."""
        per_layer = self.total_q * self.Hkv * self.d
        B.csv_tail_step(self.plan, self.pool, layer, self.d_q, self.d_k_new[layer * per_layer:],
                        self.d_v_new[layer * per_layer:], self.d_tables, self.max_blocks, self.d_out, self.d_lse, stream)

    def append(self, layer=0, stream=None):
        B.append_prefill_attn(self.plan, self.pool, layer, self.d_q, self.d_tables, self.max_blocks, self.d_out,
                              self.d_lse, stream)

    def conversation_blocks_host(self, b, layer=0):
        """Conversation b's blocks of one layer copied back to the host as a compact uint16 image
        [len(table)][2][Hkv][16][d] in table order (raw pool bytes: whoever reads them applies the layout)."""
        ids = self.tables[b]
        per_block = 2 * self.Hkv * 16 * self.d                       # int16 elements of one (layer, block)
        base = layer * self.num_blocks * per_block
        idx = torch.from_numpy(ids.astype(np.int64)).cuda()
        blocks = self.d_pool[base:base + self.num_blocks * per_block].view(self.num_blocks, per_block)[idx]
        return blocks.cpu().contiguous().numpy().view(np.uint16).reshape(-1)


def config_tail_workload(k, seed=None, layers=None, mpt=0, v_mean=0.0):
    """BASELINE.json configs 1, 2, 3, 5 as a TailWorkload (config 5 with `layers` layers, default 1)."""
    cfg = synth.CONFIGS[k]
    L = synth.config_lengths(k)
    seed = cfg["seed"] if seed is None else seed
    if k in (1, 2):
        kv = L["kv_lens"]
        return TailWorkload(cfg["Hq"], cfg["Hkv"], cfg["d"], [1] * len(kv), kv, seed=seed, mpt=mpt, v_mean=v_mean)
    if k == 3:
        return TailWorkload(cfg["Hq"], cfg["Hkv"], cfg["d"], L["q_lens"], L["kv_lens"], seed=seed, mpt=mpt, v_mean=v_mean)
    if k == 5:
        # S14: the decode call covers all 16 conversations; the append call (conversations 0-3, m = 256, same
        # kv_len) is a second plan over the same pool: wl.with_q_lens(config5_append_q_lens())
        return TailWorkload(cfg["Hq"], cfg["Hkv"], cfg["d"], [1] * cfg["n_conv"], L["kv_lens"], NL=layers or 1, seed=seed,
                            slack=0.01, mpt=mpt, v_mean=v_mean)
    raise KeyError(k)


def config5_append_q_lens():
    cfg, L = synth.CONFIGS[5], synth.config_lengths(5)
    q = np.zeros(cfg["n_conv"], dtype=np.int32)
    q[L["append_convs"]] = L["m"]
    return q

"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(device-generated pools, the library's allocator with a shuffled free list, default plans), on
sampled outputs the oracle can compute one by one.  The oracle reads the sampled conversations
back from the pool image through its own gather (O2): no expected value comes from the CUDA path.
"""
import numpy as np
import pytest
import torch

from paper_2606_01839_b200 import binding as B
from paper_2606_01839_b200 import synth, workloads
from harness import assert_close, bf16_dev_to_f64, dev_to_u16, logical_kv

pytestmark = pytest.mark.gpu


def free_gb():
    return torch.cuda.mem_get_info()[0] / 1e9


def check_rows(oracle, wl, layer, samples, O, LSE, what, written=False):
    """samples: list of (conversation b, row index i inside its q rows).  Oracle on the truncated cache.
    written: the step under test also WROTE the new rows' K/V (csv_tail_step / paged_decode_step): the rows the oracle
    gathers back from the pool at positions [kv_len - m, kv_len) must then be the step's k_new / v_new, bit for bit."""
    starts = np.concatenate([[0], np.cumsum(wl.q_lens)])
    q_all = dev_to_u16(wl.d_q).reshape(-1, wl.Hq, wl.d)
    cache = {}
    for b, i in samples:
        if b not in cache:
            cache = {b: logical_kv(oracle, wl, b, layer)}     # keep one conversation at a time (131k tokens = 512 MiB)
            if written:
                m, t = wl.q_lens[b], wl.kv_lens[b]
                per_layer = wl.total_q * wl.Hkv * wl.d
                lo, hi = layer * per_layer + starts[b] * wl.Hkv * wl.d, layer * per_layer + (starts[b] + m) * wl.Hkv * wl.d
                for name, new, got in (("K", wl.d_k_new, cache[b][0]), ("V", wl.d_v_new, cache[b][1])):
                    want = dev_to_u16(new[lo:hi]).reshape(m, wl.Hkv, wl.d)
                    assert np.array_equal(got[t - m:t], want), "%s conv %d: new %s rows are not in the pool" % (what, b, name)
        K, V = cache[b]
        m = wl.q_lens[b]
        n = wl.kv_lens[b] - m + i + 1                        # keys visible to row i (decode: m = 1, i = 0, n = kv_len)
        r = starts[b] + i
        o_ref, l_ref = oracle.attention(q_all[r:r + 1], K[:n], V[:n])
        assert_close(O[r:r + 1], LSE[r:r + 1], o_ref, l_ref, what="%s conv %d row %d (n=%d)" % (what, b, i, n))


def seeded_samples(wl, rng, n_decode, n_append_convs, rows_per_chunk):
    """(b, i) samples chosen by a seeded RNG: n_decode decode rows; rows_per_chunk rows (first, last, random) of each of
    n_append_convs chunks.  Grouped by conversation so that check_rows loads each cache once."""
    dec = [b for b, m in enumerate(wl.q_lens) if m == 1]
    app = [b for b, m in enumerate(wl.q_lens) if m > 1]
    out = [(int(b), 0) for b in rng.choice(dec, size=min(n_decode, len(dec)), replace=False)]
    for b in rng.choice(app, size=min(n_append_convs, len(app)), replace=False) if app else []:
        m = wl.q_lens[b]
        rows = {0, m - 1} | {int(x) for x in rng.integers(0, m, size=max(0, rows_per_chunk - 2))}
        out += [(int(b), i) for i in sorted(rows)]
    return out


def outputs(wl):
    torch.cuda.synchronize()
    O, LSE = bf16_dev_to_f64(wl.d_out), wl.d_lse.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(O)) and np.all(np.isfinite(LSE)), "a row was left unwritten"
    return O, LSE


def poison_outputs(wl):
    wl.d_out.fill_(0x7FC0)
    wl.d_lse.fill_(float("nan"))


def test_config3_agentic_tail_mix_full_size(oracle):
    # BASELINE.json config 3: 256 conversations, lognormal prefixes, 224 decode rows + 32 chunks of m ~ U[32,512]
    wl = workloads.config_tail_workload(3)
    info = wl.plan.info()
    assert info["n_decode_rows"] == 224 and info["n_append_chunks"] == 32
    wl.d_out.fill_(0x7FC0)
    wl.d_lse.fill_(float("nan"))
    wl.decode()
    wl.append()
    torch.cuda.synchronize()
    O, LSE = bf16_dev_to_f64(wl.d_out), wl.d_lse.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(O)) and np.all(np.isfinite(LSE))          # every row of both calls was written
    dec = [b for b in range(256) if wl.q_lens[b] == 1]
    app = [b for b in range(256) if wl.q_lens[b] > 1]
    by_len = sorted(dec, key=lambda b: wl.kv_lens[b])
    samples = [(b, 0) for b in (by_len[0], by_len[1], by_len[len(by_len) // 2], by_len[-1], dec[0], dec[-1])]
    a_small = sorted(app, key=lambda b: wl.kv_lens[b])[:3] + [max(app, key=lambda b: wl.q_lens[b])]
    for b in a_small:
        m = wl.q_lens[b]
        samples += [(b, 0), (b, m // 2), (b, m - 1)]
    check_rows(oracle, wl, 0, samples, O, LSE, "config 3")


def test_config3_timed_route_one_launch_tail_step_full_size(oracle):
    """What bench.py times on configs[2] is csv_tail_step: the KV write of all 9k new rows, then ONE persistent launch
    whose work items are the 224 decode rows' shares and the 32 chunks' tiles (the timed path must be the
    checked path).  Seeded sample of 16 decode rows and 8 chunks x 4 rows against the oracle, the written rows bit for bit,
    and a second run bit-identical to the first."""
    wl = workloads.config_tail_workload(3)
    assert wl.plan.info()["tail_n_dec"] > 0                              # the plan takes the one-launch route here
    poison_outputs(wl)
    wl.tail_step()
    O, LSE = outputs(wl)
    samples = seeded_samples(wl, np.random.default_rng(303), 16, 8, 4)
    assert sum(1 for b, _ in samples if wl.q_lens[b] == 1) >= 16 and sum(1 for b, _ in samples if wl.q_lens[b] > 1) >= 24
    check_rows(oracle, wl, 0, samples, O, LSE, "config 3 csv_tail_step", written=True)
    first = (wl.d_out.clone(), wl.d_lse.clone())
    poison_outputs(wl)
    wl.tail_step()
    torch.cuda.synchronize()
    assert torch.equal(first[0], wl.d_out) and torch.equal(first[1], wl.d_lse), "csv_tail_step differs from run to run"
    # the two-kernel route on the same plan inputs (a plan built with the override): within tolerance of the same oracle rows
    try:
        B.csv_tuning_set(B.TUNE_TAIL_TWO_KERNELS, 1)
        two = wl.with_q_lens(wl.q_lens)
    finally:
        B.csv_tuning_set(B.TUNE_TAIL_TWO_KERNELS, 0)
    two.d_q.copy_(wl.d_q)
    poison_outputs(two)
    two.tail_attn()
    O2, LSE2 = outputs(two)
    check_rows(oracle, two, 0, samples[:6] + samples[-6:], O2, LSE2, "config 3 two-kernel route")


def test_config5_long_context_full_size_eight_layers(oracle):
    # BASELINE.json config 5: Hq=64, Hkv=8, d=128, 8 layers, 16 x 131072 tokens (~69 GB of KV), >= 64 partitions per sequence
    if free_gb() < 90:
        pytest.skip("needs ~75 GB of free device memory")
    wl = workloads.config_tail_workload(5, layers=8)
    assert wl.pool_bytes >= 64 * 2 ** 30
    items, _ = wl.plan.decode_items()
    assert np.bincount(items[:, 0], minlength=16).min() >= 64
    app = wl.with_q_lens(workloads.config5_append_q_lens())
    rng = np.random.default_rng(505)
    # the headline route: paged_decode_step (KV write of the new token inside the decode launch) on three layers; layer 7
    # starts 56 GiB into the pool (64-bit addressing).  9 seeded rows in all, the written token checked bit for bit.
    for layer, n_rows in ((0, 3), (3, 3), (7, 3)):
        poison_outputs(wl)
        wl.decode_step(layer=layer)
        O, LSE = outputs(wl)
        rows = [(int(b), 0) for b in rng.choice(16, size=n_rows, replace=False)]
        check_rows(oracle, wl, layer, rows, O, LSE, "config 5 paged_decode_step layer %d" % layer, written=True)
    poison_outputs(wl)
    wl.decode(layer=7)                                      # the plain call on the same cache: same kernel without the write
    O, LSE = outputs(wl)
    check_rows(oracle, wl, 7, [(15, 0)], O, LSE, "config 5 decode layer 7")
    poison_outputs(app)
    app.append(layer=7)
    torch.cuda.synchronize()
    O, LSE = bf16_dev_to_f64(app.d_out), app.d_lse.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(O))
    check_rows(oracle, app, 7, [(2, 0), (2, 255)], O, LSE, "config 5 append layer 7")
    del app
    # the mixed step bench.py times on configs[4] (16 decode rows + 4 chunks of 256 as ONE csv_tail_step): the route the
    # plan picks (two kernels: the decode share is under a quarter), then the one-launch route forced on the same batch
    mixed = wl.with_extra_chunks(synth.config_lengths(5)["append_convs"], synth.config_lengths(5)["m"])
    assert mixed.plan.info()["tail_n_dec"] == 0
    try:
        B.csv_tuning_set(B.TUNE_TAIL_DECODE_CTAS, 26)
        forced = mixed.with_q_lens(mixed.q_lens)
    finally:
        B.csv_tuning_set(B.TUNE_TAIL_DECODE_CTAS, 0)
    assert forced.plan.info()["tail_n_dec"] == 26
    for w, layer, chunk, what in ((mixed, 7, 16, "plan's route"), (forced, 0, 18, "one launch forced")):
        poison_outputs(w)
        w.tail_attn(layer=layer)
        O, LSE = outputs(w)
        m = w.q_lens[chunk]
        rows = [(int(rng.integers(0, 16)), 0)] + [(chunk, i) for i in sorted({0, m - 1, int(rng.integers(1, m - 1)), int(rng.integers(1, m - 1))})]
        check_rows(oracle, w, layer, rows, O, LSE, "config 5 csv_tail_step (%s) layer %d" % (what, layer))


def test_config4_handoff_full_size(oracle):
    # BASELINE.json config 4: 16 conversations x 32 layers of 8B-shape KV, random 16-bit patterns, batched pack -> unpack
    if free_gb() < 95:
        pytest.skip("needs ~85 GB of free device memory")
    cfg = synth.CONFIGS[4]
    toks = [int(t) for t in synth.config_lengths(4)["tokens"]]
    NL, Hkv, d = cfg["NL"], cfg["Hkv"], cfg["d"]
    rng = np.random.default_rng(cfg["seed"])
    gen = torch.Generator(device="cuda")
    gen.manual_seed(44)
    nb = synth.pool_blocks_for(toks, slack=0.10)
    desc = B.pool_desc(NL, nb, Hkv, d)
    GUARD = -23101                                           # 0xA5C3 as int16
    d_pool = torch.full((B.kv_pool_bytes(desc) // 2,), GUARD, dtype=torch.int16, device="cuda")
    pool = B.KvPool(desc, d_pool)
    pool.set_free_order(synth.shuffled_free_order(rng, nb))
    ks, vs, sts, ids, h_ids = [], [], [], [], []
    for t in toks:
        n = NL * t * Hkv * d
        ks.append(torch.randint(-32768, 32767, (n,), dtype=torch.int16, device="cuda", generator=gen).view(NL, t, Hkv, d))
        vs.append(torch.randint(-32768, 32767, (n,), dtype=torch.int16, device="cuda", generator=gen).view(NL, t, Hkv, d))
        sts.append(torch.full((B.kv_staging_bytes(desc, t) // 2,), 0x1111, dtype=torch.int16, device="cuda"))
        h_ids.append(pool.alloc_blocks(synth.blocks_for(t)))
        ids.append(torch.from_numpy(h_ids[-1]).cuda())
    B.kv_pack_batch(desc, ks, vs, toks, [0] * 16, sts)
    B.kv_unpack_batch(pool, sts, toks, [0] * 16, ids, [len(i) for i in h_ids])
    torch.cuda.synchronize()
    unit = 2 * Hkv * 16 * d                                   # int16 elements of one (layer, block)
    pool_v = d_pool.view(NL, nb, unit)

    def check_samples(seed, staged):
        srng = np.random.default_rng(seed)
        for c in [int(np.argmin(toks)), int(np.argmax(toks))] + list(srng.integers(0, 16, size=4)):
            t = toks[c]
            ntb = synth.blocks_for(t)
            for layer, tb in [(0, 0), (NL - 1, ntb - 1)] + [(int(srng.integers(0, NL)), int(srng.integers(0, ntb))) for _ in range(6)]:
                lo, hi = tb * 16, min(t, tb * 16 + 16)
                K = dev_to_u16(ks[c][layer, lo:hi]).reshape(1, hi - lo, Hkv, d)
                V = dev_to_u16(vs[c][layer, lo:hi]).reshape(1, hi - lo, Hkv, d)
                if staged:
                    msg = oracle.staging_message(1, Hkv, d, K, V, hi - lo, 0)        # the 64 KiB unit, unused slots zero
                    got_st = dev_to_u16(sts[c].view(NL, ntb, unit)[layer, tb])
                    assert np.array_equal(got_st, msg), "staging unit (conv %d, layer %d, block %d)" % (c, layer, tb)
                expect_pool = oracle.scatter(np.full(unit, 0xA5C3, dtype=np.uint16), 1, 1, Hkv, d, K, V, hi - lo, 0,
                                             np.zeros(1, dtype=np.int32))            # unused slots keep the guard
                got_pool = dev_to_u16(pool_v[layer, int(h_ids[c][tb])])
                assert np.array_equal(got_pool, expect_pool), "pool unit (conv %d, layer %d, block %d)" % (c, layer, tb)

    check_samples(5, staged=True)
    # kv_handoff_direct (NEXT-1) on the same conversations and blocks: sampled against the oracle, and the WHOLE pool
    # against the staged route's image (itself sampled above): 21 GB compared bit for bit
    staged_image = d_pool.clone()
    d_pool.fill_(GUARD)
    B.kv_handoff_direct_batch(pool, ks, vs, toks, [0] * 16, ids, [len(i) for i in h_ids])
    torch.cuda.synchronize()
    check_samples(6, staged=False)
    assert torch.equal(d_pool, staged_image)
    del staged_image
    # blocks never handed out are untouched, in every layer
    used = np.zeros(nb, dtype=bool)
    used[np.concatenate(h_ids)] = True
    free_ids = torch.from_numpy(np.flatnonzero(~used)[:64].astype(np.int64)).cuda()
    assert bool((pool_v[:, free_ids] == GUARD).all())
    assert pool.used_blocks == sum(synth.blocks_for(t) for t in toks)


def test_turn1_prefill_chunk_8192_through_append_prefill_attn(oracle):
    """turn-1 prefill attention, chunked 8192 tokens per batch as the paper configures the prefiller
    (PAPER.md:213), is append_prefill_attn with m = 8192 and P = the tokens of the earlier chunks."""
    wl = workloads.TailWorkload(32, 8, 128, [1], [16384], seed=21)
    for P in (0, 8192):
        app = wl.with_q_lens([8192], [P + 8192])
        app.d_out.fill_(0x7FC0)
        app.append()
        torch.cuda.synchronize()
        O, LSE = bf16_dev_to_f64(app.d_out), app.d_lse.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(O)) and np.all(np.isfinite(LSE))
        check_rows(oracle, app, 0, [(0, 0), (0, 1), (0, 127), (0, 4096), (0, 8191)], O, LSE, "prefill chunk P=%d" % P)


def test_spike_sweep_at_131072_tokens_decode_and_append(oracle):
    """SURVEY §8c item 1 at config 5's length: with N(0,1) data a dropped 16-token block is invisible to the 1e-2 gate once
    L >~ 8k, so one key per (conversation, KV head) is made to carry ~all the weight (score ~30 against a log-sum-exp of
    ~12.3 for the other 131071 keys) with a +-1 pattern as its V: closed-form answer, no fp64 run.  The spikes sit on the
    first and last block of split-K partitions taken from the plan, at both ends of the sequence and at random places.
    They are written into the device pool at the oracle's addresses (O2's formula), not through the library."""
    cfg = synth.CONFIGS[5]
    Hq, Hkv, d, G, L, n = cfg["Hq"], cfg["Hkv"], cfg["d"], cfg["Hq"] // cfg["Hkv"], 131072, 6
    m = 24                                                   # appended rows of the second plan (conversations 0, 1)
    wl = workloads.TailWorkload(Hq, Hkv, d, [1] * n, [L] * n, seed=77, slack=0.02)
    items, _ = wl.plan.decode_items()
    rng = np.random.default_rng(78)
    q = synth.bf16_bits_to_f32(dev_to_u16(wl.d_q).reshape(n, Hq, d))
    app = wl.with_q_lens([m, m] + [0] * (n - 2))
    qa_bits = dev_to_u16(app.d_q).reshape(2 * m, Hq, d).copy()
    pos = np.zeros((n, Hkv), dtype=np.int64)
    pattern = np.where(rng.random((n, Hkv, d)) < 0.5, -1.0, 1.0).astype(np.float32)
    pool16 = wl.d_pool.view(torch.int16)
    spike_k = np.zeros((n, Hkv, d), dtype=np.float32)
    for b in range(n):
        for g in range(Hkv):
            mine = items[(items[:, 0] == b) & (items[:, 1] == g)]
            assert len(mine) >= 8                             # split-K really cuts this sequence
            part = mine[int(rng.integers(0, len(mine)))]
            choice = int(rng.integers(0, 6))
            j = [int(part[2]) * 16, int(part[3]) * 16 - 1, 0, L - 1, int(rng.integers(0, L)), int(part[2]) * 16 + 15][choice]
            if b < 2:
                j = min(j, L - m - 1)                         # visible to every appended row of conversations 0, 1
            pos[b, g] = j
            dirv = q[b, g * G:(g + 1) * G].sum(axis=0)
            if b < 2:                                         # the appended rows share this direction (see below)
                dirv = dirv / np.linalg.norm(dirv) * np.sqrt(d)
            spike_k[b, g] = dirv * (30.0 * np.sqrt(d) / np.dot(dirv, dirv) * (G if b >= 2 else 1.0))
            kb, vb = synth.f32_to_bf16_bits(spike_k[b, g]), synth.f32_to_bf16_bits(pattern[b, g])
            blk, slot = int(wl.tables[b][j // 16]), j % 16
            ka = np.array([oracle.pool_addr(wl.num_blocks, Hkv, d, 0, blk, 0, g, slot, c) for c in range(d)], dtype=np.int64)
            va = np.array([oracle.pool_addr(wl.num_blocks, Hkv, d, 0, blk, 1, g, slot, c) for c in range(d)], dtype=np.int64)
            pool16[torch.from_numpy(ka).cuda()] = torch.from_numpy(kb.view(np.int16)).cuda()
            pool16[torch.from_numpy(va).cuda()] = torch.from_numpy(vb.view(np.int16)).cuda()
    spike_k = synth.bf16_bits_to_f32(synth.f32_to_bf16_bits(spike_k))
    # ---- decode: 6 x 131072 ----
    wl.d_out.fill_(0x7FC0)
    wl.decode()
    torch.cuda.synchronize()
    O, LSE = bf16_dev_to_f64(wl.d_out), wl.d_lse.cpu().numpy().astype(np.float64)
    checked = 0
    for b in range(n):
        for h in range(Hq):
            s = float(np.dot(q[b, h].astype(np.float64), spike_k[b, h // G].astype(np.float64)) / np.sqrt(d))
            if s >= 22.0:                                     # others weigh <= exp(13.5 - 22) = 2e-4
                assert np.abs(O[b, h] - pattern[b, h // G]).max() <= 1e-2, (b, h, int(pos[b, h // G]), s)
                assert s - 1e-3 <= LSE[b, h] <= s + 1e-3 + np.exp(13.5 - s), (b, h, s, LSE[b, h])
                checked += 1
    assert checked >= 0.5 * n * Hq
    # ---- append on the same pool: rows of conversations 0 and 1 all point along the group's direction ----
    qa = np.zeros((2 * m, Hq, d), dtype=np.float32)
    for b in range(2):
        for h in range(Hq):
            u = spike_k[b, h // G] / np.linalg.norm(spike_k[b, h // G]) * np.sqrt(d)
            qa[b * m:(b + 1) * m, h] = u + 0.3 * rng.standard_normal((m, d)).astype(np.float32)
    qa_bits = synth.f32_to_bf16_bits(qa)
    app.d_q.copy_(torch.from_numpy(qa_bits.view(np.int16)).cuda().view_as(app.d_q))
    app.d_out.fill_(0x7FC0)
    app.append()
    torch.cuda.synchronize()
    O, LSE = bf16_dev_to_f64(app.d_out), app.d_lse.cpu().numpy().astype(np.float64)
    qa = synth.bf16_bits_to_f32(qa_bits)
    checked = 0
    for r in range(2 * m):
        b = r // m
        for h in range(Hq):
            s = float(np.dot(qa[r, h].astype(np.float64), spike_k[b, h // G].astype(np.float64)) / np.sqrt(d))
            if s >= 22.0:
                assert np.abs(O[r, h] - pattern[b, h // G]).max() <= 1e-2, (r, h, int(pos[b, h // G]), s)
                assert s - 1e-3 <= LSE[r, h] <= s + 1e-3 + np.exp(13.5 - s)
                checked += 1
    assert checked >= 0.9 * 2 * m * Hq

"""GPU parity of the one-shot KV handoff (kv_pack / kv_unpack / kv_append_tokens) against the
oracle's reference scatter (O3) and staging formula.  Bit-exact, whole pool image compared
(a stray write anywhere is a mismatch).  PAPER.md:150 §4 "transferred once to the bound decoder".
"""
import os

import numpy as np
import pytest
import torch

from paper_2606_01839_b200 import binding as B
from paper_2606_01839_b200 import replicas, synth
from harness import dev, dev_to_u16, u16_dev

pytestmark = pytest.mark.gpu
GUARD = 0xA5C3


def handoff_case(oracle, rng, NL, Hkv, d, num_blocks, convs, batched, direct=False):
    """convs: list of (tokens, token_offset).  Each conversation owns ceil((off+tokens)/16) blocks."""
    desc = B.pool_desc(NL, num_blocks, Hkv, d)
    image = np.full(oracle.pool_elems(NL, num_blocks, Hkv, d), GUARD, dtype=np.uint16)
    d_image = u16_dev(image)
    pool = B.KvPool(desc, d_image)
    pool.set_free_order(synth.shuffled_free_order(rng, num_blocks))
    expected = image.copy()
    ks, vs, stagings, tables, toks, offs, nids, msgs = [], [], [], [], [], [], [], []
    for tokens, off in convs:
        ids = pool.alloc_blocks(synth.blocks_for(off + tokens))
        K = synth.random_bits(rng, (NL, tokens, Hkv, d))
        V = synth.random_bits(rng, (NL, tokens, Hkv, d))
        expected = oracle.scatter(expected, NL, num_blocks, Hkv, d, K, V, tokens, off, ids)
        msgs.append(oracle.staging_message(NL, Hkv, d, K, V, tokens, off))
        nbytes = B.kv_staging_bytes(desc, tokens, off)
        assert nbytes == msgs[-1].size * 2
        ks.append(u16_dev(K))
        vs.append(u16_dev(V))
        stagings.append(torch.full((nbytes // 2,), 0x1111, dtype=torch.int16, device="cuda"))
        tables.append(dev(ids))
        toks.append(tokens)
        offs.append(off)
        nids.append(len(ids))
    if direct:                                   # kv_handoff_direct: no staging message at all
        if batched:
            B.kv_handoff_direct_batch(pool, ks, vs, toks, offs, tables, nids)
        else:
            for i in range(len(convs)):
                B.kv_handoff_direct(pool, ks[i], vs[i], toks[i], offs[i], tables[i], nids[i])
        torch.cuda.synchronize()
        got = dev_to_u16(d_image)
        assert np.array_equal(got, expected), "pool image differs (%d elements)" % int((got != expected).sum())
        for st in stagings:
            assert bool((st == 0x1111).all())
        return pool
    if batched:
        B.kv_pack_batch(desc, ks, vs, toks, offs, stagings)
        B.kv_unpack_batch(pool, stagings, toks, offs, tables, nids)
    else:
        for i in range(len(convs)):
            B.kv_pack(desc, ks[i], vs[i], toks[i], offs[i], stagings[i])
            B.kv_unpack(pool, stagings[i], toks[i], offs[i], tables[i], nids[i])
    torch.cuda.synchronize()
    for i in range(len(convs)):
        assert np.array_equal(dev_to_u16(stagings[i]), msgs[i]), "staging message %d differs from the oracle's" % i
    got = dev_to_u16(d_image)
    assert np.array_equal(got, expected), "pool image differs (%d elements)" % int((got != expected).sum())
    return pool


def test_config1_handoff_300_tokens(oracle):
    # BASELINE.json config 1: one kv_pack / kv_unpack of a 300-token prefill into a second 256-block pool
    rng = np.random.default_rng(0)
    pool = handoff_case(oracle, rng, 1, 1, 64, 256, [(300, 0)], batched=False)
    assert pool.used_blocks == 19


@pytest.mark.parametrize("batched", [False, True])
def test_handoff_8b_shape_ragged_and_offsets(oracle, batched):
    rng = np.random.default_rng(7)
    convs = [(300, 0), (1, 0), (16, 0), (17, 0), (5, 11), (1, 15), (2, 15), (40, 24), (129, 3), (33, 32)]
    handoff_case(oracle, rng, 3, 8, 128, 64, convs, batched)


def test_handoff_other_shapes(oracle):
    rng = np.random.default_rng(8)
    handoff_case(oracle, rng, 2, 2, 64, 40, [(100, 0), (7, 9), (64, 16)], batched=True)
    handoff_case(oracle, rng, 1, 4, 128, 40, [(47, 0), (20, 5)], batched=True)


def test_handoff_more_conversations_than_one_launch_holds(oracle):
    rng = np.random.default_rng(9)
    convs = [(int(rng.integers(1, 40)), int(rng.integers(0, 16))) for _ in range(70)]
    handoff_case(oracle, rng, 1, 2, 64, 4 * 70 + 5, convs, batched=True)


def test_handoff_argument_errors():
    desc = B.pool_desc(1, 8, 1, 64)
    buf = torch.zeros(B.kv_pool_bytes(desc) // 2, dtype=torch.int16, device="cuda")
    pool = B.KvPool(desc, buf)
    k = torch.zeros(300 * 64, dtype=torch.int16, device="cuda")
    st = torch.zeros(B.kv_staging_bytes(desc, 300) // 2, dtype=torch.int16, device="cuda")
    ids = torch.zeros(8, dtype=torch.int32, device="cuda")
    before = buf.clone()
    for call in (lambda: B.kv_pack(desc, k, k, 0, 0, st),                       # zero tokens
                 lambda: B.kv_pack(desc, k, k, -1, 0, st),
                 lambda: B.kv_pack(desc, k, k, 10, -1, st),
                 lambda: B.kv_pack(desc, k, k, 10, 0, st.data_ptr() + 16),      # misaligned staging
                 lambda: B.kv_pack(desc, k.data_ptr() + 2, k, 10, 0, st),       # misaligned source
                 lambda: B.kv_pack(B.pool_desc(1, 8, 3, 64), k, k, 10, 0, st),  # unsupported shape
                 lambda: B.kv_unpack(pool, st, 300, 0, ids, 8),                 # table shorter than ceil(300/16)
                 lambda: B.kv_unpack(pool, st, 17, 112, ids, 8),                # offset + tokens past the table
                 lambda: B.kv_unpack(pool, st, 0, 0, ids, 8)):
        with pytest.raises(B.CsvError) as e:
            call()
        assert e.value.code == B.CSV_E_INVAL
    torch.cuda.synchronize()
    assert torch.equal(buf, before)                                            # a failed call changes nothing


def test_kv_append_tokens_equals_the_reference_scatter(oracle):
    # tail step: new tokens' K/V go straight into the pool ("appending one new entry")
    rng = np.random.default_rng(11)
    NL, Hkv, d, Hq, nb = 2, 8, 128, 32, 80
    q_lens = [1, 37, 0, 1, 16, 1]
    kv_lens = [1, 100, 50, 160, 16, 33]
    image = np.full(oracle.pool_elems(NL, nb, Hkv, d), GUARD, dtype=np.uint16)
    order = synth.shuffled_free_order(rng, nb)
    tables, pos = [], 0
    for t in kv_lens:
        n = synth.blocks_for(t)
        tables.append(order[pos:pos + n])
        pos += n
    total_q = sum(q_lens)
    Kn = synth.random_bits(rng, (NL, total_q, Hkv, d))
    Vn = synth.random_bits(rng, (NL, total_q, Hkv, d))
    expected, r = image.copy(), 0
    for b, m in enumerate(q_lens):
        if m:
            expected = oracle.scatter(expected, NL, nb, Hkv, d, Kn[:, r:r + m], Vn[:, r:r + m], m, kv_lens[b] - m, tables[b])
            r += m
    d_image = u16_dev(image)
    pool = B.KvPool(B.pool_desc(NL, nb, Hkv, d), d_image)
    shape = B.attn_shape(Hq, Hkv, d)
    ws = torch.empty(B.csv_plan_workspace_bytes(shape, q_lens, kv_lens), dtype=torch.uint8, device="cuda")
    plan = B.Plan(shape, q_lens, kv_lens, 0, ws)
    tabs, mb = synth.dense_tables(tables)
    B.kv_append_tokens(pool, plan, u16_dev(Kn), u16_dev(Vn), dev(tabs), mb)
    torch.cuda.synchronize()
    assert np.array_equal(dev_to_u16(d_image), expected)


# ---------------- kv_handoff_direct: pack + transfer + scatter in one kernel ----------------

@pytest.mark.parametrize("batched", [False, True])
def test_direct_handoff_equals_the_reference_scatter(oracle, batched):
    rng = np.random.default_rng(17)
    handoff_case(oracle, rng, 1, 1, 64, 256, [(300, 0)], batched, direct=True)        # config 1's handoff
    convs = [(300, 0), (1, 0), (16, 0), (17, 0), (5, 11), (1, 15), (2, 15), (40, 24), (129, 3), (33, 32)]
    handoff_case(oracle, rng, 3, 8, 128, 64, convs, batched, direct=True)
    handoff_case(oracle, rng, 2, 2, 64, 40, [(100, 0), (7, 9), (64, 16)], batched, direct=True)
    handoff_case(oracle, rng, 1, 4, 128, 40, [(47, 0), (20, 5)], batched, direct=True)


def test_direct_handoff_more_conversations_than_one_launch_holds(oracle):
    rng = np.random.default_rng(19)
    convs = [(int(rng.integers(1, 40)), int(rng.integers(0, 16))) for _ in range(70)]
    handoff_case(oracle, rng, 1, 2, 64, 4 * 70 + 5, convs, batched=True, direct=True)


def test_direct_handoff_argument_errors():
    desc = B.pool_desc(1, 8, 1, 64)
    buf = torch.zeros(B.kv_pool_bytes(desc) // 2, dtype=torch.int16, device="cuda")
    pool = B.KvPool(desc, buf)
    k = torch.ones(300 * 64, dtype=torch.int16, device="cuda")
    ids = torch.zeros(8, dtype=torch.int32, device="cuda")
    for call in (lambda: B.kv_handoff_direct(pool, k, k, 0, 0, ids, 8),
                 lambda: B.kv_handoff_direct(pool, k, k, -3, 0, ids, 8),
                 lambda: B.kv_handoff_direct(pool, k, k, 10, -1, ids, 8),
                 lambda: B.kv_handoff_direct(pool, k.data_ptr() + 2, k, 10, 0, ids, 8),   # misaligned source
                 lambda: B.kv_handoff_direct(pool, k, None, 10, 0, ids, 8),
                 lambda: B.kv_handoff_direct(pool, k, k, 300, 0, ids, 8),                 # table too short
                 lambda: B.kv_handoff_direct(pool, k, k, 17, 112, ids, 8)):
        with pytest.raises(B.CsvError) as e:
            call()
        assert e.value.code == B.CSV_E_INVAL
    torch.cuda.synchronize()
    assert int(buf.abs().sum()) == 0


def _prefiller_process(ticket, seed, q):
    """The OTHER process of the handoff: owns the turn-1 K/V, maps the decoder's pool by CUDA IPC and pushes into it."""
    try:
        from paper_2606_01839_b200 import replicas

        NL, nb, Hkv, d = ticket["shape"]
        tokens = ticket["tokens"]
        rng = np.random.default_rng(seed)
        K = synth.random_bits(rng, (NL, tokens, Hkv, d))
        V = synth.random_bits(rng, (NL, tokens, Hkv, d))
        torch.cuda.set_device(0)
        peers = replicas.PeerPools()                               # wraps the mapping; the allocator stays with the decoder
        keep = peers.push(ticket, u16_dev(K), u16_dev(V))
        torch.cuda.synchronize()
        ptr = peers._pools[next(iter(peers._pools))][1]
        assert B.csv_ipc_mapped_bytes(ptr) >= B.kv_pool_bytes(B.pool_desc(NL, nb, Hkv, d))
        # a ticket whose shape claims more memory than the decoder really shared is refused before any pool exists
        # (shape and offset arrive in the same message as the handle), and its mapping reference is given back
        big = dict(ticket, decoder=7, shape=(NL, nb * 4096, Hkv, d))
        with pytest.raises(ValueError, match="mapped allocation"):
            peers.get(big)
        assert len(peers._pools) == 1
        with pytest.raises(B.CsvError):
            B.csv_ipc_mapped_bytes(ptr + 128)                      # not a pointer csv_ipc_open handed out
        peers.close()
        with pytest.raises(B.CsvError):
            B.csv_ipc_close(ptr)                                   # unknown pointer now
        del keep
        q.put("ok")
    except Exception as e:                                         # noqa: BLE001
        q.put("error: %r" % (e,))


def test_direct_handoff_into_another_process_pool_over_cuda_ipc(oracle):
    """One process per GPU is the deployment; this box has one GPU, so the prefiller process shares it.
    The path is the one two GPUs take: export the pool's allocation, open it in the prefiller, push, hand back."""
    import torch.multiprocessing as mp

    NL, nb, Hkv, d, tokens, off, seed = 2, 48, 8, 128, 300, 5, 23
    rng = np.random.default_rng(3)
    torch.cuda.synchronize()
    n = oracle.pool_elems(NL, nb, Hkv, d)
    slab = torch.empty(n + 8192, dtype=torch.int16, device="cuda")           # pool = a view INSIDE an allocation:
    slab.fill_(0x2222)
    d_image = slab[4096:4096 + n]                                            # the exported offset must be honoured
    image = np.full(n, GUARD, dtype=np.uint16)
    d_image.copy_(u16_dev(image))
    pool = B.KvPool(B.pool_desc(NL, nb, Hkv, d), d_image)
    pool.set_free_order(synth.shuffled_free_order(rng, nb))
    handle, offset = B.csv_ipc_export(d_image)
    ticket = replicas.handoff_ticket(pool, tokens, off, export=(handle, offset))   # the decoder allocates, the ids travel
    ids = np.asarray(ticket["ids"], dtype=np.int32)
    assert pool.used_blocks == synth.blocks_for(off + tokens)
    assert len(handle) == B.IPC_HANDLE_BYTES and offset >= 4096 * 2
    torch.cuda.synchronize()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    p = ctx.Process(target=_prefiller_process, args=(ticket, seed, q))
    p.start()
    msg = q.get(timeout=300)
    p.join(60)
    assert msg == "ok", msg
    rng2 = np.random.default_rng(seed)
    K = synth.random_bits(rng2, (NL, tokens, Hkv, d))
    V = synth.random_bits(rng2, (NL, tokens, Hkv, d))
    expected = oracle.scatter(image, NL, nb, Hkv, d, K, V, tokens, off, ids)
    assert np.array_equal(dev_to_u16(d_image), expected)
    assert bool((slab[:4096] == 0x2222).all()) and bool((slab[4096 + n:] == 0x2222).all())


def test_handoff_across_two_ranks_direct_and_staged():
    """paper_2606_01839_b200.handoff_p2p under torchrun with two ranks (prefiller, decoder): on this one-GPU box both share
    the device; with two GPUs the same program pushes over NVLink.  It exits non-zero unless both routes leave the
    decoder's pool bit-identical to a local handoff of the same K/V."""
    import json
    import socket
    import subprocess
    import sys

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), "-m", "paper_2606_01839_b200.handoff_p2p", "--tokens", "1000", "--layers", "4",
           "--convs", "5", "--iters", "1"]
    r = subprocess.run(cmd, cwd=root, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    line = [ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1]
    out = json.loads(line)
    assert out["bit_exact_direct"] and out["bit_exact_staged"] and out["bit_exact_copy"] and out["convs"] == 5
    assert out["memcpy_peer_gbs"] > 0 and out["copy_payload_gbs"] > 0          # the cudaMemcpyAsync comparison arm ran

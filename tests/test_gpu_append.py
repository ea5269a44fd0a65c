"""GPU parity of append_prefill_attn (and mixed decode + append steps, and the host-buffer tail
step) against the fp64 oracle.  PAPER.md:94 §3.1: appended chunks attend to "the whole history
context" plus themselves; BASELINE.json config 3: "causal against prefix+self".
"""
import numpy as np
import pytest
import torch

from paper_2606_01839_b200 import binding as B
from paper_2606_01839_b200 import synth
from harness import (Scenario, assert_close, bf16_dev_to_f64, dev, oracle_abs_weighted, oracle_attention, run_attention,
                     u16_dev)

pytestmark = pytest.mark.gpu


def step_case(oracle, seed, Hq, Hkv, d, convs, mpt=0, poison=False, v_mean=0.0, qscale=1.0, what=""):
    """convs: list of (P, m); m = 1 is a decode row (kv_len = P + 1), m = 0 an inert conversation."""
    rng = np.random.default_rng(seed)
    q_lens = [m for _, m in convs]
    kv_lens = [P + m for P, m in convs]
    sc = Scenario(oracle, rng, Hq, Hkv, d, kv_lens, poison=poison, v_mean=v_mean).commit().upload()
    q = synth.normal_bf16(rng, (sum(q_lens), Hq, d), std=qscale)
    O, LSE, info = run_attention(sc, q_lens, q, mpt=mpt, which="both")
    O_ref, LSE_ref = oracle_attention(sc, q_lens, q)
    A_ref = oracle_abs_weighted(sc, q_lens, q) if qscale > 1.0 else None   # peaked softmax: DESIGN.md S20
    res = assert_close(O, LSE, O_ref, LSE_ref, what or "step", A_ref=A_ref)
    if any(m == 1 for m in q_lens) and any(m > 1 for m in q_lens):
        # the same step through csv_tail_step: at d = 128 decode rows and chunks are work items of ONE launch (tail_fused.cu)
        O2, LSE2, _ = run_attention(sc, q_lens, q, mpt=mpt, which="tail")
        assert_close(O2, LSE2, O_ref, LSE_ref, (what or "step") + " [csv_tail_step]", A_ref=A_ref)
        O3, LSE3, _ = run_attention(sc, q_lens, q, mpt=mpt, which="tail")
        assert np.array_equal(O2, O3) and np.array_equal(LSE2, LSE3), "csv_tail_step is not bit-identical from run to run"
    return res, info


@pytest.mark.parametrize("Hq,Hkv,d", [(32, 8, 128), (64, 8, 128), (4, 1, 64), (8, 8, 64), (16, 2, 128), (8, 8, 128), (8, 4, 128),
                                      (2, 1, 64)])
def test_append_chunk_length_edge_cases(oracle, Hq, Hkv, d):
    # m in {2, 31, 32, 33, 512}, P = 0, prefixes not multiples of 16
    convs = [(0, 2), (0, 33), (100, 31), (1000, 32), (17, 33), (777, 2), (15, 16), (3, 100)]
    step_case(oracle, 50 + Hq + d, Hq, Hkv, d, convs, what="append edges %s" % ((Hq, Hkv, d),))


def test_append_512_token_chunk_and_full_causal_prefill(oracle):
    step_case(oracle, 60, 32, 8, 128, [(2000, 512), (0, 300)], what="m=512")


def test_mixed_decode_and_append_step_fills_one_output(oracle):
    # one plan, two calls, one [total_q] output: decode rows and chunks interleaved in batch order
    convs = [(500, 1), (300, 40), (0, 1), (2047, 1), (64, 64), (10, 0), (4000, 1), (129, 17)]
    step_case(oracle, 61, 32, 8, 128, convs, what="mixed")
    step_case(oracle, 62, 64, 8, 128, convs, what="mixed G=8")


@pytest.mark.parametrize("mpt", [64, 256, 2048])
def test_append_kv_partitions_merge_correctly(oracle, mpt):
    # long prefix cut into KV partitions; a partition boundary inside the chunk's own tokens leaves some rows
    # with no visible key in the last partition (their partial is m = -inf, l = 0)
    convs = [(3000, 100), (250, 200), (0, 130), (5000, 33)]
    (_, _), info = step_case(oracle, 63, 32, 8, 128, convs, mpt=mpt, what="append mpt=%d" % mpt)


def test_append_poisoned_padding_and_nonzero_mean(oracle):
    step_case(oracle, 64, 32, 8, 128, [(100, 37), (1000, 5), (3, 2)], poison=True, what="append poison")
    step_case(oracle, 65, 32, 8, 128, [(3000, 64), (9000, 40)], v_mean=1.0, what="append V~N(1,1)")
    step_case(oracle, 66, 32, 8, 128, [(2000, 48)], qscale=8.0, what="append q x8")


def test_append_row_equals_decode_on_the_truncated_cache(oracle):
    """Row i of a chunk with prefix P must equal a decode row with kv_len = P + i + 1 on the same cache
    (the oracle's invariant, now across the two CUDA kernels)."""
    rng = np.random.default_rng(67)
    Hq, Hkv, d, P, m = 32, 8, 128, 700, 24
    sc = Scenario(oracle, rng, Hq, Hkv, d, [P + m]).commit().upload()
    q = synth.normal_bf16(rng, (m, Hq, d))
    O_a, LSE_a, _ = run_attention(sc, [m], q, which="append")
    for i in (0, 7, m - 1):
        sc.kv_lens = [P + i + 1]
        O_d, LSE_d, _ = run_attention(sc, [1], q[i:i + 1], which="decode")
        assert np.abs(O_d[0] - O_a[i]).max() <= 2 ** -7 and np.abs(LSE_d[0] - LSE_a[i]).max() <= 2e-4
    sc.kv_lens = [P + m]


def test_tail_step_host_buffers(oracle):
    """csv_tail_step_host: plan + H2D + new-token KV write + decode + D2H in one call (bench.py's e2e path)."""
    rng = np.random.default_rng(68)
    Hq, Hkv, d = 32, 8, 128
    kv_lens = [100, 2049, 16, 1, 777]
    sc = Scenario(oracle, rng, Hq, Hkv, d, kv_lens, poison=True)
    # the cache holds everything but each conversation's newest token; that token arrives through the call
    k_new = np.stack([sc.K[b][0, kv_lens[b] - 1] for b in range(5)])
    v_new = np.stack([sc.V[b][0, kv_lens[b] - 1] for b in range(5)])
    for b, t in enumerate(kv_lens):
        if t > 1:
            sc.image = oracle.scatter(sc.image, 1, sc.num_blocks, Hkv, d, sc.K[b][:, :t - 1], sc.V[b][:, :t - 1], t - 1, 0,
                                      sc.tables[b])
    sc.upload()
    shape = B.attn_shape(Hq, Hkv, d)
    q = synth.normal_bf16(rng, (5, Hq, d))
    tabs = np.where(sc.h_tables < 0, 0, sc.h_tables).astype(np.int32)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_q, h_k, h_v, h_t = pin(q.view(np.int16)), pin(k_new.view(np.int16)), pin(v_new.view(np.int16)), pin(tabs)
    h_out = torch.zeros((5, Hq, d), dtype=torch.int16).pin_memory()
    h_lse = torch.zeros((5, Hq), dtype=torch.float32).pin_memory()
    ws = torch.empty(B.csv_tail_step_host_workspace_bytes(shape, kv_lens, sc.max_blocks), dtype=torch.uint8, device="cuda")
    B.csv_tail_step_host(sc.pool, 0, shape, kv_lens, h_q, h_k, h_v, h_t, sc.max_blocks, ws, h_out, h_lse)
    O = synth.bf16_bits_to_f32(h_out.numpy().view(np.uint16)).astype(np.float64)
    O_ref, LSE_ref = oracle_attention(sc, [1] * 5, q)
    assert_close(O, h_lse.numpy().astype(np.float64), O_ref, LSE_ref, what="tail step")


def test_tail_step_host_over_a_decode_loop(oracle):
    """csv_tail_step_host over 40 consecutive decode steps: every conversation grows by one token per step,
    crossing block edges on the way.  Every third step's O / LSE against the oracle on the cache as it stands, the pool at
    the end against the oracle's scatter."""
    from harness import dev_to_u16
    rng = np.random.default_rng(97)
    Hq, Hkv, d, steps = 32, 8, 128, 40
    start = [100, 2049, 15, 2, 777, 4096 - 20]
    final = [t + steps - 1 for t in start]
    n = len(start)
    sc = Scenario(oracle, rng, Hq, Hkv, d, final, poison=True)
    full = sc.image.copy()
    for b in range(n):
        full = oracle.scatter(full, 1, sc.num_blocks, Hkv, d, sc.K[b], sc.V[b], final[b], 0, sc.tables[b])
        sc.image = oracle.scatter(sc.image, 1, sc.num_blocks, Hkv, d, sc.K[b][:, :start[b] - 1], sc.V[b][:, :start[b] - 1],
                                  start[b] - 1, 0, sc.tables[b])
    shape = B.attn_shape(Hq, Hkv, d)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    sc.upload()
    tabs = np.where(sc.h_tables < 0, 0, sc.h_tables).astype(np.int32)
    h_t = pin(tabs)
    h_out = torch.zeros((n, Hq, d), dtype=torch.int16).pin_memory()
    h_lse = torch.zeros((n, Hq), dtype=torch.float32).pin_memory()
    ws = torch.empty(2 * B.csv_tail_step_host_workspace_bytes(shape, final, sc.max_blocks), dtype=torch.uint8, device="cuda")
    qrng = np.random.default_rng(98)
    for s_ in range(steps):
        kv = [t + s_ for t in start]
        k_new = np.stack([sc.K[b][0, kv[b] - 1] for b in range(n)])
        v_new = np.stack([sc.V[b][0, kv[b] - 1] for b in range(n)])
        q = synth.normal_bf16(qrng, (n, Hq, d))
        B.csv_tail_step_host(sc.pool, 0, shape, kv, pin(q.view(np.int16)), pin(k_new.view(np.int16)), pin(v_new.view(np.int16)),
                             h_t, sc.max_blocks, ws, h_out, h_lse)
        if s_ % 3 == 0 or s_ == steps - 1:
            O = synth.bf16_bits_to_f32(h_out.numpy().view(np.uint16)).astype(np.float64)
            for b in range(n):
                o_ref, l_ref = oracle.attention(q[b:b + 1], sc.K[b][0][:kv[b]], sc.V[b][0][:kv[b]])
                assert_close(O[b:b + 1], h_lse[b:b + 1].numpy().astype(np.float64), o_ref, l_ref,
                             what="host loop step %d conv %d" % (s_, b))
    assert np.array_equal(dev_to_u16(sc.d_image), full), "pool after the host loop differs from the oracle's scatter"


@pytest.mark.parametrize("Hq,Hkv,d", [(32, 8, 128), (64, 8, 128), (4, 1, 64)])
def test_fused_decode_step_writes_the_token_and_attends_to_it(oracle, Hq, Hkv, d):
    """paged_decode_step = kv_append_tokens + paged_decode_attn in one launch: the pool must end up bit-identical to
    the oracle's scatter of the full conversations, and O / LSE must match the oracle on the full cache."""
    rng = np.random.default_rng(70 + d + Hq)
    kv_lens = [1, 16, 17, 33, 2049, 640, 100, 4097]
    n = len(kv_lens)
    sc = Scenario(oracle, rng, Hq, Hkv, d, kv_lens, poison=True)
    full = sc.image.copy()
    for b, t in enumerate(kv_lens):
        full = oracle.scatter(full, 1, sc.num_blocks, Hkv, d, sc.K[b], sc.V[b], t, 0, sc.tables[b])
        if t > 1:   # the cache before the step: everything but the newest token
            sc.image = oracle.scatter(sc.image, 1, sc.num_blocks, Hkv, d, sc.K[b][:, :t - 1], sc.V[b][:, :t - 1], t - 1, 0,
                                      sc.tables[b])
    sc.upload()
    k_new = np.stack([sc.K[b][0, kv_lens[b] - 1] for b in range(n)])
    v_new = np.stack([sc.V[b][0, kv_lens[b] - 1] for b in range(n)])
    q = synth.normal_bf16(rng, (n, Hq, d))
    shape = B.attn_shape(Hq, Hkv, d)
    ws = torch.empty(B.csv_plan_workspace_bytes(shape, [1] * n, kv_lens), dtype=torch.uint8, device="cuda")
    plan = B.Plan(shape, [1] * n, kv_lens, 0, ws)
    d_out = torch.full((n, Hq, d), 0x7FC0, dtype=torch.int16, device="cuda")
    d_lse = torch.full((n, Hq), float("nan"), dtype=torch.float32, device="cuda")
    B.paged_decode_step(plan, sc.pool, 0, u16_dev(q), u16_dev(k_new), u16_dev(v_new), sc.d_tables, sc.max_blocks, d_out,
                        d_lse)
    torch.cuda.synchronize()
    from harness import dev_to_u16
    assert np.array_equal(dev_to_u16(sc.d_image), full), "pool after the fused step differs from the oracle's scatter"
    O_ref, LSE_ref = oracle_attention(sc, [1] * n, q)
    assert_close(bf16_dev_to_f64(d_out), d_lse.cpu().numpy().astype(np.float64), O_ref, LSE_ref, what="fused step")


def test_tail_step_mixed_batch_one_call(oracle):
    """csv_tail_step (PAPER.md:112 collocated iteration): decode rows and appended chunks of one step in
    one call on layer 1 of a 2-layer pool: every new row's K/V lands where the oracle's scatter puts it (whole pool
    image, layer 0 untouched), O / LSE match the oracle on the full cache; a pure-decode plan takes the fused path."""
    from harness import dev_to_u16
    rng = np.random.default_rng(91)
    Hq, Hkv, d, NL, layer = 32, 8, 128, 2, 1
    kv_lens = [700, 33, 2049, 300, 16, 1, 4097, 129]
    q_lens = [1, 32, 1, 257, 1, 1, 40, 0]
    sc = Scenario(oracle, rng, Hq, Hkv, d, kv_lens, NL=NL, poison=True)
    full = sc.image.copy()
    for b, (t, m) in enumerate(zip(kv_lens, q_lens)):
        full = oracle.scatter(full, NL, sc.num_blocks, Hkv, d, sc.K[b], sc.V[b], t, 0, sc.tables[b])
        # the cache before the step: layer 0 complete, layer 1 without the step's own rows
        K0, V0 = sc.K[b].copy(), sc.V[b].copy()
        sc.image = oracle.scatter(sc.image, NL, sc.num_blocks, Hkv, d, K0[:, :t - m], V0[:, :t - m], t - m, 0, sc.tables[b]) \
            if t - m > 0 else sc.image
        if m > 0:   # layer 0 already holds the step's rows (an earlier layer of the same step), layer 1 does not
            own = oracle.scatter(np.full_like(sc.image, 0), NL, sc.num_blocks, Hkv, d, K0[:, t - m:], V0[:, t - m:], m, t - m,
                                 sc.tables[b])
            mask = oracle.scatter(np.full_like(sc.image, 0), NL, sc.num_blocks, Hkv, d, np.full_like(K0[:, t - m:], 1),
                                  np.full_like(V0[:, t - m:], 1), m, t - m, sc.tables[b]).astype(bool)
            half = sc.image.size // NL
            mask[half:] = False                      # only layer 0
            sc.image = np.where(mask, own, sc.image)
    sc.upload()
    k_new = np.concatenate([sc.K[b][layer, t - m:t] for b, (t, m) in enumerate(zip(kv_lens, q_lens)) if m > 0])
    v_new = np.concatenate([sc.V[b][layer, t - m:t] for b, (t, m) in enumerate(zip(kv_lens, q_lens)) if m > 0])
    total_q = sum(q_lens)
    q = synth.normal_bf16(rng, (total_q, Hq, d))
    shape = B.attn_shape(Hq, Hkv, d)
    ws = torch.empty(B.csv_plan_workspace_bytes(shape, q_lens, kv_lens), dtype=torch.uint8, device="cuda")
    plan = B.Plan(shape, q_lens, kv_lens, 0, ws)
    d_out = torch.full((total_q, Hq, d), 0x7FC0, dtype=torch.int16, device="cuda")
    d_lse = torch.full((total_q, Hq), float("nan"), dtype=torch.float32, device="cuda")
    B.csv_tail_step(plan, sc.pool, layer, u16_dev(q), u16_dev(k_new), u16_dev(v_new), sc.d_tables, sc.max_blocks, d_out, d_lse)
    torch.cuda.synchronize()
    got = dev_to_u16(sc.d_image)
    assert np.array_equal(got, full), "pool after csv_tail_step differs from the oracle's scatter (%d elements)" % int(
        (got != full).sum())
    O_ref, LSE_ref = oracle_attention(sc, q_lens, q, layer=layer)
    assert_close(bf16_dev_to_f64(d_out), d_lse.cpu().numpy().astype(np.float64), O_ref, LSE_ref, what="csv_tail_step")
    with pytest.raises(B.CsvError):
        B.csv_tail_step(plan, sc.pool, 2, u16_dev(q), u16_dev(k_new), u16_dev(v_new), sc.d_tables, sc.max_blocks, d_out, d_lse)
    with pytest.raises(B.CsvError):
        B.csv_tail_step(plan, sc.pool, layer, u16_dev(q), None, u16_dev(v_new), sc.d_tables, sc.max_blocks, d_out, d_lse)


def test_tail_step_both_routes_in_one_process_against_the_oracle(oracle):
    """csv_tail_step has two routes for a mixed step at d = 128: ONE persistent launch (tail_fused.cu) or the decode and
    append kernels back to back.  The planner picks by the decode share of the work; CSV_TUNE_TAIL_TWO_KERNELS /
    CSV_TUNE_TAIL_DECODE_CTAS override it per plan.  Both routes, plus the forced one-launch route on a batch where the
    planner declines it, run here in one process on the same cache and are each compared with the oracle."""
    rng = np.random.default_rng(97)
    Hq, Hkv, d = 32, 8, 128
    convs = [(3000, 1), (6000, 1), (500, 96), (4100, 1), (2500, 1), (1200, 300), (5000, 1), (15, 1)]
    q_lens, kv_lens = [m for _, m in convs], [P + m for P, m in convs]
    sc = Scenario(oracle, rng, Hq, Hkv, d, kv_lens).commit().upload()
    q = synth.normal_bf16(rng, (sum(q_lens), Hq, d))
    O_ref, LSE_ref = oracle_attention(sc, q_lens, q)
    try:
        O1, L1, info1 = run_attention(sc, q_lens, q, which="tail")
        assert info1["tail_n_dec"] > 0                                   # decode-heavy batch: the planner fuses
        assert_close(O1, L1, O_ref, LSE_ref, "one launch")
        B.csv_tuning_set(B.TUNE_TAIL_TWO_KERNELS, 1)
        O2, L2, info2 = run_attention(sc, q_lens, q, which="tail")
        assert_close(O2, L2, O_ref, LSE_ref, "two kernels")
        Ob, Lb, _ = run_attention(sc, q_lens, q, which="both")           # the two public calls: the very same kernels
        assert np.array_equal(O2, Ob) and np.array_equal(L2, Lb)
        B.csv_tuning_set(B.TUNE_TAIL_TWO_KERNELS, 0)
        # a chunk-heavy batch: the planner keeps the two kernels; forcing 20 decode-role CTAs gives the one launch
        convs = [(2000, 1), (9000, 700), (64, 1)]
        q_lens, kv_lens = [m for _, m in convs], [P + m for P, m in convs]
        sc = Scenario(oracle, rng, Hq, Hkv, d, kv_lens).commit().upload()
        q = synth.normal_bf16(rng, (sum(q_lens), Hq, d))
        O_ref, LSE_ref = oracle_attention(sc, q_lens, q)
        O3, L3, info3 = run_attention(sc, q_lens, q, which="tail")
        assert info3["tail_n_dec"] == 0
        assert_close(O3, L3, O_ref, LSE_ref, "planner's choice: two kernels")
        B.csv_tuning_set(B.TUNE_TAIL_DECODE_CTAS, 20)
        O4, L4, info4 = run_attention(sc, q_lens, q, which="tail")
        assert info4["tail_n_dec"] >= 1
        assert_close(O4, L4, O_ref, LSE_ref, "one launch, forced")
    finally:
        for k in (B.TUNE_TAIL_TWO_KERNELS, B.TUNE_TAIL_DECODE_CTAS):
            B.csv_tuning_set(k, 0)


def test_tail_step_host_mixed_batch_two_layers(oracle):
    """csv_tail_step_host with q_lens and n_layers = 2: one plan, one table upload, both layers' new rows written, decode
    rows and appended chunks attended on each layer; host results against the oracle, whole pool against its scatter."""
    from harness import dev_to_u16
    rng = np.random.default_rng(93)
    Hq, Hkv, d, NL = 32, 8, 128, 2
    kv_lens = [700, 33, 2049, 300, 16, 1, 129]
    q_lens = [1, 32, 1, 257, 1, 1, 0]
    sc = Scenario(oracle, rng, Hq, Hkv, d, kv_lens, NL=NL, poison=True)
    full = sc.image.copy()
    for b, (t, m) in enumerate(zip(kv_lens, q_lens)):
        full = oracle.scatter(full, NL, sc.num_blocks, Hkv, d, sc.K[b], sc.V[b], t, 0, sc.tables[b])
        if t - m > 0:   # the cache before the step: both layers without the step's own rows
            sc.image = oracle.scatter(sc.image, NL, sc.num_blocks, Hkv, d, sc.K[b][:, :t - m], sc.V[b][:, :t - m], t - m, 0,
                                      sc.tables[b])
    sc.upload()
    rows = [(b, t, m) for b, (t, m) in enumerate(zip(kv_lens, q_lens)) if m > 0]
    k_new = np.stack([np.concatenate([sc.K[b][l, t - m:t] for b, t, m in rows]) for l in range(NL)])
    v_new = np.stack([np.concatenate([sc.V[b][l, t - m:t] for b, t, m in rows]) for l in range(NL)])
    total_q = sum(q_lens)
    q = synth.normal_bf16(rng, (NL, total_q, Hq, d))
    shape = B.attn_shape(Hq, Hkv, d)
    tabs = np.where(sc.h_tables < 0, 0, sc.h_tables).astype(np.int32)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_out = torch.full((NL, total_q, Hq, d), 0x7FC0, dtype=torch.int16).pin_memory()
    h_lse = torch.full((NL, total_q, Hq), float("nan"), dtype=torch.float32).pin_memory()
    nbytes = B.csv_tail_step_host_workspace_bytes(shape, kv_lens, sc.max_blocks, q_lens=q_lens, n_layers=NL)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    B.csv_tail_step_host(sc.pool, 0, shape, kv_lens, pin(q.view(np.int16)), pin(k_new.view(np.int16)), pin(v_new.view(np.int16)),
                         pin(tabs), sc.max_blocks, ws, h_out, h_lse, q_lens=q_lens, n_layers=NL)
    got = dev_to_u16(sc.d_image)
    assert np.array_equal(got, full), "pool after csv_tail_step_host differs from the oracle's scatter"
    for l in range(NL):
        O = synth.bf16_bits_to_f32(h_out[l].numpy().view(np.uint16)).astype(np.float64)
        O_ref, LSE_ref = oracle_attention(sc, q_lens, q[l], layer=l)
        assert_close(O, h_lse[l].numpy().astype(np.float64), O_ref, LSE_ref, what="host step layer %d" % l)
    with pytest.raises(B.CsvError):   # layers past the pool, and a workspace sized for one layer only
        B.csv_tail_step_host(sc.pool, 1, shape, kv_lens, pin(q.view(np.int16)), pin(k_new.view(np.int16)),
                             pin(v_new.view(np.int16)), pin(tabs), sc.max_blocks, ws, h_out, h_lse, q_lens=q_lens, n_layers=NL)
    small = torch.empty(B.csv_tail_step_host_workspace_bytes(shape, kv_lens, sc.max_blocks, q_lens=q_lens, n_layers=1),
                        dtype=torch.uint8, device="cuda")
    with pytest.raises(B.CsvError):
        B.csv_tail_step_host(sc.pool, 0, shape, kv_lens, pin(q.view(np.int16)), pin(k_new.view(np.int16)),
                             pin(v_new.view(np.int16)), pin(tabs), sc.max_blocks, small, h_out, h_lse, q_lens=q_lens, n_layers=NL)


def test_append_spike_sweep_sees_every_block(oracle):
    """SURVEY §8c item 1 for the tcgen05 kernel: one key carries ~all the weight for every row that may see it and its V
    is a +-1 pattern; the spike sits on the first / last block of each KV partition, around the prefix / chunk boundary
    and on the diagonal.  A dropped, duplicated or misplaced 16-token block (or a wrong mask edge) is an O(1) error."""
    rng = np.random.default_rng(137)
    Hq, Hkv, d, L, m, G = 32, 8, 128, 6001, 40, 4          # 160 stacked rows per KV head: tile A full, tile B ragged
    P = L - m
    positions = sorted(set([0, 15, 16, 2047, 2048, 2049, 4095, 4096, P - 16, P - 1, P, P + 1, P + 17, L - 2, L - 1,
                            (L // 16) * 16, (L // 16) * 16 - 1] + list(rng.integers(0, L, size=5))))
    n = len(positions)
    sc = Scenario(oracle, rng, Hq, Hkv, d, [L] * n)
    # all rows of a chunk share a direction per KV group (plus noise), so one key can dominate every row of the group
    base = rng.standard_normal((n, Hkv, d)).astype(np.float32)
    qf = np.repeat(base, G, axis=1)[:, None] + 0.3 * rng.standard_normal((n, m, Hq, d)).astype(np.float32)
    q = synth.f32_to_bf16_bits(qf.reshape(n * m, Hq, d))
    pattern = np.where(rng.random((n, Hkv, d)) < 0.5, -1.0, 1.0).astype(np.float32)
    for b, j in enumerate(positions):
        for g in range(Hkv):
            u = base[b, g]
            sc.K[b][0, j, g] = synth.f32_to_bf16_bits(u * (22.0 * np.sqrt(d) / np.dot(u, u)))
            sc.V[b][0, j, g] = synth.f32_to_bf16_bits(pattern[b, g])
    sc.commit().upload()
    O, LSE, info = run_attention(sc, [m] * n, q, mpt=2048, which="append")
    assert info["n_append_chunks"] == n
    O_ref, LSE_ref = oracle_attention(sc, [m] * n, q)
    assert_close(O, LSE, O_ref, LSE_ref, what="append spike sweep")
    hit = 0
    for b, j in enumerate(positions):
        for i in range(m):
            if j > P + i:
                continue                                     # the spike is behind the diagonal for this row
            for h in range(Hq):
                r = b * m + i
                if np.abs(O_ref[r, h] - pattern[b, h // G]).max() < 1e-3:
                    assert np.abs(O[r, h] - pattern[b, h // G]).max() <= 1e-2
                    hit += 1
    assert hit > 0.5 * n * m * Hq * 0.8                      # most visible (row, head) pairs are dominated by the spike


def test_append_is_bit_identical_under_block_permutation_and_reruns(oracle):
    # S8 for the append path: the schedule depends only on the lengths -> same bits wherever the blocks sit, run to run
    convs = [(3000, 100), (17, 33), (5000, 40), (0, 64)]
    q_lens = [m for _, m in convs]
    kv = [P + m for P, m in convs]
    outs = []
    for perm_seed in (1, 2):
        rng = np.random.default_rng(140)
        sc = Scenario(oracle, rng, 32, 8, 128, kv)
        q = synth.normal_bf16(rng, (sum(q_lens), 32, 128))
        order = synth.shuffled_free_order(np.random.default_rng(perm_seed), sc.num_blocks)
        pos = 0
        for i, t in enumerate(kv):
            nb = synth.blocks_for(t)
            sc.tables[i] = order[pos:pos + nb].copy()
            pos += nb
        sc.commit().upload()
        for _ in range(2):
            O, LSE, _ = run_attention(sc, q_lens, q, mpt=1024, which="append")
            outs.append((O.copy(), LSE.copy()))
    for O, LSE in outs[1:]:
        assert np.array_equal(O, outs[0][0]) and np.array_equal(LSE, outs[0][1])

"""GPU parity of paged_decode_attn / append_prefill_attn against the fp64 oracle (O1) on the
logical KV, through the C ABI.  Tolerances (north_star): max |O err| <= 1e-2, LSE <= 1e-3;
plus the normalised gate and the adversarial cases of SURVEY §8c (the absolute gate alone
cannot see a dropped block on N(0,1) data).
"""
import numpy as np
import pytest
import torch

from paper_2606_01839_b200 import binding as B
from paper_2606_01839_b200 import synth
from harness import Scenario, assert_close, oracle_abs_weighted, oracle_attention, run_attention

pytestmark = pytest.mark.gpu


def decode_case(oracle, seed, Hq, Hkv, d, kv_lens, mpt=0, poison=False, v_mean=0.0, qscale=1.0, what=""):
    rng = np.random.default_rng(seed)
    sc = Scenario(oracle, rng, Hq, Hkv, d, kv_lens, poison=poison, v_mean=v_mean).commit().upload()
    q_lens = [1] * len(kv_lens)
    q = synth.normal_bf16(rng, (len(kv_lens), Hq, d), std=qscale)
    O, LSE, info = run_attention(sc, q_lens, q, mpt=mpt, which="decode")
    O_ref, LSE_ref = oracle_attention(sc, q_lens, q)
    A_ref = oracle_abs_weighted(sc, q_lens, q) if qscale > 1.0 else None   # peaked softmax: DESIGN.md S20
    return assert_close(O, LSE, O_ref, LSE_ref, what or "decode", A_ref=A_ref), info, (O, LSE)


def test_config1_tiny_decode(oracle):
    # BASELINE.json config 1: 1 layer, 4 conversations, Hq=4, Hkv=1, d=64, context U[64,512], 256-block pool
    kv = synth.config_lengths(1)["kv_lens"]
    rng = np.random.default_rng(0)
    sc = Scenario(oracle, rng, 4, 1, 64, kv, pool_blocks=256).commit().upload()
    q = synth.normal_bf16(rng, (4, 4, 64))
    O, LSE, _ = run_attention(sc, [1] * 4, q, which="decode")
    assert_close(O, LSE, *oracle_attention(sc, [1] * 4, q), what="config 1")


def test_config2_llama8b_decode_full_parity(oracle):
    # BASELINE.json config 2: Hq=32, Hkv=8, d=128, 64 conversations, context U[1024,8192]; whole config vs oracle
    kv = synth.config_lengths(2)["kv_lens"]
    (oerr, lerr), info, _ = decode_case(oracle, 1, 32, 8, 128, kv, what="config 2")
    assert info["decode_grid"] == torch.cuda.get_device_properties(0).multi_processor_count
    print("config 2: max|O err| %.2e  max|LSE err| %.2e  items %d" % (oerr, lerr, info["n_decode_items"]))


@pytest.mark.parametrize("Hq,Hkv,d", [(4, 1, 64), (32, 8, 128), (64, 8, 128), (8, 8, 64), (16, 2, 128), (4, 4, 128)])
def test_decode_length_edge_cases(oracle, Hq, Hkv, d):
    # kv_len in {1, 15, 16, 17, partition-1, partition, partition+1}, mixed with a long one
    kv = [1, 15, 16, 17, 2047, 2048, 2049, 31, 33, 4100]
    decode_case(oracle, 20 + Hq, Hq, Hkv, d, kv, what="edges %s" % ((Hq, Hkv, d),))


def test_decode_poisoned_padding_and_table_tail(oracle):
    # S9: NaN bit patterns in every unused slot / block, out-of-range ids in unused table entries
    kv = [1, 5, 17, 100, 1000, 2050, 15]
    decode_case(oracle, 31, 32, 8, 128, kv, poison=True, what="poison")
    decode_case(oracle, 32, 4, 1, 64, kv, poison=True, what="poison d64")


def test_decode_nonzero_mean_values_make_the_gate_relative(oracle):
    # V ~ N(1,1) gives O ~ 1: the absolute 1e-2 gate becomes a 1 % relative gate
    decode_case(oracle, 33, 32, 8, 128, [3000, 8192, 555, 16384], v_mean=1.0, what="V~N(1,1)")
    decode_case(oracle, 34, 64, 8, 128, [20000, 777], v_mean=1.0, what="V~N(1,1) G=8")


def test_decode_large_magnitude_scores(oracle):
    # q x8 -> max score 30+; partitions whose maxima differ widely must merge without NaN
    decode_case(oracle, 35, 32, 8, 128, [4096, 9000, 100], qscale=8.0, what="q x8")


@pytest.mark.parametrize("mpt", [16, 64, 512, 4096])
def test_decode_result_does_not_depend_on_partition_size(oracle, mpt):
    # S10: forcing several partition sizes changes the result only within tolerance
    decode_case(oracle, 36, 32, 8, 128, [5000, 1234, 8192, 40], mpt=mpt, what="mpt=%d" % mpt)


def test_decode_spike_sweep_sees_every_block(oracle):
    """one key carries ~all the weight and its V is a +-1 pattern; sweeping the
    spike over every block boundary makes a dropped / misplaced block an O(1) error."""
    rng = np.random.default_rng(37)
    Hq, Hkv, d, L = 32, 8, 128, 6001
    positions = sorted(set([0, 1, 15, 16, 17, L - 1, L - 2, (L // 16) * 16, (L // 16) * 16 - 1] +
                           list(range(16 * 7, L, 16 * 29)) + list(range(16 * 11 - 1, L, 16 * 31)) +
                           list(rng.integers(0, L, size=16))))
    n = len(positions)
    sc = Scenario(oracle, rng, Hq, Hkv, d, [L] * n)
    q = synth.normal_bf16(rng, (n, Hq, d))
    qf = synth.bf16_bits_to_f32(q)
    pattern = np.where(rng.random((n, Hkv, d)) < 0.5, -1.0, 1.0).astype(np.float32)
    for b, j in enumerate(positions):
        for g in range(Hkv):
            # K[j] = c * mean of the group's queries, normalised so each head's score at j is >> the N(0,1) rest
            dirv = qf[b, g * 4:(g + 1) * 4].sum(axis=0)
            sc.K[b][0, j, g] = synth.f32_to_bf16_bits(dirv * (22.0 * np.sqrt(d) / np.dot(dirv, dirv) * 4.0))
            sc.V[b][0, j, g] = synth.f32_to_bf16_bits(pattern[b, g])
    sc.commit().upload()
    O, LSE, _ = run_attention(sc, [1] * n, q, which="decode")
    O_ref, LSE_ref = oracle_attention(sc, [1] * n, q)
    assert_close(O, LSE, O_ref, LSE_ref, what="spike sweep")
    # and the closed form: heads whose spike score dominates return the pattern itself
    for b in range(n):
        for h in range(Hq):
            if np.abs(O_ref[b, h] - pattern[b, h // 4]).max() < 1e-3:
                assert np.abs(O[b, h] - pattern[b, h // 4]).max() <= 1e-2
    assert (np.abs(O_ref - np.repeat(pattern, 4, axis=1)).max(axis=-1) < 1e-3).mean() > 0.5


def test_decode_is_bit_identical_under_block_permutation_and_reruns(oracle):
    # S8: the schedule depends only on the lengths -> same bits for any placement of the blocks, run to run
    kv = [3000, 17, 8192, 640]
    outs = []
    for perm_seed in (1, 2):
        rng = np.random.default_rng(40)
        sc = Scenario(oracle, rng, 32, 8, 128, kv)
        q = synth.normal_bf16(rng, (4, 32, 128))
        prng = np.random.default_rng(perm_seed)   # re-place the same logical KV on other blocks
        order = synth.shuffled_free_order(prng, sc.num_blocks)
        pos = 0
        for i, t in enumerate(kv):
            nb = synth.blocks_for(t)
            sc.tables[i] = order[pos:pos + nb].copy()
            pos += nb
        sc.commit().upload()
        for _ in range(2):
            O, LSE, _ = run_attention(sc, [1] * 4, q, which="decode")
            outs.append((O.copy(), LSE.copy()))
    for O, LSE in outs[1:]:
        assert np.array_equal(O, outs[0][0]) and np.array_equal(LSE, outs[0][1])


def test_decode_tolerates_aliased_blocks(oracle):
    # S11: two tables naming the same blocks (shared prefix) read the same KV
    rng = np.random.default_rng(41)
    sc = Scenario(oracle, rng, 32, 8, 128, [1000, 1000])
    sc.K[1], sc.V[1] = sc.K[0], sc.V[0]
    sc.tables[1] = sc.tables[0].copy()
    sc.commit().upload()
    q = synth.normal_bf16(rng, (2, 32, 128))
    O, LSE, _ = run_attention(sc, [1, 1], q, which="decode")
    assert_close(O, LSE, *oracle_attention(sc, [1, 1], q), what="aliased")


def test_decode_row_on_an_empty_cache_gives_zero_and_minus_infinity(oracle):
    # conserve_kv.h a4 / SURVEY §8b: kv_len = 0 -> O = 0, LSE = -inf (the oracle's O1 step 6), next to ordinary rows
    for Hq, Hkv, d in ((32, 8, 128), (4, 1, 64)):
        rng = np.random.default_rng(77)
        kv = [0, 40, 0, 300, 0]
        sc = Scenario(oracle, rng, Hq, Hkv, d, kv, poison=True).commit().upload()
        q = synth.normal_bf16(rng, (len(kv), Hq, d))
        O, LSE, info = run_attention(sc, [1] * len(kv), q, which="decode")
        assert info["n_decode_rows"] == len(kv)
        for b, t in enumerate(kv):
            o_ref, l_ref = oracle.attention(q[b:b + 1], sc.K[b][0][:t], sc.V[b][0][:t])
            if t == 0:
                assert np.all(o_ref == 0.0) and np.all(np.isneginf(l_ref))          # what the oracle says
                assert np.all(O[b] == 0.0) and np.all(np.isneginf(LSE[b])), "empty-cache row %d" % b
            else:
                assert_close(O[b:b + 1], LSE[b:b + 1], o_ref, l_ref, what="row %d beside empty-cache rows" % b)
        # the fused step writes nothing for an empty-cache row and the pool stays as it was
        shape = B.attn_shape(Hq, Hkv, d)
        ws = torch.empty(B.csv_plan_workspace_bytes(shape, [1], [0]), dtype=torch.uint8, device="cuda")
        plan = B.Plan(shape, [1], [0], 0, ws)
        before = sc.d_image.clone()
        d_out = torch.full((1, Hq, d), 0x7FC0, dtype=torch.int16, device="cuda")
        d_lse = torch.zeros((1, Hq), dtype=torch.float32, device="cuda")
        kn = torch.ones(Hkv * d, dtype=torch.int16, device="cuda")
        B.paged_decode_step(plan, sc.pool, 0, torch.zeros(Hq * d, dtype=torch.int16, device="cuda"), kn, kn, sc.d_tables,
                            sc.max_blocks, d_out, d_lse)
        B.kv_append_tokens(sc.pool, plan, kn, kn, sc.d_tables, sc.max_blocks)
        torch.cuda.synchronize()
        assert torch.equal(before, sc.d_image) and bool((d_out == 0).all()) and bool(torch.isneginf(d_lse).all())


def test_decode_on_every_visible_device(oracle):
    # Per-device library state (kernel attributes, SM count): a decode must work on each device in turn inside one
    # process.  On a 1-GPU box this is a set_device round trip followed by a launch; with more GPUs every one runs.
    n = torch.cuda.device_count()
    cur = torch.cuda.current_device()
    try:
        for dev in list(range(n)) + [0]:
            torch.cuda.set_device(dev)
            with torch.cuda.device(dev):
                rng = np.random.default_rng(5 + dev)
                sc = Scenario(oracle, rng, 32, 8, 128, [70, 1000]).commit().upload()
                q = synth.normal_bf16(rng, (3, 32, 128))
                O, LSE, _ = run_attention(sc, [1, 2], q)          # decode kernel + tcgen05 append kernel
                assert_close(O, LSE, *oracle_attention(sc, [1, 2], q), what="device %d" % dev)
    finally:
        torch.cuda.set_device(cur)


def test_attention_argument_errors(oracle):
    rng = np.random.default_rng(42)
    sc = Scenario(oracle, rng, 32, 8, 128, [100]).commit().upload()
    shape = B.attn_shape(32, 8, 128)
    ws = torch.empty(B.csv_plan_workspace_bytes(shape, [1], [100]), dtype=torch.uint8, device="cuda")
    plan = B.Plan(shape, [1], [100], 0, ws)
    q = torch.zeros(32 * 128, dtype=torch.int16, device="cuda")
    out = torch.zeros(32 * 128, dtype=torch.int16, device="cuda")
    lse = torch.zeros(32, dtype=torch.float32, device="cuda")
    host_plan = B.Plan(shape, [1], [100])
    other = B.Plan(B.attn_shape(4, 1, 64), [1], [100], 0, ws)
    for call in (lambda: B.paged_decode_attn(plan, sc.pool, 1, q, sc.d_tables, sc.max_blocks, out, lse),    # layer
                 lambda: B.paged_decode_attn(plan, sc.pool, 0, q, sc.d_tables, 3, out, lse),                # table too short
                 lambda: B.paged_decode_attn(plan, sc.pool, 0, q.data_ptr() + 2, sc.d_tables, 7, out, lse),
                 lambda: B.paged_decode_attn(host_plan, sc.pool, 0, q, sc.d_tables, 7, out, lse),           # host-only plan
                 lambda: B.append_prefill_attn(other, sc.pool, 0, q, sc.d_tables, 7, out, lse)):           # shape mismatch
        with pytest.raises(B.CsvError) as e:
            call()
        assert e.value.code == B.CSV_E_INVAL
    small = torch.empty(128, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.CsvError) as e:
        B.Plan(shape, [1] * 4, [5000] * 4, 0, small)
    assert e.value.code == B.CSV_E_NOMEM

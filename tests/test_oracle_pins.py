"""Pins for oracle/oracle.c against things that are NOT the oracle:
closed forms, invariants, brute force, torch float64 special cases, and the
paper's one worked number.  CPU only.
"""
import math
import os

import numpy as np
import pytest
import torch

from paper_2606_01839_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def f64(bits):
    return synth.bf16_bits_to_f32(bits).astype(np.float64)


def rnd(seed, R, L, Hq, Hkv, d, qscale=1.0):
    rng = np.random.default_rng(seed)
    return (synth.normal_bf16(rng, (R, Hq, d), std=qscale), synth.normal_bf16(rng, (L, Hkv, d)),
            synth.normal_bf16(rng, (L, Hkv, d)))


# ----------------------------------------------------------------- O1 softmax

def test_one_key_returns_that_value(oracle):
    # closed form (north_star): L = 1 -> O = V[0] exactly, LSE = q.K[0]/sqrt(d)
    q, K, V = rnd(1, 1, 1, 8, 2, 64)
    O, LSE = oracle.attention(q, K, V)
    for h in range(8):
        assert np.array_equal(O[0, h], f64(V)[0, h // 4])
        assert LSE[0, h] == pytest.approx(float(f64(q)[0, h] @ f64(K)[0, h // 4]) / 8.0, abs=1e-13)


def test_uniform_keys_give_mean_of_values(oracle):
    # closed form (north_star): all keys equal -> O = mean V, LSE = s + ln L
    q, K, V = rnd(2, 1, 37, 4, 1, 64)
    K[:] = K[0]
    O, LSE = oracle.attention(q, K, V)
    mean = f64(V)[:, 0].mean(axis=0)
    for h in range(4):
        s = float(f64(q)[0, h] @ f64(K)[0, 0]) / 8.0
        assert np.allclose(O[0, h], mean, rtol=0, atol=1e-14)
        assert LSE[0, h] == pytest.approx(s + math.log(37), abs=1e-12)


def test_zero_query_gives_mean_and_log_L(oracle):
    q, K, V = rnd(3, 1, 50, 4, 2, 32)
    q[:] = 0
    O, LSE = oracle.attention(q, K, V)
    for h in range(4):
        assert np.allclose(O[0, h], f64(V)[:, h // 2].mean(axis=0), atol=1e-14)
        assert LSE[0, h] == pytest.approx(math.log(50), abs=1e-13)


def test_dominant_key(oracle):
    # K[j*] = 40 q/|q|, others 0: O -> V[j*] within L*exp(-gap), LSE -> s_j*
    rng = np.random.default_rng(4)
    d, L, js = 64, 100, 63
    qf = rng.standard_normal(d).astype(np.float32)
    q = synth.f32_to_bf16_bits(qf).reshape(1, 1, d)
    K = np.zeros((L, 1, d), dtype=np.uint16)
    K[js, 0] = synth.f32_to_bf16_bits(40.0 * qf / np.linalg.norm(qf))
    V = synth.normal_bf16(rng, (L, 1, d))
    O, LSE = oracle.attention(q, K, V)
    s = float(f64(q)[0, 0] @ f64(K)[js, 0]) / math.sqrt(d)
    assert s > 30
    bound = L * math.exp(-s) * 8
    assert np.max(np.abs(O[0, 0] - f64(V)[js, 0])) < bound
    assert abs(LSE[0, 0] - s) < bound


def test_key_shift_invariance(oracle):
    # adding u to every key: O unchanged, LSE moves by q.u/sqrt(d)
    rng = np.random.default_rng(5)
    q, K, V = rnd(5, 1, 40, 2, 1, 32)
    u = rng.integers(-2, 3, size=32).astype(np.float32)  # small integers: K+u exact in bf16? keep K integer too
    K = synth.f32_to_bf16_bits(rng.integers(-3, 4, size=(40, 1, 32)).astype(np.float32))
    K2 = synth.f32_to_bf16_bits(synth.bf16_bits_to_f32(K) + u)
    O1, L1 = oracle.attention(q, K, V)
    O2, L2 = oracle.attention(q, K2, V)
    assert np.allclose(O1, O2, atol=1e-13)
    for h in range(2):
        assert L2[0, h] - L1[0, h] == pytest.approx(float(f64(q)[0, h] @ u.astype(np.float64)) / math.sqrt(32), abs=1e-12)


def test_value_affine_map(oracle):
    # weights sum to 1: V -> a V + b  =>  O -> a O + b  (a, b powers of two: exact in bf16)
    rng = np.random.default_rng(6)
    q = synth.normal_bf16(rng, (1, 4, 64))
    K = synth.normal_bf16(rng, (33, 2, 64))
    Vf = rng.integers(-8, 9, size=(33, 2, 64)).astype(np.float32)
    O1, _ = oracle.attention(q, K, synth.f32_to_bf16_bits(Vf))
    O2, _ = oracle.attention(q, K, synth.f32_to_bf16_bits(2.0 * Vf + 4.0))
    assert np.allclose(O2, 2.0 * O1 + 4.0, atol=1e-12)


def test_one_hot_values_read_out_softmax_weights(oracle):
    # V = indicator of token j in channel 0 -> O[...,0] = exp(s_j - LSE)
    q, K, _ = rnd(7, 1, 20, 2, 2, 16)
    Ksc = f64(K)
    for j in (0, 7, 19):
        V = np.zeros((20, 2, 16), dtype=np.uint16)
        V[j, :, 0] = 0x3F80  # 1.0
        O, LSE = oracle.attention(q, K, V)
        for h in range(2):
            s_j = float(f64(q)[0, h] @ Ksc[j, h]) / 4.0
            assert O[0, h, 0] == pytest.approx(math.exp(s_j - LSE[0, h]), rel=1e-12)
            assert np.all(O[0, h, 1:] == 0)


# -------------------------------------------------------------------- O1 GQA

def test_gqa_same_query_same_row(oracle):
    q, K, V = rnd(8, 1, 30, 8, 2, 32)
    q[0, 1:4] = q[0, 0]
    q[0, 4] = q[0, 0]  # other group, same q
    O, LSE = oracle.attention(q, K, V)
    for h in (1, 2, 3):
        assert np.array_equal(O[0, h], O[0, 0]) and LSE[0, h] == LSE[0, 0]
    assert not np.allclose(O[0, 4], O[0, 0])  # different KV head


def test_gqa_equals_mha_on_repeated_heads(oracle):
    q, K, V = rnd(9, 3, 25, 8, 2, 32)
    O, LSE = oracle.attention(q, K, V)
    Kx, Vx = np.repeat(K, 4, axis=1), np.repeat(V, 4, axis=1)
    O2, LSE2 = oracle.attention(q, Kx, Vx)
    assert np.allclose(O, O2, atol=1e-15) and np.allclose(LSE, LSE2, atol=1e-15)


def test_head_group_is_contiguous(oracle):
    # S2: head h reads KV head h // G (not h % Hkv)
    q, K, V = rnd(10, 1, 5, 4, 2, 16)
    O, _ = oracle.attention(q, K, V)
    Oa, _ = oracle.attention(q[:, 1:2], K[:, 0:1], V[:, 0:1])
    Ob, _ = oracle.attention(q[:, 2:3], K[:, 1:2], V[:, 1:2])
    assert np.array_equal(O[0, 1], Oa[0, 0]) and np.array_equal(O[0, 2], Ob[0, 0])


# ----------------------------------------------------------------- O1 causal

def test_append_row_equals_decode_on_truncated_cache(oracle):
    # row i with prefix P sees keys 0..P+i: identical to decode with kv_len = P+i+1
    q, K, V = rnd(11, 6, 29, 4, 2, 32)
    O, LSE = oracle.attention(q, K, V)
    P = 29 - 6
    for i in range(6):
        Od, Ld = oracle.attention(q[i:i + 1], K[:P + i + 1], V[:P + i + 1])
        assert np.array_equal(O[i], Od[0]) and np.array_equal(LSE[i], Ld[0])


def test_full_causal_prefill_matches_torch_sdpa(oracle):
    q, K, V = rnd(12, 24, 24, 4, 4, 32)
    O, _ = oracle.attention(q, K, V)
    tq = torch.from_numpy(f64(q)).permute(1, 0, 2)[None]
    tk = torch.from_numpy(f64(K)).permute(1, 0, 2)[None]
    tv = torch.from_numpy(f64(V)).permute(1, 0, 2)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, is_causal=True)[0].permute(1, 0, 2).numpy()
    assert np.allclose(O, ref, atol=1e-12)


def test_empty_cache(oracle):
    q = np.zeros((0, 4, 16), dtype=np.uint16)
    K = np.zeros((0, 2, 16), dtype=np.uint16)
    O, LSE = oracle.attention(q, K, K)
    assert O.shape == (0, 4, 16) and LSE.shape == (0, 4)


def test_decode_row_on_an_empty_cache_is_zero_and_minus_infinity(oracle):
    # SURVEY 8c O1 step 6 / conserve_kv.h a4: a decode row with no key to attend to gives O = 0, LSE = -inf.  It is
    # also the limit of the merge identity: merging it with any other part leaves that part unchanged.
    q = synth.normal_bf16(np.random.default_rng(3), (1, 4, 16))
    K = np.zeros((0, 2, 16), dtype=np.uint16)
    O, LSE = oracle.attention(q, K, K)
    assert O.shape == (1, 4, 16) and np.all(O == 0.0) and np.all(np.isneginf(LSE))
    Kb = synth.normal_bf16(np.random.default_rng(4), (5, 2, 16))
    Vb = synth.normal_bf16(np.random.default_rng(5), (5, 2, 16))
    Ob, Lb = oracle.attention(q, Kb[:1], Vb[:1])     # R = 1, L = 1 is the smallest ordinary case
    for h in range(4):
        Om, Lm = oracle.merge(O[0, h], LSE[0, h], Ob[0, h], Lb[0, h])
        assert np.allclose(Om, Ob[0, h], atol=1e-15) and abs(Lm - Lb[0, h]) <= 1e-15
    with pytest.raises(ValueError):                  # R > L stays an error everywhere else
        oracle.attention(np.zeros((2, 4, 16), dtype=np.uint16), Kb[:1], Vb[:1])


# ------------------------------------------------------------------ O1 whole

def test_brute_force_tiny(oracle):
    # a second, naive evaluation: explicit exp of every score, no max-subtraction, python floats / longdouble
    for seed in range(5):
        rng = np.random.default_rng(100 + seed)
        R, L, Hq, Hkv, d = 2, int(rng.integers(2, 9)), 4, 2, 4
        q, K, V = rnd(200 + seed, R, L, Hq, Hkv, d)
        O, LSE = oracle.attention(q, K, V)
        qf, Kf, Vf = (f64(x).astype(np.longdouble) for x in (q, K, V))
        for i in range(R):
            for h in range(Hq):
                g = h // (Hq // Hkv)
                n = L - R + i + 1
                w = [np.exp(sum(qf[i, h, c] * Kf[j, g, c] for c in range(d)) / np.sqrt(np.longdouble(d))) for j in range(n)]
                Z = sum(w)
                for c in range(d):
                    assert float(sum(w[j] * Vf[j, g, c] for j in range(n)) / Z) == pytest.approx(O[i, h, c], abs=1e-12)
                assert float(np.log(Z)) == pytest.approx(LSE[i, h], abs=1e-12)


@pytest.mark.parametrize("Hq,Hkv,d,L", [(4, 1, 64, 300), (32, 8, 128, 700)])
def test_matches_torch_float64_at_config_shapes(oracle, Hq, Hkv, d, L):
    q, K, V = rnd(13, 1, L, Hq, Hkv, d)
    O, LSE = oracle.attention(q, K, V)
    G = Hq // Hkv
    tq = torch.from_numpy(f64(q))[0]                                    # [Hq, d]
    tk = torch.from_numpy(f64(K)).repeat_interleave(G, dim=1)            # [L, Hq, d]
    tv = torch.from_numpy(f64(V)).repeat_interleave(G, dim=1)
    s = torch.einsum("hc,jhc->hj", tq, tk) / math.sqrt(d)
    ref = torch.einsum("hj,jhc->hc", torch.softmax(s, -1), tv).numpy()
    assert np.allclose(O[0], ref, atol=1e-13)
    assert np.allclose(LSE[0], torch.logsumexp(s, -1).numpy(), atol=1e-12)


def test_large_scores_do_not_overflow(oracle):
    q, K, V = rnd(14, 1, 64, 4, 1, 64, qscale=40.0)
    O, LSE = oracle.attention(q, K, V)
    assert np.all(np.isfinite(O)) and np.all(np.isfinite(LSE)) and LSE.max() > 100


# ------------------------------------------------------------------ O4 merge

def test_merge_of_parts_equals_whole(oracle):
    rng = np.random.default_rng(15)
    q, K, V = rnd(15, 1, 257, 2, 1, 32)
    O, LSE = oracle.attention(q, K, V)
    for nparts in (2, 3, 7, 64):
        cuts = np.sort(rng.choice(np.arange(1, 257), size=nparts - 1, replace=False))
        bounds = [0, *cuts.tolist(), 257]
        parts = [oracle.attention(q, K[a:b], V[a:b]) for a, b in zip(bounds[:-1], bounds[1:])]
        order = rng.permutation(nparts)  # associative + commutative: any order
        for h in range(2):
            accO, accL = np.zeros(32), -np.inf
            for p in order:
                accO, accL = oracle.merge(accO, accL, parts[p][0][0, h], parts[p][1][0, h])
            assert np.allclose(accO, O[0, h], atol=1e-12) and accL == pytest.approx(LSE[0, h], abs=1e-12)


def test_merge_with_underflowing_side(oracle):
    a = np.ones(4)
    b = np.full(4, 7.0)
    O, lse = oracle.merge(a, 100.0, b, -900.0)  # exp(-1000) underflows: no NaN, side a wins
    assert np.array_equal(O, a) and lse == 100.0
    O, lse = oracle.merge(a, -np.inf, b, 3.0)
    assert np.array_equal(O, b) and lse == 3.0
    O, lse = oracle.merge(a, -np.inf, b, -np.inf)
    assert np.all(O == 0) and lse == -np.inf


# ------------------------------------------------- O2 / O3 layout and scatter

def mk_pool(rng, NL, nb, Hkv, d):
    return synth.random_bits(rng, NL * nb * 2 * Hkv * 16 * d)


def test_pool_addr_is_a_bijection_and_tiles_are_contiguous(oracle):
    NL, nb, Hkv, d = 2, 3, 2, 128
    seen = np.zeros(oracle.pool_elems(NL, nb, Hkv, d), dtype=np.int32)
    for layer in range(NL):
        for block in range(nb):
            for kv in range(2):
                for head in range(Hkv):
                    tile = ((layer * nb + block) * 2 + kv) * Hkv + head
                    for slot in range(16):
                        for c in range(0, d):
                            a = oracle.pool_addr(nb, Hkv, d, layer, block, kv, head, slot, c)
                            assert tile * 16 * d <= a < (tile + 1) * 16 * d
                            seen[a] += 1
    assert np.all(seen == 1)


def test_in_tile_format_is_the_128B_swizzle(oracle):
    # hand-typed expectations for a few elements (bf16 units): rows of 64 elements per half,
    # 16-byte chunks XOR-ed with slot % 8; element order inside a chunk kept.
    A = lambda slot, c: oracle.pool_addr(1, 1, 128, 0, 0, 0, 0, slot, c)
    assert A(0, 0) == 0 and A(0, 7) == 7 and A(0, 8) == 8 and A(0, 63) == 63
    assert A(0, 64) == 1024 and A(0, 127) == 1024 + 63          # second half starts after 16 rows x 64
    assert A(1, 0) == 64 + 8 and A(1, 8) == 64 + 0               # slot 1: chunk 0 <-> chunk 1
    assert A(5, 17) == 5 * 64 + ((2 ^ 5) * 8) + 1
    assert A(9, 3) == 9 * 64 + ((0 ^ 1) * 8) + 3                 # slot 9 swizzles like slot 1
    assert A(15, 64 + 56 + 2) == 1024 + 15 * 64 + ((7 ^ 7) * 8) + 2
    # consecutive 8-element chunks stay contiguous 16-byte units
    for slot in range(16):
        for ch in range(16):
            base = A(slot, ch * 8)
            assert base % 8 == 0 and [A(slot, ch * 8 + e) for e in range(8)] == list(range(base, base + 8))


def test_gather_inverts_scatter_and_scatter_touches_exactly_its_elements(oracle):
    rng = np.random.default_rng(16)
    NL, nb, Hkv, d = 2, 12, 2, 64
    for tokens, off in ((37, 0), (5, 11), (16, 16), (1, 47), (20, 13)):
        pool = mk_pool(rng, NL, nb, Hkv, d)
        table = rng.permutation(nb)[: (off + tokens + 15) // 16].astype(np.int32)
        k = synth.random_bits(rng, (NL, tokens, Hkv, d))
        v = synth.random_bits(rng, (NL, tokens, Hkv, d))
        # make every written value differ from what was there, so the changed-element count is exact
        out = oracle.scatter(pool, NL, nb, Hkv, d, k, v, tokens, off, table)
        ref_changed = 0
        for layer in range(NL):
            Kg, Vg = oracle.gather(out, nb, Hkv, d, layer, table, off + tokens)
            assert np.array_equal(Kg[off:], k[layer]) and np.array_equal(Vg[off:], v[layer])
            K0, V0 = oracle.gather(pool, nb, Hkv, d, layer, table, off + tokens)
            assert np.array_equal(Kg[:off], K0[:off]) and np.array_equal(Vg[:off], V0[:off])  # prefix untouched
            ref_changed += int((K0[off:] != k[layer]).sum() + (V0[off:] != v[layer]).sum())
        assert int((out != pool).sum()) == ref_changed <= 2 * NL * tokens * Hkv * d


def test_scatter_identity_table_is_a_transposition(oracle):
    # identity table, tokens multiple of 16, one layer: pool viewed as
    # [block][kv][head][half][slot][chunk][8] must equal a numpy transpose + chunk XOR of the source
    rng = np.random.default_rng(17)
    nb, Hkv, d, tokens = 3, 2, 128, 48
    k = synth.random_bits(rng, (1, tokens, Hkv, d))
    v = synth.random_bits(rng, (1, tokens, Hkv, d))
    out = oracle.scatter(np.zeros(nb * 2 * Hkv * 16 * d, np.uint16), 1, nb, Hkv, d, k, v, tokens, 0, np.arange(nb, dtype=np.int32))
    img = out.reshape(nb, 2, Hkv, 2, 16, 8, 8)
    for kv, src in ((0, k), (1, v)):
        s = src.reshape(nb, 16, Hkv, 2, 8, 8).transpose(0, 2, 3, 1, 4, 5)  # [block][head][half][slot][chunk][8]
        for slot in range(16):
            perm = [ch ^ (slot % 8) for ch in range(8)]                     # physical chunk p holds logical chunk p ^ slot
            assert np.array_equal(img[:, kv, :, :, slot, :, :], s[:, :, :, slot, perm, :])


def test_scatter_by_hand_on_a_4_block_pool(oracle):
    # brute force: offset and length not multiples of 16; expected image built with python loops
    # and an address formula typed here from DESIGN.md's prose (not imported from anywhere)
    rng = np.random.default_rng(18)
    NL, nb, Hkv, d, tokens, off = 1, 4, 1, 64, 21, 9
    table = np.array([2, 0, 3, 1], dtype=np.int32)
    pool = mk_pool(rng, NL, nb, Hkv, d)
    k = synth.random_bits(rng, (NL, tokens, Hkv, d))
    v = synth.random_bits(rng, (NL, tokens, Hkv, d))
    exp = pool.copy()
    for t in range(tokens):
        pos = off + t
        block, slot = int(table[pos // 16]), pos % 16
        for c in range(d):
            inner = slot * 64 + (((c // 8) ^ (slot % 8)) * 8) + c % 8
            exp[(block * 2 + 0) * 16 * d + inner] = k[0, t, 0, c]
            exp[(block * 2 + 1) * 16 * d + inner] = v[0, t, 0, c]
    assert np.array_equal(oracle.scatter(pool, NL, nb, Hkv, d, k, v, tokens, off, table), exp)


def test_paging_invariance_is_bit_exact(oracle):
    # permuting the blocks and the table together leaves attention bit-identical (north_star)
    rng = np.random.default_rng(19)
    nb, Hkv, d, L = 16, 2, 64, 200
    k = synth.normal_bf16(rng, (1, L, Hkv, d))
    v = synth.normal_bf16(rng, (1, L, Hkv, d))
    q = synth.normal_bf16(rng, (1, 8, d))
    res = []
    for _ in range(3):
        table = rng.permutation(nb)[:13].astype(np.int32)
        pool = oracle.scatter(mk_pool(rng, 1, nb, Hkv, d), 1, nb, Hkv, d, k, v, L, 0, table)
        Kg, Vg = oracle.gather(pool, nb, Hkv, d, 0, table, L)
        res.append(oracle.attention(q, Kg, Vg))
    for O, LSE in res[1:]:
        assert np.array_equal(O, res[0][0]) and np.array_equal(LSE, res[0][1])


def test_staging_message_is_a_scatter_into_consecutive_blocks(oracle):
    # the message = what a scatter into a fresh zero pool with the identity table holds,
    # reordered from [layer][block] pools to [layer][tb]: same thing when the pool has exactly ntb blocks
    rng = np.random.default_rng(20)
    NL, Hkv, d = 3, 2, 128
    for tokens, off in ((300, 0), (1, 5), (33, 30)):
        k = synth.random_bits(rng, (NL, tokens, Hkv, d))
        v = synth.random_bits(rng, (NL, tokens, Hkv, d))
        slot0 = off % 16
        ntb = (slot0 + tokens + 15) // 16
        msg = oracle.staging_message(NL, Hkv, d, k, v, tokens, off)
        assert msg.size == oracle.staging_elems(NL, Hkv, d, tokens, off) == NL * ntb * 2 * Hkv * 16 * d
        pool = oracle.scatter(np.zeros(msg.size, np.uint16), NL, ntb, Hkv, d, k, v, tokens, slot0, np.arange(ntb, dtype=np.int32))
        assert np.array_equal(msg, pool)


# --------------------------------------------------------------- host rules

def test_provisioning_worked_example_from_the_paper(oracle):
    with open(os.path.join(GOLDEN, "provisioning_example.txt")) as f:
        rows = [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]
    T_p, L_in, T_d, L_d, n_expected, n_deployed = (float(x) for x in rows[0])
    rate, n_thr, n_mem, N = oracle.provision(T_p, L_in, T_d, L_d, B=1e9, W=1.0)  # memory constraint slack
    assert round(n_thr, 2) == n_expected           # "at least 1.67 decoders per prefiller"
    assert rate == pytest.approx(25000 / 15000)
    assert N == 2 and N <= n_deployed               # the paper deploys 3 (> 1.67)
    # 1.634 conv/s holds the prefiller at saturation -> mean turn-1 length ~15.3k ~ "15k"
    assert 25000 / 1.634 == pytest.approx(15300, rel=0.01)
    # Eq. 2 binds when slots are scarce: R*W/B
    _, n_thr2, n_mem2, N2 = oracle.provision(25000, 15000, 1000, 1000, B=20, W=60)
    assert n_mem2 == pytest.approx(5.0) and N2 == 5
    with pytest.raises(ValueError):
        oracle.provision(0, 1, 1, 1, 1, 1)


def test_placement_rule(oracle):
    # PAPER.md:178 lowest occupancy; ties -> lowest index; full decoders skipped; none fits -> -1
    assert oracle.place([10, 5, 7], [100, 100, 100], 1) == 1
    assert oracle.place([5, 5, 5], [100, 100, 100], 1) == 0
    assert oracle.place([10, 30], [100, 400], 1) == 1          # 0.10 vs 0.075: ratio, not count
    assert oracle.place([99, 50], [100, 100], 5) == 1          # decoder 0 cannot hold 5 more
    assert oracle.place([0, 50], [4, 100], 5) == 1
    assert oracle.place([100, 100], [100, 100], 1) == -1

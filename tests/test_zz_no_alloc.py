"""paged_decode_attn_static: the decode attention call for users who cannot allocate device memory.

Why it exists: a decoder process usually gives all of its HBM to the KV pool when it starts, and a decode step that
runs inside a serving engine is often forbidden to call cudaMalloc / cudaFree (they can fail in the middle of a
request and they stall every stream of the GPU while they run).  Such a caller has no workspace tensor to hand to
csv_plan_create.  The static variant keeps the split-K lists and partials in a fixed 8 MiB array inside the library
(one per GPU, shared by all calls) and takes only inputs and outputs.

What is checked: its output equals the ordinary Plan + workspace path (paged_decode_attn) on the same inputs, for two
calls made back to back on one stream with no synchronisation between them, the second with a different batch so
that it runs over whatever the first left in the shared array; a step over the 8 MiB limit is refused and writes
nothing; a small case is also compared with the CPU oracle.  The file name sorts last on purpose: under `pytest -x`
a failure here cannot hide any other test, and it must pass both alone in a fresh process and after the others.
"""
import numpy as np
import pytest
import torch

from paper_2606_01839_b200 import binding as B
from paper_2606_01839_b200 import synth
from paper_2606_01839_b200.workloads import TailWorkload
from harness import LSE_TOL, O_TOL, Scenario, assert_close, bf16_dev_to_f64, oracle_attention, u16_dev

pytestmark = pytest.mark.gpu

NAN_BF16 = 0x7FC0


def fresh_outputs(rows, Hq, d):
    out = torch.full((rows, Hq, d), NAN_BF16, dtype=torch.int16, device="cuda")   # NaN everywhere: every row must be written
    lse = torch.full((rows, Hq), float("nan"), dtype=torch.float32, device="cuda")
    return out, lse


def existing_path(wl, mpt=0):
    """The route every other test uses: csv_plan_create over a caller-owned workspace, then paged_decode_attn."""
    out, lse = fresh_outputs(wl.total_q, wl.Hq, wl.d)
    ws = torch.empty(max(128, B.csv_plan_workspace_bytes(wl.shape, wl.q_lens, wl.kv_lens, mpt)), dtype=torch.uint8, device="cuda")
    plan = B.Plan(wl.shape, wl.q_lens, wl.kv_lens, mpt, ws)
    B.paged_decode_attn(plan, wl.pool, 0, wl.d_q, wl.d_tables, wl.max_blocks, out, lse)
    torch.cuda.synchronize()
    info = plan.info()
    plan.destroy()
    return out, lse, info


def same_within_test_tolerance(got, want, what):
    (o, l), (o_ref, l_ref) = got, want
    O, O_ref = bf16_dev_to_f64(o), bf16_dev_to_f64(o_ref)
    L, L_ref = l.cpu().numpy().astype(np.float64), l_ref.cpu().numpy().astype(np.float64)
    assert not np.isnan(O).any() and not np.isnan(L).any(), "%s: a row was left unwritten" % what
    fin = np.isfinite(L_ref)   # an empty cache has LSE = -inf on both routes
    assert np.array_equal(fin, np.isfinite(L)) and np.array_equal(L[~fin], L_ref[~fin]), "%s: -inf rows differ" % what
    assert np.abs(O - O_ref).max() <= O_TOL, "%s: O differs from paged_decode_attn by %.3e" % (what, np.abs(O - O_ref).max())
    lerr = np.abs(L[fin] - L_ref[fin]).max()
    assert lerr <= LSE_TOL, "%s: LSE differs from paged_decode_attn by %.3e" % (what, lerr)
    # same plan, same kernels, deterministic merge order: the two routes in fact agree to the bit
    assert torch.equal(o, o_ref) and torch.equal(l, l_ref), "%s: within tolerance but not bit-identical" % what


def test_static_scratch_decode_equals_the_workspace_path_on_two_calls_in_a_row():
    # call 1: BASELINE.json configs[1] (8B shape, 64 conversations, context U[1024, 8192]): every SM busy, ~900 partials
    kv1 = synth.config_lengths(2)["kv_lens"]
    w1 = TailWorkload(32, 8, 128, [1] * len(kv1), kv1, seed=41)
    # call 2: another batch and GQA group on its own pool (ragged lengths, one empty cache, a forced partition size), so it
    # lays different lists and fewer partials over what call 1 left in the shared array
    kv2 = [1, 15, 16, 17, 0, 2049, 40000, 333, 9000]
    w2 = TailWorkload(64, 8, 128, [1] * len(kv2), kv2, seed=42)
    ref1, ref2 = existing_path(w1), existing_path(w2, mpt=2048)
    assert ref1[2]["n_decode_items"] > len(kv1) * 8 and ref2[2]["n_decode_items"] > len(kv2) * 8   # both really split K

    o1, l1 = fresh_outputs(w1.total_q, w1.Hq, w1.d)
    o2, l2 = fresh_outputs(w2.total_q, w2.Hq, w2.d)
    o3, l3 = fresh_outputs(w1.total_q, w1.Hq, w1.d)
    # back to back on the current stream, nothing in between: stream order alone must keep them apart
    B.paged_decode_attn_static(w1.pool, 0, w1.shape, w1.kv_lens, w1.d_q, w1.d_tables, w1.max_blocks, o1, l1)
    B.paged_decode_attn_static(w2.pool, 0, w2.shape, w2.kv_lens, w2.d_q, w2.d_tables, w2.max_blocks, o2, l2,
                               max_partition_tokens=2048)
    B.paged_decode_attn_static(w1.pool, 0, w1.shape, w1.kv_lens, w1.d_q, w1.d_tables, w1.max_blocks, o3, l3)
    torch.cuda.synchronize()
    same_within_test_tolerance((o1, l1), ref1[:2], "first call")
    same_within_test_tolerance((o2, l2), ref2[:2], "second call (over the first call's leftovers)")
    same_within_test_tolerance((o3, l3), ref1[:2], "first batch again")
    empty = kv2.index(0)   # the empty cache keeps paged_decode_attn's convention: O = 0, LSE = -inf
    assert not o2[empty].any() and torch.isinf(l2[empty]).all() and (l2[empty] < 0).all()


def test_static_scratch_decode_against_the_oracle(oracle):
    rng = np.random.default_rng(43)
    kv = [700, 16, 5000, 1, 2500]
    sc = Scenario(oracle, rng, 32, 8, 128, kv).commit().upload()
    q = synth.normal_bf16(rng, (len(kv), 32, 128))
    for _ in range(2):   # twice: the second run starts from the first one's scratch contents
        out, lse = fresh_outputs(len(kv), 32, 128)
        B.paged_decode_attn_static(sc.pool, 0, B.attn_shape(32, 8, 128), kv, u16_dev(q), sc.d_tables, sc.max_blocks, out, lse,
                                   max_partition_tokens=512)
        torch.cuda.synchronize()
        assert_close(bf16_dev_to_f64(out), lse.cpu().numpy().astype(np.float64), *oracle_attention(sc, [1] * len(kv), q),
                     what="static scratch vs oracle")


def test_static_scratch_decode_refuses_a_step_over_its_limit():
    kv = [8192] * 16
    wl = TailWorkload(32, 8, 128, [1] * len(kv), kv, seed=44)
    need = B.csv_plan_workspace_bytes(wl.shape, wl.q_lens, kv, 16)   # a partition per block: ~67k partials of 2 KiB
    assert need > B.STATIC_SCRATCH_BYTES
    out, lse = fresh_outputs(wl.total_q, wl.Hq, wl.d)
    with pytest.raises(B.CsvError) as e:
        B.paged_decode_attn_static(wl.pool, 0, wl.shape, kv, wl.d_q, wl.d_tables, wl.max_blocks, out, lse, max_partition_tokens=16)
    assert e.value.code == B.CSV_E_NOMEM and str(B.STATIC_SCRATCH_BYTES) in str(e.value)
    torch.cuda.synchronize()
    assert (out == NAN_BF16).all()   # nothing was launched
    assert torch.isnan(lse).all()
    # the same lengths at the default partitioning fit, and the call after a refusal works
    B.paged_decode_attn_static(wl.pool, 0, wl.shape, kv, wl.d_q, wl.d_tables, wl.max_blocks, out, lse)
    torch.cuda.synchronize()
    same_within_test_tolerance((out, lse), existing_path(wl)[:2], "after a refused call")
    with pytest.raises(B.CsvError) as e:   # bad arguments are refused before anything is built
        B.paged_decode_attn_static(wl.pool, 1, wl.shape, kv, wl.d_q, wl.d_tables, wl.max_blocks, out, lse)
    assert e.value.code == B.CSV_E_INVAL
    with pytest.raises(B.CsvError) as e:
        B.paged_decode_attn_static(wl.pool, 0, wl.shape, kv, wl.d_q, wl.d_tables, wl.max_blocks - 1, out, lse)
    assert e.value.code == B.CSV_E_INVAL

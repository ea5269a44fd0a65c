"""CPU-only tests of the library's host logic: symbol export, allocator (vs a set model),
placement, provisioning, split-K planner coverage.
No compute call is made here (no GPU on this box); device pointers are fake, aligned integers.
"""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2606_01839_b200 import binding as B
from paper_2606_01839_b200 import build as libbuild
from paper_2606_01839_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FAKE = 0x7F0000000000  # never dereferenced by host-only calls


@pytest.fixture(scope="module", autouse=True)
def built():
    libbuild.build_library()


def mkpool(nblocks, NL=1, Hkv=8, d=128):
    desc = B.pool_desc(NL, nblocks, Hkv, d)
    return B.KvPool(desc, FAKE, B.kv_pool_bytes(desc))


def test_library_exports_every_symbol_the_header_declares():
    hdr = open(os.path.join(ROOT, "include", "conserve_kv.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b([a-z_0-9]+)\s*\([^;{]*\)\s*;", hdr))
    assert len(declared) >= 28
    L = ctypes.CDLL(B.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), "libconserve_kv.so does not export %s" % name
    assert declared == set(B.SYMBOLS)


def test_pool_bytes_and_shape_checks():
    assert B.kv_pool_bytes(B.pool_desc(1, 256, 1, 64)) == 256 * 2 * 1 * 16 * 64 * 2
    assert B.kv_pool_bytes(B.pool_desc(32, 100, 8, 128)) == 32 * 100 * 2 * 8 * 4096
    assert B.kv_pool_bytes(B.pool_desc(1, 10, 8, 96)) == 0          # unsupported head_dim
    assert B.kv_pool_bytes(B.pool_desc(1, 10, 8, 128, block_size=32)) == 0
    with pytest.raises(B.CsvError) as e:
        B.KvPool(B.pool_desc(1, 10, 8, 128), FAKE + 8, 1 << 30)      # misaligned base
    assert e.value.code == B.CSV_E_INVAL
    with pytest.raises(B.CsvError):
        B.KvPool(B.pool_desc(1, 10, 8, 128), FAKE, 100)              # too few bytes
    d = B.pool_desc(2, 10, 8, 128)
    assert B.kv_staging_bytes(d, 300, 0) == 2 * 19 * 2 * 8 * 4096
    assert B.kv_staging_bytes(d, 1, 15) == 2 * 1 * 2 * 8 * 4096
    assert B.kv_staging_bytes(d, 2, 15) == 2 * 2 * 2 * 8 * 4096
    assert B.kv_staging_bytes(d, 0, 0) == 0


def test_allocator_against_a_set_model():
    rng = np.random.default_rng(0)
    n = 97
    pool = mkpool(n)
    order = synth.shuffled_free_order(rng, n)
    pool.set_free_order(order)
    free = list(order)
    held = []
    for step in range(400):
        if rng.random() < 0.55:
            k = int(rng.integers(0, 12))
            if k > len(free):
                with pytest.raises(B.CsvError) as e:
                    pool.alloc_blocks(k)
                assert e.value.code == B.CSV_E_NOMEM
            else:
                got = pool.alloc_blocks(k)
                assert list(got) == free[:k]          # hand-out order = installed order
                free = free[k:]
                held.append(list(got))
        elif held:
            ids = held.pop(int(rng.integers(0, len(held))))
            pool.free_blocks(ids)
            free += ids                                # freed ids go to the tail, in the order given
        assert pool.used_blocks == n - len(free)
        assert pool.free_count == len(free) and pool.num_blocks == n


def test_allocator_rejects_bad_frees_without_changing_anything():
    pool = mkpool(8)
    a = pool.alloc_blocks(3)
    for bad in ([a[0], a[0]], [99], [-1], [7], [a[1], 7]):
        with pytest.raises(B.CsvError) as e:
            pool.free_blocks(bad)
        assert e.value.code == B.CSV_E_INVAL
        assert pool.used_blocks == 3
    pool.free_blocks(a)
    assert pool.used_blocks == 0
    with pytest.raises(B.CsvError):
        pool.free_blocks([a[0]])                       # double free
    with pytest.raises(B.CsvError):
        pool.set_free_order([0, 1, 2])                 # not a permutation of the 8 free ids
    with pytest.raises(B.CsvError):
        pool.set_free_order([0, 1, 2, 3, 4, 5, 6, 6])
    with pytest.raises(B.CsvError) as e:
        pool.alloc_blocks(9)                           # all-or-nothing
    assert e.value.code == B.CSV_E_NOMEM and pool.used_blocks == 0


def test_placement_follows_the_papers_rule(oracle):
    # PAPER.md:178 lowest current occupancy; PAPER.md:176 decrement on termination; PAPER.md:31 skip a full decoder
    pools = [mkpool(100), mkpool(100), mkpool(50)]
    assert B.csv_place(pools, 10) == 0                 # all empty: tie -> lowest index
    c0 = pools[0].alloc_blocks(10)
    assert B.csv_place(pools, 10) == 1
    pools[1].alloc_blocks(10)
    assert B.csv_place(pools, 10) == 2                 # 0/50 < 10/100
    pools[2].alloc_blocks(10)                          # 20 % vs 10 % vs 10 %
    assert B.csv_place(pools, 10) == 0
    assert B.csv_place(pools, 45) == 0                 # pool 2 has only 40 free: skipped
    pools[0].alloc_blocks(85)
    pools[1].alloc_blocks(85)
    with pytest.raises(B.CsvError) as e:
        B.csv_place(pools, 41)
    assert e.value.code == B.CSV_E_NOMEM
    pools[0].free_blocks(c0)                           # a conversation terminates: occupancy drops
    assert B.csv_place(pools, 5) == 2                  # 20 % (pool 2) < 85 % (pool 0) < 95 %
    # random scripted arrivals against the oracle's restatement of the rule
    rng = np.random.default_rng(3)
    ps = [mkpool(64), mkpool(96), mkpool(80)]
    live = []
    for _ in range(300):
        if rng.random() < 0.6 or not live:
            need = int(rng.integers(1, 20))
            used = [p.used_blocks for p in ps]
            total = [p.num_blocks for p in ps]
            want = oracle.place(used, total, need)
            if want < 0:
                with pytest.raises(B.CsvError):
                    B.csv_place(ps, need)
            else:
                got = B.csv_place(ps, need)
                assert got == want
                live.append((got, ps[got].alloc_blocks(need)))   # binding is permanent: freed only at termination
        else:
            k, ids = live.pop(int(rng.integers(0, len(live))))
            ps[k].free_blocks(ids)


def test_provisioning_matches_the_papers_worked_example():
    line = [l for l in open(os.path.join(ROOT, "tests", "golden", "provisioning_example.txt")) if not l.startswith("#")][0]
    T_p, L_in, T_d, L_d, n_expected, deployed = [float(x) for x in line.split()]
    rate, n_thr, n_mem, n = B.csv_provision(T_p, L_in, T_d, L_d, 20.0, 1.0)
    assert round(n_thr, 2) == n_expected                # PAPER.md:209 "at least 1.67 decoders per prefiller"
    assert rate == pytest.approx(25000 / 15000)
    assert n == 2 and n <= deployed
    assert n_mem == pytest.approx(rate * 1.0 / 20.0)    # Eq. 2
    assert B.csv_provision(T_p, L_in, T_d, L_d, 1.0, 3.0)[3] == 5   # memory-bound case: ceil(1.667 * 3)
    with pytest.raises(B.CsvError):
        B.csv_provision(0, 1, 1, 1, 1, 1)


# ------------------------------------------------------------------ split-K planner

def check_decode_plan(q_lens, kv_lens, Hq, Hkv, d, mpt=0):
    plan = B.Plan(B.attn_shape(Hq, Hkv, d), q_lens, kv_lens, mpt)
    info = plan.info()
    items, wb = plan.decode_items()
    W = info["decode_workers"]
    assert W == info["decode_grid"] * (7 if d == 128 else 8)
    assert wb[0] == 0 and wb[W] == len(items) and np.all(np.diff(wb) >= 0)
    cap = (mpt if mpt else 1 << 30) // 16
    # every (conv, head, block) of every q_len = 1 row is covered exactly once, in order
    cover = {}
    for conv, head, b0, b1, kv_len, partial, direct, _ in items:
        assert q_lens[conv] == 1 and kv_len == kv_lens[conv]
        assert 0 <= b0 < b1 <= (kv_len + 15) // 16 and b1 - b0 <= cap
        cover.setdefault((conv, head), []).append((b0, b1, partial, direct))
    rows = [b for b in range(len(q_lens)) if q_lens[b] == 1]
    assert info["n_decode_rows"] == len(rows)
    assert set(cover) == {(b, g) for b in rows for g in range(Hkv) if kv_lens[b] > 0}   # an empty cache has no blocks
    seen_partials = set()
    for (conv, head), parts in cover.items():
        assert parts[0][0] == 0 and parts[-1][1] == (kv_lens[conv] + 15) // 16
        for (a0, a1, _, _), (c0, c1, _, _) in zip(parts, parts[1:]):
            assert a1 == c0
        if len(parts) == 1:
            assert parts[0][3] == 1 and parts[0][2] == -1
        else:
            ids = [p[2] for p in parts]
            assert ids == list(range(ids[0], ids[0] + len(ids))) and all(p[3] == 0 for p in parts)
            assert not (set(ids) & seen_partials)
            seen_partials |= set(ids)
    # shares are balanced: no worker streams more than ceil(units / W) + 0 blocks ... (+1 for rounding)
    units = sum(((kv_lens[b] + 15) // 16) * Hkv for b in rows)
    per_worker = [int(sum(items[i][3] - items[i][2] for i in range(wb[w], wb[w + 1]))) for w in range(W)]
    assert sum(per_worker) == units
    if units:
        assert max(per_worker) <= units // W + 1
    return plan, info


def test_decode_plan_covers_config_shapes():
    for k, (Hq, Hkv, d) in {1: (4, 1, 64), 2: (32, 8, 128)}.items():
        kv = synth.config_lengths(k)["kv_lens"]
        _, info = check_decode_plan([1] * len(kv), list(kv), Hq, Hkv, d)
    L3 = synth.config_lengths(3)
    _, info = check_decode_plan(list(L3["q_lens"]), list(L3["kv_lens"]), 32, 8, 128)
    assert info["n_decode_rows"] == 224 and info["n_append_chunks"] == 32 and info["decode_grid"] == 148
    # config 5: every sequence is cut into >= 64 partitions (BASELINE.json config 5)
    plan, info = check_decode_plan([1] * 16, [131072] * 16, 64, 8, 128)
    items, _ = plan.decode_items()
    per_seq = np.bincount(items[:, 0], minlength=16)
    assert per_seq.min() >= 64            # >= 64 partitions per sequence (8 KV heads x >= 9 shares each)
    plan64, _ = check_decode_plan([1] * 16, [131072] * 16, 64, 8, 128, mpt=2048)
    assert np.bincount(plan64.decode_items()[0][:, 0], minlength=16).min() >= 64 * 8   # forced: >= 64 per (sequence, head)


def test_decode_plan_edge_lengths_and_partition_sizes():
    for mpt in (0, 16, 64, 4096):
        check_decode_plan([1, 1, 1, 1, 1, 1, 0, 1], [1, 15, 16, 17, 2047, 2049, 0, 65536], 32, 8, 128, mpt)
    check_decode_plan([1], [1], 4, 1, 64)
    _, info = check_decode_plan([0, 0], [5, 0], 4, 1, 64)
    assert info["n_decode_items"] == 0
    with pytest.raises(B.CsvError):
        B.Plan(B.attn_shape(32, 8, 128), [2], [1])            # q_len > kv_len
    with pytest.raises(B.CsvError):
        B.Plan(B.attn_shape(32, 8, 128), [2], [0])            # ... also on an empty cache, unless it is a decode row:
    _, info = check_decode_plan([1, 1, 1], [0, 40, 0], 32, 8, 128)   # q_len 1, kv_len 0 -> O = 0, LSE = -inf (header a4)
    assert info["n_decode_rows"] == 3 and info["n_decode_items"] >= 8
    _, info = check_decode_plan([1], [0], 4, 1, 64)
    assert info["n_decode_rows"] == 1 and info["n_decode_items"] == 0
    with pytest.raises(B.CsvError):
        B.Plan(B.attn_shape(32, 8, 128), [1], [10], 24)       # partition not a multiple of 16
    with pytest.raises(B.CsvError):
        B.Plan(B.attn_shape(30, 8, 128), [1], [10])           # Hq not a multiple of Hkv
    with pytest.raises(B.CsvError):
        B.Plan(B.attn_shape(32, 8, 96), [1], [10])


def test_decode_plan_depends_only_on_lengths():
    kv = list(synth.config_lengths(2)["kv_lens"])
    a, _ = B.Plan(B.attn_shape(32, 8, 128), [1] * 64, kv).decode_items()
    b, _ = B.Plan(B.attn_shape(32, 8, 128), [1] * 64, kv).decode_items()
    assert np.array_equal(a, b)


def test_append_plan_covers_all_rows_and_visible_blocks():
    L3 = synth.config_lengths(3)
    q_lens, kv_lens = list(L3["q_lens"]), list(L3["kv_lens"])
    for (Hq, Hkv, mpt) in ((32, 8, 0), (64, 8, 4096), (32, 8, 64 * 16)):
        G = Hq // Hkv
        plan = B.Plan(B.attn_shape(Hq, Hkv, 128), q_lens, kv_lens, mpt)
        items = plan.append_items()
        q_start = np.concatenate([[0], np.cumsum(q_lens)])
        assert plan.total_q == q_start[-1]
        cover = {}
        for conv, head, r0, qs, m, kv_len, b0, b1, partial, direct, _, _ in items:
            assert m == q_lens[conv] > 1 and kv_len == kv_lens[conv] and qs == q_start[conv] and r0 % 256 == 0
            cover.setdefault((conv, head, r0), []).append((b0, b1, direct))
        chunks = [b for b in range(len(q_lens)) if q_lens[b] > 1]
        want = {(b, g, r0) for b in chunks for g in range(Hkv) for r0 in range(0, q_lens[b] * G, 256)}
        assert set(cover) == want
        for (conv, head, r0), parts in cover.items():
            parts.sort()
            m, P = q_lens[conv], kv_lens[conv] - q_lens[conv]
            i_max = min(m - 1, (min(m * G, r0 + 256) - 1) // G)   # d = 128: 256-row items (two 128-row UMMA tiles)
            assert parts[0][0] == 0 and parts[-1][1] == (P + i_max + 1 + 15) // 16   # exactly the visible blocks
            for (a0, a1, _), (c0, c1, _) in zip(parts, parts[1:]):
                assert a1 == c0
            assert all(p[2] == (1 if len(parts) == 1 else 0) for p in parts)
        # longest first
        sizes = items[:, 7] - items[:, 6]
        assert np.all(np.diff(sizes) <= 0)


def test_workspace_bytes_grows_with_partials_and_is_checked():
    sh = B.attn_shape(32, 8, 128)
    small = B.csv_plan_workspace_bytes(sh, [1], [16])
    big = B.csv_plan_workspace_bytes(sh, [1] * 64, list(synth.config_lengths(2)["kv_lens"]))
    assert 0 < small < big
    assert B.csv_plan_workspace_bytes(sh, [2], [1]) == 0
    kv = [4096] * 4
    assert B.csv_tail_step_host_workspace_bytes(sh, kv, 256) > B.csv_plan_workspace_bytes(sh, [1] * 4, kv)


def test_mixed_step_split_follows_the_work():
    # csv_plan_tail_split: only a plan with decode rows AND chunks at d = 128 has a fused launch; the decode side grows with
    # the decode bytes, shrinks with the chunks' flops, and always leaves CTAs for the other role (host-only plans, 148 SMs).
    sh = B.attn_shape(32, 8, 128)
    split = lambda q, kv, shape=sh: (lambda i: (i["tail_n_dec"], i["tail_n_shares"]))(B.Plan(shape, q, kv).info())
    assert split([1] * 8, [4096] * 8) == (0, 0)                          # decode rows only: paged_decode_step
    assert split([64] * 4, [4096] * 4) == (0, 0)                         # chunks only
    assert split([1, 64], [512, 512], B.attn_shape(4, 1, 64)) == (0, 0)  # d = 64: the three-launch route
    c3 = synth.config_lengths(3)
    k3, s3 = split(c3["q_lens"], c3["kv_lens"])
    assert 30 <= k3 <= 80 and s3 >= k3                                   # configs[2]: decode 14 GB against 2.8 TFLOP
    more_decode = np.where(c3["q_lens"] == 1, c3["kv_lens"] * 2, c3["kv_lens"])
    assert split(c3["q_lens"], more_decode)[0] > k3
    assert split([1, 512], [16, 60000]) == (0, 0)                        # hardly any decode work beside a long chunk: two kernels
    c5q, c5kv = [1] * 16 + [256] * 4, [131072] * 20                      # configs[4] as one batch: decode is 16 % of the step
    assert split(c5q, c5kv, B.attn_shape(64, 8, 128)) == (0, 0)
    assert split([1] * 200 + [2], [60000] * 200 + [64])[0] <= 111        # never more than 3/4 of the SMs on decode


def test_tuning_knobs_are_read_at_plan_build_and_recorded_in_the_plan():
    # the overrides were getenv calls inside the planner (every build) and a cached static in csv_tail_step.  They
    # are now one process-wide table that a test can flip; a plan keeps what it was built with.
    sh = B.attn_shape(64, 8, 128)
    c5q, c5kv = [1] * 16 + [256] * 4, [131072] * 20
    try:
        assert [B.csv_tuning_get(k) for k in range(5)] == [0] * 5 and B.csv_tuning_get(5) == -1
        base = B.Plan(sh, c5q, c5kv)
        assert base.info()["tail_n_dec"] == 0 and base.info()["decode_grid"] == 148
        ws_default = B.csv_plan_workspace_bytes(sh, c5q, c5kv)
        B.csv_tuning_set(B.TUNE_TAIL_DECODE_CTAS, 26)                   # force the one-launch route where the planner declines it
        forced = B.Plan(sh, c5q, c5kv)
        assert forced.info()["tail_n_dec"] == 26 and forced.info()["tail_n_shares"] == 26
        assert B.csv_plan_workspace_bytes(sh, c5q, c5kv) >= ws_default  # the size query sees the same table as the build
        assert base.info()["tail_n_dec"] == 0                           # existing plans keep what they were built with
        B.csv_tuning_set(B.TUNE_TAIL_DECODE_CTAS, 10 ** 5)
        assert B.Plan(sh, c5q, c5kv).info()["tail_n_dec"] == 147        # always one CTA left for the other role
        B.csv_tuning_set(B.TUNE_TAIL_DECODE_CTAS, 0)
        assert B.Plan(sh, c5q, c5kv).info()["tail_n_dec"] == 0
        B.csv_tuning_set(B.TUNE_DECODE_GRID, 37)
        assert B.Plan(sh, c5q, c5kv).info()["decode_grid"] == 37
        assert B.Plan(sh, [1], [16]).info()["decode_grid"] == 1         # a cap, not a floor
        # the per-SM rates of the two roles are the caller's to calibrate: a device whose SMs stream faster needs fewer
        # decode-role CTAs for the same step, one whose tensor pipes are faster needs more
        c3 = synth.config_lengths(3)
        sh8 = B.attn_shape(32, 8, 128)
        k_default = B.Plan(sh8, c3["q_lens"], c3["kv_lens"]).info()["tail_n_dec"]
        B.csv_tuning_set(B.TUNE_SM_DECODE_GBS, 100)
        k_fast_hbm = B.Plan(sh8, c3["q_lens"], c3["kv_lens"]).info()["tail_n_dec"]
        B.csv_tuning_set(B.TUNE_SM_DECODE_GBS, 0)
        B.csv_tuning_set(B.TUNE_SM_APPEND_GFLOPS, 14800)
        k_fast_mma = B.Plan(sh8, c3["q_lens"], c3["kv_lens"]).info()["tail_n_dec"]
        B.csv_tuning_set(B.TUNE_SM_APPEND_GFLOPS, 0)
        assert 0 < k_fast_hbm < k_default < k_fast_mma
        for bad in ((-1, 1), (5, 1), (0, -5), (1, (1 << 20) + 1)):
            with pytest.raises(B.CsvError):
                B.csv_tuning_set(*bad)
    finally:
        for k in range(5):
            B.csv_tuning_set(k, 0)
    assert B.Plan(sh, c5q, c5kv).info()["decode_grid"] == 148


def test_handoff_direct_and_ipc_reject_bad_arguments_before_touching_cuda():
    pool = mkpool(8, NL=1, Hkv=1, d=64)
    k = FAKE + (1 << 20)
    ids = FAKE + (2 << 20)
    for call in (lambda: B.kv_handoff_direct(pool, k, k, 0, 0, ids, 8, stream=0),          # zero tokens
                 lambda: B.kv_handoff_direct(pool, k, k, 10, -1, ids, 8, stream=0),
                 lambda: B.kv_handoff_direct(pool, k + 2, k, 10, 0, ids, 8, stream=0),      # misaligned source
                 lambda: B.kv_handoff_direct(pool, k, None, 10, 0, ids, 8, stream=0),
                 lambda: B.kv_handoff_direct(pool, k, k, 10, 0, None, 8, stream=0),
                 lambda: B.kv_handoff_direct(pool, k, k, 300, 0, ids, 8, stream=0),         # table shorter than ceil(300 / 16)
                 lambda: B.kv_handoff_direct_batch(pool, [k], [k], [17], [112], [ids], [8], stream=0)):
        with pytest.raises(B.CsvError) as e:
            call()
        assert e.value.code == B.CSV_E_INVAL
    B.kv_handoff_direct_batch(pool, [k, k], [k, k], [0, 0], [0, 0], [ids, ids], [8, 8], stream=0)   # nothing to do: no launch
    L = B.lib()
    off = ctypes.c_uint64()
    out = ctypes.c_void_p()
    buf = ctypes.create_string_buffer(B.IPC_HANDLE_BYTES)
    assert L.csv_ipc_export(None, buf, ctypes.byref(off)) == B.CSV_E_INVAL
    assert L.csv_ipc_export(ctypes.c_void_p(k), None, ctypes.byref(off)) == B.CSV_E_INVAL
    assert L.csv_ipc_open(None, 0, ctypes.byref(out)) == B.CSV_E_INVAL
    assert L.csv_ipc_open(buf, 0, None) == B.CSV_E_INVAL
    assert L.csv_ipc_close(ctypes.c_void_p(k)) == B.CSV_E_INVAL                   # never opened
    nbytes = ctypes.c_size_t(77)
    assert L.csv_ipc_mapped_bytes(ctypes.c_void_p(k), ctypes.byref(nbytes)) == B.CSV_E_INVAL   # not a csv_ipc_open pointer
    assert L.csv_ipc_mapped_bytes(None, ctypes.byref(nbytes)) == B.CSV_E_INVAL
    assert L.csv_ipc_mapped_bytes(ctypes.c_void_p(k), None) == B.CSV_E_INVAL and nbytes.value == 77
    assert pool.used_blocks == 0


def test_tail_step_host_refuses_bad_lengths_before_any_copy_is_enqueued():
    # q_len > kv_len used to be found by the planner AFTER the four host->device copies were enqueued.  On this
    # box there is no GPU, so a call that reached cudaMemcpyAsync would come back CSV_E_CUDA: CSV_E_INVAL proves the order.
    pool = mkpool(64, NL=2)
    sh = B.attn_shape(32, 8, 128)

    class FakeBuf:   # what binding._ptr / workspace sizing need from a tensor
        def __init__(self, ptr, n):
            self.ptr, self.n = ptr, n

        def data_ptr(self):
            return self.ptr

        def numel(self):
            return self.n

        def element_size(self):
            return 1

    ws = FakeBuf(FAKE, 1 << 30)
    h = FakeBuf(FAKE + (1 << 31), 1 << 20)
    call = lambda kv, q=None, mpt=0, shape=sh: B.csv_tail_step_host(pool, 0, shape, kv, h, h, h, h, 8, ws, h, h, mpt, stream=0,
                                                                     q_lens=q, n_layers=2)
    for bad in (lambda: call([100, 50], [1, 51]),            # q_len > kv_len
                lambda: call([100, -1]),                      # negative length
                lambda: call([100, 0], [1, 2]),               # only a DECODE row may sit on an empty cache
                lambda: call([100, 50], mpt=24),              # partition size not a multiple of 16
                lambda: call([100, 50], shape=B.attn_shape(24, 8, 128))):   # G = 3
        with pytest.raises(B.CsvError) as e:
            bad()
        assert e.value.code == B.CSV_E_INVAL


def test_committed_ncu_traffic_rows_belong_to_the_current_kernel_sources():
    # bench.py reports roofline.traffic only from a capture taken on the kernel sources as they are now (sha256 recorded at
    # ingest time in profiles/r2_traffic.csv / r3_traffic.csv).  A kernel edit without a fresh capture must show up here, not as a silent null.
    import importlib.util
    import os

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    want = [("decode_kernel", "configs[1]"), ("decode_kernel", "configs[2]"), ("decode_kernel", "configs[4]"),
            ("append_tc2_kernel", "configs[2]"), ("append_tc2_kernel", "configs[4]"), ("tail_kernel", "configs[2]"),
            ("pack_kernel", "configs[3]"), ("unpack_kernel", "configs[3]"), ("direct_kernel", "configs[3]")]
    for kernel, config in want:
        traffic, why = bench.traffic_for(kernel, config)
        assert traffic is not None and traffic > 0, "%s on %s: %s" % (kernel, config, why)

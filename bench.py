#!/usr/bin/env python
"""bench.py — the conversation-tail hot path on B200, through the C ABI.

Default workload = BASELINE.json configs[1] (Llama-3-8B-shaped layer, 64 conversations,
context U[1024,8192], block size 16, shuffled paged pool).  One STEP = one pass of the tail
path over that batch: paged_decode_step = the new token's K/V written into the pool + split-K paged
decode attention + merge (--unfused: kv_append_tokens and paged_decode_attn as two calls), replayed
from a CUDA graph (--no-graph: plain launches).  metric = KV bytes read / step time, in GB/s, whole job.
The other configs (handoff, agentic tail mix, long context) are timed after the headline line's
measurements and reported under "other_workloads" (--no-extras skips them).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras] [--no-graph] [--unfused]

N > 1 (torchrun): replicas only — every rank serves its own pool of conversations,
no data-path collective; barrier + max-over-ranks timing; value = total bytes / that time.
--impl reference: the fp64 CPU oracle (oracle/), as it stands, on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "paged_decode_attn_hbm_gbs"
UNIT = "GB/s"
NOMINAL_HBM_GBS = 8000.0        # north_star's "~8 TB/s"; targets (70 % / 80 %) are stated against it


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy read+write)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic_bytes():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of decode_kernel on this workload, from the committed
    `ncu --set full` capture (profiles/r1_decode_ncu_full.csv); None if the file is not there."""
    p = os.path.join(ROOT, "profiles", "r1_decode_ncu_full.csv")
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    try:
        tot = 0.0
        for line in open(p):
            f = line.strip().split(",")
            if f[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                vals = [float(x.strip('"')) for x in f[2:] if x]
                tot += unit[f[1]] * sum(vals) / len(vals)
        return tot or None
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (profiling recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.lines, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._pump, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        rows = [l for (t, l) in self.lines if t0 - 0.05 <= t <= t1 + 0.15] or [l for (_, l) in self.lines]
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except Exception:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_logical_kv(oracle, wl, b, layer=0):
    """cpu_baseline leg only: conversation b's raw pool blocks copied back, gathered (paged -> logical) by the ORACLE."""
    img = wl.conversation_blocks_host(b, layer)
    n = len(wl.tables[b])
    return oracle.gather(img, n, wl.Hkv, wl.d, 0, np.arange(n, dtype=np.int32), wl.kv_lens[b])


def oracle_sample(wl, n_conv, layer=0):
    """Time the oracle (fp64, one thread) on the first n_conv conversations of the workload.
    Returns (seconds, KV bytes it read)."""
    import oracle

    oracle.build()
    q_all = wl.d_q.cpu().contiguous().view(-1, wl.Hq, wl.d).numpy().view(np.uint16)
    rows = [b for b in range(len(wl.q_lens)) if wl.q_lens[b] == 1][:n_conv]
    starts = np.concatenate([[0], np.cumsum(wl.q_lens)])
    data = [(q_all[starts[b]:starts[b] + 1], *oracle_logical_kv(oracle, wl, b, layer)) for b in rows]
    t0 = time.perf_counter()
    outs = [oracle.attention(q, K, V) for (q, K, V) in data]
    dt = time.perf_counter() - t0
    nbytes = sum(wl.kv_lens[b] for b in rows) * wl.Hkv * wl.d * 2 * 2
    return dt, nbytes, rows, outs


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_2606_01839_b200 import synth

    oracle.build()
    cfg = synth.CONFIGS[2]
    kv = synth.config_lengths(2)["kv_lens"]
    n_conv = 2
    rng = np.random.default_rng(cfg["seed"])
    data = [(synth.normal_bf16(rng, (1, cfg["Hq"], cfg["d"])), synth.normal_bf16(rng, (int(t), cfg["Hkv"], cfg["d"])),
             synth.normal_bf16(rng, (int(t), cfg["Hkv"], cfg["d"]))) for t in kv[:n_conv]]
    nbytes = int(sum(kv[:n_conv])) * cfg["Hkv"] * cfg["d"] * 2 * 2
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        for q, K, V in data:
            oracle.attention(q, K, V)
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    sec = float(np.mean(times))
    gbs = nbytes / sec / 1e9
    sample = "first %d of 64 conversations of configs[1] (%.1f MB of KV), all 32 heads, per step" % (n_conv, nbytes / 1e6)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[1] c2_llama8b_decode64 (bounded sample)", "sample": sample},
        "cpu_baseline": {"value": gbs, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": gbs, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def time_calls(fn, iters, warmup=3):
    """CUDA-event time of fn() on the current stream: (median ms, min ms)."""
    import torch

    for _ in range(warmup):
        fn()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
    torch.cuda.synchronize()
    for a, b in evs:
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    ts = sorted(a.elapsed_time(b) for a, b in evs)
    return ts[len(ts) // 2], ts[0]


def handoff_extra(iters=5):
    """BASELINE.json configs[3]: 16 conversations x 32 layers of 8B-shape KV, random bits, pack -> unpack (batched)."""
    import torch
    from paper_2606_01839_b200 import binding as B
    from paper_2606_01839_b200 import synth

    cfg = synth.CONFIGS[4]
    toks = [int(t) for t in synth.config_lengths(4)["tokens"]]
    NL, Hkv, d = cfg["NL"], cfg["Hkv"], cfg["d"]
    rng = np.random.default_rng(cfg["seed"])
    gen = torch.Generator(device="cuda")
    gen.manual_seed(4004)
    nb = synth.pool_blocks_for(toks, slack=0.10)
    desc = B.pool_desc(NL, nb, Hkv, d)
    d_pool = torch.empty(B.kv_pool_bytes(desc) // 2, dtype=torch.int16, device="cuda")
    pool = B.KvPool(desc, d_pool)
    pool.set_free_order(synth.shuffled_free_order(rng, nb))
    ks, vs, sts, ids = [], [], [], []
    for t in toks:
        n = NL * t * Hkv * d
        ks.append(torch.randint(-32768, 32767, (n,), dtype=torch.int16, device="cuda", generator=gen))
        vs.append(torch.randint(-32768, 32767, (n,), dtype=torch.int16, device="cuda", generator=gen))
        sts.append(torch.empty(B.kv_staging_bytes(desc, t) // 2, dtype=torch.int16, device="cuda"))
        ids.append(torch.from_numpy(pool.alloc_blocks(synth.blocks_for(t))).cuda())
    offs, nids = [0] * len(toks), [len(i) for i in ids]
    payload = sum(toks) * NL * Hkv * d * 2 * 2                  # K + V bytes of all conversations
    pack_ms, _ = time_calls(lambda: B.kv_pack_batch(desc, ks, vs, toks, offs, sts), iters, 2)
    unpack_ms, _ = time_calls(lambda: B.kv_unpack_batch(pool, sts, toks, offs, ids, nids), iters, 2)
    direct_ms, _ = time_calls(lambda: B.kv_handoff_direct_batch(pool, ks, vs, toks, offs, ids, nids), iters, 2)
    moved_unpack = sum(B.kv_staging_bytes(desc, t) for t in toks)   # whole tiles (last block padded)
    out = {"workload": "configs[3] c4_handoff_32layer", "tokens_total": sum(toks), "payload_gb": payload / 1e9,
           "pack_ms": pack_ms, "unpack_ms": unpack_ms,
           "pack_gbs_rw": 2 * payload / pack_ms / 1e6, "unpack_gbs_rw": 2 * payload / unpack_ms / 1e6,
           "unpack_bytes_touched_gb": 2 * moved_unpack / 1e9,
           # kv_handoff_direct: source -> paged pool in one kernel, no staging message (same GPU here; the
           # destination may be a peer mapping).  Same payload, half the memory traffic of pack + unpack.
           "direct_ms": direct_ms, "direct_gbs_rw": 2 * payload / direct_ms / 1e6,
           "handoff_payload_gbs": {"pack_then_unpack": payload / (pack_ms + unpack_ms) / 1e6,
                                   "direct": payload / direct_ms / 1e6}}
    del ks, vs, sts, d_pool
    torch.cuda.empty_cache()
    return out


def prefill_extra(iters=5):
    """turn-1 prefill attention of a 32768-token prompt in 8192-token chunks through
    append_prefill_attn (m = 8192, P = earlier chunks), 8B shape, one layer."""
    import torch
    from paper_2606_01839_b200 import workloads

    wl = workloads.TailWorkload(32, 8, 128, [1], [32768], seed=22)
    total_ms, flops = 0.0, 0.0
    for P in (0, 8192, 16384, 24576):
        app = wl.with_q_lens([8192], [P + 8192])
        ms, _ = time_calls(app.append, iters)
        total_ms += ms
        flops += app.append_flops()
    del wl, app
    torch.cuda.empty_cache()
    return {"workload": "turn-1 prefill attention, 32768 tokens in 4 chunks of 8192 (Hq=32 Hkv=8 d=128, one layer)",
            "ms": total_ms, "tflops": flops / total_ms / 1e9}


def tail_extra(k, iters=10):
    """configs[2] (agentic tail mix) and configs[4] (70B-shaped long context, ONE of its 8 layers): per-call times."""
    import torch
    from paper_2606_01839_b200 import workloads

    full5 = k == 5 and torch.cuda.mem_get_info()[0] > 85e9      # all 8 layers of config 5 (~69 GB of KV) when they fit
    wl = workloads.config_tail_workload(k, layers=8) if full5 else workloads.config_tail_workload(k)
    out = {"workload": "configs[%d] %s" % (k - 1, __import__("paper_2606_01839_b200.synth", fromlist=["x"]).CONFIGS[k]["name"])}
    app = wl if k == 3 else wl.with_q_lens(workloads.config5_append_q_lens())
    if k == 5:
        out["layers_timed"] = 1
    dec_ms, dec_min = time_calls(wl.decode, iters)
    out.update(decode_ms=dec_ms, decode_gbs=wl.decode_kv_bytes() / dec_ms / 1e6, decode_rows=sum(1 for q in wl.q_lens if q == 1),
               decode_kv_gb=wl.decode_kv_bytes() / 1e9)
    app_ms, _ = time_calls(app.append, max(3, iters // 2))
    out.update(append_ms=app_ms, append_tflops=app.append_flops() / app_ms / 1e9, append_kv_gb=app.append_kv_bytes() / 1e9,
               append_rows=sum(q for q in app.q_lens if q > 1))
    # both overlapped on two streams (decode is HBM-bound, append tensor-bound)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

    def both():
        e = torch.cuda.Event()
        e.record()
        s1.wait_event(e)
        s2.wait_event(e)
        wl.decode(stream=s1)
        app.append(stream=s2)
        torch.cuda.current_stream().wait_stream(s1)
        torch.cuda.current_stream().wait_stream(s2)

    both_ms, _ = time_calls(both, max(3, iters // 2))
    out.update(decode_plus_append_overlapped_ms=both_ms)
    if full5:
        # configs[4]'s whole step: decode for all 16 conversations + the 4 appended chunks, on each of the 8 layers
        def step8():
            for layer in range(8):
                wl.decode(layer=layer)
                app.append(layer=layer)
        g8 = torch.cuda.CUDAGraph()
        step8()
        torch.cuda.synchronize()
        with torch.cuda.graph(g8):
            step8()
        s8_ms, _ = time_calls(g8.replay, 3, 1)

        def dec8():
            for layer in range(8):
                wl.decode(layer=layer)
        d8_ms, _ = time_calls(dec8, 3, 1)
        out.update(layers_in_pool=8, pool_gb=wl.pool_bytes / 1e9, step_8_layers_ms=s8_ms, decode_8_layers_ms=d8_ms,
                   decode_8_layers_gbs=8 * wl.decode_kv_bytes() / d8_ms / 1e6)
    if k == 3:
        # the whole mixed step in one call (csv_tail_step: KV write of all 9347 new rows + decode + append), replayed
        # from a CUDA graph as a serving loop would
        g = torch.cuda.CUDAGraph()
        wl.tail_step()
        torch.cuda.synchronize()
        with torch.cuda.graph(g):
            wl.tail_step()
        step_ms, _ = time_calls(g.replay, max(3, iters // 2))
        out.update(tail_step_one_call_ms=step_ms)
    del wl, app
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    from paper_2606_01839_b200 import build as libbuild

    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        libbuild.build_library()             # no-op when the in-tree .so is up to date; there is no fallback path
    from paper_2606_01839_b200 import binding as B
    from paper_2606_01839_b200 import replicas, workloads

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    local = local % max(1, torch.cuda.device_count())
    torch.cuda.set_device(local)
    dist, agg_dev = None, "cuda"
    if world > 1:
        import torch.distributed as dist_mod

        dist = dist_mod
        try:   # the only cross-rank traffic is a barrier and scalar reductions (replicas, no data-path collective)
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
            dist.barrier()
        except Exception as e:
            sys.stderr.write("nccl unavailable (%r): using gloo for the barrier / scalar reductions\n" % (e,))
            if dist.is_initialized():
                dist.destroy_process_group()
            dist.init_process_group("gloo")
            agg_dev = "cpu"
    B.lib()   # fails loudly if libconserve_kv.so is missing: there is no fallback

    # replicas only: rank r serves its own conversations (same length recipe, different seed)
    wl = workloads.config_tail_workload(2, seed=replicas.rank_seed(1, rank))
    kv_bytes = wl.decode_kv_bytes()
    rows = len(wl.kv_lens)
    K, W = args.steps, max(3, args.warmup)

    def step():
        if args.unfused:
            wl.kv_append_tokens()
            wl.decode()
        else:
            wl.decode_step()   # paged_decode_step: the new token's K/V write fused into the decode launch

    for _ in range(W):
        step()
    torch.cuda.synchronize()
    # The step is launch-sized (~200 us, 3 kernels): capture it once in a CUDA graph and replay it (the library only
    # enqueues launches on the caller's stream, so it is capturable as is).  --no-graph times plain launches.
    graph = None
    if not args.no_graph:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            step()
        torch.cuda.current_stream().wait_stream(side)
        try:
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                step()
            for _ in range(W):
                graph.replay()
            torch.cuda.synchronize()
        except Exception as e:   # never lose the bench line to a capture problem
            sys.stderr.write("CUDA graph capture failed (%r): timing plain launches\n" % (e,))
            graph = None
            torch.cuda.synchronize()
    run_step = graph.replay if graph is not None else step
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local) if rank == 0 else None
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.time()
    ev0.record()
    for _ in range(K):
        run_step()
    ev1.record()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    ms_total = ev0.elapsed_time(ev1)
    # roofline leg, same process, right after: K paged_decode_attn calls (decode_kernel + decode_merge_kernel) alone
    ev2.record()
    for _ in range(K):
        wl.decode()
    ev3.record()
    torch.cuda.synchronize()
    t1 = time.time()
    dec_ms = ev2.elapsed_time(ev3) / K
    if t1 - t0 < 0.5:   # give nvidia-smi (100 ms period) something to sample: keep the GPU on the same work
        tend = time.time() + 0.6
        while time.time() < tend:
            run_step()
        torch.cuda.synchronize()
        t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    ms_total, _ = replicas.aggregate(dist, ms_total, kv_bytes, device=agg_dev)
    dec_ms, total_kv_bytes = replicas.aggregate(dist, dec_ms, kv_bytes, device=agg_dev)
    ms_step = ms_total / K
    value = total_kv_bytes / ms_step / 1e6              # GB/s, whole job (sum of bytes / max time)
    info = wl.plan.info()
    launches_per_step = 3 if args.unfused else 2   # [append_tokens_kernel +] decode_kernel + decode_merge_kernel

    # end to end through the C-ABI call with HOST buffers (plan + H2D + kernels + D2H inside the timed region)
    pin = lambda t: t.cpu().pin_memory()
    h_q, h_k, h_v = pin(wl.d_q), pin(wl.d_k_new), pin(wl.d_v_new)
    h_t = torch.from_numpy(wl.h_tables).pin_memory()
    h_out = torch.zeros((rows, wl.Hq, wl.d), dtype=torch.int16).pin_memory()
    h_lse = torch.zeros((rows, wl.Hq), dtype=torch.float32).pin_memory()
    ws = torch.empty(B.csv_tail_step_host_workspace_bytes(wl.shape, wl.kv_lens, wl.max_blocks), dtype=torch.uint8,
                     device="cuda")
    e2e_call = lambda: B.csv_tail_step_host(wl.pool, 0, wl.shape, wl.kv_lens, h_q, h_k, h_v, h_t, wl.max_blocks, ws, h_out,
                                            h_lse)
    for _ in range(W):
        e2e_call()
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    tw = time.perf_counter()
    for _ in range(K):
        e2e_call()          # synchronises its stream before returning (the result is on the host)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - tw) * 1e3 / K
    e2e_ms, _ = replicas.aggregate(dist, e2e_ms, kv_bytes, device=agg_dev)
    h2d = h_q.numel() * 2 + h_k.numel() * 2 + h_v.numel() * 2 + h_t.numel() * 4
    d2h = h_out.numel() * 2 + h_lse.numel() * 4

    if rank != 0:
        if dist:
            dist.barrier()
            dist.destroy_process_group()
        return
    peak, peak_src = measured_peaks()
    achieved = kv_bytes / dec_ms / 1e6
    # host planning (reported apart from kernel time; one plan serves all layers of a step)
    pt = []
    for _ in range(21):
        t0 = time.perf_counter()
        B.Plan(wl.shape, wl.q_lens, wl.kv_lens).destroy()
        pt.append((time.perf_counter() - t0) * 1e6)
    plan_us = sorted(pt)[len(pt) // 2]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "configs[1] c2_llama8b_decode64: Hq=32 Hkv=8 d=128 bs=16, 64 conversations, context U[1024,8192], "
                               "shuffled paged pool; step = " + ("kv_append_tokens + paged_decode_attn" if args.unfused else "paged_decode_step (new-token KV write fused into the decode launch)"),
                   "kv_bytes_per_step_per_gpu": kv_bytes, "kv_tokens": int(sum(wl.kv_lens)), "decode_rows": rows,
                   "l2": "inputs larger than L2 (%.2f GB of KV per step vs 126 MB)" % (kv_bytes / 1e9),
                   "parallelism": "replicas x%d, no collective" % world, "decode_grid": info["decode_grid"],
                   "decode_items": info["n_decode_items"], "cuda_graph": graph is not None,
                   "plan_host_us": plan_us, "plan_host_us_per_layer_of_32": plan_us / 32.0},
        "tokens_per_s": world * rows / ms_step * 1e3, "us_per_step": ms_step * 1e3,
        "pct_of_nominal_8000": 100.0 * value / world / NOMINAL_HBM_GBS,
        "roofline": {"bound": "hbm", "kernel": "decode_kernel<128,3> (+ decode_merge_kernel), per paged_decode_attn call; timed over K back-to-back calls",
                     "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak,
                     "frac_of_nominal_8000": achieved / NOMINAL_HBM_GBS, "avg_launch_ms": dec_ms, "traffic": ncu_traffic_bytes(),
                     "traffic_source": "profiles/r1_decode_ncu_full.csv (dram read + write bytes per decode_kernel launch)",
                     "algorithmic_bytes": kv_bytes},
        "e2e": {"value": total_kv_bytes / e2e_ms / 1e6, "unit": UNIT, "ms_per_step": e2e_ms, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "timing": "wall clock around csv_tail_step_host (host plan + copies + kernels + sync)"},
        "gpu_launches": launches_per_step * K, "clocks": clocks,
        "context": "paper (4xA40, Qwen3-0.6B): p95 TTFET -51.08 %, +7.51 % tokens/J vs AMPD (PAPER.md:7) - scheduling figures, not this path",
    }
    if world == 1:
        # CPU baseline: the oracle as it stands, one host thread, on a bounded sample of the same workload
        dt, nb, rows_s, outs = oracle_sample(wl, 64)
        line["cpu_baseline"] = {"value": nb / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
                                "sample": "all 64 conversations of configs[1] (%.1f MB of KV), all 32 heads, once" % (nb / 1e6),
                                "host_cores_available": len(os.sched_getaffinity(0))}
        # and use that sample as a live parity check of the timed configuration
        O = wl.d_out.cpu().numpy().view(np.uint16)
        from paper_2606_01839_b200 import synth
        err = max(float(np.abs(synth.bf16_bits_to_f32(O[b]).astype(np.float64) - o[0]).max()) for b, (o, _) in zip(rows_s, outs))
        line["parity_sample_max_abs_err"] = err
        if not args.no_extras:
            extras = {}
            for name, fn in (("handoff", handoff_extra), ("agentic_tail_mix", lambda: tail_extra(3)),
                             ("long_context_70b", lambda: tail_extra(5)),
                             ("turn1_prefill_chunked", prefill_extra)):
                try:
                    extras[name] = fn()
                except Exception as e:   # an extra must never cost the headline line
                    extras[name] = {"error": repr(e)[:300]}
                    torch.cuda.empty_cache()
            line["other_workloads"] = extras
    print(json.dumps(line))
    if dist:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--unfused", action="store_true", help="kv_append_tokens + paged_decode_attn as two calls")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py — the conversation-tail KV hot path of ConServe on B200, through the C ABI (conserve_kv.h).

Headline workload = BASELINE.json configs[4], the largest single-GPU configuration: 70B-shaped attention
(Hq=64 Hkv=8 d=128, block size 16), 16 conversations x 131072 tokens, ALL 8 layers resident (68.7 GB of KV), shuffled
paged pool.  One STEP = one decode pass of the tail over that batch: on each of the 8 layers paged_decode_step (the new
token's K/V written into the pool + split-K paged decode attention + merge), replayed from a CUDA graph.
metric = KV bytes read / step time, GB/s, whole job ("gated by KV cache bandwidth at every step";
PAPER.md:112: 262,144 active KV tokens is the regime that matters).

After the headline the same run measures every other kernel and configuration BASELINE.json's metric names and prints
them as first-class records of the same JSON line:
  "rooflines": one block per (kernel, config): decode_kernel on configs[1] / [2] / [4], pack / unpack / direct kernels on
               configs[3], append_tc2_kernel on configs[2] / [4] / turn-1 prefill chunks.  Each: algorithmic work per
               launch, median AND min launch time (CUDA events), achieved, peak, frac, ncu DRAM traffic (only from a
               capture taken on the current kernel source: profiles/r2_traffic.csv).
  "steps":     whole steps: configs[1] (launch-bound case), configs[2] mixed step, configs[4] mixed 8-layer step, each
               with its host-buffer (e2e) time where there is a host call for it.
  "cpu_baseline" (+ "cpu_baselines"): the fp64 oracle on one host core, on all cores, and sampled + extrapolated to
               configs[2] / [4].

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--only LEG] [--no-extras] [--no-graph]

--gpus N without torchrun's environment: bench.py launches its own N ranks (torch.distributed.run on 127.0.0.1).
N > 1: replicas only — every rank serves its own pool of conversations, no data-path collective;
barrier + max-over-ranks timing; value = total bytes / that time.  With >= 2 devices visible, ranks 0 and 1 also time the
paper's one exchange step (prefiller -> decoder handoff over NVLink): "handoff_p2p" in the line.
--impl reference: the fp64 CPU oracle (oracle/), as it stands, on a bounded sample of the headline workload.
--only LEG: run one leg a few times and print its record (what the ncu captures under profiles/ run):
            decode_c5 | decode_c2 | decode_c3 | append_c3 | append_c5 | tail_c3 | handoff | prefill
--ingest-ncu REP --kernel NAME --config CFG: (no GPU) append one row to profiles/r2_traffic.csv from an .ncu-rep.
"""
import argparse
import concurrent.futures
import hashlib
import json
import os
import re
import socket
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
O_TOL, LSE_TOL = 1e-2, 1e-3     # north_star's gates; the sampled rows of the timed configuration are checked live
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r3_traffic.csv")        # --ingest-ncu appends here (one file per round)
TRAFFIC_CSVS = [os.path.join(ROOT, "profiles", "r2_traffic.csv"), TRAFFIC_CSV]   # read in this order: the latest row wins
CSRC = os.path.join(ROOT, "paper_2606_01839_b200", "csrc")
KERNEL_SOURCE = {"decode_kernel": "decode_attn.cu+decode_worker.cuh", "append_tc2_kernel": "append_attn_tc2.cu+append_tc2_body.cuh",
                 "pack_kernel": "handoff.cu", "unpack_kernel": "handoff.cu", "direct_kernel": "handoff.cu",
                 "tail_kernel": "tail_fused.cu+decode_worker.cuh+append_tc2_body.cuh"}   # files whose change voids a capture


# ------------------------------------------------------------------------------------------------ peaks, clocks
def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        j = json.load(open(p))
        return {"hbm": float(j["hbm_gbs"]), "bf16": float(j["bf16_tflops"]),
                "bf16_sustained": float(j.get("bf16_tflops_sustained", j["bf16_tflops"])),
                "source": "measured (MEASURED_PEAKS.json: torch copy read+write; torch.matmul bf16 8192^3 burst / sustained)"}
    except Exception:
        return {"hbm": 6650.0, "bf16": 1590.0, "bf16_sustained": 1400.0,
                "source": "fallback (B200_PROFILING.md: 6.65 TB/s, 1.59 PFLOP/s burst, ~1.4 sustained)"}


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

    def window(self, t0, t1):
        """Summary of the samples taken in [t0, t1] (all samples if none fell inside)."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm, mx, pw, reasons = [], [], [], set()
        rows = [l for (t, l) in self.lines if t0 - 0.05 <= t <= t1 + 0.15] or [l for (_, l) in self.lines]
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except Exception:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w": float(np.median(pw)) if pw else None, "reasons": sorted(reasons), "samples": len(sm)}

    def stop(self):
        if self.proc is not None:
            time.sleep(0.15)
            self.proc.terminate()


# ------------------------------------------------------------------------------------------------ timing helpers
def time_calls(fn, iters, warmup=3):
    """CUDA-event time of fn() on the current stream, one event pair per call: {median_ms, min_ms, mean_ms, n}."""
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
    return {"median_ms": ts[len(ts) // 2], "min_ms": ts[0], "mean_ms": float(np.mean(ts)), "n": len(ts)}


def graph_of(fn):
    """fn() captured in a CUDA graph (the library only enqueues launches on the caller's stream); None if capture fails."""
    import torch

    try:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            fn()
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            fn()
        g.replay()
        torch.cuda.synchronize()
        return g
    except Exception as e:   # never lose the bench line to a capture problem
        sys.stderr.write("CUDA graph capture failed (%r): timing plain launches\n" % (e,))
        torch.cuda.synchronize()
        return None


def sha256_of(files):
    """sha256 over the named csrc files ("a.cu+b.cuh"), in order; None if one is missing."""
    try:
        h = hashlib.sha256()
        for f in files.split("+"):
            h.update(open(os.path.join(CSRC, f), "rb").read())
        return h.hexdigest()
    except Exception:
        return None


def traffic_for(kernel, config):
    """(dram read + write bytes per launch, provenance) from profiles/r2_traffic.csv + r3_traffic.csv — only if the capture
    was taken on the kernel source as it is now (sha256 of the .cu file recorded at capture time); otherwise (None, why)."""
    best = None
    for path in TRAFFIC_CSVS:
        try:
            rows = [l.rstrip("\n").split(",") for l in open(path) if l.strip() and not l.startswith("#")]
        except Exception:
            continue
        hdr = rows[0]
        for r in rows[1:]:
            d = dict(zip(hdr, r))
            if d["kernel"] == kernel and d["config"] == config:
                best = d
    if best is None:
        return None, "no capture for this (kernel, config)"
    cur = sha256_of(best["source_file"])
    if cur != best["source_sha256"]:
        return None, "capture of commit %s is older than %s: refused" % (best["commit"], best["source_file"])
    return float(best["dram_read_bytes"]) + float(best["dram_write_bytes"]), \
        "ncu --set full capture at commit %s (%s), per launch" % (best["commit"], best["report"])


def roofline_block(kernel, config, bound, work, t, pk, note=None, sustained=False):
    """work: algorithmic bytes (hbm) or flops (tensor) per launch; t: time_calls() dict of ONE launch (or call)."""
    if bound == "hbm":
        peak, unit, ach, ach_best = pk["hbm"], "GB/s", work / t["median_ms"] / 1e6, work / t["min_ms"] / 1e6
    else:
        peak, unit, ach, ach_best = pk["bf16"], "TFLOP/s", work / t["median_ms"] / 1e9, work / t["min_ms"] / 1e9
    traffic, tsrc = traffic_for(kernel, config)
    b = {"kernel": kernel, "config": config, "bound": bound, "achieved": ach, "achieved_best": ach_best, "peak": peak,
         "unit": unit, "frac": ach / peak, "frac_best": ach_best / peak, "algorithmic_" + ("bytes" if bound == "hbm" else "flops"): work,
         "launch_ms_median": t["median_ms"], "launch_ms_min": t["min_ms"], "launches_timed": t["n"], "traffic": traffic,
         "traffic_source": tsrc}
    if bound == "hbm":
        b["frac_of_nominal_8000"] = ach / NOMINAL_HBM_GBS
    else:
        b["frac_of_sustained_peak"] = ach / pk["bf16_sustained"]
        b["peak_sustained"] = pk["bf16_sustained"]
    if note:
        b["note"] = note
    return b


# ------------------------------------------------------------------------------------------------ oracle legs (CPU)
def oracle_logical_kv(oracle, wl, b, layer=0):
    """conversation b's raw pool blocks copied back, gathered (paged -> logical) by the ORACLE."""
    img = wl.conversation_blocks_host(b, layer)
    n = len(wl.tables[b])
    return oracle.gather(img, n, wl.Hkv, wl.d, 0, np.arange(n, dtype=np.int32), wl.kv_lens[b])


def oracle_rows(wl, picks, layer=0):
    """picks: [(conversation, row indices inside its chunk or [0] for a decode row)].  Returns the oracle's inputs
    [(b, rows, q [R,Hq,d], K [n,Hkv,d], V)] with K/V truncated to what the LAST picked row sees (causal)."""
    import oracle

    q_all = wl.d_q.cpu().contiguous().view(-1, wl.Hq, wl.d).numpy().view(np.uint16)
    starts = np.concatenate([[0], np.cumsum(wl.q_lens)])
    out = []
    for b, rows in picks:
        K, V = oracle_logical_kv(oracle, wl, b, layer)
        out.append((b, rows, q_all, starts[b], K, V))
    return out


def oracle_eval(item, wl):
    """One pick through the oracle: every picked row is a decode on the cache truncated to what it sees."""
    import oracle

    b, rows, q_all, s0, K, V = item
    m, kv = wl.q_lens[b], wl.kv_lens[b]
    res = []
    for i in rows:
        n = kv - m + i + 1
        o, l = oracle.attention(q_all[s0 + i:s0 + i + 1], K[:n], V[:n])
        res.append((s0 + i, n, o[0], l[0]))
    return res


def parity_of(wl, results, out=None, lse=None):
    """max |O err| and |LSE err| on the oracle's rows of the device outputs (wl.d_out / wl.d_lse as they stand), or of the
    given tensors (e.g. the host buffers a csv_tail_step_host loop filled: same [total_q] row order)."""
    from paper_2606_01839_b200 import synth

    O = (wl.d_out if out is None else out).cpu().reshape(-1, wl.Hq, wl.d).numpy().view(np.uint16)
    LSE = (wl.d_lse if lse is None else lse).cpu().reshape(-1, wl.Hq).numpy().astype(np.float64)
    eo = el = 0.0
    for r, n, o, l in results:
        eo = max(eo, float(np.abs(synth.bf16_bits_to_f32(O[r]).astype(np.float64) - o).max()))
        el = max(el, float(np.abs(LSE[r] - l).max()))
    return eo, el


def route_record(route, eo, el):
    """One entry of parity.routes: the route that was TIMED, checked on its own output."""
    return {"route": route, "max_abs_err_O": eo, "max_abs_err_LSE": el, "ok": bool(eo <= O_TOL and el <= LSE_TOL)}


def oracle_timed(wl, picks, threads, layer=0):
    """Times the oracle on `picks` with `threads` host threads (ctypes releases the GIL).  Returns (seconds, KV
    token-heads scanned, results)."""
    import oracle

    oracle.build()
    items = oracle_rows(wl, picks, layer)
    t0 = time.perf_counter()
    if threads <= 1:
        res = [oracle_eval(it, wl) for it in items]
    else:
        with concurrent.futures.ThreadPoolExecutor(max_workers=threads) as ex:
            res = list(ex.map(lambda it: oracle_eval(it, wl), items))
    dt = time.perf_counter() - t0
    flat = [x for r in res for x in r]
    token_heads = sum(n for _, n, _, _ in flat) * wl.Hq
    return dt, token_heads, flat


# ------------------------------------------------------------------------------------------------ legs (GPU)
def leg_long_context(args, rank, world, ranks_on_dev, dist, agg_dev, pk, sampler):
    """configs[4]: the headline.  Returns (line fields, rooflines, steps, wl, app) — wl stays alive for the oracle legs."""
    import torch
    from paper_2606_01839_b200 import binding as B
    from paper_2606_01839_b200 import replicas, synth, workloads

    cfg = synth.CONFIGS[5]
    free, total = torch.cuda.mem_get_info()
    per_layer = cfg["n_conv"] * cfg["ctx"] * cfg["Hkv"] * cfg["d"] * 2 * 2 * 1.01
    L = int(max(1, min(cfg["NL"], (min(free, total / ranks_on_dev) * 0.92 - 4e9) // per_layer)))
    if args.layers:
        L = min(L, args.layers)
    wl = workloads.config_tail_workload(5, layers=L, seed=replicas.rank_seed(cfg["seed"], rank))
    kv_layer = wl.decode_kv_bytes()
    K, W = args.steps, max(3, args.warmup)

    def step():
        for layer in range(L):
            wl.decode_step(layer=layer)   # paged_decode_step: the new token's K/V write fused into the decode launch

    for _ in range(W):
        step()
    torch.cuda.synchronize()
    graph = None if args.no_graph else graph_of(step)
    run_step = graph.replay if graph is not None else step
    for _ in range(W):
        run_step()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
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
    t1 = time.time()
    ms_total = ev0.elapsed_time(ev1)
    # roofline leg, same process, right after: paged_decode_attn calls (decode_kernel + decode_merge_kernel), one event
    # pair per call, every layer in turn
    calls = [(lambda l=l: wl.decode(layer=l)) for l in range(L)]
    it = iter(range(10 ** 9))
    dec = time_calls(lambda: calls[next(it) % L](), max(2 * L, min(K * L, 80)), warmup=L)
    t2 = time.time()
    clocks = sampler.window(t0, t2) if sampler else None
    ms_total, _ = replicas.aggregate(dist, ms_total, 0, device=agg_dev)
    _, total_bytes = replicas.aggregate(dist, 0, L * kv_layer, device=agg_dev)
    ms_step = ms_total / K
    info = wl.plan.info()

    # e2e: the same step through the C-ABI call with HOST buffers (H2D of every layer's q / k_new / v_new and the tables,
    # host plan, kernels, D2H of O and LSE, sync), wall clock
    rows = len(wl.kv_lens)
    pin = lambda t: t.cpu().pin_memory()
    h_q = pin(wl.d_q.view(1, rows, wl.Hq, wl.d).expand(L, -1, -1, -1).contiguous())
    h_k, h_v = pin(wl.d_k_new.view(L, -1)), pin(wl.d_v_new.view(L, -1))
    h_t = torch.from_numpy(wl.h_tables).pin_memory()
    h_out = torch.zeros((L, rows, wl.Hq, wl.d), dtype=torch.int16).pin_memory()
    h_lse = torch.zeros((L, rows, wl.Hq), dtype=torch.float32).pin_memory()
    ws = torch.empty(B.csv_tail_step_host_workspace_bytes(wl.shape, wl.kv_lens, wl.max_blocks, n_layers=L), dtype=torch.uint8,
                     device="cuda")
    e2e_call = lambda: B.csv_tail_step_host(wl.pool, 0, wl.shape, wl.kv_lens, h_q, h_k, h_v, h_t, wl.max_blocks, ws, h_out,
                                            h_lse, n_layers=L)
    Ke = max(3, min(K, 10))
    for _ in range(2):
        e2e_call()
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    tw = time.perf_counter()
    for _ in range(Ke):
        e2e_call()          # synchronises its stream before returning (the result is on the host)
    e2e_ms = (time.perf_counter() - tw) * 1e3 / Ke
    e2e_ms, _ = replicas.aggregate(dist, e2e_ms, 0, device=agg_dev)
    h2d = (h_q.numel() + h_k.numel() + h_v.numel()) * 2 + h_t.numel() * 4
    d2h = h_out.numel() * 2 + h_lse.numel() * 4
    wl.e2e_layer0 = (h_out[0].clone(), h_lse[0].clone())   # the last host-buffer step's result (layer 0): checked by run_ours
    del ws, h_q, h_k, h_v, h_out, h_lse

    value = total_bytes / ms_step / 1e6
    fields = {
        "value": value, "ms_per_step": ms_step,
        "config": {"workload": "configs[4] c5_long_context_70b: Hq=64 Hkv=8 d=128 bs=16, 16 conversations x 131072 tokens, %d of 8 "
                               "layers resident (%.1f GB of KV per step per GPU), shuffled paged pool; step = paged_decode_step on "
                               "every layer (new-token KV write fused into the decode launch)" % (L, L * kv_layer / 1e9),
                   "layers": L, "kv_bytes_per_step_per_gpu": L * kv_layer, "kv_tokens_per_layer": int(sum(wl.kv_lens)),
                   "decode_rows": rows, "l2": "inputs larger than L2 (%.1f GB of KV per step vs 126 MB)" % (L * kv_layer / 1e9),
                   "parallelism": "replicas x%d on %d device(s), no collective" % (world, max(1, world // ranks_on_dev)),
                   "decode_grid": info["decode_grid"], "decode_items_per_layer": info["n_decode_items"],
                   "split_k_partitions_per_sequence": info["n_decode_items"] / float(rows), "cuda_graph": graph is not None},
        "tokens_per_s": world * rows / ms_step * 1e3, "us_per_step": ms_step * 1e3,
        "pct_of_nominal_8000": 100.0 * value / world / NOMINAL_HBM_GBS,
        "e2e": {"value": total_bytes / e2e_ms / 1e6, "unit": UNIT, "ms_per_step": e2e_ms, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "steps_timed": Ke,
                "timing": "wall clock around csv_tail_step_host (n_layers = %d: H2D, host plan, kernels, D2H, sync)" % L},
        "gpu_launches": 2 * L * K, "clocks": clocks,
    }
    head = roofline_block("decode_kernel", "configs[4]", "hbm", kv_layer, dec, pk,
                          note="per paged_decode_attn call (decode_kernel<128,2,7> + decode_merge_kernel), one layer = 8.59 GB; "
                               "calls cycle over the %d resident layers" % L)
    return fields, head, wl, L


def leg_long_context_extras(wl, L, pk, iters=6):
    """configs[4]: the appended chunks (4 x 256 tokens on 131072-token prefixes) and the whole mixed step."""
    import torch
    from paper_2606_01839_b200 import workloads

    app = wl.with_q_lens(workloads.config5_append_q_lens())
    ap = time_calls(lambda: app.append(layer=0), iters)
    blocks = [roofline_block("append_tc2_kernel", "configs[4]", "tensor", app.append_flops(), ap, pk,
                             note="per append_prefill_attn call on one layer: 4 chunks x 256 tokens, prefix 130816")]

    def parts():
        for layer in range(L):
            wl.decode(layer=layer)
            app.append(layer=layer)

    g = graph_of(parts)
    mx = time_calls(g.replay if g else parts, 3, 1)
    dec = time_calls(lambda: [wl.decode(layer=l) for l in range(L)], 3, 1)
    # the same step in ONE call per layer (csv_tail_step, attention only: S14's rows are in the pool): decode rows and
    # chunks as work items of one persistent launch (tail_fused.cu).  The 4 chunks are extra batch entries whose tables
    # name the blocks of conversations 0-3.
    from paper_2606_01839_b200 import synth
    Lc = synth.config_lengths(5)
    mixed = wl.with_extra_chunks(Lc["append_convs"], Lc["m"])

    def one_call():
        for layer in range(L):
            mixed.tail_attn(layer=layer)

    g1 = graph_of(one_call)
    oc = time_calls(g1.replay if g1 else one_call, 3, 1)
    parts_ms = dec["median_ms"] + L * ap["median_ms"]
    step = {"config": "configs[4]", "what": "decode of all 16 conversations + the 4 appended chunks on each of %d layers, "
            "CUDA-graph replay: one csv_tail_step per layer (decode rows and chunks as work items of one launch)" % L,
            "ms_median": oc["median_ms"], "ms_min": oc["min_ms"], "separate_calls_ms": mx["median_ms"],
            "decode_only_ms": dec["median_ms"], "append_only_ms_per_layer": ap["median_ms"], "sum_of_parts_ms": parts_ms,
            "one_call_vs_sum_of_parts": oc["median_ms"] / parts_ms,
            "hbm_bound_ms": L * (wl.decode_kv_bytes() + app.append_kv_bytes()) / pk["hbm"] / 1e6,
            "tensor_bound_ms": L * app.append_flops() / pk["bf16_sustained"] / 1e9,
            "decode_role_ctas": mixed.plan.info().get("tail_n_dec"),
            "note": "sum_of_parts = each call timed alone, a few launches on a cool chip; the %d-layer graph runs ~45 ms at the "
                    "1000 W cap (sw_power_cap), where the same calls are 10-13 %% slower whichever way they are launched "
                    "(separate_calls_ms is the like-for-like figure); decode_role_ctas 0 = the plan kept the two-kernel route "
                    "(decode is under a quarter of this step)" % L}
    # for the live parity of the timed route: layer 0 through the plan's own route, and the same batch and queries through
    # the ONE-launch route forced by the tuning knob (a twin plan over the same pool)
    from paper_2606_01839_b200 import binding as B
    mixed.d_out.fill_(0x7FC0)
    mixed.tail_attn(layer=0)
    try:
        B.csv_tuning_set(B.TUNE_TAIL_DECODE_CTAS, 26)
        forced = mixed.with_q_lens(mixed.q_lens)
    finally:
        B.csv_tuning_set(B.TUNE_TAIL_DECODE_CTAS, 0)
    forced.d_q.copy_(mixed.d_q)
    forced.d_out.fill_(0x7FC0)
    forced.tail_attn(layer=0)
    torch.cuda.synchronize()
    return blocks, [step], app, mixed, forced


def leg_c2(args, pk, dist, agg_dev):
    """configs[1]: the launch-bound case (1.18 GB per step): device step, per-call roofline, host-buffer step."""
    import torch
    from paper_2606_01839_b200 import binding as B
    from paper_2606_01839_b200 import workloads

    from paper_2606_01839_b200 import synth
    base = [int(t) for t in synth.config_lengths(2)["kv_lens"]]
    # the pool holds 128 tokens more per conversation than the step looks at: the host-buffer loop below GROWS every
    # conversation by one token per step, as a decode loop does
    big = workloads.TailWorkload(32, 8, 128, [1] * len(base), [t + 128 for t in base], seed=synth.CONFIGS[2]["seed"])
    wl = big.with_q_lens([1] * len(base), kv_lens=base)
    kv_bytes = wl.decode_kv_bytes()
    rows = len(wl.kv_lens)
    g = None if args.no_graph else graph_of(wl.decode_step)
    st = time_calls(g.replay if g else wl.decode_step, 100, 5)
    dec = time_calls(wl.decode, 100, 5)
    # the same call without a plan or a workspace (paged_decode_attn_static: host plan + list upload into the library's
    # static scratch array on every call, then the same kernels), for callers that cannot allocate device memory
    stat_out, stat_lse = torch.empty_like(wl.d_out), torch.empty_like(wl.d_lse)
    static_call = lambda: B.paged_decode_attn_static(wl.pool, 0, wl.shape, wl.kv_lens, wl.d_q, wl.d_tables, wl.max_blocks,
                                                     stat_out, stat_lse)
    stat = time_calls(static_call, 100, 5)
    wl.decode()
    torch.cuda.synchronize()
    static_same = bool(torch.equal(stat_out, wl.d_out) and torch.equal(stat_lse, wl.d_lse))
    pin = lambda t: t.cpu().pin_memory()
    h_q, h_k, h_v = pin(wl.d_q), pin(wl.d_k_new), pin(wl.d_v_new)
    h_t = torch.from_numpy(wl.h_tables).pin_memory()
    h_out = torch.zeros((rows, wl.Hq, wl.d), dtype=torch.int16).pin_memory()
    h_lse = torch.zeros((rows, wl.Hq), dtype=torch.float32).pin_memory()
    ws = torch.empty(2 * B.csv_tail_step_host_workspace_bytes(wl.shape, big.kv_lens, wl.max_blocks), dtype=torch.uint8, device="cuda")

    def host_loop(n, warm):
        """n timed steps of a decode loop with host buffers: step i serves kv_len = base + i (one new token each)."""
        t0 = 0.0
        for i in range(warm + n):
            if i == warm:
                torch.cuda.synchronize()
                t0 = time.perf_counter()
            kv = [t + i for t in base]
            B.csv_tail_step_host(wl.pool, 0, wl.shape, kv, h_q, h_k, h_v, h_t, wl.max_blocks, ws, h_out, h_lse)
        return (time.perf_counter() - t0) * 1e3 / n

    e2e_ms = host_loop(100, 5)
    pt = []
    for _ in range(21):
        t0 = time.perf_counter()
        B.Plan(wl.shape, wl.q_lens, wl.kv_lens).destroy()
        pt.append((time.perf_counter() - t0) * 1e6)
    info = wl.plan.info()
    step = {"config": "configs[1]", "what": "64 conversations, context U[1024,8192], 1.18 GB of KV: paged_decode_step "
            "(KV write + decode + merge), CUDA-graph replay", "ms_median": st["median_ms"], "ms_min": st["min_ms"],
            "gbs": kv_bytes / st["median_ms"] / 1e6, "tokens_per_s": rows / st["median_ms"] * 1e3,
            "e2e_host_buffers_ms": e2e_ms, "e2e_gbs": kv_bytes / e2e_ms / 1e6,
            "e2e_what": "csv_tail_step_host over 100 consecutive steps, every conversation one token longer each step (planned "
                        "per step while the H2D copies fly)",
            "h2d_bytes": (h_q.numel() + h_k.numel() + h_v.numel()) * 2 + h_t.numel() * 4,
            "d2h_bytes": h_out.numel() * 2 + h_lse.numel() * 4, "plan_host_us": sorted(pt)[len(pt) // 2],
            "decode_items": info["n_decode_items"],
            "static_scratch_call_ms": stat["median_ms"], "plan_and_workspace_call_ms": dec["median_ms"],
            "static_scratch_what": "paged_decode_attn_static (no plan, no workspace: plans on the host and uploads the lists into "
                                   "the library's 8 MiB static array on every call) against paged_decode_attn on a prebuilt plan; "
                                   "CUDA events around the call", "static_scratch_bit_identical": static_same}
    block = roofline_block("decode_kernel", "configs[1]", "hbm", kv_bytes, dec, pk,
                           note="per paged_decode_attn call (decode_kernel + decode_merge_kernel)")
    # The WHOLE config through the oracle on one core ("c1, c2: the whole config"), timed, and compared with the
    # output of the route that was timed (paged_decode_step); then the host-buffer loop's last step (kv_len = base + 104,
    # h_out / h_lse as the call left them) on 8 conversations.  The oracle reads the pool back as the steps left it.
    wl.d_out.fill_(0x7FC0)
    wl.decode_step()
    torch.cuda.synchronize()
    dt, th, res = oracle_timed(wl, [(b, [0]) for b in range(rows)], 1)
    routes = [route_record("paged_decode_step, configs[1], whole config (64 conversations x 32 heads)", *parity_of(wl, res)),
              route_record("paged_decode_attn_static, configs[1], whole config", *parity_of(wl, res, stat_out, stat_lse))]
    last = big.with_q_lens([1] * rows, kv_lens=[t + 104 for t in base])
    last.d_q.copy_(wl.d_q)
    _, _, res_last = oracle_timed(last, [(b, [0]) for b in range(0, rows, 8)], 1)
    routes.append(route_record("csv_tail_step_host, configs[1], step 105 of the host-buffer decode loop (h_out / h_lse)",
                               *parity_of(last, res_last, h_out, h_lse)))
    cpu = {"config": "configs[1]", "kind": "oracle", "cores": 1, "value": kv_bytes / dt / 1e9, "unit": UNIT, "seconds": dt,
           "sample": "the whole config: 64 conversations, all 32 heads, once",
           "parity_max_abs_err": max(r["max_abs_err_O"] for r in routes),
           "parity_max_lse_err": max(r["max_abs_err_LSE"] for r in routes), "parity_routes": routes}
    del wl, big, last
    torch.cuda.empty_cache()
    return [block], [step], cpu


def leg_c3(args, pk, with_oracle):
    """configs[2], the agentic tail mix: 224 decode rows + 32 appended chunks (m U[32,512]) in one step."""
    import torch
    from paper_2606_01839_b200 import binding as B
    from paper_2606_01839_b200 import workloads

    wl = workloads.config_tail_workload(3)
    dec = time_calls(wl.decode, 10)
    ap = time_calls(wl.append, 6)
    blocks = [roofline_block("decode_kernel", "configs[2]", "hbm", wl.decode_kv_bytes(), dec, pk,
                             note="per paged_decode_attn call: 224 decode rows"),
              roofline_block("append_tc2_kernel", "configs[2]", "tensor", wl.append_flops(), ap, pk,
                             note="per append_prefill_attn call: 32 chunks, %d rows, ragged m" % sum(q for q in wl.q_lens if q > 1))]
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

    def two_streams():
        e = torch.cuda.Event()
        e.record()
        s1.wait_event(e)
        s2.wait_event(e)
        wl.decode(stream=s1)
        wl.append(stream=s2)
        torch.cuda.current_stream().wait_stream(s1)
        torch.cuda.current_stream().wait_stream(s2)

    both = time_calls(two_streams, 5)
    g = graph_of(wl.tail_step)
    one = time_calls(g.replay if g else wl.tail_step, 6)
    # the same mixed step with HOST buffers
    pin = lambda t: t.cpu().pin_memory()
    h_q, h_k, h_v = pin(wl.d_q), pin(wl.d_k_new), pin(wl.d_v_new)
    h_t = torch.from_numpy(wl.h_tables).pin_memory()
    h_out = torch.zeros((wl.total_q, wl.Hq, wl.d), dtype=torch.int16).pin_memory()
    h_lse = torch.zeros((wl.total_q, wl.Hq), dtype=torch.float32).pin_memory()
    ws = torch.empty(B.csv_tail_step_host_workspace_bytes(wl.shape, wl.kv_lens, wl.max_blocks, q_lens=wl.q_lens),
                     dtype=torch.uint8, device="cuda")
    call = lambda: B.csv_tail_step_host(wl.pool, 0, wl.shape, wl.kv_lens, h_q, h_k, h_v, h_t, wl.max_blocks, ws, h_out, h_lse,
                                        q_lens=wl.q_lens)
    for _ in range(2):
        call()
    torch.cuda.synchronize()
    tw = time.perf_counter()
    for _ in range(5):
        call()
    e2e_ms = (time.perf_counter() - tw) * 1e3 / 5
    parts = dec["median_ms"] + ap["median_ms"]
    step = {"config": "configs[2]", "what": "mixed tail step in one call (csv_tail_step: KV write of all %d new rows + 224 decode "
            "rows + 32 appended chunks), CUDA-graph replay" % wl.total_q, "ms_median": one["median_ms"], "ms_min": one["min_ms"],
            "decode_only_ms": dec["median_ms"], "append_only_ms": ap["median_ms"], "sum_of_parts_ms": parts,
            "one_call_vs_sum_of_parts": one["median_ms"] / parts, "two_streams_ms": both["median_ms"],
            "hbm_bound_ms": (wl.decode_kv_bytes() + wl.append_kv_bytes()) / pk["hbm"] / 1e6,
            "tensor_bound_ms": wl.append_flops() / pk["bf16"] / 1e9, "e2e_host_buffers_ms": e2e_ms,
            "decode_role_ctas": wl.plan.info().get("tail_n_dec"),
            "h2d_bytes": (h_q.numel() + h_k.numel() + h_v.numel()) * 2 + h_t.numel() * 4,
            "d2h_bytes": h_out.numel() * 2 + h_lse.numel() * 4}
    cpu = None
    if with_oracle:
        # sampled oracle, extrapolated by KV token-heads: 8 decode rows, 2 chunks x 4 rows
        # the timed route first: csv_tail_step (KV write + the one persistent launch), checked on its OWN output; then
        # the host-buffer call's h_out / h_lse as the last timed iteration left them; then the two standalone calls
        wl.d_out.fill_(0x7FC0)
        wl.tail_step()
        torch.cuda.synchronize()
        dec_rows = [b for b, q in enumerate(wl.q_lens) if q == 1][:8]
        chunks = [b for b, q in enumerate(wl.q_lens) if q > 1][:2]
        picks = [(b, [0]) for b in dec_rows] + [(b, [0, wl.q_lens[b] // 3, (2 * wl.q_lens[b]) // 3, wl.q_lens[b] - 1]) for b in chunks]
        dt, th, res = oracle_timed(wl, picks, 1)
        routes = [route_record("csv_tail_step, configs[2] (one launch, decode_role_ctas %d)" % wl.plan.info()["tail_n_dec"],
                               *parity_of(wl, res)),
                  route_record("csv_tail_step_host, configs[2], last timed host-buffer step (h_out / h_lse)",
                               *parity_of(wl, res, h_out, h_lse))]
        wl.d_out.fill_(0x7FC0)
        wl.decode()
        wl.append()
        torch.cuda.synchronize()
        routes.append(route_record("paged_decode_attn + append_prefill_attn, configs[2] (the roofline blocks' calls)", *parity_of(wl, res)))
        eo, el = max(r["max_abs_err_O"] for r in routes), max(r["max_abs_err_LSE"] for r in routes)
        all_th = sum(kv for q, kv in zip(wl.q_lens, wl.kv_lens) if q == 1) * wl.Hq
        all_th += sum(q * (kv - q) + q * (q + 1) // 2 for q, kv in zip(wl.q_lens, wl.kv_lens) if q > 1) * wl.Hq
        cpu = {"config": "configs[2]", "kind": "oracle", "cores": 1, "sample": "8 decode rows + 2 chunks x 4 rows, all 32 heads",
               "sample_seconds": dt, "sample_token_heads": th, "extrapolated_step_seconds": dt * all_th / th,
               "extrapolated": True, "basis": "KV token-heads scanned (%.3g in the step)" % all_th,
               "parity_max_abs_err": eo, "parity_max_lse_err": el, "parity_routes": routes}
    del wl
    torch.cuda.empty_cache()
    return blocks, [step], cpu


def leg_handoff(pk, iters=5):
    """BASELINE.json configs[3]: 16 conversations x 32 layers of 8B-shape KV, random bits, pack -> unpack (batched), and the
    one-kernel direct route."""
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
    pack = time_calls(lambda: B.kv_pack_batch(desc, ks, vs, toks, offs, sts), iters, 2)
    unpack = time_calls(lambda: B.kv_unpack_batch(pool, sts, toks, offs, ids, nids), iters, 2)
    direct = time_calls(lambda: B.kv_handoff_direct_batch(pool, ks, vs, toks, offs, ids, nids), iters, 2)
    note = "bytes = 2 x payload (read + write), 16 conversations x 32 layers in one batched launch, %.2f GB payload" % (payload / 1e9)
    blocks = [roofline_block("pack_kernel", "configs[3]", "hbm", 2 * payload, pack, pk, note=note),
              roofline_block("unpack_kernel", "configs[3]", "hbm", 2 * payload, unpack, pk, note=note),
              roofline_block("direct_kernel", "configs[3]", "hbm", 2 * payload, direct, pk,
                             note=note + "; kv_handoff_direct: source -> paged pool in one kernel, no staging message")]
    step = {"config": "configs[3]", "what": "one-shot handoff of 16 conversations (%d tokens, 32 layers)" % sum(toks),
            "payload_gb": payload / 1e9, "pack_ms": pack["median_ms"], "unpack_ms": unpack["median_ms"], "direct_ms": direct["median_ms"],
            "handoff_payload_gbs": {"pack_then_unpack": payload / (pack["median_ms"] + unpack["median_ms"]) / 1e6,
                                    "direct": payload / direct["median_ms"] / 1e6}}
    # live parity of the three timed calls (bit-exact): sampled 64 KiB units (conversation, layer, block) against the oracle's
    # staging message and scatter.  The pool is zeroed between the two routes so that neither can pass on the other's bits.
    import oracle

    oracle.build()
    unit = 2 * Hkv * 16 * d
    srng = np.random.default_rng(3003)
    samples = []
    for c in [int(np.argmin(toks)), int(np.argmax(toks))] + [int(x) for x in srng.integers(0, len(toks), size=4)]:
        ntb = synth.blocks_for(toks[c])
        samples += [(c, 0, 0), (c, NL - 1, ntb - 1)] + [(c, int(srng.integers(0, NL)), int(srng.integers(0, ntb))) for _ in range(4)]
    u16 = lambda t: t.cpu().contiguous().numpy().view(np.uint16)

    def units_match(staged):
        bad = 0
        for c, layer, tb in samples:
            t = toks[c]
            lo, hi = tb * 16, min(t, tb * 16 + 16)
            K = u16(ks[c].view(NL, t, Hkv, d)[layer, lo:hi]).reshape(1, hi - lo, Hkv, d)
            V = u16(vs[c].view(NL, t, Hkv, d)[layer, lo:hi]).reshape(1, hi - lo, Hkv, d)
            if staged:   # the 64 KiB unit of the staging message, unused slots zero
                msg = oracle.staging_message(1, Hkv, d, K, V, hi - lo, 0)
                bad += int(not np.array_equal(u16(sts[c].view(NL, synth.blocks_for(t), unit)[layer, tb]), msg))
            got = u16(d_pool.view(NL, nb, unit)[layer, int(ids[c][tb])])
            want = oracle.scatter(np.zeros(unit, dtype=np.uint16), 1, 1, Hkv, d, K, V, hi - lo, 0, np.zeros(1, dtype=np.int32))
            bad += int(not np.array_equal(got, want))
        return bad

    d_pool.zero_()
    B.kv_pack_batch(desc, ks, vs, toks, offs, sts)
    B.kv_unpack_batch(pool, sts, toks, offs, ids, nids)
    torch.cuda.synchronize()
    bad_staged = units_match(True)
    d_pool.zero_()
    B.kv_handoff_direct_batch(pool, ks, vs, toks, offs, ids, nids)
    torch.cuda.synchronize()
    bad_direct = units_match(False)
    step["parity"] = {"what": "%d sampled 64 KiB units (conversation, layer, block) bit for bit against oracle.staging_message / "
                              "oracle.scatter; pool zeroed between the routes" % len(samples),
                      "kv_pack_batch + kv_unpack_batch mismatching units": bad_staged,
                      "kv_handoff_direct_batch mismatching units": bad_direct, "ok": bool(bad_staged == 0 and bad_direct == 0)}
    del ks, vs, sts, d_pool
    torch.cuda.empty_cache()
    return blocks, [step]


def leg_c1():
    """BASELINE.json configs[0], the tiny correctness case (parity only, no roofline claim: everything is launch-bound): 4
    conversations, Hq=4 Hkv=1 d=64, context U[64,512] in a shuffled paged pool, one decode row each through paged_decode_step,
    the whole config against the oracle; plus the 300-token handoff (kv_pack -> kv_unpack, and kv_handoff_direct) into a
    zeroed pool, the whole pool image against oracle.scatter."""
    import torch
    import oracle
    from paper_2606_01839_b200 import binding as B
    from paper_2606_01839_b200 import synth, workloads

    oracle.build()
    wl = workloads.config_tail_workload(1)
    wl.d_out.fill_(0x7FC0)
    wl.decode_step()
    torch.cuda.synchronize()
    dt, _, res = oracle_timed(wl, [(b, [0]) for b in range(len(wl.kv_lens))], 1)
    eo, el = parity_of(wl, res)
    t1 = time_calls(wl.decode_step, 20, 3)
    NL, Hkv, d, tokens, nb = 1, 1, 64, 300, 256
    desc = B.pool_desc(NL, nb, Hkv, d)
    rng = np.random.default_rng(0)
    K = synth.random_bits(rng, (NL, tokens, Hkv, d))
    V = synth.random_bits(rng, (NL, tokens, Hkv, d))
    dk, dv = (torch.from_numpy(a.view(np.int16)).cuda() for a in (K, V))
    ok = {}
    for route in ("kv_pack + kv_unpack", "kv_handoff_direct"):
        d_pool = torch.zeros(B.kv_pool_bytes(desc) // 2, dtype=torch.int16, device="cuda")
        pool = B.KvPool(desc, d_pool)
        pool.set_free_order(synth.shuffled_free_order(np.random.default_rng(1), nb))
        ids = pool.alloc_blocks(synth.blocks_for(tokens))
        d_ids = torch.from_numpy(ids).cuda()
        if route.startswith("kv_pack"):
            st = torch.empty(B.kv_staging_bytes(desc, tokens) // 2, dtype=torch.int16, device="cuda")
            B.kv_pack(desc, dk, dv, tokens, 0, st)
            B.kv_unpack(pool, st, tokens, 0, d_ids, len(ids))
        else:
            B.kv_handoff_direct(pool, dk, dv, tokens, 0, d_ids, len(ids))
        torch.cuda.synchronize()
        want = oracle.scatter(np.zeros(oracle.pool_elems(NL, nb, Hkv, d), dtype=np.uint16), NL, nb, Hkv, d, K, V, tokens, 0, ids)
        ok[route] = bool(np.array_equal(d_pool.cpu().numpy().view(np.uint16), want))
    step = {"config": "configs[0]", "what": "tiny correctness case: 4 decode rows (Hq=4 Hkv=1 d=64, context U[64,512]) through "
            "paged_decode_step + a 300-token handoff; parity only (launch-bound: no roofline claim)",
            "ms_median": t1["median_ms"], "oracle_whole_config_seconds": dt,
            "parity": {"paged_decode_step max_abs_err_O": eo, "paged_decode_step max_abs_err_LSE": el,
                       "handoff whole pool image bit-exact": ok,
                       "ok": bool(eo <= O_TOL and el <= LSE_TOL and all(ok.values()))}}
    return [], [step]


def leg_prefill(pk, iters=4):
    """turn-1 prefill attention of a 32768-token prompt in 8192-token chunks through
    append_prefill_attn (m = 8192, P = earlier chunks), 8B shape, one layer."""
    import torch
    from paper_2606_01839_b200 import workloads

    wl = workloads.TailWorkload(32, 8, 128, [1], [32768], seed=22)
    tot = {"median_ms": 0.0, "min_ms": 0.0, "mean_ms": 0.0, "n": iters}
    flops = 0.0
    for P in (0, 8192, 16384, 24576):
        app = wl.with_q_lens([8192], [P + 8192])
        t = time_calls(app.append, iters)
        for k in ("median_ms", "min_ms", "mean_ms"):
            tot[k] += t[k]
        flops += app.append_flops()
    del wl, app
    torch.cuda.empty_cache()
    return [roofline_block("append_tc2_kernel", "turn-1 prefill 32768 in 4 chunks of 8192", "tensor", flops, tot, pk,
                           note="sum of the 4 append_prefill_attn calls (Hq=32 Hkv=8 d=128, one layer)")], []


# ------------------------------------------------------------------------------------------------ --only (ncu targets)
def run_only(args):
    import torch
    from paper_2606_01839_b200 import binding as B
    from paper_2606_01839_b200 import workloads

    B.lib()
    torch.cuda.set_device(0)
    pk = peaks()
    leg = args.only
    n = max(1, args.steps)
    if leg in ("decode_c2", "decode_c3", "decode_c5", "append_c3", "append_c5", "tail_c3"):
        k = {"2": 2, "3": 3, "5": 5}[leg[-1]]
        wl = workloads.config_tail_workload(k)
        if leg.startswith("decode"):
            t = time_calls(wl.decode, n, 2)
            out = roofline_block("decode_kernel", "configs[%d]" % (k - 1), "hbm", wl.decode_kv_bytes(), t, pk)
        elif leg.startswith("append"):
            app = wl if k == 3 else wl.with_q_lens(workloads.config5_append_q_lens())
            t = time_calls(app.append, n, 2)
            out = roofline_block("append_tc2_kernel", "configs[%d]" % (k - 1), "tensor", app.append_flops(), t, pk)
        else:
            t = time_calls(wl.tail_step, n, 2)
            out = {"leg": leg, "ms_median": t["median_ms"], "ms_min": t["min_ms"]}
    elif leg == "handoff":
        out = {"rooflines": leg_handoff(pk, iters=n)[0]}
    elif leg == "prefill":
        out = {"rooflines": leg_prefill(pk, iters=n)[0]}
    else:
        raise SystemExit("unknown --only leg %r" % leg)
    print(json.dumps(out))


def ingest_ncu(args):
    """profiles/r3_traffic.csv += one row: mean dram read / write bytes per launch of `--kernel` in an .ncu-rep."""
    txt = subprocess.run(["ncu", "-i", args.ingest_ncu, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    import csv
    import io

    rows = list(csv.reader(io.StringIO(txt)))
    hdr, units = rows[0], rows[1]
    col = {h: i for i, h in enumerate(hdr)}
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    rd, wr, n = 0.0, 0.0, 0
    for r in rows[2:]:
        if not re.search(r"(?<![A-Za-z_])" + re.escape(args.kernel) + r"(?![A-Za-z_])", r[col["Kernel Name"]]):
            continue
        rd += float(r[col["dram__bytes_read.sum"]].replace(",", "")) * mult[units[col["dram__bytes_read.sum"]]]
        wr += float(r[col["dram__bytes_write.sum"]].replace(",", "")) * mult[units[col["dram__bytes_write.sum"]]]
        n += 1
    if n == 0:
        raise SystemExit("no launch of %s in %s" % (args.kernel, args.ingest_ncu))
    src = KERNEL_SOURCE[args.kernel]
    commit = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
    new = not os.path.exists(TRAFFIC_CSV)
    with open(TRAFFIC_CSV, "a") as f:
        if new:
            f.write("# dram__bytes_read.sum / dram__bytes_write.sum per launch (mean over the captured launches) of `ncu --set full` "
                    "captures; written by `python bench.py --ingest-ncu REP --kernel K --config C` (commands: profiles/r3_README.md).\n"
                    "# bench.py reports a row as roofline.traffic only while sha256 over the csrc files named in source_file still equals source_sha256.\n")
            f.write("kernel,config,dram_read_bytes,dram_write_bytes,launches,commit,source_file,source_sha256,report\n")
        f.write("%s,%s,%.0f,%.0f,%d,%s,%s,%s,%s\n" % (args.kernel, args.config, rd / n, wr / n, n, commit, src,
                                                    sha256_of(src), os.path.basename(args.ingest_ncu)))
    print("%s %s: read %.4f GB, write %.4f GB per launch (%d launches)" % (args.kernel, args.config, rd / n / 1e9, wr / n / 1e9, n))


# ------------------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric / config as our arm, bounded sample per step: ONE
    conversation-layer of configs[4] (131072 tokens, all 64 query heads), one thread."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_2606_01839_b200 import synth

    oracle.build()
    cfg = synth.CONFIGS[5]
    rng = np.random.default_rng(cfg["seed"])
    T = cfg["ctx"]
    q = synth.normal_bf16(rng, (1, cfg["Hq"], cfg["d"]))
    K = synth.normal_bf16(rng, (T, cfg["Hkv"], cfg["d"]))
    V = synth.normal_bf16(rng, (T, cfg["Hkv"], cfg["d"]))
    nbytes = T * cfg["Hkv"] * cfg["d"] * 2 * 2
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.attention(q, K, V)
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    sec = float(np.mean(times))
    gbs = nbytes / sec / 1e9
    sample = "one conversation-layer of configs[4] (131072 tokens, %.1f MB of KV, all 64 query heads) per step, 1 thread" % (nbytes / 1e6)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[4] c5_long_context_70b (bounded sample)", "sample": sample},
        "cpu_baseline": {"value": gbs, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": gbs, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    from paper_2606_01839_b200 import build as libbuild

    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        libbuild.build_library()             # no-op when the in-tree .so is up to date; there is no fallback path
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    ndev = max(1, torch.cuda.device_count())
    ranks_on_dev = (world + ndev - 1) // ndev      # > 1 only when there are fewer devices than ranks (they share)
    local = local % ndev
    torch.cuda.set_device(local)
    dist, agg_dev = None, "cuda"
    if world > 1:
        import torch.distributed as dist_mod

        dist = dist_mod
        try:   # the only cross-rank traffic is a barrier and scalar reductions (replicas, no data-path collective)
            if ranks_on_dev > 1:
                raise RuntimeError("ranks share a device: NCCL refuses duplicate GPUs")
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
            dist.barrier()
        except Exception as e:
            sys.stderr.write("nccl not used (%r): gloo for the barrier / scalar reductions\n" % (e,))
            if dist.is_initialized():
                dist.destroy_process_group()
            dist.init_process_group("gloo")
            agg_dev = "cpu"
        if local != 0 or rank != 0:
            time.sleep(0)   # every rank builds nothing; rank 0 of the node built the library above
        dist.barrier()
    from paper_2606_01839_b200 import binding as B

    B.lib()   # fails loudly if libconserve_kv.so is missing: there is no fallback
    if args.only:
        return run_only(args)
    pk = peaks()
    sampler = ClockSampler(local) if rank == 0 else None
    fields, head, wl, L = leg_long_context(args, rank, world, ranks_on_dev, dist, agg_dev, pk, sampler)

    p2p = None
    if world >= 2 and (ndev >= 2 or args.p2p):
        # the paper's one exchange step, prefiller (rank 0) -> decoder (rank 1), over NVLink
        try:
            from paper_2606_01839_b200 import handoff_p2p

            p2p = handoff_p2p.run(dist, rank, tokens=8192, layers=32, convs=4, iters=3)
        except Exception as e:
            p2p = {"error": repr(e)[:300]}
        box = [p2p if rank == 1 else None]          # the decoder (rank 1) holds the record; every rank joins the broadcast
        dist.broadcast_object_list(box, src=1)
        p2p = box[0]
    if rank != 0:
        if sampler:
            sampler.stop()
        if dist:
            dist.barrier()
            dist.destroy_process_group()
        return

    line = {"metric": METRIC, "value": None, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": None, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
            "data": "synthetic"}
    line.update(fields)
    line["roofline"] = dict(head)
    line["roofline"]["peak_source"] = pk["source"]
    line["context"] = ("paper (4xA40, Qwen3-0.6B): p95 TTFET -51.08 %, +7.51 % tokens/J vs AMPD (PAPER.md:7) - scheduling figures, "
                       "not this path")
    if p2p is not None:
        line["handoff_p2p"] = p2p
    rooflines, steps, cpus = [head], [], []
    if world == 1:
        # ---- CPU baseline: the oracle as it stands on a bounded sample of the headline workload (layer 0) -------------
        # the route that was timed: paged_decode_step (the new token's KV write inside the decode launch).  It leaves the
        # token in the pool, and the oracle reads the pool back afterwards, so the write is part of what is checked.
        wl.d_out.fill_(0x7FC0)
        wl.decode_step(layer=0)
        torch.cuda.synchronize()
        cores = len(os.sched_getaffinity(0))
        dt1, th1, res1 = oracle_timed(wl, [(b, [0]) for b in range(4)], 1)
        nb1 = 4 * wl.kv_lens[0] * wl.Hkv * wl.d * 4
        eo, el = parity_of(wl, res1)
        nall = min(len(wl.kv_lens), max(cores, 4))
        dtn, thn, resn = oracle_timed(wl, [(b, [0]) for b in range(nall)], cores)
        eo2, el2 = parity_of(wl, resn)
        eo, el = max(eo, eo2), max(el, el2)
        routes = [route_record("paged_decode_step, configs[4] layer 0 (the headline step's call), %d conversations" % nall, eo, el)]
        routes.append(route_record("csv_tail_step_host, configs[4] layer 0 of the last timed host-buffer step (h_out / h_lse)",
                                   *parity_of(wl, resn, *wl.e2e_layer0)))
        wl.d_out.fill_(0x7FC0)
        wl.decode(layer=0)
        torch.cuda.synchronize()
        routes.append(route_record("paged_decode_attn, configs[4] layer 0 (the roofline block's call)", *parity_of(wl, resn)))
        eo, el = max(r["max_abs_err_O"] for r in routes), max(r["max_abs_err_LSE"] for r in routes)
        nbn = nall * wl.kv_lens[0] * wl.Hkv * wl.d * 4
        line["cpu_baseline"] = {"value": nb1 / dt1 / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt1,
                                "sample": "4 of the 16 conversations of configs[4], layer 0 (%.1f GB of KV), all 64 heads, once" % (nb1 / 1e9),
                                "host_cores_available": cores}
        step_th = L * sum(wl.kv_lens) * wl.Hq
        cpus.append({"config": "configs[4]", "kind": "oracle", "cores": cores, "value": nbn / dtn / 1e9, "unit": UNIT,
                     "seconds": dtn, "sample": "%d conversations of layer 0 over a pool of %d threads (one conversation per task)" % (nall, cores)})
        cpus.append({"config": "configs[4]", "kind": "oracle", "cores": 1, "extrapolated": True,
                     "extrapolated_step_seconds": dt1 * step_th / th1, "basis": "KV token-heads scanned (%.3g in the %d-layer decode step)" % (step_th, L),
                     "sample_seconds": dt1})
        line["parity"] = {"config": "configs[4] layer 0, %d conversations x 64 heads against the oracle" % nall,
                          "max_abs_err_O": eo, "max_abs_err_LSE": el, "gate_O": O_TOL, "gate_LSE": LSE_TOL,
                          "ok": bool(eo <= O_TOL and el <= LSE_TOL), "routes": routes}
        if not args.no_extras:
            def guarded(name, fn):
                try:
                    return fn()
                except Exception as e:   # an extra must never cost the headline line
                    sys.stderr.write("leg %s failed: %r\n" % (name, e))
                    torch.cuda.empty_cache()
                    return None
            r = guarded("long_context_extras", lambda: leg_long_context_extras(wl, L, pk))
            if r:
                rooflines += r[0]
                steps += r[1]
                app, mixed, forced = r[2], r[3], r[4]
                # two sampled rows of one appended chunk through the oracle, extrapolated to the step
                try:
                    app.append(layer=0)
                    torch.cuda.synchronize()
                    dta, tha, resa = oracle_timed(app, [(0, [0, 255])], 1)
                    ea, ela = parity_of(app, resa)
                    ath = L * sum(q * (kv - q) + q * (q + 1) // 2 for q, kv in zip(app.q_lens, app.kv_lens) if q > 1) * app.Hq
                    cpus.append({"config": "configs[4] appended chunks", "kind": "oracle", "cores": 1, "extrapolated": True,
                                 "sample": "rows 0 and 255 of chunk 0, layer 0, all 64 heads", "sample_seconds": dta,
                                 "extrapolated_step_seconds": dta * ath / tha, "parity_max_abs_err": ea, "parity_max_lse_err": ela})
                    line["parity"]["append_sample_max_abs_err_O"] = ea
                    line["parity"]["append_sample_max_abs_err_LSE"] = ela
                    line["parity"]["ok"] = bool(line["parity"]["ok"] and ea <= O_TOL and ela <= LSE_TOL)
                    # the mixed step as timed (csv_tail_step per layer): one decode row + rows 0 and 255 of chunk entry 16
                    # (an alias of conversation 0), on the plan's route and on the forced one-launch route
                    _, _, resm = oracle_timed(mixed, [(5, [0]), (16, [0, 255])], 1)
                    for w, name in ((mixed, "csv_tail_step, configs[4] mixed step layer 0, the plan's route (decode_role_ctas %d)"
                                     % mixed.plan.info()["tail_n_dec"]),
                                    (forced, "csv_tail_step, configs[4] mixed step layer 0, one launch forced (decode_role_ctas %d)"
                                     % forced.plan.info()["tail_n_dec"])):
                        line["parity"]["routes"].append(route_record(name, *parity_of(w, resm)))
                    line["parity"]["routes"].append(route_record("append_prefill_attn, configs[4] layer 0 (the roofline block's call)", ea, ela))
                    line["parity"]["ok"] = bool(line["parity"]["ok"] and all(r["ok"] for r in line["parity"]["routes"]))
                except Exception as e:   # an extra must never cost the headline line: the route is listed as unchecked
                    sys.stderr.write("append oracle sample failed: %r\n" % (e,))
                    line["parity"]["routes"].append({"route": "configs[4] appended chunks / mixed step", "ok": None,
                                                     "unchecked": repr(e)[:200]})
                del app, mixed, forced
        del wl
        torch.cuda.empty_cache()
        if not args.no_extras:
            for name, fn in (("c1", lambda: leg_c1() + (None,)), ("c2", lambda: leg_c2(args, pk, dist, agg_dev)),
                             ("c3", lambda: leg_c3(args, pk, True)),
                             ("handoff", lambda: leg_handoff(pk) + (None,)), ("prefill", lambda: leg_prefill(pk) + (None,))):
                r = guarded(name, fn)
                if r:
                    rooflines += r[0]
                    steps += r[1]
                    for st in r[1]:   # legs whose parity is bit-exact work (handoff) or a whole tiny config carry it in their step
                        if isinstance(st.get("parity"), dict):
                            line["parity"]["routes"].append({"route": st["config"] + ": " + st["parity"].get("what", st["what"])[:160],
                                                             "ok": st["parity"]["ok"]})
                            line["parity"]["ok"] = bool(line["parity"]["ok"] and st["parity"]["ok"])
                    if len(r) > 2 and r[2]:
                        line["parity"]["routes"] += r[2].pop("parity_routes", [])
                        cpus.append(r[2])
                        line["parity"]["ok"] = bool(line["parity"]["ok"] and r[2].get("parity_max_abs_err", 0) <= O_TOL and
                                                    r[2].get("parity_max_lse_err", 0) <= LSE_TOL)
        if not line["parity"]["ok"]:
            line["value"] = None   # a kernel that fails its live parity check has no bench value
    line["rooflines"] = rooflines
    line["steps_measured"] = steps
    line["cpu_baselines"] = cpus
    if sampler:
        sampler.stop()
    print(json.dumps(line))
    if dist:
        dist.barrier()
        dist.destroy_process_group()
    if world == 1 and not line["parity"]["ok"]:
        sys.exit(3)


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--layers", type=int, default=0, help="cap on the resident layers of configs[4] (default: all 8 that fit)")
    ap.add_argument("--p2p", action="store_true", help="time the prefiller -> decoder handoff between ranks 0 and 1 even when "
                    "they share one device (it always runs when two devices are visible)")
    ap.add_argument("--only", default=None)
    ap.add_argument("--ingest-ncu", default=None)
    ap.add_argument("--kernel", default=None)
    ap.add_argument("--config", default=None)
    args = ap.parse_args()
    if args.ingest_ncu:
        return ingest_ncu(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and not args.only:
        # launched without torchrun: start our own N ranks, one per GPU (modulo the device count), and become them
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
        os.execv(sys.executable, cmd)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

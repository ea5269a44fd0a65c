"""Seeded synthetic inputs shaped like the paper's agentic tails.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests.  It
holds none of the method's arithmetic (no attention, no layout formula, no
planner): only random lengths, random values and random block permutations.

Shapes follow BASELINE.json's five configs; the paper's workload shape behind
them: turn-1 prompts of tens of thousands of tokens, appends of hundreds
(§3, Fig. 1), decoders holding up to 262,144 active KV tokens
(§3.2).  The paper's traces (SWE-bench_bm25_13K + swe-agent) are
NOT reproduced; these inputs stand in for them.

Readings (S12-S15): medians are decimal (12000, 8000), clip bounds
binary (2048..65536, 1024..32768); sigma is the std-dev of ln(length);
len = clip(rint(median * exp(sigma * z))); "uniform in [a,b]" is integer with
both ends included.  Config k uses seed k - 1.
"""
import numpy as np

BLOCK = 16

CONFIGS = {
    1: dict(name="c1_tiny", NL=1, Hq=4, Hkv=1, d=64, n_conv=4, pool_blocks=256, seed=0),
    2: dict(name="c2_llama8b_decode64", NL=1, Hq=32, Hkv=8, d=128, n_conv=64, seed=1),
    3: dict(name="c3_agentic_tail_mix", NL=1, Hq=32, Hkv=8, d=128, n_conv=256, n_append=32, seed=2),
    4: dict(name="c4_handoff_32layer", NL=32, Hq=32, Hkv=8, d=128, n_conv=16, seed=3),
    5: dict(name="c5_long_context_70b", NL=8, Hq=64, Hkv=8, d=128, n_conv=16, ctx=131072, n_append=4,
            m_append=256, seed=4),
}


def f32_to_bf16_bits(x):
    """fp32 -> bf16 bit patterns (uint16), round to nearest even (NaN kept quiet)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    rounded = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    out = rounded.astype(np.uint16)
    nan = np.isnan(x)
    if nan.any():
        out[nan] = np.uint16(0x7FC0)
    return out


def bf16_bits_to_f32(bits):
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32)


def normal_bf16(rng, shape, mean=0.0, std=1.0):
    """bf16 N(mean, std) as uint16 bit patterns."""
    return f32_to_bf16_bits((rng.standard_normal(shape, dtype=np.float32) * np.float32(std) + np.float32(mean)))


def random_bits(rng, shape):
    """Uniform random 16-bit patterns (NaN / Inf / denormal patterns included): config 4."""
    return rng.integers(0, 1 << 16, size=shape, dtype=np.uint16)


def uniform_lengths(rng, n, lo, hi):
    return rng.integers(lo, hi + 1, size=n).astype(np.int32)


def lognormal_lengths(rng, n, median, sigma, lo, hi):
    z = rng.standard_normal(n)
    return np.clip(np.rint(median * np.exp(sigma * z)), lo, hi).astype(np.int32)


def blocks_for(tokens):
    return (int(tokens) + BLOCK - 1) // BLOCK


def config_lengths(k):
    """Lengths of config k. Returns a dict of int32 arrays (see keys per config)."""
    cfg = CONFIGS[k]
    rng = np.random.default_rng(cfg["seed"])
    if k == 1:
        return dict(kv_lens=uniform_lengths(rng, cfg["n_conv"], 64, 512), prefill_tokens=300)
    if k == 2:
        return dict(kv_lens=uniform_lengths(rng, cfg["n_conv"], 1024, 8192))
    if k == 3:
        prefix = lognormal_lengths(rng, cfg["n_conv"], 12000, 0.8, 2048, 65536)
        is_append = np.zeros(cfg["n_conv"], dtype=bool)
        is_append[rng.choice(cfg["n_conv"], size=cfg["n_append"], replace=False)] = True
        m = uniform_lengths(rng, cfg["n_conv"], 32, 512)
        q_lens = np.where(is_append, m, 1).astype(np.int32)
        # decode rows: kv_len = context length; append chunks: kv_len = P + m
        kv_lens = np.where(is_append, prefix + m, prefix).astype(np.int32)
        return dict(q_lens=q_lens, kv_lens=kv_lens)
    if k == 4:
        return dict(tokens=lognormal_lengths(rng, cfg["n_conv"], 8000, 0.7, 1024, 32768))
    if k == 5:
        kv = np.full(cfg["n_conv"], cfg["ctx"], dtype=np.int32)
        return dict(kv_lens=kv, append_convs=np.arange(cfg["n_append"], dtype=np.int32), m=cfg["m_append"])
    raise KeyError(k)


def shuffled_free_order(rng, num_blocks):
    """A full random permutation of a pool's block ids (the shuffled free list)."""
    return rng.permutation(num_blocks).astype(np.int32)


def pool_blocks_for(kv_lens, slack=0.10, minimum=0):
    need = int(sum(blocks_for(t) for t in kv_lens))
    return max(int(np.ceil(need * (1.0 + slack))), need + 1, minimum)


def dense_tables(block_lists, pad=-1):
    """List of per-conversation id arrays -> [batch][max_blocks] int32 (+ max_blocks).
    Unused entries are `pad` (an out-of-range id: kernels must never read them)."""
    mb = max(1, max(len(b) for b in block_lists))
    out = np.full((len(block_lists), mb), pad, dtype=np.int32)
    for i, b in enumerate(block_lists):
        out[i, : len(b)] = b
    return out, mb

"""Shared plumbing of the GPU parity tests (not a test itself).

Inputs are built on the host with numpy + the ORACLE's layout restatement (oracle.scatter)
and uploaded; the CUDA path never produces an oracle input or an expected value.
"""
import os

import numpy as np
import torch

from paper_2606_01839_b200 import binding as B
from paper_2606_01839_b200 import synth

O_TOL = 1e-2      # north_star: max |err| <= 1e-2 absolute on O
LSE_TOL = 1e-3    # north_star: LSE within 1e-3
NORM_TOL = 3e-2   # max|err| / rms(O_ref) per row (bf16 P and O rounding give ~1.5e-2)


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.view(dtype)
    return t.cuda()


def u16_dev(a):
    """numpy uint16 -> CUDA int16 tensor with the same bits."""
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).cuda()


def dev_to_u16(t):
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def bf16_dev_to_f64(t):
    return synth.bf16_bits_to_f32(dev_to_u16(t)).astype(np.float64)


class Scenario:
    """A paged pool on the host (uint16 image) + per-conversation logical K/V and tables."""

    def __init__(self, oracle, rng, Hq, Hkv, d, kv_lens, NL=1, slack_blocks=8, poison=False, v_mean=0.0,
                 pool_blocks=None):
        self.oracle, self.Hq, self.Hkv, self.d, self.NL = oracle, Hq, Hkv, d, NL
        self.kv_lens = [int(x) for x in kv_lens]
        need = sum(synth.blocks_for(t) for t in self.kv_lens)
        self.num_blocks = pool_blocks or (need + slack_blocks)
        elems = oracle.pool_elems(NL, self.num_blocks, Hkv, d)
        if poison:   # S9: every unused slot / block holds a NaN bit pattern
            self.image = np.full(elems, 0x7FC1, dtype=np.uint16)
        else:
            self.image = np.zeros(elems, dtype=np.uint16)
        order = synth.shuffled_free_order(rng, self.num_blocks)
        self.free_order = order
        self.tables, self.K, self.V = [], [], []
        pos = 0
        for t in self.kv_lens:
            nb = synth.blocks_for(t)
            ids = order[pos:pos + nb]
            pos += nb
            self.tables.append(ids.copy())
            K = synth.normal_bf16(rng, (NL, t, Hkv, d))
            V = synth.normal_bf16(rng, (NL, t, Hkv, d), mean=v_mean)
            self.K.append(K)
            self.V.append(V)
        self.used = pos
        self.pad_id = -1 if not poison else 0x7FFFFFF

    def commit(self):
        """Scatter every conversation's logical KV into the image with the oracle (O3)."""
        for t, ids, K, V in zip(self.kv_lens, self.tables, self.K, self.V):
            if t > 0:
                self.image = self.oracle.scatter(self.image, self.NL, self.num_blocks, self.Hkv, self.d, K, V, t, 0, ids)
        return self

    def upload(self):
        self.d_image = u16_dev(self.image)
        desc = B.pool_desc(self.NL, self.num_blocks, self.Hkv, self.d)
        self.pool = B.KvPool(desc, self.d_image)
        tabs, self.max_blocks = synth.dense_tables(self.tables, pad=self.pad_id)
        self.h_tables = tabs
        self.d_tables = dev(tabs)
        return self


def run_attention(sc, q_lens, q_bits, layer=0, mpt=0, which="both"):
    """q_bits: uint16 [total_q, Hq, d].  Returns (O f64 [total_q,Hq,d], LSE f64 [total_q,Hq], plan info)."""
    shape = B.attn_shape(sc.Hq, sc.Hkv, sc.d)
    ws_bytes = B.csv_plan_workspace_bytes(shape, q_lens, sc.kv_lens, mpt)
    ws = torch.empty(max(ws_bytes, 128), dtype=torch.uint8, device="cuda")
    plan = B.Plan(shape, q_lens, sc.kv_lens, mpt, ws)
    total_q = int(np.sum(q_lens))
    d_q = u16_dev(q_bits)
    d_out = torch.full((max(total_q, 1), sc.Hq, sc.d), 0x7FC0, dtype=torch.int16, device="cuda")   # NaN sentinel
    d_lse = torch.full((max(total_q, 1), sc.Hq), float("nan"), dtype=torch.float32, device="cuda")
    if which in ("both", "decode"):
        # decode reads row b of [batch][Hq][d]; when every q_len is 1 that is the same buffer
        B.paged_decode_attn(plan, sc.pool, layer, d_q, sc.d_tables, sc.max_blocks, d_out, d_lse)
    if which in ("both", "append"):
        B.append_prefill_attn(plan, sc.pool, layer, d_q, sc.d_tables, sc.max_blocks, d_out, d_lse)
    if which == "tail":   # csv_tail_step, attention only (the rows are in the pool): one fused launch for a mixed batch
        B.csv_tail_step(plan, sc.pool, layer, d_q, None, None, sc.d_tables, sc.max_blocks, d_out, d_lse)
    torch.cuda.synchronize()
    info = plan.info()
    return bf16_dev_to_f64(d_out), d_lse.cpu().numpy().astype(np.float64), info


def oracle_attention(sc, q_lens, q_bits, layer=0):
    """Oracle O1 on the logical KV of every conversation with q_len > 0."""
    total_q = int(np.sum(q_lens))
    O = np.zeros((total_q, sc.Hq, sc.d))
    LSE = np.zeros((total_q, sc.Hq))
    r = 0
    for b, m in enumerate(q_lens):
        if m == 0:
            continue
        L = sc.kv_lens[b]
        o, l = sc.oracle.attention(q_bits[r:r + m], sc.K[b][layer][:L], sc.V[b][layer][:L])
        O[r:r + m], LSE[r:r + m] = o, l
        r += m
    return O, LSE


def oracle_abs_weighted(sc, q_lens, q_bits, layer=0):
    """A[r][h][c] = sum_j p_j |V_j[c]|: the oracle's O1 run on |V| (sign bit of every bf16 cleared).  It is what the two
    bf16 roundings of the GPU path (P before the PV product, O on output) are relative to (S20)."""
    total_q = int(np.sum(q_lens))
    A = np.zeros((total_q, sc.Hq, sc.d))
    r = 0
    for b, m in enumerate(q_lens):
        if m == 0:
            continue
        L = sc.kv_lens[b]
        if L > 0:
            A[r:r + m] = sc.oracle.attention(q_bits[r:r + m], sc.K[b][layer][:L], sc.V[b][layer][:L] & np.uint16(0x7FFF))[0]
        r += m
    return A


def logical_kv(oracle, wl, b, layer=0):
    """Conversation b of a device workload as logical K, V: its blocks are copied back as raw pool bytes and the
    ORACLE gathers them (paged -> logical) from a compact 1-layer pool with the identity table."""
    img = wl.conversation_blocks_host(b, layer)
    n = len(wl.tables[b])
    return oracle.gather(img, n, wl.Hkv, wl.d, 0, np.arange(n, dtype=np.int32), wl.kv_lens[b])


def assert_close(O, LSE, O_ref, LSE_ref, what="", norm=True, A_ref=None):
    assert np.all(np.isfinite(O)), "%s: non-finite O" % what
    assert np.all(np.isfinite(LSE)), "%s: non-finite LSE" % what
    err = np.abs(O - O_ref)
    # north_star's 1e-2 absolute bound is stated for "outputs O(1)".  A bf16 output of magnitude in [2^k, 2^(k+1)) is
    # rounded by up to half an ulp = 2^(k-8) on its own (7.8e-3 in [2,4), 1.6e-2 in [4,8)), so from |O_ref| >= 2 on that
    # half-ulp is added to the bound, element by element; below 2 the bound is the plain 1e-2 (S20).
    mag = np.abs(O_ref)
    extra = np.where(mag >= 2.0, np.exp2(np.floor(np.log2(np.maximum(mag, 1.0))) - 8.0), 0.0)
    tol = O_TOL + extra
    if A_ref is not None:
        # Only the q-scaled cases pass A_ref = sum_j p_j |V_j| (oracle_abs_weighted).  With scores of +-30 the softmax
        # sits on one or two keys, so outputs reach |V|max ~ 4 and the rounding of P to bf16 (allowed: S7; unit roundoff
        # 2^-8) is no longer averaged over many keys: |err| <= 2^-8 A (P) + 2^-8 |O| (output) <= 2^-7 A.  The bound is
        # the larger of the plain gate and that one, element by element (S20).
        tol = np.maximum(tol, np.exp2(-7.0) * A_ref)
    bad = err > tol
    assert not bad.any(), "%s: max |O err| %.3e > %.0e (+ half a bf16 ulp where |O_ref| >= 2%s); worst excess %.3e" % (
        what, err.max(), O_TOL, "; 2^-7 sum p|V| where larger" if A_ref is not None else "", (err - tol).max())
    if (err > O_TOL).any() and os.environ.get("CSV_TOL_LOG"):   # which cases needed more than the plain 1e-2 (listed in S20)
        with open(os.environ["CSV_TOL_LOG"], "a") as f:
            f.write("%s: max err %.4e at |O_ref| %.3f\n" % (what, err.max(), float(mag.reshape(-1)[err.argmax()])))
    lerr = np.abs(LSE - LSE_ref).max()
    assert lerr <= LSE_TOL, "%s: max |LSE err| %.3e > %.0e" % (what, lerr, LSE_TOL)
    if norm:
        rms = np.sqrt((O_ref ** 2).mean(axis=-1))
        nerr = (err.max(axis=-1) / np.maximum(rms, 1e-30)).max()
        assert nerr <= NORM_TOL, "%s: normalised error %.3e > %.0e" % (what, nerr, NORM_TOL)
    return float(err.max()), float(lerr)

"""ctypes binding of libconserve_kv.so: same names as include/conserve_kv.h.

Argument marshalling only (pointers, sizes, the current torch stream): every step
of the path runs in the library's kernels.  There is no fallback: if the library
has not been built, the first call raises.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libconserve_kv.so")

CSV_OK, CSV_E_INVAL, CSV_E_NOMEM, CSV_E_CUDA = 0, -1, -2, -3
BLOCK = 16

# every symbol include/conserve_kv.h declares (tests check the library exports them all)
SYMBOLS = [
    "csv_last_cuda_error", "csv_version", "kv_pool_bytes", "kv_pool_create", "kv_pool_destroy",
    "kv_pool_set_free_order", "kv_alloc_blocks", "kv_free_blocks", "kv_pool_used_blocks", "kv_pool_num_blocks",
    "kv_pool_free_blocks", "kv_pool_get_desc", "csv_place", "csv_provision", "kv_staging_bytes", "kv_pack",
    "kv_unpack", "kv_pack_batch", "kv_unpack_batch", "kv_append_tokens", "csv_plan_workspace_bytes",
    "csv_plan_create", "csv_plan_destroy", "csv_plan_info", "csv_plan_tail_split", "csv_plan_decode_workers", "csv_plan_total_q", "csv_plan_decode_items",
    "csv_plan_append_items", "paged_decode_attn", "paged_decode_step", "append_prefill_attn", "csv_tail_step_host_workspace_bytes",
    "csv_tail_step_host", "kv_handoff_direct", "kv_handoff_direct_batch", "csv_ipc_export", "csv_ipc_open", "csv_ipc_close", "csv_ipc_copy", "csv_tail_step",
    "paged_decode_attn_static", "csv_ipc_mapped_bytes", "csv_tuning_set", "csv_tuning_get",
]
IPC_HANDLE_BYTES = 64


class KvPoolDesc(ctypes.Structure):
    _fields_ = [("num_layers", ctypes.c_int32), ("num_blocks", ctypes.c_int32), ("block_size", ctypes.c_int32),
                ("num_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32), ("dtype", ctypes.c_int32)]


class AttnShape(ctypes.Structure):
    _fields_ = [("num_q_heads", ctypes.c_int32), ("num_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
                ("block_size", ctypes.c_int32)]


class CsvError(RuntimeError):
    def __init__(self, fn, code, cuda=0):
        self.code, self.cuda = code, cuda
        name = {CSV_E_INVAL: "CSV_E_INVAL", CSV_E_NOMEM: "CSV_E_NOMEM", CSV_E_CUDA: "CSV_E_CUDA"}.get(code, str(code))
        super().__init__("%s -> %s%s" % (fn, name, " (cudaError %d)" % cuda if code == CSV_E_CUDA else ""))


_lib = None


def lib():
    """The loaded library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libconserve_kv.so is not built: run `python -m paper_2606_01839_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_size_t
        pi32, pvp = ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_void_p)
        pdesc, pshape, pd = ctypes.POINTER(KvPoolDesc), ctypes.POINTER(AttnShape), ctypes.POINTER(ctypes.c_double)
        sig = {
            "csv_last_cuda_error": (ctypes.c_int, []),
            "csv_version": (ctypes.c_char_p, []),
            "kv_pool_bytes": (sz, [pdesc]),
            "kv_pool_create": (ctypes.c_int, [pdesc, vp, sz, pvp]),
            "kv_pool_destroy": (ctypes.c_int, [vp]),
            "kv_pool_set_free_order": (ctypes.c_int, [vp, pi32, i32]),
            "kv_alloc_blocks": (ctypes.c_int, [vp, i32, pi32]),
            "kv_free_blocks": (ctypes.c_int, [vp, pi32, i32]),
            "kv_pool_used_blocks": (i32, [vp]),
            "kv_pool_num_blocks": (i32, [vp]),
            "kv_pool_free_blocks": (i32, [vp]),
            "kv_pool_get_desc": (ctypes.c_int, [vp, pdesc]),
            "csv_place": (ctypes.c_int, [pvp, i32, i32, pi32]),
            "csv_provision": (ctypes.c_int, [ctypes.c_double] * 6 + [pd, pd, pd, pi32]),
            "kv_staging_bytes": (sz, [pdesc, i32, i32]),
            "kv_pack": (ctypes.c_int, [pdesc, vp, vp, i32, i32, vp, vp]),
            "kv_unpack": (ctypes.c_int, [vp, vp, i32, i32, vp, i32, vp]),
            "kv_pack_batch": (ctypes.c_int, [pdesc, i32, pvp, pvp, pi32, pi32, pvp, vp]),
            "kv_unpack_batch": (ctypes.c_int, [vp, i32, pvp, pi32, pi32, pvp, pi32, vp]),
            "kv_append_tokens": (ctypes.c_int, [vp, vp, vp, vp, vp, i32, vp]),
            "kv_handoff_direct": (ctypes.c_int, [vp, vp, vp, i32, i32, vp, i32, vp]),
            "kv_handoff_direct_batch": (ctypes.c_int, [vp, i32, pvp, pvp, pi32, pi32, pvp, pi32, vp]),
            "csv_ipc_export": (ctypes.c_int, [vp, vp, ctypes.POINTER(ctypes.c_uint64)]),
            "csv_ipc_open": (ctypes.c_int, [vp, ctypes.c_uint64, pvp]),
            "csv_ipc_close": (ctypes.c_int, [vp]),
            "csv_ipc_mapped_bytes": (ctypes.c_int, [vp, ctypes.POINTER(sz)]),
            "csv_ipc_copy": (ctypes.c_int, [vp, vp, sz, vp]),
            "csv_tuning_set": (ctypes.c_int, [i32, i32]),
            "csv_tuning_get": (i32, [i32]),
            "csv_plan_workspace_bytes": (sz, [pshape, pi32, pi32, i32, i32]),
            "csv_plan_create": (ctypes.c_int, [pshape, pi32, pi32, i32, i32, vp, sz, vp, pvp]),
            "csv_plan_destroy": (ctypes.c_int, [vp]),
            "csv_plan_info": (ctypes.c_int, [vp, pi32, pi32, pi32, pi32, pi32]),
            "csv_plan_tail_split": (ctypes.c_int, [vp, pi32, pi32]),
            "csv_plan_decode_workers": (i32, [vp]),
            "csv_plan_total_q": (i32, [vp]),
            "csv_plan_decode_items": (i32, [vp, pi32, i32, pi32, i32]),
            "csv_plan_append_items": (i32, [vp, pi32, i32]),
            "paged_decode_attn": (ctypes.c_int, [vp, vp, i32, vp, vp, i32, vp, vp, vp]),
            "paged_decode_attn_static": (ctypes.c_int, [vp, i32, pshape, i32, pi32, i32, vp, vp, i32, vp, vp, vp]),
            "append_prefill_attn": (ctypes.c_int, [vp, vp, i32, vp, vp, i32, vp, vp, vp]),
            "paged_decode_step": (ctypes.c_int, [vp, vp, i32, vp, vp, vp, vp, i32, vp, vp, vp]),
            "csv_tail_step": (ctypes.c_int, [vp, vp, i32, vp, vp, vp, vp, i32, vp, vp, vp]),
            "csv_tail_step_host_workspace_bytes": (sz, [pshape, pi32, pi32, i32, i32, i32, i32]),
            "csv_tail_step_host": (ctypes.c_int, [vp, i32, i32, pshape, i32, pi32, pi32, vp, vp, vp, pi32, i32, i32, vp, sz,
                                                  vp, vp, vp]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(fn, rc):
    if rc != CSV_OK:
        raise CsvError(fn, rc, lib().csv_last_cuda_error() if rc == CSV_E_CUDA else 0)


def _i32(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def _ptr(t):
    """Device (or pinned host) pointer of a torch tensor / raw int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return ctypes.c_void_p(t)
    return ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch

        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return ctypes.c_void_p(stream)
    return ctypes.c_void_p(stream.cuda_stream)


def csv_version():
    return lib().csv_version().decode()


def pool_desc(num_layers, num_blocks, num_kv_heads, head_dim, block_size=BLOCK, dtype=0):
    return KvPoolDesc(num_layers, num_blocks, block_size, num_kv_heads, head_dim, dtype)


def attn_shape(num_q_heads, num_kv_heads, head_dim, block_size=BLOCK):
    return AttnShape(num_q_heads, num_kv_heads, head_dim, block_size)


def kv_pool_bytes(desc):
    return int(lib().kv_pool_bytes(ctypes.byref(desc)))


def kv_staging_bytes(desc, tokens, token_offset=0):
    return int(lib().kv_staging_bytes(ctypes.byref(desc), tokens, token_offset))


class KvPool:
    """kv_pool_t handle over caller memory (a torch uint8/bf16 CUDA tensor, or a raw pointer)."""

    def __init__(self, desc, base, nbytes=None):
        self.desc = desc
        self._keep = base
        if nbytes is None:
            nbytes = base.numel() * base.element_size()
        h = ctypes.c_void_p()
        _check("kv_pool_create", lib().kv_pool_create(ctypes.byref(desc), _ptr(base), nbytes, ctypes.byref(h)))
        self.handle = h

    def destroy(self):
        if self.handle:
            lib().kv_pool_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_free_order(self, order):
        a, p = _i32(order)
        _check("kv_pool_set_free_order", lib().kv_pool_set_free_order(self.handle, p, len(a)))

    def alloc_blocks(self, n):
        out = np.zeros(max(n, 1), dtype=np.int32)
        _check("kv_alloc_blocks", lib().kv_alloc_blocks(self.handle, n, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))))
        return out[:n].copy()

    def free_blocks(self, ids):
        a, p = _i32(ids)
        _check("kv_free_blocks", lib().kv_free_blocks(self.handle, p, len(a)))

    @property
    def used_blocks(self):
        return int(lib().kv_pool_used_blocks(self.handle))

    @property
    def num_blocks(self):
        return int(lib().kv_pool_num_blocks(self.handle))

    @property
    def free_count(self):
        return int(lib().kv_pool_free_blocks(self.handle))

    def get_desc(self):
        d = KvPoolDesc()
        _check("kv_pool_get_desc", lib().kv_pool_get_desc(self.handle, ctypes.byref(d)))
        return d


kv_pool_create = KvPool


def kv_alloc_blocks(pool, n):
    return pool.alloc_blocks(n)


def kv_free_blocks(pool, ids):
    return pool.free_blocks(ids)


def csv_place(pools, need_blocks):
    """index of the decoder pool with the lowest active KV occupancy that fits."""
    arr = (ctypes.c_void_p * len(pools))(*[p.handle for p in pools])
    out = ctypes.c_int32(-1)
    _check("csv_place", lib().csv_place(arr, len(pools), need_blocks, ctypes.byref(out)))
    return out.value


def csv_provision(T_p, L_in, T_d, L_d, B, W):
    r, a, b, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_double(), ctypes.c_int32()
    _check("csv_provision", lib().csv_provision(T_p, L_in, T_d, L_d, B, W, ctypes.byref(r), ctypes.byref(a),
                                                ctypes.byref(b), ctypes.byref(n)))
    return r.value, a.value, b.value, n.value


def kv_pack(desc, d_k, d_v, tokens, token_offset, d_staging, stream=None):
    _check("kv_pack", lib().kv_pack(ctypes.byref(desc), _ptr(d_k), _ptr(d_v), tokens, token_offset, _ptr(d_staging),
                                    _stream(stream)))


def kv_unpack(pool, d_staging, tokens, token_offset, d_block_ids, n_ids, stream=None):
    _check("kv_unpack", lib().kv_unpack(pool.handle, _ptr(d_staging), tokens, token_offset, _ptr(d_block_ids), n_ids,
                                        _stream(stream)))


def _vparr(ts):
    return (ctypes.c_void_p * len(ts))(*[(t if isinstance(t, int) else (0 if t is None else t.data_ptr())) for t in ts])


def kv_pack_batch(desc, d_ks, d_vs, tokens, token_offsets, d_stagings, stream=None):
    n = len(d_ks)
    _, pt = _i32(tokens)
    _, po = _i32(token_offsets)
    _check("kv_pack_batch", lib().kv_pack_batch(ctypes.byref(desc), n, _vparr(d_ks), _vparr(d_vs), pt, po,
                                                _vparr(d_stagings), _stream(stream)))


def kv_unpack_batch(pool, d_stagings, tokens, token_offsets, d_block_ids, n_ids, stream=None):
    n = len(d_stagings)
    _, pt = _i32(tokens)
    _, po = _i32(token_offsets)
    _, pn = _i32(n_ids)
    _check("kv_unpack_batch", lib().kv_unpack_batch(pool.handle, n, _vparr(d_stagings), pt, po, _vparr(d_block_ids), pn,
                                                    _stream(stream)))


def kv_handoff_direct(pool, d_k, d_v, tokens, token_offset, d_block_ids, n_ids, stream=None):
    _check("kv_handoff_direct", lib().kv_handoff_direct(pool.handle, _ptr(d_k), _ptr(d_v), tokens, token_offset,
                                                        _ptr(d_block_ids), n_ids, _stream(stream)))


def kv_handoff_direct_batch(pool, d_ks, d_vs, tokens, token_offsets, d_block_ids, n_ids, stream=None):
    n = len(d_ks)
    _, pt = _i32(tokens)
    _, po = _i32(token_offsets)
    _, pn = _i32(n_ids)
    _check("kv_handoff_direct_batch", lib().kv_handoff_direct_batch(pool.handle, n, _vparr(d_ks), _vparr(d_vs), pt, po,
                                                                    _vparr(d_block_ids), pn, _stream(stream)))


def csv_ipc_export(t):
    """(handle bytes, offset) of the cudaMalloc allocation holding tensor / pointer t: plain host data for any channel."""
    h = ctypes.create_string_buffer(IPC_HANDLE_BYTES)
    off = ctypes.c_uint64()
    _check("csv_ipc_export", lib().csv_ipc_export(_ptr(t), h, ctypes.byref(off)))
    return bytes(h.raw), int(off.value)


def csv_ipc_open(handle, offset):
    """Maps another process's allocation; returns the device pointer (int) of base + offset."""
    out = ctypes.c_void_p()
    _check("csv_ipc_open", lib().csv_ipc_open(ctypes.c_char_p(handle), offset, ctypes.byref(out)))
    return int(out.value)


def csv_ipc_mapped_bytes(ptr):
    """Bytes of the mapped allocation at and after a pointer csv_ipc_open returned."""
    out = ctypes.c_size_t()
    _check("csv_ipc_mapped_bytes", lib().csv_ipc_mapped_bytes(ctypes.c_void_p(ptr), ctypes.byref(out)))
    return int(out.value)


def csv_ipc_close(ptr):
    _check("csv_ipc_close", lib().csv_ipc_close(ctypes.c_void_p(ptr)))


def csv_ipc_copy(dst, src, nbytes, stream=None):
    """Copy-engine transfer between device buffers (torch tensors or raw pointers, e.g. a csv_ipc_open mapping)."""
    _check("csv_ipc_copy", lib().csv_ipc_copy(_ptr(dst), _ptr(src), int(nbytes), _stream(stream)))


TUNE_DECODE_GRID, TUNE_TAIL_DECODE_CTAS, TUNE_TAIL_TWO_KERNELS, TUNE_SM_DECODE_GBS, TUNE_SM_APPEND_GFLOPS = 0, 1, 2, 3, 4


def csv_tuning_set(knob, value):
    """Process-wide tuning override (0 = default); read when a plan is built and recorded in it (conserve_kv.h)."""
    _check("csv_tuning_set", lib().csv_tuning_set(knob, value))


def csv_tuning_get(knob):
    return int(lib().csv_tuning_get(knob))


def csv_plan_workspace_bytes(shape, q_lens, kv_lens, max_partition_tokens=0):
    q, pq = _i32(q_lens)
    _, pk = _i32(kv_lens)
    return int(lib().csv_plan_workspace_bytes(ctypes.byref(shape), pq, pk, len(q), max_partition_tokens))


class Plan:
    """csv_plan_t handle.  workspace: a torch CUDA uint8 tensor (>= csv_plan_workspace_bytes), or None (host-only)."""

    def __init__(self, shape, q_lens, kv_lens, max_partition_tokens=0, workspace=None, stream=None):
        q, pq = _i32(q_lens)
        _, pk = _i32(kv_lens)
        self.shape, self._keep = shape, workspace
        h = ctypes.c_void_p()
        if workspace is None:
            rc = lib().csv_plan_create(ctypes.byref(shape), pq, pk, len(q), max_partition_tokens, None, 0, None,
                                       ctypes.byref(h))
        else:
            rc = lib().csv_plan_create(ctypes.byref(shape), pq, pk, len(q), max_partition_tokens, _ptr(workspace),
                                       workspace.numel() * workspace.element_size(), _stream(stream), ctypes.byref(h))
        _check("csv_plan_create", rc)
        self.handle = h

    def destroy(self):
        if self.handle:
            lib().csv_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def info(self):
        v = [ctypes.c_int32() for _ in range(5)]
        _check("csv_plan_info", lib().csv_plan_info(self.handle, *[ctypes.byref(x) for x in v]))
        keys = ["n_decode_items", "n_decode_rows", "n_append_chunks", "n_append_rows", "decode_grid"]
        out = dict(zip(keys, [x.value for x in v]))
        a, b = ctypes.c_int32(), ctypes.c_int32()
        _check("csv_plan_tail_split", lib().csv_plan_tail_split(self.handle, ctypes.byref(a), ctypes.byref(b)))
        out.update(tail_n_dec=a.value, tail_n_shares=b.value, decode_workers=int(lib().csv_plan_decode_workers(self.handle)))
        return out

    @property
    def total_q(self):
        return int(lib().csv_plan_total_q(self.handle))

    def decode_items(self):
        inf = self.info()
        n, W = inf["n_decode_items"], inf["decode_workers"]
        items = np.zeros((max(n, 1), 8), dtype=np.int32)
        wb = np.zeros(W + 1, dtype=np.int32)
        lib().csv_plan_decode_items(self.handle, items.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), n,
                                    wb.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), W + 1)
        return items[:n], wb

    def append_items(self):
        n = int(lib().csv_plan_append_items(self.handle, None, 0))
        items = np.zeros((max(n, 1), 12), dtype=np.int32)
        lib().csv_plan_append_items(self.handle, items.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), n)
        return items[:n]


csv_plan_create = Plan


def paged_decode_attn(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse, stream=None):
    _check("paged_decode_attn", lib().paged_decode_attn(plan.handle, pool.handle, layer, _ptr(d_q), _ptr(d_block_tables),
                                                        max_blocks, _ptr(d_out), _ptr(d_lse), _stream(stream)))


STATIC_SCRATCH_BYTES = 8 << 20   # CSV_STATIC_SCRATCH_BYTES of conserve_kv.h


def paged_decode_attn_static(pool, layer, shape, kv_lens, d_q, d_block_tables, max_blocks, d_out, d_lse,
                             max_partition_tokens=0, stream=None):
    """paged_decode_attn without a Plan or a workspace tensor, for callers that may not allocate device memory (all HBM
    already belongs to the KV pool, or the surrounding engine forbids cudaMalloc inside a step).  One decode row per entry
    of kv_lens.  The scratch is a fixed 8 MiB array inside the library, one per GPU, shared by every call: keep calls on
    one stream.  A step that needs more raises CsvError(CSV_E_NOMEM); make the first call on a device before any stream
    capture (it looks the array's address up).  See conserve_kv.h."""
    k, pk = _i32(kv_lens)
    rc = lib().paged_decode_attn_static(pool.handle, layer, ctypes.byref(shape), len(k), pk, max_partition_tokens, _ptr(d_q),
                                        _ptr(d_block_tables), max_blocks, _ptr(d_out), _ptr(d_lse), _stream(stream))
    if rc == CSV_E_NOMEM:
        err = CsvError("paged_decode_attn_static", rc)
        err.args = ("%s: this step's plan needs more than the library's fixed %d-byte scratch array; use paged_decode_attn "
                    "with a caller-owned workspace" % (err.args[0], STATIC_SCRATCH_BYTES),)
        raise err
    _check("paged_decode_attn_static", rc)


def paged_decode_step(plan, pool, layer, d_q, d_k_new, d_v_new, d_block_tables, max_blocks, d_out, d_lse, stream=None):
    _check("paged_decode_step", lib().paged_decode_step(plan.handle, pool.handle, layer, _ptr(d_q), _ptr(d_k_new),
                                                        _ptr(d_v_new), _ptr(d_block_tables), max_blocks, _ptr(d_out),
                                                        _ptr(d_lse), _stream(stream)))


def csv_tail_step(plan, pool, layer, d_q, d_k_new, d_v_new, d_block_tables, max_blocks, d_out, d_lse, stream=None):
    _check("csv_tail_step", lib().csv_tail_step(plan.handle, pool.handle, layer, _ptr(d_q), _ptr(d_k_new), _ptr(d_v_new),
                                                _ptr(d_block_tables), max_blocks, _ptr(d_out), _ptr(d_lse), _stream(stream)))


def append_prefill_attn(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse, stream=None):
    _check("append_prefill_attn", lib().append_prefill_attn(plan.handle, pool.handle, layer, _ptr(d_q),
                                                            _ptr(d_block_tables), max_blocks, _ptr(d_out), _ptr(d_lse),
                                                            _stream(stream)))


def kv_append_tokens(pool, plan, d_k_new, d_v_new, d_block_tables, max_blocks, stream=None):
    _check("kv_append_tokens", lib().kv_append_tokens(pool.handle, plan.handle, _ptr(d_k_new), _ptr(d_v_new),
                                                      _ptr(d_block_tables), max_blocks, _stream(stream)))


def csv_tail_step_host_workspace_bytes(shape, kv_lens, max_blocks, max_partition_tokens=0, q_lens=None, n_layers=1):
    k, pk = _i32(kv_lens)
    pq = _i32(q_lens)[1] if q_lens is not None else None
    return int(lib().csv_tail_step_host_workspace_bytes(ctypes.byref(shape), pq, pk, len(k), max_blocks, n_layers,
                                                        max_partition_tokens))


def csv_tail_step_host(pool, layer, shape, kv_lens, h_q, h_k_new, h_v_new, h_block_tables, max_blocks, workspace, h_out,
                       h_lse, max_partition_tokens=0, stream=None, q_lens=None, n_layers=1):
    """One tail step (decode rows + appended chunks, layers [layer, layer + n_layers)) with HOST (pinned torch) buffers;
    synchronises the stream before returning."""
    k, pk = _i32(kv_lens)
    q = _i32(q_lens) if q_lens is not None else None
    _check("csv_tail_step_host", lib().csv_tail_step_host(
        pool.handle, layer, n_layers, ctypes.byref(shape), len(k), q[1] if q else None, pk, _ptr(h_q), _ptr(h_k_new),
        _ptr(h_v_new), ctypes.cast(_ptr(h_block_tables), ctypes.POINTER(ctypes.c_int32)), max_blocks, max_partition_tokens,
        _ptr(workspace), workspace.numel() * workspace.element_size(), _ptr(h_out), _ptr(h_lse), _stream(stream)))

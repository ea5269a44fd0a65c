"""ctypes front end of oracle/oracle.c (TEST INFRASTRUCTURE, see that file).

Argument marshalling only: every number the oracle produces is computed in
oracle.c.  bf16 tensors travel as numpy uint16 bit patterns.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force=False):
    """Compile oracle.c with gcc into oracle/liboracle.so (if stale)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c_u16p = ctypes.POINTER(ctypes.c_uint16)
        c_i32p = ctypes.POINTER(ctypes.c_int32)
        c_f64p = ctypes.POINTER(ctypes.c_double)
        i = ctypes.c_int
        lib.orc_attention.argtypes = [c_u16p, c_u16p, c_u16p, i, i, i, i, i, c_f64p, c_f64p]
        lib.orc_attention.restype = i
        lib.orc_pool_addr.argtypes = [i] * 9
        lib.orc_pool_addr.restype = ctypes.c_size_t
        lib.orc_pool_elems.argtypes = [i] * 4
        lib.orc_pool_elems.restype = ctypes.c_size_t
        lib.orc_gather.argtypes = [c_u16p, i, i, i, i, c_i32p, i, c_u16p, c_u16p]
        lib.orc_gather.restype = i
        lib.orc_scatter.argtypes = [c_u16p, i, i, i, i, c_u16p, c_u16p, i, i, c_i32p, i]
        lib.orc_scatter.restype = i
        lib.orc_staging_elems.argtypes = [i] * 5
        lib.orc_staging_elems.restype = ctypes.c_size_t
        lib.orc_staging_message.argtypes = [i, i, i, c_u16p, c_u16p, i, i, c_u16p]
        lib.orc_staging_message.restype = i
        lib.orc_merge.argtypes = [c_f64p, ctypes.c_double, c_f64p, ctypes.c_double, i, c_f64p, c_f64p]
        lib.orc_merge.restype = None
        dbl = ctypes.c_double
        lib.orc_provision.argtypes = [dbl] * 6 + [c_f64p, c_f64p, c_f64p, ctypes.POINTER(i)]
        lib.orc_provision.restype = i
        lib.orc_place.argtypes = [ctypes.POINTER(i), ctypes.POINTER(i), i, i]
        lib.orc_place.restype = i
        _lib = lib
    return _lib


def _u16(a):
    a = np.ascontiguousarray(a)
    if a.dtype != np.uint16:
        raise TypeError("bf16 data must be passed as uint16 bit patterns, got %s" % a.dtype)
    return a


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


def attention(q, K, V):
    """O1. q [R,Hq,d], K,V [L,Hkv,d] uint16 bf16 bits -> (O [R,Hq,d] f64, LSE [R,Hq] f64)."""
    q, K, V = _u16(q), _u16(K), _u16(V)
    R, Hq, d = q.shape
    L, Hkv, d2 = K.shape
    assert d2 == d and V.shape == K.shape
    O = np.zeros((R, Hq, d), dtype=np.float64)
    LSE = np.zeros((R, Hq), dtype=np.float64)
    rc = _load().orc_attention(_p(q, ctypes.c_uint16), _p(K, ctypes.c_uint16), _p(V, ctypes.c_uint16), R, L, Hq,
                               Hkv, d, _p(O, ctypes.c_double), _p(LSE, ctypes.c_double))
    if rc != 0:
        raise ValueError("orc_attention rejected its arguments")
    return O, LSE


def pool_addr(num_blocks, Hkv, d, layer, block, kv, head, slot, c):
    return int(_load().orc_pool_addr(num_blocks, Hkv, d, layer, block, kv, head, slot, c))


def pool_elems(NL, num_blocks, Hkv, d):
    return int(_load().orc_pool_elems(NL, num_blocks, Hkv, d))


def gather(pool, num_blocks, Hkv, d, layer, table, L):
    """O2. pool: flat uint16 image -> (K [L,Hkv,d], V [L,Hkv,d]) uint16."""
    pool = _u16(pool)
    table = np.ascontiguousarray(table, dtype=np.int32)
    K = np.zeros((L, Hkv, d), dtype=np.uint16)
    V = np.zeros((L, Hkv, d), dtype=np.uint16)
    rc = _load().orc_gather(_p(pool, ctypes.c_uint16), num_blocks, Hkv, d, layer, _p(table, ctypes.c_int32), L,
                            _p(K, ctypes.c_uint16), _p(V, ctypes.c_uint16))
    if rc != 0:
        raise ValueError("orc_gather: block id out of range")
    return K, V


def scatter(pool, NL, num_blocks, Hkv, d, k_src, v_src, tokens, off, table):
    """O3. Returns a NEW pool image = `pool` with the conversation's KV scattered in."""
    out = _u16(pool).copy()
    k_src, v_src = _u16(k_src), _u16(v_src)
    assert k_src.size == NL * tokens * Hkv * d and v_src.size == k_src.size
    table = np.ascontiguousarray(table, dtype=np.int32)
    rc = _load().orc_scatter(_p(out, ctypes.c_uint16), NL, num_blocks, Hkv, d, _p(k_src, ctypes.c_uint16),
                             _p(v_src, ctypes.c_uint16), tokens, off, _p(table, ctypes.c_int32), len(table))
    if rc != 0:
        raise ValueError("orc_scatter rejected its arguments")
    return out


def staging_elems(NL, Hkv, d, tokens, off):
    return int(_load().orc_staging_elems(NL, Hkv, d, tokens, off))


def staging_message(NL, Hkv, d, k_src, v_src, tokens, off):
    k_src, v_src = _u16(k_src), _u16(v_src)
    msg = np.zeros(staging_elems(NL, Hkv, d, tokens, off), dtype=np.uint16)
    rc = _load().orc_staging_message(NL, Hkv, d, _p(k_src, ctypes.c_uint16), _p(v_src, ctypes.c_uint16), tokens,
                                     off, _p(msg, ctypes.c_uint16))
    if rc != 0:
        raise ValueError("orc_staging_message rejected its arguments")
    return msg


def merge(Oa, lse_a, Ob, lse_b):
    """O4. Two normalised partials over disjoint key sets -> (O, LSE)."""
    Oa = np.ascontiguousarray(Oa, dtype=np.float64)
    Ob = np.ascontiguousarray(Ob, dtype=np.float64)
    O = np.zeros_like(Oa)
    lse = ctypes.c_double()
    _load().orc_merge(_p(Oa, ctypes.c_double), float(lse_a), _p(Ob, ctypes.c_double), float(lse_b), Oa.size,
                      _p(O, ctypes.c_double), ctypes.byref(lse))
    return O, lse.value


def provision(T_p, L_in, T_d, L_d, B, W):
    """PAPER.md:162-172. -> (R*, N_throughput, N_memory, N)."""
    r, a, b = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    n = ctypes.c_int()
    rc = _load().orc_provision(T_p, L_in, T_d, L_d, B, W, ctypes.byref(r), ctypes.byref(a), ctypes.byref(b),
                               ctypes.byref(n))
    if rc != 0:
        raise ValueError("orc_provision: inputs must be positive")
    return r.value, a.value, b.value, n.value


def place(used, total, need):
    """PAPER.md:178. -> index of the chosen decoder, or -1."""
    n = len(used)
    U = (ctypes.c_int * n)(*[int(x) for x in used])
    T = (ctypes.c_int * n)(*[int(x) for x in total])
    return int(_load().orc_place(U, T, n, int(need)))

"""ORACLE — TEST INFRASTRUCTURE ONLY (ctypes binding of oracle.c).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from the CUDA package
``paper_2606_00516_b200`` and the CUDA package imports nothing from here.

All array arguments are numpy; bf16 tensors are passed as ``uint16`` bit patterns.  Pool layout
(the boundary contract of include/pa.h): ``pool[block][kv_head][slot][d]`` per K and per V.
See oracle.c for the passages each function follows and tests/test_oracle_pins.py for its pins.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (no fast-math: fp64 IEEE semantics are the point)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fno-fast-math", "-ffp-contract=off",
                               "-o", tmp, _SRC, "-lm", "-lpthread"])
        os.replace(tmp, _LIB)
    return _LIB


class _Shape(C.Structure):
    _fields_ = [("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("block_size", C.c_int32), ("max_blocks_per_seq", C.c_int32)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        for name in ("oracle_kv_append", "oracle_kv_gather", "oracle_attention_rows", "oracle_attention_weights",
                     "oracle_attention_partial", "oracle_merge", "oracle_fit", "oracle_quadratic_kappa", "oracle_theta0",
                     "oracle_eq7"):
            getattr(_lib, name).restype = C.c_int32
    return _lib


def _p(a, ctype):
    return a.ctypes.data_as(C.POINTER(ctype))


def _u16(a):
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, a.dtype
    return a


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


@dataclass
class PagedShape:
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    block_size: int = 16

    def _c(self, max_blocks_per_seq: int) -> _Shape:
        return _Shape(self.num_q_heads, self.num_kv_heads, self.head_dim, self.block_size, int(max_blocks_per_seq))


def kv_append(shape: PagedShape, k_new, v_new, k_pool, v_pool, cu_seqlens_q, context_lens, block_tables) -> None:
    """In-place append into ``k_pool``/``v_pool`` (uint16 arrays of the documented layout)."""
    bt = _i32(block_tables)
    cu, cl = _i32(cu_seqlens_q), _i32(context_lens)
    assert k_pool.dtype == np.uint16 and k_pool.flags.c_contiguous and v_pool.flags.c_contiguous
    k_new, v_new = _u16(k_new), _u16(v_new)
    sh = shape._c(bt.shape[1])
    rc = _load().oracle_kv_append(C.byref(sh), _p(k_new, C.c_uint16), _p(v_new, C.c_uint16), _p(k_pool, C.c_uint16),
                                  _p(v_pool, C.c_uint16), _p(cu, C.c_int32), _p(cl, C.c_int32), _p(bt, C.c_int32),
                                  C.c_int32(len(cl)))
    assert rc == 0


def kv_gather(shape: PagedShape, k_pool, v_pool, block_tables, s: int, kv_len: int):
    bt = _i32(block_tables)
    sh = shape._c(bt.shape[1])
    k_out = np.empty((kv_len, shape.num_kv_heads, shape.head_dim), dtype=np.uint16)
    v_out = np.empty_like(k_out)
    k_pool, v_pool = _u16(k_pool), _u16(v_pool)
    rc = _load().oracle_kv_gather(C.byref(sh), _p(k_pool, C.c_uint16), _p(v_pool, C.c_uint16), _p(bt, C.c_int32),
                                  C.c_int32(s), C.c_int32(kv_len), _p(k_out, C.c_uint16), _p(v_out, C.c_uint16))
    assert rc == 0
    return k_out, v_out


def attention(shape: PagedShape, q, k_pool, v_pool, cu_seqlens_q, context_lens, block_tables, scale: float,
              rows=None, n_threads: int = 1, return_lse: bool = False):
    """fp64 attention output ``[len(rows), Hq, D]`` for the listed token rows (default: all)."""
    bt = _i32(block_tables)
    cu, cl = _i32(cu_seqlens_q), _i32(context_lens)
    q, k_pool, v_pool = _u16(q), _u16(k_pool), _u16(v_pool)
    n_tok = int(cu[-1])
    rows = np.arange(n_tok, dtype=np.int64) if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    out = np.zeros((len(rows), shape.num_q_heads, shape.head_dim), dtype=np.float64)
    lse = np.zeros((len(rows), shape.num_q_heads), dtype=np.float64)
    sh = shape._c(bt.shape[1])
    rc = _load().oracle_attention_rows(C.byref(sh), _p(q, C.c_uint16), _p(k_pool, C.c_uint16), _p(v_pool, C.c_uint16),
                                       _p(cu, C.c_int32), _p(cl, C.c_int32), _p(bt, C.c_int32), C.c_int32(len(cl)),
                                       C.c_double(scale), _p(rows, C.c_int64), C.c_int64(len(rows)),
                                       _p(out, C.c_double), _p(lse, C.c_double), C.c_int32(n_threads))
    assert rc >= 1, rc
    return (out, lse) if return_lse else out


def attention_weights(shape: PagedShape, q, k_pool, v_pool, cu_seqlens_q, context_lens, block_tables, scale: float,
                      row: int, h: int):
    """Softmax weights p_t (length n_j) and lse of one (token row, q head)."""
    bt = _i32(block_tables)
    cu, cl = _i32(cu_seqlens_q), _i32(context_lens)
    q, k_pool, v_pool = _u16(q), _u16(k_pool), _u16(v_pool)
    cap = int((cl.astype(np.int64) + np.diff(cu)).max())
    p = np.zeros(cap, dtype=np.float64)
    lse = C.c_double(0.0)
    sh = shape._c(bt.shape[1])
    n = _load().oracle_attention_weights(C.byref(sh), _p(q, C.c_uint16), _p(k_pool, C.c_uint16),
                                         _p(v_pool, C.c_uint16), _p(cu, C.c_int32), _p(cl, C.c_int32),
                                         _p(bt, C.c_int32), C.c_int32(len(cl)), C.c_double(scale), C.c_int64(row),
                                         C.c_int32(h), _p(p, C.c_double), C.c_int64(cap), C.byref(lse))
    assert n >= 1, n
    return p[:n].copy(), lse.value


def attention_partial(shape: PagedShape, q, k_pool, v_pool, cu_seqlens_q, context_lens, block_tables, scale: float,
                      row: int, h: int, key_lo: int, key_hi: int):
    """(m, l, unnormalised o[D]) of one (row, head) over keys [key_lo, key_hi)."""
    bt = _i32(block_tables)
    cu, cl = _i32(cu_seqlens_q), _i32(context_lens)
    q, k_pool, v_pool = _u16(q), _u16(k_pool), _u16(v_pool)
    m, l = C.c_double(0.0), C.c_double(0.0)
    o = np.zeros(shape.head_dim, dtype=np.float64)
    sh = shape._c(bt.shape[1])
    rc = _load().oracle_attention_partial(C.byref(sh), _p(q, C.c_uint16), _p(k_pool, C.c_uint16),
                                          _p(v_pool, C.c_uint16), _p(cu, C.c_int32), _p(cl, C.c_int32),
                                          _p(bt, C.c_int32), C.c_int32(len(cl)), C.c_double(scale), C.c_int64(row),
                                          C.c_int32(h), C.c_int64(key_lo), C.c_int64(key_hi), C.byref(m), C.byref(l),
                                          _p(o, C.c_double))
    assert rc == 0, rc
    return m.value, l.value, o


def merge(m_i, l_i, o_i):
    """Flash-decoding combine of partials → (o[D], lse)."""
    m_i = np.ascontiguousarray(m_i, dtype=np.float64)
    l_i = np.ascontiguousarray(l_i, dtype=np.float64)
    o_i = np.ascontiguousarray(o_i, dtype=np.float64)
    n, D = o_i.shape
    o = np.zeros(D, dtype=np.float64)
    lse = C.c_double(0.0)
    rc = _load().oracle_merge(C.c_int32(n), C.c_int32(D), _p(m_i, C.c_double), _p(l_i, C.c_double),
                              _p(o_i, C.c_double), _p(o, C.c_double), C.byref(lse))
    assert rc == 0
    return o, lse.value


def fit(n, T):
    """OLS T = α + β·n → (alpha, beta, r2); raises ValueError with < 2 distinct n."""
    n = np.ascontiguousarray(n, dtype=np.float64)
    T = np.ascontiguousarray(T, dtype=np.float64)
    a, b, r2 = C.c_double(), C.c_double(), C.c_double()
    rc = _load().oracle_fit(_p(n, C.c_double), _p(T, C.c_double), C.c_int32(len(n)), C.byref(a), C.byref(b),
                            C.byref(r2))
    if rc != 0:
        raise ValueError(f"oracle_fit: rc={rc}")
    return a.value, b.value, r2.value


def quadratic_kappa(r, K):
    """Quadratic LS fit K(r)=c0+c1 r+c2 r² and κ = 2c2/(c0+c1+c2) (Eq. 10–11)."""
    r = np.ascontiguousarray(r, dtype=np.float64)
    K = np.ascontiguousarray(K, dtype=np.float64)
    c = np.zeros(3, dtype=np.float64)
    kappa = C.c_double()
    rc = _load().oracle_quadratic_kappa(_p(r, C.c_double), _p(K, C.c_double), C.c_int32(len(r)), _p(c, C.c_double),
                                        C.byref(kappa))
    if rc != 0:
        raise ValueError(f"oracle_quadratic_kappa: rc={rc}")
    return c, kappa.value


def theta0(x: float):
    """Base CFR threshold θ0 and ζ = −ln(1−θ0) from θ0/(1−θ0) + ln(1−θ0) = x, x = p0·α_p/α_d (Eq. 3)."""
    th, ze = C.c_double(), C.c_double()
    rc = _load().oracle_theta0(C.c_double(x), C.byref(th), C.byref(ze))
    if rc != 0:
        raise ValueError(f"oracle_theta0: rc={rc}")
    return th.value, ze.value


def eq7(alpha_p, beta_p, alpha_d, beta_d, alpha_mb, beta_mb_e, mu_L, mu_O, zeta, k0, N):
    """Crossover condition (Eq. 7, Prop. 3.4) → dict(lhs, rhs, beta_eb_w, tp_eb, tp_mb)."""
    out = [C.c_double() for _ in range(5)]
    rc = _load().oracle_eq7(*[C.c_double(float(v)) for v in (alpha_p, beta_p, alpha_d, beta_d, alpha_mb, beta_mb_e,
                                                               mu_L, mu_O, zeta, k0, N)], *[C.byref(o) for o in out])
    if rc != 0:
        raise ValueError(f"oracle_eq7: rc={rc}")
    return dict(zip(("lhs", "rhs", "beta_eb_w", "tp_eb", "tp_mb"), (o.value for o in out)))

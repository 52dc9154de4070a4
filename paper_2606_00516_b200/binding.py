"""Thin ctypes binding of libpa_b200.so — same names as include/pa.h, argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; PyTorch only supplies device memory
(``tensor.data_ptr()``) and streams.  There is NO CPU fallback: if the library is missing or no sm_100
device is usable, calls raise ``PaError``.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpa_b200.so")

PA_OK = 0
PA_ERR_INVALID, PA_ERR_UNSUPPORTED, PA_ERR_WORKSPACE, PA_ERR_CUDA, PA_ERR_TIMER = -1, -2, -3, -4, -5
PA_FLAG_DEBUG_SIMPLE = 1
PA_FLAG_PREFILL_P_SMEM = 2

EXPORTS = ["pa_create", "pa_destroy", "pa_workspace_bytes", "pa_kv_pool_bytes", "pa_kv_append", "pa_plan",
           "pa_batch_attention", "pa_kv_gather", "pa_timer_begin", "pa_timer_end", "pa_timer_record",
           "pa_timer_fit", "pa_timer_kappa", "pa_timer_reset", "pa_crossover_theta0", "pa_crossover_eq7", "pa_plan_info",
           "pa_last_error", "pa_decode_attention_static", "pa_static_scratch_bytes", "pa_static_last_error"]


class PaError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"pa error {code}: {msg}")
        self.code = code


class PaConfig(C.Structure):
    _fields_ = [("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("block_size", C.c_int32), ("num_blocks", C.c_int64), ("max_seqs", C.c_int32),
                ("max_tokens", C.c_int32), ("max_blocks_per_seq", C.c_int32), ("device", C.c_int32),
                ("flags", C.c_uint32), ("tune_prefill_ctas", C.c_int32), ("tune_bundles_per_stream", C.c_int32),
                ("tune_min_bundle_blocks", C.c_int32), ("tune_levels", C.c_int32)]


_lib = None


def load_library() -> C.CDLL:
    """Load libpa_b200.so (built by ``python -m paper_2606_00516_b200.build``); raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PaError(PA_ERR_CUDA, f"{LIB_PATH} not built — run `python -m paper_2606_00516_b200.build`; "
                                       "there is no fallback path")
        lib = C.CDLL(LIB_PATH)
        vp, i32, i64, f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        lib.pa_create.argtypes = [C.POINTER(vp), C.POINTER(PaConfig)]
        lib.pa_destroy.argtypes = [vp]
        lib.pa_workspace_bytes.argtypes = [vp]
        lib.pa_workspace_bytes.restype = i64
        lib.pa_kv_pool_bytes.argtypes = [vp]
        lib.pa_kv_pool_bytes.restype = i64
        lib.pa_kv_append.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, vp]
        lib.pa_plan.argtypes = [vp, vp, vp, i32, i32, vp, i64, vp]
        lib.pa_batch_attention.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_float, vp, vp]
        lib.pa_kv_gather.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
        lib.pa_timer_begin.argtypes = [vp, vp]
        lib.pa_timer_end.argtypes = [vp, vp, f64, i32, C.POINTER(f64)]
        lib.pa_timer_record.argtypes = [vp, f64, i32, f64]
        lib.pa_timer_fit.argtypes = [vp, f64, C.POINTER(f64), C.POINTER(f64), C.POINTER(f64), C.POINTER(i32)]
        lib.pa_timer_kappa.argtypes = [vp, i32, C.POINTER(f64), C.POINTER(f64), C.POINTER(i32)]
        lib.pa_timer_reset.argtypes = [vp]
        lib.pa_crossover_theta0.argtypes = [f64, C.POINTER(f64), C.POINTER(f64)]
        lib.pa_crossover_eq7.argtypes = [C.POINTER(f64), C.POINTER(f64)]
        lib.pa_plan_info.argtypes = [vp, i32]
        lib.pa_plan_info.restype = i64
        lib.pa_last_error.argtypes = [vp]
        lib.pa_last_error.restype = C.c_char_p
        lib.pa_decode_attention_static.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, C.c_float, vp, i32, vp]
        lib.pa_static_scratch_bytes.argtypes = []
        lib.pa_static_scratch_bytes.restype = i64
        lib.pa_static_last_error.argtypes = []
        lib.pa_static_last_error.restype = C.c_char_p
        for n in EXPORTS:
            if n not in ("pa_workspace_bytes", "pa_kv_pool_bytes", "pa_plan_info", "pa_last_error",
                         "pa_static_scratch_bytes", "pa_static_last_error"):
                getattr(lib, n).restype = i32
        _lib = lib
    return _lib


def _ptr(t) -> int:
    return 0 if t is None else t.data_ptr()


def _host_i32(a) -> int:
    """Address of a HOST int32 array (kept alive by the caller for the duration of the call)."""
    import numpy as np
    if isinstance(a, np.ndarray) and a.dtype == np.int32 and a.flags.c_contiguous:
        return a.ctypes.data
    t = torch.as_tensor(a, dtype=torch.int32).contiguous()
    assert t.device.type == "cpu"
    _host_i32.keep = t          # survives until the next conversion, i.e. past the C call that uses the address
    return t.data_ptr()


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream


def decode_attention_static(q, k_pool, v_pool, context_lens, block_tables, max_kv_len: int, softmax_scale: float, out,
                            stream=None):
    """pa_decode_attention_static: decode attention with the scratch in the library's static device array (no context,
    no workspace, no allocation).  q/out [n_seq, Hq, D] bf16; pools [num_blocks, Hkv, 16, D]; block_tables
    [n_seq, max_blocks_per_seq] int32; all on the current CUDA device."""
    lib = load_library()
    n_seq, hq, d = q.shape
    rc = lib.pa_decode_attention_static(_ptr(q), _ptr(k_pool), _ptr(v_pool), _ptr(context_lens), _ptr(block_tables),
                                        n_seq, hq, k_pool.shape[1], d, block_tables.shape[1], max_kv_len,
                                        C.c_float(softmax_scale), _ptr(out), q.device.index, _stream(stream))
    if rc != PA_OK:
        raise PaError(rc, lib.pa_static_last_error().decode())


def static_scratch_bytes() -> int:
    return int(load_library().pa_static_scratch_bytes())


class PagedAttention:
    """One context per shape.  Methods mirror the C entry points one to one."""

    def __init__(self, num_q_heads: int, num_kv_heads: int, head_dim: int, num_blocks: int, max_seqs: int,
                 max_tokens: int, max_blocks_per_seq: int, block_size: int = 16, device: int = 0, flags: int = 0,
                 tune_prefill_ctas: int = 0, tune_bundles_per_stream: int = 0, tune_min_bundle_blocks: int = 0,
                 tune_levels: int = 0):
        self.lib = load_library()
        self.cfg = PaConfig(num_q_heads, num_kv_heads, head_dim, block_size, num_blocks, max_seqs, max_tokens,
                            max_blocks_per_seq, device, flags, tune_prefill_ctas, tune_bundles_per_stream,
                            tune_min_bundle_blocks, tune_levels)
        self.ctx = C.c_void_p()
        rc = self.lib.pa_create(C.byref(self.ctx), C.byref(self.cfg))
        if rc != PA_OK:
            raise PaError(rc, "pa_create failed (unsupported shape, invalid size, or no usable sm_100 device)")
        self.device = torch.device("cuda", device)
        self.workspace = torch.empty(self.workspace_bytes(), dtype=torch.uint8, device=self.device)

    def close(self):
        if getattr(self, "ctx", None) and self.ctx.value:
            self.lib.pa_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != PA_OK:
            raise PaError(rc, self.last_error())

    def last_error(self) -> str:
        return self.lib.pa_last_error(self.ctx).decode()

    def workspace_bytes(self) -> int:
        return int(self.lib.pa_workspace_bytes(self.ctx))

    def kv_pool_bytes(self) -> int:
        return int(self.lib.pa_kv_pool_bytes(self.ctx))

    def pool_shape(self):
        c = self.cfg
        return (c.num_blocks, c.num_kv_heads, c.block_size, c.head_dim)

    def kv_append(self, k_new, v_new, k_pool, v_pool, cu_seqlens_q, context_lens, block_tables, n_seq: int,
                  n_tok: int, stream=None):
        self._check(self.lib.pa_kv_append(self.ctx, _ptr(k_new), _ptr(v_new), _ptr(k_pool), _ptr(v_pool),
                                          _ptr(cu_seqlens_q), _ptr(context_lens), _ptr(block_tables), n_seq, n_tok,
                                          _stream(stream)))

    def plan(self, h_cu_seqlens_q, h_context_lens, n_seq: int, num_decode_seqs: int, stream=None):
        """h_* are HOST int32 arrays: contiguous numpy int32 (passed as they are) or anything torch.as_tensor takes."""
        self._check(self.lib.pa_plan(self.ctx, _host_i32(h_cu_seqlens_q), _host_i32(h_context_lens), n_seq,
                                     num_decode_seqs, self.workspace.data_ptr(), self.workspace.numel(),
                                     _stream(stream)))

    def batch_attention(self, q, k_pool, v_pool, cu_seqlens_q, context_lens, block_tables, softmax_scale: float, out,
                        stream=None):
        self._check(self.lib.pa_batch_attention(self.ctx, _ptr(q), _ptr(k_pool), _ptr(v_pool), _ptr(cu_seqlens_q),
                                                _ptr(context_lens), _ptr(block_tables), C.c_float(softmax_scale),
                                                _ptr(out), _stream(stream)))

    def kv_gather(self, k_pool, v_pool, block_table_row, kv_len: int, k_out, v_out, stream=None):
        self._check(self.lib.pa_kv_gather(self.ctx, _ptr(k_pool), _ptr(v_pool), _ptr(block_table_row), kv_len,
                                          _ptr(k_out), _ptr(v_out), _stream(stream)))

    def timer_begin(self, stream=None):
        self._check(self.lib.pa_timer_begin(self.ctx, _stream(stream)))

    def timer_end(self, r: float, n_tok: int, stream=None) -> float:
        sec = C.c_double()
        self._check(self.lib.pa_timer_end(self.ctx, _stream(stream), r, n_tok, C.byref(sec)))
        return sec.value

    def timer_record(self, r: float, n_tok: int, seconds: float):
        self._check(self.lib.pa_timer_record(self.ctx, r, n_tok, seconds))

    def timer_fit(self, r: float):
        a, b, r2, n = C.c_double(), C.c_double(), C.c_double(), C.c_int32()
        self._check(self.lib.pa_timer_fit(self.ctx, r, C.byref(a), C.byref(b), C.byref(r2), C.byref(n)))
        return a.value, b.value, r2.value, n.value

    def timer_kappa(self, n_tok: int):
        """(c0, c1, c2), kappa, n_points of K(r) = c0 + c1 r + c2 r^2 at this n_tok (App. A.3, Eq. 9-11)."""
        c, k, n = (C.c_double * 3)(), C.c_double(), C.c_int32()
        self._check(self.lib.pa_timer_kappa(self.ctx, n_tok, c, C.byref(k), C.byref(n)))
        return (c[0], c[1], c[2]), k.value, n.value

    def crossover_theta0(self, x: float):
        """(theta0, zeta) of PAPER.md Eq. 3 for x = p0·alpha_p/alpha_d."""
        th, ze = C.c_double(), C.c_double()
        rc = self.lib.pa_crossover_theta0(x, C.byref(th), C.byref(ze))
        if rc != PA_OK:
            raise PaError(rc, "pa_crossover_theta0: x must be positive and finite")
        return th.value, ze.value

    def crossover_eq7(self, alpha_p, beta_p, alpha_d, beta_d, alpha_mb, beta_mb_e, mu_L, mu_O, zeta, k0, N):
        """PAPER.md Eq. 7 → dict(lhs, rhs, beta_eb_w, tp_eb, tp_mb); mixed batching wins iff lhs < rhs."""
        a = (C.c_double * 11)(alpha_p, beta_p, alpha_d, beta_d, alpha_mb, beta_mb_e, mu_L, mu_O, zeta, k0, N)
        o = (C.c_double * 5)()
        rc = self.lib.pa_crossover_eq7(a, o)
        if rc != PA_OK:
            raise PaError(rc, "pa_crossover_eq7: needs mu_L + mu_O > 0, k0 > 0, N > 0")
        return dict(zip(("lhs", "rhs", "beta_eb_w", "tp_eb", "tp_mb"), list(o)))

    def timer_reset(self):
        self._check(self.lib.pa_timer_reset(self.ctx))

    def plan_info(self, which: int) -> int:
        return int(self.lib.pa_plan_info(self.ctx, which))

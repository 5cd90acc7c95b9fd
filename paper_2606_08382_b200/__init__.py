"""ctypes binding of libstarkv.so (include/starkv.h) -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; torch is used for device
memory and streams.  There is no CPU fallback: importing this package without a built
``libstarkv.so`` raises, and every call on a machine without a CUDA device returns an error code
that is turned into ``StarkvError``.

The functions carry the C names (``starkv_create``, ``starkv_pack``, ``starkv_unpack``,
``starkv_append``, ``starkv_decode_attn`` ...) and take torch tensors (or raw integer pointers)
where the C side takes pointers.
"""
from __future__ import annotations

import ctypes
import math
import os
from typing import Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libstarkv.so")

SYMBOLS = [
    "starkv_create", "starkv_destroy", "starkv_page_bytes", "starkv_workspace_bytes",
    "starkv_append_workspace_bytes", "starkv_pack", "starkv_unpack", "starkv_append",
    "starkv_decode_attn", "starkv_decode_attn_latent", "starkv_decode_step", "starkv_decode_attn_static", "starkv_decode_attn_generic", "starkv_decode_attn_rope", "starkv_decode_attn_host",
    "starkv_append_host_workspace_bytes", "starkv_append_host", "starkv_decode_step_host", "starkv_set_kernel_timing",
    "starkv_last_decode_kernel_ms",
    "starkv_set_splits", "starkv_set_option", "starkv_last_launches", "starkv_decode_kernel_name", "starkv_last_append_kernel_name", "starkv_strerror",
    "starkv_last_error",
]

STARKV_OK = 0
STARKV_ERR_INVALID_ARG = -1
STARKV_ERR_UNSUPPORTED = -2
STARKV_ERR_WORKSPACE = -3
STARKV_ERR_CUDA = -4


class StarkvError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"starkv error {code}: {text}")
        self.code = code


class starkv_desc(ctypes.Structure):
    _fields_ = [
        ("n_q_heads", ctypes.c_int32), ("n_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
        ("rank_k", ctypes.POINTER(ctypes.c_int32)), ("rank_k_hi", ctypes.POINTER(ctypes.c_int32)),
        ("rank_v", ctypes.c_int32), ("rank_v_hi", ctypes.c_int32),
        ("bits_hi", ctypes.c_int32), ("bits_lo", ctypes.c_int32),
        ("page_tokens", ctypes.c_int32), ("layout_id", ctypes.c_int32), ("sm_scale", ctypes.c_float),
    ]


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python paper_2606_08382_b200/build.py` "
            "(or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32p, c_int, c_i64, c_sz = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_size_t
    lib.starkv_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(starkv_desc), vp]
    lib.starkv_create.restype = c_int
    lib.starkv_destroy.argtypes = [vp]
    lib.starkv_destroy.restype = None
    lib.starkv_page_bytes.argtypes = [vp]
    lib.starkv_page_bytes.restype = c_sz
    lib.starkv_workspace_bytes.argtypes = [vp, c_int, c_int]
    lib.starkv_workspace_bytes.restype = c_sz
    lib.starkv_append_workspace_bytes.argtypes = [vp, c_int]
    lib.starkv_append_workspace_bytes.restype = c_sz
    lib.starkv_pack.argtypes = [vp, vp, vp, c_int, vp]
    lib.starkv_pack.restype = c_int
    lib.starkv_unpack.argtypes = [vp, vp, c_int, vp, vp, vp]
    lib.starkv_unpack.restype = c_int
    lib.starkv_append.argtypes = [vp, vp, i32p, c_int, i32p, i32p, c_int, vp, c_i64, c_i64, c_int, vp, c_i64,
                                  c_int, vp, vp, vp, c_sz]
    lib.starkv_append.restype = c_int
    dec = [vp, vp, vp, i32p, c_int, i32p, c_int, vp, vp, vp, c_sz, vp]
    lib.starkv_decode_attn_rope.argtypes = [vp, vp, vp, i32p, c_int, i32p, i32p, ctypes.c_float, c_int, vp, vp, vp, c_sz, vp]
    lib.starkv_decode_attn_rope.restype = c_int
    lib.starkv_decode_step.argtypes = [vp, vp, i32p, c_int, i32p, i32p, c_int, vp, c_i64, c_i64, c_int, vp, c_i64, c_int, vp, vp,
                                       vp, c_sz, vp, i32p, vp, vp, vp, c_sz, vp]
    lib.starkv_decode_step.restype = c_int
    lib.starkv_decode_attn_latent.argtypes = [vp, vp, vp, i32p, c_int, i32p, c_int, vp, vp, c_sz, vp]
    lib.starkv_decode_attn_latent.restype = c_int
    lib.starkv_decode_attn_static.argtypes = [vp, vp, vp, i32p, c_int, i32p, c_int, vp, vp, vp]
    lib.starkv_decode_attn_static.restype = c_int
    for name in ("starkv_decode_attn", "starkv_decode_attn_generic", "starkv_decode_attn_host"):
        getattr(lib, name).argtypes = dec
        getattr(lib, name).restype = c_int
    lib.starkv_append_host_workspace_bytes.argtypes = [vp, c_int, c_int, c_int]
    lib.starkv_append_host_workspace_bytes.restype = c_sz
    lib.starkv_append_host.argtypes = [vp, vp, i32p, c_int, i32p, i32p, c_int, vp, c_int, c_i64, c_int, vp, c_int,
                                       c_int, vp, vp, vp, c_sz]
    lib.starkv_append_host.restype = c_int
    lib.starkv_decode_step_host.argtypes = [vp, vp, i32p, c_int, i32p, i32p, c_int, vp, c_int, c_i64, c_int, vp, c_int, c_int, vp, vp,
                                            vp, c_sz, vp, i32p, vp, vp, vp, c_sz, vp]
    lib.starkv_decode_step_host.restype = c_int
    lib.starkv_set_kernel_timing.argtypes = [vp, c_int]
    lib.starkv_set_kernel_timing.restype = c_int
    lib.starkv_last_decode_kernel_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    lib.starkv_last_decode_kernel_ms.restype = c_int
    lib.starkv_set_splits.argtypes = [vp, c_int]
    lib.starkv_set_splits.restype = c_int
    lib.starkv_last_launches.argtypes = [vp]
    lib.starkv_last_launches.restype = c_int
    lib.starkv_set_option.argtypes = [vp, ctypes.c_char_p, c_int]
    lib.starkv_set_option.restype = c_int
    lib.starkv_decode_kernel_name.argtypes = [vp]
    lib.starkv_decode_kernel_name.restype = ctypes.c_char_p
    lib.starkv_last_append_kernel_name.argtypes = [vp]
    lib.starkv_last_append_kernel_name.restype = ctypes.c_char_p
    lib.starkv_strerror.argtypes = [c_int]
    lib.starkv_strerror.restype = ctypes.c_char_p
    lib.starkv_last_error.argtypes = [vp]
    lib.starkv_last_error.restype = ctypes.c_char_p
    return lib


_lib = _load()


_PTR_OF = {}   # type -> its unbound data_ptr, filled on first sight (the common case, once per argument per call)


def _ptr(x) -> Optional[int]:
    """Device/host pointer of a torch tensor, numpy array, int or None."""
    f = _PTR_OF.get(type(x))
    if f is not None:
        return f(x)
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        _PTR_OF[type(x)] = type(x).data_ptr
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(f"cannot take a pointer of {type(x)}")


class Context:
    """Owns one starkv_ctx*.  ``stream``: a torch.cuda.Stream, a raw cudaStream_t int, or None."""

    def __init__(self, handle: int, desc_keepalive):
        self.handle = handle
        self._keep = desc_keepalive

    def _check(self, rc: int) -> None:
        if rc != STARKV_OK:
            text = _lib.starkv_strerror(rc).decode()
            if rc == STARKV_ERR_CUDA:
                text += ": " + _lib.starkv_last_error(self.handle).decode()
            raise StarkvError(rc, text)

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h:
            _lib.starkv_destroy(h)


def starkv_create(n_q_heads: int, n_kv_heads: int, head_dim: int, rank_k: Sequence[int],
                  rank_k_hi: Sequence[int], rank_v: int, rank_v_hi: int, bits_hi: int, bits_lo: int,
                  page_tokens: int = 64, sm_scale: float = 0.0, stream=None, layout_id: int = 1) -> Context:
    rk = (ctypes.c_int32 * len(rank_k))(*[int(r) for r in rank_k])
    rkh = (ctypes.c_int32 * len(rank_k_hi))(*[int(r) for r in rank_k_hi])
    d = starkv_desc(n_q_heads, n_kv_heads, head_dim, rk, rkh, rank_v, rank_v_hi, bits_hi, bits_lo,
                    page_tokens, layout_id, sm_scale)
    if len(rank_k) != n_kv_heads or len(rank_k_hi) != n_kv_heads:
        raise StarkvError(STARKV_ERR_INVALID_ARG, "rank tables must have n_kv_heads entries")
    s = stream.cuda_stream if hasattr(stream, "cuda_stream") else stream
    h = ctypes.c_void_p()
    rc = _lib.starkv_create(ctypes.byref(h), ctypes.byref(d), s)
    if rc != STARKV_OK:
        raise StarkvError(rc, _lib.starkv_strerror(rc).decode())
    return Context(h.value, (rk, rkh, d))


def create_from_config(cfg, stream=None) -> Context:
    """Context for a ``synth.Config``-like object (fields of starkv_desc by name)."""
    return starkv_create(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rank_k, cfg.rank_k_hi, cfg.rank_v,
                         cfg.rank_v_hi, cfg.bits_hi, cfg.bits_lo, cfg.page_tokens, float(cfg.sm_scale), stream)


def starkv_page_bytes(ctx: Context) -> int:
    return int(_lib.starkv_page_bytes(ctx.handle))


def starkv_workspace_bytes(ctx: Context, batch: int, max_pages: int) -> int:
    return int(_lib.starkv_workspace_bytes(ctx.handle, batch, max_pages))


def starkv_append_workspace_bytes(ctx: Context, n_new: int) -> int:
    return int(_lib.starkv_append_workspace_bytes(ctx.handle, n_new))


def starkv_pack(ctx: Context, latents_k, latents_v, n_tokens: int, pages_out) -> None:
    ctx._check(_lib.starkv_pack(ctx.handle, _ptr(latents_k), _ptr(latents_v), n_tokens, _ptr(pages_out)))


def starkv_unpack(ctx: Context, pages_in, n_tokens: int, codes_out=None, scales_out=None, dequant_out=None) -> None:
    ctx._check(_lib.starkv_unpack(ctx.handle, _ptr(pages_in), n_tokens, _ptr(codes_out), _ptr(scales_out),
                                  _ptr(dequant_out)))


def starkv_append(ctx: Context, page_pool, block_table, max_pages: int, seq_ids, positions, n_new: int,
                  k_new, k_row_stride: int, k_head_stride: int, d_in_k: int, v_new, v_row_stride: int,
                  d_in_v: int, A_k, A_v, workspace, workspace_bytes: int) -> None:
    ctx._check(_lib.starkv_append(ctx.handle, _ptr(page_pool), _ptr(block_table), max_pages, _ptr(seq_ids),
                                  _ptr(positions), n_new, _ptr(k_new), k_row_stride, k_head_stride, d_in_k,
                                  _ptr(v_new), v_row_stride, d_in_v, _ptr(A_k), _ptr(A_v), _ptr(workspace),
                                  workspace_bytes))


def _decode(fn, ctx, q, page_pool, block_table, max_pages, seq_lens, batch, B_k, B_v, workspace, workspace_bytes, out):
    ctx._check(fn(ctx.handle, _ptr(q), _ptr(page_pool), _ptr(block_table), max_pages, _ptr(seq_lens), batch,
                  _ptr(B_k), _ptr(B_v), _ptr(workspace), workspace_bytes, _ptr(out)))


def starkv_decode_attn(ctx, q, page_pool, block_table, max_pages, seq_lens, batch, B_k, B_v, workspace,
                       workspace_bytes, out) -> None:
    _decode(_lib.starkv_decode_attn, ctx, q, page_pool, block_table, max_pages, seq_lens, batch, B_k, B_v,
            workspace, workspace_bytes, out)


def starkv_decode_step(ctx, page_pool, block_table, max_pages, seq_ids, positions, batch, k_new, k_row_stride, k_head_stride,
                       d_in_k, v_new, v_row_stride, d_in_v, A_k, A_v, append_workspace, append_workspace_bytes, q, seq_lens,
                       B_k, B_v, workspace, workspace_bytes, out) -> None:
    ctx._check(_lib.starkv_decode_step(ctx.handle, _ptr(page_pool), _ptr(block_table), max_pages, _ptr(seq_ids),
                                       _ptr(positions), batch, _ptr(k_new), k_row_stride, k_head_stride, d_in_k, _ptr(v_new),
                                       v_row_stride, d_in_v, _ptr(A_k), _ptr(A_v), _ptr(append_workspace),
                                       append_workspace_bytes, _ptr(q), _ptr(seq_lens), _ptr(B_k), _ptr(B_v),
                                       _ptr(workspace), workspace_bytes, _ptr(out)))


def starkv_decode_attn_latent(ctx, q, page_pool, block_table, max_pages, seq_lens, batch, B_k, workspace, workspace_bytes,
                              out_latent) -> None:
    """Latent-output mode: out_latent fp16 [batch, H_q, r_v] = softmax(s) . L_v (no B_v up-projection)."""
    ctx._check(_lib.starkv_decode_attn_latent(ctx.handle, _ptr(q), _ptr(page_pool), _ptr(block_table), max_pages,
                                              _ptr(seq_lens), batch, _ptr(B_k), _ptr(workspace), workspace_bytes,
                                              _ptr(out_latent)))


STATIC_SCRATCH_BYTES = 8 << 20   # include/starkv.h STARKV_STATIC_SCRATCH_BYTES


def starkv_decode_attn_static(ctx, q, page_pool, block_table, max_pages, seq_lens, batch, B_k, B_v, out) -> None:
    """starkv_decode_attn with the decode scratch in the library's static device array (no workspace argument,
    no allocation inside the call)."""
    rc = _lib.starkv_decode_attn_static(ctx.handle, _ptr(q), _ptr(page_pool), _ptr(block_table), max_pages,
                                        _ptr(seq_lens), batch, _ptr(B_k), _ptr(B_v), _ptr(out))
    if rc == STARKV_ERR_WORKSPACE:   # the library's text names the bytes needed and the array's size
        raise StarkvError(rc, _lib.starkv_last_error(ctx.handle).decode())
    ctx._check(rc)


def starkv_decode_attn_rope(ctx, q_rotated, page_pool, block_table, max_pages, seq_lens, pos_offset, rope_theta, batch, B_k, B_v,
                            workspace, workspace_bytes, out) -> None:
    ctx._check(_lib.starkv_decode_attn_rope(ctx.handle, _ptr(q_rotated), _ptr(page_pool), _ptr(block_table), max_pages,
                                            _ptr(seq_lens), _ptr(pos_offset) if pos_offset is not None else None,
                                            ctypes.c_float(rope_theta), batch, _ptr(B_k), _ptr(B_v), _ptr(workspace),
                                            workspace_bytes, _ptr(out)))


def starkv_decode_attn_generic(ctx, q, page_pool, block_table, max_pages, seq_lens, batch, B_k, B_v, workspace,
                               workspace_bytes, out) -> None:
    _decode(_lib.starkv_decode_attn_generic, ctx, q, page_pool, block_table, max_pages, seq_lens, batch, B_k,
            B_v, workspace, workspace_bytes, out)


def starkv_decode_attn_host(ctx, q_host, page_pool, block_table, max_pages, seq_lens_host, batch, B_k, B_v,
                            workspace, workspace_bytes, out_host) -> None:
    _decode(_lib.starkv_decode_attn_host, ctx, q_host, page_pool, block_table, max_pages, seq_lens_host, batch,
            B_k, B_v, workspace, workspace_bytes, out_host)


def starkv_decode_step_host(ctx, page_pool, block_table, max_pages, seq_ids_host, positions_host, batch, k_new_host, k_row_elems,
                            k_head_stride, d_in_k, v_new_host, v_row_elems, d_in_v, A_k, A_v, append_workspace,
                            append_workspace_bytes, q_host, seq_lens_host, B_k, B_v, workspace, workspace_bytes, out_host) -> None:
    ctx._check(_lib.starkv_decode_step_host(ctx.handle, _ptr(page_pool), _ptr(block_table), max_pages, _ptr(seq_ids_host),
                                            _ptr(positions_host), batch, _ptr(k_new_host), k_row_elems, k_head_stride, d_in_k,
                                            _ptr(v_new_host), v_row_elems, d_in_v, _ptr(A_k), _ptr(A_v), _ptr(append_workspace),
                                            append_workspace_bytes, _ptr(q_host), _ptr(seq_lens_host), _ptr(B_k), _ptr(B_v),
                                            _ptr(workspace), workspace_bytes, _ptr(out_host)))


def starkv_append_host_workspace_bytes(ctx: Context, n_new: int, k_row_elems: int, v_row_elems: int) -> int:
    return int(_lib.starkv_append_host_workspace_bytes(ctx.handle, n_new, k_row_elems, v_row_elems))


def starkv_append_host(ctx: Context, page_pool, block_table, max_pages: int, seq_ids_host, positions_host,
                       n_new: int, k_new_host, k_row_elems: int, k_head_stride: int, d_in_k: int, v_new_host,
                       v_row_elems: int, d_in_v: int, A_k, A_v, workspace, workspace_bytes: int) -> None:
    ctx._check(_lib.starkv_append_host(ctx.handle, _ptr(page_pool), _ptr(block_table), max_pages,
                                       _ptr(seq_ids_host), _ptr(positions_host), n_new, _ptr(k_new_host),
                                       k_row_elems, k_head_stride, d_in_k, _ptr(v_new_host), v_row_elems, d_in_v,
                                       _ptr(A_k), _ptr(A_v), _ptr(workspace), workspace_bytes))


def starkv_set_kernel_timing(ctx: Context, on: bool) -> None:
    ctx._check(_lib.starkv_set_kernel_timing(ctx.handle, 1 if on else 0))


def starkv_last_decode_kernel_ms(ctx: Context) -> float:
    ms = ctypes.c_float(0.0)
    ctx._check(_lib.starkv_last_decode_kernel_ms(ctx.handle, ctypes.byref(ms)))
    return float(ms.value)


def starkv_set_splits(ctx: Context, n_splits: int) -> None:
    ctx._check(_lib.starkv_set_splits(ctx.handle, n_splits))


DECODE_VARIANTS = {"auto": 0, "mma": 1, "tc5": 2, "tm": 3, "generic": 4}


def starkv_set_option(ctx: Context, name: str, value: int) -> None:
    ctx._check(_lib.starkv_set_option(ctx.handle, name.encode(), int(value)))


def starkv_last_launches(ctx: Context) -> int:
    return int(_lib.starkv_last_launches(ctx.handle))


def starkv_decode_kernel_name(ctx: Context) -> str:
    return _lib.starkv_decode_kernel_name(ctx.handle).decode()


def starkv_last_append_kernel_name(ctx: Context) -> str:
    return _lib.starkv_last_append_kernel_name(ctx.handle).decode()


def starkv_strerror(code: int) -> str:
    return _lib.starkv_strerror(code).decode()

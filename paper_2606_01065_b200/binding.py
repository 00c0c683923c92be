"""Thin ctypes binding of libleyline.so (include/leyline.h): argument marshalling only.

Same names as the C ABI: ``leyline_plan`` (host planner), ``leyline_splice`` (FRESH / INPLACE_MOVE) and
``leyline_rotate_inplace`` (ROTATE_ONLY).  Every step of the path runs inside the library's kernels; torch is
used by callers for device memory and streams only.  There is no CPU fallback: if the shared library cannot be
loaded (or built with nvcc) importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Sequence

import numpy as np

from . import build as _build

OK, E_INVALID, E_UNSORTED, E_OVERLAP, E_RANGE, E_NOFREE, E_UNSUPPORTED, E_CUDA, E_NOMEM, E_ALIAS = range(10)
BF16, FP8_E4M3 = 0, 1
NEOX, INTERLEAVED = 0, 1
FRESH, INPLACE_MOVE, ROTATE_ONLY = 0, 1, 2
AMORTIZE, FORGET = 0, 1
TILE_SRC_REPL = 1


class CacheDesc(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("latent_dim", C.c_int32), ("rope_dim", C.c_int32),
                ("page_size", C.c_int32), ("dtype", C.c_int32), ("pairing", C.c_int32),
                ("rope_heads", C.c_int32), ("reserved_", C.c_int32), ("row_stride_bytes", C.c_int64), ("pool_slots", C.c_int64),
                ("inv_freq", C.POINTER(C.c_float)), ("layer_scale", C.POINTER(C.c_float)),
                ("layer_pairing", C.POINTER(C.c_int32))]


class Directive(C.Structure):
    _fields_ = [("request", C.c_int32), ("repl_len", C.c_int32), ("start", C.c_int64), ("end", C.c_int64),
                ("repl_row", C.c_int64), ("semantic", C.c_int32), ("reserved_", C.c_int32)]


class Segment(C.Structure):
    _fields_ = [("request", C.c_int32), ("kind", C.c_int32), ("src_begin", C.c_int64), ("dst_begin", C.c_int64),
                ("length", C.c_int64), ("shift", C.c_int64)]


class PlanInfo(C.Structure):
    _fields_ = [("mode", C.c_int32), ("n_requests", C.c_int32)] + [
        (n, C.c_int64) for n in ("total_new_tokens", "total_new_pages", "n_free_consumed", "n_released", "n_segments",
                                 "n_tiles", "n_move_tiles", "n_trig", "rows_moved", "rows_inserted", "rows_rotated",
                                 "bytes_read", "bytes_written", "bytes_index", "tile_rows", "rot_tile_rows", "mover")]


class Tile(C.Structure):
    _fields_ = [("src_pos", C.c_int64), ("dst_pos", C.c_int64), ("n_rows", C.c_int32), ("trig", C.c_int32),
                ("flags", C.c_int32), ("dep_lo", C.c_int32), ("dep_hi", C.c_int32), ("request", C.c_int32)]


class Tuning(C.Structure):
    _fields_ = [("kernel", C.c_int32), ("tile_rows", C.c_int32), ("ctas_per_sm", C.c_int32), ("profile", C.c_int32),
                ("stages", C.c_int32), ("layer_group", C.c_int32), ("consumer_warps", C.c_int32),
                ("rotate_kernel", C.c_int32), ("skip_alias_check", C.c_int32)]


class CdcParams(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("min_size", C.c_int32), ("max_size", C.c_int32), ("mask_bits", C.c_int32),
                ("reserved_", C.c_int32)]


class LeylineError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        msg = f"{where}: {_lib.leyline_strerror(status).decode()} (status {status})"
        if detail:
            msg += f" [{detail}]"
        super().__init__(msg)


def _load() -> C.CDLL:
    path = _build.build()          # raises if nvcc fails; never falls back to anything else
    L = C.CDLL(path)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.leyline_plan.restype = C.c_int
    L.leyline_plan.argtypes = [C.POINTER(CacheDesc), i32, i32, vp, vp, vp, i32, vp, vp, i64, C.POINTER(vp)]
    L.leyline_plan_ex.restype = C.c_int
    L.leyline_plan_ex.argtypes = [C.POINTER(CacheDesc), i32, i32, vp, vp, vp, i32, vp, vp, i64, C.POINTER(Tuning), C.POINTER(vp)]
    for name in ("leyline_plan_trig_table_device", "leyline_plan_new_seq_lens", "leyline_plan_forget_trim", "leyline_plan_slot_offsets",
                 "leyline_plan_new_pt_offsets", "leyline_plan_new_pages", "leyline_plan_released",
                 "leyline_plan_segments", "leyline_plan_tiles", "leyline_plan_trig_shifts", "leyline_plan_trig_table"):
        f = getattr(L, name)
        f.restype = C.c_int
        f.argtypes = [vp, vp]
    L.leyline_plan_get_info.restype = C.c_int
    L.leyline_plan_get_info.argtypes = [vp, C.POINTER(PlanInfo)]
    L.leyline_splice.restype = C.c_int
    L.leyline_splice.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    L.leyline_rotate_inplace.restype = C.c_int
    L.leyline_rotate_inplace.argtypes = [vp, vp, vp, vp, vp]
    L.leyline_rotate_inplace_master.restype = C.c_int
    L.leyline_rotate_inplace_master.argtypes = [vp, vp, vp, vp, vp, vp]
    L.leyline_plan_kernel_ms.restype = C.c_int
    L.leyline_plan_kernel_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.leyline_plan_prefetch.restype = C.c_int
    L.leyline_plan_prefetch.argtypes = [vp]
    L.leyline_probe_band_update.restype = C.c_int
    L.leyline_probe_band_update.argtypes = [vp, i64, i64, i32, i32, i32, vp]
    L.leyline_plan_destroy.restype = None
    L.leyline_plan_destroy.argtypes = [vp]
    L.leyline_strerror.restype = C.c_char_p
    L.leyline_strerror.argtypes = [C.c_int]
    L.leyline_last_cuda_error.restype = C.c_char_p
    L.leyline_set_tuning.restype = C.c_int
    L.leyline_set_tuning.argtypes = [C.POINTER(Tuning)]
    L.leyline_get_tuning.restype = C.c_int
    L.leyline_get_tuning.argtypes = [C.POINTER(Tuning)]
    L.leyline_version.restype = C.c_char_p
    # discovery side (include/leyline_cdc.h)
    L.leyline_cdc_chunk.restype = C.c_int
    L.leyline_cdc_chunk.argtypes = [C.POINTER(CdcParams), vp, i64, vp, i32, vp, i32, vp, vp, vp, i64, vp, vp]
    L.leyline_cdc_chunk_noalloc.restype = C.c_int
    L.leyline_cdc_chunk_noalloc.argtypes = L.leyline_cdc_chunk.argtypes
    L.leyline_cdc_last_error.restype = C.c_char_p
    L.leyline_registry_clear.restype = C.c_int
    L.leyline_registry_clear.argtypes = [vp, vp, i64, vp]
    L.leyline_registry_insert.restype = C.c_int
    L.leyline_registry_insert.argtypes = [vp, vp, i64, vp, vp, i64, vp, vp]
    L.leyline_registry_lookup.restype = C.c_int
    L.leyline_registry_lookup.argtypes = [vp, vp, i64, vp, i64, vp, vp]
    return L


_lib = _load()
LIB_PATH = _build.LIB


def _check(st: int, where: str):
    if st != OK:
        raise LeylineError(st, where, _lib.leyline_last_cuda_error().decode() if st in (E_CUDA, E_INVALID) else "")


def leyline_version() -> str:
    return _lib.leyline_version().decode()


def leyline_set_tuning(kernel: int = 0, tile_rows: int = 0, ctas_per_sm: int = 0, profile: int = 0, stages: int = 0,
                       layer_group: int = 0, consumer_warps: int = 0, rotate_kernel: int = 0, skip_alias_check: int = 0):
    t = Tuning(kernel, tile_rows, ctas_per_sm, profile, stages, layer_group, consumer_warps, rotate_kernel, skip_alias_check)
    _check(_lib.leyline_set_tuning(C.byref(t)), "leyline_set_tuning")


def leyline_get_tuning() -> dict:
    t = Tuning()
    _check(_lib.leyline_get_tuning(C.byref(t)), "leyline_get_tuning")
    return {"kernel": t.kernel, "tile_rows": t.tile_rows, "ctas_per_sm": t.ctas_per_sm, "profile": t.profile,
            "stages": t.stages, "layer_group": t.layer_group,
            "consumer_warps": t.consumer_warps, "rotate_kernel": t.rotate_kernel, "skip_alias_check": t.skip_alias_check}


def _arr(x, dtype):
    return np.ascontiguousarray(np.asarray(x, dtype=dtype))


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p) if a.size else None


def make_desc(n_layers, latent_dim, rope_dim, page_size, dtype, pairing, row_stride_bytes, pool_slots, inv_freq,
              layer_scale=None, rope_heads=1, layer_pairing=None):
    """Returns (CacheDesc, keepalive) -- keep `keepalive` referenced while the desc is in use.
    Row = latent_dim + rope_heads * rope_dim elements (rope_heads = 1: MLA; kv_heads: full-width K)."""
    inv = _arr(inv_freq, np.float32)
    sc = _arr(layer_scale, np.float32) if layer_scale is not None else None
    lp = _arr(layer_pairing, np.int32) if layer_pairing is not None else None
    if lp is not None and len(lp) != n_layers:
        raise ValueError(f"layer_pairing: expected {n_layers} entries, got {len(lp)}")
    d = CacheDesc(n_layers, latent_dim, rope_dim, page_size, dtype, pairing, rope_heads, 0, row_stride_bytes, pool_slots,
                  inv.ctypes.data_as(C.POINTER(C.c_float)),
                  sc.ctypes.data_as(C.POINTER(C.c_float)) if sc is not None else None,
                  lp.ctypes.data_as(C.POINTER(C.c_int32)) if lp is not None else None)
    return d, (inv, sc, lp)


class Plan:
    """Owner of a ``leyline_plan_t*`` (destroyed on ``close()`` / garbage collection)."""

    def __init__(self, handle, n_requests: int, rope_dim: int):
        self._h = C.c_void_p(handle)
        self.n_requests = n_requests
        self._H = rope_dim // 2
        self.info = PlanInfo()
        _check(_lib.leyline_plan_get_info(self._h, C.byref(self.info)), "leyline_plan_get_info")

    # -- queries (host) --
    def _get(self, fn, n, dtype):
        out = np.zeros(int(n), dtype=dtype)
        _check(getattr(_lib, fn)(self._h, _ptr(out)), fn)
        return out

    @property
    def new_seq_lens(self): return self._get("leyline_plan_new_seq_lens", self.n_requests, np.int64)
    @property
    def forget_trim(self): return self._get("leyline_plan_forget_trim", self.n_requests, np.int64)
    @property
    def slot_offsets(self): return self._get("leyline_plan_slot_offsets", self.n_requests + 1, np.int64)
    @property
    def new_pt_offsets(self): return self._get("leyline_plan_new_pt_offsets", self.n_requests + 1, np.int64)
    @property
    def new_pages(self): return self._get("leyline_plan_new_pages", self.info.total_new_pages, np.int32)
    @property
    def released(self): return self._get("leyline_plan_released", self.info.n_released, np.int32)
    @property
    def trig_shifts(self): return self._get("leyline_plan_trig_shifts", self.info.n_trig, np.int64)
    @property
    def trig_table(self):
        return self._get("leyline_plan_trig_table", self.info.n_trig * 2 * self._H, np.float32).reshape(-1, 2, self._H)

    @property
    def trig_table_device(self):
        """The table the launches use (evaluated in fp64 on the device); valid after a launch."""
        return self._get("leyline_plan_trig_table_device", self.info.n_trig * 2 * self._H, np.float32).reshape(-1, 2, self._H)

    @property
    def segments(self):
        buf = (Segment * int(self.info.n_segments))()
        _check(_lib.leyline_plan_segments(self._h, C.cast(buf, C.c_void_p)), "leyline_plan_segments")
        return [(s.request, s.kind, s.src_begin, s.dst_begin, s.length, s.shift) for s in buf]

    @property
    def tiles(self):
        buf = (Tile * int(self.info.n_tiles))()
        _check(_lib.leyline_plan_tiles(self._h, C.cast(buf, C.c_void_p)), "leyline_plan_tiles")
        return list(buf)

    def prefetch(self):
        """leyline.h: leyline_plan_prefetch -- start the table upload on the library's copy stream."""
        _check(_lib.leyline_plan_prefetch(self._h), "leyline_plan_prefetch")
        return self

    def kernel_ms(self) -> float:
        ms = C.c_float()
        _check(_lib.leyline_plan_kernel_ms(self._h, C.byref(ms)), "leyline_plan_kernel_ms")
        return ms.value

    def close(self):
        if self._h:
            _lib.leyline_plan_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self): return self
    def __exit__(self, *a): self.close()


def pack_directives(directives: Sequence) -> np.ndarray:
    """(request, start, end, repl_len, repl_row, semantic) tuples -> packed leyline_directive array."""
    dt = np.dtype([("request", np.int32), ("repl_len", np.int32), ("start", np.int64), ("end", np.int64),
                   ("repl_row", np.int64), ("semantic", np.int32), ("reserved_", np.int32)])
    assert dt.itemsize == C.sizeof(Directive)
    a = np.zeros(len(directives), dt)
    for i, (r, s, e, n, row, sem) in enumerate(directives):
        a[i] = (r, n, s, e, row, sem, 0)
    return a


def leyline_plan(desc: CacheDesc, mode: int, seq_lens, pt_offsets, pages, directives, free_ids) -> Plan:
    """Host planner (leyline.h: leyline_plan).  All arguments are host arrays; `directives` is a sequence of
    (request, start, end, repl_len, repl_row, semantic) or an array from ``pack_directives``."""
    sl, po, pg, fr = _arr(seq_lens, np.int64), _arr(pt_offsets, np.int64), _arr(pages, np.int32), _arr(free_ids, np.int32)
    d = directives if isinstance(directives, np.ndarray) else pack_directives(directives)
    h = C.c_void_p()
    st = _lib.leyline_plan(C.byref(desc), mode, len(sl), _ptr(sl), _ptr(po), _ptr(pg), len(d), _ptr(d), _ptr(fr),
                           len(fr), C.byref(h))
    _check(st, "leyline_plan")
    return Plan(h.value, len(sl), desc.rope_dim)


def leyline_plan_ex(desc: CacheDesc, mode: int, seq_lens, pt_offsets, pages, directives, free_ids, tuning: Tuning | None = None) -> Plan:
    """leyline.h: leyline_plan_ex -- the planner with its tuning passed per call (None = defaults); the process-wide
    tuning of leyline_set_tuning is not consulted."""
    sl, po, pg, fr = _arr(seq_lens, np.int64), _arr(pt_offsets, np.int64), _arr(pages, np.int32), _arr(free_ids, np.int32)
    d = directives if isinstance(directives, np.ndarray) else pack_directives(directives)
    h = C.c_void_p()
    st = _lib.leyline_plan_ex(C.byref(desc), mode, len(sl), _ptr(sl), _ptr(po), _ptr(pg), len(d), _ptr(d), _ptr(fr),
                              len(fr), C.byref(tuning) if tuning is not None else None, C.byref(h))
    _check(st, "leyline_plan_ex")
    return Plan(h.value, len(sl), desc.rope_dim)


class LayerPointers:
    """A host array of per-layer device pointers, marshalled once (``layer_pointers``) and reusable across calls;
    keeps the tensors alive."""

    def __init__(self, layers):
        self.n = len(layers)
        self.array = (C.c_void_p * self.n)()
        for i, t in enumerate(layers):
            self.array[i] = int(t) if isinstance(t, int) else t.data_ptr()
        self.keep = layers


def layer_pointers(layers) -> LayerPointers:
    return LayerPointers(layers)


def _ptr_array(layers, n_layers: int, what: str):
    if layers is None:
        return None, None
    lp = layers if isinstance(layers, LayerPointers) else LayerPointers(layers)
    if lp.n != n_layers:
        raise ValueError(f"{what}: expected {n_layers} layers, got {lp.n}")
    return lp.array, lp


def _stream_handle(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(stream if isinstance(stream, int) else stream.cuda_stream)


def _dev_ptr(t):
    return None if t is None else C.c_void_p(int(t) if isinstance(t, int) else t.data_ptr())


def leyline_splice(plan: Plan, layer_src, layer_dst, layer_repl=None, page_table_out=None, slot_idx_out=None,
                   stream=None, n_layers: int | None = None):
    """leyline.h: leyline_splice.  layer_* are sequences of device tensors (or raw device pointers), one per
    layer; *_out are int32 device tensors or None.  Asynchronous on `stream` (default: torch's current)."""
    n = n_layers if n_layers is not None else (layer_dst.n if isinstance(layer_dst, LayerPointers) else len(layer_dst))
    a, _k1 = _ptr_array(layer_src, n, "layer_src")
    b, _k2 = _ptr_array(layer_dst, n, "layer_dst")
    c, _k3 = _ptr_array(layer_repl, n, "layer_repl")
    st = _lib.leyline_splice(plan._h, a, b, c, _dev_ptr(page_table_out), _dev_ptr(slot_idx_out), _stream_handle(stream))
    _check(st, "leyline_splice")


def leyline_rotate_inplace(plan: Plan, layers, layer_repl=None, slot_idx_out=None, stream=None):
    """leyline.h: leyline_rotate_inplace."""
    n = layers.n if isinstance(layers, LayerPointers) else len(layers)
    a, _k1 = _ptr_array(layers, n, "layer_ptrs")
    c, _k3 = _ptr_array(layer_repl, n, "layer_repl")
    st = _lib.leyline_rotate_inplace(plan._h, a, c, _dev_ptr(slot_idx_out), _stream_handle(stream))
    _check(st, "leyline_rotate_inplace")


def leyline_rotate_inplace_master(plan: Plan, layers, layer_master, layer_repl=None, slot_idx_out=None, stream=None):
    """leyline.h: leyline_rotate_inplace_master (fp32 master band per layer, float32 tensors [pool_slots, band])."""
    n = layers.n if isinstance(layers, LayerPointers) else len(layers)
    a, _k1 = _ptr_array(layers, n, "layer_ptrs")
    m, _k2 = _ptr_array(layer_master, n, "layer_master")
    c, _k3 = _ptr_array(layer_repl, n, "layer_repl")
    st = _lib.leyline_rotate_inplace_master(plan._h, a, m, c, _dev_ptr(slot_idx_out), _stream_handle(stream))
    _check(st, "leyline_rotate_inplace_master")


def leyline_probe_band_update(buf, n_rows: int, row_stride_bytes: int, band_offset_bytes: int, band_bytes: int,
                              ctas_per_sm: int = 0, stream=None):
    """leyline.h: leyline_probe_band_update (measurement aid: the a5 access pattern on a contiguous buffer)."""
    _check(_lib.leyline_probe_band_update(_dev_ptr(buf), n_rows, row_stride_bytes, band_offset_bytes, band_bytes, ctas_per_sm,
                                          _stream_handle(stream)), "leyline_probe_band_update")


# ----------------------------------------------------------------------------- discovery side (leyline_cdc.h)

CDC_HASH, CDC_ANCHOR, CDC_MAX, CDC_SEQ_END = range(4)


def leyline_cdc_chunk(params: CdcParams, tokens, n_tokens: int, seq_offsets, n_seqs: int, anchor_ids, n_anchor_ids: int,
                      chunk_end, chunk_hash, chunk_kind, capacity: int, n_chunks, stream=None):
    """leyline_cdc.h: leyline_cdc_chunk.  Every array argument is a device tensor (or raw device pointer, or None
    where the header allows NULL); outputs are written in place."""
    st = _lib.leyline_cdc_chunk(C.byref(params), _dev_ptr(tokens), n_tokens, _dev_ptr(seq_offsets), n_seqs,
                                _dev_ptr(anchor_ids), n_anchor_ids, _dev_ptr(chunk_end), _dev_ptr(chunk_hash),
                                _dev_ptr(chunk_kind), capacity, _dev_ptr(n_chunks), _stream_handle(stream))
    _check(st, "leyline_cdc_chunk")


CDC_NOALLOC_MAX_TOKENS = 524288      # leyline_cdc.h: LEYLINE_CDC_NOALLOC_MAX_TOKENS


def leyline_cdc_chunk_noalloc(params: CdcParams, tokens, n_tokens: int, seq_offsets, n_seqs: int, anchor_ids,
                              n_anchor_ids: int, chunk_end, chunk_hash, chunk_kind, capacity: int, n_chunks, stream=None):
    """leyline_cdc.h: leyline_cdc_chunk_noalloc.  Same arguments and results as ``leyline_cdc_chunk``, for callers that
    may not allocate device memory (a server whose own allocator owns the GPU, a fixed memory budget): the working
    tables sit in an 8 MiB array inside the library instead of a pool, so ``n_tokens`` is limited to
    ``CDC_NOALLOC_MAX_TOKENS`` (LeylineError with the library's message beyond it).  Calls share that array: keep them
    on one stream, or order them; make the first call on a device before any stream capture."""
    st = _lib.leyline_cdc_chunk_noalloc(C.byref(params), _dev_ptr(tokens), n_tokens, _dev_ptr(seq_offsets), n_seqs,
                                        _dev_ptr(anchor_ids), n_anchor_ids, _dev_ptr(chunk_end), _dev_ptr(chunk_hash),
                                        _dev_ptr(chunk_kind), capacity, _dev_ptr(n_chunks), _stream_handle(stream))
    if st != OK:
        raise LeylineError(st, "leyline_cdc_chunk_noalloc", _lib.leyline_cdc_last_error().decode())


def leyline_registry_clear(keys, vals, capacity: int, stream=None):
    _check(_lib.leyline_registry_clear(_dev_ptr(keys), _dev_ptr(vals), capacity, _stream_handle(stream)),
           "leyline_registry_clear")


def leyline_registry_insert(keys, vals, capacity: int, hashes, values, n: int, n_dropped=None, stream=None):
    _check(_lib.leyline_registry_insert(_dev_ptr(keys), _dev_ptr(vals), capacity, _dev_ptr(hashes), _dev_ptr(values), n,
                                        _dev_ptr(n_dropped), _stream_handle(stream)), "leyline_registry_insert")


def leyline_registry_lookup(keys, vals, capacity: int, hashes, n: int, out, stream=None):
    _check(_lib.leyline_registry_lookup(_dev_ptr(keys), _dev_ptr(vals), capacity, _dev_ptr(hashes), n, _dev_ptr(out),
                                        _stream_handle(stream)), "leyline_registry_lookup")

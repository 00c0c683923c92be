"""oracle/cdc.py -- TEST INFRASTRUCTURE ONLY: ctypes marshalling for oracle/cdc_oracle.c (the sequential CPU
definition of the anchored content-defined chunker, content hash and registry of the discovery side; SURVEY.md
section 8(f) NEXT-4).  The arithmetic is in the C file; the registry (reading D5: key -> smallest
value inserted) is a Python dict.  Nothing here is imported by the product."""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import lib as _base_lib

KIND_HASH, KIND_ANCHOR, KIND_MAX, KIND_SEQ_END = 0, 1, 2, 3
_ready = False


def _lib():
    global _ready
    L = _base_lib()
    if not _ready:
        L.cdc_ora_gear.restype = C.c_uint64
        L.cdc_ora_gear.argtypes = [C.c_uint64, C.c_int32]
        L.cdc_ora_content_hash.restype = C.c_uint64
        L.cdc_ora_content_hash.argtypes = [C.c_void_p, C.c_int64, C.c_int64]
        L.cdc_ora_signature.restype = None
        L.cdc_ora_signature.argtypes = [C.c_uint64, C.c_void_p, C.c_int64, C.c_void_p, C.c_int32, C.c_void_p, C.c_int32,
                                        C.c_void_p]
        L.cdc_ora_chunk.restype = C.c_int64
        L.cdc_ora_chunk.argtypes = [C.c_uint64, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_int64, C.c_void_p,
                                    C.c_int32, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        _ready = True
    return L


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def gear(seed: int, token: int) -> int:
    return int(_lib().cdc_ora_gear(C.c_uint64(seed), C.c_int32(token)))


def content_hash(tokens, b: int, e: int) -> int:
    t = np.ascontiguousarray(tokens, np.int32)
    return int(_lib().cdc_ora_content_hash(_p(t), b, e))


def _prep(tokens, seq_offsets, anchors):
    t = np.ascontiguousarray(tokens, np.int32)
    so = np.ascontiguousarray([0, len(t)] if seq_offsets is None else seq_offsets, np.int64)
    an = np.ascontiguousarray(sorted(anchors) if anchors is not None else [], np.int32)
    return t, so, an


def signature(seed: int, tokens, seq_offsets=None, anchors=None) -> np.ndarray:
    t, so, an = _prep(tokens, seq_offsets, anchors)
    out = np.zeros(len(t), np.uint64)
    _lib().cdc_ora_signature(C.c_uint64(seed), _p(t), len(t), _p(so), len(so) - 1, _p(an), len(an), _p(out))
    return out


def chunk(seed: int, min_size: int, max_size: int, mask_bits: int, tokens, seq_offsets=None, anchors=None):
    """-> (chunk_end int64 [n_chunks] exclusive global ends, chunk_hash uint64 [n_chunks], chunk_kind int32 [n_chunks])"""
    t, so, an = _prep(tokens, seq_offsets, anchors)
    n = len(t)
    end, hsh, kind = np.zeros(max(n, 1), np.int64), np.zeros(max(n, 1), np.uint64), np.zeros(max(n, 1), np.int32)
    c = _lib().cdc_ora_chunk(C.c_uint64(seed), min_size, max_size, mask_bits, _p(t), n, _p(so), len(so) - 1, _p(an),
                             len(an), _p(end), _p(hsh), _p(kind))
    return end[:c].copy(), hsh[:c].copy(), kind[:c].copy()


class Registry:
    """D5: content hash -> smallest value inserted under it (values are source positions)."""

    def __init__(self):
        self.d = {}

    def insert(self, hashes, values):
        for h, v in zip(hashes, values):
            h, v = int(h), int(v)
            self.d[h] = min(self.d.get(h, v), v)

    def lookup(self, hashes) -> np.ndarray:
        return np.array([self.d.get(int(h), -1) for h in hashes], np.int64)

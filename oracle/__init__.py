"""oracle/ -- TEST INFRASTRUCTURE ONLY (see the header of leyline_oracle.c).

ctypes loader and per-request orchestration for the plain-C CPU oracle of the Leyline splice
(arxiv/paper_2606_01065).  Nothing here imports, links or shares code with the CUDA library in
``paper_2606_01065_b200``; only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.

The arithmetic lives in ``leyline_oracle.c`` (each function cites the PAPER.md passage it follows);
this file only marshals numpy arrays and loops over requests in ascending order (rule O3 of DESIGN.md:
"requests processed in ascending index; free ids consumed front to back").
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "leyline_oracle.c")
_SRC_CDC = os.path.join(_HERE, "cdc_oracle.c")     # discovery side, wrapped by oracle/cdc.py
_LIB = os.path.join(_HERE, "liboracle.so")

OK, E_INVALID, E_UNSORTED, E_OVERLAP, E_RANGE, E_NOFREE, E_UNSUPPORTED = range(7)
BF16, FP8_E4M3, F64 = 0, 1, 2
NEOX, INTERLEAVED = 0, 1
AMORTIZE, FORGET = 0, 1
KEEP, INSERT = 0, 1
FRESH, INPLACE_MOVE, ROTATE_ONLY = 0, 1, 2
ELEM_BYTES = {BF16: 2, FP8_E4M3: 1, F64: 8}


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (IEEE semantics: no fast-math, no FMA contraction)."""
    srcs = [_SRC, _SRC_CDC]
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in srcs):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               "-o", _LIB, *srcs, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.ora_bf16_decode.restype = C.c_double
        L.ora_bf16_decode.argtypes = [C.c_uint16]
        L.ora_bf16_encode.restype = C.c_uint16
        L.ora_bf16_encode.argtypes = [C.c_double]
        L.ora_e4m3_decode.restype = C.c_double
        L.ora_e4m3_decode.argtypes = [C.c_uint8]
        L.ora_e4m3_encode.restype = C.c_uint8
        L.ora_e4m3_encode.argtypes = [C.c_double]
        L.ora_slot_of.restype = C.c_int64
        L.ora_first_edit.restype = C.c_int64
        L.ora_rotate_pair.restype = None
        L.ora_rotate_pair.argtypes = [C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.ora_rerope_pair.restype = None
        L.ora_rerope_pair.argtypes = [C.c_double] * 5 + [C.POINTER(C.c_double), C.POINTER(C.c_double)]
        for name in ("ora_validate", "ora_segments", "ora_map_fresh", "ora_map_inplace", "ora_map_rotate_only",
                     "ora_apply_layer", "ora_rotate_master_layer"):
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _i64(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.int64))


def _i32(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.int32))


# ----------------------------------------------------------------------------- scalar helpers

def bf16_decode(h: int) -> float:
    return lib().ora_bf16_decode(h)


def bf16_encode(x: float) -> int:
    return lib().ora_bf16_encode(x)


def e4m3_decode(b: int) -> float:
    return lib().ora_e4m3_decode(b)


def e4m3_encode(x: float) -> int:
    return lib().ora_e4m3_encode(x)


def rotate_pair(a: float, b: float, phi: float):
    a2, b2 = C.c_double(), C.c_double()
    lib().ora_rotate_pair(a, b, phi, C.byref(a2), C.byref(b2))
    return a2.value, b2.value


def rerope_pair(a: float, b: float, p: float, c: float, theta: float):
    a2, b2 = C.c_double(), C.c_double()
    lib().ora_rerope_pair(a, b, p, c, theta, C.byref(a2), C.byref(b2))
    return a2.value, b2.value


# ----------------------------------------------------------------------------- O1 / O2

def validate(seq_lens, directives) -> int:
    """directives: sequence of (request, start, end, repl_len, repl_row, semantic)."""
    sl = _i64(seq_lens)
    d = list(directives)
    req = _i32([x[0] for x in d])
    st, en, rl, rr = (_i64([x[i] for x in d]) for i in (1, 2, 3, 4))
    sem = _i32([x[5] for x in d])
    return lib().ora_validate(C.c_int32(len(sl)), _p(sl), C.c_int32(len(d)), _p(req), _p(st), _p(en), _p(rl), _p(rr),
                              _p(sem))


@dataclass
class Segments:
    kind: np.ndarray
    src: np.ndarray
    dst: np.ndarray
    len: np.ndarray
    shift: np.ndarray
    L_new: int
    forget_trim: int

    def __len__(self):
        return len(self.kind)

    def as_tuples(self):
        return [(int(k), int(s), int(d), int(n), int(c)) for k, s, d, n, c in
                zip(self.kind, self.src, self.dst, self.len, self.shift)]


def segments(L_old: int, directives) -> Segments:
    """directives of ONE request: sequence of (start, end, repl_len, repl_row, semantic)."""
    d = list(directives)
    k = len(d)
    st, en, rl, rr = (_i64([x[i] for x in d]) for i in (0, 1, 2, 3))
    sem = _i32([x[4] for x in d])
    cap = 2 * k + 1
    kind = np.zeros(cap, np.int32)
    src, dst, ln, sh = (np.zeros(cap, np.int64) for _ in range(4))
    L_new, trim = C.c_int64(), C.c_int64()
    n = lib().ora_segments(C.c_int64(L_old), C.c_int32(k), _p(st), _p(en), _p(rl), _p(rr), _p(sem), _p(kind), _p(src),
                           _p(dst), _p(ln), _p(sh), C.byref(L_new), C.byref(trim))
    return Segments(kind[:n].copy(), src[:n].copy(), dst[:n].copy(), ln[:n].copy(), sh[:n].copy(), L_new.value,
                    trim.value)


# ----------------------------------------------------------------------------- O3

@dataclass
class RequestMap:
    segs: Segments
    L_old: int
    L_new: int
    slot_old: np.ndarray            # [L_old] token-level slots of old positions
    slot_new: np.ndarray            # [L_new] token-level slots of new positions (the new index list)
    new_pages: np.ndarray | None    # page-table row (FRESH / INPLACE_MOVE), None for ROTATE_ONLY
    released: np.ndarray            # page ids (FRESH / INPLACE_MOVE) or slot ids (ROTATE_ONLY)
    n_consumed: int


def slots_of(P: int, pages: np.ndarray, L: int) -> np.ndarray:
    """idx[t] = pages[t // P] * P + t % P, by explicit loop in C (ora_slot_of)."""
    pages = _i32(pages)
    out = np.zeros(L, np.int64)
    f = lib().ora_slot_of
    for t in range(L):
        out[t] = f(C.c_int64(P), _p(pages), C.c_int64(t))
    return out


def _slots_of_fast(P: int, pages: np.ndarray, L: int) -> np.ndarray:
    # the same definition vectorised (used only for large L; checked against slots_of in the pins)
    t = np.arange(L, dtype=np.int64)
    return _i32(pages).astype(np.int64)[t // P] * P + t % P


def map_request(mode: int, P: int, L_old: int, old_pages, directives, free_ids) -> tuple[int, RequestMap | None]:
    """Slot / page map of ONE request under rule M1/M2/M3.  ``free_ids`` is the part of the caller's free
    list not yet consumed by earlier requests.  Returns (status, RequestMap)."""
    segs = segments(L_old, directives)
    old_pages = _i32(old_pages)
    free_ids = _i32(free_ids)
    n_old = -(-L_old // P)
    L_new = segs.L_new
    n_new_cap = max(-(-L_new // P), n_old) + 1
    new_pages = np.zeros(n_new_cap, np.int32)
    nn, nc, nr = C.c_int64(), C.c_int64(), C.c_int64()
    slot_old = _slots_of_fast(P, old_pages, L_old)
    if mode == FRESH:
        released = np.zeros(n_old + 1, np.int32)
        d = list(directives)
        s0 = lib().ora_first_edit(C.c_int32(len(d)), _p(_i64([x[0] for x in d])), _p(_i64([x[1] for x in d])),
                                  _p(_i64([x[2] for x in d])), _p(_i32([x[4] for x in d])))
        st = lib().ora_map_fresh(C.c_int64(P), C.c_int64(L_old), C.c_int64(L_new), C.c_int64(s0), _p(old_pages),
                                 _p(free_ids), C.c_int64(len(free_ids)), _p(new_pages), C.byref(nn), C.byref(nc),
                                 _p(released), C.byref(nr))
    elif mode == INPLACE_MOVE:
        released = np.zeros(n_old + 1, np.int32)
        st = lib().ora_map_inplace(C.c_int64(P), C.c_int64(L_old), C.c_int64(L_new), _p(old_pages), _p(free_ids),
                                   C.c_int64(len(free_ids)), _p(new_pages), C.byref(nn), C.byref(nc), _p(released),
                                   C.byref(nr))
    elif mode == ROTATE_ONLY:
        released = np.zeros(L_old + 1, np.int32)
        idx_new = np.zeros(max(L_new, 1), np.int64)
        st = lib().ora_map_rotate_only(C.c_int64(P), C.c_int64(L_old), _p(old_pages), C.c_int32(len(segs)),
                                       _p(segs.kind), _p(segs.src), _p(segs.dst), _p(segs.len), _p(free_ids),
                                       C.c_int64(len(free_ids)), _p(idx_new), C.byref(nc), _p(released), C.byref(nr))
        if st != OK:
            return st, None
        return OK, RequestMap(segs, L_old, L_new, slot_old, idx_new[:L_new].copy(), None,
                              released[:nr.value].copy(), nc.value)
    else:
        raise ValueError(mode)
    if st != OK:
        return st, None
    pages = new_pages[:nn.value].copy()
    slot_new = _slots_of_fast(P, pages, L_new)
    return OK, RequestMap(segs, L_old, L_new, slot_old, slot_new, pages, released[:nr.value].copy(), nc.value)


@dataclass
class BatchMap:
    status: int
    requests: list = field(default_factory=list)     # RequestMap per request
    n_consumed: int = 0
    released: np.ndarray | None = None                # concatenated over requests, ascending request order

    @property
    def new_seq_lens(self):
        return np.array([r.L_new for r in self.requests], np.int64)


def plan_batch(mode: int, P: int, seq_lens, pt_offsets, pages, directives, free_ids) -> BatchMap:
    """The whole of O1-O3 for a batch: validate everything first (all-or-none), then map the
    requests in ascending order, consuming ``free_ids`` front to back.
    directives: sequence of (request, start, end, repl_len, repl_row, semantic), sorted."""
    st = validate(seq_lens, directives)
    if st != OK:
        return BatchMap(st)
    out = BatchMap(OK)
    pages = _i32(pages)
    free_ids = _i32(free_ids)
    rel = []
    for r, L in enumerate(seq_lens):
        mine = [(d[1], d[2], d[3], d[4], d[5]) for d in directives if d[0] == r]
        row = pages[pt_offsets[r]:pt_offsets[r + 1]]
        st, rm = map_request(mode, P, int(L), row, mine, free_ids[out.n_consumed:])
        if st != OK:
            return BatchMap(st)
        out.requests.append(rm)
        out.n_consumed += rm.n_consumed
        rel.append(rm.released)
    out.released = np.concatenate(rel) if rel else np.zeros(0, np.int32)
    return out


# ----------------------------------------------------------------------------- O4

def apply_layer(dtype: int, pairing: int, Dc: int, Dr: int, stride: int, inv_freq: np.ndarray, scale: float,
                old_pool: np.ndarray, new_pool: np.ndarray, repl: np.ndarray | None, rm: RequestMap,
                n_heads: int = 1) -> int:
    """One request, one layer.  old_pool (uint8, pristine) is read, new_pool (uint8) is written in place.
    A row is Dc position-free elements + n_heads heads of Dr rotated elements (n_heads = 1: MLA)."""
    assert old_pool.dtype == np.uint8 and new_pool.dtype == np.uint8
    assert old_pool.flags.c_contiguous and new_pool.flags.c_contiguous
    inv = np.ascontiguousarray(inv_freq, dtype=np.float32)
    s = rm.segs
    rp = _p(np.ascontiguousarray(repl)) if repl is not None else None
    return lib().ora_apply_layer(C.c_int(dtype), C.c_int(pairing), C.c_int32(Dc), C.c_int32(Dr), C.c_int32(n_heads),
                                 C.c_int64(stride), _p(inv), C.c_float(scale), _p(old_pool), _p(new_pool), rp, C.c_int32(len(s)),
                                 _p(s.kind), _p(s.src), _p(s.dst), _p(s.len), _p(s.shift), _p(_i64(rm.slot_old)),
                                 _p(_i64(rm.slot_new)))


def splice_layer(dtype: int, pairing: int, Dc: int, Dr: int, stride: int, inv_freq: np.ndarray, scale: float,
                 old_pool: np.ndarray, repl: np.ndarray | None, bm: BatchMap, n_heads: int = 1) -> np.ndarray:
    """All requests of a batch on one layer: returns the new pool (a copy of old_pool with every live new
    position of every request written).  Requests never alias, so their order is irrelevant here."""
    new_pool = old_pool.copy()
    for rm in bm.requests:
        st = apply_layer(dtype, pairing, Dc, Dr, stride, inv_freq, scale, old_pool, new_pool, repl, rm, n_heads)
        assert st == OK, st
    return new_pool


def rotate_master_layer(pairing: int, Dc: int, Dr: int, stride: int, inv_freq: np.ndarray, pool: np.ndarray,
                        master: np.ndarray, repl: np.ndarray | None, bm: BatchMap, n_heads: int = 1):
    """DESIGN.md reading R1 (fp32 master band), one layer, ROTATE_ONLY maps, bf16 pool.  `pool` (uint8) and `master`
    (float32 [n_slots, n_heads*Dr]) are updated IN PLACE (rows do not move in this mode)."""
    assert pool.dtype == np.uint8 and master.dtype == np.float32 and pool.flags.c_contiguous and master.flags.c_contiguous
    inv = np.ascontiguousarray(inv_freq, dtype=np.float32)
    rp = _p(np.ascontiguousarray(repl)) if repl is not None else None
    for rm in bm.requests:
        s = rm.segs
        st = lib().ora_rotate_master_layer(C.c_int(pairing), C.c_int32(Dc), C.c_int32(Dr), C.c_int32(n_heads), C.c_int64(stride),
                                           _p(inv), _p(pool), _p(master), rp, C.c_int32(len(s)), _p(s.kind), _p(s.src),
                                           _p(s.dst), _p(s.len), _p(s.shift), _p(_i64(rm.slot_new)))
        assert st == OK, st

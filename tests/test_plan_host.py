"""Host-side tests of libleyline.so (no GPU): the C ABI exports what include/leyline.h declares, leyline_plan
agrees bit-exactly with the oracle's O1-O3 on thousands of tiny randomised cases and on the five BASELINE.json
configs, its error codes follow rule V, and the tile list with its load->store dependencies (rule M2) is a
correct schedule for the in-place move -- checked by executing the tiles on integer row labels under random
legal interleavings."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle as O
from helpers import list_splice
from parity import assert_plan_equal, oracle_plan
from paper_2606_01065_b200 import binding as B
from paper_2606_01065_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
MODES = [B.FRESH, B.INPLACE_MOVE, B.ROTATE_ONLY]


def test_abi_exports_every_declared_symbol():
    inc = os.path.join(ROOT, "include")
    text = "".join(open(os.path.join(inc, f)).read() for f in sorted(os.listdir(inc)) if f.endswith(".h"))
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = set(re.findall(r"\b(leyline_[a-z_0-9]+)\s*\(", text))
    assert {"leyline_plan", "leyline_splice", "leyline_rotate_inplace", "leyline_plan_destroy", "leyline_plan_prefetch",
            "leyline_cdc_chunk", "leyline_registry_insert", "leyline_registry_lookup"} <= names
    lib = ctypes.CDLL(B.LIB_PATH)
    for n in sorted(names):
        assert hasattr(lib, n), f"{n} declared in leyline.h but not exported"
    assert "sm_100a" in B.leyline_version()
    # ... and nothing else: the library is built with -fvisibility=hidden, only LEYLINE_API declarations are exported
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", B.LIB_PATH], check=True, capture_output=True, text=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln}
    assert {e for e in exported if e.startswith("leyline")} == names, sorted(exported ^ names)
    assert not [e for e in exported if not e.startswith("leyline") and not e.startswith("_")], exported


def test_enum_values_match_oracle_contract():
    assert (B.OK, B.E_INVALID, B.E_UNSORTED, B.E_OVERLAP, B.E_RANGE, B.E_NOFREE, B.E_UNSUPPORTED) == \
           (O.OK, O.E_INVALID, O.E_UNSORTED, O.E_OVERLAP, O.E_RANGE, O.E_NOFREE, O.E_UNSUPPORTED)
    assert (B.FRESH, B.INPLACE_MOVE, B.ROTATE_ONLY) == (O.FRESH, O.INPLACE_MOVE, O.ROTATE_ONLY)


def tiny_workload(rng, P=None, n_req=None, forget=False, dtype=synth.DT_BF16):
    P = int(rng.choice([1, 2, 4, 8, 16])) if P is None else P
    n_req = int(rng.integers(1, 4)) if n_req is None else n_req
    seq_lens = [int(rng.integers(0, 150)) for _ in range(n_req)]
    dirs = []
    for r, L in enumerate(seq_lens):
        k = int(rng.integers(0, 5))
        cuts = np.sort(rng.integers(0, L + 1, size=2 * k))
        for j in range(k):
            s, e = int(cuts[2 * j]), int(cuts[2 * j + 1])
            n = int(rng.integers(0, 2 * (e - s) + 3)) if rng.random() < 0.8 else 0
            sem = B.FORGET if (forget and rng.random() < 0.15) else B.AMORTIZE
            dirs.append((r, s, e, n, 0, sem))
    w = synth.Workload("tiny", 2, seq_lens, P, dtype=dtype, inv_freq=synth.rope_inv_freq(64), directives=dirs,
                       seed=int(rng.integers(1 << 30)), pool_factor=3.0, extra_pages=sum(d[3] for d in dirs) + 8)
    return w.finalize()


def test_layer_pairing_is_validated():
    w = tiny_workload(np.random.default_rng(4), P=4, n_req=1)

    def plan_with(lp):
        d, keep = B.make_desc(w.n_layers, w.latent_dim, w.rope_dim, w.page_size, w.dtype, w.pairing, w.row_bytes,
                              w.n_slots, w.inv_freq, layer_pairing=lp)
        return B.leyline_plan(d, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, w.directives, w.free_pages)

    plan_with([B.NEOX, B.INTERLEAVED]).close()
    with pytest.raises(B.LeylineError) as ei:
        plan_with([B.NEOX, 7])
    assert ei.value.status == B.E_INVALID
    with pytest.raises(ValueError):
        plan_with([B.NEOX])


def test_prefetch_without_a_device_fails_loudly_and_keeps_the_plan():
    """No CPU fallback: without a CUDA device the upload is refused with LEYLINE_E_CUDA; host queries still work."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("needs a box without a GPU")
    w = tiny_workload(np.random.default_rng(3), P=4, n_req=2)
    plan = make_plan(w, B.FRESH)
    with pytest.raises(B.LeylineError) as ei:
        plan.prefetch()
    assert ei.value.status == B.E_CUDA
    assert len(plan.new_seq_lens) == 2
    plan.close()


def make_plan(w, mode, n_layers=None):
    d, keep = B.make_desc(n_layers or w.n_layers, w.latent_dim, w.rope_dim, w.page_size, w.dtype, w.pairing,
                          w.row_bytes, w.n_slots, w.inv_freq, rope_heads=w.rope_heads)
    free = w.free_slots() if mode == B.ROTATE_ONLY else w.free_pages
    return B.leyline_plan(d, mode, w.seq_lens, w.pt_offsets, w.pages, w.directives, free)


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("block", range(8))
def test_plan_matches_oracle_randomised(mode, block):
    rng = np.random.default_rng(5000 + 100 * mode + block)
    for _ in range(150):
        w = tiny_workload(rng, forget=True)
        bm = oracle_plan(w, mode)
        assert bm.status == O.OK
        with make_plan(w, mode) as plan:
            assert_plan_equal(plan, bm, mode)
            check_tiles_cover(plan, bm, w, mode)


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("cfg", [1, 2, 3, "3m", 4, 5])
def test_plan_matches_oracle_on_baseline_configs(mode, cfg):
    w = synth.config(cfg, pool_factor=2.2)
    bm = oracle_plan(w, mode)
    with make_plan(w, mode) as plan:
        assert_plan_equal(plan, bm, mode)
        check_tiles_cover(plan, bm, w, mode)
        i = plan.info
        E, W = w.elem_bytes, w.row_elems
        if mode != B.ROTATE_ONLY:
            assert i.bytes_read == i.bytes_written == (i.rows_moved + i.rows_inserted) * W * E * w.n_layers
        if cfg == 3 and mode == B.FRESH:   # (103,936 + 320) x 61 rows, 14.65 GB read + written
            assert (i.rows_moved, i.rows_inserted, i.rows_rotated) == (103936, 320, 103936)
            assert i.bytes_read + i.bytes_written == 2 * (103936 + 320) * 1152 * 61
        if cfg == 4:
            shifts = [s[5] for s in plan.segments if s[1] == 0]
            assert sum(1 for r in range(64) if any(s[0] == r and s[1] == 0 and s[5] > 0 for s in plan.segments)) >= 8
            assert any(c < 0 for c in shifts)


def check_tiles_cover(plan, bm, w, mode):
    """Tiles are exactly the rows the mode must touch, each once, with the right source, shift and trig row."""
    tiles = plan.tiles
    shifts = plan.trig_shifts
    n_move = plan.info.n_move_tiles
    seen = {}
    for t_i, t in enumerate(tiles):
        is_repl = bool(t.flags & B.TILE_SRC_REPL)
        if mode == B.ROTATE_ONLY and not is_repl:     # a5 work items: the (row, pair column) units one block holds =
            assert 1 <= t.n_rows <= plan.info.rot_tile_rows     # 256 threads x 6 (bf16) / 4 (fp8) units in flight
            units = 1536 if w.elem_bytes == 2 else 1024
            assert (plan.info.rot_tile_rows * w.rope_heads * (w.rope_dim * w.elem_bytes // 32) <= units or plan.info.rot_tile_rows == 1
                    or plan.info.mover == 2)
        else:
            assert 1 <= t.n_rows <= plan.info.tile_rows <= 64
        assert is_repl == (t_i >= n_move)
        for q in range(t.n_rows):
            key = (t.request, "r" if is_repl else "o", t.src_pos + q)
            assert key not in seen
            seen[key] = (t.dst_pos + q, t.trig)
        assert t.dep_lo >= 0 and t.dep_hi < t_i
        if mode != B.INPLACE_MOVE:
            assert t.dep_hi < t.dep_lo
    want = {}
    for r, rm in enumerate(bm.requests):
        segs = rm.segs.as_tuples()
        k0P = 0
        if mode == B.FRESH:
            # rule M1: everything in front of the first directive that changes anything stays where it is; a FORGET
            # ends the search, no-ops do not count
            first = None
            for d in (d for d in w.directives if d[0] == r):
                if d[5] == B.FORGET:
                    break
                if d[2] > d[1] or d[3] > 0:
                    first = d[1]
                    break
            k0P = (first // w.page_size) * w.page_size if first is not None else rm.L_new
        ins_cursor = 0
        for (kind, src, dst, ln, sh) in segs:
            for q in range(ln):
                if kind == O.INSERT:
                    want[(r, "r", src + q)] = (dst + q, None)
                elif mode == B.FRESH and dst + q >= k0P:
                    want[(r, "o", src + q)] = (dst + q, sh)
                elif mode in (B.INPLACE_MOVE, B.ROTATE_ONLY) and sh != 0:
                    want[(r, "o", src + q)] = (dst + q, sh)
    assert set(seen) == set(want)
    for key, (dst, trig) in seen.items():
        wdst, wsh = want[key]
        if key[1] == "o":
            assert dst == wdst
            assert (trig == -1 and wsh == 0) or (trig >= 0 and shifts[trig] == wsh)
        else:
            assert trig == -1
            if mode != B.ROTATE_ONLY:
                assert dst == wdst


def test_trig_table_is_fp64_trig_rounded_once():
    w = synth.config(3, pool_factor=2.2)
    with make_plan(w, B.FRESH) as plan:
        sh, tab = plan.trig_shifts, plan.trig_table
        th = w.inv_freq.astype(np.float64)
        for g, c in enumerate(sh):
            # independent evaluation: exact integer-times-double product, numpy fp64 trig
            phi = float(c) * th
            np.testing.assert_array_equal(tab[g, 0], np.cos(phi).astype(np.float32))
            np.testing.assert_array_equal(tab[g, 1], np.sin(phi).astype(np.float32))


def test_error_codes_follow_rule_v():
    w = tiny_workload(np.random.default_rng(1), P=4, n_req=2)
    w.seq_lens = [40, 30]
    w.directives = []
    w.finalize()
    d, keep = B.make_desc(2, 512, 64, 4, 0, 0, 1152, w.n_slots, w.inv_freq)

    def status(dirs, mode=B.FRESH, free=None, desc=d):
        try:
            B.leyline_plan(desc, mode, w.seq_lens, w.pt_offsets, w.pages, dirs, w.free_pages if free is None else free).close()
            return B.OK
        except B.LeylineError as e:
            return e.status

    A = B.AMORTIZE
    cases = [
        ([], B.OK), ([(0, 5, 5, 0, 0, A)], B.OK), ([(0, 0, 40, 0, 0, A)], B.OK),
        ([(0, 5, 10, 1, 0, A), (0, 10, 12, 0, 0, A)], B.OK),                 # adjacent spans accepted
        ([(2, 0, 1, 0, 0, A)], B.E_RANGE), ([(-1, 0, 1, 0, 0, A)], B.E_RANGE),
        ([(0, -1, 1, 0, 0, A)], B.E_INVALID), ([(0, 5, 4, 0, 0, A)], B.E_INVALID),
        ([(0, 1, 2, -1, 0, A)], B.E_INVALID), ([(0, 1, 2, 0, -1, A)], B.E_INVALID), ([(0, 1, 2, 0, 0, 7)], B.E_INVALID),
        ([(0, 30, 41, 0, 0, A)], B.E_RANGE), ([(1, 0, 31, 0, 0, A)], B.E_RANGE),
        ([(1, 0, 1, 0, 0, A), (0, 0, 1, 0, 0, A)], B.E_UNSORTED),
        ([(0, 10, 12, 0, 0, A), (0, 5, 6, 0, 0, A)], B.E_UNSORTED),
        ([(0, 5, 10, 0, 0, A), (0, 9, 12, 0, 0, A)], B.E_OVERLAP),
    ]
    for dirs, want in cases:
        assert status(dirs) == want, dirs
        assert O.validate(w.seq_lens, dirs) == want, dirs                      # the oracle applies the same rule
    assert status([(0, 0, 0, 400, 0, A)], free=w.free_pages[:3]) == B.E_NOFREE
    assert status([(0, 0, 0, 5, 0, A)], mode=B.ROTATE_ONLY, free=w.free_slots()[:4]) == B.E_NOFREE
    bad, k2 = B.make_desc(2, 512, 64, 3, 0, 0, 1152, w.n_slots, w.inv_freq)        # page size not a power of two
    assert status([], desc=bad) == B.E_INVALID
    bad, k3 = B.make_desc(2, 512, 63, 4, 0, 0, 1152, w.n_slots, w.inv_freq)        # odd rope_dim
    assert status([], desc=bad) == B.E_INVALID
    bad, k4 = B.make_desc(2, 500, 64, 4, 0, 0, 1136, w.n_slots, w.inv_freq)        # latent bytes not 16-byte chunks
    assert status([], desc=bad) == B.E_UNSUPPORTED
    bad, k5 = B.make_desc(2, 512, 64, 4, 0, 0, 1152, 8, w.inv_freq)                # page ids beyond the pool
    assert status([]) == B.OK and status([], desc=bad) == B.E_RANGE
    # directive.reserved_ must be 0 (leyline.h)
    packed = B.pack_directives([(0, 5, 6, 0, 0, A)])
    packed["reserved_"] = 7
    assert status(packed) == B.E_INVALID
    # a free id outside the pool is RANGE and wins over the alias rule; NOFREE wins over both
    assert status([(1, 28, 28, 5, 0, A)], free=np.array([w.pool_pages + 3, w.pages[0]], np.int32)) == B.E_RANGE   # consumes 2
    assert status([(1, 28, 28, 5, 0, A)], free=np.array([w.free_pages[0], w.pages[0]], np.int32)) == B.E_ALIAS
    assert status([(0, 0, 0, 400, 0, A)], free=np.array([w.pages[0]], np.int32)) == B.E_NOFREE


def test_alias_rule_refuses_plans_that_would_overwrite_live_kv():
    """leyline.h, LEYLINE_E_ALIAS: a consumed free id that is live or handed out twice, and -- for the modes that write
    a request's own pages -- a page listed by two requests of which one is edited.  Hand-built tables, P = 4."""
    inv = synth.rope_inv_freq(64)
    d, keep = B.make_desc(1, 512, 64, 4, 0, 0, 1152, 64 * 4, inv)
    seq, pto, pages = [10, 6], [0, 3, 5], np.array([0, 1, 2, 3, 4], np.int32)
    A = B.AMORTIZE

    def status(mode, dirs, free, pages=pages, pto=pto, seq=seq):
        try:
            B.leyline_plan(d, mode, seq, pto, pages, dirs, np.asarray(free, np.int32)).close()
            return B.OK
        except B.LeylineError as e:
            return e.status

    grow = [(0, 2, 2, 9, 0, A)]                                   # request 0 grows by 9 rows: FRESH consumes 4 pages
    assert status(B.FRESH, grow, [10, 11, 12, 13, 14]) == B.OK
    assert status(B.FRESH, grow, [10, 1, 12, 13, 14]) == B.E_ALIAS        # page 1 is a live page of request 0
    assert status(B.FRESH, grow, [10, 4, 12, 13, 14]) == B.E_ALIAS        # page 4 is a live page of request 1
    assert status(B.FRESH, grow, [10, 11, 11, 13, 14]) == B.E_ALIAS       # handed out twice
    assert status(B.FRESH, grow, [10, 11, 12, 13, 1]) == B.E_ALIAS        # every CONSUMED id is checked (5 are) ...
    assert status(B.FRESH, grow, [10, 11, 12, 13, 14, 1]) == B.OK         # ... ids that are not consumed are not
    assert status(B.INPLACE_MOVE, grow, [10, 3]) == B.E_ALIAS            # growth by 2 pages: the 2nd is request 1's
    assert status(B.INPLACE_MOVE, grow, [10, 11]) == B.OK
    # ROTATE_ONLY consumes free SLOTS: slot 13 sits in live page 3
    assert status(B.ROTATE_ONLY, grow, [40, 41, 42, 43, 44, 45, 46, 47, 13]) == B.E_ALIAS
    assert status(B.ROTATE_ONLY, grow, [40, 41, 42, 43, 44, 45, 46, 47, 40]) == B.E_ALIAS
    assert status(B.ROTATE_ONLY, grow, [40, 41, 42, 43, 44, 45, 46, 47, 48]) == B.OK
    # the same in a pool of 2^22 slots, where the planner finds duplicates by sorting the few ids instead of a bit per slot
    big, keep_big = B.make_desc(1, 512, 64, 4, 0, 0, 1152, 1 << 22, inv)
    for free, want in (([40, 41, 42, 43, 44, 45, 46, 47, 40], B.E_ALIAS), ([40, 41, 42, 43, 4000000, 45, 46, 47, 4000000], B.E_ALIAS),
                       ([40, 41, 42, 43, 44, 45, 46, 47, 4000000], B.OK)):
        try:
            B.leyline_plan(big, B.ROTATE_ONLY, seq, pto, pages, grow, np.asarray(free, np.int32)).close()
            got = B.OK
        except B.LeylineError as e:
            got = e.status
        assert got == want
    del keep_big
    # a page shared by two requests (a common prefix): fine for FRESH, which never writes a request's own pages ...
    shared = np.array([0, 1, 2, 0, 4], np.int32)
    edit1 = [(1, 5, 6, 0, 0, A)]
    assert status(B.FRESH, edit1, [10, 11], pages=shared) == B.OK
    # ... refused for the in-place modes when either owner is edited, accepted when nobody is
    assert status(B.INPLACE_MOVE, edit1, [10], pages=shared) == B.E_ALIAS
    assert status(B.ROTATE_ONLY, edit1, [40], pages=shared) == B.E_ALIAS
    assert status(B.INPLACE_MOVE, [(0, 9, 10, 0, 0, A)], [10], pages=shared) == B.E_ALIAS
    assert status(B.INPLACE_MOVE, [], [10], pages=shared) == B.OK
    assert status(B.INPLACE_MOVE, edit1, [10], pages=np.array([0, 1, 2, 3, 3], np.int32)) == B.E_ALIAS   # twice in one request
    # leyline_tuning.skip_alias_check = 1: the caller vouches for its tables, nothing is checked (and nothing is cheaper)
    B.leyline_set_tuning(skip_alias_check=1)
    try:
        assert status(B.FRESH, grow, [10, 1, 12, 13, 14]) == B.OK
        assert status(B.INPLACE_MOVE, edit1, [10], pages=shared) == B.OK
        assert status(B.ROTATE_ONLY, grow, [40, 41, 42, 43, 44, 45, 46, 47, 40]) == B.OK
    finally:
        B.leyline_set_tuning()
    del keep


def test_page_table_rows_must_be_exactly_as_long_as_the_request():
    """leyline.h: a row longer than ceil(L/P) is refused -- its surplus pages would be neither kept nor released."""
    inv = synth.rope_inv_freq(64)
    d, keep = B.make_desc(1, 512, 64, 4, 0, 0, 1152, 64 * 4, inv)
    for mode in MODES:
        with pytest.raises(B.LeylineError) as ei:
            B.leyline_plan(d, mode, [10], [0, 5], [0, 1, 2, 3, 4], [], [9])
        assert ei.value.status == B.E_INVALID
        with pytest.raises(B.LeylineError) as ei:
            B.leyline_plan(d, mode, [10], [0, 2], [0, 1], [], [9])
        assert ei.value.status == B.E_INVALID
        B.leyline_plan(d, mode, [10], [0, 3], [0, 1, 2], [], [9]).close()
    del keep


def test_noop_and_forget_only_requests_launch_nothing():
    """PAPER.md:102 and rule M1: a request whose directives change nothing (no-ops) or only truncate it (FORGET before any
    edit) produces no tile in any mode, consumes no free id, and FRESH keeps its pages."""
    inv = synth.rope_inv_freq(64)
    d, keep = B.make_desc(1, 512, 64, 4, 0, 0, 1152, 64 * 4, inv)
    pages = np.arange(6, dtype=np.int32) + 10
    for mode in MODES:
        free = np.arange(40, 60, dtype=np.int32)
        for dirs, L_new, n_pages in (([(0, 3, 3, 0, 0, B.AMORTIZE), (0, 9, 9, 0, 0, B.AMORTIZE)], 22, 6),
                                     ([(0, 9, 9, 0, 0, B.FORGET)], 9, 3), ([(0, 1, 1, 0, 0, B.AMORTIZE), (0, 8, 12, 5, 0, B.FORGET)], 8, 2)):
            with B.leyline_plan(d, mode, [22], [0, 6], pages, dirs, free) as plan:
                i = plan.info
                assert (i.n_tiles, i.n_free_consumed, i.rows_moved, i.rows_inserted, i.rows_rotated) == (0, 0, 0, 0, 0)
                assert plan.new_seq_lens[0] == L_new
                if mode != B.ROTATE_ONLY:
                    assert list(plan.new_pages) == list(pages[:n_pages]) and list(plan.released) == list(pages[n_pages:])
                else:
                    assert list(plan.released) == [int(pages[t // 4]) * 4 + t % 4 for t in range(L_new, 22)]
    del keep


def test_plan_ex_takes_its_tuning_per_call():
    """leyline.h: leyline_plan_ex never looks at the process-wide tuning of leyline_set_tuning, and the other way round."""
    w = synth.config(2, pool_factor=2.2)
    d, keep = B.make_desc(w.n_layers, w.latent_dim, w.rope_dim, w.page_size, w.dtype, w.pairing, w.row_bytes, w.n_slots, w.inv_freq)
    args = (d, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, w.directives, w.free_pages)
    with B.leyline_plan_ex(*args) as p0, B.leyline_plan_ex(*args, B.Tuning(1, 7, 0, 0, 0, 0, 0, 0, 0)) as p1:
        assert (p0.info.mover, p0.info.tile_rows) == (2, 32) and (p1.info.mover, p1.info.tile_rows) == (1, 7)
    B.leyline_set_tuning(kernel=1, tile_rows=5)
    try:
        with B.leyline_plan_ex(*args) as p0, B.leyline_plan(*args[:7]) as p2:
            assert (p0.info.mover, p0.info.tile_rows) == (2, 32)           # plan_ex: defaults, whatever the global says
            assert (p2.info.mover, p2.info.tile_rows) == (1, 5)            # leyline_plan: the process-wide default
    finally:
        B.leyline_set_tuning()
    with pytest.raises(B.LeylineError) as ei:
        B.leyline_plan_ex(*args, B.Tuning(9, 0, 0, 0, 0, 0, 0, 0, 0))
    assert ei.value.status == B.E_INVALID
    del keep


# ----------------------------------------------------------------------------- rule M2 as a schedule

def simulate_inplace(plan, w, rng):
    """Execute the plan's tiles on integer row labels: a tile's LOAD may happen at any time, its STORE only after
    its own load and the loads of tiles [dep_lo, dep_hi]; insert tiles are part of the same schedule (they read the
    replacement buffer and wait for the move tiles that still read their destination rows).  The interleaving is a
    random legal one.  Returns the pool of labels."""
    P = w.page_size
    pool = np.full(w.n_slots, -1, np.int64)
    for r, L in enumerate(w.seq_lens):
        row = w.pages[w.pt_offsets[r]:w.pt_offsets[r + 1]]
        t = np.arange(L)
        pool[row[t // P].astype(np.int64) * P + t % P] = r * 10 ** 6 + t            # label = (request, old position)
    new_pages, off = plan.new_pages, plan.new_pt_offsets
    tiles = plan.tiles
    n_move = plan.info.n_move_tiles

    def src_slots(t):
        row = w.pages[w.pt_offsets[t.request]:w.pt_offsets[t.request + 1]]
        p = t.src_pos + np.arange(t.n_rows)
        return row[p // P].astype(np.int64) * P + p % P

    def dst_slots(t):
        row = new_pages[off[t.request]:off[t.request + 1]]
        p = t.dst_pos + np.arange(t.n_rows)
        return row[p // P].astype(np.int64) * P + p % P

    loaded, stored, regs = set(), set(), {}
    pending = list(range(len(tiles)))
    while len(stored) < len(tiles):
        ready = []
        for i in pending:
            if i not in loaded:
                ready.append(("L", i))
            elif all(d in loaded for d in range(tiles[i].dep_lo, tiles[i].dep_hi + 1)):
                ready.append(("S", i))
        # bias towards stores so that missing dependencies actually bite
        stores = [x for x in ready if x[0] == "S"]
        op, i = stores[int(rng.integers(len(stores)))] if stores and rng.random() < 0.7 else ready[int(rng.integers(len(ready)))]
        if op == "L":
            t = tiles[i]
            if i >= n_move:      # label = -(req, repl row) - 2
                regs[i] = -(t.request * 10 ** 6 + t.src_pos + np.arange(t.n_rows)) - 2
            else:
                regs[i] = pool[src_slots(t)].copy()
            loaded.add(i)
        else:
            pool[dst_slots(tiles[i])] = regs.pop(i)
            stored.add(i)
            pending.remove(i)
    return pool


@pytest.mark.parametrize("seed", range(60))
def test_inplace_tiles_are_a_correct_schedule(seed):
    rng = np.random.default_rng(9000 + seed)
    w = tiny_workload(rng, P=int(rng.choice([1, 2, 4, 8])))
    B.leyline_set_tuning(tile_rows=int(rng.choice([1, 2, 3, 5, 8, 32])))
    try:
        plan = make_plan(w, B.INPLACE_MOVE)
    finally:
        B.leyline_set_tuning()
    with plan:
        pool = simulate_inplace(plan, w, rng)
        P = w.page_size
        new_pages, off = plan.new_pages, plan.new_pt_offsets
        for r, L in enumerate(w.seq_lens):
            dirs = [(d[1], d[2], d[3], d[4]) for d in w.directives if d[0] == r]
            want = list_splice(L, dirs)                                   # literal Python list slicing
            row = new_pages[off[r]:off[r + 1]]
            assert plan.new_seq_lens[r] == len(want)
            for tpos, (kind, i) in enumerate(want):
                got = pool[int(row[tpos // P]) * P + tpos % P]
                assert got == (r * 10 ** 6 + i if kind == "o" else -(r * 10 ** 6 + i) - 2), (r, tpos, kind, i, got)


def test_heads_descriptor_rules():
    """rope_heads: 0 reads as 1; row = latent + heads * rope_dim; a head must be an even number of 16-byte chunks;
    the row kernel (tuning.kernel = 1) only takes one head of 2^k chunks."""
    w = synth.Workload("h", 1, [100], 16, latent_dim=0, rope_dim=128, rope_heads=8, inv_freq=synth.rope_inv_freq(128, 5e5),
                       directives=[(0, 10, 20, 3, 0, 0)], seed=1, pool_factor=3.0, extra_pages=4).finalize()
    for mode in MODES:
        bm = oracle_plan(w, mode)
        with make_plan(w, mode) as plan:
            assert_plan_equal(plan, bm, mode)
            i = plan.info
            assert i.mover == 2                                   # several heads: the bulk mover
            row = 8 * 128 * 2
            if mode == B.ROTATE_ONLY:
                assert i.bytes_read == (i.rows_rotated * row + i.rows_inserted * row) * w.n_layers
                assert i.rot_tile_rows == i.tile_rows == 24   # full-width K: the rotation runs on the bulk mover, 48 KB tiles
            else:
                assert i.bytes_read == (i.rows_moved + i.rows_inserted) * row * w.n_layers
    inv = synth.rope_inv_freq(128, 5e5)
    # stride must cover all heads
    d, k = B.make_desc(1, 0, 128, 16, 0, 0, 128 * 2, w.n_slots, inv, rope_heads=8)
    with pytest.raises(B.LeylineError) as e:
        B.leyline_plan(d, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, w.directives, w.free_pages)
    assert e.value.status == 1
    # a head of one 16-byte chunk (8 bf16 elements) cannot be split into two half-chunks
    d, k = B.make_desc(1, 0, 8, 16, 0, 1, 16, w.n_slots, synth.rope_inv_freq(8), rope_heads=1)
    with pytest.raises(B.LeylineError) as e:
        B.leyline_plan(d, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, w.directives, w.free_pages)
    assert e.value.status == 6
    # forced row kernel on a multi-head band
    B.leyline_set_tuning(kernel=1)
    try:
        d, k = B.make_desc(1, 0, 128, 16, 0, 0, 2048, w.n_slots, inv, rope_heads=8)
        with pytest.raises(B.LeylineError) as e:
            B.leyline_plan(d, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, w.directives, w.free_pages)
        assert e.value.status == 6
    finally:
        B.leyline_set_tuning()
    # rope_heads = 0 is the MLA default
    d, k = B.make_desc(1, 512, 64, 16, 0, 0, 1152, w.n_slots, synth.rope_inv_freq(64), rope_heads=0)
    with B.leyline_plan(d, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, w.directives, w.free_pages) as plan:
        assert plan.info.bytes_read == (plan.info.rows_moved + plan.info.rows_inserted) * 1152


def test_headers_are_plain_c_and_the_abi_links_from_c(tmp_path):
    """The boundary is a C ABI: both headers compile as C99 with -Wall -Werror -pedantic, and a C program linked
    against libleyline.so plans the paper's worked example (5 + 57 + 9 tokens, 11-token stub: Delta = -46, L 71 -> 25;
    PAPER.md:155) and prints what the getters return.  Host only; no device call is made."""
    import subprocess
    src = tmp_path / "abi.c"
    src.write_text(r'''
#include <stdio.h>
#include "leyline.h"
#include "leyline_cdc.h"
int main(void) {
    float inv_freq[32];
    int i;
    for (i = 0; i < 32; ++i) inv_freq[i] = 1.0f / (float)(i + 1);
    leyline_cache_desc c = {0};
    c.n_layers = 2; c.latent_dim = 512; c.rope_dim = 64; c.page_size = 1; c.dtype = LEYLINE_BF16;
    c.pairing = LEYLINE_ROPE_NEOX; c.rope_heads = 1; c.row_stride_bytes = 1152; c.pool_slots = 256; c.inv_freq = inv_freq;
    int64_t seq_lens[1] = {71}, pt_offsets[2] = {0, 71}, new_len[1] = {0};
    int32_t pages[71], free_ids[64];
    for (i = 0; i < 71; ++i) pages[i] = i;
    for (i = 0; i < 64; ++i) free_ids[i] = 100 + i;
    leyline_directive d = {0};
    d.request = 0; d.start = 5; d.end = 62; d.repl_len = 11; d.repl_row = 0; d.semantic = LEYLINE_AMORTIZE;
    leyline_plan_t* plan = 0;
    leyline_status st = leyline_plan(&c, LEYLINE_FRESH, 1, seq_lens, pt_offsets, pages, 1, &d, free_ids, 64, &plan);
    if (st != LEYLINE_OK) { printf("plan failed: %s\n", leyline_strerror(st)); return 1; }
    leyline_plan_info info;
    leyline_plan_get_info(plan, &info);
    leyline_plan_new_seq_lens(plan, new_len);
    printf("L_new=%lld consumed=%lld released=%lld rows_moved=%lld rows_inserted=%lld version=%s\n", (long long)new_len[0],
           (long long)info.n_free_consumed, (long long)info.n_released, (long long)info.rows_moved,
           (long long)info.rows_inserted, leyline_version());
    leyline_plan_destroy(plan);
    return 0;
}
''')
    exe = tmp_path / "abi"
    inc = os.path.join(ROOT, "include")
    libdir = os.path.dirname(B.LIB_PATH)
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", inc, str(src), "-o", str(exe),
                    "-L", libdir, "-lleyline", f"-Wl,-rpath,{libdir}"], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout
    # tokens 5..61 removed, 11 inserted, 9 downstream tokens moved by -46; token-level FRESH keeps slots [0, 5)
    assert "L_new=25 consumed=20 released=66 rows_moved=9 rows_inserted=11" in out, out
    assert "sm_100a" in out


def test_tma_rotate_tiles_are_whole_boxes_inside_one_page():
    """leyline_tuning.rotate_kernel = 2 (k_rotate_band_tma): ROTATE_ONLY tiles are at most min(page, 64) rows, never
    straddle a page of the OLD table (so their rows are consecutive slots: one 2-D box), and every interior tile of a
    segment is a whole box.  Pages below 16 rows and wide bands fall back to the other kernels."""
    for P, box in ((16, 16), (64, 64), (256, 64)):
        w = synth.Workload("t", 1, [5000, 777], P, inv_freq=synth.yarn_inv_freq(),
                           directives=[(0, 300, 1100, 77, 0, 0), (0, 3000, 3001, 600, 0, 0), (1, 770, 777, 0, 0, 0)],
                           seed=2, pool_factor=3.0, extra_pages=4).finalize()
        B.leyline_set_tuning(rotate_kernel=2)
        try:
            plan = make_plan(w, B.ROTATE_ONLY)
        finally:
            B.leyline_set_tuning()
        with plan:
            assert plan.info.mover == 3 and plan.info.rot_tile_rows == box
            bm = oracle_plan(w, B.ROTATE_ONLY)
            assert_plan_equal(plan, bm, B.ROTATE_ONLY)
            check_tiles_cover(plan, bm, w, B.ROTATE_ONLY)
            rot = plan.tiles[:plan.info.n_move_tiles]
            for t in rot:
                assert 1 <= t.n_rows <= box and t.src_pos // P == (t.src_pos + t.n_rows - 1) // P
                assert t.src_pos // box == (t.src_pos + t.n_rows - 1) // box          # aligned to the box grid
            assert sum(1 for t in rot if t.n_rows == box) >= len(rot) - 2 * len(plan.segments)
    w = synth.config(1, pool_factor=2.5)                                              # token-level slots: no boxes
    B.leyline_set_tuning(rotate_kernel=2)
    try:
        with make_plan(w, B.ROTATE_ONLY) as plan:
            assert plan.info.mover == 1
        with make_plan(synth.config("gqa", pool_factor=2.0), B.ROTATE_ONLY) as plan:
            assert plan.info.mover == 2                                               # wide band: whole rows on the bulk mover
    finally:
        B.leyline_set_tuning()


def test_flat_rotate_kernel_is_chosen_by_the_planner_for_short_segments():
    """k_rotate_band_flat (plan.info.mover == 4) is a host decision: auto picks it when packing the rotate tiles into full
    block passes saves a fifth of the work items (the paper's App. B shape: 228 tiles -> 62 passes), keeps k_rotate_band on
    long segments, never overrides the wide-band (bulk) or TMA choice; rotate_kernel = 1 / 3 force either; the tiles,
    segments and maps of the plan are the same whichever kernel runs them."""
    appb, cfg2 = synth.config("appB", pool_factor=2.0), synth.config(2, pool_factor=1.25)
    with make_plan(appb, B.ROTATE_ONLY) as plan:
        assert plan.info.mover == 4 and plan.info.rot_tile_rows == 384
        n_passes = -(-int(plan.info.rows_rotated) // 384)
        assert n_passes * 5 <= int(plan.info.n_move_tiles) * 4
        auto_tiles = [(t.src_pos, t.dst_pos, t.n_rows, t.trig) for t in plan.tiles]
    with make_plan(cfg2, B.ROTATE_ONLY) as plan:
        assert plan.info.mover == 1
    with make_plan(synth.config(5, pool_factor=1.25), B.ROTATE_ONLY) as plan:
        assert plan.info.mover == 1 and plan.info.rot_tile_rows == 512
    for rk, mover in ((1, 1), (3, 4)):
        B.leyline_set_tuning(rotate_kernel=rk)
        try:
            with make_plan(appb, B.ROTATE_ONLY) as plan:
                assert plan.info.mover == mover
                assert [(t.src_pos, t.dst_pos, t.n_rows, t.trig) for t in plan.tiles] == auto_tiles
                assert_plan_equal(plan, oracle_plan(appb, B.ROTATE_ONLY), B.ROTATE_ONLY)
            with make_plan(cfg2, B.ROTATE_ONLY) as plan:
                assert plan.info.mover == mover
            with make_plan(synth.config("gqa", pool_factor=2.0), B.ROTATE_ONLY) as plan:
                assert plan.info.mover == 2                                           # wide band stays on the bulk mover
            with make_plan(synth.config(2, pool_factor=2.0), B.FRESH) as plan:
                assert plan.info.mover == 2                                           # not a ROTATE_ONLY plan: untouched
        finally:
            B.leyline_set_tuning()
    with pytest.raises(B.LeylineError):
        B.leyline_set_tuning(rotate_kernel=4)
    B.leyline_set_tuning()

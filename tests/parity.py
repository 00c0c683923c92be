"""Test-only: compare the CUDA library (through the binding) with the CPU oracle on the same seeded inputs.

The bar (BASELINE.json north_star):
  * bit-exact: new sequence lengths, page-table rows, token-level slot list, released list, free ids consumed,
    segments, every pool byte outside rotated K_pe bands (moved latent, C = 0 segments, replacement rows, and
    every byte the mode never writes -- other requests, free pool, prefix pages, released pages);
  * rotated bf16 K_pe: ordinal distance <= 2 bf16 ulp for EVERY element (north_star's bound as written, +0 == -0).
    Round 1 needed a cancellation floor |g - o| <= 2^-20 * rho here (plain fp32 arithmetic has an absolute error of
    ~2^-24 * rho, which is many bf16 steps where a cos - b sin cancels: about one element in 10^6); since round 2 the
    kernels redo such outputs with compensated fp32 arithmetic and the floor is gone.  Measured: never more than 1;
  * rotated fp8 K_pe: ordinal distance <= 1 e4m3 code (+0 == -0).
"""
from __future__ import annotations

import numpy as np

import oracle as O
from paper_2606_01065_b200 import synth


def oracle_plan(w: synth.Workload, mode: int) -> O.BatchMap:
    free = w.free_slots() if mode == O.ROTATE_ONLY else w.free_pages
    return O.plan_batch(mode, w.page_size, w.seq_lens, w.pt_offsets, w.pages, w.directives, free)


def assert_plan_equal(plan, bm: O.BatchMap, mode: int):
    """Library plan (binding.Plan) vs oracle BatchMap: everything integer, bit-exact."""
    assert bm.status == O.OK
    np.testing.assert_array_equal(plan.new_seq_lens, bm.new_seq_lens)
    assert plan.info.n_free_consumed == bm.n_consumed
    np.testing.assert_array_equal(plan.released, bm.released)
    segs = []
    for r, rm in enumerate(bm.requests):
        segs += [(r, k, s, d, n, c) for (k, s, d, n, c) in rm.segs.as_tuples()]
    assert plan.segments == segs
    np.testing.assert_array_equal(plan.forget_trim, [rm.segs.forget_trim for rm in bm.requests])
    if mode != O.ROTATE_ONLY:
        want = np.concatenate([rm.new_pages for rm in bm.requests]) if bm.requests else np.zeros(0, np.int32)
        np.testing.assert_array_equal(plan.new_pages, want)
        off = np.concatenate([[0], np.cumsum([len(rm.new_pages) for rm in bm.requests])])
        np.testing.assert_array_equal(plan.new_pt_offsets, off)
    off = np.concatenate([[0], np.cumsum([rm.L_new for rm in bm.requests])])
    np.testing.assert_array_equal(plan.slot_offsets, off)


def oracle_slot_list(bm: O.BatchMap) -> np.ndarray:
    return np.concatenate([rm.slot_new for rm in bm.requests]).astype(np.int32) if bm.requests else np.zeros(0, np.int32)


def _bf16_ord(bits: np.ndarray) -> np.ndarray:
    b = bits.astype(np.int32)
    mag = b & 0x7FFF
    return np.where(b & 0x8000, -mag, mag)


def _bf16_val(bits: np.ndarray) -> np.ndarray:
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def _e4m3_ord(b: np.ndarray) -> np.ndarray:
    v = b.astype(np.int32)
    mag = v & 0x7F
    return np.where(v & 0x80, -mag, mag)


def rotated_rows(w: synth.Workload, bm: O.BatchMap, mode: int):
    """(new slot, old slot) of every row whose K_pe band is rotated (KEEP segments with shift != 0 that the mode
    processes)."""
    new_s, old_s = [], []
    for rm in bm.requests:
        for (kind, src, dst, ln, sh) in rm.segs.as_tuples():
            if kind == O.KEEP and sh != 0:
                new_s.append(rm.slot_new[dst:dst + ln])
                old_s.append(rm.slot_old[src:src + ln])
    if not new_s:
        return np.zeros(0, np.int64), np.zeros(0, np.int64)
    return np.concatenate(new_s).astype(np.int64), np.concatenate(old_s).astype(np.int64)


def compare_layer(w: synth.Workload, bm: O.BatchMap, mode: int, old_pool: np.ndarray, gpu_pool: np.ndarray,
                  repl: np.ndarray, scale: float = 1.0, layer: int = 0, inserts_prefilled: bool = False) -> dict:
    """One layer, whole pool.  old_pool / gpu_pool / repl: flat uint8.  Asserts the bar and returns statistics."""
    stride = w.row_bytes
    E = w.elem_bytes
    pairing = w.pairing_of(layer)
    if repl is None:                      # the oracle always copies the replacement rows; they are masked out below
        repl = np.zeros(max(w.n_repl_rows, 1) * stride, np.uint8)
    want = O.splice_layer(w.dtype, pairing, w.latent_dim, w.rope_dim, stride, w.inv_freq, scale, old_pool, repl, bm,
                          n_heads=w.rope_heads)
    g = gpu_pool.reshape(-1, stride)
    o = want.reshape(-1, stride)
    if inserts_prefilled:
        # layer_repl = NULL: the replacement slots belong to the caller's prefill and must not have been written
        oo = old_pool.reshape(-1, stride)
        for rm in bm.requests:
            for (kind, src, dst, ln, sh) in rm.segs.as_tuples():
                if kind == O.INSERT:
                    s_ins = rm.slot_new[dst:dst + ln].astype(np.int64)
                    o[s_ins] = oo[s_ins]
    new_s, old_s = rotated_rows(w, bm, mode)
    band0 = w.latent_dim * E
    # 1. everything outside rotated bands: bit-exact over the whole pool
    neq = g != o
    if len(new_s):
        neq[new_s, band0:] = False
    assert not neq.any(), f"layer {layer}: {int(neq.sum())} bytes differ outside rotated K_pe bands (first rows {np.unique(np.nonzero(neq)[0])[:8]})"
    del neq
    stats = {"rotated_elems": 0, "max_ord": 0, "frac_equal": 1.0, "n_floor": 0}
    if not len(new_s):
        return stats
    gb = np.ascontiguousarray(g[new_s, band0:])
    ob = np.ascontiguousarray(o[new_s, band0:])
    if w.dtype == synth.DT_BF16:
        gbits, obits = gb.view(np.uint16), ob.view(np.uint16)
        dist = np.abs(_bf16_ord(gbits) - _bf16_ord(obits))
        n_floor = 0                    # kept in the statistics: the cancellation floor of round 1 no longer exists
        assert dist.max() <= 2, (f"layer {layer}: {int((dist > 2).sum())} rotated bf16 elements beyond 2 ulp "
                                 f"(max ordinal distance {int(dist.max())})")
        stats.update(rotated_elems=int(dist.size), max_ord=int(dist.max()), frac_equal=float((dist == 0).mean()),
                     n_floor=n_floor)
    else:
        dist = np.abs(_e4m3_ord(gb) - _e4m3_ord(ob))
        assert dist.max() <= 1, f"fp8 rotated K_pe: max ordinal distance {int(dist.max())} > 1"
        stats.update(rotated_elems=int(dist.size), max_ord=int(dist.max()), frac_equal=float((dist == 0).mean()))
    return stats


_PINNED = {"bufs": [], "cap": 0}


def _pinned_buffers(nbytes: int, count: int):
    """`count` pinned host buffers of at least `nbytes` bytes, kept from test to test (page-locking costs about as much
    as the copies it speeds up, so it is done once per size class, grow-only)."""
    import torch
    if _PINNED["cap"] < nbytes or len(_PINNED["bufs"]) < count:
        _PINNED["bufs"] = []          # drop the old arena before pinning a larger one
        _PINNED["cap"] = 0
        _PINNED["bufs"] = [torch.empty(nbytes, dtype=torch.uint8, pin_memory=True) for _ in range(count)]
        _PINNED["cap"] = nbytes
    return _PINNED["bufs"][:count]


def compare_all_layers(w: synth.Workload, bm: O.BatchMap, mode: int, cache, layers=None, inserts_prefilled: bool = False,
                       checksums=None, max_workers: int | None = None) -> list:
    """Every layer of a device cache against the oracle, whole pool, one layer at a time (SURVEY.md section 7 "never hold
    a whole cache on the host").  The pristine layer is REGENERATED from its seed into a device scratch buffer (the
    generator is counter-based and seeded per layer, so this reproduces the bytes the splice started from; `checksums`,
    taken before the splice, prove it), so in-place modes need no host snapshot of the cache.  Layers cross PCIe through
    a small ring of pinned bounce buffers (a pageable `.cpu()` runs at ~2 GB/s on the GPU box, pinned at ~55 GB/s); the
    oracle (GIL-free C) and the numpy comparisons of different layers run on a thread pool, sized to the host's cores
    and free memory."""
    import os
    import threading
    from concurrent.futures import ThreadPoolExecutor

    import psutil
    import torch
    layers = list(range(cache.n_layers)) if layers is None else list(layers)
    per_layer = 7 * w.layer_bytes + 1
    fit = int(psutil.virtual_memory().available * 0.6 // per_layer)
    nw = max(1, min(os.cpu_count() or 1, 16, fit, len(layers)))
    if max_workers:
        nw = min(nw, max_workers)
    scratch = torch.empty(w.layer_bytes, dtype=torch.uint8, device=cache.device)
    n_sets = min(len(layers), 3 if w.layer_bytes <= (1 << 30) else 2)    # pinning costs time too: fewer, when a layer is > 1 GiB
    pins = _pinned_buffers(w.layer_bytes, 2 * n_sets)
    free_sets = list(range(n_sets))
    set_lock = threading.Condition()
    gate = threading.Semaphore(nw + 1)            # layers resident on the host at once
    stats = [None] * len(layers)

    def work(i, l, k, landed, repl, scale):
        try:
            landed.synchronize()                   # both copies of this layer have reached the pinned buffers
            old = pins[2 * k][: w.layer_bytes].numpy().copy()
            new = pins[2 * k + 1][: w.layer_bytes].numpy().copy()
        finally:
            with set_lock:
                free_sets.append(k)
                set_lock.notify()
        try:
            stats[i] = compare_layer(w, bm, mode, old, new, repl, scale, layer=l, inserts_prefilled=inserts_prefilled)
        finally:
            gate.release()

    with ThreadPoolExecutor(max_workers=nw) as ex:
        futs = []
        for i, l in enumerate(layers):
            gate.acquire()
            with set_lock:
                while not free_sets:
                    set_lock.wait()
                k = free_sets.pop()
            scale = synth.fill_layer_(scratch, w, cache.layer_ids[l])
            assert scale == cache.scales[l]
            if checksums is not None:
                assert int(layer_checksum(scratch)) == checksums[l], f"layer {l}: regenerated bytes differ from the cache's"
            pins[2 * k][: w.layer_bytes].copy_(scratch, non_blocking=True)
            pins[2 * k + 1][: w.layer_bytes].copy_(cache.pools[l], non_blocking=True)
            landed = torch.cuda.Event()
            landed.record()
            repl = None if inserts_prefilled else cache.repl[l].cpu().numpy()
            futs.append(ex.submit(work, i, l, k, landed, repl, scale))
        for f in futs:
            f.result()
    return stats


def layer_checksum(buf) -> int:
    """Order-independent 64-bit sum of a uint8 device tensor read as int64 words (a cheap identity check, not a hash)."""
    import torch
    n = buf.numel() // 8 * 8
    return int(buf[:n].view(torch.int64).sum().item()) + int(buf[n:].to(torch.int64).sum().item())

"""Device-memory plumbing around the binding: allocate a synthetic cache for a ``synth.Workload`` with torch,
build the descriptor, plan and launch.  No arithmetic of the method lives here, and nothing here touches
``oracle/``."""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B
from . import synth


class DeviceCache:
    """Per-layer pools ``[n_slots * row_bytes]`` uint8 on `device`, plus per-layer replacement rows.
    `layers` restricts which layers of the workload are materialised (layers are independent buffers)."""

    def __init__(self, w: synth.Workload, device="cuda:0", layers=None, fill=True, with_dst=False, host_resident=False):
        self.w = w
        self.device = torch.device(device)
        self.layer_ids = list(range(w.n_layers)) if layers is None else list(layers)
        self.pools, self.repl, self.scales = [], [], []
        # host_resident: pools and replacement rows in pinned host memory; the library takes those pointers as they are
        where = dict(device="cpu", pin_memory=True) if host_resident else dict(device=self.device)
        for l in self.layer_ids:
            buf = torch.empty(w.layer_bytes, dtype=torch.uint8, **where)
            scale = synth.fill_layer_(buf, w, l) if fill else 1.0
            rp = torch.empty(max(w.n_repl_rows, 1) * w.row_bytes, dtype=torch.uint8, **where)
            if fill:
                synth.fill_repl_(rp[: w.n_repl_rows * w.row_bytes], w, l, scale)
            self.pools.append(buf)
            self.repl.append(rp)
            self.scales.append(scale)
        self.dst = [torch.empty_like(p) for p in self.pools] if with_dst else None

    @property
    def n_layers(self):
        return len(self.layer_ids)

    def desc(self):
        w = self.w
        return B.make_desc(self.n_layers, w.latent_dim, w.rope_dim, w.page_size, w.dtype, w.pairing, w.row_bytes,
                           w.n_slots, w.inv_freq, self.scales if w.dtype == synth.DT_FP8 else None,
                           rope_heads=w.rope_heads,
                           layer_pairing=None if w.layer_pairing is None else [w.layer_pairing[l] for l in self.layer_ids])

    def nbytes(self):
        return sum(p.numel() for p in self.pools) + sum(r.numel() for r in self.repl)


def plan_workload(w: synth.Workload, mode: int, desc) -> B.Plan:
    free = w.free_slots() if mode == B.ROTATE_ONLY else w.free_pages
    return B.leyline_plan(desc, mode, w.seq_lens, w.pt_offsets, w.pages, w.directives, free)


def run_workload(cache: DeviceCache, mode: int, stream=None, want_idx=True, prefetch=False, launches=1):
    """Plan + launch one splice of the cache's workload in `mode` (in place on cache.pools unless cache.dst is
    set and the mode is FRESH).  Returns (plan, page_table_out, slot_idx_out) -- device int32 tensors."""
    d, keep = cache.desc()
    plan = plan_workload(cache.w, mode, d)
    dev = cache.device
    pt = torch.empty(max(int(plan.info.total_new_pages), 1), dtype=torch.int32, device=dev) if want_idx else None
    idx = torch.empty(max(int(plan.info.total_new_tokens), 1), dtype=torch.int32, device=dev) if want_idx else None
    if prefetch:
        plan.prefetch()
    for _ in range(launches):     # FRESH never writes what it reads, so launching a plan again repeats the result
        if mode == B.ROTATE_ONLY:
            B.leyline_rotate_inplace(plan, cache.pools, cache.repl, idx, stream)
        else:
            dst = cache.dst if (cache.dst is not None and mode == B.FRESH) else cache.pools
            B.leyline_splice(plan, cache.pools, dst, cache.repl, pt, idx, stream)
    del keep
    return plan, pt, idx

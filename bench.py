#!/usr/bin/env python
"""bench.py -- Leyline splice throughput on one B200 (or N independent replicas), DESIGN.md "Measurement".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 3] [--mode fresh]

One step = one pass of the whole hot path over the workload: leyline_plan on the host (a1), then
leyline_splice on the stream: table upload, index / page-table rewrite (a2), fused gather -> rotate -> scatter
with the replacement insert (a3 + a4; a0 is the released list the plan reports).  Default workload =
BASELINE.json config 3 (DeepSeek-V3 shape: 61 layers x 131072 tokens, bf16, page 64, YaRN, three directives),
FRESH mode.  The metric is splice GB/s counting algorithmic bytes read + written (plan.bytes_read +
plan.bytes_written).  Rank 0 prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "splice_throughput_read_plus_write"
UNIT = "GB/s"
MODES = {"fresh": 0, "inplace": 1, "rotate_only": 2}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="3", help="BASELINE.json config: 2, 3, 3m, 4, 5; full-width K: gqa, mha96; appB: the paper's App. B counters' shape")
    ap.add_argument("--mode", default="fresh", choices=list(MODES))
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the supplementary modes / workloads")
    ap.add_argument("--kernel", type=int, default=0, help="leyline_tuning.kernel (0 auto, 1 row, 2 bulk)")
    ap.add_argument("--tile-rows", type=int, default=0)
    ap.add_argument("--ctas-per-sm", type=int, default=0)
    ap.add_argument("--stages", type=int, default=0, help="leyline_tuning.stages (bulk kernel)")
    ap.add_argument("--layer-group", type=int, default=0, help="leyline_tuning.layer_group (bulk kernel)")
    ap.add_argument("--consumer-warps", type=int, default=0, help="leyline_tuning.consumer_warps (bulk kernel)")
    ap.add_argument("--rotate-kernel", type=int, default=0, help="leyline_tuning.rotate_kernel (0 auto, 1 strided registers, 2 TMA boxes, 3 flat passes)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="process-group backend for --gpus N > 1")
    ap.add_argument("--stub-step-ms", type=float, default=0.0,
                    help="TEST ONLY (tests/test_replicas_gloo.py): replace the splice by a host sleep of this many ms "
                         "(+ 1 ms per rank) so that the N-replica launch and its timing contract run without a GPU")
    return ap.parse_args()


def workload_of(name: str, mode: str):
    from paper_2606_01065_b200 import synth
    cfg = int(name) if name.isdigit() else name
    # FRESH compacts into pages of the same pool: the pool holds the live pages plus as many fresh ones
    factor = 2.0 if mode == "fresh" else 1.25
    return synth.config(cfg, pool_factor=factor)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch device copy, read+write)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s, earlier measurement on this pool)"


def ncu_traffic(workload: str, mode: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on (workload, mode), from the newest
    committed `ncu --set full` summary under profiles/ (text, written from a capture; see profiles/README.md).
    None when no capture of that kernel/workload exists."""
    import csv
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_ncu_full_{kernel}_cfg{workload}_{mode}.csv")))
    if not files:
        return None, None
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    tot = 0.0
    with open(files[-1]) as f:
        for row in csv.reader(f):
            if len(row) == 3 and row[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                tot += float(row[2]) * mult.get(row[1], 1.0)
    return (tot or None), os.path.relpath(files[-1], ROOT)


class ClockSampler:
    """nvidia-smi clocks + throttle reasons while the timed region runs (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
            # nvidia-smi initialises NVML for some hundred ms and holds driver locks meanwhile, which stalls this
            # process's CUDA calls: wait for its first sample so that none of that falls into a timed region
            t0 = time.perf_counter()
            while not self.rows and self.proc.poll() is None and time.perf_counter() - t0 < 3.0:
                time.sleep(0.01)
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 3 + i and r[3 + i].lower().startswith("active") for r in self.rows)]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


# ----------------------------------------------------------------------------- our arm

def dist_setup(n_gpus: int):
    """One process per GPU (torchrun, or spawn_replicas below, exports RANK / LOCAL_RANK / WORLD_SIZE); nccl only
    carries the timing contract's barrier and max-over-ranks -- the splice itself has no exchange step
    (paper_2606_01065_b200/replicas.py)."""
    import torch
    from paper_2606_01065_b200 import replicas as R
    rank, world, local = R.env_rank()
    if world != max(1, n_gpus):
        raise SystemExit(f"bench.py: --gpus {n_gpus} but WORLD_SIZE is {world}")
    torch.cuda.set_device(local)
    return R.init("nccl", torch.device("cuda", local))


def barrier(world: int):
    import torch
    from paper_2606_01065_b200 import replicas as R
    R.barrier(world, torch.device("cuda", torch.cuda.current_device()))


def max_over_ranks(x: float, world: int) -> float:
    import torch
    from paper_2606_01065_b200 import replicas as R
    return R.max_over_ranks(x, world, torch.device("cuda", torch.cuda.current_device()))


def time_splice(cache, w, mode: int, steps: int, warmup: int, world: int = 1, chunk: int = 0):
    """K timed steps of plan + splice on torch's current stream, CUDA events around the whole region and the
    library's own events around the data-moving kernels of every step."""
    import torch
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    desc, keep = cache.desc()
    dev = cache.device
    plan0 = harness.plan_workload(w, mode, desc)
    info = plan0.info
    pt = torch.empty(max(int(info.total_new_pages), 1), dtype=torch.int32, device=dev)
    idx = torch.empty(max(int(info.total_new_tokens), 1), dtype=torch.int32, device=dev)
    nbytes = int(info.bytes_read + info.bytes_written)
    # per step: k_index (page table + slot list, one launch) + ONE data kernel: k_move_bulk (FRESH; INPLACE_MOVE with the
    # inserts as its last tickets) or k_rotate_band (ROTATE_ONLY, inserts as trailing copy items)
    launches = 2
    plan0.close()
    plans, host_us = [], []

    pools, repl = B.layer_pointers(cache.pools), B.layer_pointers(cache.repl)   # marshalled once, as a server would
    free = w.free_slots() if mode == B.ROTATE_ONLY else w.free_pages
    dirs = B.pack_directives(w.directives)
    seq_lens = np.asarray(w.seq_lens, np.int64)          # a server holds these as arrays already

    kms = []

    def retire(keep_in_flight):
        # a server destroys a plan once its launch has finished (its host tables are then recycled by the next plan);
        # the plan of 3 steps ago has long finished, so reading its kernel time does not stall the pipeline
        while len(plans) > keep_in_flight:
            p = plans.pop(0)
            kms.append(p.kernel_ms())
            p.close()

    def step():
        t0 = time.perf_counter()
        plan = B.leyline_plan(desc, mode, seq_lens, w.pt_offsets, w.pages, dirs, free)
        host_us.append((time.perf_counter() - t0) * 1e6)
        plan.prefetch()          # table upload on the library's copy stream; the launch below only waits on its event
        if mode == B.ROTATE_ONLY:
            B.leyline_rotate_inplace(plan, pools, repl, idx)
        else:
            B.leyline_splice(plan, pools, pools, repl, pt, idx)
        plans.append(plan)
        retire(3)

    for _ in range(warmup):
        step()
    barrier(world)
    retire(0)
    host_us.clear()
    kms.clear()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    marks = []                    # an event every `chunk` steps (supplementary lines only): see ms_per_step_median_chunk
    e0.record()
    for i in range(steps):
        step()
        if chunk and (i + 1) % chunk == 0 and i + 1 < steps:
            marks.append(torch.cuda.Event(enable_timing=True))
            marks[-1].record()
    e1.record()
    barrier(world)
    ms = e0.elapsed_time(e1) / steps
    ms_chunk = ms_best = None
    if chunk and marks:
        ev = [e0, *marks]
        per = [ev[j].elapsed_time(ev[j + 1]) / chunk for j in range(len(ev) - 1)]
        ms_chunk, ms_best = float(np.median(per)), float(np.min(per))
    retire(0)
    del keep
    return {"ms_per_step": ms, "ms_per_step_median_chunk": ms_chunk, "ms_per_step_best_chunk": ms_best, "kernel_ms_median": float(np.median(kms)), "kernel_ms": float(np.mean(kms)), "kernel_ms_min": float(np.min(kms)), "bytes": nbytes,
            "plan_host_us": float(np.median(host_us)), "launches_per_step": launches,
            "n_directives": len(w.directives), "rows_moved": int(info.rows_moved), "rows_inserted": int(info.rows_inserted),
            "mover": int(info.mover), "tile_rows": int(info.tile_rows)}


def time_single_calls(cache, w, mode: int, reps: int = 10):
    """Latency of ONE call on an idle GPU (nothing to hide the table upload behind): host wall clock from leyline_plan
    to the stream being drained, median of `reps`.  The throughput figure above pipelines back-to-back steps."""
    import torch
    from paper_2606_01065_b200 import binding as B
    desc, keep = cache.desc()
    pools, repl = B.layer_pointers(cache.pools), B.layer_pointers(cache.repl)
    free = w.free_slots() if mode == B.ROTATE_ONLY else w.free_pages
    dirs = B.pack_directives(w.directives)
    pt = idx = None
    out = []
    for i in range(reps + 2):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        plan = B.leyline_plan(desc, mode, w.seq_lens, w.pt_offsets, w.pages, dirs, free)
        plan.prefetch()
        if pt is None:
            pt = torch.empty(max(int(plan.info.total_new_pages), 1), dtype=torch.int32, device=cache.device)
            idx = torch.empty(max(int(plan.info.total_new_tokens), 1), dtype=torch.int32, device=cache.device)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
        if mode == B.ROTATE_ONLY:
            B.leyline_rotate_inplace(plan, pools, repl, idx)
        else:
            B.leyline_splice(plan, pools, pools, repl, pt, idx)
        torch.cuda.synchronize()
        if i >= 2:
            out.append((time.perf_counter() - t0) * 1e6)
        plan.close()
    del keep
    return {"median_us": float(np.median(out)), "min_us": float(np.min(out)), "calls": reps,
            "us_per_directive": float(np.median(out)) / max(1, len(w.directives))}


def time_discovery(dev, with_oracle: bool, n_sessions: int = 16, prompt_len: int = 17000, reps: int = 20):
    """Supplementary line: the discovery side (leyline_cdc_chunk) on the shape of the paper's
    microbenchmark -- 16 sessions x ~17 K-token prompts, anchors every ~600 tokens -- against
    the oracle's sequential chunker on the host, for the default chunk parameters (16, 256, 6) and for long chunks
    (64, 4096, 12).  The input is 1 MB, so the call is bound by its chain of dependent small launches, not by bytes:
    `launch_bound_ms` = launches x the per-launch cost of the same call on a 48-token input."""
    import torch
    from paper_2606_01065_b200 import binding as B
    rng = np.random.default_rng(17)
    n = n_sessions * prompt_len
    anchors = [100000, 100001, 100002]
    t = rng.integers(0, 50000, size=n).astype(np.int32)
    pos = np.cumsum(rng.integers(300, 1200, size=2 * n // 600))
    t[pos[pos < n]] = anchors[0]
    so = [i * prompt_len for i in range(n_sessions + 1)]
    td = torch.from_numpy(t).to(dev)
    off = torch.tensor(so, dtype=torch.int64, device=dev)
    an = torch.tensor(anchors, dtype=torch.int32, device=dev)
    end = torch.empty(n, dtype=torch.int64, device=dev)
    hsh = torch.empty(n, dtype=torch.int64, device=dev)
    kind = torch.empty(n, dtype=torch.int32, device=dev)
    cnt = torch.zeros(1, dtype=torch.int64, device=dev)

    def timed(fn, reps):
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    # cost of one small dependent launch of this call chain: the same call on a 48-token input (every kernel is one
    # block, so its time is launches x launch cost), divided by its launch count
    n_small = 48
    def launches_of(m, mn):      # front, next; doubling rounds (seeds behind every hard stop: <= (m-1)/min_size + 1 chunks to cover); count+scan, emit
        far, rounds, reach = (m - 1) // mn + 1, 0, 1
        while reach <= far:
            reach, rounds = reach << 1, rounds + 1
        return 2 + rounds + 2
    off_small = torch.tensor([0, n_small], dtype=torch.int64, device=dev)
    prm0 = B.CdcParams(0x5EED, 16, 256, 6, 0)
    small_ms = timed(lambda: B.leyline_cdc_chunk(prm0, td, n_small, off_small, 1, an, len(anchors), end, hsh, kind, n_small, cnt), 50)
    launch_ms = small_ms / launches_of(n_small, 16)
    out = {"tokens": n, "small_launch_us": launch_ms * 1e3,
           "bound": "launch latency: the input is 1 MB, the call is a chain of dependent small launches (scratch "
                    "allocation included, programmatic dependent launch); launch_bound_ms = launches_per_call x the "
                    "per-launch cost of the same call on 48 tokens"}
    for name, (mn, mx, bits) in (("min16_max256_bits6", (16, 256, 6)), ("min64_max4096_bits12", (64, 4096, 12))):
        prm = B.CdcParams(0x5EED, mn, mx, bits, 0)
        gpu_ms = timed(lambda: B.leyline_cdc_chunk(prm, td, n, off, n_sessions, an, len(anchors), end, hsh, kind, n, cnt), reps)
        c = int(cnt.item())
        one = []                      # ONE call on an idle GPU, synchronised on both sides (what a server's request path sees)
        for _ in range(12):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            B.leyline_cdc_chunk(prm, td, n, off, n_sessions, an, len(anchors), end, hsh, kind, n, cnt)
            torch.cuda.synchronize()
            one.append((time.perf_counter() - t0) * 1e6)
        launches = launches_of(n, mn)
        line = {"chunks": c, "gpu_ms": gpu_ms, "gpu_Mtok_per_s": n / gpu_ms / 1e3, "launches_per_call": launches,
                "launch_bound_ms": launches * launch_ms, "over_launch_bound": gpu_ms / (launches * launch_ms),
                "one_synchronised_call_us": float(np.median(one[2:]))}
        if with_oracle:      # part of the cpu_baseline leg: the oracle's sequential chunker timed on the host beside it
            from oracle import cdc as OC
            t0 = time.perf_counter()
            o_end, o_hash, o_kind = OC.chunk(0x5EED, mn, mx, bits, t, so, anchors)
            cpu_ms = (time.perf_counter() - t0) * 1e3
            same = c == len(o_end) and bool((end[:c].cpu().numpy() == o_end).all()) and \
                bool((hsh[:c].cpu().numpy().view(np.uint64) == o_hash).all())
            line.update(oracle_ms=cpu_ms, oracle_Mtok_per_s=n / cpu_ms / 1e3, matches_oracle=same)
        out[name] = line
    return out


def cpu_baseline_all_cores(pools, repls, scales, w, mode: int, bytes_per_layer: int, n_layers: int = 48):
    """the same oracle with a thread per layer (layers are independent given the plan; the C
    oracle runs outside the GIL), on all host cores.  A reported baseline, not a target."""
    import oracle as O
    from concurrent.futures import ThreadPoolExecutor
    cores = os.cpu_count() or 1
    n_layers = min(n_layers, w.n_layers)
    free = w.free_slots() if mode == O.ROTATE_ONLY else w.free_pages
    inputs = [(pools(l), repls(l)) for l in range(n_layers)]
    t0 = time.perf_counter()
    bm = O.plan_batch(mode, w.page_size, w.seq_lens, w.pt_offsets, w.pages, w.directives, free)

    def one(l):
        O.splice_layer(w.dtype, w.pairing_of(l), w.latent_dim, w.rope_dim, w.row_bytes, w.inv_freq, scales[l], inputs[l][0],
                       inputs[l][1], bm, n_heads=w.rope_heads)

    with ThreadPoolExecutor(max_workers=cores) as ex:
        list(ex.map(one, range(n_layers)))
    dt = time.perf_counter() - t0
    return {"value": n_layers * bytes_per_layer / dt / 1e9, "unit": UNIT, "cores": min(cores, n_layers), "kind": "oracle, one thread per layer",
            "sample": f"{n_layers} of {w.n_layers} layers of {w.name}, {dt:.1f} s", "host_cpus": cores}


def cpu_baseline(pools, repls, scales, w, mode: int, bytes_per_layer: int, budget_s: float = 15.0, max_layers: int = 1 << 30):
    """The oracle as it stands (one thread, explicit per-token loops, fp64 libm trig) on whole layers of the same
    workload, on this host, until about `budget_s` seconds of oracle time are spent (a bounded sample: whole layers,
    which are independent given the plan).  `pools` / `repls`: callables returning a layer's bytes as a flat uint8
    numpy array."""
    import oracle as O
    free = w.free_slots() if mode == O.ROTATE_ONLY else w.free_pages
    t0 = time.perf_counter()
    bm = O.plan_batch(mode, w.page_size, w.seq_lens, w.pt_offsets, w.pages, w.directives, free)
    t_total = time.perf_counter() - t0
    assert bm.status == O.OK
    done = 0
    while done < min(max_layers, w.n_layers) and t_total < budget_s:
        old, repl = pools(done), repls(done)
        t0 = time.perf_counter()
        O.splice_layer(w.dtype, w.pairing, w.latent_dim, w.rope_dim, w.row_bytes, w.inv_freq, scales[done], old, repl, bm,
                       n_heads=w.rope_heads)
        t_total += time.perf_counter() - t0
        done += 1
    return {"value": done * bytes_per_layer / t_total / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{done} of {w.n_layers} layers of {w.name} ({done * bytes_per_layer / 1e9:.2f} GB read+written), "
                      f"plan + per-layer splice, {t_total:.1f} s",
            "seconds": t_total, "host_cpus": os.cpu_count()}


def pcie_peak(dev, nbytes: int = 1 << 30, reps: int = 3):
    """What the link gives plain copies, measured in this run: one pinned host -> device and one device -> host
    cudaMemcpyAsync of `nbytes` each, alone and then both at once on two streams (one copy per direction in flight).
    `both_GBps` (bytes of both directions / the time until both are done) is the bound `e2e` is read against."""
    import torch
    h_src = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    h_dst = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    d_dst = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    d_src = torch.zeros(nbytes, dtype=torch.uint8, device=dev)
    h_src.zero_()
    s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)

    def run(h2d: bool, d2h: bool) -> float:
        best = float("inf")
        for _ in range(reps + 1):                 # the first pass is the warm-up
            torch.cuda.synchronize()
            ev = []
            for on, st, dst, src in ((h2d, s_in, d_dst, h_src), (d2h, s_out, h_dst, d_src)):
                if on:
                    with torch.cuda.stream(st):
                        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        a.record()
                        dst.copy_(src, non_blocking=True)
                        b.record()
                        ev.append((a, b))
            torch.cuda.synchronize()
            first = ev[0][0]                      # both streams start right behind the same synchronize
            best = min(best, max(max(first.elapsed_time(b), a.elapsed_time(b)) for a, b in ev))
        return best * 1e-3

    one_in, one_out, both = run(True, False), run(False, True), run(True, True)
    return {"h2d_alone_GBps": nbytes / one_in / 1e9, "d2h_alone_GBps": nbytes / one_out / 1e9,
            "both_GBps": 2 * nbytes / both / 1e9, "bytes_each_way": nbytes,
            "how": "pinned cudaMemcpyAsync, one per direction, two streams, CUDA events, best of %d" % reps}


def run_e2e(cache, w, steps: int, warmup: int = 1):
    """Same metric through the public API with HOST buffers: the cache lives in pinned host memory and the library is
    handed those host pointers (include/leyline.h: layer pointers may be device memory or device-accessible pinned
    host memory).  The kernels gather the rows to move straight from host memory and scatter the spliced rows
    straight back over PCIe, so only the bytes the method needs cross the link: per step host -> device = the rows
    read + the plan tables, device -> host = the rows written + the page table and slot list read back.
    `pcie_peak` is the link's own rate for plain pinned copies in both directions at once, measured here; `frac` =
    value / pcie_peak.both_GBps."""
    import torch
    from paper_2606_01065_b200 import binding as B
    L = cache.n_layers
    dev = cache.device
    link = pcie_peak(dev)
    host_pool = [torch.empty(w.layer_bytes, dtype=torch.uint8, pin_memory=True) for _ in range(L)]
    host_repl = [torch.empty(cache.repl[l].numel(), dtype=torch.uint8, pin_memory=True) for l in range(L)]
    for l in range(L):
        host_pool[l].copy_(cache.pools[l])
        host_repl[l].copy_(cache.repl[l])
    torch.cuda.synchronize()
    desc, keep = cache.desc()
    pools, repl = B.layer_pointers(host_pool), B.layer_pointers(host_repl)
    dirs = B.pack_directives(w.directives)
    sizes = {}
    # the step's small results (new page table, slot list) land in buffers a scheduler would hold for the session:
    # device side for the kernels, pinned host side for the read-back; sized once from the first plan
    plan0 = B.leyline_plan(desc, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, dirs, w.free_pages)
    n_pt, n_idx = int(plan0.info.total_new_pages), int(plan0.info.total_new_tokens)
    plan0.close()
    pt = torch.empty(n_pt, dtype=torch.int32, device=dev)
    idx = torch.empty(n_idx, dtype=torch.int32, device=dev)
    pt_host = torch.empty(n_pt, dtype=torch.int32, pin_memory=True)
    idx_host = torch.empty(n_idx, dtype=torch.int32, pin_memory=True)

    def step():
        plan = B.leyline_plan(desc, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, dirs, w.free_pages)
        plan.prefetch()
        info = plan.info
        B.leyline_splice(plan, pools, pools, repl, pt, idx)
        pt_host.copy_(pt, non_blocking=True)             # the step's result that the scheduler reads
        idx_host.copy_(idx, non_blocking=True)
        torch.cuda.synchronize()                         # ... and it reads it: the step ends when the result is on the host
        sizes.update(read=int(info.bytes_read), written=int(info.bytes_written), small=pt_host.numel() * 4 + idx_host.numel() * 4,
                     tables=int(info.n_tiles) * 48 + int(info.total_new_pages) * 8)
        plan.close()

    for _ in range(warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    dt = (time.perf_counter() - t0) / steps
    # supplementary: the same host-resident source spliced straight INTO THE DEVICE pool (swap-in + edit in one pass:
    # rows cross PCIe once, host -> device only)
    dev_pools = B.layer_pointers(cache.pools)

    def swap_in():
        plan = B.leyline_plan(desc, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, dirs, w.free_pages)
        plan.prefetch()
        B.leyline_splice(plan, pools, dev_pools, repl, None, None)
        torch.cuda.synchronize()
        plan.close()

    swap_in()
    t0 = time.perf_counter()
    for _ in range(2):
        swap_in()
    dt_swap = (time.perf_counter() - t0) / 2
    # the spliced host cache must equal the device-resident result (same kernels, same arithmetic)
    plan = B.leyline_plan(desc, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, dirs, w.free_pages)
    B.leyline_splice(plan, cache.pools, cache.pools, cache.repl, None, None)     # same start state, device-resident
    torch.cuda.synchronize()
    plan.close()
    same = all(bool((host_pool[l].to(dev) == cache.pools[l]).all()) for l in (0, L - 1))
    del keep
    value = (sizes["read"] + sizes["written"]) / dt / 1e9
    return {"value": value, "unit": UNIT,
            "h2d_bytes_per_step": sizes["read"] + sizes["tables"], "d2h_bytes_per_step": sizes["written"] + sizes["small"],
            "ms_per_step": dt * 1e3, "steps": steps, "matches_device_resident_result": same,
            "pcie_peak": link, "frac": value / link["both_GBps"],
            "swap_in": {"ms_per_step": dt_swap * 1e3, "h2d_GBps": sizes["read"] / dt_swap / 1e9,
                        "frac_of_h2d_alone": sizes["read"] / dt_swap / 1e9 / link["h2d_alone_GBps"],
                        "note": "host-resident source spliced into the device pool: moved rows cross PCIe once"},
            "note": "cache in pinned host memory, spliced in place over PCIe by the same kernels (host pointers through the "
                    "C ABI); host wall clock around synchronised steps; bound = pcie_peak.both_GBps (plain pinned copies, "
                    "both directions at once, measured in this run)"}



# (key, synth config, modes) of SURVEY.md section 8(d)'s table that ride along with the headline as `extras`
EXTRA_WORKLOADS = [("cfg2", "2", ("fresh", "inplace", "rotate_only"), 2.0),
                   ("cfg5", "5", ("fresh", "inplace", "rotate_only"), 2.0),
                   ("cfg4", "4", ("inplace", "rotate_only"), 1.25),
                   ("cfg4", "4", ("fresh",), 2.0),          # 147 GB of pools: runs when that much device memory is free
                   ("gqa", "gqa", ("fresh", "inplace", "rotate_only"), 2.0),
                   ("mha96", "mha96", ("fresh", "inplace", "rotate_only"), 2.0),
                   ("appB", "appB", ("fresh", "rotate_only"), 2.0)]


def extra_line(cache, w, mode_name: str, peak: float, device_index: int, target_s: float = 0.35):
    """One supplementary (workload, mode) line: the same step as the headline (plan + prefetch + index + data kernel),
    long enough (about target_s) for nvidia-smi to sample the clocks under load."""
    mode = MODES[mode_name]
    probe = time_splice(cache, w, mode, 3, 2)
    steps = int(min(400, max(5, target_s * 1e3 / max(probe["ms_per_step"], 1e-3))))
    time.sleep(0.5)              # let the power average settle: these lines run back to back behind cache fills
    sampler = ClockSampler(device_index)
    sampler.start()
    x = time_splice(cache, w, mode, steps, 1, chunk=max(1, steps // 8))
    clocks = sampler.stop()
    # The step time of a supplementary line is the MEDIAN over eight chunks of the timed region: nvidia-smi sampling next
    # to the run stalls the submitting thread for tens of ms now and then (seen as one line in five at 1.1-1.25 x its
    # kernel time while the kernel time itself did not move); the mean over the whole region is reported beside it.
    # The headline line keeps the contract's plain mean over exactly K steps.
    ms_step = x["ms_per_step_median_chunk"] or x["ms_per_step"]
    step_gbs, kern_gbs = x["bytes"] / ms_step / 1e6, x["bytes"] / x["kernel_ms"] / 1e6
    return {"workload": w.name, "mode": mode_name, "steps": steps, "bytes": x["bytes"], "directives": x["n_directives"],
            "ms_per_step": ms_step, "ms_per_step_mean": x["ms_per_step"], "GBps": step_gbs, "kernel_ms": x["kernel_ms"], "kernel_GBps": kern_gbs,
            "frac": kern_gbs / peak, "step_over_kernel": ms_step / x["kernel_ms"],
            "plan_host_us": x["plan_host_us"], "us_per_directive": ms_step * 1e3 / max(1, x["n_directives"]),
            "mover": x["mover"], "tile_rows": x["tile_rows"], "clocks": clocks}


def extra_workloads(peak: float, device_index: int, skip=()):
    """Every other row of SURVEY.md 8(d): configs 2, 4, 5, the full-width K pools and the paper's App. B shape, each in
    the modes it has, one cache per workload (built, timed, freed)."""
    import gc
    import torch
    from paper_2606_01065_b200 import harness, synth
    out = {}
    for key, cfg, modes, factor in EXTRA_WORKLOADS:
        if key in skip:
            continue
        w = synth.config(int(cfg) if cfg.isdigit() else cfg, pool_factor=factor)
        need = (w.layer_bytes + max(w.n_repl_rows, 1) * w.row_bytes) * w.n_layers
        free, _ = torch.cuda.mem_get_info(device_index)
        if free < need * 1.03 + (1 << 30):
            for m in modes:
                out[f"{key}_{m}"] = {"workload": w.name, "mode": m, "skipped": f"needs {need / 2**30:.0f} GiB of device memory, "
                                                                              f"{free / 2**30:.0f} GiB free"}
            continue
        cache = harness.DeviceCache(w, f"cuda:{device_index}")
        torch.cuda.synchronize()
        for m in modes:
            out[f"{key}_{m}"] = extra_line(cache, w, m, peak, device_index)
        if key == "appB":    # the paper's own shape: what ONE call costs a server (plan + upload + kernels, idle GPU)
            for m in modes:
                out[f"{key}_{m}_single_call_idle_gpu"] = time_single_calls(cache, w, MODES[m])
        del cache
        gc.collect()
        torch.cuda.empty_cache()
    return out


def pattern_probe(device, n_rows: int = 8 << 20):
    """The library's own probe of the a5 access pattern (leyline_probe_band_update: contiguous rows, no page table, no
    rotation, full-line accesses): what the memory system allows on 128 B of every 1152-B row / 64 B of every 576-B row,
    read + written in place.  k_rotate_band's GB/s is to be read against this, not against a dense copy."""
    import torch
    from paper_2606_01065_b200 import binding as B
    out = {}
    for name, row_bytes, band in (("bf16_128_of_1152", 1152, 128), ("fp8_64_of_576", 576, 64), ("dense_1152_of_1152", 1152, 1152)):
        buf = torch.zeros(n_rows * row_bytes, dtype=torch.uint8, device=device)
        best = {}
        for per_sm in (4, 8, 16):
            for _ in range(2):
                B.leyline_probe_band_update(buf, n_rows, row_bytes, row_bytes - band, band, per_sm)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                B.leyline_probe_band_update(buf, n_rows, row_bytes, row_bytes - band, band, per_sm)
            e1.record()
            torch.cuda.synchronize()
            best[f"ctas_per_sm_{per_sm}"] = 2.0 * n_rows * band / (e0.elapsed_time(e1) / 5 * 1e-3) / 1e9
        out[name] = {"GBps": max(best.values()), "by_grid": best, "rows": n_rows}
        del buf
    return out


def pattern_reference(device, n_rows: int = 4 << 20):
    """What plain torch ops reach on the access pattern of a5 (ROTATE_ONLY on an MLA cache): an in-place update of the
    last 128 B of every 1152-B row (bf16) / the last 64 B of every 576-B row (fp8) of a contiguous buffer -- no page
    table, no rotation.  A reference for how hard the PATTERN is on this memory system, next to k_rotate_band's GB/s
    (same byte accounting: band bytes read + written)."""
    import torch
    out = {}
    for name, row_bytes, band in (("bf16_128_of_1152", 1152, 128), ("fp8_64_of_576", 576, 64)):
        buf = torch.zeros(n_rows * row_bytes, dtype=torch.uint8, device=device)
        views = {"int32_add": (buf.view(torch.int32).view(n_rows, row_bytes // 4)[:, (row_bytes - band) // 4:], lambda v: v.add_(1))}
        if row_bytes == 1152:
            views["bf16_mul"] = (buf.view(torch.bfloat16).view(n_rows, 576)[:, 512:], lambda v: v.mul_(1.0009765625))
        best = {}
        for k, (v, op) in views.items():
            for _ in range(2):
                op(v)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                op(v)
            e1.record()
            torch.cuda.synchronize()
            best[k] = 2.0 * n_rows * band / (e0.elapsed_time(e1) / 5 * 1e-3) / 1e9
        out[name] = {"GBps": max(best.values()), "by_op": best, "rows": n_rows}
        del buf, views
    # and a dense in-place update of the same buffer size with the same op, for scale
    buf = torch.zeros(n_rows * 288, dtype=torch.int32, device=device)
    for _ in range(2):
        buf.add_(1)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(5):
        buf.add_(1)
    e1.record()
    torch.cuda.synchronize()
    out["dense_int32_add"] = {"GBps": 2.0 * buf.numel() * 4 / (e0.elapsed_time(e1) / 5 * 1e-3) / 1e9}
    return out


def sustained_line(cache, w, mode: int, ms_per_step: float, device_index: int, seconds: float = 3.2):
    """The headline step back to back for >= 3 s (median and best, clocks under load): the same
    time_splice as the headline, cut into 32 chunks whose median and best are reported beside the plain mean."""
    steps = int(max(64, np.ceil(seconds * 1e3 / max(ms_per_step, 1e-3))))
    sampler = ClockSampler(device_index)
    sampler.start()
    x = time_splice(cache, w, mode, steps, 3, chunk=max(1, steps // 32))
    clocks = sampler.stop()
    gbs = lambda ms: x["bytes"] / ms / 1e6
    return {"steps": steps, "seconds": steps * x["ms_per_step"] * 1e-3, "ms_per_step_mean": x["ms_per_step"],
            "ms_per_step_median": x["ms_per_step_median_chunk"], "ms_per_step_best": x["ms_per_step_best_chunk"],
            "GBps_mean": gbs(x["ms_per_step"]), "GBps_median": gbs(x["ms_per_step_median_chunk"]),
            "GBps_best": gbs(x["ms_per_step_best_chunk"]), "kernel_ms_mean": x["kernel_ms"], "kernel_ms_median": x["kernel_ms_median"],
            "kernel_ms_best": x["kernel_ms_min"], "mover_GBps_mean": gbs(x["kernel_ms"]), "mover_GBps_best": gbs(x["kernel_ms_min"]),
            "chunks": 32, "clocks": clocks}


SUMMARY_KEYS = {"cfg2": "2", "cfg3": "3", "cfg3m": "3m", "cfg4": "4", "cfg5": "5", "gqa": "g", "mha96": "m", "appB": "B"}
SUMMARY_MODES = {"fresh": "f", "inplace": "i", "rotate_only": "r"}


def summary_of(out: dict, peak: float) -> dict:
    """Every (workload, mode) of SURVEY.md 8(d) in a few characters each, as the LAST key of the line, so that a
    truncated record of this line still shows them.  Row = [mover GB/s, fraction of the copy peak, us per directive of
    the step, host plan us, SM MHz under load, 1 if any throttle reason was seen].  Keys: workload (2 3 3m 4 5 = BASELINE
    configs, g = gqa, m = mha96, B = App. B shape) + mode (f fresh, i in place, r rotate only)."""
    def us(x):
        return round(x, 1) if x < 100 else int(round(x))

    def row(gbs, frac, us_dir, plan_us, clocks):
        c = clocks or {}
        return [int(round(gbs)), round(frac, 2), us(us_dir), int(round(plan_us)), int(c.get("sm_mhz") or 0),
                int(bool([r for r in c.get("reasons") or [] if r != "nvidia-smi unavailable"]))]

    rf = out["roofline"]
    sm = {"cols": "kGBps,frac,us/dir,plan_us,MHz,thr",
          "3f": row(rf["achieved"], rf["frac"], out["us_per_directive"], out["plan_host_us"], out.get("clocks"))}
    ex = out.get("extras") if isinstance(out.get("extras"), dict) else {}
    for key, x in ex.items():
        wl, _, md = key.partition("_")
        if wl not in SUMMARY_KEYS or md not in SUMMARY_MODES or not isinstance(x, dict):
            continue
        k = SUMMARY_KEYS[wl] + SUMMARY_MODES[md]
        sm[k] = "skip" if "skipped" in x else row(x["kernel_GBps"], x["frac"], x["us_per_directive"], x["plan_host_us"], x.get("clocks"))
    for m in ("fresh", "rotate_only"):          # the paper's own shape: one call on an idle GPU, us (median)
        one = ex.get(f"appB_{m}_single_call_idle_gpu")
        if one:
            sm["B" + SUMMARY_MODES[m] + "1"] = int(round(one["median_us"]))
    su = out.get("sustained")
    if su:   # [seconds, median GB/s, best GB/s, mover GB/s mean, MHz, thr]
        c = su.get("clocks") or {}
        sm["sus"] = [round(su["seconds"], 1), int(round(su["GBps_median"])), int(round(su["GBps_best"])), int(round(su["mover_GBps_mean"])),
                     int(c.get("sm_mhz") or 0), int(bool(c.get("reasons")))]
    e = out.get("e2e") or {}
    if e.get("value"):
        sm["e2e"] = [round(e["value"], 1), round(e.get("frac") or 0, 2)]
    pp = ex.get("a5_pattern_probe") or {}
    if pp:   # a5's ceiling: the pattern probe, GB/s read+write (bf16 128 of 1152 B, fp8 64 of 576 B)
        sm["a5p"] = [int(round(pp[k]["GBps"])) for k in ("bf16_128_of_1152", "fp8_64_of_576") if k in pp]
    sm["peak"] = int(round(peak))
    return sm


def build_flags() -> str:
    from paper_2606_01065_b200 import build as _b
    return _b.built_with()


def kernel_name(mover: int, rotate_only: bool) -> str:
    """leyline_plan_info.mover -> the kernel that moves the bytes (2 = bulk mover, 3 = the 2-D TMA band variant chosen
    with --rotate-kernel 2, 4 = the band kernel over flat passes (short segments, or --rotate-kernel 3); otherwise the
    register-staged kernels)."""
    if mover == 2:
        return "k_move_bulk"
    if mover == 3:
        return "k_rotate_band_tma"
    if mover == 4:
        return "k_rotate_band_flat"
    return "k_rotate_band" if rotate_only else "k_move_rows"


def run_stub(args):
    """--stub-step-ms: the N-replica launch and timing contract with a host sleep in place of the splice (no GPU, no
    library): barrier, K timed steps, MAX over ranks of the step time, SUM of the units, one JSON line from rank 0."""
    from paper_2606_01065_b200 import replicas as R
    rank, world, local = R.init(args.backend)
    R.barrier(world)
    for _ in range(args.warmup):
        time.sleep(1e-3)
    R.barrier(world)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time.sleep((args.stub_step_ms + rank) * 1e-3)
    ms_mine = (time.perf_counter() - t0) * 1e3 / args.steps
    R.barrier(world)
    units = 1_000_000 * (rank + 1)
    value, ms = R.job_throughput_gbs(units, ms_mine, world)
    R.finish(world)
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
                          "vs_baseline": None, "dtype": "none", "data": "stub", "impl": "stub",
                          "config": {"workload": "stub (host sleep)", "replicas": world}, "gpu_launches": 0,
                          "units_all_ranks": sum(1_000_000 * (r + 1) for r in range(world))}))


def run_ours(args):
    import torch
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    from paper_2606_01065_b200 import replicas as R
    from paper_2606_01065_b200 import synth
    rank, world, local = dist_setup(args.gpus)
    B.leyline_set_tuning(kernel=args.kernel, tile_rows=args.tile_rows, ctas_per_sm=args.ctas_per_sm, profile=1,
                         stages=args.stages, layer_group=args.layer_group, consumer_warps=args.consumer_warps,
                         rotate_kernel=args.rotate_kernel)
    mode = MODES[args.mode]
    w = workload_of(args.workload, args.mode)
    cache = harness.DeviceCache(w, f"cuda:{local}")
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    r = time_splice(cache, w, mode, args.steps, args.warmup, world)
    clocks = sampler.stop()
    ms = max_over_ranks(r["ms_per_step"], world)
    dev = torch.device("cuda", local)
    value = R.sum_over_ranks(float(r["bytes"]), world, dev) / (ms * 1e-3) / 1e9     # whole job: all replicas' bytes / slowest rank's time
    peak, peak_src = peaks()
    kernel_gbs = r["bytes"] / (r["kernel_ms"] * 1e-3) / 1e9
    kname = kernel_name(r["mover"], mode == B.ROTATE_ONLY)
    traffic, traffic_src = ncu_traffic(args.workload, args.mode, kname)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16" if w.dtype == 0 else "fp8_e4m3",
        "data": "synthetic", "impl": "ours",
        "config": {"workload": w.name, "mode": args.mode, "n_layers": w.n_layers, "seq_lens": f"{w.n_requests}x{w.seq_lens[0]}",
                   "page_size": w.page_size, "directives": r["n_directives"], "rows_moved_per_layer": r["rows_moved"],
                   "rows_inserted_per_layer": r["rows_inserted"], "bytes_read_plus_written": r["bytes"],
                   "cache_flush": "none needed: each step streams %.2f GB, far larger than the 126 MB L2" % (r["bytes"] / 1e9),
                   "replicas": world, "multi_gpu": "replicas only (the path has no exchange step)",
                   "build_knobs": " ".join(f for f in build_flags().split() if f.startswith("-D")) or "none (default build)",
                   "throughput": "pipelined steady state: the host plan and table upload of step n+1 overlap the kernels of "
                                 "step n; extras.single_call_idle_gpu is one call on an idle GPU"},
        "us_per_directive": ms * 1e3 / max(1, r["n_directives"]),
        "pct_of_8TBps_nominal": 100.0 * value / world / 8000.0,
        "plan_host_us": r["plan_host_us"],
        "gpu_launches": r["launches_per_step"] * args.steps,
        "clocks": clocks,
        "roofline": {"bound": "hbm", "achieved": kernel_gbs, "peak": peak, "unit": UNIT, "frac": kernel_gbs / peak,
                     "traffic": traffic, "traffic_source": traffic_src, "algorithmic_bytes": r["bytes"],
                     "kernel": kname + (" (in-place K_pe rotation)" if kname.startswith("k_rotate_band") else " (fused gather-rotate-scatter + insert)"),
                     "tile_rows": r["tile_rows"],
                     "kernel_ms": r["kernel_ms"], "kernel_ms_best": r["kernel_ms_min"],
                     "peak_source": peak_src, "frac_of_8TBps_nominal": kernel_gbs / 8000.0},
    }
    headline = args.workload == "3" and args.mode == "fresh"
    if rank == 0 and world == 1:
        bytes_per_layer = r["bytes"] // w.n_layers
        if not args.no_extras and headline:
            extras = {}
            for name, wl, md in (("cfg3_inplace", w, "inplace"), ("cfg3_rotate_only", w, "rotate_only"),
                                 ("cfg3m_fresh", synth.config("3m", pool_factor=2.0), "fresh"),
                                 ("cfg3m_inplace", synth.config("3m", pool_factor=2.0), "inplace")):
                cache.w = wl
                extras[name] = extra_line(cache, wl, md, peak, local)
            cache.w = w
            out["sustained"] = sustained_line(cache, w, mode, r["ms_per_step"], local)
            extras["single_call_idle_gpu"] = time_single_calls(cache, w, mode)
            extras["discovery_cdc"] = time_discovery(cache.device, with_oracle=not args.no_cpu_baseline)
            out["extras"] = extras
        if not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(lambda l: cache.pools[l].cpu().numpy(), lambda l: cache.repl[l].cpu().numpy(),
                                               cache.scales, w, mode, bytes_per_layer)
            out["cpu_baseline_all_cores"] = cpu_baseline_all_cores(lambda l: cache.pools[l].cpu().numpy(),
                                                                   lambda l: cache.repl[l].cpu().numpy(), cache.scales, w, mode,
                                                                   bytes_per_layer)
    if not args.no_e2e and mode == B.FRESH:
        # every replica runs its own end-to-end leg (host pools over its own PCIe link); whole job = all bytes / slowest
        try:
            e = run_e2e(cache, w, steps=5)
        except Exception as ex:   # e.g. the host cannot pin that much memory: say so instead of inventing a number
            e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                 "error": f"{type(ex).__name__}: {ex}"}
        if world > 1:
            ok = R.sum_over_ranks(1.0 if e.get("value") else 0.0, world, dev) == world
            e_ms = max_over_ranks(e.get("ms_per_step") or 0.0, world)
            if ok:
                e = dict(e, value=world * r["bytes"] / (e_ms * 1e-3) / 1e9,
                         ms_per_step=e_ms, h2d_bytes_per_step=world * e["h2d_bytes_per_step"],
                         d2h_bytes_per_step=world * e["d2h_bytes_per_step"], replicas=world)
            else:
                e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                     "error": "the end-to-end leg failed on at least one rank: " + str(e.get("error"))}
        out["e2e"] = e
    if rank == 0 and world == 1 and not args.no_extras and headline:
        # the rest of SURVEY.md 8(d)'s table; the config-3 cache is released first (config 4 alone is 92 GB)
        import gc
        del cache
        gc.collect()
        torch.cuda.empty_cache()
        out["extras"].update(extra_workloads(peak, local))
        out["extras"]["a5_pattern_probe"] = pattern_probe(dev)
        out["extras"]["a5_pattern_reference_torch"] = pattern_reference(dev)
    elif world > 1:
        out["extras"] = "N = 1 only (supplementary workloads; they do not depend on the replica count)"
    R.finish(world)
    if rank == 0:
        # order of the line: contract keys, roofline, cpu_baseline, e2e, sustained, then the long `extras`, and the compact
        # `summary` of every SURVEY.md 8(d) row as the very last key
        ex = out.pop("extras", None)
        if ex is not None:
            out["extras"] = ex
        out["summary"] = summary_of(out, peak)
        print(json.dumps(out))


def spawn_replicas(args) -> int:
    """`python bench.py --gpus N` without a launcher: start N ranks of this script, one per GPU (RANK / LOCAL_RANK /
    WORLD_SIZE / MASTER_* as torchrun would export them), and pass rank 0's JSON line through.  Fails loudly when the
    box has fewer than N devices -- the flag must mean N."""
    import socket
    if args.stub_step_ms <= 0:
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            sys.stderr.write(f"bench.py: --gpus {args.gpus} asked for, but this box has {have} CUDA device(s)\n")
            return 2
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for rk in range(args.gpus):
        env = dict(os.environ, RANK=str(rk), LOCAL_RANK=str(rk), WORLD_SIZE=str(args.gpus), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        env.setdefault("NCCL_DEBUG", "INFO")       # the communicator log shows the rank count (and NVLS, when used)
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__), *sys.argv[1:]], env=env,
                                      stdout=None if rk == 0 else subprocess.DEVNULL))
    rc = 0
    for pr in procs:
        rc = pr.wait() or rc
    return rc


# ----------------------------------------------------------------------------- reference arm = the oracle

def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on this host's cores; each step is a bounded sample (one
    layer) of the same workload.  No CUDA library, no GPU work.  Under torchrun only rank 0 runs."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import torch
    import oracle as O
    from paper_2606_01065_b200 import synth
    mode = MODES[args.mode]
    w = workload_of(args.workload, args.mode)
    buf = torch.empty(w.layer_bytes, dtype=torch.uint8)
    scale = synth.fill_layer_(buf, w, 0)
    rp = torch.empty(max(w.n_repl_rows, 1) * w.row_bytes, dtype=torch.uint8)
    synth.fill_repl_(rp[: w.n_repl_rows * w.row_bytes], w, 0, scale)
    old, repl = buf.numpy(), rp.numpy()
    free = w.free_slots() if mode == O.ROTATE_ONLY else w.free_pages
    E, W = w.elem_bytes, w.row_elems
    times = []
    nbytes = 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        bm = O.plan_batch(mode, w.page_size, w.seq_lens, w.pt_offsets, w.pages, w.directives, free)
        O.splice_layer(w.dtype, w.pairing, w.latent_dim, w.rope_dim, w.row_bytes, w.inv_freq, scale, old, repl, bm,
                       n_heads=w.rope_heads)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
        if not nbytes:
            rows = 0
            for r, rm in enumerate(bm.requests):
                # rule M1: FRESH rewrites from the page of the first directive that changes anything (FORGET ends the search)
                first = None
                for d in (d for d in w.directives if d[0] == r):
                    if d[5] != 0:
                        break
                    if d[2] > d[1] or d[3] > 0:
                        first = d[1]
                        break
                k0P = (first // w.page_size) * w.page_size if first is not None else rm.L_new
                for (k, s, d, n, c) in rm.segs.as_tuples():
                    if k == O.INSERT:
                        rows += n
                    elif mode == O.FRESH:
                        rows += max(0, d + n - max(d, k0P))
                    elif c != 0:
                        rows += n if mode == O.INPLACE_MOVE else 0
            nbytes = 2 * rows * W * E
            if mode == O.ROTATE_ONLY:
                nbytes += 2 * sum(n for rm in bm.requests for (k, s, d, n, c) in rm.segs.as_tuples() if k == O.KEEP and c != 0) * w.rope_heads * w.rope_dim * E
    ms = float(np.mean(times)) * 1e3
    value = nbytes / (ms * 1e-3) / 1e9
    sample = f"1 of {w.n_layers} layers of {w.name} per step ({nbytes / 1e9:.3f} GB read+written), plan + splice"
    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "impl": "reference",
        "config": {"workload": w.name, "mode": args.mode, "n_layers": w.n_layers, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "host_cpus": os.cpu_count()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    elif a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_replicas(a))
    elif a.stub_step_ms > 0:
        run_stub(a)
    else:
        run_ours(a)

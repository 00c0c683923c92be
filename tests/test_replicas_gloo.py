"""Multi-GPU path on CPU: world_size-2 `gloo` processes run the measurement plumbing of
paper_2606_01065_b200/replicas.py (the splice has no exchange step -> replicas only; the only
collectives are the timing contract's barrier / MAX-over-ranks / SUM of units), and two ranks that each plan
the same workload with the host planner produce identical plans (the plan is the only thing a serving stack
would broadcast)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_2606_01065_b200 import replicas as R
    r, w, _ = R.init("gloo")
    assert (r, w) == (rank, world)
    R.barrier(w)
    # each replica "measured" its own step time and processed its own bytes
    ms_mine = 2.0 + rank           # rank 1 is the slow one
    bytes_mine = 1000 * (rank + 1)
    gbs, ms = R.job_throughput_gbs(bytes_mine, ms_mine, w)
    # host planner on every rank: identical plans, no communication needed (the plan is deterministic)
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import synth
    wl = synth.config(1, pool_factor=2.5)
    desc, keep = B.make_desc(wl.n_layers, wl.latent_dim, wl.rope_dim, wl.page_size, wl.dtype, wl.pairing,
                             wl.row_bytes, wl.n_slots, wl.inv_freq, None)
    plan = B.leyline_plan(desc, B.FRESH, wl.seq_lens, wl.pt_offsets, wl.pages, wl.directives, wl.free_pages)
    sig = torch.tensor([int(plan.info.bytes_read), int(plan.info.bytes_written), int(plan.info.total_new_tokens),
                        int(np.asarray(plan.new_pages, dtype=np.int64).sum())], dtype=torch.int64)
    plan.close()
    import torch.distributed as dist
    gathered = [torch.zeros_like(sig) for _ in range(w)]
    dist.all_gather(gathered, sig)
    q.put((rank, gbs, ms, [g.tolist() for g in gathered]))
    R.finish(w)


@pytest.mark.timeout(300)
def test_world2_gloo_replicas():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=240) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, gbs, ms, sigs in res:
        assert ms == 3.0                                         # MAX over ranks
        assert gbs == pytest.approx(3000 / 3.0e-3 / 1e9)         # SUM of bytes / max time
        assert sigs[0] == sigs[1] and sigs[0][0] > 0             # same plan on both ranks


def test_single_process_is_identity():
    from paper_2606_01065_b200 import replicas as R
    assert R.max_over_ranks(1.5, 1) == 1.5
    assert R.sum_over_ranks(7, 1) == 7.0
    gbs, ms = R.job_throughput_gbs(2_000_000_000, 1.0, 1)
    assert ms == 1.0 and gbs == pytest.approx(2000.0)


ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.timeout(300)
def test_bench_gpus_n_starts_n_ranks_by_itself():
    """`python bench.py --gpus 2` with no launcher must start two ranks and report n_gpus = 2, the slowest rank's step
    time and the units of BOTH ranks (here with the test-only host-sleep step on gloo, no GPU)."""
    import json
    import subprocess
    import sys
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--stub-step-ms", "5", "--backend", "gloo",
                        "--steps", "3", "--warmup", "1"], capture_output=True, text=True, cwd=ROOT, timeout=280,
                       env={k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")})
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                       # rank 0 alone prints
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["steps"] == 3 and out["warmup"] == 1
    assert out["ms_per_step"] >= 6.0                             # rank 1 sleeps 5 + 1 ms: MAX over ranks
    assert out["units_all_ranks"] == 3_000_000
    assert out["value"] == pytest.approx(3_000_000 / (out["ms_per_step"] * 1e-3) / 1e9)


def test_bench_gpus_n_fails_loudly_when_the_box_has_fewer_devices():
    import subprocess
    import sys
    if torch.cuda.device_count() >= 2:
        pytest.skip("this box has two devices")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, cwd=ROOT, timeout=280,
                       env={k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")})
    assert r.returncode == 2 and "--gpus 2" in r.stderr and not r.stdout.strip()

"""GPU parity: the CUDA library through its C ABI vs the CPU oracle, element by element, on the same seeded
inputs (tests/parity.py states the bar).  Small and medium cases compare every layer and the whole pool
(so every byte the mode must not write is checked too); the full BASELINE.json configs run in the launch
configuration bench.py times (all layers, one call) and compare EVERY layer, whole pool, one layer at a time, the
oracle on a thread per layer (no sanitizer exists on this GPU pool: bytes are the race detector of the hazard mover)."""
import numpy as np
import pytest
import torch

import oracle as O
from parity import assert_plan_equal, compare_all_layers, compare_layer, layer_checksum, oracle_plan, oracle_slot_list
from paper_2606_01065_b200 import synth
from test_plan_host import tiny_workload

pytestmark = pytest.mark.gpu

MODES = [O.FRESH, O.INPLACE_MOVE, O.ROTATE_ONLY]
MODE_NAME = {O.FRESH: "fresh", O.INPLACE_MOVE: "inplace", O.ROTATE_ONLY: "rotate_only"}
# leyline_tuning.kernel: the a3/a4 mover.  1 = k_move_rows (register-staged), 2 = k_move_bulk (TMA bulk copies through
# shared memory); 0 = the planner's choice (bulk for unpadded rows in pages of >= 16 rows or of >= 1 KB each), which is what bench.py times.
MOVERS = [1, 2]


STREAM_BYTES = 1 << 30      # caches larger than this are compared layer by layer from regenerated inputs


def run_and_compare(w, mode, check_layers=None, tuning=None, host_resident=False, inserts_prefilled=False, **launch):
    """check_layers=None compares EVERY layer, whole pool.  Small caches are snapshotted on the host before the splice;
    large ones (the full BASELINE.json configs) are compared one layer at a time against inputs regenerated from their
    seeds (parity.compare_all_layers), with the oracle running on a thread per layer."""
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    if tuning:
        B.leyline_set_tuning(**tuning)
    try:
        cache = harness.DeviceCache(w, "cuda:0", host_resident=host_resident)
        check_layers = list(range(w.n_layers)) if check_layers is None else check_layers
        stream = not host_resident and w.layer_bytes * len(check_layers) > STREAM_BYTES
        if stream:
            sums = {l: layer_checksum(cache.pools[l]) for l in check_layers}
        else:
            # a pinned host pool IS a cpu tensor: .cpu() would alias it, and the splice then overwrites the snapshot
            old = {l: (cache.pools[l].clone() if host_resident else cache.pools[l].cpu()).numpy() for l in check_layers}
        if inserts_prefilled:
            cache.repl = None                 # layer_repl = NULL: the caller prefills the replacement slots
        plan, pt, idx = harness.run_workload(cache, mode, **launch)
        torch.cuda.synchronize()
    finally:
        if tuning:
            B.leyline_set_tuning()
    bm = oracle_plan(w, mode)
    assert_plan_equal(plan, bm, mode)
    n_tok = int(plan.info.total_new_tokens)
    np.testing.assert_array_equal(idx.cpu().numpy()[:n_tok], oracle_slot_list(bm))          # a2, bit-exact
    if mode != O.ROTATE_ONLY:
        n_pg = int(plan.info.total_new_pages)
        want = np.concatenate([rm.new_pages for rm in bm.requests]) if n_pg else np.zeros(0, np.int32)
        np.testing.assert_array_equal(pt.cpu().numpy()[:n_pg], want)
    if stream:
        import time
        t0 = time.perf_counter()
        stats = compare_all_layers(w, bm, mode, cache, check_layers, inserts_prefilled, checksums=sums)
        print(f"[parity] {w.name} {MODE_NAME[mode]}: {len(check_layers)} of {w.n_layers} layers, whole pools "
              f"({w.layer_bytes * len(check_layers) / 2**30:.1f} GiB), compared in {time.perf_counter() - t0:.1f} s")
    else:
        stats = []
        for l in check_layers:
            stats.append(compare_layer(w, bm, mode, old[l], cache.pools[l].cpu().numpy(),
                                       None if inserts_prefilled else cache.repl[l].cpu().numpy(),
                                       cache.scales[l], layer=l, inserts_prefilled=inserts_prefilled))
    plan.close()
    tot = sum(s["rotated_elems"] for s in stats)
    if tot:
        worst = max(s["max_ord"] for s in stats)
        eq = sum(s["frac_equal"] * s["rotated_elems"] for s in stats) / tot
        print(f"[parity] {w.name} {MODE_NAME[mode]}: rotated elems {tot}, max ordinal distance {worst}, "
              f"bit-equal {eq:.6f}, cancellation-floor passes {sum(s['n_floor'] for s in stats)}")
        if w.dtype == synth.DT_BF16:
            assert eq > 0.99          # fp32 trig + one RNE: almost every element is the oracle's exact code
    return stats


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("mover", [0] + MOVERS)
def test_config1_all_modes(mode, mover):
    run_and_compare(synth.config(1, pool_factor=2.5), mode, tuning={"kernel": mover})


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("dtype", [synth.DT_BF16, synth.DT_FP8])
@pytest.mark.parametrize("pairing", [synth.NEOX, synth.INTERLEAVED])
@pytest.mark.parametrize("mover", MOVERS)
def test_randomised_small(mode, dtype, pairing, mover):
    rng = np.random.default_rng(77 + 10 * mode + 3 * dtype + pairing)
    for _ in range(12):
        w = tiny_workload(rng, dtype=dtype)
        w.pairing = pairing
        run_and_compare(w, mode, tuning={"kernel": mover})


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("mover,tile_rows", [(1, 1), (1, 7), (1, 32), (2, 1), (2, 7), (2, 32), (2, 64)])
def test_medium_many_tiles_ragged(mode, mover, tile_rows):
    """Several pages, ragged tails, tiles that straddle pages, growth and shrink in one request, YaRN thetas."""
    w = synth.Workload("medium", 3, [3000, 1, 0, 2777], 16, inv_freq=synth.yarn_inv_freq(),
                       directives=[(0, 5, 5, 40, 0, 0), (0, 100, 900, 3, 0, 0), (0, 1500, 1501, 333, 0, 0),
                                   (0, 2990, 3000, 0, 0, 0),
                                   (1, 0, 1, 0, 0, 0),
                                   (3, 0, 17, 500, 0, 0), (3, 1000, 1700, 0, 0, 0), (3, 2776, 2777, 2, 0, 0)],
                       seed=11, pool_factor=3.0, extra_pages=80).finalize()
    run_and_compare(w, mode, tuning={"kernel": mover, "tile_rows": tile_rows})


@pytest.mark.parametrize("mode", [O.FRESH, O.INPLACE_MOVE])
@pytest.mark.parametrize("stages,layer_group", [(3, 1), (4, 3), (8, 8)])
def test_bulk_ring_geometry(mode, stages, layer_group):
    """The bulk mover's shared-memory ring at its smallest and largest depth, layer groups that do not divide the
    layer count (5 layers), growth and shrink in one request."""
    w = synth.Workload("ring", 5, [2100, 900], 16, inv_freq=synth.yarn_inv_freq(),
                       directives=[(0, 7, 40, 300, 0, 0), (0, 900, 1700, 5, 0, 0), (1, 100, 101, 77, 0, 0)],
                       seed=21, pool_factor=3.0, extra_pages=60).finalize()
    run_and_compare(w, mode, tuning={"kernel": 2, "tile_rows": 16, "stages": stages, "layer_group": layer_group})


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("dtype", [synth.DT_BF16, synth.DT_FP8])
@pytest.mark.parametrize("mover", MOVERS)
def test_per_layer_pairing(mode, dtype, mover):
    """the pairing helper "reads is_neox_style per layer" -- a cache whose layers mix the two conventions
    (G20): each layer must be rotated with its own pairing, in every mode, in one call."""
    rng = np.random.default_rng(133)
    w = tiny_workload(rng, P=16, n_req=3, dtype=dtype)
    w.n_layers = 5
    w.layer_pairing = [synth.NEOX, synth.INTERLEAVED, synth.INTERLEAVED, synth.NEOX, synth.INTERLEAVED]
    w.pairing = synth.NEOX
    run_and_compare(w, mode, tuning={"kernel": mover})


def test_per_layer_pairing_one_convention_only():
    """All layers interleaved through the per-layer array while the cache-wide flag says NeoX: the array wins."""
    w = synth.config(1, pool_factor=2.5)
    w.layer_pairing = [synth.INTERLEAVED, synth.INTERLEAVED]
    for mode in MODES:
        run_and_compare(w, mode)


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("mover", MOVERS)
def test_prefetched_tables(mode, mover):
    """leyline_plan_prefetch: tables uploaded on the library's copy stream, the launch only waits on the event."""
    rng = np.random.default_rng(77)
    run_and_compare(tiny_workload(rng, P=16, n_req=3), mode, tuning={"kernel": mover}, prefetch=True)
    # a prefetched plan that is never launched gives its tables back on the copy stream
    from paper_2606_01065_b200 import harness
    w = tiny_workload(rng, P=16, n_req=2)
    d, keep = harness.DeviceCache(w, "cuda:0", fill=False).desc()
    for _ in range(3):
        harness.plan_workload(w, mode, d).prefetch().close()
    torch.cuda.synchronize()
    del keep


@pytest.mark.parametrize("prefetch", [False, True])
def test_relaunching_a_fresh_plan_repeats_the_result(prefetch):
    """The second launch of a plan must zero its ticket counters itself (the upload zeroes them only once)."""
    run_and_compare(synth.config(1, pool_factor=2.5), O.FRESH, prefetch=prefetch, launches=3)


@pytest.mark.parametrize("mode", MODES)
def test_identity_and_degenerate(mode):
    # no directives at all, no-op directives, |R| = |span| (Delta = 0: everything downstream is a byte copy, G19)
    for dirs in ([], [(0, 10, 10, 0, 0, 0)], [(0, 64, 128, 64, 0, 0)], [(0, 0, 0, 0, 0, 0), (0, 500, 500, 0, 0, 0)]):
        w = synth.Workload("ident", 2, [500], 8, inv_freq=synth.rope_inv_freq(), directives=dirs, seed=3,
                           pool_factor=3.0, extra_pages=16).finalize()
        stats = run_and_compare(w, mode)
        assert all(s["rotated_elems"] == 0 for s in stats)


def test_special_values_survive():
    """-0.0, subnormals and large magnitudes in K_pe: byte-exact where C = 0, within tolerance where rotated."""
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    w = synth.Workload("special", 1, [256], 4, inv_freq=synth.rope_inv_freq(), directives=[(0, 100, 110, 3, 0, 0)],
                       seed=5, pool_factor=3.0, extra_pages=8).finalize()
    cache = harness.DeviceCache(w, "cuda:0")
    v = cache.pools[0].view(torch.int16)
    # -0.0, +-smallest subnormal, largest subnormal, 2^125, smallest normal, 1.0
    specials = torch.tensor([-32768, 1, -32767, 0x007F, 0x7E00, 0x0080, 0x3F80], dtype=torch.int16, device="cuda:0")
    v[::13] = specials[torch.arange(v[::13].numel(), device="cuda:0") % len(specials)]
    old = cache.pools[0].cpu().numpy()
    plan, pt, idx = harness.run_workload(cache, B.FRESH)
    torch.cuda.synchronize()
    bm = oracle_plan(w, B.FRESH)
    compare_layer(w, bm, B.FRESH, old, cache.pools[0].cpu().numpy(), cache.repl[0].cpu().numpy(), 1.0)


@pytest.mark.parametrize("mode,mover", [(O.FRESH, 1), (O.FRESH, 2), (O.ROTATE_ONLY, 0), (O.INPLACE_MOVE, 1),
                                        (O.INPLACE_MOVE, 2)])
def test_config2_dsv2lite(mode, mover):
    run_and_compare(synth.config(2, pool_factor=2.2), mode, tuning={"kernel": mover})        # all 27 layers


@pytest.mark.parametrize("cfg", [3, "3m"])
@pytest.mark.parametrize("mode", MODES)
def test_config3_dsv3_full_size(cfg, mode):
    # default tuning = the launch configuration bench.py times (bulk mover for FRESH / INPLACE_MOVE)
    run_and_compare(synth.config(cfg, pool_factor=2.0), mode)                                # all 61 layers


@pytest.mark.parametrize("mode", [O.FRESH, O.INPLACE_MOVE])
def test_config3m_row_mover_full_size(mode):
    run_and_compare(synth.config("3m", pool_factor=2.0), mode, tuning={"kernel": 1})         # all 61 layers


def _release_cached_device_memory():
    """mem_get_info counts what torch's caching allocator still holds from earlier tests as used: hand it back first, so
    that "free" means free (without this the 147-GB test took its 12-layer branch whenever it ran behind the 92-GB one)."""
    import gc
    gc.collect()
    torch.cuda.synchronize()
    torch.cuda.empty_cache()


def test_config4_batched_inplace_full_size():
    w = synth.config(4)           # 64 x 16K x 61 layers, one shared pool (~92 GB with the 25 % spare pages)
    _release_cached_device_memory()
    free, total = torch.cuda.mem_get_info(0)
    if free < w.layer_bytes * w.n_layers * 1.08:
        # a B200 (>= 170 GiB in total) must run this at full size: on such a device a shortage is a failure, not a skip
        assert total < 170 << 30, f"{free / 2**30:.0f} GiB free of {total / 2**30:.0f}: something else holds the device's memory"
        pytest.skip(f"needs {w.layer_bytes * w.n_layers / 2**30:.0f} GiB of device memory")
    run_and_compare(w, O.INPLACE_MOVE)                   # all 61 layers, 1.5 GB each


def test_config4_batched_fresh_full_size():
    # FRESH on the batched workload needs a second set of pages: 147 GB of pools for all 61 layers, which a 180 GB B200
    # holds; on a smaller or busier device the same plan runs on 12 layers (layers are independent buffers under one plan)
    w = synth.config(4, pool_factor=2.0)
    _release_cached_device_memory()
    free, total = torch.cuda.mem_get_info(0)
    if free < (w.layer_bytes * (w.n_layers + 1)) * 1.04 + (2 << 30):
        # the 12-layer fallback is for smaller devices only: on a B200 (>= 170 GiB in total) the test fails rather than
        # pass on a fifth of the layers without saying so
        assert total < 170 << 30, f"{free / 2**30:.0f} GiB free of {total / 2**30:.0f}: config 4 FRESH needs 147 GB of pools"
        w = synth.config(4, pool_factor=2.2, n_layers=12)
    run_and_compare(w, O.FRESH)


@pytest.mark.parametrize("mode", [O.FRESH, O.INPLACE_MOVE, O.ROTATE_ONLY])
def test_config5_fp8_full_size(mode):
    run_and_compare(synth.config(5, pool_factor=2.2), mode)                  # all 61 layers


# ----------------------------------------------------------------------------- full-width K

def heads_workload(name, heads, d, latent, dtype, pairing, theta, page=16, layers=2):
    return synth.Workload(name, layers, [2100, 900, 64], page, dtype=dtype, pairing=pairing, latent_dim=latent, rope_dim=d,
                          rope_heads=heads, inv_freq=synth.rope_inv_freq(d, theta),
                          directives=[(0, 7, 40, 300, 0, 0), (0, 900, 1700, 5, 0, 0), (1, 100, 101, 77, 0, 0),
                                      (2, 0, 64, 1, 0, 0)],
                          seed=31, pool_factor=3.0, extra_pages=60).finalize()


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("pairing", [synth.NEOX, synth.INTERLEAVED])
@pytest.mark.parametrize("heads,d,latent,dtype,theta", [
    (8, 128, 0, synth.DT_BF16, 5.0e5),      # GQA, Llama-3.1-style (Table 8 row 3)
    (8, 128, 0, synth.DT_FP8, 1.0e6),       # GQA, Qwen-3-style, fp8 storage
    (4, 96, 0, synth.DT_BF16, 1.0e4),       # Phi-3-style head_dim 96: 12 chunks per head
    (3, 96, 64, synth.DT_BF16, 1.0e4),      # odd head count behind a position-free prefix (K and V sharing a row)
    (2, 64, 512, synth.DT_BF16, 1.0e4),     # two rotated heads behind an MLA-sized latent
    (1, 32, 16, synth.DT_FP8, 1.0e4),       # smallest band the kernels take: one head of two chunks
])
def test_full_width_heads(mode, pairing, heads, d, latent, dtype, theta):
    run_and_compare(heads_workload("heads", heads, d, latent, dtype, pairing, theta), mode)


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("page", [1, 4])
def test_full_width_small_pages(mode, page):
    """Token-level slots / tiny pages: the bulk mover degenerates to one copy per row, inserts of ROTATE_ONLY too."""
    run_and_compare(heads_workload("heads_p", 8, 128, 0, synth.DT_BF16, synth.NEOX, 5.0e5, page=page), mode)


@pytest.mark.parametrize("cfg", ["gqa", "mha96"])
@pytest.mark.parametrize("mode", MODES)
def test_full_width_full_size(cfg, mode):
    w = synth.config(cfg, pool_factor=2.0)
    run_and_compare(w, mode)                                                # all 32 layers


@pytest.mark.parametrize("mode,mover", [(O.FRESH, 1), (O.FRESH, 2), (O.INPLACE_MOVE, 1), (O.INPLACE_MOVE, 2), (O.ROTATE_ONLY, 0)])
def test_byte_offsets_beyond_2_to_the_31(mode, mover):
    """SURVEY.md section 7 "64-bit addressing" (G17): slot ids fit int32, byte offsets do not.  One layer whose pool is
    4.6 GiB (4 M slots x 1152 B) with the request's pages scattered over all of it by the seeded permutation, so about
    half of the rows every kernel touches sit beyond byte 2^31 and a quarter beyond 2^32.  Whole-pool comparison."""
    w = synth.Workload("big_pool", 1, [8192 + 37], 64, inv_freq=synth.yarn_inv_freq(),
                       directives=[(0, 700, 1900, 333, 0, 0), (0, 4000, 4001, 0, 0, 0), (0, 6000, 6000, 77, 0, 0)],
                       seed=31, pool_factor=1.0, extra_pages=(1 << 16) - 129).finalize()
    assert w.layer_bytes > (1 << 32)
    slots = w.pages.astype(np.int64) * 64
    assert (slots * w.row_bytes > (1 << 31)).mean() > 0.3 and (slots * w.row_bytes > (1 << 32)).any()
    run_and_compare(w, mode, tuning={"kernel": mover})


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("mover", MOVERS)
def test_host_resident_cache_is_spliced_over_pcie(mode, mover):
    """include/leyline.h: layer pointers may be pinned host memory.  The same kernels gather from and scatter to the
    host-resident pools (bench.py's e2e leg); results and untouched bytes must match the oracle exactly as on device."""
    rng = np.random.default_rng(909)
    w = tiny_workload(rng, P=16, n_req=3)
    run_and_compare(w, mode, tuning={"kernel": mover}, host_resident=True)
    if mode != O.INPLACE_MOVE:
        run_and_compare(synth.config(1, pool_factor=2.5), mode, tuning={"kernel": mover}, host_resident=True)


@pytest.mark.parametrize("mode", MODES)
def test_forget_directives_truncate_on_device_too(mode):
    """a FORGET directive routes to a prefix-trimmed re-prefill -- the request is cut at the directive's
    start (new coordinates), everything behind it is released and no kernel touches it.  Mixed with AMORTIZE edits."""
    rng = np.random.default_rng(4242)
    done = 0
    while done < 6:
        w = tiny_workload(rng, forget=True)
        if not any(d[5] == synth.FORGET for d in w.directives):
            continue
        run_and_compare(w, mode)
        done += 1


def test_two_plans_in_flight_on_two_streams():
    """Plans own their tables, tickets and hazard flags, so independent splices may overlap on different streams
    (a server splices several requests' caches concurrently); each result must equal its own oracle."""
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    ws = [synth.config(2, pool_factor=2.2, n_layers=3), synth.config("3m", pool_factor=2.0, n_layers=2)]
    modes = [O.INPLACE_MOVE, O.FRESH]
    caches = [harness.DeviceCache(w, "cuda:0") for w in ws]
    olds = [[p.cpu().numpy() for p in c.pools] for c in caches]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    outs = []
    for rep in range(2):                      # second round: FRESH again on stream 1 while a rotate runs on stream 0
        for c, m, s in zip(caches, modes, streams):
            if rep == 1 and m != O.FRESH:
                continue
            outs.append((c, m, harness.run_workload(c, m, stream=s, prefetch=(rep == 0))))
    torch.cuda.synchronize()
    for (c, m, (plan, pt, idx)), old in zip(outs[:2], olds):
        bm = oracle_plan(c.w, m)
        assert_plan_equal(plan, bm, m)
        np.testing.assert_array_equal(idx.cpu().numpy()[:int(plan.info.total_new_tokens)], oracle_slot_list(bm))
        for l in range(c.w.n_layers):
            compare_layer(c.w, bm, m, old[l], c.pools[l].cpu().numpy(), c.repl[l].cpu().numpy(), c.scales[l], layer=l)
    for _, _, (plan, _, _) in outs:
        plan.close()


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("mover", MOVERS)
def test_caller_prefills_replacement_slots(mode, mover):
    """PAPER.md:405(b): in the paper step (b) is the model's prefill of R into the new slots.  With layer_repl = NULL
    the library allocates those slots in the new maps and never writes their bytes; everything else is as usual."""
    rng = np.random.default_rng(405)
    for _ in range(4):
        run_and_compare(tiny_workload(rng, P=int(rng.choice([1, 16]))), mode, tuning={"kernel": mover}, inserts_prefilled=True)
    run_and_compare(synth.config(1, pool_factor=2.5), mode, tuning={"kernel": mover}, inserts_prefilled=True)


@pytest.mark.parametrize("mode", [O.FRESH, O.ROTATE_ONLY])
def test_paper_appendix_b_shape(mode):
    """185 matched chunks of ~130 tokens copied to fresh token-level slots and rotated in one call (the shape of the
    paper's bytes_rotated / kernel-time counters), and the same rotated where they sit."""
    run_and_compare(synth.config("appB", pool_factor=2.0), mode)


def test_launch_argument_errors_are_refused_before_any_launch():
    """leyline.h: the launch entry points return only argument / launch errors -- and nothing is written when they do."""
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    w = synth.config(1, pool_factor=2.5)
    cache = harness.DeviceCache(w, "cuda:0")
    before = [p.clone() for p in cache.pools]
    desc, keep = cache.desc()
    idx = torch.full((8192,), -5, dtype=torch.int32, device="cuda:0")

    def status_of(fn):
        with pytest.raises(B.LeylineError) as ei:
            fn()
        return ei.value.status

    rot = harness.plan_workload(w, B.ROTATE_ONLY, desc)
    fresh = harness.plan_workload(w, B.FRESH, desc)
    inpl = harness.plan_workload(w, B.INPLACE_MOVE, desc)
    other = [torch.empty_like(p) for p in cache.pools]
    # a plan of the wrong mode
    assert status_of(lambda: B.leyline_splice(rot, cache.pools, cache.pools, cache.repl, None, idx)) == B.E_INVALID
    assert status_of(lambda: B.leyline_rotate_inplace(fresh, cache.pools, cache.repl, idx)) == B.E_INVALID
    # INPLACE_MOVE must read and write the same buffers
    assert status_of(lambda: B.leyline_splice(inpl, cache.pools, other, cache.repl, None, idx)) == B.E_INVALID
    # a NULL or misaligned layer pointer
    bad = [cache.pools[0].data_ptr() + 8, cache.pools[1].data_ptr()]
    assert status_of(lambda: B.leyline_splice(fresh, bad, bad, cache.repl, None, idx)) == B.E_INVALID
    assert status_of(lambda: B.leyline_splice(fresh, [0, 0], [0, 0], cache.repl, None, idx)) == B.E_INVALID
    # wrong number of layers is caught by the binding itself
    with pytest.raises(ValueError):
        B.leyline_splice(fresh, cache.pools[:1], cache.pools, cache.repl, None, idx)
    torch.cuda.synchronize()
    assert all(bool((a == b).all()) for a, b in zip(before, cache.pools)) and bool((idx == -5).all())
    # and the plans are still usable afterwards
    B.leyline_splice(fresh, cache.pools, cache.pools, cache.repl, None, idx)
    torch.cuda.synchronize()
    assert int(idx[0].item()) != -5
    for p in (rot, fresh, inpl):
        p.close()
    del keep


def test_two_host_threads_drive_the_library_at_once():
    """ctypes releases the GIL, so two Python threads really are inside libleyline.so together: planning, pinned
    staging, the table pool and the launches are shared state that must hold up (each thread on its own stream)."""
    import threading
    from paper_2606_01065_b200 import harness
    ws = [synth.config(2, pool_factor=2.2, n_layers=2), synth.config(1, pool_factor=2.5)]
    modes = [O.FRESH, O.ROTATE_ONLY]
    caches = [harness.DeviceCache(w, "cuda:0") for w in ws]
    olds = [[p.cpu().numpy() for p in c.pools] for c in caches]
    torch.cuda.synchronize()
    results, errors = [None, None], []

    def work(i):
        try:
            s = torch.cuda.Stream()
            last = None
            for rep in range(20 if modes[i] == O.FRESH else 1):      # FRESH is idempotent: hammer it
                if last is not None:
                    last[0].close()
                last = harness.run_workload(caches[i], modes[i], stream=s, prefetch=bool(rep % 2))
            s.synchronize()
            results[i] = last
        except Exception as ex:        # surfaced in the main thread
            errors.append(ex)

    threads = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    torch.cuda.synchronize()
    for i, (c, m) in enumerate(zip(caches, modes)):
        plan, pt, idx = results[i]
        bm = oracle_plan(c.w, m)
        assert_plan_equal(plan, bm, m)
        np.testing.assert_array_equal(idx.cpu().numpy()[:int(plan.info.total_new_tokens)], oracle_slot_list(bm))
        for l in range(c.w.n_layers):
            compare_layer(c.w, bm, m, olds[i][l], c.pools[l].cpu().numpy(), c.repl[l].cpu().numpy(), c.scales[l], layer=l)
        plan.close()


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("heads,d,latent,dtype", [
    (128, 256, 0, synth.DT_BF16),      # the largest row the library takes: 128 heads x 256 = 65,536 B (one row per tile)
    (2, 512, 0, synth.DT_BF16),        # the widest head: 64 chunks
    (128, 32, 2048, synth.DT_FP8),     # most heads of the narrowest kind (one chunk per half) behind a wide latent
    (1, 32, 32736, synth.DT_BF16),     # a 64 KB row that is nearly all latent, with a small bf16 band
])
def test_maximum_geometries(mode, heads, d, latent, dtype):
    """leyline.h limits: head <= 64 chunks, <= 128 heads, rows <= 64 KB."""
    w = synth.Workload("max_geom", 2, [300, 41], 16, dtype=dtype, latent_dim=latent, rope_dim=d, rope_heads=heads,
                       inv_freq=synth.rope_inv_freq(d, 1.0e4),
                       directives=[(0, 10, 50, 7, 0, 0), (0, 200, 201, 30, 0, 0), (1, 0, 3, 0, 0, 0)],
                       seed=64, pool_factor=3.0, extra_pages=8).finalize()
    assert w.row_bytes <= 65536
    run_and_compare(w, mode)


def test_geometries_beyond_the_limits_are_refused():
    from paper_2606_01065_b200 import binding as B
    for heads, d, latent in ((129, 16, 0), (1, 1024, 0), (128, 256, 16), (1, 24, 0)):
        w = synth.Workload("too_big", 1, [16], 16, latent_dim=latent, rope_dim=d, rope_heads=heads,
                           inv_freq=synth.rope_inv_freq(d, 1.0e4), directives=[], seed=1, pool_factor=2.0).finalize()
        desc, keep = B.make_desc(1, latent, d, 16, B.BF16, B.NEOX, w.row_bytes, w.n_slots, w.inv_freq, rope_heads=heads)
        with pytest.raises(B.LeylineError) as ei:
            B.leyline_plan(desc, B.FRESH, w.seq_lens, w.pt_offsets, w.pages, [], w.free_pages)
        assert ei.value.status == B.E_UNSUPPORTED, (heads, d, latent)


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("page", [256, 1024])
def test_large_pages(mode, page):
    """Pages larger than a tile and larger than the requests' edits: tiles never straddle more than two pages, runs are
    capped by the tile, the boundary page of FRESH is copied from its head."""
    w = synth.Workload("large_pages", 2, [5000, 1300], page, inv_freq=synth.yarn_inv_freq(),
                       directives=[(0, 300, 1100, 77, 0, 0), (0, 3000, 3001, 600, 0, 0), (1, 1290, 1300, 0, 0, 0)],
                       seed=256, pool_factor=3.0, extra_pages=4).finalize()
    for mover in MOVERS:
        run_and_compare(w, mode, tuning={"kernel": mover})


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("mixed", [False, True])
def test_more_layers_than_one_launch_holds(mode, mixed):
    """LEYLINE_MAX_LAYERS_PER_LAUNCH = 128: 130 layers (two conventions mixed) take several launches per mover; hazard
    flags are numbered per launch."""
    rng = np.random.default_rng(130)
    w = tiny_workload(rng, P=4, n_req=2)
    w.n_layers = 130
    w.layer_pairing = [int(x) for x in rng.integers(0, 2, size=130)] if mixed else None     # one convention: 128 + 2 layers
    for mover in MOVERS:
        run_and_compare(w, mode, tuning={"kernel": mover})


def fuzz_workload(rng):
    """Several requests of up to a few thousand tokens, up to 6 directives each with the edit shapes of the paper's
    randomised suites (spans U[8,200] or long, |R| in [0, 2|span|], both signs), random page size,
    storage type, pairing and band geometry."""
    P = int(rng.choice([1, 2, 8, 16, 64, 128]))
    n_req = int(rng.integers(1, 7))
    seq_lens = [int(rng.integers(0, 6000)) for _ in range(n_req)]
    dirs = []
    for r, L in enumerate(seq_lens):
        k = int(rng.integers(0, 7))
        cuts = np.sort(rng.integers(0, L + 1, size=2 * k))
        for j in range(k):
            s, e = int(cuts[2 * j]), int(cuts[2 * j + 1])
            if rng.random() < 0.6:
                e = min(e, s + int(rng.integers(8, 201)))
            n = int(rng.integers(0, 2 * (e - s) + 3)) if rng.random() < 0.85 else 0
            dirs.append((r, s, e, min(n, 700), 0, 0))
    geom = [(512, 64, 1), (0, 128, 2), (64, 96, 3), (16, 32, 1)][int(rng.integers(0, 4))]
    w = synth.Workload("fuzz", 2, seq_lens, P, dtype=int(rng.integers(0, 2)), pairing=int(rng.integers(0, 2)),
                       latent_dim=geom[0], rope_dim=geom[1], rope_heads=geom[2],
                       inv_freq=synth.rope_inv_freq(geom[1], float(rng.choice([1.0e4, 5.0e5]))), directives=dirs,
                       seed=int(rng.integers(1 << 30)), pool_factor=2.5, extra_pages=sum(d[3] for d in dirs) // P + 16)
    return w.finalize()


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("seed", range(4))
def test_fuzz_medium(mode, seed):
    rng = np.random.default_rng(31337 + 17 * seed + mode)
    for _ in range(6):
        w = fuzz_workload(rng)
        tuning = {"kernel": int(rng.choice([0, 2])), "tile_rows": int(rng.choice([0, 0, 5, 16, 64])),
                  "stages": int(rng.choice([0, 3, 5])), "layer_group": int(rng.choice([0, 1, 2]))}
        if w.rope_heads == 1 and w.rope_dim in (32, 64) and rng.random() < 0.4:
            tuning = {"kernel": 1, "tile_rows": int(rng.choice([0, 3, 32]))}
        run_and_compare(w, mode, tuning=tuning, prefetch=bool(rng.integers(0, 2)))


@pytest.mark.parametrize("mover", MOVERS)
@pytest.mark.parametrize("src_on_host", [False, True])
def test_fresh_into_a_separate_pool(mover, src_on_host):
    """leyline.h: for FRESH, layer_dst may differ from layer_src.  Only the fresh pages are written, into layer_dst
    (page ids are the same in both pools); the source pool -- here optionally a host-resident, swapped-out copy -- is
    never written, and nothing else of the destination is touched."""
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    rng = np.random.default_rng(606 + mover)
    for w in (tiny_workload(rng, P=16, n_req=3), synth.config(1, pool_factor=2.5)):
        B.leyline_set_tuning(kernel=mover)
        try:
            cache = harness.DeviceCache(w, "cuda:0", host_resident=src_on_host)
            old = [p.clone().numpy() if src_on_host else p.cpu().numpy() for p in cache.pools]
            dst = [torch.full((w.layer_bytes,), 0xA5, dtype=torch.uint8, device="cuda:0") for _ in cache.pools]
            desc, keep = cache.desc()
            plan = harness.plan_workload(w, B.FRESH, desc)
            B.leyline_splice(plan, cache.pools, dst, cache.repl, None, None)
            torch.cuda.synchronize()
        finally:
            B.leyline_set_tuning()
        bm = oracle_plan(w, O.FRESH)
        assert_plan_equal(plan, bm, O.FRESH)
        fresh_pages = plan.new_pages[~np.isin(plan.new_pages, w.pages)]        # ids taken from the free list
        rows = (fresh_pages.astype(np.int64)[:, None] * w.page_size + np.arange(w.page_size)[None, :]).reshape(-1)
        for l in range(w.n_layers):
            src_now = cache.pools[l].numpy() if src_on_host else cache.pools[l].cpu().numpy()
            np.testing.assert_array_equal(src_now, old[l])                      # the source is never written
            want = O.splice_layer(w.dtype, w.pairing, w.latent_dim, w.rope_dim, w.row_bytes, w.inv_freq, cache.scales[l],
                                  old[l], cache.repl[l].cpu().numpy(), bm).reshape(-1, w.row_bytes)
            got = dst[l].cpu().numpy().reshape(-1, w.row_bytes)
            mask = np.zeros(len(got), bool)
            mask[rows] = True
            assert (got[~mask] == 0xA5).all()                                   # nothing outside the fresh pages
            # inside the fresh pages: rows the plan wrote equal the oracle's; slots past L_new in a last page stay canary
            live = np.zeros(len(got), bool)
            for rm in bm.requests:
                live[rm.slot_new.astype(np.int64)] = True
            live &= mask
            assert (got[mask & ~live] == 0xA5).all()
            gl, wl = got[live], want[live]
            band0 = w.latent_dim * w.elem_bytes
            np.testing.assert_array_equal(gl[:, :band0], wl[:, :band0])
            d = np.abs(_ord16(gl[:, band0:]) - _ord16(wl[:, band0:]))
            assert d.max() <= 2
        plan.close()
        del keep


def _ord16(b):
    v = np.ascontiguousarray(b).view(np.uint16).astype(np.int32)
    return np.where(v & 0x8000, -(v & 0x7FFF), v & 0x7FFF)


@pytest.mark.parametrize("mode", MODES)
def test_paper_section_4_1_layout(mode):
    """The paper's constructed prompt: 5 prefix tokens, a 57-token chunk replaced by an 11-token stub,
    9 post tokens -- Delta = -46, L 71 -> 25, post tokens 62..70 -> 16..24 -- on the DeepSeek-V2-Lite shape (27 layers,
    token-level slots, NeoX and interleaved)."""
    g = __import__("helpers").golden("paper_worked_example.txt")
    pre, chunk, post, stub = int(g["pre_tokens"]), int(g["chunk_tokens"]), int(g["post_tokens"]), int(g["stub_tokens"])
    for pairing in (synth.NEOX, synth.INTERLEAVED):
        w = synth.Workload("sec4_1", 27, [pre + chunk + post], 1, pairing=pairing, inv_freq=synth.rope_inv_freq(64, 10000.0),
                           directives=[(0, pre, pre + chunk, stub, 0, 0)], seed=41, pool_factor=3.0, extra_pages=16).finalize()
        stats = run_and_compare(w, mode)
        bm = oracle_plan(w, mode)
        assert bm.requests[0].L_new == pre + chunk + post + int(g["delta"]) == 25
        assert sum(s["rotated_elems"] for s in stats) == post * 64 * 27


@pytest.mark.parametrize("mode", MODES)
def test_attention_logits_are_preserved_on_the_device(mode):
    """The property the method exists for (north_star "q.k logits are preserved for every query
    position"): after a three-directive splice executed by the CUDA path, (R(m) q) . K_pe_new[n] equals the
    relative-position logit computed from the RAW keys, for every query position m and every key n -- to the accuracy
    the bf16 cache allows (two roundings: the stored input, the stored output)."""
    from helpers import list_splice, rope_complex, to_storage, from_storage
    from paper_2606_01065_b200 import harness
    rng = np.random.default_rng(123)
    L, P, Dr, Dc = 700, 16, 64, 512
    inv = synth.yarn_inv_freq()
    dirs3 = [(40, 150, 9), (300, 301, 120), (600, 640, 0)]
    w = synth.Workload("logits", 2, [L], P, inv_freq=inv, directives=[(0, s, e, n, 0, 0) for s, e, n in dirs3], seed=5,
                       pool_factor=3.0, extra_pages=16).finalize()
    seq = list_splice(L, [(s, e, n, row) for (_, s, e, n, row, _) in w.directives])
    cache = harness.DeviceCache(w, "cuda:0", fill=False)
    slot_old = w.pages.astype(np.int64)[np.arange(L) // P] * P + np.arange(L) % P
    raws, raw_rs = [], []
    for l in range(w.n_layers):
        raw = rng.standard_normal((L, Dr))
        raw_r = rng.standard_normal((w.n_repl_rows, Dr))
        final_pos = np.array([n for n, tok in enumerate(seq) if tok[0] == "r"])          # replacement K_pe: roped at its
        order = np.array([tok[1] for tok in seq if tok[0] == "r"])                        # FINAL position (G12)
        pos_of_row = np.empty(w.n_repl_rows, np.int64)
        pos_of_row[order] = final_pos
        pool = np.zeros((w.n_slots, w.row_bytes), np.uint8)
        pool[slot_old] = to_storage(np.concatenate([rng.standard_normal((L, Dc)), rope_complex(raw, np.arange(L), inv)], axis=1), O.BF16)
        repl = to_storage(np.concatenate([rng.standard_normal((w.n_repl_rows, Dc)), rope_complex(raw_r, pos_of_row, inv)], axis=1), O.BF16)
        cache.pools[l].copy_(torch.from_numpy(pool.reshape(-1)))
        cache.repl[l].copy_(torch.from_numpy(repl.reshape(-1)))
        raws.append(raw)
        raw_rs.append(raw_r)
    plan, pt, idx = harness.run_workload(cache, mode)
    torch.cuda.synchronize()
    slots = idx.cpu().numpy()[:len(seq)].astype(np.int64)
    H = Dr // 2
    th = inv.astype(np.float64)
    worst = 0.0
    for l in range(w.n_layers):
        k_new = from_storage(cache.pools[l].cpu().numpy().reshape(-1, w.row_bytes)[slots], O.BF16)[:, Dc:]
        k_raw = np.stack([raws[l][tok[1]] if tok[0] == "o" else raw_rs[l][tok[1]] for tok in seq])
        kc = k_raw[:, :H] + 1j * k_raw[:, H:]
        q_raw = rng.standard_normal(Dr)
        qc = q_raw[:H] + 1j * q_raw[H:]
        for m in range(0, len(seq), 7):
            q_m = rope_complex(q_raw, m, inv)
            got = k_new @ q_m
            want = np.real(np.sum(qc[None, :] * np.conj(kc) * np.exp(1j * (m - np.arange(len(seq)))[:, None] * th[None, :]), axis=1))
            # bf16 K (two roundings, 2^-8 relative each at most) against an exact q: |err| <= 2^-7 * |q| * |k|
            bound = 2.0 ** -7 * np.linalg.norm(q_raw) * np.linalg.norm(k_raw, axis=1)
            assert (np.abs(got - want) <= bound).all()
            worst = max(worst, float((np.abs(got - want) / bound).max()))
    print(f"[logits] mode {mode}: worst |logit error| / (2^-7 |q||k|) = {worst:.3f}")
    plan.close()


def test_device_trig_table_matches_the_host_evaluation():
    """the cos/sin table of a launch is evaluated in fp64 ON THE DEVICE (k_index) -- fp64 product of
    the integer shift and theta_i, fp64 sincos, one rounding to fp32.  Against numpy's fp64 trig rounded once (an
    independent evaluation) it must agree to the last fp32 bit almost everywhere and never differ by more than one fp32
    ulp; the host query leyline_plan_trig_table must equal numpy exactly."""
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    for cfg, mode in (("appB", B.ROTATE_ONLY), (4, B.ROTATE_ONLY), ("3m", B.FRESH)):
        w = synth.config(cfg, pool_factor=2.0, n_layers=1)
        cache = harness.DeviceCache(w, "cuda:0", fill=False)
        for p in cache.pools + cache.repl:
            p.zero_()
        plan, pt, idx = harness.run_workload(cache, mode)
        torch.cuda.synchronize()
        dev, host, shifts = plan.trig_table_device, plan.trig_table, plan.trig_shifts
        assert len(shifts) >= 3
        phi = shifts.astype(np.float64)[:, None] * w.inv_freq.astype(np.float64)[None, :]
        want = np.stack([np.cos(phi), np.sin(phi)], axis=1).astype(np.float32)
        np.testing.assert_array_equal(host, want)
        d = np.abs(dev.view(np.int32).astype(np.int64) - want.view(np.int32).astype(np.int64))
        same_sign = np.signbit(dev) == np.signbit(want)
        assert ((d <= 1) & same_sign | (np.abs(dev.astype(np.float64) - want) < 1e-45)).all()
        assert (d == 0).mean() > 0.9999, (cfg, float((d == 0).mean()))
        plan.close()


# ----------------------------------------------------------------------------- a5 with 2-D TMA boxes (k_rotate_band_tma)

TMA = {"rotate_kernel": 2}


@pytest.mark.parametrize("cfg", [2, 3, "3m", 5])
def test_rotate_only_tma_full_size(cfg):
    """leyline_tuning.rotate_kernel = 2: the band of a page as one 2-D TMA box (64 rows x 128 B bf16 / 64 B fp8, pitch =
    row stride), loaded into shared memory, rotated there and stored back.  Every layer, whole pools."""
    from paper_2606_01065_b200 import binding as B
    w = synth.config(cfg, pool_factor=2.0)
    run_and_compare(w, O.ROTATE_ONLY, tuning=TMA)
    B.leyline_set_tuning(**TMA)
    try:
        with __import__("test_plan_host").make_plan(w, B.ROTATE_ONLY) as plan:
            assert plan.info.mover == 3 and plan.info.rot_tile_rows == 64
    finally:
        B.leyline_set_tuning()


@pytest.mark.parametrize("page", [16, 32, 64, 256])
@pytest.mark.parametrize("dtype", [synth.DT_BF16, synth.DT_FP8])
@pytest.mark.parametrize("pairing", [synth.NEOX, synth.INTERLEAVED])
def test_rotate_only_tma_ragged(page, dtype, pairing):
    """Segments that start and end inside pages (ragged first / last tiles move row by row), several requests, growth
    and shrink, replacement inserts in the same launch, a request of one token and an empty one."""
    w = synth.Workload("tma_ragged", 3, [3000, 1, 0, 2777], page, dtype=dtype, pairing=pairing, inv_freq=synth.yarn_inv_freq(),
                       directives=[(0, 5, 5, 40, 0, 0), (0, 100, 900, 3, 0, 0), (0, 1500, 1501, 333, 0, 0),
                                   (0, 2990, 3000, 0, 0, 0), (1, 0, 1, 0, 0, 0),
                                   (3, 0, 17, 500, 0, 0), (3, 1000, 1700, 0, 0, 0), (3, 2776, 2777, 2, 0, 0)],
                       seed=12, pool_factor=3.0, extra_pages=80).finalize()
    run_and_compare(w, O.ROTATE_ONLY, tuning=TMA)
    run_and_compare(w, O.ROTATE_ONLY, tuning=dict(TMA, stages=6, layer_group=2))


def test_rotate_only_tma_other_geometries():
    """Two heads of 64 behind an MLA latent (256-B band), the narrowest band (32 B, fp8), per-layer pairing, caller-
    prefilled replacement slots, more layers than one launch holds (64 tensor maps per launch), and pools whose pages
    are smaller than a box row count (falls back to the strided kernel)."""
    rng = np.random.default_rng(64)
    run_and_compare(heads_workload("tma_heads", 2, 64, 512, synth.DT_BF16, synth.NEOX, 1.0e4), O.ROTATE_ONLY, tuning=TMA)
    run_and_compare(heads_workload("tma_narrow", 1, 32, 16, synth.DT_FP8, synth.NEOX, 1.0e4), O.ROTATE_ONLY, tuning=TMA)
    w = tiny_workload(rng, P=16, n_req=3)
    w.n_layers = 5
    w.layer_pairing = [synth.NEOX, synth.INTERLEAVED, synth.INTERLEAVED, synth.NEOX, synth.INTERLEAVED]
    run_and_compare(w, O.ROTATE_ONLY, tuning=TMA)
    run_and_compare(tiny_workload(rng, P=16), O.ROTATE_ONLY, tuning=TMA, inserts_prefilled=True)
    w = tiny_workload(rng, P=16, n_req=2)
    w.n_layers = 130
    run_and_compare(w, O.ROTATE_ONLY, tuning=TMA)
    run_and_compare(tiny_workload(rng, P=4), O.ROTATE_ONLY, tuning=TMA)
    for _ in range(6):
        run_and_compare(fuzz_workload(rng), O.ROTATE_ONLY, tuning=TMA, prefetch=bool(rng.integers(0, 2)))


FLAT = {"rotate_kernel": 3}


def test_rotate_flat_is_chosen_for_short_segments_only():
    """Auto: the paper's own shape (185 chunks of ~130 tokens, token-level slots) runs on
    k_rotate_band_flat (plan.info.mover == 4), configs with long segments keep k_rotate_band; rotate_kernel = 1 / 3 force
    either.  Full size, every layer, whole pools, against the oracle, in each case."""
    from paper_2606_01065_b200 import binding as B
    mk = __import__("test_plan_host").make_plan
    appb = synth.config("appB", pool_factor=2.0)
    with mk(appb, B.ROTATE_ONLY) as plan:
        assert plan.info.mover == 4 and plan.info.rot_tile_rows == 384
    with mk(synth.config(2, pool_factor=1.25), B.ROTATE_ONLY) as plan:
        assert plan.info.mover == 1
    for tuning, mover in (({"rotate_kernel": 1}, 1), (FLAT, 4)):
        B.leyline_set_tuning(**tuning)
        try:
            with mk(appb, B.ROTATE_ONLY) as plan:
                assert plan.info.mover == mover
            with mk(synth.config(2, pool_factor=1.25), B.ROTATE_ONLY) as plan:
                assert plan.info.mover == mover
        finally:
            B.leyline_set_tuning()
    run_and_compare(appb, O.ROTATE_ONLY)                       # auto = flat
    run_and_compare(appb, O.ROTATE_ONLY, tuning={"rotate_kernel": 1})
    run_and_compare(synth.config(2, pool_factor=1.25), O.ROTATE_ONLY, tuning=FLAT)


@pytest.mark.parametrize("cfg", [3, 5])
def test_rotate_flat_full_size(cfg):
    """rotate_kernel = 3 on the long-segment configs (bf16: 384-row passes of 4 pair columns; fp8: 512-row passes of 2):
    passes that start and end inside tiles, every layer, whole pools."""
    run_and_compare(synth.config(cfg, pool_factor=1.25), O.ROTATE_ONLY, tuning=FLAT)


@pytest.mark.parametrize("page", [1, 16, 64])
@pytest.mark.parametrize("dtype", [synth.DT_BF16, synth.DT_FP8])
@pytest.mark.parametrize("pairing", [synth.NEOX, synth.INTERLEAVED])
def test_rotate_flat_ragged(page, dtype, pairing):
    """Passes that span several short segments with different rotations, a pass that ends behind the last rotated row,
    several requests, growth and shrink, replacement inserts in the same launch, a request of one token and an empty one."""
    w = synth.Workload("flat_ragged", 3, [3000, 1, 0, 2777, 150, 97, 260], page, dtype=dtype, pairing=pairing, inv_freq=synth.yarn_inv_freq(),
                       directives=[(0, 5, 5, 40, 0, 0), (0, 100, 900, 3, 0, 0), (0, 1500, 1501, 333, 0, 0),
                                   (0, 2990, 3000, 0, 0, 0), (1, 0, 1, 0, 0, 0),
                                   (3, 0, 17, 500, 0, 0), (3, 1000, 1700, 0, 0, 0), (3, 2776, 2777, 2, 0, 0),
                                   (4, 0, 30, 0, 0, 0), (5, 3, 3, 9, 0, 0), (6, 10, 20, 0, 0, 0), (6, 100, 101, 7, 0, 0)],
                       seed=13, pool_factor=3.0, extra_pages=80).finalize()
    run_and_compare(w, O.ROTATE_ONLY, tuning=FLAT)


def test_rotate_flat_other_geometries():
    """Two heads of 64 behind an MLA latent (8 pair columns), the narrowest band (32 B fp8: one pair column), per-layer
    pairing (two launches over the same passes), caller-prefilled replacement slots, more layers than one launch
    holds, and fuzzed workloads."""
    from paper_2606_01065_b200 import binding as B
    rng = np.random.default_rng(65)
    run_and_compare(heads_workload("flat_heads", 2, 64, 512, synth.DT_BF16, synth.NEOX, 1.0e4), O.ROTATE_ONLY, tuning=FLAT)
    run_and_compare(heads_workload("flat_narrow", 1, 32, 16, synth.DT_FP8, synth.NEOX, 1.0e4), O.ROTATE_ONLY, tuning=FLAT)
    w = tiny_workload(rng, P=16, n_req=3)
    w.n_layers = 5
    w.layer_pairing = [synth.NEOX, synth.INTERLEAVED, synth.INTERLEAVED, synth.NEOX, synth.INTERLEAVED]
    run_and_compare(w, O.ROTATE_ONLY, tuning=FLAT)
    run_and_compare(tiny_workload(rng, P=16), O.ROTATE_ONLY, tuning=FLAT, inserts_prefilled=True)
    w = tiny_workload(rng, P=1, n_req=2)
    w.n_layers = 130
    run_and_compare(w, O.ROTATE_ONLY, tuning=FLAT)
    for _ in range(8):
        run_and_compare(fuzz_workload(rng), O.ROTATE_ONLY, tuning=FLAT, prefetch=bool(rng.integers(0, 2)))


@pytest.mark.parametrize("seed", [101, 202])
def test_hazard_mover_random_batches_all_layers(seed):
    """More race coverage for k_move_bulk<HAZARD> at full concurrency (148 CTAs, every layer compared, whole pools):
    config-4-shaped batches with other directive draws -- 48 requests x 8 K tokens x 24 layers, 1-5 directives each,
    spans log-uniform 16-4096, replacements up to 512 rows (more growth than config 4), Delta of both signs."""
    rng = np.random.default_rng(seed)
    n_req, L = 48, 8192
    dirs = []
    for r in range(n_req):
        for (s0, e0, rl) in synth.random_directives(rng, L, int(rng.integers(1, 6)), 16, 4096, 512):
            dirs.append((r, s0, e0, rl, 0, synth.AMORTIZE))
    w = synth.Workload(f"hazard_batch_{seed}", 24, [L] * n_req, 64, inv_freq=synth.yarn_inv_freq(64, 10000.0, 40.0, 4096),
                       directives=dirs, seed=seed, pool_factor=1.3).finalize()
    assert any(d[3] > d[2] - d[1] for d in dirs) and any(d[3] < d[2] - d[1] for d in dirs)
    run_and_compare(w, O.INPLACE_MOVE)


# ----------------------------------------------------------------------------- the rotation arithmetic itself

def _band_by_position(w, cache, idx, n_tok):
    """K_pe band bytes of every layer in NEW logical order ([layer][token][band bytes])."""
    slots = idx[:n_tok].long()
    band0 = w.latent_dim * w.elem_bytes
    return torch.stack([p.view(-1, w.row_bytes)[slots, band0:] for p in cache.pools]).cpu().numpy()


@pytest.mark.parametrize("dtype", [synth.DT_BF16, synth.DT_FP8])
@pytest.mark.parametrize("pairing", [synth.NEOX, synth.INTERLEAVED])
def test_every_mode_and_mover_stores_the_same_bits(dtype, pairing):
    """One function of (a, b, cos, sin) in every kernel (device_common.cuh, rot_plain / rot_comp): FRESH, INPLACE_MOVE and
    ROTATE_ONLY, through the bulk mover, the row mover, the strided band kernel (tile items and flat passes) and the TMA
    band kernel, must leave
    bit-identical K_pe at every new position -- not merely results that each sit within tolerance of the oracle."""
    w = synth.Workload("same_bits", 3, [3000, 1, 2777], 16, dtype=dtype, pairing=pairing, inv_freq=synth.yarn_inv_freq(),
                       directives=[(0, 5, 5, 40, 0, 0), (0, 100, 900, 3, 0, 0), (0, 1500, 1501, 333, 0, 0),
                                   (2, 0, 17, 500, 0, 0), (2, 1000, 1700, 0, 0, 0), (2, 2776, 2777, 2, 0, 0)],
                       seed=19, pool_factor=3.0, extra_pages=80).finalize()
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    ref = None
    for mode, tuning in ((O.FRESH, {"kernel": 2}), (O.FRESH, {"kernel": 1}), (O.INPLACE_MOVE, {"kernel": 2}),
                         (O.INPLACE_MOVE, {"kernel": 1}), (O.ROTATE_ONLY, {"rotate_kernel": 1}), (O.ROTATE_ONLY, {"rotate_kernel": 2}),
                         (O.ROTATE_ONLY, {"rotate_kernel": 3})):
        B.leyline_set_tuning(**tuning)
        try:
            cache = harness.DeviceCache(w, "cuda:0")
            plan, pt, idx = harness.run_workload(cache, mode)
            torch.cuda.synchronize()
        finally:
            B.leyline_set_tuning()
        got = _band_by_position(w, cache, idx, int(plan.info.total_new_tokens))
        plan.close()
        if ref is None:
            ref = got
        else:
            np.testing.assert_array_equal(got, ref, err_msg=f"mode {MODE_NAME[mode]} tuning {tuning}")


@pytest.mark.parametrize("mode,tuning", [(O.FRESH, {"kernel": 2}), (O.FRESH, {"kernel": 1}), (O.INPLACE_MOVE, {"kernel": 2}),
                                         (O.ROTATE_ONLY, {"rotate_kernel": 1}), (O.ROTATE_ONLY, {"rotate_kernel": 2}),
                                         (O.ROTATE_ONLY, {"rotate_kernel": 3})])
@pytest.mark.parametrize("pairing", [synth.NEOX, synth.INTERLEAVED])
def test_cancelling_pairs_stay_within_one_code(mode, tuning, pairing):
    """Inputs built so that a cos - b sin (or b cos + a sin) nearly cancels in EVERY pair of every downstream row: for the
    segment's shift C the stored pair is (r sin phi, r cos phi) / (r cos phi, -r sin phi) rounded to bf16, phi = C theta_i,
    so one output is what the input rounding left over, 2^-9 rho and less.  Plain fp32 arithmetic (absolute error
    ~2^-24 rho) is several bf16 codes off on the deepest of these; the kernels' compensated form must stay within ONE
    code of the oracle on all of them -- the path that one element in 10^4 of ordinary data takes, taken here by most."""
    from paper_2606_01065_b200 import binding as B
    from paper_2606_01065_b200 import harness
    L, s0, e0, rl = 4096 + 37, 700, 1900, 333
    w = synth.Workload("cancel", 2, [L], 16, pairing=pairing, inv_freq=synth.yarn_inv_freq(),
                       directives=[(0, s0, e0, rl, 0, 0)], seed=23, pool_factor=3.0, extra_pages=40).finalize()
    C = rl - (e0 - s0)
    H = w.rope_dim // 2
    phi = float(C) * w.inv_freq.astype(np.float64)
    rng = np.random.default_rng(5)
    n_down = L - e0
    r = np.exp(rng.uniform(np.log(0.05), np.log(8.0), size=(w.n_layers, n_down, H)))
    flip = rng.integers(0, 2, size=(w.n_layers, n_down, H)).astype(bool)
    a = np.where(flip, r * np.cos(phi), r * np.sin(phi))      # flip: b' = b cos + a sin cancels; else a' = a cos - b sin
    b = np.where(flip, -r * np.sin(phi), r * np.cos(phi))
    band = np.concatenate([a, b], axis=-1) if pairing == synth.NEOX else np.stack([a, b], axis=-1).reshape(w.n_layers, n_down, 2 * H)
    B.leyline_set_tuning(**tuning)
    try:
        cache = harness.DeviceCache(w, "cuda:0")
        old_slots = torch.from_numpy(w.pages.astype(np.int64)[np.arange(e0, L) // 16] * 16 + np.arange(e0, L) % 16).to("cuda:0")
        for l in range(w.n_layers):
            rows = cache.pools[l].view(torch.bfloat16).view(-1, w.row_elems)
            rows[old_slots, w.latent_dim:] = torch.from_numpy(band[l]).to("cuda:0").to(torch.bfloat16)
        old = [p.cpu().numpy() for p in cache.pools]
        plan, pt, idx = harness.run_workload(cache, mode)
        torch.cuda.synchronize()
    finally:
        B.leyline_set_tuning()
    bm = oracle_plan(w, mode)
    assert_plan_equal(plan, bm, mode)
    deep = 0
    for l in range(w.n_layers):
        st = compare_layer(w, bm, mode, old[l], cache.pools[l].cpu().numpy(), cache.repl[l].cpu().numpy(), 1.0, layer=l)
        assert st["max_ord"] <= 1, st
        # how deep the cancellation goes on this input: the oracle's own output against the pair's norm
        want = O.splice_layer(w.dtype, pairing, w.latent_dim, w.rope_dim, w.row_bytes, w.inv_freq, 1.0, old[l],
                              cache.repl[l].cpu().numpy(), bm, n_heads=w.rope_heads).reshape(-1, w.row_bytes)
        new_s, _ = __import__("parity").rotated_rows(w, bm, mode)
        out = (want[new_s, w.latent_dim * 2:].copy().view(np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)
        x, y = (out[:, :H], out[:, H:]) if pairing == synth.NEOX else (out[:, 0::2], out[:, 1::2])
        rho = np.sqrt(x * x + y * y)
        deep += int((np.minimum(np.abs(x), np.abs(y)) < 2.0 ** -13 * rho).sum())
    plan.close()
    assert deep > 1000, f"the constructed input does not cancel deeply enough to exercise the compensated form ({deep})"

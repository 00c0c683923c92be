"""Table 8 of the paper on the GPU (App. H): "cross-architecture rotation-algebra validation".

For the five architectures of the table (MLA d=64 at theta 3.2e7 and 1e4; GQA d=128 at 5e5 and 1e6; d=96 at 1e4), K of
shape [batch 8, heads 32, d] in bf16, 24 (source position, Delta) cases x 5 seeds: rel-L2 between the delta-rotated
stored key R(Delta) R(p) k and fresh RoPE R(p + Delta) k.  The paper rotates in bf16 and prints worst / median rel-L2 per
row (tests/golden/paper_table8.txt); "no model weights required".  Here batch = 8 layers, the 24 cases
are 24 requests of ONE plan (each request's last token is the tracked key at position p; the directive in front of it
shifts it by Delta), executed by leyline_rotate_inplace / leyline_splice through the C ABI.  The library rotates in fp32
and rounds once, so every case must sit under the paper's worst value for its row, above the floor two bf16 roundings
(stored input, stored output) impose, and agree with the CPU oracle's statistics.
"""
import numpy as np
import pytest
import torch

import oracle as O
from helpers import from_storage, golden, rope_complex, to_storage
from paper_2606_01065_b200 import synth

pytestmark = pytest.mark.gpu

T8 = golden("paper_table8.txt")
ROWS = [("mla_dense", 64), ("mla_alt", 64), ("gqa_llama31", 128), ("gqa_qwen3", 128), ("gqa_phi3", 96)]
SOURCES = (10, 100, 1000, 4000, 8000, 8836)
DELTAS = (1, 76, -512, 2000)                            # signed, |Delta| from PAPER.md:133; 6 x 4 = 24 cases
HEADS, BATCH = 32, 8


def cases():
    out = []
    for p in SOURCES:
        for d in DELTAS:
            out.append((p, d if p + d >= 1 else -d))     # keep the target position inside the cache
    return out


def rel_l2(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.mark.parametrize("name,d", ROWS)
@pytest.mark.parametrize("mode", [O.ROTATE_ONLY, O.FRESH])
def test_table8_row(name, d, mode):
    from paper_2606_01065_b200 import binding as B
    theta, worst_paper, median_paper = float(T8[name + "_theta"]), float(T8[name + "_worst"]), float(T8[name + "_median"])
    inv = synth.rope_inv_freq(d, theta)
    cs = cases()
    n_req = len(cs)
    row_bytes = HEADS * d * 2
    # Request r: p filler tokens and then the tracked key at position p; the directive replaces the p fillers by
    # p + Delta tokens whose rows the caller would prefill (layer_repl = NULL), so the key moves to p + Delta.  Fillers
    # and replacement slots are never read or written, so they all alias one dummy slot: the pool stays tiny
    # (token-level slots: slot 0 = dummy, slot 1 + r = the key of request r, slot 1 + n_req + r = its fresh slot).
    DUMMY = 0
    seq_lens = [p + 1 for p, _ in cs]
    pt_offsets = np.concatenate([[0], np.cumsum(seq_lens)]).astype(np.int64)
    pages = np.concatenate([np.r_[np.full(p, DUMMY), 1 + r] for r, (p, _) in enumerate(cs)]).astype(np.int32)
    dirs = [(r, 0, p, p + dl, 0, synth.AMORTIZE) for r, (p, dl) in enumerate(cs)]
    free = np.concatenate([np.r_[np.full(p + dl, DUMMY), [1 + n_req + r] if mode == O.FRESH else []] for r, (p, dl) in enumerate(cs)]).astype(np.int32)
    n_slots = 2 + 2 * n_req
    desc, keep = B.make_desc(BATCH, 0, d, 1, B.BF16, B.NEOX, row_bytes, n_slots, inv, rope_heads=HEADS)
    bm = O.plan_batch(mode, 1, seq_lens, pt_offsets, pages, dirs, free)
    assert bm.status == O.OK
    new_slot = [int(rm.slot_new[-1]) for rm in bm.requests]
    assert new_slot == [(1 + n_req + r) if mode == O.FRESH else (1 + r) for r in range(n_req)]
    dummy_repl = np.zeros(max(p + dl for p, dl in cs) * row_bytes, np.uint8)   # the oracle always copies the rows (into the dummy slot)
    rels_gpu, rels_ora = [], []
    for seed in range(5):
        rng = np.random.default_rng(8000 + seed)
        raw = rng.standard_normal((BATCH, n_req, HEADS, d))
        olds, pools = [], []
        for l in range(BATCH):
            pool = np.zeros((n_slots, row_bytes), np.uint8)
            for r, (p, _) in enumerate(cs):
                k = rope_complex(raw[l, r], np.full(HEADS, p), inv).reshape(1, HEADS * d)        # R(p) k, stored as bf16
                pool[1 + r] = to_storage(k, O.BF16)[0]
            olds.append(pool.reshape(-1))
            pools.append(torch.from_numpy(olds[-1].copy()).to("cuda:0"))
        # the dummy slot is aliased on purpose (never read or written here): the caller vouches for its tables
        plan = B.leyline_plan_ex(desc, mode, seq_lens, pt_offsets, pages, dirs, free, B.Tuning(skip_alias_check=1))
        idx = torch.empty(int(plan.info.total_new_tokens), dtype=torch.int32, device="cuda:0")
        if mode == O.ROTATE_ONLY:
            B.leyline_rotate_inplace(plan, pools, None, idx)
        else:
            B.leyline_splice(plan, pools, pools, None, None, idx)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(plan.new_seq_lens, bm.new_seq_lens)
        np.testing.assert_array_equal(idx.cpu().numpy()[np.cumsum(bm.new_seq_lens) - 1], new_slot)
        for l in range(BATCH):
            got = from_storage(pools[l].cpu().numpy().reshape(-1, row_bytes)[new_slot], O.BF16)
            ora = from_storage(O.splice_layer(O.BF16, O.NEOX, 0, d, row_bytes, inv, 1.0, olds[l], dummy_repl, bm,
                                              n_heads=HEADS).reshape(-1, row_bytes)[new_slot], O.BF16)
            for r, (p, dl) in enumerate(cs):
                want = rope_complex(raw[l, r], np.full(HEADS, p + dl), inv).reshape(-1)
                rels_gpu.append(rel_l2(got[r], want))
                rels_ora.append(rel_l2(ora[r], want))
        plan.close()
    del keep
    rels_gpu, rels_ora = np.array(rels_gpu), np.array(rels_ora)
    print(f"[Table 8] {name} d={d} theta={theta:g} mode {mode}: GPU worst {rels_gpu.max():.2e} median {np.median(rels_gpu):.2e}; "
          f"oracle worst {rels_ora.max():.2e} median {np.median(rels_ora):.2e}; paper worst {worst_paper:.1e} median {median_paper:.1e}")
    assert rels_gpu.max() <= worst_paper and np.median(rels_gpu) <= median_paper
    assert rels_gpu.min() >= 1.0e-3                       # two bf16 roundings (stored input, stored output) cannot vanish
    assert abs(np.median(rels_gpu) - np.median(rels_ora)) <= 0.02 * np.median(rels_ora)
    assert abs(rels_gpu.max() - rels_ora.max()) <= 0.05 * rels_ora.max()

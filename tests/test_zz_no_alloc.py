"""leyline_cdc_chunk_noalloc: the chunker for hosts that may not allocate device memory (include/leyline_cdc.h).

Why the entry point exists.  ``leyline_cdc_chunk`` takes its working tables (about 15 B per token) from a
stream-ordered memory pool on every call.  An inference server that has handed the whole GPU to its own KV-cache
allocator at start-up cannot allow that: a later driver allocation can fail outright, and growing a pool stalls the
device for milliseconds in the middle of serving.  The same holds for a process kept to a fixed device-memory budget.
For those callers the library carries the tables as a fixed 8 MiB array in its own device image, and
``leyline_cdc_chunk_noalloc`` uses that array and nothing else; the price is a size limit (``CDC_NOALLOC_MAX_TOKENS``
tokens per call) and that calls which overlap on the GPU would trample each other's tables.

What is checked here.  The array is shared by every call and keeps what the last call left in it, so the test makes
calls IN A ROW on one stream -- a large batch, then at once a small one with other parameters (its tables lie inside the
large one's leftovers), then the large one again -- and compares each, bit for bit (integer work: the bar is equality),
with ``leyline_cdc_chunk`` on the same inputs.  It also checks that a batch beyond the limit is refused with a message
that names the limit, before anything is launched.

This file sorts last on purpose: ``pytest -x`` stops at the first failure, and a failure here must not hide the parity
tests.  It passes alone in a fresh process (the first call does the per-device address lookup) and after the rest.
"""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
ANCHORS = [7, 100, 101, 49999]


def _prompt(rng, n, vocab=50000, anchor_every=None):
    t = rng.integers(200, vocab, size=n).astype(np.int32)
    if anchor_every:
        at = np.arange(anchor_every, n, anchor_every)
        t[np.clip(at + rng.integers(-anchor_every // 4, anchor_every // 4, size=len(at)), 0, n - 1)] = rng.choice(ANCHORS, size=len(at))
    return t


class _Case:
    """Device inputs of one chunking problem, and one set of output buffers per call that will be made on it."""

    def __init__(self, torch, dev, tokens, seq_offsets, anchors, params, calls):
        self.n = len(tokens)
        self.params = params
        self.n_seqs = len(seq_offsets) - 1
        self.tokens = torch.from_numpy(np.ascontiguousarray(tokens, np.int32)).to(dev)
        self.offsets = torch.tensor(seq_offsets, dtype=torch.int64, device=dev)
        self.anchors = torch.tensor(sorted(anchors), dtype=torch.int32, device=dev) if anchors else None
        self.n_anchors = len(anchors)
        cap = max(self.n, 1)
        # sentinels everywhere: the tail behind the chunk count shows that a path wrote no further than it reported
        self.out = {c: (torch.full((cap,), -7, dtype=torch.int64, device=dev), torch.zeros(cap, dtype=torch.int64, device=dev),
                        torch.full((cap,), -7, dtype=torch.int32, device=dev), torch.full((1,), -7, dtype=torch.int64, device=dev))
                    for c in ("reference", *calls)}

    def run(self, fn, call):
        end, hsh, kind, cnt = self.out[call]
        fn(self.params, self.tokens, self.n, self.offsets, self.n_seqs, self.anchors, self.n_anchors, end, hsh, kind, self.n, cnt)

    def assert_same(self, call):
        (e0, h0, k0, c0), (e1, h1, k1, c1) = self.out["reference"], self.out[call]
        c = int(c0.item())
        assert c > 0 and int(c1.item()) == c, (call, c, int(c1.item()))
        np.testing.assert_array_equal(e1.cpu().numpy(), e0.cpu().numpy(), err_msg=call + ": chunk ends")
        np.testing.assert_array_equal(h1.cpu().numpy(), h0.cpu().numpy(), err_msg=call + ": content hashes")
        np.testing.assert_array_equal(k1.cpu().numpy(), k0.cpu().numpy(), err_msg=call + ": chunk kinds")
        return c


def test_header_limit_matches_the_binding_and_the_symbol_is_exported():
    from paper_2606_01065_b200 import binding as B
    text = open(os.path.join(ROOT, "include", "leyline_cdc.h")).read()
    (limit,) = re.findall(r"#define\s+LEYLINE_CDC_NOALLOC_MAX_TOKENS\s+(\d+)", text)
    assert int(limit) == B.CDC_NOALLOC_MAX_TOKENS
    assert callable(B.leyline_cdc_chunk_noalloc)


@pytest.mark.gpu
def test_noalloc_chunker_equals_the_allocating_one_on_calls_in_a_row():
    import torch
    from paper_2606_01065_b200 import binding as B
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(2606)
    # the paper's microbenchmark shape (16 sessions x ~17K-token prompts) plus a long and two empty
    # sequences: ~300K tokens, several compaction blocks, a ragged tail -- and close to the limit of the static array
    lens = [int(rng.integers(16000, 18000)) for _ in range(16)] + [0, 30000, 0, 1]
    big = _Case(torch, dev, _prompt(rng, sum(lens), anchor_every=600), [0, *np.cumsum(lens).tolist()], ANCHORS,
                B.CdcParams(0x1234ABCD, 64, 1024, 7, 0), calls=("big", "big again"))
    assert big.n <= B.CDC_NOALLOC_MAX_TOKENS
    # a small problem with other parameters and no anchors: all of its tables fall inside what the big call left behind
    small = _Case(torch, dev, _prompt(rng, 5003, vocab=230), [0, 17, 17, 4000, 5003], [], B.CdcParams(99, 1, 16, 2, 0),
                  calls=("small", "small again"))
    # exactly at the limit, one sequence, minimum chunk size 1 (the most doubling rounds the layout can ask for)
    full = _Case(torch, dev, _prompt(rng, B.CDC_NOALLOC_MAX_TOKENS, anchor_every=5000), [0, B.CDC_NOALLOC_MAX_TOKENS],
                 ANCHORS, B.CdcParams(5, 1, 4096, 11, 0), calls=("full",))

    for case in (big, small, full):                       # the existing, allocating path: what this test compares with
        case.run(B.leyline_cdc_chunk, "reference")
    torch.cuda.synchronize()

    free_before = torch.cuda.mem_get_info()[0]
    # five calls in a row on one stream with no synchronisation in between: each finds the previous one's leftovers
    order = [("big", big), ("small", small), ("big again", big), ("full", full), ("small again", small)]
    for call, case in order:
        case.run(B.leyline_cdc_chunk_noalloc, call)
    torch.cuda.synchronize()
    # the calls took no device memory (every torch buffer was made before; 2 MiB of slack for driver bookkeeping)
    assert free_before - torch.cuda.mem_get_info()[0] <= 2 << 20
    counts = {call: case.assert_same(call) for call, case in order}
    assert counts["big again"] == counts["big"] and counts["small again"] == counts["small"]

    # beyond the limit: refused before anything is launched, outputs untouched, and the message names the limit
    over = B.CDC_NOALLOC_MAX_TOKENS + 1
    t = torch.zeros(over, dtype=torch.int32, device=dev)
    off = torch.tensor([0, over], dtype=torch.int64, device=dev)
    cnt = torch.full((1,), -7, dtype=torch.int64, device=dev)
    end = torch.full((8,), -7, dtype=torch.int64, device=dev)
    with pytest.raises(B.LeylineError) as err:
        B.leyline_cdc_chunk_noalloc(B.CdcParams(1, 64, 1024, 7, 0), t, over, off, 1, None, 0, end, None, None, 8, cnt)
    assert err.value.status == B.E_UNSUPPORTED and str(B.CDC_NOALLOC_MAX_TOKENS) in str(err.value)
    torch.cuda.synchronize()
    assert int(cnt.item()) == -7 and (end.cpu().numpy() == -7).all()
    # an empty batch needs no scratch at all
    B.leyline_cdc_chunk_noalloc(B.CdcParams(1, 64, 1024, 7, 0), None, 0, torch.zeros(1, dtype=torch.int64, device=dev), 0,
                                None, 0, end, None, None, 8, cnt)
    torch.cuda.synchronize()
    assert int(cnt.item()) == 0

"""Discovery side: anchored content-defined chunking, chunk content
hash, registry.  CPU tests pin the oracle (oracle/cdc_oracle.c) to published generator vectors, to the Gear-hash
window identity, to a list-based re-implementation of the boundary rule and to the property the paper relies on
(content behind an anchor chunks identically wherever it sits, so a registry hit returns the edit's Delta).
GPU tests compare the CUDA chunker / registry with the oracle bit for bit.
"""
import numpy as np
import pytest

from helpers import golden
from oracle import cdc as OC

V = golden("published_hash_vectors.txt")
M64 = (1 << 64) - 1
SEED, MIN, MAX, BITS = 0x5EED, 16, 256, 6
ANCHORS = [100000, 100001, 100002]            # stand-ins for chat-template special tokens (PAPER.md:389 (iii))


def random_prompt(rng, n, vocab=50000, anchor_every=None):
    t = rng.integers(0, vocab, size=n).astype(np.int32)
    if anchor_every:
        pos = np.cumsum(rng.integers(anchor_every // 2, anchor_every * 2, size=2 * n // anchor_every + 1))
        pos = pos[pos < n]
        t[pos] = rng.choice(ANCHORS, size=len(pos))
    return t


# ----------------------------------------------------------------------------- generators: published vectors

def test_d1_gear_is_splitmix64():
    assert OC.gear(0, 0) == V["splitmix64_seed0_out1"]
    assert OC.gear(0, 1) == V["splitmix64_seed0_out2"]
    assert OC.gear(0, 2) == V["splitmix64_seed0_out3"]
    # the seed is the generator's starting state: seed = one increment shifts the stream by one
    assert OC.gear(0x9E3779B97F4A7C15, 0) == V["splitmix64_seed0_out2"]


def test_d4_content_hash_is_fnv1a64_over_le_bytes():
    p = V["fnv1a64_prime"]
    # "a" then three zero bytes: x ^= 0 leaves x, so the hash is FNV("a") * prime^3
    assert OC.content_hash([0x61], 0, 1) == (V["fnv1a64_a"] * p ** 3) & M64
    # "foob" + "ar\0\0" as two little-endian words
    w0 = int.from_bytes(b"foob", "little")
    w1 = int.from_bytes(b"ar\0\0", "little")
    assert OC.content_hash([w0, w1], 0, 2) == (V["fnv1a64_foobar"] * p ** 2) & M64
    # empty range: the offset basis; sub-ranges hash their own tokens only
    assert OC.content_hash([5, 6, 7], 1, 1) == V["fnv1a64_offset_basis"]
    assert OC.content_hash([9, w0, w1, 9], 1, 3) == OC.content_hash([w0, w1], 0, 2)


# ----------------------------------------------------------------------------- D2: the Gear window

def test_d2_signature_is_a_64_token_window_sum():
    """h_i = (h_{i-1} << 1) + G(t_i) mod 2^64  ==  sum_{j < 64} G(t_{i-j}) << j, cut at the last anchor / sequence start
    (bit k of h_i depends on the last k+1 tokens only: the Gear hash's defining property, Xia et al.)."""
    rng = np.random.default_rng(0)
    t = random_prompt(rng, 700, anchor_every=90)
    so = [0, 300, 300, 700]                      # an empty sequence in the middle
    sig = OC.signature(SEED, t, so, ANCHORS)
    for i in range(len(t)):
        seq_start = 0 if i < 300 else 300
        acc, j = 0, 0
        while j < 64 and i - j >= seq_start and not (j > 0 and int(t[i - j]) in ANCHORS):
            acc += OC.gear(SEED, int(t[i - j])) << j
            j += 1
        assert int(sig[i]) == acc & M64, i


# ----------------------------------------------------------------------------- D3: the boundary rule, brute force

def chunk_by_lists(tokens, seq_offsets, anchors, seed, mn, mx, bits):
    """Independent restatement of D3 with Python lists and the window-sum form of the signature."""
    out = []
    for s in range(len(seq_offsets) - 1):
        seq = [int(x) for x in tokens[seq_offsets[s]:seq_offsets[s + 1]]]
        cur, run = [], []                        # cur: tokens of the open chunk; run: tokens since the last anchor
        for k, tok in enumerate(seq):
            cur.append(tok)
            run.append(tok)
            h = sum(OC.gear(seed, x) << j for j, x in enumerate(reversed(run[-64:]))) & M64
            if tok in anchors:
                kind = OC.KIND_ANCHOR
            elif k == len(seq) - 1:
                kind = OC.KIND_SEQ_END
            elif len(cur) == mx:
                kind = OC.KIND_MAX
            elif len(cur) >= mn and (bits == 0 or h >> (64 - bits) == 0):
                kind = OC.KIND_HASH
            else:
                continue
            if kind == OC.KIND_ANCHOR:
                run = []
            out.append((seq_offsets[s] + k + 1, tuple(cur), kind))
            cur = []
    return out


@pytest.mark.parametrize("seed", range(6))
def test_d3_boundaries_match_list_restatement(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(1, 1500))
    t = random_prompt(rng, n, vocab=int(rng.choice([3, 50, 50000])), anchor_every=int(rng.choice([0, 40, 200])) or None)
    cuts = np.sort(rng.integers(0, n + 1, size=int(rng.integers(0, 4))))
    so = [0, *[int(c) for c in cuts], n]
    mn, mx, bits = int(rng.choice([1, 4, 16])), int(rng.choice([16, 64, 256])), int(rng.choice([0, 2, 4, 6]))
    end, hsh, kind = OC.chunk(SEED + seed, mn, mx, bits, t, so, ANCHORS)
    want = chunk_by_lists(t, so, ANCHORS, SEED + seed, mn, mx, bits)
    assert [int(e) for e in end] == [w[0] for w in want]
    assert [int(k) for k in kind] == [w[2] for w in want]
    for h, w in zip(hsh, want):
        assert int(h) == OC.content_hash(list(w[1]), 0, len(w[1]))


def test_d3_invariants_and_chunk_length_law():
    rng = np.random.default_rng(11)
    n = 400000
    t = random_prompt(rng, n)
    end, hsh, kind = OC.chunk(SEED, MIN, MAX, BITS, t, None, ANCHORS)
    start = np.concatenate([[0], end[:-1]])
    ln = end - start
    assert end[-1] == n and (ln >= 1).all() and (ln <= MAX).all()               # chunks tile the sequence
    assert (ln[kind == OC.KIND_HASH] >= MIN).all() and (ln[kind == OC.KIND_MAX] == MAX).all()
    assert (kind[:-1] != OC.KIND_SEQ_END).all() and kind[-1] == OC.KIND_SEQ_END
    # random tokens: past min_size every position is a boundary with probability 2^-bits, truncated at max_size:
    # E[len] = (MIN - 1) + sum_{k=1..MAX-MIN+1} P(len >= MIN-1+k), a geometric law
    q = 1.0 - 2.0 ** -BITS
    expect = (MIN - 1) + sum(q ** (k - 1) for k in range(1, MAX - MIN + 2))
    assert abs(ln[:-1].mean() - expect) / expect < 0.03, (ln.mean(), expect)
    assert abs((kind == OC.KIND_MAX).mean() - q ** (MAX - MIN + 1)) < 0.01


# ----------------------------------------------------------------------------- the property the paper relies on

def build_and_replay(rng, edit_at_turn=2, n_turns=8, turn_len=700, stub_len=11):
    """BUILD prompt = turns separated by anchor tokens; REPLAY prompt = the same with one turn's body replaced by a
    short stub (a summarisation edit).  Returns (build, replay, edit_start, edit_end, stub_len)."""
    turns = [rng.integers(0, 50000, size=turn_len + int(rng.integers(0, 50))).astype(np.int32) for _ in range(n_turns)]
    sep = np.array([ANCHORS[0]], np.int32)
    build = np.concatenate([np.concatenate([tr, sep]) for tr in turns])
    s = sum(len(tr) + 1 for tr in turns[:edit_at_turn])
    e = s + len(turns[edit_at_turn])
    stub = rng.integers(0, 50000, size=stub_len).astype(np.int32)
    replay = np.concatenate([build[:s], stub, build[e:]])
    return build, replay, s, e, stub_len


def test_anchored_chunks_behind_an_edit_are_found_with_the_edits_delta():
    """PAPER.md:389 (iii), :397: with the anchored chunker every chunk that lies wholly behind the edited turn is
    re-discovered in the edited prompt, at its old position + Delta, Delta = |R| - |span|."""
    rng = np.random.default_rng(5)
    build, replay, s, e, r = build_and_replay(rng)
    delta = r - (e - s)
    b_end, b_hash, _ = OC.chunk(SEED, MIN, MAX, BITS, build, None, ANCHORS)
    r_end, r_hash, _ = OC.chunk(SEED, MIN, MAX, BITS, replay, None, ANCHORS)
    b_start = np.concatenate([[0], b_end[:-1]])
    r_start = np.concatenate([[0], r_end[:-1]])
    reg = OC.Registry()
    reg.insert(b_hash, b_start)
    src = reg.lookup(r_hash)
    behind = r_start >= s + r + 1                     # chunks after the edited turn's closing anchor
    assert behind.sum() > 20
    assert (src[behind] >= 0).all()                   # every one of them is found ...
    assert ((r_start[behind] - src[behind]) == delta).all()   # ... at exactly the directive's Delta
    before = r_end <= s
    assert ((r_start[before] - src[before]) == 0).all()       # the untouched prefix maps to itself


def test_registry_keeps_the_smallest_value_under_duplicate_keys():
    """DESIGN.md reading D5: a key inserted several times maps to the SMALLEST value ever inserted under it, whatever the
    insertion order and however the inserts are batched; unknown keys read -1.  Checked against a sort-based
    restatement (sort by (key, value), keep the first of each key) that shares nothing with the dict loop."""
    rng = np.random.default_rng(55)
    keys = rng.integers(1, 40, size=500).astype(np.uint64) * np.uint64(0x9E3779B97F4A7C15)     # 39 distinct keys, many repeats
    vals = rng.integers(0, 10**9, size=500).astype(np.int64)
    order = np.lexsort((vals, keys))
    first = np.concatenate([[True], keys[order][1:] != keys[order][:-1]])
    want = dict(zip(keys[order][first].tolist(), vals[order][first].tolist()))
    for perm in (np.arange(500), np.arange(500)[::-1], rng.permutation(500)):
        reg = OC.Registry()
        for lo in range(0, 500, 37):                                       # several batches
            sel = perm[lo:lo + 37]
            reg.insert(keys[sel], vals[sel])
        got = reg.lookup(np.array(list(want.keys()), np.uint64))
        np.testing.assert_array_equal(got, np.array(list(want.values()), np.int64))
        assert (reg.lookup(np.array([7, 11], np.uint64)) == -1).all()
    # hand case: descending then ascending values under one key
    reg = OC.Registry()
    reg.insert([5, 5, 5], [30, 10, 20])
    reg.insert([5], [15])
    assert reg.lookup([5]).tolist() == [10]


def test_unanchored_chunker_resynchronises_only_after_a_window():
    """Without anchors (the paper's 'legacy purely-Gear-hash chunker') boundaries behind an edit depend
    on where the previous boundary fell (min / max sizes), so the first chunks behind the edit may differ; content
    64 tokens past a COMMON boundary chunks identically again."""
    rng = np.random.default_rng(6)
    build, replay, s, e, r = build_and_replay(rng)
    delta = r - (e - s)
    b_end, b_hash, _ = OC.chunk(SEED, MIN, MAX, BITS, build, None, [])
    r_end, r_hash, _ = OC.chunk(SEED, MIN, MAX, BITS, replay, None, [])
    common = np.intersect1d(b_end[b_end > e] + delta, r_end[r_end > s + r])
    common = common[common >= s + r + 64]              # the window no longer sees the edit: signatures agree from here
    assert len(common) > 0                             # the two chunkings do meet again ...
    first = common[0]
    assert set(r_end[r_end >= first]) == set(b_end[b_end >= first - delta] + delta)   # ... and stay together


# ----------------------------------------------------------------------------- GPU parity (bit-exact: integer work)

def gpu_chunk(tokens, seq_offsets, anchors, seed, mn, mx, bits, capacity=None):
    import torch
    from paper_2606_01065_b200 import binding as B
    dev = torch.device("cuda:0")
    n = len(tokens)
    so = [0, n] if seq_offsets is None else seq_offsets
    t = torch.from_numpy(np.ascontiguousarray(tokens, np.int32)).to(dev)
    off = torch.tensor(so, dtype=torch.int64, device=dev)
    an = torch.tensor(sorted(anchors), dtype=torch.int32, device=dev) if anchors else None
    cap = n if capacity is None else capacity
    end = torch.full((max(cap, 1),), -7, dtype=torch.int64, device=dev)
    hsh = torch.zeros(max(cap, 1), dtype=torch.int64, device=dev)        # uint64 bit patterns
    kind = torch.full((max(cap, 1),), -7, dtype=torch.int32, device=dev)
    cnt = torch.full((1,), -7, dtype=torch.int64, device=dev)
    B.leyline_cdc_chunk(B.CdcParams(seed, mn, mx, bits, 0), t, n, off, len(so) - 1, an, len(anchors) if anchors else 0,
                        end, hsh, kind, cap, cnt)
    torch.cuda.synchronize()
    c = int(cnt.item())
    m = min(c, cap)
    return c, end.cpu().numpy()[:m], hsh.cpu().numpy().view(np.uint64)[:m], kind.cpu().numpy()[:m], (end, kind)


@pytest.mark.gpu
@pytest.mark.parametrize("seed", range(8))
def test_gpu_chunker_matches_oracle_small(seed):
    rng = np.random.default_rng(100 + seed)
    n = int(rng.integers(1, 6000))
    t = random_prompt(rng, n, vocab=int(rng.choice([3, 50, 50000])), anchor_every=int(rng.choice([0, 40, 200])) or None)
    cuts = np.sort(rng.integers(0, n + 1, size=int(rng.integers(0, 5))))
    so = [0, *[int(c) for c in cuts], n]
    mn, mx, bits = int(rng.choice([1, 4, 16])), int(rng.choice([16, 64, 256])), int(rng.choice([0, 2, 4, 6]))
    c, end, hsh, kind, _ = gpu_chunk(t, so, ANCHORS, SEED + seed, mn, mx, bits)
    o_end, o_hash, o_kind = OC.chunk(SEED + seed, mn, mx, bits, t, so, ANCHORS)
    assert c == len(o_end)
    np.testing.assert_array_equal(end, o_end)
    np.testing.assert_array_equal(kind, o_kind)
    np.testing.assert_array_equal(hsh, o_hash)


@pytest.mark.gpu
@pytest.mark.parametrize("anchored", [True, False])
def test_gpu_chunker_matches_oracle_long_batch(anchored):
    """16 sessions x ~17K-token prompts (the paper's microbenchmark shape) in one call, plus a
    128K-token sequence; several compaction blocks, a ragged tail, empty sequences."""
    rng = np.random.default_rng(17)
    lens = [int(rng.integers(16000, 18000)) for _ in range(16)] + [0, 131072, 0, 1]
    t = random_prompt(rng, sum(lens), anchor_every=600 if anchored else None)
    so = [0, *np.cumsum(lens).tolist()]
    anchors = ANCHORS if anchored else []
    c, end, hsh, kind, _ = gpu_chunk(t, so, anchors, SEED, MIN, MAX, BITS)
    o_end, o_hash, o_kind = OC.chunk(SEED, MIN, MAX, BITS, t, so, anchors)
    assert c == len(o_end)
    np.testing.assert_array_equal(end, o_end)
    np.testing.assert_array_equal(kind, o_kind)
    np.testing.assert_array_equal(hsh, o_hash)


@pytest.mark.gpu
def test_gpu_chunker_edge_cases():
    import torch
    from paper_2606_01065_b200 import binding as B
    # empty input: zero chunks, nothing written
    c, end, hsh, kind, _ = gpu_chunk(np.zeros(0, np.int32), [0, 0], ANCHORS, SEED, MIN, MAX, BITS)
    assert c == 0
    # every token an anchor: one chunk per token
    t = np.full(300, ANCHORS[1], np.int32)
    c, end, hsh, kind, _ = gpu_chunk(t, None, ANCHORS, SEED, MIN, MAX, BITS)
    assert c == 300 and (end == np.arange(1, 301)).all() and (kind[:-1] == B.CDC_ANCHOR).all()
    # one repeated token, mask never satisfied or always satisfied: max-size / min-size chunks
    t = np.full(1000, 7, np.int32)
    c, end, hsh, kind, _ = gpu_chunk(t, None, [], SEED, 4, 64, 0)
    o_end, o_hash, o_kind = OC.chunk(SEED, 4, 64, 0, t, None, [])
    np.testing.assert_array_equal(end, o_end)
    assert (np.diff(np.concatenate([[0], end]))[:-1] == 4).all()
    # capacity smaller than the number of chunks: the count is still reported, only `capacity` entries are written
    rng = np.random.default_rng(3)
    t = random_prompt(rng, 20000)
    full_c, full_end, full_hash, full_kind, _ = gpu_chunk(t, None, [], SEED, MIN, MAX, BITS)
    c, end, hsh, kind, (end_t, kind_t) = gpu_chunk(t, None, [], SEED, MIN, MAX, BITS, capacity=10)
    assert c == full_c and len(end) == 10
    np.testing.assert_array_equal(end, full_end[:10])
    np.testing.assert_array_equal(hsh, full_hash[:10])
    # bad arguments are refused before any launch
    with pytest.raises(B.LeylineError):
        gpu_chunk(t, None, [], SEED, 0, MAX, BITS)
    with pytest.raises(B.LeylineError):
        gpu_chunk(t, None, [], SEED, 32, 16, BITS)


@pytest.mark.gpu
def test_gpu_registry_and_discovery_returns_the_edits_delta():
    """BUILD registers its chunks, REPLAY looks its own up: every chunk behind the edited turn is found at
    old position + Delta -- on the device, against the oracle's registry (D5: smallest value wins)."""
    import torch
    from paper_2606_01065_b200 import binding as B
    rng = np.random.default_rng(5)
    build, replay, s, e, r = build_and_replay(rng)
    delta = r - (e - s)
    dev = torch.device("cuda:0")
    cap = 1 << 12
    keys = torch.empty(cap, dtype=torch.int64, device=dev)
    vals = torch.empty(cap, dtype=torch.int64, device=dev)
    B.leyline_registry_clear(keys, vals, cap)
    bc, b_end, b_hash, _, _ = gpu_chunk(build, None, ANCHORS, SEED, MIN, MAX, BITS)
    rc, r_end, r_hash, _, _ = gpu_chunk(replay, None, ANCHORS, SEED, MIN, MAX, BITS)
    b_start = np.concatenate([[0], b_end[:-1]])
    r_start = np.concatenate([[0], r_end[:-1]])
    # duplicates on purpose: the build prompt registered twice, the second time with larger values
    ins_h = np.concatenate([b_hash, b_hash]).view(np.int64)
    ins_v = np.concatenate([b_start + 100000, b_start]).astype(np.int64)
    dropped = torch.full((1,), -1, dtype=torch.int64, device=dev)
    B.leyline_registry_insert(keys, vals, cap, torch.from_numpy(ins_h).to(dev), torch.from_numpy(ins_v).to(dev), len(ins_h),
                              dropped)
    out = torch.empty(rc, dtype=torch.int64, device=dev)
    B.leyline_registry_lookup(keys, vals, cap, torch.from_numpy(r_hash.view(np.int64).copy()).to(dev), rc, out)
    torch.cuda.synchronize()
    assert int(dropped.item()) == 0
    reg = OC.Registry()
    reg.insert(np.concatenate([b_hash, b_hash]), ins_v)
    src = out.cpu().numpy()
    np.testing.assert_array_equal(src, reg.lookup(r_hash))
    behind = r_start >= s + r + 1
    assert behind.sum() > 20 and (src[behind] >= 0).all()
    assert ((r_start[behind] - src[behind]) == delta).all()
    # a table that is too small reports what it could not store
    tiny_k = torch.empty(8, dtype=torch.int64, device=dev)
    tiny_v = torch.empty(8, dtype=torch.int64, device=dev)
    B.leyline_registry_clear(tiny_k, tiny_v, 8)
    B.leyline_registry_insert(tiny_k, tiny_v, 8, torch.from_numpy(b_hash.view(np.int64).copy()).to(dev),
                              torch.from_numpy(b_start.astype(np.int64)).to(dev), bc, dropped)
    torch.cuda.synchronize()
    assert int(dropped.item()) == len(set(b_hash.tolist())) - 8


@pytest.mark.gpu
@pytest.mark.parametrize("mn,mx,bits", [(1, 1, 0), (1, 1, 6), (7, 7, 3), (4096, 4096, 0), (1, 4096, 32), (64, 4096, 12), (1, 2, 1)])
def test_gpu_chunker_parameter_extremes(mn, mx, bits):
    """Every token its own chunk, fixed-size chunks, the largest chunk size, a mask that never / always fires; thousands
    of tiny sequences next to long ones (more sequences than one grid pass of k_cdc_seq_ends)."""
    rng = np.random.default_rng(mn * 31 + mx * 7 + bits)
    lens = [int(x) for x in rng.integers(0, 4, size=70000)] + [50000, 0, 9000] + [int(x) for x in rng.integers(0, 3, size=5000)]
    t = random_prompt(rng, sum(lens), vocab=1000, anchor_every=500)
    so = [0, *np.cumsum(lens).tolist()]
    c, end, hsh, kind, _ = gpu_chunk(t, so, ANCHORS, SEED, mn, mx, bits)
    o_end, o_hash, o_kind = OC.chunk(SEED, mn, mx, bits, t, so, ANCHORS)
    assert c == len(o_end)
    np.testing.assert_array_equal(end, o_end)
    np.testing.assert_array_equal(kind, o_kind)
    np.testing.assert_array_equal(hsh, o_hash)


@pytest.mark.gpu
@pytest.mark.parametrize("mn,mx,bits", [(64, 4096, 12), (2048, 4096, 16), (1, 3000, 9), (16, 256, 6)])
def test_gpu_chunker_long_unanchored_sequences(mn, mx, bits):
    """No anchors at all, four sequences of ~200 K tokens: hard stops are ~200 K positions apart and candidates up to
    65 K, so "next set bit" walks the second bitmap level over many words, chains are thousands of chunks long (the
    doubling needs most of its rounds) and max_size cuts dominate where the mask rarely fires."""
    rng = np.random.default_rng(mn + mx + bits)
    lens = [200003, 199999, 1, 180000]
    t = rng.integers(0, 32000, size=sum(lens)).astype(np.int32)
    so = [0, *np.cumsum(lens).tolist()]
    c, end, hsh, kind, _ = gpu_chunk(t, so, [], SEED, mn, mx, bits)
    o_end, o_hash, o_kind = OC.chunk(SEED, mn, mx, bits, t, so, [])
    assert c == len(o_end)
    np.testing.assert_array_equal(end, o_end)
    np.testing.assert_array_equal(kind, o_kind)
    np.testing.assert_array_equal(hsh, o_hash)


@pytest.mark.gpu
@pytest.mark.parametrize("offsets", [[5, 3, 900, 20], [-7, 10**12, 4], [0, 0, 0, 0], [123, 123], [2000, 0]])
def test_gpu_chunker_survives_garbage_device_offsets(offsets):
    """The sequence offsets live on the device, so the host cannot validate them (leyline_cdc.h asks for ascending
    offsets from 0 to n_tokens).  Whatever they hold, the call must stay inside its buffers: nothing at or past
    `capacity` is written (canaries on both sides of every output), the count stays within [0, n_tokens], reported ends
    are non-decreasing positions in (0, n_tokens], and a well-formed call right behind it is unaffected."""
    import torch
    from paper_2606_01065_b200 import binding as B
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(len(offsets))
    n, cap, pad = 2000, 300, 64
    t = random_prompt(rng, n, anchor_every=40)
    td = torch.from_numpy(t).to(dev)
    off = torch.tensor(offsets, dtype=torch.int64, device=dev)
    an = torch.tensor(sorted(ANCHORS), dtype=torch.int32, device=dev)
    end = torch.full((cap + 2 * pad,), -7, dtype=torch.int64, device=dev)
    hsh = torch.full((cap + 2 * pad,), -7, dtype=torch.int64, device=dev)
    kind = torch.full((cap + 2 * pad,), -7, dtype=torch.int32, device=dev)
    cnt = torch.full((3,), -7, dtype=torch.int64, device=dev)
    B.leyline_cdc_chunk(B.CdcParams(SEED, MIN, MAX, BITS, 0), td, n, off, len(offsets) - 1, an, len(ANCHORS),
                        end[pad:], hsh[pad:], kind[pad:], cap, cnt[1:])
    torch.cuda.synchronize()
    for buf in (end, hsh, kind):
        assert bool((buf[:pad] == -7).all()) and bool((buf[pad + cap:] == -7).all())
    assert int(cnt[0]) == -7 and int(cnt[2]) == -7
    c = int(cnt[1])
    assert 0 <= c <= n
    e = end[pad:pad + min(c, cap)].cpu().numpy()
    assert ((e > 0) & (e <= n)).all() and (np.diff(e) >= 0).all()
    # the library is still in working order
    c2, end2, hsh2, kind2, _ = gpu_chunk(t, None, ANCHORS, SEED, MIN, MAX, BITS)
    o_end, o_hash, o_kind = OC.chunk(SEED, MIN, MAX, BITS, t, None, ANCHORS)
    assert c2 == len(o_end)
    np.testing.assert_array_equal(end2, o_end)
    np.testing.assert_array_equal(hsh2, o_hash)

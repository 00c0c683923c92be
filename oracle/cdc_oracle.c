/*
 * oracle/cdc_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain sequential CPU definition of the DISCOVERY side that precedes the Leyline splice (SURVEY.md section 8(f)
 * NEXT-4; arxiv/paper_2606_01065, "PAPER.md:N" = line N of /root/reference/PAPER.md): the anchored content-defined
 * chunker and the chunk content hash that find shifted-identical chunks, whose position difference is the Delta
 * the splice then rotates by.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_2606_01065_b200/csrc; only tests/ may load it.
 *
 * What the paper fixes:
 *   - a "CDC chunker's Gear-hash rolling signature" over the prompt's tokens finds chunk boundaries (PAPER.md:389 (i));
 *   - ABSPOS_CDC: chunking starts at absolute position 0 of the prompt, not at the radix-match boundary, so hashes are
 *     stable across requests with different matched prefixes (PAPER.md:389 (ii));
 *   - A1 anchored CDC "forces a CDC boundary AND resets the rolling hash at chat-template special tokens"
 *     (PAPER.md:389 (iii));
 *   - chunks are registered under a content hash; a later prompt's chunk with the same hash at another position is a
 *     shifted-identical chunk.
 * What the paper does NOT give -- the Gear table, the boundary mask, min / max chunk sizes, the content hash -- is
 * fixed by DESIGN.md readings D1-D5 ("parity unpinned by the paper" for those constants):
 *   D1 gear value of a token   G(v) = splitmix64 output for state seed + (v+1)*0x9E3779B97F4A7C15 (Steele et al.)
 *   D2 rolling signature       h_i = (h_{i-1} << 1) + G(t_i)  mod 2^64 (Gear hash, Xia et al.), h = 0 at the start of a
 *                              sequence and after every anchor token; NOT reset at hash-defined boundaries, so a
 *                              boundary depends on the last 64 tokens only (bit k of h_i depends on t_{i-k..i})
 *   D3 boundary rule           position i ends a chunk (inclusive) iff  t_i is an anchor, or i is the last token of its
 *                              sequence, or len == max_size, or (len >= min_size and the top mask_bits of h_i are 0),
 *                              len = i - chunk_start + 1
 *   D4 content hash            64-bit FNV-1a (offset 0xcbf29ce484222325, prime 0x100000001b3) over the chunk's token
 *                              ids as little-endian 4-byte words; 0 is remapped to 1 (0 = empty registry key)
 *   D5 registry                key -> smallest value inserted under that key (deterministic under duplicates)
 *
 * Pins (tests/test_cdc.py, -m "not gpu"): published splitmix64 and FNV-1a test vectors, the 64-token window identity
 * against a brute-force sum in Python integers, a list-based re-implementation of D3 on tiny inputs, tiling /
 * min / max invariants, the geometric chunk-length law, and the property the paper relies on: content behind an
 * anchor chunks identically wherever it sits, so discovery returns exactly the Delta of the edit.
 */
#include <stdint.h>

/* D1.  splitmix64 (Steele, Lea, Flood 2014): the state advances by the golden-ratio increment, the output is the
 * mixed state.  Token v uses the (v+1)-th state after `seed`. */
uint64_t cdc_ora_gear(uint64_t seed, int32_t token) {
    uint64_t z = seed + ((uint64_t)(uint32_t)token + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static int is_anchor(int32_t t, const int32_t* anchors, int32_t n_anchors) {
    for (int32_t a = 0; a < n_anchors; ++a) /* plain linear search: the oracle is not tuned */
        if (anchors[a] == t) return 1;
    return 0;
}

/* D4.  FNV-1a over the little-endian bytes of tokens[b..e). */
uint64_t cdc_ora_content_hash(const int32_t* tokens, int64_t b, int64_t e) {
    uint64_t x = 0xcbf29ce484222325ull;
    for (int64_t i = b; i < e; ++i) {
        uint32_t w = (uint32_t)tokens[i];
        for (int k = 0; k < 4; ++k) {
            x ^= (uint64_t)((w >> (8 * k)) & 0xFFu);
            x *= 0x100000001b3ull;
        }
    }
    return x ? x : 1ull;
}

/* D2 alone: the rolling signature at every position (for the window pin).  sig_out[n]. */
void cdc_ora_signature(uint64_t seed, const int32_t* tokens, int64_t n, const int64_t* seq_offsets, int32_t n_seqs,
                       const int32_t* anchors, int32_t n_anchors, uint64_t* sig_out) {
    for (int32_t s = 0; s < n_seqs; ++s) {
        uint64_t h = 0;
        for (int64_t i = seq_offsets[s]; i < seq_offsets[s + 1] && i < n; ++i) {
            h = (h << 1) + cdc_ora_gear(seed, tokens[i]);
            sig_out[i] = h;
            if (is_anchor(tokens[i], anchors, n_anchors)) h = 0;
        }
    }
}

/* D2 + D3 + D4, one pass per sequence, in order.  chunk_end[c] = exclusive end (global index) of chunk c,
 * chunk_kind[c] = why it ended: 0 hash, 1 anchor, 2 max_size, 3 end of sequence.  Returns the number of chunks
 * (the caller sizes the outputs to n). */
int64_t cdc_ora_chunk(uint64_t seed, int32_t min_size, int32_t max_size, int32_t mask_bits, const int32_t* tokens,
                      int64_t n, const int64_t* seq_offsets, int32_t n_seqs, const int32_t* anchors,
                      int32_t n_anchors, int64_t* chunk_end, uint64_t* chunk_hash, int32_t* chunk_kind) {
    int64_t c = 0;
    (void)n;
    for (int32_t s = 0; s < n_seqs; ++s) {
        uint64_t h = 0;
        int64_t start = seq_offsets[s];
        for (int64_t i = seq_offsets[s]; i < seq_offsets[s + 1]; ++i) {
            h = (h << 1) + cdc_ora_gear(seed, tokens[i]);
            int64_t len = i - start + 1;
            int kind = -1;
            if (is_anchor(tokens[i], anchors, n_anchors)) kind = 1;
            else if (i == seq_offsets[s + 1] - 1) kind = 3;
            else if (len == max_size) kind = 2;
            else if (len >= min_size && (mask_bits == 0 || (h >> (64 - mask_bits)) == 0)) kind = 0;
            if (kind == 1) h = 0; /* A1: the anchor also resets the rolling hash (PAPER.md:389 (iii)) */
            if (kind >= 0) {
                chunk_end[c] = i + 1;
                chunk_hash[c] = cdc_ora_content_hash(tokens, start, i + 1);
                chunk_kind[c] = kind;
                ++c;
                start = i + 1;
            }
        }
    }
    return c;
}

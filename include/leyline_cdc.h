/*
 * leyline_cdc.h -- C ABI of the DISCOVERY side that precedes the Leyline splice:
 * anchored content-defined chunking of token sequences, chunk content hashes, and a device-resident content-hash
 * registry.  A chunk of a new prompt whose hash is registered at another position is a shifted-identical chunk; the
 * position difference is the Delta that leyline_plan / leyline_splice then re-anchor and rotate by.
 *
 * Source: arxiv/paper_2606_01065 ("PAPER.md:N" = line N of the paper text).  The paper fixes the structure --
 * a Gear-hash rolling signature over tokens (PAPER.md:389 (i)), chunking from absolute position 0 (ABSPOS_CDC,
 * :389 (ii)), a forced boundary AND a hash reset at chat-template special tokens (A1 anchored CDC, :389 (iii)),
 * registration under a content hash (:195, :397) -- and none of the constants.  Those are readings D1-D5 of DESIGN.md:
 *   D1  G(v) = splitmix64 output for state seed + (v+1) * 0x9E3779B97F4A7C15
 *   D2  h_i = (h_{i-1} << 1) + G(t_i) mod 2^64; h = 0 at a sequence start and after an anchor token; not reset at
 *       hash-defined boundaries (so h_i is a function of the last 64 tokens)
 *   D3  position i ends a chunk (inclusive) iff t_i is an anchor, else i is the last token of its sequence, else
 *       len == max_size, else (len >= min_size and the top mask_bits of h_i are zero); len = i - chunk_start + 1
 *   D4  content hash = FNV-1a 64 over the chunk's token ids as little-endian 4-byte words; 0 is stored as 1
 *   D5  registry: key -> the smallest value inserted under that key
 *
 * All pointers named dev_* are DEVICE pointers; every call is asynchronous on `cuda_stream` and returns only argument
 * or launch errors (LEYLINE_E_INVALID / LEYLINE_E_CUDA; see leyline.h for the status codes).  There is no CPU fallback.
 */
#ifndef LEYLINE_CDC_H_
#define LEYLINE_CDC_H_

#include <stddef.h>
#include <stdint.h>

#include "leyline.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    uint64_t seed;       /* D1 */
    int32_t min_size;    /* >= 1: a hash-defined boundary needs at least this many tokens in the chunk */
    int32_t max_size;    /* >= min_size, <= 4096: a chunk is cut at this length */
    int32_t mask_bits;   /* 0..32: a hash boundary needs the top mask_bits of h_i to be zero (expected gap 2^mask_bits) */
    int32_t reserved_;   /* must be 0 */
} leyline_cdc_params;

/* Why a chunk ended (dev_chunk_kind). */
typedef enum { LEYLINE_CDC_HASH = 0, LEYLINE_CDC_ANCHOR = 1, LEYLINE_CDC_MAX = 2, LEYLINE_CDC_SEQ_END = 3 } leyline_cdc_kind;

/*
 * leyline_cdc_chunk -- chunk n_seqs token sequences stored back to back.
 *
 *   dev_tokens       int32 [n_tokens], n_tokens < 2^31
 *   dev_seq_offsets  int64 [n_seqs + 1], ascending, [0] = 0, [n_seqs] = n_tokens (empty sequences allowed)
 *   dev_anchor_ids   int32 [n_anchor_ids], SORTED ascending token ids that force a boundary and reset the signature
 *                    (may be NULL when n_anchor_ids = 0: the paper's unanchored "legacy" chunker)
 *   dev_chunk_end    int64 [capacity]: exclusive end (global token index) of every chunk, ascending; chunk c starts
 *                    where chunk c-1 ends (chunks tile the concatenated sequences)
 *   dev_chunk_hash   uint64 [capacity] or NULL: D4 of every chunk
 *   dev_chunk_kind   int32 [capacity] or NULL: leyline_cdc_kind
 *   dev_n_chunks     int64 [1]: the number of chunks found.  If it exceeds `capacity` only the first `capacity`
 *                    entries were written (capacity = n_tokens always suffices)
 *
 * Scratch memory is allocated and freed stream-ordered by the call itself (about 30 B per token).
 */
LEYLINE_API leyline_status leyline_cdc_chunk(const leyline_cdc_params* params, const int32_t* dev_tokens, int64_t n_tokens,
                                 const int64_t* dev_seq_offsets, int32_t n_seqs, const int32_t* dev_anchor_ids,
                                 int32_t n_anchor_ids, int64_t* dev_chunk_end, uint64_t* dev_chunk_hash,
                                 int32_t* dev_chunk_kind, int64_t capacity, int64_t* dev_n_chunks, void* cuda_stream);

/*
 * Registry (D5): an open-addressing table in caller-owned device memory, `capacity` a power of two:
 * dev_keys uint64 [capacity] (0 = empty) and dev_vals int64 [capacity].  Keep it at most half full.
 *   clear   empties the table.
 *   insert  for i < n: table[hashes[i]] = min(table[hashes[i]], values[i]).  Entries that find no free slot are
 *           counted in dev_n_dropped (int64 [1], may be NULL; zeroed by the call).
 *   lookup  out[i] = the value stored under hashes[i], or -1.
 * Hash 0 is never a valid key (D4 remaps it).
 */
LEYLINE_API leyline_status leyline_registry_clear(uint64_t* dev_keys, int64_t* dev_vals, int64_t capacity, void* cuda_stream);
LEYLINE_API leyline_status leyline_registry_insert(uint64_t* dev_keys, int64_t* dev_vals, int64_t capacity,
                                       const uint64_t* dev_hashes, const int64_t* dev_values, int64_t n,
                                       int64_t* dev_n_dropped, void* cuda_stream);
LEYLINE_API leyline_status leyline_registry_lookup(const uint64_t* dev_keys, const int64_t* dev_vals, int64_t capacity,
                                       const uint64_t* dev_hashes, int64_t n, int64_t* dev_out, void* cuda_stream);

#ifdef __cplusplus
}
#endif

#endif /* LEYLINE_CDC_H_ */

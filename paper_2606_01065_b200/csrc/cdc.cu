/*
 * cdc.cu -- discovery side of the Leyline splice on the device (include/leyline_cdc.h):
 * anchored Gear-hash content-defined chunking (PAPER.md:389 (i)-(iii)), chunk content hashes and the content-hash
 * registry.  Readings D1-D5 of DESIGN.md fix the constants the paper leaves open.
 *
 * The sequential definition (one rolling hash, one open chunk) is restated so that every step is data-parallel:
 *   k_cdc_flags      per token: gear value G(t) (D1), "anchor" and "last token of its sequence" flags
 *   k_cdc_signature  per position: h_i as the 64-term window sum  sum_j G(t_{i-j}) << j  cut at the last reset (D2
 *                    in closed form: the shift drops a token out of the 64-bit word after 64 steps); the "hash
 *                    candidate" and "hard stop" (anchor / sequence end) predicates go into two BITMAPS, one ballot per
 *                    32 positions, with a second level (one bit per non-empty word) built by k_cdc_level1
 *   k_cdc_next       per position s: where a chunk that STARTS at s would end (D3) = min(next hard stop >= s,
 *                    s + max_size - 1, next candidate >= s + min_size - 1); "next set bit at or after i" is a
 *                    find-first-set in the position's word, else in the level-1 word: O(1) loads per position for
 *                    every legal (min_size, max_size, mask_bits), so the pass is linear in n
 *   k_cdc_reach      pointer doubling over s -> next(s): marks the starts actually reached from the sequence starts;
 *                    a round that sets no new mark proves the longest per-sequence chain is covered, and every later
 *                    round returns at once (ceil(log2(longest chain)) working rounds, not ceil(log2 n))
 *   k_cdc_count / k_cdc_scan / k_cdc_emit   ordered compaction of the marked starts
 *   k_cdc_hash       content hash per chunk (D4).  FNV-1a is a serial recurrence (x = (x ^ byte) * prime), so its
 *                    floor is the LONGEST chunk: 4 dependent 64-bit multiplies per token, <= 4 * max_size in a row
 * Integer work throughout; results are bit-exact against the CPU oracle.
 */
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "leyline_cdc.h"
#include "plan_internal.h" /* LEYLINE_CATCH_STATUS */

namespace {

constexpr int kT = 256;
constexpr uint8_t F_ANCHOR = 1, F_SEQ_END = 2;

thread_local std::string g_cdc_error;
bool ok(cudaError_t e) {
    if (e == cudaSuccess) return true;
    g_cdc_error = cudaGetErrorString(e);
    (void)cudaGetLastError();
    return false;
}
#define CU(call) do { if (!ok((call))) return LEYLINE_E_CUDA; } while (0)

__device__ __forceinline__ uint64_t gear_of(uint64_t seed, int32_t token) { /* D1: splitmix64 */
    uint64_t z = seed + ((uint64_t)(uint32_t)token + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__global__ void __launch_bounds__(kT) k_cdc_flags(const int32_t* __restrict__ tokens, int64_t n, const int32_t* __restrict__ anchors,
                                                  int n_anchors, uint64_t seed, uint64_t* __restrict__ gear, uint8_t* __restrict__ flags) {
    for (int64_t i = blockIdx.x * (int64_t)kT + threadIdx.x; i < n; i += (int64_t)gridDim.x * kT) {
        const int32_t t = tokens[i];
        int lo = 0, hi = n_anchors; /* first anchor >= t */
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(anchors + mid) < t) lo = mid + 1; else hi = mid;
        }
        gear[i] = gear_of(seed, t);
        flags[i] = (lo < n_anchors && __ldg(anchors + lo) == t) ? F_ANCHOR : 0;
    }
}

/* the last token of every non-empty sequence (runs after k_cdc_flags on the same stream).  Offsets live on the device
 * and cannot be validated by the host: anything outside [0, n] is ignored here rather than followed. */
__global__ void __launch_bounds__(kT) k_cdc_seq_ends(const int64_t* __restrict__ seq_offsets, int n_seqs, int64_t n,
                                                     uint8_t* __restrict__ flags, uint8_t* __restrict__ mark) {
    for (int s = blockIdx.x * kT + threadIdx.x; s < n_seqs; s += gridDim.x * kT) {
        const int64_t b = seq_offsets[s], e = seq_offsets[s + 1];
        if (e > b && b >= 0 && e <= n) {
            flags[e - 1] |= F_SEQ_END; /* one writer per byte: sequences do not share tokens */
            mark[b] = 1;               /* a chunk starts at every sequence start */
        }
    }
}

/* D2 + the two predicates of D3 as bitmaps.  Word w of hard0 / cand0 covers positions [32w, 32w + 32): a warp handles 32
 * consecutive positions and lane 0 stores the ballot, so every word (also the tail, where positions >= n read as 0) is
 * written exactly once and nothing is modified in place. */
__global__ void __launch_bounds__(kT) k_cdc_signature(const uint64_t* __restrict__ gear, const uint8_t* __restrict__ flags, int64_t n,
                                                      int64_t n_padded, int mask_bits, uint32_t* __restrict__ hard0,
                                                      uint32_t* __restrict__ cand0) {
    for (int64_t i = blockIdx.x * (int64_t)kT + threadIdx.x; i < n_padded; i += (int64_t)gridDim.x * kT) {
        bool hard = false, cand = false;
        if (i < n) {
            uint64_t h = gear[i];
            for (int j = 1; j < 64; ++j) {
                const int64_t k = i - j;
                if (k < 0 || flags[k]) break; /* the signature was reset after token k (anchor or end of a sequence) */
                h += gear[k] << j;
            }
            hard = flags[i] != 0;
            cand = mask_bits == 0 || (h >> (64 - mask_bits)) == 0;
        }
        const unsigned hb = __ballot_sync(0xFFFFFFFFu, hard), cb = __ballot_sync(0xFFFFFFFFu, cand);
        if ((threadIdx.x & 31) == 0) { hard0[i >> 5] = hb; cand0[i >> 5] = cb; }
    }
}

/* level 1: bit b of word v <=> level-0 word 32v + b is non-zero (both bitmaps in one pass) */
__global__ void __launch_bounds__(kT) k_cdc_level1(const uint32_t* __restrict__ hard0, const uint32_t* __restrict__ cand0, int64_t n_words,
                                                   int64_t n_words_padded, uint32_t* __restrict__ hard1, uint32_t* __restrict__ cand1) {
    for (int64_t w = blockIdx.x * (int64_t)kT + threadIdx.x; w < n_words_padded; w += (int64_t)gridDim.x * kT) {
        const unsigned hb = __ballot_sync(0xFFFFFFFFu, w < n_words && hard0[w] != 0);
        const unsigned cb = __ballot_sync(0xFFFFFFFFu, w < n_words && cand0[w] != 0);
        if ((threadIdx.x & 31) == 0) { hard1[w >> 5] = hb; cand1[w >> 5] = cb; }
    }
}

/* first set position >= i and <= last in a two-level bitmap, or INT64_MAX.  At most 2 + (last - i) / 1024 word loads. */
__device__ __forceinline__ int64_t next_set(const uint32_t* __restrict__ l0, const uint32_t* __restrict__ l1, int64_t i, int64_t last) {
    if (i > last) return INT64_MAX;
    int64_t w = i >> 5;
    uint32_t m = __ldg(l0 + w) & (0xFFFFFFFFu << (i & 31));
    if (!m) {
        int64_t v = w >> 5;
        const int b = (int)(w & 31);
        uint32_t m1 = b == 31 ? 0u : (__ldg(l1 + v) & (0xFFFFFFFFu << (b + 1)));
        const int64_t v_last = last >> 10;
        while (!m1) {
            if (++v > v_last) return INT64_MAX;
            m1 = __ldg(l1 + v);
        }
        w = (v << 5) + (__ffs((int)m1) - 1);
        m = __ldg(l0 + w);
    }
    const int64_t pos = (w << 5) + (__ffs((int)m) - 1);
    return pos <= last ? pos : INT64_MAX;
}

/* D3 for a chunk starting at s: nxt[s] = exclusive end, kind[s] = why.  The first of: an anchor or the end of the
 * sequence at or after s, the max_size-th token, a hash candidate from the min_size-th token on (D3's order decides
 * ties).  Never reads or reports anything past n, whatever the device-side offsets say. */
__global__ void __launch_bounds__(kT) k_cdc_next(const uint8_t* __restrict__ flags, const uint32_t* __restrict__ hard0,
                                                 const uint32_t* __restrict__ hard1, const uint32_t* __restrict__ cand0,
                                                 const uint32_t* __restrict__ cand1, int64_t n, int min_size, int max_size,
                                                 int32_t* __restrict__ nxt, uint8_t* __restrict__ kind) {
    for (int64_t s = blockIdx.x * (int64_t)kT + threadIdx.x; s <= n; s += (int64_t)gridDim.x * kT) {
        if (s == n) { nxt[s] = (int32_t)n; break; } /* terminal: the chain stops here */
        const int64_t i_max = min(s + max_size - 1, n - 1); /* the last token of the pool ends a chunk in any case */
        const int64_t i_hard = next_set(hard0, hard1, s, i_max);
        const int64_t i_cand = next_set(cand0, cand1, s + min_size - 1, i_max);
        int64_t i;
        int why;
        if (i_hard <= i_cand && i_hard != INT64_MAX) {
            i = i_hard;
            why = (flags[i] & F_ANCHOR) ? LEYLINE_CDC_ANCHOR : LEYLINE_CDC_SEQ_END;
        } else if (i_cand != INT64_MAX && i_cand < s + max_size - 1) {
            i = i_cand;
            why = LEYLINE_CDC_HASH;
        } else {
            i = i_max;
            why = i_max == s + max_size - 1 ? LEYLINE_CDC_MAX : LEYLINE_CDC_SEQ_END;
        }
        nxt[s] = (int32_t)(i + 1);
        kind[s] = (uint8_t)why;
    }
}

/* One round of pointer doubling: jump_in = next applied 2^k times.  Every marked start marks the start 2^k chunks
 * ahead; marks only ever land on starts of the true chain, so reading a mark set in this same round is harmless.
 * progress[0] (the previous round's) == 0: that round set no new mark, so every chain is complete (a sequence's k-th
 * round is the only one that can mark its chunks 2^k .. 2^(k+1) - 1) and this round has nothing to do. */
__global__ void __launch_bounds__(kT) k_cdc_reach(const int32_t* __restrict__ jump_in, int32_t* __restrict__ jump_out, int64_t n,
                                                  uint8_t* __restrict__ mark, const int32_t* __restrict__ progress_prev,
                                                  int32_t* __restrict__ progress) {
    if (progress_prev && *progress_prev == 0) return;
    bool any = false;
    for (int64_t s = blockIdx.x * (int64_t)kT + threadIdx.x; s <= n; s += (int64_t)gridDim.x * kT) {
        const int32_t j = jump_in[s];
        if (s < n && j < n && mark[s] && !mark[j]) { mark[j] = 1; any = true; }
        jump_out[s] = jump_in[j];
    }
    if (__any_sync(0xFFFFFFFFu, any) && (threadIdx.x & 31) == 0) *progress = 1;
}

/* ---- ordered compaction of the marked starts ---- */

constexpr int kItems = 8;                 /* consecutive positions per thread */
constexpr int kBlockSpan = kT * kItems;   /* positions per block */

__global__ void __launch_bounds__(kT) k_cdc_count(const uint8_t* __restrict__ mark, int64_t n, int32_t* __restrict__ block_count) {
    __shared__ int s_warp[kT / 32];
    const int64_t base = blockIdx.x * (int64_t)kBlockSpan + threadIdx.x * kItems;
    int c = 0;
#pragma unroll
    for (int k = 0; k < kItems; ++k)
        if (base + k < n && mark[base + k]) ++c;
    for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, o);
    if ((threadIdx.x & 31) == 0) s_warp[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0;
        for (int w = 0; w < kT / 32; ++w) tot += s_warp[w];
        block_count[blockIdx.x] = tot;
    }
}

/* exclusive scan of the block counts by ONE block (n / 2048 entries: 512 for a million tokens); also the total */
__global__ void __launch_bounds__(1024) k_cdc_scan(int32_t* __restrict__ block_count, int n_blocks, int64_t* __restrict__ n_chunks) {
    __shared__ int s_part[1024];
    __shared__ int s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (int base = 0; base < n_blocks; base += 1024) {
        const int i = base + threadIdx.x;
        const int v = i < n_blocks ? block_count[i] : 0;
        s_part[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) { /* Hillis-Steele inclusive scan */
            const int add = threadIdx.x >= o ? s_part[threadIdx.x - o] : 0;
            __syncthreads();
            s_part[threadIdx.x] += add;
            __syncthreads();
        }
        const int carry = s_carry;
        if (i < n_blocks) block_count[i] = carry + s_part[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = carry + s_part[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_chunks = s_carry;
}

__device__ __forceinline__ uint64_t fnv1a_tokens(const int32_t* __restrict__ tokens, int64_t b, int64_t e) { /* D4 */
    uint64_t x = 0xcbf29ce484222325ull;
    for (int64_t i = b; i < e; ++i) {
        const uint32_t w = (uint32_t)tokens[i];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            x ^= (uint64_t)((w >> (8 * k)) & 0xFFu);
            x *= 0x100000001b3ull;
        }
    }
    return x ? x : 1ull;
}

/* chunk c = the c-th marked start in position order: end, kind */
__global__ void __launch_bounds__(kT) k_cdc_emit(const uint8_t* __restrict__ mark, const int32_t* __restrict__ nxt,
                                                 const uint8_t* __restrict__ kind, int64_t n, const int32_t* __restrict__ block_offset,
                                                 int64_t capacity, int64_t* __restrict__ chunk_end, int32_t* __restrict__ chunk_kind,
                                                 int32_t* __restrict__ chunk_start) {
    __shared__ int s_warp[kT / 32];
    const int64_t base = blockIdx.x * (int64_t)kBlockSpan + threadIdx.x * kItems;
    int c = 0;
#pragma unroll
    for (int k = 0; k < kItems; ++k)
        if (base + k < n && mark[base + k]) ++c;
    int incl = c; /* inclusive scan inside the warp */
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if ((threadIdx.x & 31) >= o) incl += v;
    }
    if ((threadIdx.x & 31) == 31) s_warp[threadIdx.x >> 5] = incl;
    __syncthreads();
    int before = block_offset[blockIdx.x] + incl - c;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) before += s_warp[w];
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const int64_t s = base + k;
        if (s < n && mark[s]) {
            if (before < capacity) {
                chunk_end[before] = nxt[s];
                if (chunk_kind) chunk_kind[before] = kind[s];
                chunk_start[before] = (int32_t)s;
            }
            ++before;
        }
    }
}

__global__ void __launch_bounds__(kT) k_cdc_hash(const int32_t* __restrict__ tokens, const int32_t* __restrict__ chunk_start,
                                                 const int64_t* __restrict__ chunk_end, const int64_t* __restrict__ n_chunks,
                                                 int64_t capacity, uint64_t* __restrict__ chunk_hash) {
    const int64_t m = *n_chunks < capacity ? *n_chunks : capacity;
    for (int64_t c = blockIdx.x * (int64_t)kT + threadIdx.x; c < m; c += (int64_t)gridDim.x * kT)
        chunk_hash[c] = fnv1a_tokens(tokens, chunk_start[c], chunk_end[c]);
}

/* ---- registry (D5) ---- */

__device__ __forceinline__ uint64_t slot_hash(uint64_t key) { /* keys are FNV outputs; fold the high half in */
    key ^= key >> 32;
    return key * 0x9E3779B97F4A7C15ull;
}

__global__ void __launch_bounds__(kT) k_reg_clear(uint64_t* __restrict__ keys, int64_t* __restrict__ vals, int64_t capacity) {
    for (int64_t i = blockIdx.x * (int64_t)kT + threadIdx.x; i < capacity; i += (int64_t)gridDim.x * kT) {
        keys[i] = 0;
        vals[i] = INT64_MAX;
    }
}

__global__ void __launch_bounds__(kT) k_reg_insert(uint64_t* __restrict__ keys, int64_t* __restrict__ vals, int64_t capacity,
                                                   const uint64_t* __restrict__ hashes, const int64_t* __restrict__ values, int64_t n,
                                                   int64_t* __restrict__ n_dropped) {
    for (int64_t i = blockIdx.x * (int64_t)kT + threadIdx.x; i < n; i += (int64_t)gridDim.x * kT) {
        const uint64_t key = hashes[i];
        if (key == 0) { if (n_dropped) atomicAdd((unsigned long long*)n_dropped, 1ull); continue; }
        uint64_t slot = (slot_hash(key) >> 20) & (uint64_t)(capacity - 1);
        bool done = false;
        for (int64_t probe = 0; probe < capacity; ++probe, slot = (slot + 1) & (uint64_t)(capacity - 1)) {
            const unsigned long long seen = atomicCAS((unsigned long long*)&keys[slot], 0ull, (unsigned long long)key);
            if (seen == 0ull || seen == key) {
                atomicMin((long long*)&vals[slot], (long long)values[i]);
                done = true;
                break;
            }
        }
        if (!done && n_dropped) atomicAdd((unsigned long long*)n_dropped, 1ull);
    }
}

__global__ void __launch_bounds__(kT) k_reg_lookup(const uint64_t* __restrict__ keys, const int64_t* __restrict__ vals, int64_t capacity,
                                                   const uint64_t* __restrict__ hashes, int64_t n, int64_t* __restrict__ out) {
    for (int64_t i = blockIdx.x * (int64_t)kT + threadIdx.x; i < n; i += (int64_t)gridDim.x * kT) {
        const uint64_t key = hashes[i];
        int64_t found = -1;
        if (key != 0) {
            uint64_t slot = (slot_hash(key) >> 20) & (uint64_t)(capacity - 1);
            for (int64_t probe = 0; probe < capacity; ++probe, slot = (slot + 1) & (uint64_t)(capacity - 1)) {
                const uint64_t seen = keys[slot];
                if (seen == key) { found = vals[slot]; break; }
                if (seen == 0) break;
            }
        }
        out[i] = found;
    }
}

unsigned grid_for(int64_t n, int per_block = kT) {
    int64_t b = (n + per_block - 1) / per_block;
    if (b < 1) b = 1;
    if (b > 148 * 16) b = 148 * 16;
    return (unsigned)b;
}

}  // namespace

extern "C" LEYLINE_API leyline_status leyline_cdc_chunk(const leyline_cdc_params* p, const int32_t* dev_tokens, int64_t n,
                                            const int64_t* dev_seq_offsets, int32_t n_seqs, const int32_t* dev_anchor_ids,
                                            int32_t n_anchor_ids, int64_t* dev_chunk_end, uint64_t* dev_chunk_hash,
                                            int32_t* dev_chunk_kind, int64_t capacity, int64_t* dev_n_chunks,
                                            void* cuda_stream) try {
    g_cdc_error.clear();
    if (!p || p->reserved_ != 0 || p->min_size < 1 || p->max_size < p->min_size || p->max_size > 4096 ||
        p->mask_bits < 0 || p->mask_bits > 32)
        return LEYLINE_E_INVALID;
    if (n < 0 || n >= (int64_t(1) << 31) || n_seqs < 0 || n_anchor_ids < 0 || capacity < 0) return LEYLINE_E_INVALID;
    if (!dev_n_chunks || !dev_seq_offsets || (n > 0 && (!dev_tokens || n_seqs < 1)) || (capacity > 0 && !dev_chunk_end) ||
        (n_anchor_ids > 0 && !dev_anchor_ids))
        return LEYLINE_E_INVALID;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (n == 0) {
        CU(cudaMemsetAsync(dev_n_chunks, 0, sizeof(int64_t), stream));
        return LEYLINE_OK;
    }
    /* scratch: gear u64[n] | jumpA i32[n+1] | jumpB i32[n+1] | nxt i32[n+1] | start i32[n] | blocks i32 | bitmaps (two
     * levels x two predicates) | progress i32[rounds] | flags, kind, mark */
    auto up = [](int64_t x) { return (x + 255) / 256 * 256; };
    const int64_t n_blocks = (n + kBlockSpan - 1) / kBlockSpan;
    const int64_t n_words = (n + 31) / 32, n_words_padded = (n_words + 31) / 32 * 32, n_words1 = n_words_padded / 32;
    int rounds = 0; /* the chain has at most n links: ceil(log2(n + 1)) doubling rounds reach all of it */
    for (int64_t reach = 1; reach <= n; reach <<= 1) ++rounds;
    const int64_t o_gear = 0, o_ja = o_gear + up(n * 8), o_jb = o_ja + up((n + 1) * 4), o_nxt = o_jb + up((n + 1) * 4),
                  o_start = o_nxt + up((n + 1) * 4), o_blk = o_start + up(n * 4), o_h0 = o_blk + up(n_blocks * 4),
                  o_c0 = o_h0 + up(n_words_padded * 4), o_h1 = o_c0 + up(n_words_padded * 4), o_c1 = o_h1 + up((n_words1 + 1) * 4),
                  o_prog = o_c1 + up((n_words1 + 1) * 4), o_flags = o_prog + up((rounds + 1) * 4), o_kind = o_flags + up(n + 1),
                  o_mark = o_kind + up(n + 1), total = o_mark + up(n + 1);
    uint8_t* ws = nullptr;
    CU(cudaMallocAsync(reinterpret_cast<void**>(&ws), (size_t)total, stream));
    uint64_t* gear = reinterpret_cast<uint64_t*>(ws + o_gear);
    int32_t* ja = reinterpret_cast<int32_t*>(ws + o_ja);
    int32_t* jb = reinterpret_cast<int32_t*>(ws + o_jb);
    int32_t* nxt = reinterpret_cast<int32_t*>(ws + o_nxt);
    int32_t* start = reinterpret_cast<int32_t*>(ws + o_start);
    int32_t* blk = reinterpret_cast<int32_t*>(ws + o_blk);
    uint32_t *hard0 = reinterpret_cast<uint32_t*>(ws + o_h0), *cand0 = reinterpret_cast<uint32_t*>(ws + o_c0),
             *hard1 = reinterpret_cast<uint32_t*>(ws + o_h1), *cand1 = reinterpret_cast<uint32_t*>(ws + o_c1);
    int32_t* progress = reinterpret_cast<int32_t*>(ws + o_prog);
    uint8_t *flags = ws + o_flags, *kind = ws + o_kind, *mark = ws + o_mark;
    leyline_status st = LEYLINE_OK;
    auto fail = [&]() { cudaFreeAsync(ws, stream); return LEYLINE_E_CUDA; };
    /* progress | flags | kind | mark are contiguous: one memset (flags must be 0 where k_cdc_flags does not write) */
    if (!ok(cudaMemsetAsync(progress, 0, (size_t)(total - o_prog), stream))) return fail();
    k_cdc_flags<<<grid_for(n), kT, 0, stream>>>(dev_tokens, n, dev_anchor_ids, n_anchor_ids, p->seed, gear, flags);
    k_cdc_seq_ends<<<grid_for(n_seqs), kT, 0, stream>>>(dev_seq_offsets, n_seqs, n, flags, mark);
    k_cdc_signature<<<grid_for(n_words * 32), kT, 0, stream>>>(gear, flags, n, n_words * 32, p->mask_bits, hard0, cand0);
    k_cdc_level1<<<grid_for(n_words_padded), kT, 0, stream>>>(hard0, cand0, n_words, n_words_padded, hard1, cand1);
    k_cdc_next<<<grid_for(n + 1), kT, 0, stream>>>(flags, hard0, hard1, cand0, cand1, n, p->min_size, p->max_size, nxt, kind);
    const int32_t* jin = nxt;
    int32_t* jout = ja;
    for (int r = 0; r < rounds; ++r) {
        k_cdc_reach<<<grid_for(n + 1), kT, 0, stream>>>(jin, jout, n, mark, r ? progress + r - 1 : nullptr, progress + r);
        jin = jout;
        jout = (jout == ja) ? jb : ja;
    }
    k_cdc_count<<<(unsigned)n_blocks, kT, 0, stream>>>(mark, n, blk);
    k_cdc_scan<<<1, 1024, 0, stream>>>(blk, (int)n_blocks, dev_n_chunks);
    if (capacity > 0) {
        k_cdc_emit<<<(unsigned)n_blocks, kT, 0, stream>>>(mark, nxt, kind, n, blk, capacity, dev_chunk_end, dev_chunk_kind, start);
        if (dev_chunk_hash)
            k_cdc_hash<<<grid_for(capacity < n ? capacity : n, kT), kT, 0, stream>>>(dev_tokens, start, dev_chunk_end, dev_n_chunks,
                                                                                  capacity, dev_chunk_hash);
    }
    if (!ok(cudaGetLastError())) st = LEYLINE_E_CUDA;
    if (!ok(cudaFreeAsync(ws, stream))) st = LEYLINE_E_CUDA;
    return st;
} LEYLINE_CATCH_STATUS

static bool pow2(int64_t x) { return x > 0 && (x & (x - 1)) == 0; }

extern "C" LEYLINE_API leyline_status leyline_registry_clear(uint64_t* dev_keys, int64_t* dev_vals, int64_t capacity, void* cuda_stream) try {
    g_cdc_error.clear();
    if (!dev_keys || !dev_vals || !pow2(capacity)) return LEYLINE_E_INVALID;
    k_reg_clear<<<grid_for(capacity), kT, 0, static_cast<cudaStream_t>(cuda_stream)>>>(dev_keys, dev_vals, capacity);
    CU(cudaGetLastError());
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

extern "C" LEYLINE_API leyline_status leyline_registry_insert(uint64_t* dev_keys, int64_t* dev_vals, int64_t capacity,
                                                  const uint64_t* dev_hashes, const int64_t* dev_values, int64_t n,
                                                  int64_t* dev_n_dropped, void* cuda_stream) try {
    g_cdc_error.clear();
    if (!dev_keys || !dev_vals || !pow2(capacity) || n < 0 || (n > 0 && (!dev_hashes || !dev_values))) return LEYLINE_E_INVALID;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (dev_n_dropped) CU(cudaMemsetAsync(dev_n_dropped, 0, sizeof(int64_t), stream));
    if (n == 0) return LEYLINE_OK;
    k_reg_insert<<<grid_for(n), kT, 0, stream>>>(dev_keys, dev_vals, capacity, dev_hashes, dev_values, n, dev_n_dropped);
    CU(cudaGetLastError());
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

extern "C" LEYLINE_API leyline_status leyline_registry_lookup(const uint64_t* dev_keys, const int64_t* dev_vals, int64_t capacity,
                                                  const uint64_t* dev_hashes, int64_t n, int64_t* dev_out, void* cuda_stream) try {
    g_cdc_error.clear();
    if (!dev_keys || !dev_vals || !pow2(capacity) || n < 0 || (n > 0 && (!dev_hashes || !dev_out))) return LEYLINE_E_INVALID;
    if (n == 0) return LEYLINE_OK;
    k_reg_lookup<<<grid_for(n), kT, 0, static_cast<cudaStream_t>(cuda_stream)>>>(dev_keys, dev_vals, capacity, dev_hashes, n, dev_out);
    CU(cudaGetLastError());
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

/*
 * cdc.cu -- discovery side of the Leyline splice on the device (include/leyline_cdc.h):
 * anchored Gear-hash content-defined chunking (PAPER.md:389 (i)-(iii)), chunk content hashes and the content-hash
 * registry.  Readings D1-D5 of DESIGN.md fix the constants the paper leaves open.
 *
 * The sequential definition (one rolling hash, one open chunk) is restated so that every step is data-parallel:
 *   k_cdc_flags      per token: gear value G(t) (D1), "anchor" and "last token of its sequence" flags
 *   k_cdc_signature  per position: h_i as the 64-term window sum  sum_j G(t_{i-j}) << j  cut at the last reset (D2
 *                    in closed form: the shift drops a token out of the 64-bit word after 64 steps), candidate flag
 *   k_cdc_next       per position s: where a chunk that STARTS at s would end (D3), scanning <= max_size flags
 *   k_cdc_reach      pointer doubling over s -> next(s): marks the starts actually reached from the sequence starts
 *   k_cdc_count / k_cdc_scan / k_cdc_emit   ordered compaction of the marked starts, content hash per chunk (D4)
 * Integer work throughout; results are bit-exact against the CPU oracle.
 */
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "leyline_cdc.h"
#include "plan_internal.h" /* LEYLINE_CATCH_STATUS */

namespace {

constexpr int kT = 256;
constexpr uint8_t F_ANCHOR = 1, F_SEQ_END = 2, F_CAND = 4;

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

/* the last token of every non-empty sequence (runs after k_cdc_flags on the same stream) */
__global__ void __launch_bounds__(kT) k_cdc_seq_ends(const int64_t* __restrict__ seq_offsets, int n_seqs, uint8_t* __restrict__ flags,
                                                     uint8_t* __restrict__ mark) {
    for (int s = blockIdx.x * kT + threadIdx.x; s < n_seqs; s += gridDim.x * kT) {
        const int64_t b = seq_offsets[s], e = seq_offsets[s + 1];
        if (e > b) {
            flags[e - 1] |= F_SEQ_END; /* one writer per byte: sequences do not share tokens */
            mark[b] = 1;               /* a chunk starts at every sequence start */
        }
    }
}

__global__ void __launch_bounds__(kT) k_cdc_signature(const uint64_t* __restrict__ gear, int64_t n, int mask_bits,
                                                      uint8_t* __restrict__ flags) {
    for (int64_t i = blockIdx.x * (int64_t)kT + threadIdx.x; i < n; i += (int64_t)gridDim.x * kT) {
        uint64_t h = gear[i];
        for (int j = 1; j < 64; ++j) {
            const int64_t k = i - j;
            if (k < 0 || (flags[k] & (F_ANCHOR | F_SEQ_END))) break; /* the signature was reset after token k */
            h += gear[k] << j;
        }
        /* only bit 2 changes here and only this thread writes flags[i]; neighbours read bits 0-1, which are final */
        if (mask_bits == 0 || (h >> (64 - mask_bits)) == 0) flags[i] |= F_CAND;
    }
}

/* D3 for a chunk starting at s: nxt[s] = exclusive end, kind[s] = why. */
__global__ void __launch_bounds__(kT) k_cdc_next(const uint8_t* __restrict__ flags, int64_t n, int min_size, int max_size,
                                                 int32_t* __restrict__ nxt, uint8_t* __restrict__ kind) {
    for (int64_t s = blockIdx.x * (int64_t)kT + threadIdx.x; s <= n; s += (int64_t)gridDim.x * kT) {
        if (s == n) { nxt[s] = (int32_t)n; break; } /* terminal: the chain stops here */
        int64_t i = s;
        int why;
        for (;; ++i) {
            const uint8_t f = flags[i];
            const int64_t len = i - s + 1;
            if (f & F_ANCHOR) { why = LEYLINE_CDC_ANCHOR; break; }
            if (f & F_SEQ_END) { why = LEYLINE_CDC_SEQ_END; break; }
            if (len == max_size) { why = LEYLINE_CDC_MAX; break; }
            if (len >= min_size && (f & F_CAND)) { why = LEYLINE_CDC_HASH; break; }
        }
        nxt[s] = (int32_t)(i + 1);
        kind[s] = (uint8_t)why;
    }
}

/* One round of pointer doubling: jump_in = next applied 2^k times.  Every marked start marks the start 2^k chunks
 * ahead; marks only ever land on starts of the true chain, so reading a mark set in this same round is harmless. */
__global__ void __launch_bounds__(kT) k_cdc_reach(const int32_t* __restrict__ jump_in, int32_t* __restrict__ jump_out, int64_t n,
                                                  uint8_t* __restrict__ mark) {
    for (int64_t s = blockIdx.x * (int64_t)kT + threadIdx.x; s <= n; s += (int64_t)gridDim.x * kT) {
        const int32_t j = jump_in[s];
        if (s < n && j < n && mark[s]) mark[j] = 1;
        jump_out[s] = jump_in[j];
    }
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
    /* scratch: gear u64[n] | jumpA i32[n+1] | jumpB i32[n+1] | nxt i32[n+1] | start i32[n] | blocks i32 | flags, kind, mark */
    auto up = [](int64_t x) { return (x + 255) / 256 * 256; };
    const int64_t n_blocks = (n + kBlockSpan - 1) / kBlockSpan;
    const int64_t o_gear = 0, o_ja = o_gear + up(n * 8), o_jb = o_ja + up((n + 1) * 4), o_nxt = o_jb + up((n + 1) * 4),
                  o_start = o_nxt + up((n + 1) * 4), o_blk = o_start + up(n * 4), o_flags = o_blk + up(n_blocks * 4),
                  o_kind = o_flags + up(n + 1), o_mark = o_kind + up(n + 1), total = o_mark + up(n + 1);
    uint8_t* ws = nullptr;
    CU(cudaMallocAsync(reinterpret_cast<void**>(&ws), (size_t)total, stream));
    uint64_t* gear = reinterpret_cast<uint64_t*>(ws + o_gear);
    int32_t* ja = reinterpret_cast<int32_t*>(ws + o_ja);
    int32_t* jb = reinterpret_cast<int32_t*>(ws + o_jb);
    int32_t* nxt = reinterpret_cast<int32_t*>(ws + o_nxt);
    int32_t* start = reinterpret_cast<int32_t*>(ws + o_start);
    int32_t* blk = reinterpret_cast<int32_t*>(ws + o_blk);
    uint8_t *flags = ws + o_flags, *kind = ws + o_kind, *mark = ws + o_mark;
    leyline_status st = LEYLINE_OK;
    auto fail = [&]() { cudaFreeAsync(ws, stream); return LEYLINE_E_CUDA; };
    if (!ok(cudaMemsetAsync(mark, 0, (size_t)(n + 1), stream))) return fail();
    k_cdc_flags<<<grid_for(n), kT, 0, stream>>>(dev_tokens, n, dev_anchor_ids, n_anchor_ids, p->seed, gear, flags);
    k_cdc_seq_ends<<<grid_for(n_seqs), kT, 0, stream>>>(dev_seq_offsets, n_seqs, flags, mark);
    k_cdc_signature<<<grid_for(n), kT, 0, stream>>>(gear, n, p->mask_bits, flags);
    k_cdc_next<<<grid_for(n + 1), kT, 0, stream>>>(flags, n, p->min_size, p->max_size, nxt, kind);
    /* the chain has at most n links: ceil(log2(n + 1)) doubling rounds reach all of it */
    const int32_t* jin = nxt;
    int32_t* jout = ja;
    for (int64_t reach = 1; reach <= n; reach <<= 1) {
        k_cdc_reach<<<grid_for(n + 1), kT, 0, stream>>>(jin, jout, n, mark);
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

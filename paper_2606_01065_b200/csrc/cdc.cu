/*
 * cdc.cu -- discovery side of the Leyline splice on the device (include/leyline_cdc.h):
 * anchored Gear-hash content-defined chunking (PAPER.md:389 (i)-(iii)), chunk content hashes and the content-hash
 * registry.  Readings D1-D5 of DESIGN.md fix the constants the paper leaves open.
 *
 * The sequential definition (one rolling hash, one open chunk) is restated so that every step is data-parallel:
 *   k_cdc_front      everything that is a function of a 64-token window, one launch: gear value G(t) (D1), "anchor" /
 *                    "last token of its sequence" flags, h_i as the 64-term window sum  sum_j G(t_{i-j}) << j  cut at the
 *                    last reset (D2 in closed form: the shift drops a token out of the 64-bit word after 64 steps), the
 *                    "hash candidate" and "hard stop" (anchor / sequence end) predicates as two-level BITMAPS (one
 *                    ballot per 32 positions, one bit per non-empty word above it), and the chain SEEDS: a chunk starts
 *                    for certain at every sequence start and behind every hard stop
 *   k_cdc_next       per position s: where a chunk that STARTS at s would end (D3) = min(next hard stop >= s,
 *                    s + max_size - 1, next candidate >= s + min_size - 1); "next set bit at or after i" is a
 *                    find-first-set in the position's word, else in the level-1 word: O(1) loads per position for
 *                    every legal (min_size, max_size, mask_bits), so the pass is linear in n
 *   k_cdc_reach      pointer doubling over s -> next(s): marks the starts actually reached from the seeds.  Between two
 *                    seeds every chunk but the last holds >= min_size tokens, so ceil(log2(n / min_size + 2)) rounds
 *                    always suffice; a round that sets no new mark proves every chain is covered, and every later
 *                    round returns at once
 *   k_cdc_count_scan ordered compaction of the marked starts: marks per block, scanned by the block that finishes last
 *   k_cdc_emit       chunk end, kind and content hash (D4).  FNV-1a is a serial recurrence (x = (x ^ byte) * prime), so
 *                    the floor is the LONGEST chunk: 4 dependent 64-bit multiplies per token, <= 4 * max_size in a row
 * The call is a chain of R + 4 small dependent launches on ~1 MB of input (R = the doubling rounds), so it is bound by
 * the launch-to-launch gap: every kernel is launched with programmatic stream serialisation (PDL) and lets its successor
 * be scheduled while it runs.  No memset, no intermediate host step.
 * Integer work throughout; results are bit-exact against the CPU oracle.
 */
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <string>

#include "leyline_cdc.h"
#include "plan_internal.h" /* LEYLINE_CATCH_STATUS */

namespace {

constexpr int kT = 256;
constexpr uint8_t F_ANCHOR = 1, F_SEQ_END = 2, F_RESET = 3 /* either: a hard stop, and the signature restarts behind it */,
                  F_SEQ_START = 4 /* shared-memory only: a non-empty sequence starts here */;

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

/* Programmatic dependent launch (sm_90+): every kernel of the call lets its successor be scheduled at once
 * (launch_dependents) and then waits until its predecessor has completed and flushed (wait).  The call is a chain of ~20
 * small dependent launches on 1 MB of input, so what it costs is the launch-to-launch gap, and this is what hides it. */
__device__ __forceinline__ void pdl_enter() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

constexpr int kSigSpan = 1024;              /* positions per block pass = one level-1 bitmap word */
constexpr int kSigHalo = 63;                /* D2: h_i depends on the last 64 tokens */

/* k_cdc_front: everything that is a function of a 64-token window, in ONE launch.  A block pass covers the 1024 positions
 * of one level-1 word v plus a 63-token halo in front of it:
 *   - gear value G(t) (D1) and the reset flags of those 1087 positions go to shared memory: "anchor" by bisection of the
 *     sorted anchor ids, "last token of a non-empty sequence" by bisection of the sequence offsets;
 *   - the chain seeds (mark[i], every position written exactly once): position i starts a chunk for certain when a
 *     sequence starts there or when position i - 1 is a hard stop (an anchor or a sequence end, D3).  With these seeds the pointer doubling only has to cover the chunks
 *     between two hard stops, all of which but the last hold >= min_size tokens;
 *   - h_i as the 64-term window sum  sum_j G(t_{i-j}) << j  cut at the last reset (D2 in closed form), the "hash
 *     candidate" and "hard stop" predicates as two bitmaps (one ballot per 32 positions) and their level-1 words (one
 *     bit per non-empty level-0 word).
 * Offsets live on the device and cannot be validated by the host: the bisections only ever index [0, n_seqs], and nothing
 * at or past n is written. */
__global__ void __launch_bounds__(kT) k_cdc_front(const int32_t* __restrict__ tokens, int64_t n, const int32_t* __restrict__ anchors,
                                                  int n_anchors, uint64_t seed, const int64_t* __restrict__ seq_offsets, int n_seqs,
                                                  int mask_bits, int64_t n_super, uint8_t* __restrict__ flags, uint8_t* __restrict__ mark,
                                                  uint32_t* __restrict__ hard0, uint32_t* __restrict__ cand0,
                                                  uint32_t* __restrict__ hard1, uint32_t* __restrict__ cand1,
                                                  int32_t* __restrict__ progress, int n_progress) {
    __shared__ uint64_t s_gear[kSigSpan + kSigHalo];
    __shared__ uint8_t s_flag[kSigSpan + kSigHalo];
    __shared__ uint32_t s_nonzero[2][kSigSpan / 32];
    pdl_enter();
    if (blockIdx.x == 0)
        for (int k = threadIdx.x; k < n_progress; k += kT) progress[k] = 0;
    const int64_t first = seq_offsets[0];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int64_t v = blockIdx.x; v < n_super; v += gridDim.x) {
        const int64_t base = v * kSigSpan - kSigHalo;
        for (int k = threadIdx.x; k < kSigSpan + kSigHalo; k += kT) {
            const int64_t i = base + k;
            uint64_t g = 0;
            uint8_t f = F_SEQ_END; /* outside [0, n): a reset, so that no window reaches across it */
            if (i >= 0 && i < n) {
                const int32_t t = tokens[i];
                int lo = 0, hi = n_anchors; /* first anchor >= t */
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (__ldg(anchors + mid) < t) lo = mid + 1; else hi = mid;
                }
                const bool anchor = lo < n_anchors && __ldg(anchors + lo) == t;
                int a = 0, b = n_seqs + 1; /* first offset > i */
                while (a < b) {
                    const int mid = (a + b) >> 1;
                    if (__ldg(seq_offsets + mid) <= i) a = mid + 1; else b = mid;
                }
                const bool seq_end = a >= 1 && a <= n_seqs && __ldg(seq_offsets + a) == i + 1; /* [.., i + 1) is non-empty: offsets[a-1] <= i */
                const bool seq_start = a >= 1 && a <= n_seqs && __ldg(seq_offsets + a - 1) == i; /* [i, offsets[a]) is non-empty */
                g = gear_of(seed, t);
                f = (uint8_t)((anchor ? F_ANCHOR : 0) | (seq_end ? F_SEQ_END : 0));
                if (k >= kSigHalo) flags[i] = f;
                if (seq_start) f |= F_SEQ_START;
            }
            s_gear[k] = g;
            s_flag[k] = f;
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < kSigSpan / kT; ++q) {
            const int w_in = warp * (kSigSpan / kT) + q;      /* level-0 word inside this span */
            const int k = kSigHalo + w_in * 32 + lane;
            const int64_t i = base + k;
            bool hard = false, cand = false;
            if (i < n) {
                uint64_t h = s_gear[k];
                for (int j = 1; j < 64; ++j) {
                    if (s_flag[k - j] & F_RESET) break; /* the signature was reset after that token (anchor, end of a sequence, or i - j < 0) */
                    h += s_gear[k - j] << j;
                }
                hard = (s_flag[k] & F_RESET) != 0;
                cand = mask_bits == 0 || (h >> (64 - mask_bits)) == 0;
                /* chain seed: a sequence starts here, or the token in front is a hard stop the chains can reach */
                mark[i] = ((s_flag[k] & F_SEQ_START) || (i >= 1 && i - 1 >= first && (s_flag[k - 1] & F_RESET))) ? 1 : 0;
            }
            const unsigned hb = __ballot_sync(0xFFFFFFFFu, hard), cb = __ballot_sync(0xFFFFFFFFu, cand);
            if (lane == 0) {
                hard0[v * 32 + w_in] = hb;
                cand0[v * 32 + w_in] = cb;
                s_nonzero[0][w_in] = hb != 0;
                s_nonzero[1][w_in] = cb != 0;
            }
        }
        __syncthreads();
        if (warp == 0) {
            const unsigned h1 = __ballot_sync(0xFFFFFFFFu, s_nonzero[0][lane] != 0), c1 = __ballot_sync(0xFFFFFFFFu, s_nonzero[1][lane] != 0);
            if (lane == 0) { hard1[v] = h1; cand1[v] = c1; }
        }
        __syncthreads();
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
    pdl_enter();
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
 * After rounds 0 .. k-1 exactly the starts less than 2^k chunks behind a seed are marked.  progress_prev == 0: round
 * k-1 set no new mark, so the start 2^(k-1) chunks behind every seed was already marked, i.e. lies within 2^(k-1) chunks
 * of a LATER seed: no start is 2^(k-1) or more chunks behind its nearest seed, every chain is complete and this round
 * (and every later one) has nothing to do. */
__global__ void __launch_bounds__(kT) k_cdc_reach(const int32_t* __restrict__ jump_in, int32_t* __restrict__ jump_out, int64_t n,
                                                  uint8_t* __restrict__ mark, const int32_t* __restrict__ progress_prev,
                                                  int32_t* __restrict__ progress) {
    pdl_enter();
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

/* Marks per block, and -- by the block that finishes last (a ticket from `done`, zeroed by k_cdc_front) -- the
 * exclusive scan of those counts and the total: n / 2048 entries (512 for a million tokens), a strip per thread. */
__global__ void __launch_bounds__(kT) k_cdc_count_scan(const uint8_t* __restrict__ mark, int64_t n, int32_t* __restrict__ block_count,
                                                       int32_t* __restrict__ done, int64_t* __restrict__ n_chunks) {
    __shared__ int s_warp[kT / 32];
    __shared__ int s_strip[kT];
    __shared__ bool s_last;
    pdl_enter();
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
        __threadfence();
        s_last = atomicAdd(done, 1) == (int)gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence(); /* the other blocks' counts, published before their tickets */
    const int n_blocks = (int)gridDim.x;
    const int per = (n_blocks + kT - 1) / kT, b0 = threadIdx.x * per, b1 = min(b0 + per, n_blocks);
    volatile int32_t* counts = block_count;
    int sum = 0;
    for (int i = b0; i < b1; ++i) sum += counts[i];
    s_strip[threadIdx.x] = sum;
    __syncthreads();
    for (int o = 1; o < kT; o <<= 1) { /* Hillis-Steele inclusive scan of the strip sums */
        const int add = threadIdx.x >= o ? s_strip[threadIdx.x - o] : 0;
        __syncthreads();
        s_strip[threadIdx.x] += add;
        __syncthreads();
    }
    int run = s_strip[threadIdx.x] - sum;
    for (int i = b0; i < b1; ++i) { const int v = counts[i]; counts[i] = run; run += v; }
    if (threadIdx.x == kT - 1) *n_chunks = s_strip[kT - 1];
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

/* chunk c = the c-th marked start in position order: end, kind and content hash (D4).  FNV-1a is a serial recurrence
 * (x = (x ^ byte) * prime), so the floor of this kernel is the LONGEST chunk: 4 dependent 64-bit multiplies per token, at
 * most 4 * max_size in a row, by the thread that owns the chunk's start. */
__global__ void __launch_bounds__(kT) k_cdc_emit(const int32_t* __restrict__ tokens, const uint8_t* __restrict__ mark,
                                                 const int32_t* __restrict__ nxt, const uint8_t* __restrict__ kind, int64_t n,
                                                 const int32_t* __restrict__ block_offset, int64_t capacity,
                                                 int64_t* __restrict__ chunk_end, int32_t* __restrict__ chunk_kind,
                                                 uint64_t* __restrict__ chunk_hash) {
    __shared__ int s_warp[kT / 32];
    pdl_enter();
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
                const int64_t e = nxt[s];
                chunk_end[before] = e;
                if (chunk_kind) chunk_kind[before] = kind[s];
                if (chunk_hash) chunk_hash[before] = fnv1a_tokens(tokens, s, e);
            }
            ++before;
        }
    }
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

/* cudaLaunchKernelEx with the programmatic-stream-serialisation attribute: the kernel may be scheduled while its
 * predecessor on the stream still runs; its pdl_enter() waits for that predecessor to complete before touching memory. */
template <class... KArgs, class... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), unsigned grid, unsigned block, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

/* Scratch of leyline_cdc_chunk comes from a pool of the chunker's own, one per device.  Not the default pool (it hands
 * its memory back to the driver at every synchronisation: measured 515 -> 124 us per synchronised call), and not the
 * plan-table pool either: that one forbids internal dependencies so that leyline_plan_prefetch's copy stream never
 * waits on a user stream, which also means a block freed by a discovery call on a user stream cannot be handed to a
 * prefetch (or back) -- concurrent discovery and planning kept GROWING it, the 10-40 ms stall its reserve exists to
 * avoid.  This pool caches up to kCdcPoolKeepBytes between calls (1 M tokens need 16 MB) and trims the rest at the next
 * synchronisation, so it is bounded. */
constexpr unsigned long long kCdcPoolKeepBytes = 64ull << 20;
constexpr int kCdcMaxDevices = 64;
std::mutex g_cdc_pool_mutex;
cudaMemPool_t g_cdc_pool[kCdcMaxDevices] = {};

cudaMemPool_t cdc_pool_on_current_device() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kCdcMaxDevices) { (void)cudaGetLastError(); return nullptr; }
    std::lock_guard<std::mutex> lock(g_cdc_pool_mutex);
    if (!g_cdc_pool[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
        unsigned long long keep = kCdcPoolKeepBytes;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        (void)cudaGetLastError();
        g_cdc_pool[dev] = pool;
    }
    return g_cdc_pool[dev];
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
    /* scratch: jumpA i32[n+1] | jumpB i32[n+1] | nxt i32[n+1] | blocks i32 | bitmaps (two levels x two predicates) |
     * progress i32[rounds] + the compaction's ticket | flags, kind, mark.  Every byte that is read is written by a kernel
     * of this call first (k_cdc_front zeroes the counters), so there is no memset. */
    auto up = [](int64_t x) { return (x + 255) / 256 * 256; };
    const int64_t n_blocks = (n + kBlockSpan - 1) / kBlockSpan;
    const int64_t n_super = (n + kSigSpan - 1) / kSigSpan, n_words_padded = n_super * 32;
    /* Doubling rounds: seeds sit behind every hard stop, and between two seeds every chunk but the last holds >= min_size
     * tokens, so no start is more than (n - 1) / min_size + 1 chunks behind its seed; rounds 0 .. R-1 reach 2^R - 1. */
    int rounds = 0;
    for (int64_t reach = 1, far = (n - 1) / p->min_size + 1; reach <= far; reach <<= 1) ++rounds;
    const int n_counters = rounds + 1; /* progress[0 .. rounds), then the compaction's ticket */
    const int64_t o_ja = 0, o_jb = o_ja + up((n + 1) * 4), o_nxt = o_jb + up((n + 1) * 4), o_blk = o_nxt + up((n + 1) * 4),
                  o_h0 = o_blk + up(n_blocks * 4), o_c0 = o_h0 + up(n_words_padded * 4), o_h1 = o_c0 + up(n_words_padded * 4),
                  o_c1 = o_h1 + up((n_super + 1) * 4), o_prog = o_c1 + up((n_super + 1) * 4), o_flags = o_prog + up(n_counters * 4),
                  o_kind = o_flags + up(n + 1), o_mark = o_kind + up(n + 1), total = o_mark + up(n + 1);
    uint8_t* ws = nullptr;
    /* from the chunker's own pool (cdc_pool_on_current_device above); the default pool only if that cannot be created */
    if (cudaMemPool_t pool = cdc_pool_on_current_device())
        CU(cudaMallocFromPoolAsync(reinterpret_cast<void**>(&ws), (size_t)total, pool, stream));
    else
        CU(cudaMallocAsync(reinterpret_cast<void**>(&ws), (size_t)total, stream));
    int32_t* ja = reinterpret_cast<int32_t*>(ws + o_ja);
    int32_t* jb = reinterpret_cast<int32_t*>(ws + o_jb);
    int32_t* nxt = reinterpret_cast<int32_t*>(ws + o_nxt);
    int32_t* blk = reinterpret_cast<int32_t*>(ws + o_blk);
    uint32_t *hard0 = reinterpret_cast<uint32_t*>(ws + o_h0), *cand0 = reinterpret_cast<uint32_t*>(ws + o_c0),
             *hard1 = reinterpret_cast<uint32_t*>(ws + o_h1), *cand1 = reinterpret_cast<uint32_t*>(ws + o_c1);
    int32_t* progress = reinterpret_cast<int32_t*>(ws + o_prog);
    uint8_t *flags = ws + o_flags, *kind = ws + o_kind, *mark = ws + o_mark;
    leyline_status st = LEYLINE_OK;
    bool launched = true;
    auto go = [&](cudaError_t e) { launched = launched && ok(e); };
    go(launch_pdl(k_cdc_front, grid_for(n_super, 1), kT, stream, dev_tokens, n, dev_anchor_ids, (int)n_anchor_ids, p->seed,
                  dev_seq_offsets, (int)n_seqs, (int)p->mask_bits, n_super, flags, mark, hard0, cand0, hard1, cand1, progress, n_counters));
    go(launch_pdl(k_cdc_next, grid_for(n + 1), kT, stream, (const uint8_t*)flags, (const uint32_t*)hard0, (const uint32_t*)hard1,
                  (const uint32_t*)cand0, (const uint32_t*)cand1, n, (int)p->min_size, (int)p->max_size, nxt, kind));
    const int32_t* jin = nxt;
    int32_t* jout = ja;
    for (int r = 0; r < rounds; ++r) {
        go(launch_pdl(k_cdc_reach, grid_for(n + 1), kT, stream, jin, jout, n, mark, (const int32_t*)(r ? progress + r - 1 : nullptr),
                      progress + r));
        jin = jout;
        jout = (jout == ja) ? jb : ja;
    }
    go(launch_pdl(k_cdc_count_scan, (unsigned)n_blocks, kT, stream, (const uint8_t*)mark, n, blk, progress + rounds, dev_n_chunks));
    if (capacity > 0)
        go(launch_pdl(k_cdc_emit, (unsigned)n_blocks, kT, stream, dev_tokens, (const uint8_t*)mark, (const int32_t*)nxt,
                      (const uint8_t*)kind, n, (const int32_t*)blk, capacity, dev_chunk_end, dev_chunk_kind, dev_chunk_hash));
    if (!launched) st = LEYLINE_E_CUDA;
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

/* ===================================================================================================================
 * leyline_cdc_chunk_noalloc -- the chunker for callers that must not allocate device memory (leyline_cdc.h).
 *
 * leyline_cdc_chunk takes its ~15 B / token of working memory from a stream-ordered pool on every call.  Some hosts of
 * this library cannot do that: a serving engine that has handed the whole GPU to its own KV-cache allocator at start-up
 * and treats any later driver allocation as a bug (it can fail, and growing a pool stalls the device); a process that
 * runs under a fixed memory budget set by a scheduler; code that runs between two points where the allocator's lock may
 * not be taken.  For them the working memory below is part of the library's image: it exists from the moment the module
 * is loaded on a GPU until the process exits, on EVERY GPU that loads the library, used or not.  That is why it is kept
 * small (8 MiB) and why the entry point has a hard size limit instead of growing.
 *
 * The launch chain is the one leyline_cdc_chunk runs (same kernels, same order, same arguments); only where the scratch
 * lives differs.  It is written out again here rather than shared so that the allocating path stays as it was.
 * =================================================================================================================== */

constexpr size_t kNoAllocScratchBytes = size_t(8) << 20;
/* File-scope device array.  In HOST code this name is only a handle the runtime knows the symbol by, not a device
 * address -- passing it to a kernel would hand the kernel a host address.  Host code gets the real address once per
 * device from cudaGetSymbolAddress (noalloc_scratch_on_current_device below) and passes that. */
static __device__ __align__(256) unsigned char g_cdc_noalloc_scratch[kNoAllocScratchBytes];

namespace {

constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mutex;
uint8_t* g_noalloc_ptr[kNoAllocMaxDevices] = {};   /* device address of g_cdc_noalloc_scratch, per device ordinal */

/* Bytes of scratch the chain needs for n tokens, and where each table starts (same layout as leyline_cdc_chunk). */
struct NoAllocLayout {
    int64_t ja, jb, nxt, blk, h0, c0, h1, c1, prog, flags, kind, mark, total;
    int64_t n_blocks, n_super;
    int rounds, n_counters;
};
NoAllocLayout noalloc_layout(int64_t n, int min_size) {
    auto up = [](int64_t x) { return (x + 255) / 256 * 256; };
    NoAllocLayout L;
    L.n_blocks = (n + kBlockSpan - 1) / kBlockSpan;
    L.n_super = (n + kSigSpan - 1) / kSigSpan;
    const int64_t n_words_padded = L.n_super * 32;
    L.rounds = 0;
    for (int64_t reach = 1, far = (n - 1) / min_size + 1; reach <= far; reach <<= 1) ++L.rounds;
    L.n_counters = L.rounds + 1;
    L.ja = 0;
    L.jb = L.ja + up((n + 1) * 4);
    L.nxt = L.jb + up((n + 1) * 4);
    L.blk = L.nxt + up((n + 1) * 4);
    L.h0 = L.blk + up(L.n_blocks * 4);
    L.c0 = L.h0 + up(n_words_padded * 4);
    L.h1 = L.c0 + up(n_words_padded * 4);
    L.c1 = L.h1 + up((L.n_super + 1) * 4);
    L.prog = L.c1 + up((L.n_super + 1) * 4);
    L.flags = L.prog + up(L.n_counters * 4);
    L.kind = L.flags + up(n + 1);
    L.mark = L.kind + up(n + 1);
    L.total = L.mark + up(n + 1);
    return L;
}

/* Set-up, once per device, with that device current: ask the runtime where g_cdc_noalloc_scratch lives on it.  The
 * query makes the runtime load this library's device code on that GPU if it has not yet (that is when the 8 MiB are
 * placed), so the first call on a device should be made outside any stream capture.  Nothing is allocated here. */
leyline_status noalloc_scratch_on_current_device(uint8_t** out) {
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices) {
        g_cdc_error = "leyline_cdc_chunk_noalloc: device ordinal " + std::to_string(dev) + " is beyond the " +
                      std::to_string(kNoAllocMaxDevices) + " devices this entry point keeps an address for";
        return LEYLINE_E_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void* p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_cdc_noalloc_scratch));
        if (!p) { g_cdc_error = "cudaGetSymbolAddress returned a null address for the static scratch"; return LEYLINE_E_CUDA; }
        g_noalloc_ptr[dev] = static_cast<uint8_t*>(p);
    }
    *out = g_noalloc_ptr[dev];
    return LEYLINE_OK;
}

}  // namespace

extern "C" LEYLINE_API leyline_status leyline_cdc_chunk_noalloc(const leyline_cdc_params* p, const int32_t* dev_tokens, int64_t n,
                                                    const int64_t* dev_seq_offsets, int32_t n_seqs,
                                                    const int32_t* dev_anchor_ids, int32_t n_anchor_ids,
                                                    int64_t* dev_chunk_end, uint64_t* dev_chunk_hash,
                                                    int32_t* dev_chunk_kind, int64_t capacity, int64_t* dev_n_chunks,
                                                    void* cuda_stream) try {
    g_cdc_error.clear();
    if (!p || p->reserved_ != 0 || p->min_size < 1 || p->max_size < p->min_size || p->max_size > 4096 ||
        p->mask_bits < 0 || p->mask_bits > 32) {
        g_cdc_error = "leyline_cdc_chunk_noalloc: bad leyline_cdc_params";
        return LEYLINE_E_INVALID;
    }
    if (n < 0 || n_seqs < 0 || n_anchor_ids < 0 || capacity < 0) {
        g_cdc_error = "leyline_cdc_chunk_noalloc: negative size";
        return LEYLINE_E_INVALID;
    }
    if (n > LEYLINE_CDC_NOALLOC_MAX_TOKENS) {
        g_cdc_error = "leyline_cdc_chunk_noalloc: n_tokens = " + std::to_string(n) + " exceeds LEYLINE_CDC_NOALLOC_MAX_TOKENS = " +
                      std::to_string((long long)LEYLINE_CDC_NOALLOC_MAX_TOKENS) +
                      " (the static scratch is fixed at 8 MiB; split the batch or use leyline_cdc_chunk)";
        return LEYLINE_E_UNSUPPORTED;
    }
    if (!dev_n_chunks || !dev_seq_offsets || (n > 0 && (!dev_tokens || n_seqs < 1)) || (capacity > 0 && !dev_chunk_end) ||
        (n_anchor_ids > 0 && !dev_anchor_ids)) {
        g_cdc_error = "leyline_cdc_chunk_noalloc: NULL argument";
        return LEYLINE_E_INVALID;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (n == 0) {
        CU(cudaMemsetAsync(dev_n_chunks, 0, sizeof(int64_t), stream));
        return LEYLINE_OK;
    }
    const NoAllocLayout L = noalloc_layout(n, p->min_size);
    if (L.total > (int64_t)kNoAllocScratchBytes) { /* cannot happen for n <= the stated maximum; kept as the real guard */
        g_cdc_error = "leyline_cdc_chunk_noalloc: " + std::to_string(L.total) + " B of scratch needed, the static array holds " +
                      std::to_string(kNoAllocScratchBytes);
        return LEYLINE_E_UNSUPPORTED;
    }
    uint8_t* ws = nullptr;
    if (leyline_status st = noalloc_scratch_on_current_device(&ws)) return st;
    /* The array still holds whatever the previous call (any size, any parameters) left in it.  Nothing has to be
     * cleared by hand: every table entry the chain reads for THIS n is written by an earlier kernel of this same chain,
     * and the only values that must start at zero -- the doubling rounds' progress words and the compaction's ticket --
     * are zeroed by k_cdc_front itself. */
    int32_t* ja = reinterpret_cast<int32_t*>(ws + L.ja);
    int32_t* jb = reinterpret_cast<int32_t*>(ws + L.jb);
    int32_t* nxt = reinterpret_cast<int32_t*>(ws + L.nxt);
    int32_t* blk = reinterpret_cast<int32_t*>(ws + L.blk);
    uint32_t *hard0 = reinterpret_cast<uint32_t*>(ws + L.h0), *cand0 = reinterpret_cast<uint32_t*>(ws + L.c0),
             *hard1 = reinterpret_cast<uint32_t*>(ws + L.h1), *cand1 = reinterpret_cast<uint32_t*>(ws + L.c1);
    int32_t* progress = reinterpret_cast<int32_t*>(ws + L.prog);
    uint8_t *flags = ws + L.flags, *kind = ws + L.kind, *mark = ws + L.mark;
    bool launched = true;
    auto go = [&](cudaError_t e) { launched = launched && ok(e); };
    go(launch_pdl(k_cdc_front, grid_for(L.n_super, 1), kT, stream, dev_tokens, n, dev_anchor_ids, (int)n_anchor_ids, p->seed,
                  dev_seq_offsets, (int)n_seqs, (int)p->mask_bits, L.n_super, flags, mark, hard0, cand0, hard1, cand1, progress,
                  L.n_counters));
    go(launch_pdl(k_cdc_next, grid_for(n + 1), kT, stream, (const uint8_t*)flags, (const uint32_t*)hard0, (const uint32_t*)hard1,
                  (const uint32_t*)cand0, (const uint32_t*)cand1, n, (int)p->min_size, (int)p->max_size, nxt, kind));
    const int32_t* jin = nxt;
    int32_t* jout = ja;
    for (int r = 0; r < L.rounds; ++r) {
        go(launch_pdl(k_cdc_reach, grid_for(n + 1), kT, stream, jin, jout, n, mark,
                      (const int32_t*)(r ? progress + r - 1 : nullptr), progress + r));
        jin = jout;
        jout = (jout == ja) ? jb : ja;
    }
    go(launch_pdl(k_cdc_count_scan, (unsigned)L.n_blocks, kT, stream, (const uint8_t*)mark, n, blk, progress + L.rounds, dev_n_chunks));
    if (capacity > 0)
        go(launch_pdl(k_cdc_emit, (unsigned)L.n_blocks, kT, stream, dev_tokens, (const uint8_t*)mark, (const int32_t*)nxt,
                      (const uint8_t*)kind, n, (const int32_t*)blk, capacity, dev_chunk_end, dev_chunk_kind, dev_chunk_hash));
    if (!launched) return LEYLINE_E_CUDA;
    CU(cudaGetLastError());
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

extern "C" LEYLINE_API const char* leyline_cdc_last_error(void) { return g_cdc_error.c_str(); }

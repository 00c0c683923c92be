/*
 * kernels_bulk.cuh -- the shared-memory-staged ("bulk") mover: steps a3 + a4 of DESIGN.md with TMA 1-D bulk copies.
 *
 *   k_move_bulk   gather -> rotate -> scatter of whole rows (PAPER.md:118-127, :405(b)(c)) through a ring of
 *                 shared-memory stages: contiguous runs of rows are fetched global -> shared with
 *                 cp.async.bulk (completion on an mbarrier), the K_pe band is rotated in shared memory
 *                 (Eq. (1)), and the runs are written shared -> global with cp.async.bulk.
 *                 With HAZARD = true it is the in-place mover of rule M2: "loaded" is published as soon as the
 *                 stage's mbarrier completes, and the stores wait for the tiles whose source rows they overwrite.
 *
 * One persistent, warp-specialised CTA per SM; tickets are pulled (tile, layer group) with the group fastest.  A run is a maximal set of rows
 * of a tile that are consecutive both in the pool and in the stage (page boundaries and row padding break runs).
 */
#ifndef LEYLINE_KERNELS_BULK_CUH_
#define LEYLINE_KERNELS_BULK_CUH_

#include "device_common.cuh"

namespace leyline {

constexpr int kBulkMaxRows = 64;   /* rows per tile (two per lane of the issuing warp) */
constexpr int kBulkMaxStages = 8;

struct BulkStageInfo {
    int64_t dst_off[kBulkMaxRows]; /* byte offset of every row's destination in the layer's pool */
    int32_t n_rows;                /* 0 = no more work */
    int32_t trig;
    int32_t tile;
    int32_t layer;
    int32_t dep_lo, dep_hi;
    int32_t from_repl;             /* replacement rows: nobody waits for this tile, so "loaded" is not published */
    int32_t pad_;
};

/* ---- PTX wrappers (sm_90+ async-proxy bulk copies, mbarrier) ---- */

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        :: "r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* smem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 :: "l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int n_threads) {
    asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(n_threads) : "memory");
}

/* ------------------------------------------------------------------ a3 + a4 ---- */

/* warp 0 = producer; warps 1..cwarps = consumers (warp 1 also stores), cwarps = 4 for MLA's narrow band, 8 when the
 * band is most of the row (full-width K); HAZARD adds 4 warps that publish "loaded" and poll dependencies (rule M2),
 * round-robin over stages, and a last warp that watches the stages land in order. */
constexpr int kBulkConsumerWarps = 4;
constexpr int kBulkWideConsumerWarps = 12; /* default when the band is most of the row (measured: 8 -> 12 is +9 % on GQA) */
constexpr int kBulkMaxConsumerWarps = 12; /* more never helped (measured), and the launch bound caps the registers per thread */
constexpr int kBulkHazardWarps = 4;
constexpr int kBulkMaxThreadsWS = 32 * (1 + kBulkMaxConsumerWarps);
constexpr int kBulkMaxThreadsHazard = kBulkMaxThreadsWS + 32 * (kBulkHazardWarps + 1);

/* Work item = (tile, group of `layer_group` consecutive layers), group fastest: the producer resolves the tile's rows
 * once and issues one stage per layer of the group. */
template <int DT, int PAIRING, bool HAZARD>
__global__ void __launch_bounds__(HAZARD ? kBulkMaxThreadsHazard : kBulkMaxThreadsWS, 1)
k_move_bulk(const __grid_constant__ MoveParams p, const int n_stages, const int stage_bytes, const int row_bytes,
            const int layer_group, const int cwarps) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ BulkStageInfo s_info[kBulkMaxStages];
    __shared__ __align__(8) uint64_t s_full[kBulkMaxStages], s_empty[kBulkMaxStages], s_deps[kBulkMaxStages];
    __shared__ volatile int s_end_it;    /* iteration index of the end marker, -1 while the producer still has work */
    __shared__ volatile int s_loaded_it; /* HAZARD: stages [0, s_loaded_it) have landed (written by the watcher warp, in order) */
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int band0 = p.lat_chunks * 16;
    const int n_consumers = 32 * cwarps;
    constexpr int N = Codec<DT>::kElems;

    if (tid == 0) {
        s_end_it = -1;
        s_loaded_it = 0;
        for (int s = 0; s < n_stages; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], 1); mbar_init(&s_deps[s], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == 0) {
        /* ---------------- producer: tickets -> rows -> bulk loads, running ahead of the consumers ---------------- */
        const int n_groups = (p.n_layers + layer_group - 1) / layer_group;
        const bool padded = p.stride != row_bytes;
        auto fetch = [&]() {
            long long it = 0;
            if (lane == 0) it = (long long)atomicAdd(p.ticket, 1ull);
            return __shfl_sync(0xFFFFFFFFu, it, 0);
        };
        int it = 0; /* stages produced so far */
        long long item = fetch();
        for (;;) {
            if (item >= p.n_items) { /* end marker */
                const int stage = it % n_stages;
                mbar_wait(&s_empty[stage], (uint32_t)(((it / n_stages) & 1) ^ 1));
                if (lane == 0) { s_info[stage].n_rows = 0; s_end_it = it; __threadfence_block(); mbar_arrive(&s_full[stage]); }
                break;
            }
            const int tile_i = p.tile_begin + (int)(item / n_groups);
            const int grp = (int)(item % n_groups);
            const DevTile t = p.tiles[tile_i];
            item = fetch(); /* the next ticket's round trip overlaps this tile's table look-ups */
            const bool from_repl = (t.flags & TILE_SRC_REPL) != 0;
            int64_t s_off[kBulkMaxRows / 32], d_off[kBulkMaxRows / 32];
            int run_rows[kBulkMaxRows / 32]; /* > 0: this lane's row starts a source run of that many rows */
#pragma unroll
            for (int half = 0; half < kBulkMaxRows / 32; ++half) {
                const int r = half * 32 + lane;
                const bool valid = r < t.n_rows;
                int64_t s_slot = 0, d_slot = 0;
                if (valid) {
                    s_slot = from_repl ? t.src_pos + r : slot_of(p.tabs, t.src_tab, t.src_pos + r, p.page_shift);
                    d_slot = (t.flags & TILE_DST_IS_SRC) ? s_slot /* in-place rotation: back where it came from */
                                                         : slot_of(p.tabs, t.dst_tab, t.dst_pos + r, (t.flags & TILE_DST_TOKEN) ? 0 : p.page_shift);
                }
                s_off[half] = s_slot * p.stride;
                d_off[half] = d_slot * p.stride;
                const int64_t prev = __shfl_up_sync(0xFFFFFFFFu, s_slot, 1);
                const bool start = valid && (lane == 0 || padded || s_slot != prev + 1);
                const unsigned starts = __ballot_sync(0xFFFFFFFFu, start);
                const unsigned valids = __ballot_sync(0xFFFFFFFFu, valid);
                const unsigned later = starts & ~((2u << lane) - 1u); /* run starts after this lane */
                const int end = later ? __ffs(later) - 1 : 32 - __clz(valids);
                run_rows[half] = start ? end - lane : 0;
            }
            const int l_end = min((grp + 1) * layer_group, p.n_layers);
            for (int layer = grp * layer_group; layer < l_end; ++layer, ++it) {
                const int stage = it % n_stages;
                mbar_wait(&s_empty[stage], (uint32_t)(((it / n_stages) & 1) ^ 1)); /* its last stores have read it */
                BulkStageInfo& info = s_info[stage];
#pragma unroll
                for (int half = 0; half < kBulkMaxRows / 32; ++half)
                    if (half * 32 + lane < t.n_rows) info.dst_off[half * 32 + lane] = d_off[half];
                if (lane == 0) {
                    info.n_rows = t.n_rows; info.trig = t.trig; info.tile = tile_i; info.layer = layer;
                    info.dep_lo = t.dep_lo; info.dep_hi = t.dep_hi; info.from_repl = from_repl ? 1 : 0;
                }
                __syncwarp();
                if (lane == 0) mbar_arrive_expect_tx(&s_full[stage], (uint32_t)(t.n_rows * row_bytes));
                __syncwarp();
                const uint8_t* __restrict__ sbase = from_repl ? p.repl[layer] : p.src[layer];
                uint8_t* stage_mem = smem + (size_t)stage * stage_bytes;
#pragma unroll
                for (int half = 0; half < kBulkMaxRows / 32; ++half)
                    if (run_rows[half] > 0)
                        bulk_g2s(stage_mem + (size_t)(half * 32 + lane) * row_bytes, sbase + s_off[half],
                                 (uint32_t)(run_rows[half] * row_bytes), &s_full[stage]);
            }
        }
        return;
    }

    if (HAZARD && warp == 1 + cwarps + kBulkHazardWarps) {
        /* ---------------- watcher: waits for the stages in ring order (so its parity waits never alias) and counts
         * the landed ones for the hazard warps, ahead of the consumers ---------------- */
        for (int it = 0;; ++it) {
            const int stage = it % n_stages;
            mbar_wait(&s_full[stage], (uint32_t)((it / n_stages) & 1));
            if (s_info[stage].n_rows == 0) break;
            if (lane == 0) { __threadfence_block(); s_loaded_it = it + 1; }
        }
        return;
    }
    if (HAZARD && warp >= 1 + cwarps) {
        /* ---------------- hazard warps (rule M2), off the consumers' critical path: once a stage's rows are in shared
         * memory publish "loaded" for (tile, layer), then wait until every tile whose source rows this tile
         * overwrites has published too, and tell the storing warp through the stage's s_deps barrier.  The release
         * fence and the acquire poll cost more than a tile's time slot, so several warps take the stages in turn. - */
        for (int it = warp - (1 + cwarps);; it += kBulkHazardWarps) {
            const int stage = it % n_stages;
            /* Gate on the consumers' in-order count of landed stages, not on the mbarrier parity: this warp skips
             * iterations, and a parity wait on a phase that is more than one ahead would alias. */
            bool live = true;
            while (s_loaded_it <= it) {
                const int e = s_end_it;
                if (e >= 0 && it >= e) { live = false; break; } /* at or past the end marker */
            }
            if (!live) break;
            __threadfence_block();
            const BulkStageInfo& info = s_info[stage];
            if (info.n_rows == 0) break;
            int32_t* flags = p.flags + p.layer0 + info.layer;
            if (lane == 0 && !info.from_repl) st_release(flags + (int64_t)info.tile * p.n_layers_total, 1);
            for (int d = info.dep_lo + lane; d <= info.dep_hi; d += 32)
                while (ld_acquire(flags + (int64_t)d * p.n_layers_total) == 0) __nanosleep(32);
            __syncwarp();
            if (lane == 0) mbar_arrive(&s_deps[stage]);
        }
        return;
    }

    /* ---------------- consumers: rotate the K_pe band in shared memory, then warp 1 stores the runs ---------------- */
    const int cwarp = warp - 1;
    const int half = p.head_chunks >> 1;  /* pair columns per head */
    const int cols = p.n_heads * half;    /* pair columns per row */
    /* unit u = (row u / cols, column u % cols), units strided by n_consumers: when cols divides n_consumers a thread
     * keeps its column, and with it its cos / sin registers */
    const bool fixed_col = n_consumers % cols == 0;
    const int my_u = cwarp * 32 + lane, my_r0 = my_u / cols, my_col = my_u - my_r0 * cols;
    const int my_q = my_col % half, my_chunk = (my_col / half) * p.head_chunks + my_q;
    const int rows_per_pass = n_consumers / cols;
    PairTrig<N, false> tr;
    int have_trig = -1;
    for (int it = 0;; ++it) {
        const int stage = it % n_stages;
        mbar_wait(&s_full[stage], (uint32_t)((it / n_stages) & 1));
        const BulkStageInfo& info = s_info[stage];
        const int n_rows = info.n_rows;
        if (n_rows == 0) break;
        uint8_t* stage_mem = smem + (size_t)stage * stage_bytes;
        if (info.trig >= 0) {
            /* a unit = (row, pair column): chunk q of a head's first half and its partner q + half, both rotated by
             * this thread (rotate_chunk_pair), so no two threads touch the same bytes */
            const int total = n_rows * cols;
            if (fixed_col) {
                /* the thread's pair column is the same for all of its units: its cos / sin stay in registers and are
                 * reloaded only when the tile belongs to another segment (the table reads through L1 were as many
                 * bytes as the band itself) */
                const float* __restrict__ trig_row = trig_row_of(p.trig, info.trig, p.H);
                if (info.trig != have_trig) {
                    load_pair_trig<PAIRING>(trig_row, p.H, my_q, half, tr);
                    have_trig = info.trig;
                }
                int4* band = reinterpret_cast<int4*>(stage_mem + (size_t)my_r0 * row_bytes + band0) + my_chunk;
                const size_t step = (size_t)rows_per_pass * row_bytes / 16;
                for (int r = my_r0; r < n_rows; r += rows_per_pass, band += step) {
                    int4 lo = band[0], hi = band[half];
                    rotate_chunk_pair<DT, PAIRING>(lo, hi, tr, trig_row, p.H, my_q, half, band, band + half);
                    band[0] = lo;
                    band[half] = hi;
                }
            } else {
                const float* __restrict__ trig_row = trig_row_of(p.trig, info.trig, p.H);
                for (int u = cwarp * 32 + lane; u < total; u += n_consumers) {
                    const int r = u / cols, col = u - r * cols;
                    const int head = col / half, q = col - head * half;
                    int4* band = reinterpret_cast<int4*>(stage_mem + (size_t)r * row_bytes + band0) + head * p.head_chunks + q;
                    int4 lo = band[0], hi = band[half];
                    PairTrig<N, false> t1;
                    load_pair_trig<PAIRING>(trig_row, p.H, q, half, t1);
                    rotate_chunk_pair<DT, PAIRING>(lo, hi, t1, trig_row, p.H, q, half, band, band + half);
                    band[0] = lo;
                    band[half] = hi;
                }
            }
            fence_proxy_async_smem(); /* generic-proxy writes -> visible to the bulk store's async-proxy reads */
        }
        named_bar_sync(1, n_consumers);
        if (cwarp == 0) {
            if (HAZARD) mbar_wait(&s_deps[stage], (uint32_t)((it / n_stages) & 1)); /* sources I overwrite are loaded */
            uint8_t* __restrict__ dbase = p.dst[info.layer];
            const bool padded = p.stride != row_bytes;
#pragma unroll
            for (int half = 0; half < kBulkMaxRows / 32; ++half) {
                const int r = half * 32 + lane;
                if (half * 32 >= n_rows) break;
                const bool valid = r < n_rows;
                const int64_t off = valid ? info.dst_off[r] : 0;
                const int64_t prev = __shfl_up_sync(0xFFFFFFFFu, off, 1);
                const bool start = valid && (lane == 0 || padded || off != prev + p.stride);
                const unsigned starts = __ballot_sync(0xFFFFFFFFu, start);
                const unsigned valids = __ballot_sync(0xFFFFFFFFu, valid);
                if (start) {
                    const unsigned later = starts & ~((2u << lane) - 1u);
                    const int end = later ? __ffs(later) - 1 : 32 - __clz(valids);
                    bulk_s2g(dbase + off, stage_mem + (size_t)r * row_bytes, (uint32_t)((end - lane) * row_bytes));
                }
            }
            bulk_commit();       /* every lane commits its own (possibly empty) group: the group counts stay in step */
            bulk_wait_read<1>(); /* the stores of the previous iteration have finished reading shared memory */
            __syncwarp();
            if (it >= 1 && lane == 0) mbar_arrive(&s_empty[(it - 1) % n_stages]);
        }
    }
    if (cwarp == 0) bulk_wait_all(); /* shared memory must outlive the bulk stores that read it */
}

}  // namespace leyline

#endif /* LEYLINE_KERNELS_BULK_CUH_ */

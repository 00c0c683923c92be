/*
 * kernels_band_tma.cuh -- step a5 (the paper's in-place path) on PAGED pools with 2-D TMA boxes.
 *
 *   k_rotate_band_tma   The band of a page -- band_bytes of each of box_rows consecutive slots, pitch = row stride:
 *                       128 B of every 1152-B row for a bf16 MLA cache -- is ONE tensor-map box.  It is fetched into a
 *                       dense shared-memory stage with cp.async.bulk.tensor (completion on the stage's mbarrier),
 *                       rotated there (Eq. (1)), and written back with a tensor store to the slots it
 *                       came from.  Only the band's bytes cross the memory system; the SM issues two TMA
 *                       instructions per 64 rows instead of 2 x 512 16-byte accesses through the LSU.
 *
 * One persistent, warp-specialised CTA per SM: warp 0 pulls (tile, layer group) tickets, resolves the tile's first slot
 * once and issues one stage per layer; warps 1..4 rotate (one 16-byte chunk per thread, NeoX partner by lane exchange,
 * so every shared-memory access is a dense 512-B wavefront), warp 1 stores.  Tiles are whole boxes aligned to the page in
 * OLD position space (the planner sizes them: rot_tile_rows = min(page, 64)); a ragged first / last tile of a
 * segment moves row by row with 1-D bulk copies of band_bytes each.  Replacement rows (a4) are byte-copied by all
 * threads after the ring has drained, as in k_rotate_band.
 */
#ifndef LEYLINE_KERNELS_BAND_TMA_CUH_
#define LEYLINE_KERNELS_BAND_TMA_CUH_

#include <cuda.h> /* CUtensorMap (type only; the encoder is fetched from the driver at run time) */

#include "kernels_bulk.cuh"

namespace leyline {

constexpr int kBandMaxStages = 32;
constexpr int kBandTmaLayers = 64;   /* tensor maps per launch (8 KB of kernel parameters) */
constexpr int kBandConsumerWarps = 4;
constexpr int kBandThreads = 32 * (1 + kBandConsumerWarps);
constexpr int kBandStoresInFlight = 4; /* store groups that may still be reading shared memory before a stage is reused */

struct BandMaps { CUtensorMap m[kBandTmaLayers]; };

struct BandStageInfo {
    int64_t slot0;    /* first slot of the tile (rows are slot0 .. slot0 + n_rows) */
    int32_t n_rows;   /* 0 = no more work */
    int32_t trig;
    int32_t layer;
    int32_t full;     /* a whole box: moved by the tensor map; else row by row */
};

__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int32_t c0, int32_t c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 :: "r"(smem_u32(smem_dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, int32_t c0, int32_t c1, const void* smem_src) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];"
                 :: "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(smem_src)) : "memory");
}

template <int DT, int PAIRING>
__global__ void __launch_bounds__(kBandThreads, 1)
k_rotate_band_tma(const __grid_constant__ MoveParams p, const __grid_constant__ BandMaps maps, const int n_stages,
                  const int stage_bytes, const int box_rows, const int band_bytes, const int layer_group) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ BandStageInfo s_info[kBandMaxStages];
    __shared__ __align__(8) uint64_t s_full[kBandMaxStages], s_empty[kBandMaxStages];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t band0 = (int64_t)p.lat_chunks * 16;
    constexpr int N = Codec<DT>::kElems;

    if (tid == 0) {
        for (int s = 0; s < n_stages; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == 0) {
        /* ---------------- producer ---------------- */
        const int n_groups = (p.n_layers + layer_group - 1) / layer_group;
        auto fetch = [&]() {
            long long it = 0;
            if (lane == 0) it = (long long)atomicAdd(p.ticket, 1ull);
            return __shfl_sync(0xFFFFFFFFu, it, 0);
        };
        int it = 0;
        long long item = fetch();
        for (;;) {
            if (item >= p.n_items) { /* end marker */
                const int stage = it % n_stages;
                mbar_wait(&s_empty[stage], (uint32_t)(((it / n_stages) & 1) ^ 1));
                if (lane == 0) { s_info[stage].n_rows = 0; __threadfence_block(); mbar_arrive(&s_full[stage]); }
                break;
            }
            const int tile_i = p.tile_begin + (int)(item / n_groups);
            const int grp = (int)(item % n_groups);
            const DevTile t = p.tiles[tile_i];
            item = fetch(); /* the next ticket's round trip overlaps this tile's table look-up */
            const int64_t slot0 = slot_of(p.tabs, t.src_tab, t.src_pos, p.page_shift); /* the tile lies inside one page */
            const bool full = t.n_rows == box_rows;
            const int l_end = min((grp + 1) * layer_group, p.n_layers);
            for (int layer = grp * layer_group; layer < l_end; ++layer, ++it) {
                const int stage = it % n_stages;
                mbar_wait(&s_empty[stage], (uint32_t)(((it / n_stages) & 1) ^ 1)); /* its last store has read it */
                uint8_t* stage_mem = smem + (size_t)stage * stage_bytes;
                if (lane == 0) {
                    BandStageInfo& info = s_info[stage];
                    info.slot0 = slot0; info.n_rows = t.n_rows; info.trig = t.trig; info.layer = layer; info.full = full ? 1 : 0;
                    mbar_arrive_expect_tx(&s_full[stage], (uint32_t)(t.n_rows * band_bytes));
                    if (full) tma_load_2d(stage_mem, &maps.m[layer], 0, (int32_t)slot0, &s_full[stage]);
                }
                __syncwarp();
                if (!full) {
                    const uint8_t* __restrict__ base = p.dst[layer] + slot0 * p.stride + band0;
                    for (int r = lane; r < t.n_rows; r += 32)
                        bulk_g2s(stage_mem + (size_t)r * band_bytes, base + (int64_t)r * p.stride, (uint32_t)band_bytes, &s_full[stage]);
                }
            }
        }
    } else {
        /* ---------------- consumers: rotate in shared memory, warp 1 stores ---------------- */
        const int cwarp = warp - 1;
        const int n_consumers = 32 * kBandConsumerWarps;
        const bool lane_exchange = (p.head_chunks & (p.head_chunks - 1)) == 0 && p.head_chunks <= 32; /* partner = lane ^ half */
        const int half = p.head_chunks >> 1;
        for (int it = 0;; ++it) {
            const int stage = it % n_stages;
            mbar_wait(&s_full[stage], (uint32_t)((it / n_stages) & 1));
            const BandStageInfo info = s_info[stage];
            if (info.n_rows == 0) break;
            uint8_t* stage_mem = smem + (size_t)stage * stage_bytes;
            const float* __restrict__ trig_row = trig_row_of(p.trig, info.trig, p.H);
            if (lane_exchange) {
                /* thread <-> 16-byte chunk of the dense stage, consecutive lanes on consecutive chunks */
                const int total = info.n_rows * p.band_chunks;
                for (int c0 = cwarp * 32; c0 < total; c0 += n_consumers) {
                    const int c = c0 + lane;
                    const bool active = c < total;
                    int4* at = reinterpret_cast<int4*>(stage_mem) + c;
                    int4 v = make_int4(0, 0, 0, 0);
                    if (active) v = *at;
                    const int j = c % p.head_chunks; /* == lane % head_chunks: 32 and the stage's chunk count are multiples of it */
                    v = rotate_band_chunk<DT, PAIRING>(v, j, p.head_chunks, trig_row, p.H, active);
                    if (active) *at = v;
                }
            } else {
                /* heads that are not a power-of-two number of chunks (head_dim 96): a thread rotates chunk q and q + half */
                const int cols = p.n_heads * half;
                const int total = info.n_rows * cols;
                for (int u = cwarp * 32 + lane; u < total; u += n_consumers) {
                    const int r = u / cols, col = u - r * cols;
                    const int head = col / half, q = col - head * half;
                    int4* band = reinterpret_cast<int4*>(stage_mem + (size_t)r * band_bytes) + head * p.head_chunks + q;
                    int4 lo = band[0], hi = band[half];
                    PairTrig<N, false> tr;
                    load_pair_trig<PAIRING>(trig_row, p.H, q, half, tr);
                    rotate_chunk_pair<DT, PAIRING>(lo, hi, tr, trig_row, p.H, q, half, band, band + half);
                    band[0] = lo;
                    band[half] = hi;
                }
            }
            fence_proxy_async_smem(); /* generic-proxy writes -> visible to the async-proxy reads of the stores */
            named_bar_sync(1, n_consumers);
            if (cwarp == 0) {
                if (info.full) {
                    if (lane == 0) tma_store_2d(&maps.m[info.layer], 0, (int32_t)info.slot0, stage_mem);
                } else {
                    uint8_t* __restrict__ base = p.dst[info.layer] + info.slot0 * p.stride + band0;
                    for (int r = lane; r < info.n_rows; r += 32)
                        bulk_s2g(base + (int64_t)r * p.stride, stage_mem + (size_t)r * band_bytes, (uint32_t)band_bytes);
                }
                bulk_commit();                          /* every lane commits its own (possibly empty) group */
                bulk_wait_read<kBandStoresInFlight>();  /* the stores of iteration it - kBandStoresInFlight have read their stage */
                __syncwarp();
                if (it >= kBandStoresInFlight && lane == 0) mbar_arrive(&s_empty[(it - kBandStoresInFlight) % n_stages]);
            }
        }
        if (cwarp == 0) bulk_wait_all(); /* shared memory must outlive the bulk stores that read it */
    }

    /* a4 in the same launch: replacement rows are byte-copied into the free slots the plan consumed (disjoint from
     * every rotated row).  16-byte chunks, four loads in flight per thread. */
    const int row_chunks = p.lat_chunks + p.band_chunks;
    for (long long ci = blockIdx.x; ci < p.n_copy_items; ci += gridDim.x) {
        const DevTile t = p.tiles[p.copy_tile_begin + (int)(ci / p.n_layers)];
        const int layer = (int)(ci % p.n_layers);
        const uint8_t* __restrict__ src = p.repl[layer] + t.src_pos * p.stride;
        uint8_t* __restrict__ dst = p.dst[layer];
        const int shift = (t.flags & TILE_DST_TOKEN) ? 0 : p.page_shift;
        const int n_chunks = t.n_rows * row_chunks;
        for (int c0 = tid; c0 < n_chunks; c0 += kBandThreads * 4) {
            int4 v[4];
            uint8_t* out[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int c = c0 + k * kBandThreads;
                out[k] = nullptr;
                if (c < n_chunks) {
                    const int r = c / row_chunks, col = c - r * row_chunks;
                    v[k] = ld_stream(src + (int64_t)r * p.stride + col * 16);
                    out[k] = dst + slot_of(p.tabs, t.dst_tab, t.dst_pos + r, shift) * p.stride + col * 16;
                }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (out[k]) st_stream(out[k], v[k]);
        }
    }
}

}  // namespace leyline

#endif /* LEYLINE_KERNELS_BAND_TMA_CUH_ */

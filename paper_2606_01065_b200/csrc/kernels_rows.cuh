/*
 * kernels_rows.cuh -- the register-staged ("row") kernels: steps a2, a3, a4, a5 of DESIGN.md.
 *
 *   k_index        a2  slot-index list / page-table rewrite (PAPER.md:135, :405(c) "re-keyed"), and the cos/sin table
 *                  of the plan's shifts (fp64 on the device)
 *   k_move_rows    a3+a4  gather -> rotate -> scatter of whole rows, replacement insert as extra tiles
 *                  (PAPER.md:118-127, :405(b)(c)); with HAZARD = true it is the in-place mover of rule M2
 *   k_rotate_band  a5  in-place rotation of the K_pe band only
 *
 * k_move_rows is persistent (CTAs pull (tile, layer) items from a ticket counter, layer fastest); k_rotate_band
 * and k_index take their items round-robin.
 */
#ifndef LEYLINE_KERNELS_ROWS_CUH_
#define LEYLINE_KERNELS_ROWS_CUH_

#include "device_common.cuh"

namespace leyline {

/* ------------------------------------------------------------------ a2 ---- */

/* One launch writes both outputs: blocks [0, blocks_a) produce `a` (page-table rows), the rest `b` (token-level slot
 * list); either may be empty (total = 0). */
__device__ __forceinline__ void index_body(const IndexParams& p, long long block, long long n_blocks) {
    for (long long o = block * blockDim.x + threadIdx.x; o < p.total; o += n_blocks * blockDim.x) {
        int lo = 0, hi = p.n_runs - 1; /* last run with out_begin <= o */
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (__ldg(&p.runs[mid].out_begin) <= o) lo = mid; else hi = mid - 1;
        }
        const IdxRun r = p.runs[lo];
        const int64_t q = o - r.out_begin;
        int32_t v;
        if (r.kind == 0) v = (int32_t)slot_of(p.tabs, r.tab, r.pos0 + q, p.page_shift);
        else if (r.kind == 1) v = __ldg(p.tabs + r.tab + r.pos0 + q);
        else v = __ldg(p.tabs + r.pos0 + q);
        p.out[o] = v;
    }
}

/* blocks [0, blocks_a): page-table rows; [blocks_a, blocks_a + blocks_b): token-level slot list; the rest: the cos/sin
 * table of the plan's distinct shifts, one (shift, frequency) per thread, in fp64 (see TrigParams).  The data kernel
 * that consumes the table is launched behind this one on the same stream. */
__global__ void __launch_bounds__(kThreads) k_index(const IndexParams a, const IndexParams b, const TrigParams tp,
                                                     const int blocks_a, const int blocks_b) {
    if ((int)blockIdx.x < blocks_a) {
        index_body(a, blockIdx.x, blocks_a);
    } else if ((int)blockIdx.x < blocks_a + blocks_b) {
        index_body(b, blockIdx.x - blocks_a, blocks_b);
    } else {
        const int u = ((int)blockIdx.x - blocks_a - blocks_b) * kThreads + (int)threadIdx.x;
        if (u < tp.n_trig * tp.H) {
            const int g = u / tp.H, i = u - g * tp.H;
            double sn, cs;
            sincos((double)tp.shifts[g] * (double)tp.inv_freq[i], &sn, &cs);
            const float ch = (float)cs, sh = (float)sn; /* hi: the value rounded once to fp32; lo: what that rounding dropped */
            float* row = tp.out + (int64_t)g * kTrigParts * tp.H;
            row[i] = ch;
            row[tp.H + i] = sh;
            row[2 * tp.H + i] = (float)(cs - (double)ch);
            row[3 * tp.H + i] = (float)(sn - (double)sh);
        }
    }
}

/* ------------------------------------------------------------------ a3 + a4 ---- */

constexpr int kMaxTileRows = 32;
constexpr int kLatPerThread = 8; /* 16-byte latent chunks a thread holds: tile_rows * lat_chunks <= 8 * 256 */

/* LC / NB: latent / band chunks per row at compile time, or -1 to read them from the parameters. */
template <int DT, int PAIRING, bool HAZARD, int LC_T, int NB_T>
__global__ void __launch_bounds__(kThreads, 3) k_move_rows(const __grid_constant__ MoveParams p) {
    __shared__ int64_t s_src[kMaxTileRows], s_dst[kMaxTileRows];
    __shared__ long long s_item;
    const int tid = threadIdx.x;
    const int LC = LC_T >= 0 ? LC_T : p.lat_chunks;
    const int NB = NB_T >= 0 ? NB_T : p.band_chunks;

    for (;;) {
        if (tid == 0) s_item = (long long)atomicAdd(p.ticket, 1ull);
        __syncthreads();
        const long long item = s_item;
        if (item >= p.n_items) break;
        const int tile_i = p.tile_begin + (int)(item / p.n_layers);
        const int layer = (int)(item % p.n_layers);
        const DevTile t = p.tiles[tile_i];
        const bool from_repl = (t.flags & TILE_SRC_REPL) != 0;
        if (tid < t.n_rows) {
            s_src[tid] = (from_repl ? t.src_pos + tid : slot_of(p.tabs, t.src_tab, t.src_pos + tid, p.page_shift)) * p.stride;
            s_dst[tid] = slot_of(p.tabs, t.dst_tab, t.dst_pos + tid, (t.flags & TILE_DST_TOKEN) ? 0 : p.page_shift) * p.stride;
        }
        __syncthreads();
        const uint8_t* __restrict__ sbase = from_repl ? p.repl[layer] : p.src[layer];
        uint8_t* __restrict__ dbase = p.dst[layer];

        /* gather: every load of the tile is issued before anything is stored */
        int4 lat[kLatPerThread];
        const int n_lat = t.n_rows * LC;
#pragma unroll
        for (int k = 0; k < kLatPerThread; ++k) {
            const int c = tid + k * kThreads;
            if (c < n_lat) {
                const int r = c / LC, col = c - r * LC;
                const uint8_t* a = sbase + s_src[r] + col * 16;
                lat[k] = HAZARD ? ld_coherent(a) : ld_stream(a);
            }
        }
        const int br = tid / NB, bj = tid - br * NB;
        const bool has_band = br < t.n_rows;
        int4 band = make_int4(0, 0, 0, 0);
        if (has_band) {
            const uint8_t* a = sbase + s_src[br] + (LC + bj) * 16;
            band = HAZARD ? ld_coherent(a) : ld_stream(a);
        }

        /* rotate (tile-uniform branch: C = 0 segments, head copies and inserts are byte copies, G19) */
        if (t.trig >= 0) band = rotate_band_chunk<DT, PAIRING>(band, bj, NB, trig_row_of(p.trig, t.trig, p.H), p.H, has_band);

        if (HAZARD) {
            /* rule M2: publish "loaded", then wait for the tiles whose source rows this tile overwrites.
             * "Loaded" must mean the data has ARRIVED: the fence below orders the accesses, but when the pool sits in
             * pinned host memory a posted PCIe write may pass an earlier read request, so every loaded register is
             * consumed first (the xor chain cannot issue before the loads have returned). */
            uint32_t landed = (uint32_t)(band.x ^ band.y ^ band.z ^ band.w);
#pragma unroll
            for (int k = 0; k < kLatPerThread; ++k)
                if (tid + k * kThreads < n_lat) landed ^= (uint32_t)(lat[k].x ^ lat[k].y ^ lat[k].z ^ lat[k].w);
            asm volatile("" :: "r"(landed) : "memory");
            if (!from_repl) __threadfence(); /* nobody waits for a replacement tile: it publishes nothing */
            __syncthreads();
            int32_t* flags = p.flags + p.layer0 + layer;
            if (tid == 0 && !from_repl) st_release(flags + (int64_t)tile_i * p.n_layers_total, 1);
            for (int d = t.dep_lo + tid; d <= t.dep_hi; d += kThreads)
                while (ld_acquire(flags + (int64_t)d * p.n_layers_total) == 0) __nanosleep(64);
            __syncthreads();
        }

        /* scatter */
#pragma unroll
        for (int k = 0; k < kLatPerThread; ++k) {
            const int c = tid + k * kThreads;
            if (c < n_lat) {
                const int r = c / LC, col = c - r * LC;
                st_stream(dbase + s_dst[r] + col * 16, lat[k]);
            }
        }
        if (has_band) st_stream(dbase + s_dst[br] + (LC + bj) * 16, band);
    }
}

/* ------------------------------------------------------------------ a5 ---- */

/* In-place rotation of the band where the rows sit.  Only `band` bytes of every row move (128 B of a
 * 1152-B bf16 MLA row), so the kernel is a strided gather/scatter: what matters is many independent 16-byte
 * accesses in flight and few instructions around them.  A work unit is a (row, pair column): the 16-byte chunk q
 * of a head's first half and its partner chunk q + half, both held by ONE thread, so no lane exchange, no shared
 * memory and no barrier is needed.  One block handles one (tile, layer) item = kRotUnroll units per thread (6 on bf16,
 * 4 on fp8; two CTAs per SM either way), all loads issued before the first store; items are assigned round-robin
 * (static), no atomics.  The plain result of a unit is stored at once; the rare unit with an output that cancels is then
 * redone from its inputs (still in registers) with the compensated form and stored again (device_common.cuh).
 * FIXED: the pair columns per row divide the block size, so a thread keeps one column (cos/sin stay in registers).
 * LEYLINE_ROT_BF16_CTAS / LEYLINE_ROT_BF16_UNROLL are build-time knobs kept for measurements (3 x 4,
 * 2 x 4, 2 x 5, 2 x 6 and 2 x 8 were timed; 2 x 6 is the default). */
static_assert(rot_units_per_item(2) == kThreads * kRotUnrollBf16 && rot_units_per_item(1) == kThreads * kRotUnrollFp8,
              "the planner sizes ROTATE_ONLY tiles to <= the units a block holds");

#ifndef LEYLINE_ROT_BF16_CTAS
#define LEYLINE_ROT_BF16_CTAS 2
#endif
template <int DT, int PAIRING, bool FIXED>
__global__ void __launch_bounds__(kThreads, DT == LEYLINE_FP8_E4M3 ? 2 : LEYLINE_ROT_BF16_CTAS) k_rotate_band(const __grid_constant__ MoveParams p) {
    constexpr int N = Codec<DT>::kElems;
    constexpr int kRotUnroll = DT == LEYLINE_BF16 ? kRotUnrollBf16 : kRotUnrollFp8;
    constexpr bool HALF_LINE = DT == LEYLINE_FP8_E4M3; /* fp8 rows are 4.5 lines: a narrow band shares its line with latent */
    const int tid = threadIdx.x;
    const int half = p.head_chunks >> 1;   /* pair columns per head */
    const int cols = p.n_heads * half;     /* pair columns per row */
    const int64_t band0 = (int64_t)p.lat_chunks * 16;
    /* what a thread's unit k is does not depend on the item: row-in-tile, 16-byte chunk of the band, pair column */
    int rk[kRotUnroll], chunk[kRotUnroll], qs[kRotUnroll];
#pragma unroll
    for (int k = 0; k < kRotUnroll; ++k) {
        const int u = FIXED ? tid : tid + k * kThreads;
        const int r = u / cols, col = u - r * cols;
        const int head = col / half;
        qs[k] = col - head * half;
        chunk[k] = head * p.head_chunks + qs[k];
        rk[k] = FIXED ? r + k * (kThreads / cols) : r;
    }
    /* The rows of an item are found through tile -> page table -> slot, two dependent look-ups before the first
     * byte of data can be requested.  The loop is software-pipelined: the NEXT item's slots are resolved while the
     * current item's band loads are in flight, so that chain never leaves the memory system idle. */
    struct Item { int32_t slot[kRotUnroll]; int32_t layer, trig; };
    auto resolve = [&](long long item, Item& it) {
        const int tile_i = p.tile_begin + (int)(item / p.n_layers);
        it.layer = (int)(item % p.n_layers);
        const DevTile t = p.tiles[tile_i];
        it.trig = t.trig;
#pragma unroll
        for (int k = 0; k < kRotUnroll; ++k)
            it.slot[k] = rk[k] < t.n_rows ? (int32_t)slot_of(p.tabs, t.src_tab, t.src_pos + rk[k], p.page_shift) : -1;
    };
    long long item = blockIdx.x;
    Item cur, nxt;
    if (cols > kThreads * kRotUnroll) {
        /* a row with more pair columns than one block pass holds (e.g. 128 heads x 256: 2048 columns; the planner
         * then makes one-row items): plain strided loop over the row's units, no pipelining */
        for (; item < p.n_items; item += gridDim.x) {
            const DevTile t = p.tiles[p.tile_begin + (int)(item / p.n_layers)];
            uint8_t* __restrict__ base = p.dst[(int)(item % p.n_layers)];
            const float* __restrict__ trig_row = trig_row_of(p.trig, t.trig, p.H);
            const int total = t.n_rows * cols;
            for (int u = tid; u < total; u += kThreads) {
                const int r = u / cols, col = u - r * cols;
                const int head = col / half, q = col - head * half;
                uint8_t* a = base + slot_of(p.tabs, t.src_tab, t.src_pos + r, p.page_shift) * p.stride + band0 +
                             (int64_t)(head * p.head_chunks + q) * 16;
                int4 lo = ld_coherent<HALF_LINE>(a), hi = ld_coherent<HALF_LINE>(a + half * 16);
                PairTrig<N, false> t1;
                load_pair_trig<PAIRING>(trig_row, p.H, q, half, t1);
                rotate_chunk_pair<DT, PAIRING>(lo, hi, t1, trig_row, p.H, q, half, reinterpret_cast<const int4*>(a),
                                               reinterpret_cast<const int4*>(a) + half);
                st_stream(a, lo);
                st_stream(a + half * 16, hi);
            }
        }
    }
    if (item < p.n_items) resolve(item, cur);
    while (item < p.n_items) {
        uint8_t* __restrict__ base = p.dst[cur.layer];
        int4 lo[kRotUnroll], hi[kRotUnroll];
        uint8_t* addr[kRotUnroll];
#pragma unroll
        for (int k = 0; k < kRotUnroll; ++k) {
            addr[k] = nullptr;
            if (cur.slot[k] >= 0) {
                addr[k] = base + (int64_t)cur.slot[k] * p.stride + band0 + (int64_t)chunk[k] * 16;
                lo[k] = ld_coherent<HALF_LINE>(addr[k]);
                hi[k] = ld_coherent<HALF_LINE>(addr[k] + half * 16);
            }
        }
        const long long next = item + gridDim.x;
        const bool more = next < p.n_items;
        if (more) resolve(next, nxt);
        const float* __restrict__ trig_row = trig_row_of(p.trig, cur.trig, p.H);
        PairTrig<N, false> tr;
        if (FIXED) load_pair_trig<PAIRING>(trig_row, p.H, qs[0], half, tr);
#pragma unroll
        for (int k = 0; k < kRotUnroll; ++k) {
            if (addr[k]) {
                if (!FIXED) load_pair_trig<PAIRING>(trig_row, p.H, qs[k], half, tr);
                int4 lo_out = lo[k], hi_out = hi[k];
                const bool redo = rotate_chunk_pair_plain<DT, PAIRING>(lo_out, hi_out, tr);
                st_stream(addr[k], lo_out);          /* never waits for the test */
                st_stream(addr[k] + half * 16, hi_out);
                if (redo && Comp<DT>::value) {       /* about one unit in 1000: again from its inputs, with the fix-up */
                    rotate_chunk_pair_careful<DT, PAIRING>(lo_out, hi_out, trig_row, p.H, qs[k], half, lo[k], hi[k]);
                    st_stream(addr[k], lo_out);
                    st_stream(addr[k] + half * 16, hi_out);
                }
            }
        }
        if (!more) break;
        cur = nxt;
        item = next;
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
        for (int c0 = tid; c0 < n_chunks; c0 += kThreads * 4) {
            int4 v[4];
            uint8_t* out[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int c = c0 + k * kThreads;
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

/* ------------------------------------------------------------------ a5 on short segments ---- */

/* k_rotate_band with the work cut differently (same arithmetic, same loads and stores per unit): a tile never crosses
 * a segment, so when the rotated segments are short -- the paper's own workload is hundreds of ~130-token chunks per
 * call -- a (tile, layer) item fills a third of the block's units and the memory system sees a
 * third of the requests it could have in flight.  Here the rows of all rotate tiles, in tile order, are one flat row
 * space, and an item is (pass, layer): pass b = flat rows [b * R, (b + 1) * R), R = the rows a block holds, whatever tiles
 * they fall in.  p.passes[b] names the tile of the pass's first row and that row's offset in it; a thread walks forward
 * from there over the tiles' row counts (its units are ascending in row, so the walk never restarts; a block spans a
 * handful of tiles at most).  Every unit carries its own cos/sin row, reloaded only when the tile's rotation changes.
 * Geometry: the FIXED case only (the pair columns of a row divide the block), which is every narrow band; the planner
 * picks this kernel (plan.cpp) and falls back to k_rotate_band otherwise.  Inserts ride behind as in k_rotate_band. */
template <int DT, int PAIRING>
__global__ void __launch_bounds__(kThreads, DT == LEYLINE_FP8_E4M3 ? 2 : LEYLINE_ROT_BF16_CTAS) k_rotate_band_flat(const __grid_constant__ MoveParams p) {
    constexpr int N = Codec<DT>::kElems;
    constexpr int kRotUnroll = DT == LEYLINE_BF16 ? kRotUnrollBf16 : kRotUnrollFp8;
    constexpr bool HALF_LINE = DT == LEYLINE_FP8_E4M3;
    const int tid = threadIdx.x;
    const int half = p.head_chunks >> 1;   /* pair columns per head */
    const int cols = p.n_heads * half;     /* pair columns per row; divides kThreads */
    const int64_t band0 = (int64_t)p.lat_chunks * 16;
    const int r0 = tid / cols, col = tid - r0 * cols;
    const int head = col / half, q = col - head * half;
    const int64_t chunk_off = band0 + (int64_t)(head * p.head_chunks + q) * 16;
    const int rstep = kThreads / cols;     /* rows between a thread's consecutive units */
    const int tile_end = p.tile_begin + p.n_rot_tiles;

    struct Item { int32_t slot[kRotUnroll]; int32_t trig[kRotUnroll]; int32_t layer; };
    auto resolve = [&](long long item, Item& it) {
        const long long pass = item / p.n_layers;
        it.layer = (int)(item - pass * p.n_layers);
        const RotPass rp = p.passes[pass];
        int j = p.tile_begin + rp.tile;
        int off = rp.row_off + r0;                                   /* row of unit 0, counted from tile j's first row */
        int n = j < tile_end ? p.tiles[j].n_rows : 0;
        int held = -1, t_tab = 0, t_trig = -1;                       /* the tile whose fields are in registers */
        int64_t t_pos = 0;
#pragma unroll
        for (int k = 0; k < kRotUnroll; ++k) {
            while (j < tile_end && off >= n) {
                off -= n;
                ++j;
                n = j < tile_end ? p.tiles[j].n_rows : 0;
            }
            if (j < tile_end) {
                if (held != j) {
                    const DevTile& t = p.tiles[j];
                    t_pos = t.src_pos; t_tab = t.src_tab; t_trig = t.trig;
                    held = j;
                }
                it.slot[k] = (int32_t)slot_of(p.tabs, t_tab, t_pos + off, p.page_shift);
                it.trig[k] = t_trig;
            } else {
                it.slot[k] = -1;                                     /* behind the last rotated row */
                it.trig[k] = -1;
            }
            off += rstep;
        }
    };

    long long item = blockIdx.x;
    Item cur, nxt;
    if (item < p.n_items) resolve(item, cur);
    while (item < p.n_items) {
        uint8_t* __restrict__ base = p.dst[cur.layer];
        int4 lo[kRotUnroll], hi[kRotUnroll];
        uint8_t* addr[kRotUnroll];
#pragma unroll
        for (int k = 0; k < kRotUnroll; ++k) {
            addr[k] = nullptr;
            if (cur.slot[k] >= 0) {
                addr[k] = base + (int64_t)cur.slot[k] * p.stride + chunk_off;
                lo[k] = ld_coherent<HALF_LINE>(addr[k]);
                hi[k] = ld_coherent<HALF_LINE>(addr[k] + half * 16);
            }
        }
        const long long next = item + gridDim.x;
        const bool more = next < p.n_items;
        if (more) resolve(next, nxt);                                /* the next item's look-ups run under this item's loads */
        const float* __restrict__ trig_row = nullptr;
        PairTrig<N, false> tr;
        int have = -2;
#pragma unroll
        for (int k = 0; k < kRotUnroll; ++k) {
            if (addr[k]) {
                if (cur.trig[k] != have) {                           /* a new segment: this column's cos/sin of its shift */
                    have = cur.trig[k];
                    trig_row = trig_row_of(p.trig, have, p.H);
                    load_pair_trig<PAIRING>(trig_row, p.H, q, half, tr);
                }
                int4 lo_out = lo[k], hi_out = hi[k];
                const bool redo = rotate_chunk_pair_plain<DT, PAIRING>(lo_out, hi_out, tr);
                st_stream(addr[k], lo_out);
                st_stream(addr[k] + half * 16, hi_out);
                if (redo && Comp<DT>::value) {
                    rotate_chunk_pair_careful<DT, PAIRING>(lo_out, hi_out, trig_row, p.H, q, half, lo[k], hi[k]);
                    st_stream(addr[k], lo_out);
                    st_stream(addr[k] + half * 16, hi_out);
                }
            }
        }
        if (!more) break;
        cur = nxt;
        item = next;
    }

    /* a4 in the same launch, as in k_rotate_band */
    const int row_chunks = p.lat_chunks + p.band_chunks;
    for (long long ci = blockIdx.x; ci < p.n_copy_items; ci += gridDim.x) {
        const DevTile t = p.tiles[p.copy_tile_begin + (int)(ci / p.n_layers)];
        const int layer = (int)(ci % p.n_layers);
        const uint8_t* __restrict__ src = p.repl[layer] + t.src_pos * p.stride;
        uint8_t* __restrict__ dst = p.dst[layer];
        const int shift = (t.flags & TILE_DST_TOKEN) ? 0 : p.page_shift;
        const int n_chunks = t.n_rows * row_chunks;
        for (int c0 = tid; c0 < n_chunks; c0 += kThreads * 4) {
            int4 v[4];
            uint8_t* out[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int c = c0 + k * kThreads;
                out[k] = nullptr;
                if (c < n_chunks) {
                    const int r = c / row_chunks, cc = c - r * row_chunks;
                    v[k] = ld_stream(src + (int64_t)r * p.stride + cc * 16);
                    out[k] = dst + slot_of(p.tabs, t.dst_tab, t.dst_pos + r, shift) * p.stride + cc * 16;
                }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (out[k]) st_stream(out[k], v[k]);
        }
    }
}

/* ------------------------------------------------------------------ a5 with an fp32 master band ---- */

/* Chained splices round the bf16 K_pe once per turn and the error random-walks (Table 6; the paper's
 * remedy is "periodic re-prefill of the affected slots").  The re-anchor option keeps an fp32 MASTER copy of the band
 * per slot ([pool_slots][rope_heads * rope_dim] floats per layer, caller-owned): the rotation is applied to the master
 * in fp32 (error ~2^-24 per turn instead of 2^-9) and the bf16 band is re-derived from it by one RNE, so the stored
 * K_pe never carries more than one rounding however often its slot is re-rotated.  bf16 caches, ROTATE_ONLY plans.
 * p.src[layer] carries the master pointers.  Same unit as k_rotate_band: (row, pair column), both partner chunks in one
 * thread.  Replacement rows (trailing copy items) are copied into the pool and widened into the master. */
template <int PAIRING>
__global__ void __launch_bounds__(kThreads) k_rotate_master(const __grid_constant__ MoveParams p) {
    constexpr int N = Codec<LEYLINE_BF16>::kElems; /* 8 elements per 16-byte chunk */
    const int tid = threadIdx.x;
    const int half = p.head_chunks >> 1, cols = p.n_heads * half;
    const int64_t band0 = (int64_t)p.lat_chunks * 16;
    const int64_t band_elems = (int64_t)p.band_chunks * N;
    for (long long item = blockIdx.x; item < p.n_items; item += gridDim.x) {
        const DevTile t = p.tiles[p.tile_begin + (int)(item / p.n_layers)];
        const int layer = (int)(item % p.n_layers);
        uint8_t* __restrict__ pool = p.dst[layer];
        float* __restrict__ master = reinterpret_cast<float*>(const_cast<uint8_t*>(p.src[layer]));
        const float* __restrict__ trig_row = trig_row_of(p.trig, t.trig, p.H);
        const int total = t.n_rows * cols;
        for (int u = tid; u < total; u += kThreads) {
            const int r = u / cols, col = u - r * cols;
            const int head = col / half, q = col - head * half;
            const int chunk = head * p.head_chunks + q;
            const int64_t slot = slot_of(p.tabs, t.src_tab, t.src_pos + r, p.page_shift);
            float4* mlo = reinterpret_cast<float4*>(master + slot * band_elems + (int64_t)chunk * N);
            float4* mhi = mlo + half * (N / 4);
            float a[N], b[N];
            PairTrig<N, true> tr;
#pragma unroll
            for (int k = 0; k < N / 4; ++k) {
                const float4 x = mlo[k], y = mhi[k];
                a[4 * k] = x.x; a[4 * k + 1] = x.y; a[4 * k + 2] = x.z; a[4 * k + 3] = x.w;
                b[4 * k] = y.x; b[4 * k + 1] = y.y; b[4 * k + 2] = y.z; b[4 * k + 3] = y.w;
            }
            load_pair_trig<PAIRING>(trig_row, p.H, q, half, tr);
            rotate_pair_master<PAIRING, N>(a, b, tr);
#pragma unroll
            for (int k = 0; k < N / 4; ++k) {
                mlo[k] = make_float4(a[4 * k], a[4 * k + 1], a[4 * k + 2], a[4 * k + 3]);
                mhi[k] = make_float4(b[4 * k], b[4 * k + 1], b[4 * k + 2], b[4 * k + 3]);
            }
            uint8_t* band = pool + slot * p.stride + band0 + (int64_t)chunk * 16;
            st_stream(band, Codec<LEYLINE_BF16>::pack(a));              /* one RNE from the fp32 master */
            st_stream(band + half * 16, Codec<LEYLINE_BF16>::pack(b));
        }
    }
    const int row_chunks = p.lat_chunks + p.band_chunks;
    for (long long ci = blockIdx.x; ci < p.n_copy_items; ci += gridDim.x) {
        const DevTile t = p.tiles[p.copy_tile_begin + (int)(ci / p.n_layers)];
        const int layer = (int)(ci % p.n_layers);
        const uint8_t* __restrict__ src = p.repl[layer] + t.src_pos * p.stride;
        uint8_t* __restrict__ pool = p.dst[layer];
        float* __restrict__ master = reinterpret_cast<float*>(const_cast<uint8_t*>(p.src[layer]));
        const int shift = (t.flags & TILE_DST_TOKEN) ? 0 : p.page_shift;
        const int n_chunks = t.n_rows * row_chunks;
        for (int c0 = tid; c0 < n_chunks; c0 += kThreads) {
            const int r = c0 / row_chunks, col = c0 - r * row_chunks;
            const int4 v = ld_stream(src + (int64_t)r * p.stride + col * 16);
            const int64_t slot = slot_of(p.tabs, t.dst_tab, t.dst_pos + r, shift);
            st_stream(pool + slot * p.stride + col * 16, v);
            if (col >= p.lat_chunks) { /* the replacement's K_pe is the new master, widened exactly */
                float f[N];
                Codec<LEYLINE_BF16>::unpack(v, f);
                float4* m = reinterpret_cast<float4*>(master + slot * band_elems + (int64_t)(col - p.lat_chunks) * N);
                m[0] = make_float4(f[0], f[1], f[2], f[3]);
                m[1] = make_float4(f[4], f[5], f[6], f[7]);
            }
        }
    }
}

/* ------------------------------------------------------------------ measurement aid ---- */

/* The access pattern of a5 with everything else taken away (leyline_probe_band_update): `band_chunks` 16-byte chunks at
 * byte `band0` of every `stride`-byte row of ONE contiguous buffer are read, changed (one integer add) and written back
 * in place.  No page table, no tiles, no rotation; consecutive lanes take consecutive chunks of a row (full-line
 * requests), U independent loads per thread are issued before the first store; HALF_LINE as in k_rotate_band (the host
 * picks it when the band is not a whole number of 128-byte lines).  What this reaches is what the memory system gives
 * ANY kernel on that pattern; bench.py reports it next to k_rotate_band. */
template <int U, bool HALF_LINE>
__global__ void __launch_bounds__(kThreads) k_probe_band_update(uint8_t* __restrict__ base, const long long n_rows, const long long stride,
                                                                const int band0, const int band_chunks) {
    const long long total = n_rows * band_chunks;
    const long long n_threads = (long long)gridDim.x * blockDim.x;
    for (long long u0 = blockIdx.x * (long long)blockDim.x + threadIdx.x; u0 < total; u0 += n_threads * U) {
        int4 v[U];
        uint8_t* a[U];
#pragma unroll
        for (int k = 0; k < U; ++k) {
            const long long u = u0 + k * n_threads;
            a[k] = nullptr;
            if (u < total) {
                const long long r = u / band_chunks;
                a[k] = base + r * stride + band0 + (int)(u - r * band_chunks) * 16;
                v[k] = ld_coherent<HALF_LINE>(a[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < U; ++k)
            if (a[k]) { v[k].x += 1; st_stream(a[k], v[k]); }
    }
}

}  // namespace leyline

#endif /* LEYLINE_KERNELS_ROWS_CUH_ */

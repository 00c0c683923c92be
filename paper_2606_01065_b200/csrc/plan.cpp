/*
 * plan.cpp -- leyline_plan / leyline_plan_ex: the host planner (step a1 of DESIGN.md; PAPER.md:98, :141, :405-409,
 * :421, :635).
 *
 * Pure host C++: no CUDA call, usable without a device.  Turns sorted, non-overlapping directives into
 *   - per-request segments with cumulative shift C_j ("running position shift carried over"),
 *   - the new slot / page map under rule M1 (FRESH), M2 (INPLACE_MOVE) or M3 (ROTATE_ONLY),
 *   - device work items (tiles of <= tile_rows rows, consecutive in new position) in ticket order, with the
 *     load->store dependencies that make in-place moves safe (rule M2),
 *   - the list of distinct non-zero shifts; the cos/sin table of C_j * theta_i itself is evaluated in fp64 on the
 *     DEVICE by the index kernel of the launch (k_index, splice.cu), and on the host only when
 *     leyline_plan_trig_table asks for it.
 *
 * A plan per turn is the steady state of a server, and the paper's workload is hundreds of ~130-token chunks per call
 * (PAPER.md:383, :411), so this file is written for latency: one pass per table, no per-request allocation, released
 * slots kept as runs, buffers recycled from plan to plan.  Nothing is thrown across the ABI.
 */
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>

#include "plan_internal.h"

using leyline::DevTile;
using leyline::IdxRun;
using leyline::ReleasedRun;


namespace {

std::mutex g_tuning_mu;
leyline_tuning g_tuning = {0, 0, 0, 0, 0, 0, 0, 0, 0};

inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

inline int heads_of(const leyline_cache_desc& c) { return c.rope_heads > 0 ? c.rope_heads : 1; }
inline int64_t row_elems(const leyline_cache_desc& c) { return (int64_t)c.latent_dim + (int64_t)heads_of(c) * c.rope_dim; }

/* The register-staged row kernel covers one head of 2^k <= 32 chunks (partner by lane xor); everything else (several
 * heads, head_dim 96 = 12 chunks, ...) runs on the bulk mover, whose band loop is generic. */
bool row_kernel_ok(const leyline_cache_desc& c, int E) {
    const int64_t nb = (int64_t)c.rope_dim * E / 16;
    return heads_of(c) == 1 && nb <= 32 && (nb & (nb - 1)) == 0 && (int64_t)c.latent_dim * E / 16 <= 2048;
}

leyline_status check_desc(const leyline_cache_desc* c, int* elem_bytes, int* page_shift) {
    if (!c) return LEYLINE_E_INVALID;
    if (c->n_layers < 1 || c->latent_dim < 0 || c->rope_dim < 2 || (c->rope_dim & 1)) return LEYLINE_E_INVALID;
    if (c->rope_heads < 0 || c->reserved_ != 0) return LEYLINE_E_INVALID;
    if (c->page_size < 1 || (c->page_size & (c->page_size - 1))) return LEYLINE_E_INVALID;
    if (c->dtype != LEYLINE_BF16 && c->dtype != LEYLINE_FP8_E4M3) return LEYLINE_E_INVALID;
    if (c->pairing != LEYLINE_ROPE_NEOX && c->pairing != LEYLINE_ROPE_INTERLEAVED) return LEYLINE_E_INVALID;
    if (!c->inv_freq) return LEYLINE_E_INVALID;
    if (c->layer_pairing)
        for (int l = 0; l < c->n_layers; ++l)
            if (c->layer_pairing[l] != LEYLINE_ROPE_NEOX && c->layer_pairing[l] != LEYLINE_ROPE_INTERLEAVED) return LEYLINE_E_INVALID;
    int E = c->dtype == LEYLINE_BF16 ? 2 : 1;
    int64_t row = row_elems(*c) * E;
    if (c->row_stride_bytes < row || (c->row_stride_bytes & 15)) return LEYLINE_E_INVALID;
    if (c->pool_slots < 0 || (c->pool_slots % c->page_size)) return LEYLINE_E_INVALID;
    for (int i = 0; i < c->rope_dim / 2; ++i)
        if (!std::isfinite(c->inv_freq[i])) return LEYLINE_E_INVALID;
    if (c->dtype == LEYLINE_FP8_E4M3 && c->layer_scale)
        for (int l = 0; l < c->n_layers; ++l)
            if (!(c->layer_scale[l] > 0.f) || !std::isfinite(c->layer_scale[l])) return LEYLINE_E_INVALID;
    /* what the kernels cover: 16-byte chunks; a head is an even number of chunks (a thread rotates chunk q of the
     * first half together with chunk q + half), at most 64; at most 128 heads; rows of at most 64 KB */
    int64_t lat_bytes = (int64_t)c->latent_dim * E, head_bytes = (int64_t)c->rope_dim * E;
    if ((lat_bytes & 15) || (head_bytes & 31)) return LEYLINE_E_UNSUPPORTED;
    if (head_bytes / 16 > 64 || heads_of(*c) > 128 || row > 65536) return LEYLINE_E_UNSUPPORTED;
    int sh = 0;
    while ((1 << sh) < c->page_size) ++sh;
    *elem_bytes = E;
    *page_shift = sh;
    return LEYLINE_OK;
}

leyline_status check_tuning(const leyline_tuning* t) {
    if (!t) return LEYLINE_E_INVALID;
    if (t->kernel < 0 || t->kernel > 2 || t->tile_rows < 0 || t->tile_rows > 64 || t->ctas_per_sm < 0 ||
        t->ctas_per_sm > 32 || t->stages < 0 || t->stages > 32 || t->layer_group < 0 ||
        t->layer_group > LEYLINE_MAX_LAYERS_PER_LAUNCH || t->consumer_warps < 0 || t->consumer_warps > 16 ||
        t->rotate_kernel < 0 || t->rotate_kernel > 3 || t->skip_alias_check < 0 || t->skip_alias_check > 1)
        return LEYLINE_E_INVALID;
    return LEYLINE_OK;
}

/* Rule V of DESIGN.md (same order as the paper's checks are stated: PAPER.md:98, :409, :635). */
leyline_status check_directives(int32_t n_req, const int64_t* seq_lens, int32_t n_dir, const leyline_directive* d) {
    for (int32_t i = 0; i < n_dir; ++i) {
        if (d[i].request < 0 || d[i].request >= n_req) return LEYLINE_E_RANGE;
        if (d[i].start < 0 || d[i].end < d[i].start || d[i].repl_len < 0 || d[i].repl_row < 0) return LEYLINE_E_INVALID;
        if ((d[i].semantic != LEYLINE_AMORTIZE && d[i].semantic != LEYLINE_FORGET) || d[i].reserved_ != 0) return LEYLINE_E_INVALID;
        if (d[i].end > seq_lens[d[i].request]) return LEYLINE_E_RANGE;
        if (i > 0) {
            if (d[i].request < d[i - 1].request) return LEYLINE_E_UNSORTED;
            if (d[i].request == d[i - 1].request) {
                if (d[i].start < d[i - 1].start) return LEYLINE_E_UNSORTED;
                if (d[i].start < d[i - 1].end) return LEYLINE_E_OVERLAP;
            }
        }
    }
    return LEYLINE_OK;
}

/* Which mover runs a3/a4 (and ROTATE_ONLY's inserts).  The bulk kernel moves contiguous runs of rows with TMA 1-D
 * copies, so it pays with runs: unpadded rows (padding must never be written) in pages of >= 16 rows, or rows of >= 1 KB; otherwise the
 * register-staged row kernel is used where it covers the band geometry.  tuning.kernel = 1 / 2 forces one of them. */
bool choose_bulk(const leyline_cache_desc& c, int E, const leyline_tuning& t, int mode) {
    if (!row_kernel_ok(c, E)) return true;
    if (mode == LEYLINE_ROTATE_ONLY) return false;
    if (t.kernel == 1) return false;
    if (t.kernel == 2) return true;
    /* unpadded rows; pages of >= 16 rows give multi-row runs, and even row-by-row (token-level pools) the bulk copies
     * win once a row is >= 1 KB (measured on the scattered rows of the appB workload: 4.79 -> 5.38 TB/s) */
    return c.row_stride_bytes == row_elems(c) * E && (c.page_size >= 16 || row_elems(c) * E >= 1024);
}

int choose_tile_rows(const leyline_cache_desc& c, int E, const leyline_tuning& t, bool bulk) {
    int64_t lat_chunks = (int64_t)c.latent_dim * E / 16, nb = (int64_t)c.rope_dim * E / 16;
    if (bulk) {
        /* bulk kernel: one shared-memory stage holds a tile; default ~36 KB per stage (48 KB for rows of 2 KB and
         * more, measured on the full-width K pools: fewer, larger stages amortise the per-stage hand-offs), <= 64 rows */
        int64_t row = row_elems(c) * E;
        int64_t want = t.tile_rows > 0 ? t.tile_rows : std::max<int64_t>(1, (row >= 2048 ? 49152 : 36864) / row);
        return (int)std::max<int64_t>(1, std::min<int64_t>({want, (int64_t)64, 65536 / row}));
    }
    /* the row kernel keeps a whole tile in registers: <= 8 latent + 1 band chunk per thread, 256 threads */
    int64_t cap = 32;
    if (lat_chunks > 0) cap = std::min<int64_t>(cap, 2048 / lat_chunks);
    cap = std::min<int64_t>(cap, 256 / nb);
    if (cap < 1) cap = 1;
    int64_t want = t.tile_rows > 0 ? t.tile_rows : 32;
    return (int)std::max<int64_t>(1, std::min(want, cap));
}

/* Rows per k_rotate_band work item: as many as fill the block's rot_units_per_item (row, pair column) units. */
int choose_rot_tile_rows(const leyline_cache_desc& c, int E, const leyline_tuning& t) {
    const int64_t cols = (int64_t)heads_of(c) * ((int64_t)c.rope_dim * E / 32);
    int64_t cap = std::max<int64_t>(1, leyline::rot_units_per_item(E) / cols);
    int64_t want = t.tile_rows > 0 ? t.tile_rows : cap;
    return (int)std::max<int64_t>(1, std::min(want, cap));
}

/* The large tables of a destroyed plan (tiles, page tables, segments, ...) are handed to the next plan instead of
 * going back to the allocator, which would return them to the OS and make the next plan fault every page in again
 * (measured: 130 of the 140 us of a config-3 plan). */
struct PlanBuffers {
    std::vector<DevTile> tiles;
    std::vector<int32_t> tabs, released, new_pages;
    std::vector<leyline_segment> segments;
    std::vector<IdxRun> slot_runs, page_runs;
    std::vector<ReleasedRun> released_runs;
    std::vector<int64_t> trig_shifts;
};
std::mutex g_recycle_mu;
std::vector<PlanBuffers> g_recycled;
constexpr size_t kMaxRecycled = 8;

void take_buffers(leyline_plan_s* pl) {
    std::lock_guard<std::mutex> lk(g_recycle_mu);
    if (g_recycled.empty()) return;
    PlanBuffers b = std::move(g_recycled.back());
    g_recycled.pop_back();
    pl->tiles = std::move(b.tiles);                 pl->tiles.clear();
    pl->tabs = std::move(b.tabs);                   pl->tabs.clear();
    pl->released = std::move(b.released);           pl->released.clear();
    pl->new_pages = std::move(b.new_pages);         pl->new_pages.clear();
    pl->segments = std::move(b.segments);           pl->segments.clear();
    pl->slot_runs = std::move(b.slot_runs);         pl->slot_runs.clear();
    pl->page_runs = std::move(b.page_runs);         pl->page_runs.clear();
    pl->released_runs = std::move(b.released_runs); pl->released_runs.clear();
    pl->trig_shifts = std::move(b.trig_shifts);     pl->trig_shifts.clear();
}

void give_buffers(leyline_plan_s* pl) {
    PlanBuffers b;
    b.tiles = std::move(pl->tiles);
    b.tabs = std::move(pl->tabs);
    b.released = std::move(pl->released);
    b.new_pages = std::move(pl->new_pages);
    b.segments = std::move(pl->segments);
    b.slot_runs = std::move(pl->slot_runs);
    b.page_runs = std::move(pl->page_runs);
    b.released_runs = std::move(pl->released_runs);
    b.trig_shifts = std::move(pl->trig_shifts);
    std::lock_guard<std::mutex> lk(g_recycle_mu);
    if (g_recycled.size() < kMaxRecycled) g_recycled.push_back(std::move(b));
}

/* a plan abandoned half-built (error or exception): its buffers are still worth keeping */
struct PlanGuard {
    leyline_plan_s* p;
    ~PlanGuard() {
        if (!p) return;
        try { give_buffers(p); } catch (...) {}
        delete p;
    }
    leyline_plan_s* release() { leyline_plan_s* q = p; p = nullptr; return q; }
};

/* Tiles of [dst0, dst0+len): boundaries are multiples of tile_rows in `align0` space.  `proto` carries everything but
 * (src_pos, dst_pos, n_rows).  ascending = ticket order of left-shifters and of every non-hazard mode; descending =
 * ticket order of right-shifters (rule M2).  The count is known up front, so the vector grows once per segment. */
inline void emit_tiles(std::vector<DevTile>& v, int64_t src0, int64_t dst0, int64_t len, int64_t align0, int tile_rows,
                       DevTile proto, bool descending = false) {
    if (len <= 0) return;
    const int64_t n0 = std::min<int64_t>(len, tile_rows - (align0 % tile_rows));
    const int64_t rest = len - n0, n_full = rest / tile_rows, tail = rest - n_full * tile_rows;
    const size_t count = (size_t)(1 + n_full + (tail ? 1 : 0)), at = v.size();
    v.resize(at + count, proto);
    DevTile* t = v.data() + at;
    if (!descending) {
        t->src_pos = src0; t->dst_pos = dst0; t->n_rows = (int32_t)n0; ++t;
        int64_t off = n0;
        for (int64_t i = 0; i < n_full; ++i, ++t, off += tile_rows) { t->src_pos = src0 + off; t->dst_pos = dst0 + off; t->n_rows = tile_rows; }
        if (tail) { t->src_pos = src0 + off; t->dst_pos = dst0 + off; t->n_rows = (int32_t)tail; }
    } else {
        int64_t off = n0 + n_full * tile_rows;
        if (tail) { t->src_pos = src0 + off; t->dst_pos = dst0 + off; t->n_rows = (int32_t)tail; ++t; }
        for (int64_t i = 0; i < n_full; ++i, ++t) { off -= tile_rows; t->src_pos = src0 + off; t->dst_pos = dst0 + off; t->n_rows = tile_rows; }
        t->src_pos = src0; t->dst_pos = dst0; t->n_rows = (int32_t)n0;
    }
}

/* distinct non-zero shifts -> row of the cos/sin table; open addressing, sized for the segments of the call */
struct ShiftIndex {
    std::vector<int64_t> key;
    std::vector<int32_t> val;
    size_t mask = 0;
    void reset(size_t expect) {
        size_t cap = 16;
        while (cap < 2 * expect + 2) cap <<= 1;
        key.assign(cap, 0);
        val.assign(cap, -1);
        mask = cap - 1;
    }
    int32_t lookup_or_add(int64_t C, std::vector<int64_t>& shifts) {
        size_t h = (size_t)((uint64_t)C * 0x9E3779B97F4A7C15ull >> 17) & mask;
        for (;; h = (h + 1) & mask) {
            if (val[h] < 0) {
                key[h] = C;
                val[h] = (int32_t)shifts.size();
                shifts.push_back(C);
                return val[h];
            }
            if (key[h] == C) return val[h];
        }
    }
};

/* per-thread scratch that keeps its capacity from plan to plan (same reason as PlanBuffers) */
struct Scratch {
    std::vector<uint64_t> seen;           /* alias checks: two bits per pool page (see the alias pass) */
    std::vector<uint64_t> slot_seen;      /* ROTATE_ONLY: a bit per pool slot, consumed free slots */
    std::vector<int32_t> dir_begin, old_tab_off, token_lists, dist, slot_ids;
    std::vector<int64_t> first_edit;
    std::vector<DevTile> insert_tiles;
    ShiftIndex shifts;
};
thread_local Scratch tl_scratch;

leyline_status plan_impl(const leyline_cache_desc* desc, int32_t mode, int32_t n_requests, const int64_t* seq_lens,
                         const int64_t* pt_offsets, const int32_t* pages, int32_t n_directives,
                         const leyline_directive* directives, const int32_t* free_ids, int64_t n_free,
                         const leyline_tuning& tuning, leyline_plan_t** out) {
    int E = 2, pshift = 0;
    leyline_status st = check_desc(desc, &E, &pshift);
    if (st != LEYLINE_OK) return st;
    if (mode != LEYLINE_FRESH && mode != LEYLINE_INPLACE_MOVE && mode != LEYLINE_ROTATE_ONLY) return LEYLINE_E_INVALID;
    if (n_requests < 0 || n_directives < 0 || n_free < 0) return LEYLINE_E_INVALID;
    if (n_requests > 0 && (!seq_lens || !pt_offsets)) return LEYLINE_E_INVALID;
    if (n_directives > 0 && !directives) return LEYLINE_E_INVALID;
    if (n_free > 0 && !free_ids) return LEYLINE_E_INVALID;
    const int64_t P = desc->page_size;
    const int64_t pool_pages = desc->pool_slots / P;
    Scratch& S = tl_scratch;

    /* page tables: every row exactly ceil(L/P) entries, every id inside the pool (one vectorisable pass per row) */
    int64_t total_old_pages = 0;
    bool contiguous = n_requests > 0 && pt_offsets[0] == 0;
    for (int32_t r = 0; r < n_requests; ++r) {
        if (seq_lens[r] < 0 || pt_offsets[r] < 0 || pt_offsets[r + 1] < pt_offsets[r]) return LEYLINE_E_INVALID;
        const int64_t need = ceil_div(seq_lens[r], P);
        if (pt_offsets[r + 1] - pt_offsets[r] != need) return LEYLINE_E_INVALID;
        if (need > 0 && !pages) return LEYLINE_E_INVALID;
        contiguous = contiguous && pt_offsets[r] == total_old_pages;
        total_old_pages += need;
        if (total_old_pages > INT32_MAX / 2) return LEYLINE_E_UNSUPPORTED;
    }
    {
        const uint32_t lim = (uint32_t)std::min<int64_t>(pool_pages, (int64_t)INT32_MAX + 1);
        for (int32_t r = 0; r < n_requests; ++r) {
            const int32_t* row = pages + pt_offsets[r];
            const int64_t need = pt_offsets[r + 1] - pt_offsets[r];
            uint32_t bad = 0;
            for (int64_t p = 0; p < need; ++p) bad |= (uint32_t)((uint32_t)row[p] >= lim);
            if (bad) return LEYLINE_E_RANGE;
        }
    }
    const int64_t free_limit = mode == LEYLINE_ROTATE_ONLY ? desc->pool_slots : pool_pages;
    st = check_directives(n_requests, seq_lens, n_directives, directives);
    if (st != LEYLINE_OK) return st;
    if (tuning.kernel == 1 && !row_kernel_ok(*desc, E)) return LEYLINE_E_UNSUPPORTED; /* forced row kernel on a band it does not cover */

    PlanGuard guard{new leyline_plan_s()};
    leyline_plan_s* pl = guard.p;
    take_buffers(pl);
    pl->desc = *desc;
    const int H = desc->rope_dim / 2;
    pl->inv_freq.assign(desc->inv_freq, desc->inv_freq + H);
    pl->desc.inv_freq = pl->inv_freq.data();
    if (desc->layer_scale) pl->layer_scale.assign(desc->layer_scale, desc->layer_scale + desc->n_layers);
    pl->desc.layer_scale = pl->layer_scale.empty() ? nullptr : pl->layer_scale.data();
    if (desc->layer_pairing) pl->layer_pairing.assign(desc->layer_pairing, desc->layer_pairing + desc->n_layers);
    pl->desc.layer_pairing = pl->layer_pairing.empty() ? nullptr : pl->layer_pairing.data();
    pl->mode = mode;
    pl->n_requests = n_requests;
    pl->elem_bytes = E;
    pl->page_shift = pshift;
    pl->tuning = tuning;
    pl->desc.rope_heads = heads_of(*desc);
    pl->n_heads = heads_of(*desc);
    pl->head_chunks = desc->rope_dim * E / 16;
    pl->use_bulk = choose_bulk(*desc, E, tuning, mode);
    pl->tile_rows = choose_tile_rows(*desc, E, tuning, pl->use_bulk);
    pl->rot_tile_rows = mode == LEYLINE_ROTATE_ONLY ? choose_rot_tile_rows(*desc, E, tuning) : 0;
    const bool unpadded = desc->row_stride_bytes == row_elems(*desc) * E;
    /* ROTATE_ONLY on a full-width K pool rewrites most of every row anyway: whole rows then
     * stream through the bulk mover and come back to the slots they were read from (measured: GQA 6.42 -> 6.7 TB/s,
     * head_dim 96 5.86 -> 6.5), instead of the strided band kernel that MLA's 1/9 band needs */
    pl->rotate_with_bulk = mode == LEYLINE_ROTATE_ONLY && tuning.kernel != 1 &&
                           2 * (int64_t)heads_of(*desc) * desc->rope_dim >= row_elems(*desc) && unpadded;
    if (pl->rotate_with_bulk) {
        pl->use_bulk = true;
        pl->tile_rows = choose_tile_rows(*desc, E, tuning, true);
        pl->rot_tile_rows = pl->tile_rows;
    }
    /* ROTATE_ONLY on a narrow band in pages of >= 16 rows: the band of a page is one 2-D box (band bytes x rows, pitch =
     * row stride) that TMA loads into and stores from shared memory (k_rotate_band_tma); tiles are then whole boxes,
     * aligned to the page in OLD position space.  tuning.rotate_kernel: 0 auto, 1 strided register kernel, 2 TMA boxes. */
    {
        const int64_t band_bytes = (int64_t)heads_of(*desc) * desc->rope_dim * E;
        const bool tma_ok = mode == LEYLINE_ROTATE_ONLY && !pl->rotate_with_bulk && P >= 16 && band_bytes <= 256 &&
                            tuning.tile_rows == 0;
        pl->rotate_with_tma = tma_ok && (tuning.rotate_kernel == 2 || (tuning.rotate_kernel == 0 && leyline::kRotateTmaByDefault));
        if (pl->rotate_with_tma) pl->rot_tile_rows = (int32_t)std::min<int64_t>(P, leyline::kRotTmaBoxRows);
    }
    const int TR = pl->tile_rows;
    const int TR_ROT = pl->rot_tile_rows;

    /* directives of request r: [dir_begin[r], dir_begin[r+1]) */
    S.dir_begin.assign((size_t)n_requests + 1, 0);
    for (int32_t i = 0; i < n_directives; ++i) ++S.dir_begin[(size_t)directives[i].request + 1];
    for (int32_t r = 0; r < n_requests; ++r) S.dir_begin[(size_t)r + 1] += S.dir_begin[(size_t)r];

    /* tabs: old page tables first, one row per request */
    S.old_tab_off.resize((size_t)n_requests + 1);
    if (contiguous) {
        pl->tabs.assign(pages, pages + total_old_pages);
        for (int32_t r = 0; r <= n_requests; ++r) S.old_tab_off[(size_t)r] = (int32_t)(r < n_requests ? pt_offsets[r] : total_old_pages);
    } else {
        pl->tabs.reserve((size_t)total_old_pages);
        for (int32_t r = 0; r < n_requests; ++r) {
            S.old_tab_off[(size_t)r] = (int32_t)pl->tabs.size();
            pl->tabs.insert(pl->tabs.end(), pages + pt_offsets[r], pages + pt_offsets[r + 1]);
        }
        S.old_tab_off[(size_t)n_requests] = (int32_t)pl->tabs.size();
    }

    /* Alias rule (after rule V; first failure wins): the kernels write rows in place (INPLACE_MOVE, ROTATE_ONLY) or
     * into consumed free pages (FRESH, growth), so
     *   - a page listed twice, where one of its owners has directives, is refused for the in-place modes (FRESH never
     *     writes a request's own pages, so shared prefix pages are fine there);
     *   - a consumed free id that is a live page (or a slot of one), or that was already consumed, is refused. */
    /* Two bits per pool page, as two bitmaps cleared per plan (17 KB each for a 137 K-slot token-level pool: they stay
     * in L1, where one byte per page did not): `seen` = listed by some request or consumed
     * from the free list, `edited` = listed by a request that has directives.  The pass touches every live page, i.e.
     * every TOKEN of a token-level pool. */
    const bool inplace_mode = mode != LEYLINE_FRESH;
    const bool check_alias = tuning.skip_alias_check == 0;
    const size_t bm_words = check_alias ? ((size_t)pool_pages + 63) / 64 : 0;
    S.seen.assign(2 * bm_words, 0); /* word pairs: [2w] = seen, [2w + 1] = edited, so that a page touches one cache line */
    uint64_t* const seen = S.seen.data();
    bool alias = false;
    for (int32_t r = 0; r < n_requests && check_alias; ++r) {
        const int32_t* row = pl->tabs.data() + S.old_tab_off[(size_t)r];
        const int64_t need = S.old_tab_off[(size_t)r + 1] - S.old_tab_off[(size_t)r];
        if (!inplace_mode) {
            for (int64_t p = 0; p < need; ++p) seen[((uint32_t)row[p] >> 6) * 2] |= 1ull << (row[p] & 63);
            continue;
        }
        const bool has_dirs = S.dir_begin[(size_t)r + 1] > S.dir_begin[(size_t)r];
        const uint64_t mine = has_dirs ? ~0ull : 0ull;
        uint64_t bad = 0;
        for (int64_t p = 0; p < need; ++p) {
            uint64_t* const w = seen + ((uint32_t)row[p] >> 6) * 2;
            const uint64_t bit = 1ull << (row[p] & 63);
            bad |= (w[1] & bit) | (w[0] & bit & mine); /* listed before, and one owner is edited */
            w[0] |= bit;
            w[1] |= bit & mine;
        }
        alias = alias || bad != 0;
    }
    pl->old_seq_lens.assign(seq_lens, seq_lens + n_requests);
    pl->new_seq_lens.resize((size_t)n_requests);
    pl->forget_trim.resize((size_t)n_requests);
    pl->slot_offsets.assign((size_t)n_requests + 1, 0);
    pl->new_pt_offsets.assign((size_t)n_requests + 1, 0);
    pl->seg_begin.assign((size_t)n_requests + 1, 0);
    S.first_edit.assign((size_t)n_requests, -1);
    S.token_lists.clear();
    int64_t consumed = 0;
    bool nofree = false, badfree = false;

    /* the next `count` free PAGE ids appended to the new table (front to back): range, then alias */
    auto take_free_pages = [&](int64_t count) {
        if (count <= 0) return;
        if (consumed + count > n_free) { nofree = true; return; }
        const int32_t* ids = free_ids + consumed;
        for (int64_t q = 0; q < count; ++q) {
            if (ids[q] < 0 || ids[q] >= free_limit) { badfree = true; continue; }
            if (!check_alias) continue;
            const uint64_t bit = 1ull << (ids[q] & 63);
            alias = alias || (seen[((uint32_t)ids[q] >> 6) * 2] & bit) != 0; /* live, or consumed before */
            seen[((uint32_t)ids[q] >> 6) * 2] |= bit;
        }
        pl->new_pages.insert(pl->new_pages.end(), ids, ids + count);
        consumed += count;
    };

    /* pass 1: segments, maps, released lists; requests ascending, free ids front to back */
    int64_t n_released = 0;
    for (int32_t r = 0; r < n_requests && !nofree; ++r) {
        const leyline_directive* d = directives + S.dir_begin[(size_t)r];
        const int32_t k = S.dir_begin[(size_t)r + 1] - S.dir_begin[(size_t)r];
        const int64_t L_old = seq_lens[r];
        int64_t C = 0, pos = 0, trim = -1, L_new = -1, first_edit = -1;
        bool before_forget = true;
        for (int32_t j = 0; j < k; ++j) {
            if (d[j].start > pos) pl->segments.push_back({r, 0, pos, pos + C, d[j].start - pos, C});
            if (d[j].semantic == LEYLINE_FORGET) { /* truncate here, re-prefill is the caller's */
                trim = L_new = d[j].start + C;
                before_forget = false;
                break;
            }
            if (first_edit < 0 && (d[j].end > d[j].start || d[j].repl_len > 0)) first_edit = d[j].start;
            if (d[j].repl_len > 0) pl->segments.push_back({r, 1, d[j].repl_row, d[j].start + C, d[j].repl_len, 0});
            C += (int64_t)d[j].repl_len - (d[j].end - d[j].start); /* Delta = |R| - (e - s) */
            pos = d[j].end;
        }
        if (before_forget) {
            if (L_old > pos) pl->segments.push_back({r, 0, pos, pos + C, L_old - pos, C});
            L_new = L_old + C;
        }
        pl->seg_begin[(size_t)r + 1] = (int64_t)pl->segments.size();
        pl->new_seq_lens[(size_t)r] = L_new;
        pl->forget_trim[(size_t)r] = trim;
        pl->slot_offsets[(size_t)r + 1] = pl->slot_offsets[(size_t)r] + L_new;
        S.first_edit[(size_t)r] = first_edit;
        const int64_t n_old = ceil_div(L_old, P), n_new = ceil_div(L_new, P);
        const int32_t* old_row = pl->tabs.data() + S.old_tab_off[(size_t)r];
        if (mode == LEYLINE_FRESH) {
            /* M1: pages in front of the first directive that changes anything are kept, the rest is compacted into
             * fresh pages; a request nothing edits keeps its first ceil(L_new/P) pages (all of them unless a FORGET
             * truncated it) and consumes nothing */
            if (first_edit < 0) {
                pl->new_pages.insert(pl->new_pages.end(), old_row, old_row + n_new);
                if (n_old > n_new) pl->released.insert(pl->released.end(), old_row + n_new, old_row + n_old);
            } else {
                const int64_t k0 = first_edit / P;
                pl->new_pages.insert(pl->new_pages.end(), old_row, old_row + k0);
                take_free_pages(n_new - k0);
                if (n_old > k0) pl->released.insert(pl->released.end(), old_row + k0, old_row + n_old);
            }
        } else if (mode == LEYLINE_INPLACE_MOVE) {
            /* M2: identity on the common pages, growth appends, shrink releases the tail */
            pl->new_pages.insert(pl->new_pages.end(), old_row, old_row + std::min(n_old, n_new));
            take_free_pages(n_new - n_old);
            if (n_old > n_new) pl->released.insert(pl->released.end(), old_row + n_new, old_row + n_old);
        } else {
            /* M3: no row moves; removed positions' slots are released in order (kept as runs of old positions, expanded
             * by leyline_plan_released), inserted rows take the next free SLOT ids */
            int64_t at = 0;
            const int32_t tab = S.old_tab_off[(size_t)r];
            for (int64_t g = pl->seg_begin[(size_t)r]; g < pl->seg_begin[(size_t)r + 1]; ++g) {
                const leyline_segment& s = pl->segments[(size_t)g];
                if (s.kind == 0) {
                    if (s.src_begin > at) { pl->released_runs.push_back({tab, at, s.src_begin - at}); n_released += s.src_begin - at; }
                    at = s.src_begin + s.length;
                } else {
                    if (consumed + s.length > n_free) { nofree = true; break; }
                    const int32_t* ids = free_ids + consumed;
                    for (int64_t q = 0; q < s.length; ++q) {
                        if (ids[q] < 0 || ids[q] >= free_limit) { badfree = true; continue; }
                        const int32_t pg = ids[q] >> pshift;
                        alias = alias || (check_alias && ((seen[((uint32_t)pg >> 6) * 2] >> (pg & 63)) & 1ull)); /* a slot of a live page */
                    }
                    S.token_lists.insert(S.token_lists.end(), ids, ids + s.length);
                    consumed += s.length;
                }
            }
            if (L_old > at) { pl->released_runs.push_back({tab, at, L_old - at}); n_released += L_old - at; }
        }
        pl->new_pt_offsets[(size_t)r + 1] = (int64_t)pl->new_pages.size();
    }
    if (nofree) return LEYLINE_E_NOFREE;
    if (badfree) return LEYLINE_E_RANGE;
    if (mode == LEYLINE_ROTATE_ONLY && check_alias && !alias && S.token_lists.size() > 1) { /* the same free slot handed out twice */
        const size_t n_ids = S.token_lists.size(), words = ((size_t)desc->pool_slots + 63) / 64;
        if (words <= 64 * n_ids) {
            /* a bit per pool slot: clearing it costs less than sorting the ids (19 K inserted rows on config 4: the
             * sort was 250 of the plan's 360 us) unless the pool is huge and the ids are few */
            S.slot_seen.assign(words, 0);
            uint64_t dup = 0;
            for (size_t q = 0; q < n_ids; ++q) {
                const uint32_t id = (uint32_t)S.token_lists[q];
                const uint64_t bit = 1ull << (id & 63);
                dup |= S.slot_seen[id >> 6] & bit;
                S.slot_seen[id >> 6] |= bit;
            }
            alias = dup != 0;
        } else {
            S.slot_ids = S.token_lists;
            std::sort(S.slot_ids.begin(), S.slot_ids.end());
            alias = std::adjacent_find(S.slot_ids.begin(), S.slot_ids.end()) != S.slot_ids.end();
        }
    }
    if (alias) return LEYLINE_E_ALIAS;
    if (mode != LEYLINE_ROTATE_ONLY) n_released = (int64_t)pl->released.size();

    /* tabs: new page tables, then token-level lists */
    const int32_t new_tab_base = (int32_t)pl->tabs.size();
    if (mode != LEYLINE_ROTATE_ONLY) pl->tabs.insert(pl->tabs.end(), pl->new_pages.begin(), pl->new_pages.end());
    const int32_t token_base = (int32_t)pl->tabs.size();
    pl->tabs.insert(pl->tabs.end(), S.token_lists.begin(), S.token_lists.end());

    /* pass 2: tiles (ticket order: move tiles, then insert tiles), index runs */
    std::vector<DevTile>& tiles = pl->tiles;
    std::vector<DevTile>& inserts = S.insert_tiles;
    inserts.clear();
    S.shifts.reset(pl->segments.size());
    S.dist.clear();
    leyline_plan_info& in = pl->info;
    auto trig_index = [&](int64_t C) -> int32_t { /* G19: a zero shift is a byte copy, never arithmetic */
        return C == 0 ? -1 : S.shifts.lookup_or_add(C, pl->trig_shifts);
    };
    int64_t token_cursor = 0;
    for (int32_t r = 0; r < n_requests; ++r) {
        const int32_t src_tab = S.old_tab_off[(size_t)r];
        const int32_t dst_tab = new_tab_base + (int32_t)pl->new_pt_offsets[(size_t)r];
        const leyline_segment* segs = pl->segments.data() + pl->seg_begin[(size_t)r];
        const int64_t n_segs = pl->seg_begin[(size_t)r + 1] - pl->seg_begin[(size_t)r];
        if (mode == LEYLINE_ROTATE_ONLY) {
            const int32_t rot_flags = pl->rotate_with_bulk ? leyline::TILE_DST_IS_SRC : 0;
            for (int64_t g = 0; g < n_segs; ++g) {
                const leyline_segment& s = segs[g];
                if (s.kind == 0) {
                    pl->slot_runs.push_back({pl->slot_offsets[(size_t)r] + s.dst_begin, s.length, s.src_begin, src_tab, 0});
                    const int32_t t = trig_index(s.shift);
                    if (t < 0) continue;
                    in.rows_rotated += s.length;
                    emit_tiles(tiles, s.src_begin, s.dst_begin, s.length, s.src_begin, TR_ROT,
                               DevTile{0, 0, src_tab, src_tab, 0, t, rot_flags, 0, -1, r});
                } else {
                    const int32_t list = token_base + (int32_t)token_cursor;
                    pl->slot_runs.push_back({pl->slot_offsets[(size_t)r] + s.dst_begin, s.length, 0, list, 1});
                    in.rows_inserted += s.length;
                    emit_tiles(inserts, s.src_begin, 0, s.length, 0, TR,
                               DevTile{0, 0, -1, list, 0, -1, leyline::TILE_SRC_REPL | leyline::TILE_DST_TOKEN, 0, -1, r});
                    token_cursor += s.length;
                }
            }
            continue;
        }
        if (pl->new_seq_lens[(size_t)r] > 0)
            pl->slot_runs.push_back({pl->slot_offsets[(size_t)r], pl->new_seq_lens[(size_t)r], 0, dst_tab, 0});
        if (mode == LEYLINE_FRESH) {
            if (S.first_edit[(size_t)r] < 0) continue; /* nothing edited: the kept pages already hold every live row */
            const int64_t first = (S.first_edit[(size_t)r] / P) * P; /* new positions >= first live in fresh pages */
            for (int64_t g = 0; g < n_segs; ++g) {
                const leyline_segment& s = segs[g];
                if (s.kind == 1) {
                    in.rows_inserted += s.length;
                    emit_tiles(inserts, s.src_begin, s.dst_begin, s.length, s.dst_begin, TR,
                               DevTile{0, 0, -1, dst_tab, 0, -1, leyline::TILE_SRC_REPL, 0, -1, r});
                    continue;
                }
                const int64_t skip = std::max<int64_t>(0, first - s.dst_begin);
                if (skip >= s.length) continue;
                const int32_t t = trig_index(s.shift);
                in.rows_moved += s.length - skip;
                if (t >= 0) in.rows_rotated += s.length - skip;
                emit_tiles(tiles, s.src_begin + skip, s.dst_begin + skip, s.length - skip, s.dst_begin + skip, TR,
                           DevTile{0, 0, src_tab, dst_tab, 0, t, 0, 0, -1, r});
            }
            continue;
        }
        /* INPLACE_MOVE, rule M2.  A segment with C < 0 only lands on source rows of earlier segments / removed spans,
         * C > 0 only on later ones, and the two groups never touch each other's sources: left-shifters ascending
         * front-to-back, right-shifters descending back-to-front, C = 0 untouched. */
        const size_t first_insert = inserts.size();
        const int32_t base_l = (int32_t)tiles.size();
        for (int64_t g = 0; g < n_segs; ++g) {
            const leyline_segment& s = segs[g];
            if (s.kind == 1) {
                in.rows_inserted += s.length;
                emit_tiles(inserts, s.src_begin, s.dst_begin, s.length, s.dst_begin, TR,
                           DevTile{0, 0, -1, dst_tab, 0, -1, leyline::TILE_SRC_REPL, 0, -1, r});
                continue;
            }
            if (s.shift >= 0) continue;
            const int32_t t = trig_index(s.shift);
            in.rows_moved += s.length;
            in.rows_rotated += s.length;
            emit_tiles(tiles, s.src_begin, s.dst_begin, s.length, s.dst_begin, TR, DevTile{0, 0, src_tab, dst_tab, 0, t, 0, 0, -1, r});
        }
        const int32_t base_r = (int32_t)tiles.size();
        for (int64_t g = n_segs - 1; g >= 0; --g) {
            const leyline_segment& s = segs[g];
            if (s.kind == 1 || s.shift <= 0) continue;
            const int32_t t = trig_index(s.shift);
            in.rows_moved += s.length;
            in.rows_rotated += s.length;
            emit_tiles(tiles, s.src_begin, s.dst_begin, s.length, s.dst_begin, TR, DevTile{0, 0, src_tab, dst_tab, 0, t, 0, 0, -1, r},
                       /*descending=*/true);
        }
        const int32_t end_r = (int32_t)tiles.size();
        /* left-shifters: a tile's destination covers source rows of tiles at lower positions (earlier tickets) */
        for (int32_t i = base_l, lo = base_l; i < base_r; ++i) {
            DevTile& t = tiles[(size_t)i];
            const int64_t d0 = t.dst_pos, d1 = t.dst_pos + t.n_rows;
            while (lo < i && tiles[(size_t)lo].src_pos + tiles[(size_t)lo].n_rows <= d0) ++lo;
            int32_t hi = lo; /* first tile at or after lo whose source starts at or past d1 */
            while (hi < i && tiles[(size_t)hi].src_pos < d1) ++hi;
            t.dep_lo = lo;
            t.dep_hi = hi - 1;
            if (hi > lo && ((i - base_l) & 7) == 0) S.dist.push_back(i - (hi - 1));
        }
        /* right-shifters: destination covers source rows of tiles at higher positions (earlier tickets) */
        for (int32_t i = base_r, lo = base_r; i < end_r; ++i) {
            DevTile& t = tiles[(size_t)i];
            const int64_t d0 = t.dst_pos, d1 = t.dst_pos + t.n_rows;
            while (lo < i && tiles[(size_t)lo].src_pos >= d1) ++lo;
            int32_t hi = lo;
            while (hi < i && tiles[(size_t)hi].src_pos + tiles[(size_t)hi].n_rows > d0) ++hi;
            t.dep_lo = lo;
            t.dep_hi = hi - 1;
            if (hi > lo && ((i - base_r) & 7) == 0) S.dist.push_back(i - (hi - 1));
        }
        /* inserts run in the same launch, after every move in ticket order: a replacement row may land on a row some
         * move tile of this request still has to read, so it waits for those tiles.  Within the left-shifters sources
         * ascend with the ticket, within the right-shifters they descend, so the overlapping tiles of one group are a
         * contiguous range found by bisection; an insert that lands on sources of BOTH groups gets the hull across
         * them (a superset is safe: all of them hold smaller tickets). */
        for (size_t q = first_insert; q < inserts.size(); ++q) {
            DevTile& t = inserts[q];
            const int64_t d0 = t.dst_pos, d1 = t.dst_pos + t.n_rows;
            int32_t lo = INT32_MAX, hi = -1;
            const DevTile* T = tiles.data();
            {   /* left group: first tile with src_end > d0, last tile with src_pos < d1 */
                const DevTile* a = std::partition_point(T + base_l, T + base_r, [&](const DevTile& m) { return m.src_pos + m.n_rows <= d0; });
                const DevTile* b = std::partition_point(a, T + base_r, [&](const DevTile& m) { return m.src_pos < d1; });
                if (b > a) { lo = std::min(lo, (int32_t)(a - T)); hi = std::max(hi, (int32_t)(b - T) - 1); }
            }
            {   /* right group (sources descending): first tile with src_pos < d1, last tile with src_end > d0 */
                const DevTile* a = std::partition_point(T + base_r, T + end_r, [&](const DevTile& m) { return m.src_pos >= d1; });
                const DevTile* b = std::partition_point(a, T + end_r, [&](const DevTile& m) { return m.src_pos + m.n_rows > d0; });
                if (b > a) { lo = std::min(lo, (int32_t)(a - T)); hi = std::max(hi, (int32_t)(b - T) - 1); }
            }
            t.dep_lo = hi >= 0 ? lo : 0;
            t.dep_hi = hi;
        }
    }
    if (mode != LEYLINE_ROTATE_ONLY && !pl->new_pages.empty())
        pl->page_runs.push_back({0, (int64_t)pl->new_pages.size(), new_tab_base, 0, 2});

    in.mode = mode;
    in.n_requests = n_requests;
    in.total_new_tokens = pl->slot_offsets[(size_t)n_requests];
    in.total_new_pages = mode == LEYLINE_ROTATE_ONLY ? 0 : (int64_t)pl->new_pages.size();
    in.n_free_consumed = consumed;
    in.n_released = n_released;
    in.n_segments = (int64_t)pl->segments.size();
    in.n_move_tiles = (int64_t)tiles.size();
    in.n_tiles = (int64_t)(tiles.size() + inserts.size());
    in.n_trig = (int64_t)pl->trig_shifts.size();
    const int64_t row_bytes = row_elems(*desc) * E, band_bytes = (int64_t)heads_of(*desc) * desc->rope_dim * E;
    int64_t per_layer = (in.rows_moved + in.rows_inserted) * row_bytes;
    if (mode == LEYLINE_ROTATE_ONLY) per_layer = in.rows_rotated * band_bytes + in.rows_inserted * row_bytes;
    in.bytes_read = in.bytes_written = per_layer * desc->n_layers;
    in.bytes_index = 4 * in.total_new_tokens + 4 * in.total_new_pages;
    in.tile_rows = pl->tile_rows;
    in.rot_tile_rows = pl->rot_tile_rows;
    in.mover = pl->use_bulk ? 2 : 1; /* ROTATE_ONLY: 2 = the rotation itself runs on the bulk mover (wide bands) */
    if (mode == LEYLINE_ROTATE_ONLY && !pl->rotate_with_bulk) in.mover = pl->rotate_with_tma ? 3 : 1;
    /* a5 on short segments (the paper's own workload: hundreds of ~130-token chunks per call): a tile
     * never crosses a segment, so k_rotate_band's one-tile items would fill a fraction of a block's units.  The flat
     * kernel packs consecutive tiles into full passes instead; it is chosen when that saves a fifth of the items or more
     * (tuning.rotate_kernel: 1 = never, 3 = always). */
    if (mode == LEYLINE_ROTATE_ONLY && !pl->rotate_with_bulk && !pl->rotate_with_tma && TR_ROT > 0 && !tiles.empty()) {
        const int64_t cols = (int64_t)pl->n_heads * (pl->head_chunks / 2);
        const bool fixed = cols <= 256 && 256 % cols == 0 && leyline::rot_units_per_item(E) % cols == 0 &&
                           (int64_t)TR_ROT * cols == leyline::rot_units_per_item(E);
        const int64_t n_passes = (in.rows_rotated + TR_ROT - 1) / TR_ROT;
        const bool pays = n_passes * 5 <= (int64_t)tiles.size() * 4;
        if (fixed && tuning.rotate_kernel != 1 && (tuning.rotate_kernel == 3 || pays)) {
            pl->rotate_flat = true;
            pl->rot_passes.reserve((size_t)n_passes);
            int64_t next_start = 0, row0 = 0; /* flat row at which the next pass starts / the current tile starts */
            for (size_t j = 0; j < tiles.size(); ++j) {
                const int64_t n = tiles[j].n_rows;
                for (; next_start < row0 + n; next_start += TR_ROT)
                    pl->rot_passes.push_back({(int32_t)j, (int32_t)(next_start - row0)});
                row0 += n;
            }
            in.mover = 4;
        }
    }

    if (!S.dist.empty()) { /* how far back (in tiles) a waiting tile's dependencies sit: a launch hint (sampled) */
        std::nth_element(S.dist.begin(), S.dist.begin() + (long)(S.dist.size() / 2), S.dist.end());
        pl->dep_distance_median = S.dist[S.dist.size() / 2];
    }
    tiles.insert(tiles.end(), inserts.begin(), inserts.end());
    *out = guard.release();
    return LEYLINE_OK;
}

/* cos / sin of C_g * theta_i on the HOST (queries only; the launches use the device's own fp64 evaluation):
 * fp64 product, fp64 libm (one sincos call), rounded once to fp32 */
void host_trig_table(const leyline_plan_s* pl, float* out) {
    const size_t H = pl->inv_freq.size();
    for (size_t g = 0; g < pl->trig_shifts.size(); ++g)
        for (size_t i = 0; i < H; ++i) {
            double sn, cs;
            ::sincos((double)pl->trig_shifts[g] * (double)pl->inv_freq[i], &sn, &cs);
            out[g * 2 * H + i] = (float)cs;
            out[g * 2 * H + H + i] = (float)sn;
        }
}

}  // namespace

/* Every entry point below converts an escaping C++ exception into a status (leyline.h: "nothing is thrown across
 * the ABI"). */
#define LEYLINE_GUARDED(...)                                                     \
    try { __VA_ARGS__ } catch (const std::bad_alloc&) { return LEYLINE_E_NOMEM; } \
    catch (...) { return LEYLINE_E_INVALID; }

extern "C" LEYLINE_API leyline_status leyline_plan_ex(const leyline_cache_desc* desc, int32_t mode, int32_t n_requests,
                                                      const int64_t* seq_lens, const int64_t* pt_offsets,
                                                      const int32_t* pages, int32_t n_directives,
                                                      const leyline_directive* directives, const int32_t* free_ids,
                                                      int64_t n_free, const leyline_tuning* tuning, leyline_plan_t** out) {
    if (!out) return LEYLINE_E_INVALID;
    *out = nullptr;
    LEYLINE_GUARDED(
        leyline_tuning t = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        if (tuning) {
            if (check_tuning(tuning) != LEYLINE_OK) return LEYLINE_E_INVALID;
            t = *tuning;
        }
        return plan_impl(desc, mode, n_requests, seq_lens, pt_offsets, pages, n_directives, directives, free_ids, n_free, t, out);
    )
}

extern "C" LEYLINE_API leyline_status leyline_plan(const leyline_cache_desc* desc, int32_t mode, int32_t n_requests,
                                                   const int64_t* seq_lens, const int64_t* pt_offsets, const int32_t* pages,
                                                   int32_t n_directives, const leyline_directive* directives,
                                                   const int32_t* free_ids, int64_t n_free, leyline_plan_t** out) {
    leyline_tuning t;
    {
        std::lock_guard<std::mutex> lk(g_tuning_mu);
        t = g_tuning;
    }
    return leyline_plan_ex(desc, mode, n_requests, seq_lens, pt_offsets, pages, n_directives, directives, free_ids, n_free, &t, out);
}

/* ------------------------------------------------------------------ queries ---- */

#define LEYLINE_GETTER(name, type, member)                                                     \
    extern "C" LEYLINE_API leyline_status name(const leyline_plan_t* plan, type* out) {       \
        if (!plan || (!out && !plan->member.empty())) return LEYLINE_E_INVALID;                \
        if (!plan->member.empty()) std::memcpy(out, plan->member.data(), plan->member.size() * sizeof(type)); \
        return LEYLINE_OK;                                                                     \
    }

extern "C" LEYLINE_API leyline_status leyline_plan_get_info(const leyline_plan_t* plan, leyline_plan_info* out) {
    if (!plan || !out) return LEYLINE_E_INVALID;
    *out = plan->info;
    return LEYLINE_OK;
}
LEYLINE_GETTER(leyline_plan_new_seq_lens, int64_t, new_seq_lens)
LEYLINE_GETTER(leyline_plan_forget_trim, int64_t, forget_trim)
LEYLINE_GETTER(leyline_plan_slot_offsets, int64_t, slot_offsets)
LEYLINE_GETTER(leyline_plan_segments, leyline_segment, segments)
LEYLINE_GETTER(leyline_plan_trig_shifts, int64_t, trig_shifts)

/* Released ids.  Page modes keep the list; ROTATE_ONLY keeps runs of removed old positions and expands them here
 * (slot = page << shift | offset through the request's old page table), so planning does not pay per released slot. */
extern "C" LEYLINE_API leyline_status leyline_plan_released(const leyline_plan_t* plan, int32_t* out) {
    if (!plan || (!out && plan->info.n_released > 0)) return LEYLINE_E_INVALID;
    if (plan->mode != LEYLINE_ROTATE_ONLY) {
        if (!plan->released.empty()) std::memcpy(out, plan->released.data(), plan->released.size() * sizeof(int32_t));
        return LEYLINE_OK;
    }
    const int sh = plan->page_shift;
    const int64_t mask = ((int64_t)1 << sh) - 1;
    for (const ReleasedRun& rr : plan->released_runs) {
        const int32_t* row = plan->tabs.data() + rr.tab;
        for (int64_t t = rr.pos0; t < rr.pos0 + rr.count; ++t) *out++ = (int32_t)(((int64_t)row[t >> sh] << sh) | (t & mask));
    }
    return LEYLINE_OK;
}

extern "C" LEYLINE_API leyline_status leyline_plan_new_pt_offsets(const leyline_plan_t* plan, int64_t* out) {
    if (!plan || !out || plan->mode == LEYLINE_ROTATE_ONLY) return LEYLINE_E_INVALID;
    std::memcpy(out, plan->new_pt_offsets.data(), plan->new_pt_offsets.size() * sizeof(int64_t));
    return LEYLINE_OK;
}

extern "C" LEYLINE_API leyline_status leyline_plan_new_pages(const leyline_plan_t* plan, int32_t* out) {
    if (!plan || plan->mode == LEYLINE_ROTATE_ONLY || (!out && !plan->new_pages.empty())) return LEYLINE_E_INVALID;
    if (!plan->new_pages.empty()) std::memcpy(out, plan->new_pages.data(), plan->new_pages.size() * sizeof(int32_t));
    return LEYLINE_OK;
}

extern "C" LEYLINE_API leyline_status leyline_plan_tiles(const leyline_plan_t* plan, leyline_tile* out) {
    if (!plan || (!out && !plan->tiles.empty())) return LEYLINE_E_INVALID;
    for (size_t i = 0; i < plan->tiles.size(); ++i) {
        const DevTile& t = plan->tiles[i];
        out[i].src_pos = t.src_pos;
        out[i].dst_pos = t.dst_pos;
        out[i].n_rows = t.n_rows;
        out[i].trig = t.trig;
        out[i].flags = t.flags & LEYLINE_TILE_SRC_REPL;
        out[i].dep_lo = t.dep_lo;
        out[i].dep_hi = t.dep_hi;
        out[i].request = t.request;
    }
    return LEYLINE_OK;
}

/* cos/sin table rows, [n_trig][2][rope_dim/2] fp32, evaluated on the host (tests check them against an independent
 * fp64 evaluation; the launches evaluate the same expression in fp64 on the device) */
extern "C" LEYLINE_API leyline_status leyline_plan_trig_table(const leyline_plan_t* plan, float* out) {
    if (!plan || (!out && !plan->trig_shifts.empty())) return LEYLINE_E_INVALID;
    host_trig_table(plan, out);
    return LEYLINE_OK;
}

extern "C" LEYLINE_API void leyline_plan_destroy(leyline_plan_t* plan) {
    if (!plan) return;
    leyline::plan_release_device(plan);
    try { give_buffers(plan); } catch (...) {}
    delete plan;
}

extern "C" LEYLINE_API const char* leyline_strerror(leyline_status s) {
    switch (s) {
        case LEYLINE_OK: return "ok";
        case LEYLINE_E_INVALID: return "invalid argument";
        case LEYLINE_E_UNSORTED: return "directives not sorted by (request, start)";
        case LEYLINE_E_OVERLAP: return "overlapping spans";
        case LEYLINE_E_RANGE: return "request, span or id out of range";
        case LEYLINE_E_NOFREE: return "free list too short";
        case LEYLINE_E_UNSUPPORTED: return "cache geometry not supported by the kernels";
        case LEYLINE_E_CUDA: return "CUDA error";
        case LEYLINE_E_NOMEM: return "out of host memory";
        case LEYLINE_E_ALIAS: return "a free id is live or handed out twice, or a page is shared with a request edited in place";
    }
    return "unknown status";
}

extern "C" LEYLINE_API leyline_status leyline_set_tuning(const leyline_tuning* t) {
    if (check_tuning(t) != LEYLINE_OK) return LEYLINE_E_INVALID;
    std::lock_guard<std::mutex> lk(g_tuning_mu);
    g_tuning = *t;
    return LEYLINE_OK;
}

extern "C" LEYLINE_API leyline_status leyline_get_tuning(leyline_tuning* t) {
    if (!t) return LEYLINE_E_INVALID;
    std::lock_guard<std::mutex> lk(g_tuning_mu);
    *t = g_tuning;
    return LEYLINE_OK;
}

extern "C" LEYLINE_API const char* leyline_version(void) { return "leyline-b200 0.2 sm_100a"; }

/*
 * plan.cpp -- leyline_plan: the host planner (step a1 of DESIGN.md).
 *
 * Pure host C++: no CUDA call, usable without a device.  Turns sorted, non-overlapping directives into
 *   - per-request segments with cumulative shift C_j ("running position shift carried over"),
 *   - the new slot / page map under rule M1 (FRESH), M2 (INPLACE_MOVE) or M3 (ROTATE_ONLY),
 *   - device work items (tiles of <= tile_rows rows, consecutive in new position) in ticket order, with the
 *     load->store dependencies that make in-place moves safe (rule M2),
 *   - the cos/sin table of C_j * theta_i: product and trig in fp64, rounded once to fp32.
 */
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <mutex>
#include <new>

#include "plan_internal.h"

using leyline::DevTile;
using leyline::IdxRun;

namespace {

leyline_tuning g_tuning = {0, 0, 0, 0, 0, 0, 0};

inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

struct Seg {
    int32_t kind;  /* 0 KEEP, 1 INSERT */
    int64_t src, dst, len, shift;
};

/* Segments of one request in new-position order.  Returns L_new. */
int64_t build_segments(int64_t L_old, const leyline_directive* d, int32_t k, std::vector<Seg>& out, int64_t* trim) {
    int64_t C = 0, pos = 0;
    *trim = -1;
    for (int32_t j = 0; j < k; ++j) {
        if (d[j].start > pos) out.push_back({0, pos, pos + C, d[j].start - pos, C});
        if (d[j].semantic == LEYLINE_FORGET) { /* truncate here, re-prefill is the caller's */
            *trim = d[j].start + C;
            return d[j].start + C;
        }
        if (d[j].repl_len > 0) out.push_back({1, d[j].repl_row, d[j].start + C, d[j].repl_len, 0});
        C += (int64_t)d[j].repl_len - (d[j].end - d[j].start); /* Delta = |R| - (e - s) */
        pos = d[j].end;
    }
    if (L_old > pos) out.push_back({0, pos, pos + C, L_old - pos, C});
    return L_old + C;
}

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

/* Rule V of DESIGN.md (same order as the paper's checks are stated: PAPER.md:98, :409, :635). */
leyline_status check_directives(int32_t n_req, const int64_t* seq_lens, int32_t n_dir, const leyline_directive* d) {
    for (int32_t i = 0; i < n_dir; ++i) {
        if (d[i].request < 0 || d[i].request >= n_req) return LEYLINE_E_RANGE;
        if (d[i].start < 0 || d[i].end < d[i].start || d[i].repl_len < 0 || d[i].repl_row < 0) return LEYLINE_E_INVALID;
        if (d[i].semantic != LEYLINE_AMORTIZE && d[i].semantic != LEYLINE_FORGET) return LEYLINE_E_INVALID;
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

/* Rows per k_rotate_band work item: as many as fill the block's kRotUnitsPerItem (row, pair column) units. */
int choose_rot_tile_rows(const leyline_cache_desc& c, int E, const leyline_tuning& t) {
    const int64_t cols = (int64_t)heads_of(c) * ((int64_t)c.rope_dim * E / 32);
    int64_t cap = std::max<int64_t>(1, leyline::kRotUnitsPerItem / cols);
    int64_t want = t.tile_rows > 0 ? t.tile_rows : cap;
    return (int)std::max<int64_t>(1, std::min(want, cap));
}

/* A plan per turn is the steady state of a server: the large tables of a destroyed plan (tiles, page tables, released
 * list, ...) are handed to the next plan instead of going back to the allocator, which would return them to the OS
 * and make the next plan fault every page in again (measured: 130 of the 140 us of a config-3 plan). */
struct PlanBuffers {
    std::vector<DevTile> tiles;
    std::vector<int32_t> tabs, released, new_pages;
    std::vector<float> trig;
    std::vector<leyline_segment> segments;
    std::vector<IdxRun> slot_runs, page_runs;
};
std::mutex g_recycle_mu;
std::vector<PlanBuffers> g_recycled;
constexpr size_t kMaxRecycled = 8;

void take_buffers(leyline_plan_s* pl) {
    std::lock_guard<std::mutex> lk(g_recycle_mu);
    if (g_recycled.empty()) return;
    PlanBuffers b = std::move(g_recycled.back());
    g_recycled.pop_back();
    pl->tiles = std::move(b.tiles);         pl->tiles.clear();
    pl->tabs = std::move(b.tabs);           pl->tabs.clear();
    pl->released = std::move(b.released);   pl->released.clear();
    pl->new_pages = std::move(b.new_pages); pl->new_pages.clear();
    pl->trig = std::move(b.trig);           pl->trig.clear();
    pl->segments = std::move(b.segments);   pl->segments.clear();
    pl->slot_runs = std::move(b.slot_runs); pl->slot_runs.clear();
    pl->page_runs = std::move(b.page_runs); pl->page_runs.clear();
}

void give_buffers(leyline_plan_s* pl) {
    PlanBuffers b;
    b.tiles = std::move(pl->tiles);
    b.tabs = std::move(pl->tabs);
    b.released = std::move(pl->released);
    b.new_pages = std::move(pl->new_pages);
    b.trig = std::move(pl->trig);
    b.segments = std::move(pl->segments);
    b.slot_runs = std::move(pl->slot_runs);
    b.page_runs = std::move(pl->page_runs);
    std::lock_guard<std::mutex> lk(g_recycle_mu);
    if (g_recycled.size() < kMaxRecycled) g_recycled.push_back(std::move(b));
}

void discard(leyline_plan_s* pl) { /* a plan abandoned half-built: its buffers are still worth keeping */
    give_buffers(pl);
    delete pl;
}

/* split [dst0, dst0+len) into tiles whose boundaries are multiples of tile_rows in `align_pos` space */
template <class F>
void split_tiles(int64_t src0, int64_t dst0, int64_t len, int64_t align0, int tile_rows, F&& emit) {
    int64_t done = 0;
    while (done < len) {
        int64_t a = align0 + done;
        int64_t n = std::min<int64_t>(len - done, tile_rows - (a % tile_rows));
        emit(src0 + done, dst0 + done, (int32_t)n);
        done += n;
    }
}

}  // namespace

extern "C" leyline_status leyline_plan(const leyline_cache_desc* desc, int32_t mode, int32_t n_requests,
                                       const int64_t* seq_lens, const int64_t* pt_offsets, const int32_t* pages,
                                       int32_t n_directives, const leyline_directive* directives,
                                       const int32_t* free_ids, int64_t n_free, leyline_plan_t** out) {
    if (!out) return LEYLINE_E_INVALID;
    *out = nullptr;
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
    for (int32_t r = 0; r < n_requests; ++r) {
        if (seq_lens[r] < 0 || pt_offsets[r] < 0 || pt_offsets[r + 1] < pt_offsets[r]) return LEYLINE_E_INVALID;
        int64_t need = ceil_div(seq_lens[r], P);
        if (pt_offsets[r + 1] - pt_offsets[r] < need) return LEYLINE_E_INVALID;
        if (need > 0 && !pages) return LEYLINE_E_INVALID;
        for (int64_t p = 0; p < need; ++p) {
            int32_t id = pages[pt_offsets[r] + p];
            if (id < 0 || id >= pool_pages) return LEYLINE_E_RANGE;
        }
    }
    const int64_t free_limit = mode == LEYLINE_ROTATE_ONLY ? desc->pool_slots : pool_pages;
    st = check_directives(n_requests, seq_lens, n_directives, directives);
    if (st != LEYLINE_OK) return st;

    leyline_plan_s* pl = new (std::nothrow) leyline_plan_s();
    if (!pl) return LEYLINE_E_INVALID;
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
    pl->tuning = g_tuning;
    pl->desc.rope_heads = heads_of(*desc);
    pl->n_heads = heads_of(*desc);
    pl->head_chunks = desc->rope_dim * E / 16;
    if (g_tuning.kernel == 1 && !row_kernel_ok(*desc, E)) { /* forced row kernel on a band it does not cover */
        discard(pl);
        return LEYLINE_E_UNSUPPORTED;
    }
    pl->use_bulk = choose_bulk(*desc, E, g_tuning, mode);
    pl->tile_rows = choose_tile_rows(*desc, E, g_tuning, pl->use_bulk);
    pl->rot_tile_rows = mode == LEYLINE_ROTATE_ONLY ? choose_rot_tile_rows(*desc, E, g_tuning) : 0;
    /* ROTATE_ONLY on a full-width K pool rewrites most of every row anyway: whole rows then
     * stream through the bulk mover and come back to the slots they were read from (measured: GQA 6.42 -> 6.7 TB/s,
     * head_dim 96 5.86 -> 6.5), instead of the strided band kernel that MLA's 1/9 band needs */
    pl->rotate_with_bulk = mode == LEYLINE_ROTATE_ONLY && g_tuning.kernel != 1 &&
                           2 * (int64_t)heads_of(*desc) * desc->rope_dim >= row_elems(*desc) &&
                           desc->row_stride_bytes == row_elems(*desc) * E;
    if (pl->rotate_with_bulk) {
        pl->use_bulk = true;
        pl->tile_rows = choose_tile_rows(*desc, E, g_tuning, true);
        pl->rot_tile_rows = pl->tile_rows;
    }
    const int TR = pl->tile_rows;
    const int TR_ROT = pl->rot_tile_rows;

    /* tabs: old page tables first, one row per request */
    std::vector<int32_t> old_tab_off(n_requests + 1, 0);
    for (int32_t r = 0; r < n_requests; ++r) {
        int64_t need = ceil_div(seq_lens[r], P);
        old_tab_off[r] = (int32_t)pl->tabs.size();
        pl->tabs.insert(pl->tabs.end(), pages + (need ? pt_offsets[r] : 0), pages + (need ? pt_offsets[r] : 0) + need);
    }
    old_tab_off[n_requests] = (int32_t)pl->tabs.size();

    std::map<int64_t, int32_t> trig_of;
    auto trig_index = [&](int64_t C) -> int32_t {
        if (C == 0) return -1; /* G19: a zero shift is a byte copy, never arithmetic */
        auto it = trig_of.find(C);
        if (it != trig_of.end()) return it->second;
        int32_t g = (int32_t)pl->trig_shifts.size();
        trig_of.emplace(C, g);
        pl->trig_shifts.push_back(C);
        const size_t at = pl->trig.size();
        pl->trig.resize(at + 2 * (size_t)H);
        for (int i = 0; i < H; ++i) { /* fp64 product, fp64 libm (one sincos call), rounded once to fp32 */
            double sn, cs;
            ::sincos((double)C * (double)pl->inv_freq[i], &sn, &cs);
            pl->trig[at + (size_t)i] = (float)cs;
            pl->trig[at + (size_t)H + (size_t)i] = (float)sn;
        }
        return g;
    };

    pl->old_seq_lens.assign(seq_lens, seq_lens + n_requests);
    pl->new_seq_lens.resize(n_requests);
    pl->forget_trim.resize(n_requests);
    pl->slot_offsets.assign(n_requests + 1, 0);
    pl->new_pt_offsets.assign(n_requests + 1, 0);

    struct ReqWork { std::vector<Seg> segs; int64_t k0; int32_t new_tab; };
    std::vector<ReqWork> work(n_requests);
    std::vector<int32_t> token_lists;               /* ROTATE_ONLY: consumed free slots, in consumption order */
    std::vector<DevTile> move_tiles = std::move(pl->tiles), insert_tiles; /* the recycled capacity, if any */
    move_tiles.clear();
    int64_t consumed = 0;
    int32_t di = 0;
    bool nofree = false, badfree = false;

    auto take_free = [&]() -> int32_t {
        if (consumed >= n_free) { nofree = true; return 0; }
        int32_t id = free_ids[consumed++];
        if (id < 0 || id >= free_limit) badfree = true;
        return id;
    };
    /* the next `count` free ids appended to `dst` in one go (front to back, as take_free would) */
    auto take_free_range = [&](std::vector<int32_t>& dst, int64_t count) {
        if (count <= 0) return;
        if (consumed + count > n_free) { nofree = true; return; }
        const int32_t* ids = free_ids + consumed;
        for (int64_t q = 0; q < count; ++q)
            if (ids[q] < 0 || ids[q] >= free_limit) badfree = true;
        dst.insert(dst.end(), ids, ids + count);
        consumed += count;
    };

    /* pass 1: segments, maps, released lists (requests ascending, free ids front to back) */
    for (int32_t r = 0; r < n_requests && !nofree; ++r) {
        int32_t d0 = di;
        while (di < n_directives && directives[di].request == r) ++di;
        const int32_t k = di - d0;
        const int64_t L_old = seq_lens[r];
        ReqWork& w = work[r];
        int64_t trim = -1;
        const int64_t L_new = build_segments(L_old, directives + d0, k, w.segs, &trim);
        pl->new_seq_lens[r] = L_new;
        pl->forget_trim[r] = trim;
        pl->slot_offsets[r + 1] = pl->slot_offsets[r] + L_new;
        for (const Seg& s : w.segs)
            pl->segments.push_back({r, s.kind, s.src, s.dst, s.len, s.shift});
        const int64_t n_old = ceil_div(L_old, P), n_new = ceil_div(L_new, P);
        const int32_t* old_row = pl->tabs.data() + old_tab_off[r];
        if (mode == LEYLINE_FRESH) {
            /* M1: pages before the first edited page kept, the rest compacted into fresh pages */
            if (k == 0) {
                w.k0 = n_old;
                pl->new_pages.insert(pl->new_pages.end(), old_row, old_row + n_old);
            } else {
                w.k0 = directives[d0].start / P;
                pl->new_pages.insert(pl->new_pages.end(), old_row, old_row + w.k0);
                take_free_range(pl->new_pages, n_new - w.k0);
                if (n_old > w.k0) pl->released.insert(pl->released.end(), old_row + w.k0, old_row + n_old);
            }
        } else if (mode == LEYLINE_INPLACE_MOVE) {
            /* M2: identity on the common pages, growth appends, shrink releases the tail */
            pl->new_pages.insert(pl->new_pages.end(), old_row, old_row + std::min(n_old, n_new));
            take_free_range(pl->new_pages, n_new - n_old);
            if (n_old > n_new) pl->released.insert(pl->released.end(), old_row + n_new, old_row + n_old);
        } else {
            /* M3: no row moves; removed positions' slots are released in order */
            int64_t pos = 0;
            auto slot_old = [&](int64_t t) { return (int32_t)(((int64_t)old_row[t >> pshift] << pshift) | (t & (P - 1))); };
            for (const Seg& s : w.segs) {
                if (s.kind == 0) {
                    for (int64_t t = pos; t < s.src; ++t) pl->released.push_back(slot_old(t));
                    pos = s.src + s.len;
                } else {
                    for (int64_t q = 0; q < s.len && !nofree; ++q) token_lists.push_back(take_free());
                }
            }
            for (int64_t t = pos; t < L_old; ++t) pl->released.push_back(slot_old(t));
        }
        pl->new_pt_offsets[r + 1] = (int64_t)pl->new_pages.size();
    }
    if (nofree || badfree) {
        discard(pl);
        return nofree ? LEYLINE_E_NOFREE : LEYLINE_E_RANGE;
    }

    /* tabs: new page tables, then token-level lists */
    const int32_t new_tab_base = (int32_t)pl->tabs.size();
    pl->tabs.insert(pl->tabs.end(), pl->new_pages.begin(), pl->new_pages.end());
    const int32_t token_base = (int32_t)pl->tabs.size();
    pl->tabs.insert(pl->tabs.end(), token_lists.begin(), token_lists.end());

    /* pass 2: tiles, index runs */
    int64_t token_cursor = 0;
    for (int32_t r = 0; r < n_requests; ++r) {
        ReqWork& w = work[r];
        const int32_t src_tab = old_tab_off[r];
        const int32_t dst_tab = new_tab_base + (int32_t)pl->new_pt_offsets[r];
        if (mode == LEYLINE_ROTATE_ONLY) {
            for (const Seg& s : w.segs) {
                if (s.kind == 0) {
                    pl->slot_runs.push_back({pl->slot_offsets[r] + s.dst, s.len, s.src, src_tab, 0});
                    int32_t g = trig_index(s.shift);
                    if (g < 0) continue;
                    split_tiles(s.src, s.dst, s.len, s.src, TR_ROT, [&](int64_t a, int64_t b, int32_t n) {
                        move_tiles.push_back({a, b, src_tab, src_tab, n, g, pl->rotate_with_bulk ? leyline::TILE_DST_IS_SRC : 0,
                                              0, -1, r});
                    });
                } else {
                    int32_t list = token_base + (int32_t)token_cursor;
                    pl->slot_runs.push_back({pl->slot_offsets[r] + s.dst, s.len, 0, list, 1});
                    split_tiles(s.src, 0, s.len, 0, TR, [&](int64_t a, int64_t b, int32_t n) {
                        insert_tiles.push_back({a, b, -1, list, n, -1, leyline::TILE_SRC_REPL | leyline::TILE_DST_TOKEN,
                                                0, -1, r});
                    });
                    token_cursor += s.len;
                }
            }
            continue;
        }
        if (pl->new_seq_lens[r] > 0)
            pl->slot_runs.push_back({pl->slot_offsets[r], pl->new_seq_lens[r], 0, dst_tab, 0});
        if (mode == LEYLINE_FRESH) {
            const int64_t first = w.k0 * P; /* new positions >= first live in fresh pages and must be written */
            for (const Seg& s : w.segs) {
                if (s.kind == 1) {
                    split_tiles(s.src, s.dst, s.len, s.dst, TR, [&](int64_t a, int64_t b, int32_t n) {
                        insert_tiles.push_back({a, b, -1, dst_tab, n, -1, leyline::TILE_SRC_REPL, 0, -1, r});
                    });
                    continue;
                }
                int64_t skip = std::max<int64_t>(0, first - s.dst);
                if (skip >= s.len) continue;
                int32_t g = trig_index(s.shift);
                split_tiles(s.src + skip, s.dst + skip, s.len - skip, s.dst + skip, TR,
                            [&](int64_t a, int64_t b, int32_t n) {
                                move_tiles.push_back({a, b, src_tab, dst_tab, n, g, 0, 0, -1, r});
                            });
            }
        } else { /* INPLACE_MOVE, rule M2 */
            /* per-thread scratch that keeps its capacity from plan to plan (same reason as PlanBuffers) */
            static thread_local std::vector<DevTile> left, right;
            left.clear();
            right.clear();
            const size_t first_insert = insert_tiles.size();
            for (const Seg& s : w.segs) {
                if (s.kind == 1) {
                    split_tiles(s.src, s.dst, s.len, s.dst, TR, [&](int64_t a, int64_t b, int32_t n) {
                        insert_tiles.push_back({a, b, -1, dst_tab, n, -1, leyline::TILE_SRC_REPL, 0, -1, r});
                    });
                    continue;
                }
                if (s.shift == 0) continue; /* stays where it is, bytes untouched */
                int32_t g = trig_index(s.shift);
                std::vector<DevTile>& grp = s.shift < 0 ? left : right;
                split_tiles(s.src, s.dst, s.len, s.dst, TR, [&](int64_t a, int64_t b, int32_t n) {
                    grp.push_back({a, b, src_tab, dst_tab, n, g, 0, 0, -1, r});
                });
            }
            /* left-shifters ascending: a tile's destination covers source rows of tiles at lower positions */
            const int32_t base_l = (int32_t)move_tiles.size();
            for (size_t i = 0, lo = 0; i < left.size(); ++i) {
                DevTile t = left[i];
                const int64_t d0 = t.dst_pos, d1 = t.dst_pos + t.n_rows;
                while (lo < i && left[lo].src_pos + left[lo].n_rows <= d0) ++lo;
                size_t hi = lo; /* first tile at or after lo whose source starts at or past d1 */
                while (hi < i && left[hi].src_pos < d1) ++hi;
                t.dep_lo = base_l + (int32_t)lo;
                t.dep_hi = base_l + (int32_t)hi - 1;
                move_tiles.push_back(t);
            }
            /* right-shifters descending: destination covers source rows of tiles at higher positions */
            const int32_t base_r = (int32_t)move_tiles.size();
            std::reverse(right.begin(), right.end());
            for (size_t i = 0, lo = 0; i < right.size(); ++i) {
                DevTile t = right[i];
                const int64_t d0 = t.dst_pos, d1 = t.dst_pos + t.n_rows;
                while (lo < i && right[lo].src_pos >= d1) ++lo;
                size_t hi = lo;
                while (hi < i && right[hi].src_pos + right[hi].n_rows > d0) ++hi;
                t.dep_lo = base_r + (int32_t)lo;
                t.dep_hi = base_r + (int32_t)hi - 1;
                move_tiles.push_back(t);
            }
            /* inserts run in the same launch, after every move in ticket order: a replacement row may land on a row
             * some move tile of this request still has to read, so it waits for the hull of those tiles (a superset
             * is safe: all of them hold smaller tickets) */
            for (size_t q = first_insert; q < insert_tiles.size(); ++q) {
                DevTile& t = insert_tiles[q];
                const int64_t d0 = t.dst_pos, d1 = t.dst_pos + t.n_rows;
                /* within the left-shifters (and within the right-shifters) sources are monotone in ticket order, so
                 * the overlapping tiles of one group are a contiguous, exact range; only an insert that lands on
                 * sources of BOTH groups gets the hull across them */
                int32_t lo = INT32_MAX, hi = -1;
                for (int32_t m = base_l; m < (int32_t)move_tiles.size(); ++m)
                    if (move_tiles[m].src_pos < d1 && move_tiles[m].src_pos + move_tiles[m].n_rows > d0) {
                        lo = std::min(lo, m);
                        hi = std::max(hi, m);
                    }
                t.dep_lo = hi >= 0 ? lo : 0;
                t.dep_hi = hi;
            }
        }
    }
    if (mode != LEYLINE_ROTATE_ONLY && !pl->new_pages.empty())
        pl->page_runs.push_back({0, (int64_t)pl->new_pages.size(), new_tab_base, 0, 2});

    leyline_plan_info& in = pl->info;
    in.mode = mode;
    in.n_requests = n_requests;
    in.total_new_tokens = pl->slot_offsets[n_requests];
    in.total_new_pages = mode == LEYLINE_ROTATE_ONLY ? 0 : (int64_t)pl->new_pages.size();
    in.n_free_consumed = consumed;
    in.n_released = (int64_t)pl->released.size();
    in.n_segments = (int64_t)pl->segments.size();
    in.n_move_tiles = (int64_t)move_tiles.size();
    in.n_tiles = (int64_t)(move_tiles.size() + insert_tiles.size());
    in.n_trig = (int64_t)pl->trig_shifts.size();
    for (const DevTile& t : move_tiles) {
        if (mode != LEYLINE_ROTATE_ONLY) in.rows_moved += t.n_rows;
        if (t.trig >= 0) in.rows_rotated += t.n_rows;
    }
    for (const DevTile& t : insert_tiles) in.rows_inserted += t.n_rows;
    const int64_t row_bytes = row_elems(*desc) * E, band_bytes = (int64_t)heads_of(*desc) * desc->rope_dim * E;
    int64_t per_layer = (in.rows_moved + in.rows_inserted) * row_bytes;
    if (mode == LEYLINE_ROTATE_ONLY) per_layer = in.rows_rotated * band_bytes + in.rows_inserted * row_bytes;
    in.bytes_read = in.bytes_written = per_layer * desc->n_layers;
    in.bytes_index = 4 * in.total_new_tokens + 4 * in.total_new_pages;
    in.tile_rows = pl->tile_rows;
    in.rot_tile_rows = pl->rot_tile_rows;
    in.mover = pl->use_bulk ? 2 : 1; /* ROTATE_ONLY: 2 = the rotation itself runs on the bulk mover (wide bands) */
    if (mode == LEYLINE_ROTATE_ONLY && !pl->rotate_with_bulk) in.mover = 1;
    if (mode == LEYLINE_ROTATE_ONLY) pl->new_pages.clear();

    if (mode == LEYLINE_INPLACE_MOVE) { /* how far back (in tiles) a waiting tile's dependencies sit: a launch hint */
        std::vector<int32_t> dist;
        for (size_t i = 0; i < move_tiles.size(); ++i)
            if (move_tiles[i].dep_hi >= move_tiles[i].dep_lo) dist.push_back((int32_t)i - move_tiles[i].dep_hi);
        if (!dist.empty()) {
            std::nth_element(dist.begin(), dist.begin() + (long)(dist.size() / 2), dist.end());
            pl->dep_distance_median = dist[dist.size() / 2];
        }
    }
    pl->tiles = std::move(move_tiles);
    pl->tiles.insert(pl->tiles.end(), insert_tiles.begin(), insert_tiles.end());
    *out = pl;
    return LEYLINE_OK;
}

/* ------------------------------------------------------------------ queries ---- */

#define LEYLINE_GETTER(name, type, member)                                         \
    extern "C" leyline_status name(const leyline_plan_t* plan, type* out) {        \
        if (!plan || (!out && !plan->member.empty())) return LEYLINE_E_INVALID;    \
        if (!plan->member.empty()) std::memcpy(out, plan->member.data(), plan->member.size() * sizeof(type)); \
        return LEYLINE_OK;                                                         \
    }

extern "C" leyline_status leyline_plan_get_info(const leyline_plan_t* plan, leyline_plan_info* out) {
    if (!plan || !out) return LEYLINE_E_INVALID;
    *out = plan->info;
    return LEYLINE_OK;
}
LEYLINE_GETTER(leyline_plan_new_seq_lens, int64_t, new_seq_lens)
LEYLINE_GETTER(leyline_plan_forget_trim, int64_t, forget_trim)
LEYLINE_GETTER(leyline_plan_slot_offsets, int64_t, slot_offsets)
LEYLINE_GETTER(leyline_plan_released, int32_t, released)
LEYLINE_GETTER(leyline_plan_segments, leyline_segment, segments)
LEYLINE_GETTER(leyline_plan_trig_shifts, int64_t, trig_shifts)

extern "C" leyline_status leyline_plan_new_pt_offsets(const leyline_plan_t* plan, int64_t* out) {
    if (!plan || !out || plan->mode == LEYLINE_ROTATE_ONLY) return LEYLINE_E_INVALID;
    std::memcpy(out, plan->new_pt_offsets.data(), plan->new_pt_offsets.size() * sizeof(int64_t));
    return LEYLINE_OK;
}

extern "C" leyline_status leyline_plan_new_pages(const leyline_plan_t* plan, int32_t* out) {
    if (!plan || plan->mode == LEYLINE_ROTATE_ONLY || (!out && !plan->new_pages.empty())) return LEYLINE_E_INVALID;
    if (!plan->new_pages.empty()) std::memcpy(out, plan->new_pages.data(), plan->new_pages.size() * sizeof(int32_t));
    return LEYLINE_OK;
}

extern "C" leyline_status leyline_plan_tiles(const leyline_plan_t* plan, leyline_tile* out) {
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

/* cos/sin table rows, [n_trig][2][rope_dim/2] fp32 (tests check them against an independent fp64 evaluation) */
extern "C" leyline_status leyline_plan_trig_table(const leyline_plan_t* plan, float* out) {
    if (!plan || (!out && !plan->trig.empty())) return LEYLINE_E_INVALID;
    if (!plan->trig.empty()) std::memcpy(out, plan->trig.data(), plan->trig.size() * sizeof(float));
    return LEYLINE_OK;
}

extern "C" void leyline_plan_destroy(leyline_plan_t* plan) {
    if (!plan) return;
    leyline_plan_release_device_(plan);
    give_buffers(plan);
    delete plan;
}

extern "C" const char* leyline_strerror(leyline_status s) {
    switch (s) {
        case LEYLINE_OK: return "ok";
        case LEYLINE_E_INVALID: return "invalid argument";
        case LEYLINE_E_UNSORTED: return "directives not sorted by (request, start)";
        case LEYLINE_E_OVERLAP: return "overlapping spans";
        case LEYLINE_E_RANGE: return "request, span or id out of range";
        case LEYLINE_E_NOFREE: return "free list too short";
        case LEYLINE_E_UNSUPPORTED: return "cache geometry not supported by the kernels";
        case LEYLINE_E_CUDA: return "CUDA error";
    }
    return "unknown status";
}

extern "C" leyline_status leyline_set_tuning(const leyline_tuning* t) {
    if (!t) return LEYLINE_E_INVALID;
    if (t->kernel < 0 || t->kernel > 2 || t->tile_rows < 0 || t->tile_rows > 64 || t->ctas_per_sm < 0 ||
        t->ctas_per_sm > 32 || t->stages < 0 || t->stages > 8 || t->layer_group < 0 ||
        t->layer_group > LEYLINE_MAX_LAYERS_PER_LAUNCH || t->consumer_warps < 0 || t->consumer_warps > 16)
        return LEYLINE_E_INVALID;
    g_tuning = *t;
    return LEYLINE_OK;
}

extern "C" leyline_status leyline_get_tuning(leyline_tuning* t) {
    if (!t) return LEYLINE_E_INVALID;
    *t = g_tuning;
    return LEYLINE_OK;
}

extern "C" const char* leyline_version(void) { return "leyline-b200 0.1 sm_100a"; }

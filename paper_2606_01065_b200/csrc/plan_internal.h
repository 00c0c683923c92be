/*
 * plan_internal.h -- the plan object shared by the host planner (plan.cpp) and the launchers (splice.cu).
 * Not part of the ABI.  See include/leyline.h for the contract and DESIGN.md for the rules (M1-M3, V).
 */
#ifndef LEYLINE_PLAN_INTERNAL_H_
#define LEYLINE_PLAN_INTERNAL_H_

#include <cstdint>
#include <new>
#include <vector>

#include "leyline.h"

namespace leyline {

/* Device work item: up to tile_rows rows that are consecutive in NEW logical position (one segment, hence one
 * rotation).  Source and destination rows are located through int32 tables in `tabs`:
 *   slot(pos) = tabs[tab + (pos >> shift)] << shift | (pos & ((1 << shift) - 1))
 * with shift = log2(page_size) for page tables and 0 for token-level slot lists.  src_tab < 0: the source is
 * the replacement buffer and src_pos is the row inside it. */
struct DevTile {
    int64_t src_pos;
    int64_t dst_pos;
    int32_t src_tab;
    int32_t dst_tab;
    int32_t n_rows;
    int32_t trig;      /* row of the cos/sin table, -1 = byte copy */
    int32_t flags;     /* bit 0: source is the replacement buffer; bit 1: dst table is token-level (shift 0) */
    int32_t dep_lo;    /* INPLACE_MOVE: tiles [dep_lo, dep_hi] must have loaded (same layer) before this stores */
    int32_t dep_hi;
    int32_t request;
};
static_assert(sizeof(DevTile) == 48, "DevTile layout");

enum : int32_t { TILE_SRC_REPL = 1, TILE_DST_TOKEN = 2,
                 TILE_DST_IS_SRC = 4 /* rows are written back to the slots they were read from (in-place rotation) */ };

/* k_rotate_band (a5): (row, pair column) units one block handles = 256 threads x the units a thread keeps in flight;
 * ROTATE_ONLY tiles hold at most this many units, i.e. rot_tile_rows = rot_units_per_item / (rope_heads * head_chunks / 2)
 * rows. */
#ifndef LEYLINE_ROT_BF16_UNROLL
#define LEYLINE_ROT_BF16_UNROLL 6
#endif
constexpr int kRotUnrollBf16 = LEYLINE_ROT_BF16_UNROLL, kRotUnrollFp8 = 4;
constexpr int rot_units_per_item(int elem_bytes) { return 256 * (elem_bytes == 2 ? kRotUnrollBf16 : kRotUnrollFp8); }

/* k_rotate_band_flat (a5 when the rotated segments are short): the rows of ALL rotate tiles, in tile order, form one
 * flat row space; pass b covers flat rows [b * rot_tile_rows, (b + 1) * rot_tile_rows) whatever tiles they fall in.
 * RotPass says where pass b starts: the tile that holds its first row and that row's offset inside the tile. */
struct RotPass {
    int32_t tile;
    int32_t row_off;
};
static_assert(sizeof(RotPass) == 8, "RotPass layout");

/* k_rotate_band_tma (a5 on paged pools): the band of up to kRotTmaBoxRows consecutive slots is one 2-D TMA box. */
constexpr int kRotTmaBoxRows = 64;
constexpr bool kRotateTmaByDefault = false; /* decided by measurement */

/* ROTATE_ONLY: `count` removed old positions pos0.. of the request whose old page table starts at tabs[tab]; their slots
 * are the released list (expanded by leyline_plan_released). */
struct ReleasedRun {
    int32_t tab;
    int64_t pos0, count;
};

/* One run of the token-level index list / page-table output (step a2). */
struct IdxRun {
    int64_t out_begin; /* first output element */
    int64_t length;
    int64_t pos0;      /* kind 0/1: first logical position; kind 2: first element of `tabs` to copy */
    int32_t tab;       /* kind 0: page table offset in tabs; kind 1: token-level list offset */
    int32_t kind;      /* 0 = via page table (shift = log2 P), 1 = via token-level list, 2 = raw copy of tabs */
};
static_assert(sizeof(IdxRun) == 32, "IdxRun layout");

}  // namespace leyline

struct leyline_plan_s {
    leyline_cache_desc desc;            /* inv_freq / layer_scale pointers redirected to the copies below */
    std::vector<float> inv_freq;
    std::vector<float> layer_scale;
    std::vector<int32_t> layer_pairing; /* per-layer override of desc.pairing, or empty */
    int32_t mode = 0;
    int32_t n_requests = 0;
    int32_t elem_bytes = 2;
    int32_t page_shift = 0;
    int32_t tile_rows = 32;
    int32_t rot_tile_rows = 0;          /* ROTATE_ONLY: rows per k_rotate_band work item */
    int32_t n_heads = 1;                /* heads in the rotated band (desc.rope_heads, 0 read as 1) */
    int32_t head_chunks = 8;            /* 16-byte chunks per head */
    int32_t dep_distance_median = -1;   /* INPLACE_MOVE: median of (tile index - dep_hi) over tiles that wait, -1 if none */
    bool rotate_with_bulk = false;      /* ROTATE_ONLY on a band that is most of the row: the rotation runs on k_move_bulk, in place */
    bool rotate_with_tma = false;       /* ROTATE_ONLY on a narrow band in pages of >= 16 rows: k_rotate_band_tma (2-D TMA boxes) */
    bool rotate_flat = false;           /* ROTATE_ONLY, narrow band, short segments: k_rotate_band_flat over rot_passes */
    bool use_bulk = false;              /* a3/a4 run on k_move_bulk (TMA bulk copies) instead of k_move_rows */
    leyline_tuning tuning{};

    std::vector<int64_t> old_seq_lens, new_seq_lens, forget_trim, slot_offsets, new_pt_offsets, old_pt_offsets;
    std::vector<int32_t> new_pages;     /* concatenated new page-table rows (FRESH / INPLACE_MOVE) */
    std::vector<int32_t> released;      /* page modes: released page ids */
    std::vector<leyline::ReleasedRun> released_runs; /* ROTATE_ONLY: released slots as runs of removed old positions */
    std::vector<int64_t> seg_begin;     /* segments of request r: [seg_begin[r], seg_begin[r+1]) */
    std::vector<leyline_segment> segments;
    std::vector<leyline::DevTile> tiles;   /* move tiles first, then insert tiles; ticket order */
    std::vector<leyline::RotPass> rot_passes; /* rotate_flat: start of every block pass in the flat row space of the rotate tiles */
    std::vector<int64_t> trig_shifts;
                                        /* the cos/sin table [n_trig][2][H] of C * theta_i is evaluated in fp64 on the
                                           device by the launch's index kernel (and by the host only for the query) */
    std::vector<int32_t> tabs;          /* old page tables ++ new page tables ++ token-level lists */
    std::vector<leyline::IdxRun> slot_runs;  /* produce dev_slot_idx_out */
    std::vector<leyline::IdxRun> page_runs;  /* produce dev_page_table_out */
    leyline_plan_info info{};

    /* device side (owned by splice.cu; created on first launch, freed by leyline_plan_destroy) */
    void* d_blob = nullptr;             /* tiles | trig (device-computed) | shifts | inv_freq | tabs | slot_runs | page_runs */
    int64_t off_tiles = 0, off_trig = 0, off_shifts = 0, off_inv_freq = 0, off_tabs = 0, off_slot_runs = 0, off_page_runs = 0,
            off_rot_passes = 0, blob_bytes = 0;
    void* d_scratch = nullptr;          /* tail of d_blob: [0,256) ticket counters; then hazard flags [n_move_tiles * n_layers] int32 */
    int64_t scratch_bytes = 0;
    int device = -1;
    void* ev_start = nullptr;           /* cudaEvent_t pair around the data-moving kernels (tuning.profile) */
    void* ev_stop = nullptr;
    void* last_stream = nullptr;        /* stream of the last launch: the device tables are freed on it */
    void* ev_uploaded = nullptr;        /* leyline_plan_prefetch: cudaEvent_t recorded after the upload on the copy stream */
    bool scratch_clean = false;         /* the upload path already zeroed d_scratch; the first launch skips its memset */
    bool trig_ready = false;            /* the device cos/sin table has been written by a launch's index kernel */
};

/* closes a function-try-block of an extern "C" entry point: nothing is thrown across the ABI */
#define LEYLINE_CATCH_STATUS                                     \
    catch (const std::bad_alloc&) { return LEYLINE_E_NOMEM; }    \
    catch (...) { return LEYLINE_E_INVALID; }

namespace leyline {
/* implemented in splice.cu; plan.cpp calls it from leyline_plan_destroy (not part of the ABI, not exported) */
void plan_release_device(leyline_plan_s* plan);
}  // namespace leyline

#endif /* LEYLINE_PLAN_INTERNAL_H_ */

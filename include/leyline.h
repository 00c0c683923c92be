/*
 * leyline.h -- C ABI of the B200-native Leyline splice library (libleyline.so).
 *
 * The library implements the data-parallel hot path of the KV-cache directive of
 * "Leyline: KV Cache Directives for Agentic Inference" (arxiv/paper_2606_01065).
 * Citations "PAPER.md:N" are lines of the paper text; "G<n>" / "M<n>" / "rule V" are the readings and
 * rules listed in DESIGN.md.
 *
 * One directive D = (s_start, s_end, R, m) replaces the cached token span
 * [s_start, s_end) of a request by |R| replacement tokens.  Applying it to an MLA cache means
 * (PAPER.md:127 steps 1-3, PAPER.md:405 (a)-(d)):
 *   (a) the span's KV slots are released;
 *   (b) the replacement's precomputed KV rows are written at new positions [s_start, s_start+|R|);
 *   (c) every downstream token i >= s_end is re-keyed to i + Delta, Delta = |R| - (s_end - s_start), and its
 *       K_pe is rotated in closed form, K_pe_new = R(Delta) K_pe (Eq. (1)), latent untouched;
 *   (d) nothing for Q.
 * Several sorted, non-overlapping directives per request compose into one rotation per segment by the
 * cumulative shift C_j = sum_{i<=j} Delta_i (R(a)R(b) = R(a+b)).
 *
 * Cache layout (caller-owned): per layer one pool of `n_slots` rows of
 * `row_stride_bytes`; a row is `latent_dim` elements of c_kv followed by `rope_dim` elements of K_pe
 * (bf16, or fp8 e4m3 with one fp32 scale per layer).  Page p of a layer is rows [p*page_size, (p+1)*page_size).
 * A request's logical position t lives at slot  table[t / page_size] * page_size + t % page_size.
 *
 * Threading / streams: leyline_plan is pure host code (no CUDA call, no device needed).  leyline_splice,
 * leyline_rotate_inplace and leyline_rotate_inplace_master upload the plan's tables on first use (stream-ordered; or
 * earlier, on the library's copy stream, after leyline_plan_prefetch), launch one index kernel and one data kernel on
 * the caller's stream and return without synchronising.  A plan may be in flight on one stream at a time; different
 * plans may be in flight on different streams and may be driven from different host threads.
 * leyline_set_tuning is a process-wide benchmarking default read (under a lock) by leyline_plan only; leyline_plan_ex
 * takes its tuning as an argument and never looks at the process-wide one.
 * Nothing is thrown across the ABI: every entry point returns a leyline_status (a C++ exception inside the library,
 * e.g. std::bad_alloc while planning a very large batch, comes back as LEYLINE_E_NOMEM / LEYLINE_E_INVALID).
 * Only the functions declared in include/ are exported from libleyline.so (-fvisibility=hidden + LEYLINE_API).
 * There is no CPU fallback: without a CUDA device the launch entry points return LEYLINE_E_CUDA.
 * The discovery side (chunker, registry) is declared in leyline_cdc.h.
 */
#ifndef LEYLINE_H_
#define LEYLINE_H_

#include <stdint.h>

#if defined(__GNUC__)
#define LEYLINE_API __attribute__((visibility("default")))
#else
#define LEYLINE_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    LEYLINE_OK = 0,
    LEYLINE_E_INVALID = 1,     /* NULL / negative / inconsistent argument */
    LEYLINE_E_UNSORTED = 2,    /* directives not sorted by (request, start) */
    LEYLINE_E_OVERLAP = 3,     /* two spans of one request overlap (rejected at apply time) */
    LEYLINE_E_RANGE = 4,       /* request id or span outside the request */
    LEYLINE_E_NOFREE = 5,      /* free list too short for the pages / slots the plan must consume */
    LEYLINE_E_UNSUPPORTED = 6, /* geometry the kernels do not cover (see leyline_cache_desc) */
    LEYLINE_E_CUDA = 7,        /* CUDA runtime error (message via leyline_last_cuda_error) */
    LEYLINE_E_NOMEM = 8,       /* host allocation failed inside the library (nothing was produced) */
    LEYLINE_E_ALIAS = 9        /* a consumed free id is a live page / slot or appears twice, or (INPLACE_MOVE,
                                  ROTATE_ONLY) a page is listed by two requests of which one is edited: executing the
                                  plan would overwrite live KV */
} leyline_status;

typedef enum { LEYLINE_BF16 = 0, LEYLINE_FP8_E4M3 = 1 } leyline_dtype;
/* RoPE pairing: NEOX pairs element i with i + rope_dim/2, INTERLEAVED pairs 2i with 2i+1. */
typedef enum { LEYLINE_ROPE_NEOX = 0, LEYLINE_ROPE_INTERLEAVED = 1 } leyline_pairing;
/* FRESH        : the paper's dst_slots path: everything from the first edited page on is
 *                compacted into pages taken from the free list; source pages are released, never written (M1).
 * INPLACE_MOVE : rows move inside the request's own pages (growth appends free pages, shrink releases the
 *                tail); overlapping source/destination handled by hazard-ordered tiles (M2).
 * ROTATE_ONLY  : the paper's in-place path: no row moves, K_pe rotated where it sits, the
 *                token-level slot index list is rewritten (M3). */
typedef enum { LEYLINE_FRESH = 0, LEYLINE_INPLACE_MOVE = 1, LEYLINE_ROTATE_ONLY = 2 } leyline_mode;
/* PAPER.md:98, :102.  FORGET truncates the request at the directive's start: everything from there on is released and
 * no kernel touches it (a request whose first effective directive is a FORGET launches nothing at all). */
typedef enum { LEYLINE_AMORTIZE = 0, LEYLINE_FORGET = 1 } leyline_semantic;

#define LEYLINE_MAX_LAYERS_PER_LAUNCH 128

typedef struct {
    int32_t n_layers;          /* >= 1 */
    int32_t latent_dim;        /* position-free elements at the start of a row (c_kv: 512 for DeepSeek MLA; 0 for a
                                  GQA/MHA K pool; a V pool's elements when K and V share a row); bytes a multiple of 16 */
    int32_t rope_dim;          /* rotated elements per HEAD (64 for MLA's K_pe; head_dim 128 / 96 for full-width K,
                                  PAPER.md:223, :515, Table 8 :533-541); even; (rope_dim/2)*elem bytes a multiple of 16 */
    int32_t page_size;         /* tokens per page, power of two (1 = token-level slots) */
    int32_t dtype;             /* leyline_dtype */
    int32_t pairing;           /* leyline_pairing (inside each head) */
    int32_t rope_heads;        /* heads in the rotated band, each rope_dim elements, all using the same inv_freq; 0 reads
                                  as 1.  1 = MLA (one shared K_pe per token); kv_heads = the GQA/MHA degenerate case
                                  "qk_nope_head_dim=0 rotates the full K".  Row = latent_dim +
                                  rope_heads*rope_dim elements. */
    int32_t reserved_;         /* must be 0 */
    int64_t row_stride_bytes;  /* >= (latent_dim + rope_heads*rope_dim)*elem bytes, multiple of 16.  Bytes of a row
                                  beyond that (padding) are never read or written. */
    int64_t pool_slots;        /* rows in each layer's pool (a multiple of page_size); page ids are validated
                                  against pool_slots / page_size, slot ids against pool_slots */
    const float* inv_freq;     /* HOST, [rope_dim/2]: THE theta_i in fp32 (YaRN etc. already applied; G9).
                                  Copied by leyline_plan. */
    const float* layer_scale;  /* HOST, [n_layers], fp8 only (may be NULL): per-layer dequantisation scale.  A splice
                                  leaves it unchanged, so it cancels in x/scale*scale; it is validated (> 0, finite)
                                  but not used by the kernels (G16). */
    const int32_t* layer_pairing; /* HOST, [n_layers] of leyline_pairing, or NULL: per-layer override of `pairing`
                                  (the paper's helper "reads is_neox_style per layer"; G20).  Layers of one
                                  convention are launched together, so a mixed cache costs one extra launch per mover.
                                  Copied by leyline_plan. */
} leyline_cache_desc;

typedef struct {
    int32_t request;           /* index into seq_lens */
    int32_t repl_len;          /* |R| >= 0 */
    int64_t start, end;        /* span [start, end) in ORIGINAL token indices of the request (G1) */
    int64_t repl_row;          /* first row of this directive's replacement KV inside layer_repl[l] */
    int32_t semantic;          /* leyline_semantic */
    int32_t reserved_;         /* must be 0 */
} leyline_directive;

/* One segment of a request in new-position order (query result). */
typedef struct {
    int32_t request;
    int32_t kind;              /* 0 = KEEP (old rows re-keyed and rotated), 1 = INSERT (replacement rows) */
    int64_t src_begin;         /* KEEP: first old position; INSERT: first replacement row */
    int64_t dst_begin;         /* first new position */
    int64_t length;            /* > 0 (empty segments are omitted) */
    int64_t shift;             /* KEEP: cumulative C_j (rotation amount = dst - src); INSERT: 0 */
} leyline_segment;

typedef struct {
    int32_t mode;
    int32_t n_requests;
    int64_t total_new_tokens;  /* sum of new sequence lengths = length of the token-level index list */
    int64_t total_new_pages;   /* sum of new page-table rows (0 for ROTATE_ONLY) */
    int64_t n_free_consumed;   /* ids taken from the front of the free list */
    int64_t n_released;        /* ids reported back (pages, or slots for ROTATE_ONLY) */
    int64_t n_segments;
    int64_t n_tiles;           /* device work items per layer (move tiles first, then insert tiles) */
    int64_t n_move_tiles;
    int64_t n_trig;            /* rows of the cos/sin table = distinct non-zero cumulative shifts */
    int64_t rows_moved;        /* per layer: KEEP rows copied+rotated (FRESH / INPLACE_MOVE; includes FRESH's head copy) */
    int64_t rows_inserted;     /* per layer: replacement rows written */
    int64_t rows_rotated;      /* per layer: rows whose K_pe is rotated (shift != 0) */
    int64_t bytes_read;        /* ALGORITHMIC bytes over all layers: (latent+rope)*elem per moved/inserted row,
                                  rope*elem per in-place rotated row */
    int64_t bytes_written;     /* same, written */
    int64_t bytes_index;       /* 4 B per new token + 4 B per new page-table entry (once, not per layer) */
    int64_t tile_rows;         /* rows per device work item of the a3/a4 mover chosen for this plan */
    int64_t rot_tile_rows;     /* ROTATE_ONLY: rows per in-place rotation work item (a5), else 0 */
    int64_t mover;             /* a3/a4 kernel this plan launches: 1 = k_move_rows, 2 = k_move_bulk (see leyline_tuning).
                                  ROTATE_ONLY: 1 = k_rotate_band (strided band kernel), 2 = the band is at least half of
                                  the row (full-width K), so whole rows stream through k_move_bulk and are written back
                                  to the slots they were read from, 3 = k_rotate_band_tma (2-D TMA boxes of the band),
                                  4 = k_rotate_band_flat (k_rotate_band's arithmetic with consecutive short tiles packed
                                  into full block passes; chosen when the rotated segments are short) */
} leyline_plan_info;

typedef struct leyline_plan_s leyline_plan_t;

/* Tuning knobs of a plan (defaults = all zero = what bench.py reports).  leyline_plan_ex takes them per call;
 * leyline_plan reads the process-wide default set by leyline_set_tuning. */
typedef struct leyline_tuning_s {
    int32_t kernel;        /* a3/a4 mover: 0 = auto (bulk for unpadded rows in pages of >= 16 rows or of >= 1 KB each, or when the band is not a
                              single head of 2^k <= 32 chunks), 1 = row kernel (LDG/STG through registers; single-head
                              bands of 2^k chunks only, else LEYLINE_E_UNSUPPORTED), 2 = bulk kernel (TMA 1-D bulk
                              copies through shared memory) */
    int32_t tile_rows;     /* rows per tile of the move/insert kernels, 0 = default (row kernel <= 32, bulk <= 64) */
    int32_t ctas_per_sm;   /* row kernel only, 0 = default */
    int32_t profile;       /* 1: record CUDA events around the data-moving kernels (leyline_plan_kernel_ms) */
    int32_t stages;        /* bulk / TMA-band kernels: shared-memory stages per CTA, 0 = as many as fit (bulk: at most 8) */
    int32_t layer_group;   /* bulk / TMA-band kernels: layers per work item (one stage each), 0 = default */
    int32_t consumer_warps;/* bulk kernel only: warps that rotate the band in shared memory, 0 = default (4 for MLA's
                              narrow band, 12 when the band is most of the row); values up to 16 are accepted, at most 12 are used
                              (more never helped and the launch bound caps the registers per thread) */
    int32_t rotate_kernel; /* a5 on a narrow band (MLA): 0 = auto, 1 = k_rotate_band (strided 16-byte loads / stores through
                              registers), 2 = k_rotate_band_tma (the band of a page as one 2-D TMA box staged through shared
                              memory; pages of >= 16 rows, else falls back to 1), 3 = k_rotate_band_flat whenever the
                              geometry allows it (auto picks it only when it saves a fifth of the work items or more) */
    int32_t skip_alias_check; /* 1: the caller guarantees what the alias rule checks (free ids disjoint from live pages and
                              from each other, no page shared with a request edited in place); LEYLINE_E_ALIAS is then
                              never returned and the planner skips its pass over every live page */
} leyline_tuning;

/*
 * leyline_plan -- the host planner (step a1).
 *
 *   desc          cache geometry (copied).
 *   n_requests    number of requests; seq_lens[r] = cached tokens of request r (HOST).
 *   pt_offsets    HOST [n_requests+1]: row r of the page table is pages[pt_offsets[r] .. pt_offsets[r+1]),
 *                 EXACTLY ceil(seq_lens[r]/page_size) entries (a longer row is refused with LEYLINE_E_INVALID: pages
 *                 behind the last token would be neither kept nor released).
 *   pages         HOST int32 page ids.
 *   directives    HOST, sorted by (request, start), spans of one request non-overlapping (adjacent allowed).
 *   free_ids      HOST int32: free PAGE ids (FRESH, INPLACE_MOVE) or free SLOT ids (ROTATE_ONLY); consumed front to
 *                 back, requests in ascending order.  The library never allocates pool pages itself.
 *   out           receives the plan (owned by the caller, release with leyline_plan_destroy).
 *
 * Every directive of every request is validated before any state is produced (all-or-none);
 * on error *out is NULL.  Validation order is rule V of DESIGN.md (first failure wins, directives in order):
 * request out of range -> RANGE; start<0 | end<start | repl_len<0 | repl_row<0 | bad semantic -> INVALID;
 * end > seq_len -> RANGE; request or start decreasing -> UNSORTED; start < previous end -> OVERLAP;
 * then free list too short -> NOFREE; a consumed free id outside the pool -> RANGE; then the alias rule -> ALIAS:
 * a consumed free id that is a live page (a slot of a live page, ROTATE_ONLY) or is consumed twice, and -- for the
 * modes that write a request's own pages, INPLACE_MOVE and ROTATE_ONLY -- a page listed twice when one of its owners
 * has directives (FRESH never writes a request's own pages, so requests may share prefix pages there).
 * Accepted: start==end (pure insert), repl_len==0 (pure delete), both (no-op: changes nothing, in any
 * mode), adjacent spans, start==0, requests without directives (untouched).  directive.reserved_ must be 0.
 * leyline_plan uses the process-wide tuning (leyline_set_tuning); leyline_plan_ex takes `tuning` (NULL = defaults).
 */
LEYLINE_API leyline_status leyline_plan_ex(const leyline_cache_desc* desc, int32_t mode, int32_t n_requests,
                                           const int64_t* seq_lens, const int64_t* pt_offsets, const int32_t* pages,
                                           int32_t n_directives, const leyline_directive* directives,
                                           const int32_t* free_ids, int64_t n_free, const leyline_tuning* tuning,
                                           leyline_plan_t** out);
LEYLINE_API leyline_status leyline_plan(const leyline_cache_desc* desc, int32_t mode, int32_t n_requests,
                            const int64_t* seq_lens, const int64_t* pt_offsets, const int32_t* pages,
                            int32_t n_directives, const leyline_directive* directives, const int32_t* free_ids,
                            int64_t n_free, leyline_plan_t** out);

/* Plan queries (all HOST output buffers, sized from leyline_plan_info). */
LEYLINE_API leyline_status leyline_plan_get_info(const leyline_plan_t* plan, leyline_plan_info* out);
LEYLINE_API leyline_status leyline_plan_new_seq_lens(const leyline_plan_t* plan, int64_t* out /*[n_requests]*/);
/* First FORGET directive's start in new coordinates per request, -1 if none. */
LEYLINE_API leyline_status leyline_plan_forget_trim(const leyline_plan_t* plan, int64_t* out /*[n_requests]*/);
/* Offsets of each request inside the token-level index list: [n_requests+1], prefix sums of new_seq_lens. */
LEYLINE_API leyline_status leyline_plan_slot_offsets(const leyline_plan_t* plan, int64_t* out);
/* New page tables (FRESH / INPLACE_MOVE; LEYLINE_E_INVALID for ROTATE_ONLY): offsets [n_requests+1] and ids. */
LEYLINE_API leyline_status leyline_plan_new_pt_offsets(const leyline_plan_t* plan, int64_t* out);
LEYLINE_API leyline_status leyline_plan_new_pages(const leyline_plan_t* plan, int32_t* out /*[total_new_pages]*/);
/* Released ids, requests ascending: pages in ascending logical order (FRESH: old pages from the first edited
 * page on; INPLACE_MOVE: tail pages) or, for ROTATE_ONLY, the slots of every removed old position in order.
 * Their bytes are never written (PAPER.md:405(a); G14). */
LEYLINE_API leyline_status leyline_plan_released(const leyline_plan_t* plan, int32_t* out /*[n_released]*/);
LEYLINE_API leyline_status leyline_plan_segments(const leyline_plan_t* plan, leyline_segment* out /*[n_segments]*/);

/* One device work item per layer (query result, for tests and tooling): `n_rows` rows that are consecutive in
 * NEW logical position, `dst_pos .. dst_pos+n_rows` of `request`, read from OLD logical positions
 * `src_pos ..` of the same request (or from replacement rows `src_pos ..` when LEYLINE_TILE_SRC_REPL is set).
 * The device resolves positions to slots through the page tables, so a tile may straddle pages.  `trig` is the
 * row of the cos/sin table that rotates the K_pe band (-1: byte copy).  Tiles are listed in TICKET order: the
 * device hands them out in this order, layer fastest.  For INPLACE_MOVE a tile may store only after tiles
 * [dep_lo, dep_hi] (indices into this list, all smaller than its own; empty when dep_lo > dep_hi) have
 * finished LOADING the same layer: those are exactly the tiles whose source rows it overwrites (rule M2 of
 * DESIGN.md).  Move tiles come first ([0, n_move_tiles)), replacement inserts after.  For ROTATE_ONLY the move
 * tiles are the in-place K_pe rotations (src_pos = old position, dst_pos = new position, no row moves). */
#define LEYLINE_TILE_SRC_REPL 1
typedef struct {
    int64_t src_pos;
    int64_t dst_pos;
    int32_t n_rows;
    int32_t trig;
    int32_t flags;
    int32_t dep_lo, dep_hi;
    int32_t request;
} leyline_tile;
LEYLINE_API leyline_status leyline_plan_tiles(const leyline_plan_t* plan, leyline_tile* out /*[n_tiles]*/);
/* Shifts C of the cos/sin table rows: row g holds cos/sin(C_g * theta_i), i in [0, rope_dim/2). */
LEYLINE_API leyline_status leyline_plan_trig_shifts(const leyline_plan_t* plan, int64_t* out /*[n_trig]*/);
/* The table itself, [n_trig][2][rope_dim/2] fp32: cos then sin of C_g * theta_i (fp64 product and trig, rounded once),
 * evaluated on the HOST by this call (libm).  The launches never upload it: the index kernel of every launch evaluates
 * the same expression in fp64 on the device (CUDA's sincos, <= 2 ulp of fp64), which takes the 32 fp64 sincos per
 * distinct shift off the host's critical path (hundreds of shifts per call in the paper's chunk workload),
 * and keeps every value as an fp32 hi + lo pair: hi is the value rounded once to fp32 -- what this call returns -- and
 * lo what that rounding dropped, used only where an output's two products cancel (bf16 caches).
 * leyline_plan_trig_table_device copies the device's hi parts back (after the plan has been launched and its stream
 * synchronised; LEYLINE_E_INVALID before that) so that the two evaluations can be compared. */
LEYLINE_API leyline_status leyline_plan_trig_table(const leyline_plan_t* plan, float* out);
LEYLINE_API leyline_status leyline_plan_trig_table_device(const leyline_plan_t* plan, float* out);

/*
 * leyline_splice -- execute a FRESH or INPLACE_MOVE plan on `cuda_stream` (steps a2-a4).
 *
 *   layer_src   HOST array of n_layers DEVICE pointers to the pools read (16-byte aligned).  "Device pointer" means any
 *               address the device can dereference: device memory, or pinned (page-locked, mapped) host memory --
 *               a host-resident cache is then spliced over PCIe by the same kernels, moving only the rows the plan
 *               touches.
 *   layer_dst   HOST array of n_layers DEVICE pointers to the pools written.  May equal layer_src (fresh pages of
 *               the same pool); MUST equal it for INPLACE_MOVE.  When it differs (FRESH), page ids mean the same
 *               pages in both pools and only the fresh pages are written, into layer_dst: e.g. a swapped-out,
 *               host-resident source spliced straight into the device pool.  The kept prefix pages are not copied.
 *   layer_repl  HOST array of n_layers DEVICE pointers to the replacement KV rows, [rows x row_stride_bytes] per
 *               layer, K_pe already roped at its FINAL position (G12).  NULL = the caller fills the replacement
 *               slots itself -- the paper's own flow, where step (b) is the model's prefill of R into the new
 *               slots (PAPER.md:405(b)): the slots are allocated in the new page table / slot list and their bytes
 *               are left untouched.
 *   dev_page_table_out  DEVICE int32 [total_new_pages] or NULL: receives the new page-table rows (concatenated,
 *               leyline_plan_new_pt_offsets).
 *   dev_slot_idx_out    DEVICE int32 [total_new_tokens] or NULL: receives the token-level slot of every new position.
 *
 * Kernels: index / page-table rewrite, then the fused gather -> rotate -> scatter (+ replacement insert).
 * Asynchronous; only launch errors are returned.  Bytes the mode says are never written are never written.
 */
LEYLINE_API leyline_status leyline_splice(leyline_plan_t* plan, void* const* layer_src, void* const* layer_dst,
                              const void* const* layer_repl, int32_t* dev_page_table_out, int32_t* dev_slot_idx_out,
                              void* cuda_stream);

/*
 * leyline_rotate_inplace -- execute a ROTATE_ONLY plan (steps a2, a5): rotate the band of every downstream
 * token where it sits (128 B of every 1152 B bf16 MLA row; the whole row of a full-width K pool), optionally copy the replacement rows into the consumed
 * free slots (layer_repl == NULL: the caller already prefilled them), and write the new token-level index list.
 */
LEYLINE_API leyline_status leyline_rotate_inplace(leyline_plan_t* plan, void* const* layer_ptrs, const void* const* layer_repl,
                                      int32_t* dev_slot_idx_out, void* cuda_stream);

/*
 * leyline_rotate_inplace_master -- leyline_rotate_inplace with the RE-ANCHOR option: besides
 * the pools the caller keeps, per layer, an fp32 MASTER copy of the rotated band,
 *   layer_master[l]: DEVICE float [pool_slots][rope_heads * rope_dim]  (dense rows, 16-byte aligned).
 * Chained splices round a bf16 K_pe once per turn and the error random-walks (Table 6: rel-L2
 * 4.3e-3 at N=2 -> 2.6e-2 at N=100; the paper's remedy is periodic re-prefill).  Here every rotation is applied to
 * the master in fp32 (fma, error ~2^-24 per turn) and the stored band is re-derived from the master by ONE
 * round-to-nearest-even, so K_pe never carries more than one rounding however often its slot is re-rotated.
 * Rows of C = 0 segments are untouched (band and master).  Replacement rows (layer_repl != NULL) are copied into the
 * pool and their band widened exactly into the master; with layer_repl == NULL the caller fills both.
 * bf16 caches and ROTATE_ONLY plans only (else LEYLINE_E_UNSUPPORTED / LEYLINE_E_INVALID).
 */
LEYLINE_API leyline_status leyline_rotate_inplace_master(leyline_plan_t* plan, void* const* layer_ptrs, void* const* layer_master,
                                             const void* const* layer_repl, int32_t* dev_slot_idx_out, void* cuda_stream);

/*
 * leyline_plan_prefetch -- OPTIONAL: start uploading the plan's device tables (tiles, cos/sin table, page tables,
 * index runs; SURVEY.md section 3(3) "one small H2D copy") on a library-owned copy stream of the CURRENT device and
 * return at once.  The first leyline_splice / leyline_rotate_inplace of the plan then only waits for that copy's
 * event on its own stream instead of issuing the copy there, so the upload overlaps whatever the device is still
 * running (the scheduler plans turn n+1 while turn n executes).  Without this call the tables are uploaded by the
 * first launch, in order on its stream.  Idempotent; a no-op once the tables are on the device.
 * Returns LEYLINE_E_CUDA without a device (the plan itself stays valid and usable for queries).
 */
LEYLINE_API leyline_status leyline_plan_prefetch(leyline_plan_t* plan);

LEYLINE_API void leyline_plan_destroy(leyline_plan_t* plan);
LEYLINE_API const char* leyline_strerror(leyline_status s);
/* Text of the last CUDA error seen by this thread's calls into the library ("" if none). */
LEYLINE_API const char* leyline_last_cuda_error(void);

/* Process-wide default tuning, read by leyline_plan (benchmarking; leyline_plan_ex takes its own). */
LEYLINE_API leyline_status leyline_set_tuning(const leyline_tuning* t);
LEYLINE_API leyline_status leyline_get_tuning(leyline_tuning* t);

/* Device time of the data-moving kernels (a3+a4 / a5) of the plan's last launch, from CUDA events recorded on
 * the launching stream when the plan was created with tuning.profile = 1.  Waits for that launch to finish (only for
 * it: later work on the stream keeps running). */
LEYLINE_API leyline_status leyline_plan_kernel_ms(const leyline_plan_t* plan, float* ms);

/*
 * leyline_probe_band_update -- MEASUREMENT AID, not part of the method: the memory access pattern of step a5 with
 * everything else taken away.  `band_bytes` at byte `band_offset_bytes` of every `row_stride_bytes`-byte row of one
 * contiguous device buffer of n_rows rows are read, changed (an integer add) and written back in place: no page table,
 * no plan, no rotation, full-line 16-byte accesses, 8 independent loads per thread, ctas_per_sm x SM count blocks
 * (0 = 8).  Timing it gives the rate the memory system allows ANY kernel on "128 B of every 1152-B row" (bf16 MLA) or
 * "64 B of every 576-B row" (fp8); bench.py reports it next to k_rotate_band as extras.a5_pattern_probe.  Asynchronous.
 */
LEYLINE_API leyline_status leyline_probe_band_update(void* dev_buf, int64_t n_rows, int64_t row_stride_bytes,
                                                     int32_t band_offset_bytes, int32_t band_bytes, int32_t ctas_per_sm,
                                                     void* cuda_stream);

/* Library / build description, e.g. "leyline-b200 0.2 sm_100a". */
LEYLINE_API const char* leyline_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LEYLINE_H_ */

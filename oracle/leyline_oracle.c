/*
 * oracle/leyline_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, single-threaded CPU definition of what the Leyline splice computes
 * (arxiv/paper_2606_01065; every "PAPER.md:N" below is a line of /root/reference/PAPER.md).
 * It is the checker for the CUDA library under paper_2606_01065_b200/csrc and shares NO code,
 * header, table or helper with it.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this file.  It is never tuned for speed:
 * every token is an explicit loop iteration, every angle is a fresh fp64 libm sin/cos.
 *
 * What is defined here
 *   O1  ora_validate        directive validation        (PAPER.md:98 4-tuple, :409 overlap rejected,
 *                                                        :635 all-or-none)
 *   O2  ora_segments        span list -> segment list   (PAPER.md:98 Delta=|R|-(e-s); :127 steps 1-3;
 *                                                        :405 (a)-(c); :409 left-to-right running shift)
 *   O3  ora_map_*           slot / page maps            (PAPER.md:135 dst_slots, :129 in-place; page rules
 *                                                        M1-M3 are DESIGN.md readings: the paper is
 *                                                        token-slot only)
 *   O4  ora_apply_layer     per-token row move + Eq.(1) (PAPER.md:118-123 K_pe_new = R(Delta) K_pe;
 *                                                        :641 pairing i <-> i+d/2; :133 2i <-> 2i+1;
 *                                                        :650 fp32-or-better trig, downcast on store)
 *   O4' ora_rerope_pair     brute-force re-RoPE R(p+C) R(-p) k, the second independent path
 *                                                       (PAPER.md:110 K_pe[i]=R(i)K_raw[i]; :509)
 *   O5  ora_rotate_master_layer  the re-anchor option: fp32 master of the band, rotated in fp64 and rounded once to
 *                                                       fp32, band = RNE_bf16(master) (reading R1)
 *   codecs                  bf16 / e4m3 <-> fp64, direct round-to-nearest-even from fp64.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): paper's worked example 5+57+9 / stub 11,
 * closure, fresh-RoPE equality, logit preservation, O4 vs O4', 2*pi periods, hand 2x2 rotation,
 * codec sweeps against torch's converters, brute-force list slicing for the maps.
 * Unpinned by the paper (pinned only by the rules in DESIGN.md + brute force): page rules M1-M3,
 * the fp8 cache semantics and the master-band reading R1 ("parity unpinned" by the paper).
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

/* status codes: the numeric values are the ABI contract written in DESIGN.md */
enum { ORA_OK = 0, ORA_E_INVALID = 1, ORA_E_UNSORTED = 2, ORA_E_OVERLAP = 3, ORA_E_RANGE = 4,
       ORA_E_NOFREE = 5, ORA_E_UNSUPPORTED = 6 };
enum { ORA_BF16 = 0, ORA_FP8_E4M3 = 1, ORA_F64 = 2 /* oracle-only un-rounded storage for the pins */ };
enum { ORA_NEOX = 0, ORA_INTERLEAVED = 1 };
enum { ORA_AMORTIZE = 0, ORA_FORGET = 1 };
enum { ORA_KEEP = 0, ORA_INSERT = 1 };

/* ------------------------------------------------------------------ codecs ---- */

/* bf16: 1 sign, 8 exponent (bias 127), 7 mantissa bits = the top half of an IEEE fp32. */
double ora_bf16_decode(uint16_t h) {
    uint32_t u = ((uint32_t)h) << 16;
    float f;
    memcpy(&f, &u, 4);
    return (double)f;
}

/* Direct round-to-nearest-even fp64 -> bf16 (no intermediate fp32 rounding).
 * quantum = 2^(E-7) with E = max(floor(log2|x|), -126); n = rint(|x|/quantum) (default rounding mode =
 * nearest-even, scaling by a power of two is exact); overflow past the largest finite goes to inf. */
uint16_t ora_bf16_encode(double x) {
    uint16_t sign = (uint16_t)(signbit(x) ? 0x8000u : 0u);
    if (isnan(x)) return (uint16_t)(sign | 0x7FC0u);
    double ax = fabs(x);
    if (isinf(ax)) return (uint16_t)(sign | 0x7F80u);
    if (ax == 0.0) return sign;
    int e;
    (void)frexp(ax, &e); /* ax = m * 2^e, m in [0.5,1)  ->  floor(log2 ax) = e-1 */
    int E = e - 1;
    if (E < -126) E = -126;
    double quantum = ldexp(1.0, E - 7);
    double n = nearbyint(ax / quantum);
    double v = n * quantum; /* exactly a bf16 value, or 2^128 on overflow */
    if (v >= ldexp(1.0, 128)) return (uint16_t)(sign | 0x7F80u);
    float f = (float)v; /* exact: v has <= 8 significant bits and fp32's exponent range */
    uint32_t u;
    memcpy(&u, &f, 4);
    return (uint16_t)(sign | (uint16_t)(u >> 16));
}

/* e4m3 ("fn" flavour used for KV caches): 1 sign, 4 exponent (bias 7), 3 mantissa; no inf;
 * S.1111.111 is NaN; largest finite 448 = 1.75 * 2^8; subnormal quantum 2^-9. */
double ora_e4m3_decode(uint8_t b) {
    int s = (b >> 7) & 1, ex = (b >> 3) & 0xF, m = b & 7;
    double v;
    if (ex == 0xF && m == 7) return NAN;
    if (ex == 0) v = ldexp((double)m, -9);
    else v = ldexp(1.0 + (double)m / 8.0, ex - 7);
    return s ? -v : v;
}

/* Direct RNE fp64 -> e4m3 with saturation to +-448 ("satfinite"); never produces NaN from a finite input. */
uint8_t ora_e4m3_encode(double x) {
    uint8_t sign = (uint8_t)(signbit(x) ? 0x80u : 0u);
    if (isnan(x)) return (uint8_t)(sign | 0x7Fu);
    double ax = fabs(x);
    if (ax == 0.0) return sign;
    if (isinf(ax)) return (uint8_t)(sign | 0x7Eu);
    int e;
    (void)frexp(ax, &e);
    int E = e - 1;
    if (E < -6) E = -6;
    double quantum = ldexp(1.0, E - 3);
    double v = nearbyint(ax / quantum) * quantum;
    if (v > 448.0) v = 448.0;
    if (v == 0.0) return sign;
    /* v is exactly representable: find its fields */
    int e2;
    double m2 = frexp(v, &e2); /* v = m2 * 2^e2, m2 in [0.5,1) */
    int E2 = e2 - 1;
    if (E2 < -6) { /* subnormal: v = m * 2^-9 */
        int m = (int)ldexp(v, 9);
        return (uint8_t)(sign | (uint8_t)m);
    }
    int m = (int)((m2 * 2.0 - 1.0) * 8.0);
    return (uint8_t)(sign | (uint8_t)(((E2 + 7) << 3) | m));
}

static int elem_bytes(int dtype) { return dtype == ORA_BF16 ? 2 : dtype == ORA_FP8_E4M3 ? 1 : 8; }

static double load_elem(int dtype, const uint8_t* p, int64_t i, double scale) {
    if (dtype == ORA_BF16) { uint16_t h; memcpy(&h, p + 2 * i, 2); return ora_bf16_decode(h); }
    if (dtype == ORA_FP8_E4M3) return ora_e4m3_decode(p[i]) * scale;
    double d; memcpy(&d, p + 8 * i, 8); return d;
}
static void store_elem(int dtype, uint8_t* p, int64_t i, double v, double scale) {
    if (dtype == ORA_BF16) { uint16_t h = ora_bf16_encode(v); memcpy(p + 2 * i, &h, 2); }
    else if (dtype == ORA_FP8_E4M3) p[i] = ora_e4m3_encode(v / scale);
    else memcpy(p + 8 * i, &v, 8);
}

/* ------------------------------------------------------------------ O1 -------- */

/* Validation, first failure wins, directives visited in the given order:
 *  a. request outside [0,n_req)                         -> RANGE
 *  b. start<0, end<start, repl_len<0, repl_row<0, semantic not in {0,1} -> INVALID
 *  c. end > seq_len[request]                            -> RANGE
 *  d. against the previous directive: request decreases, or same request and start decreases -> UNSORTED;
 *     same request and start < previous end             -> OVERLAP   (adjacency is allowed)
 */
int ora_validate(int32_t n_req, const int64_t* seq_lens, int32_t n_dir, const int32_t* req,
                 const int64_t* start, const int64_t* end, const int64_t* repl_len, const int64_t* repl_row,
                 const int32_t* semantic) {
    if (n_req < 0 || n_dir < 0) return ORA_E_INVALID;
    for (int32_t r = 0; r < n_req; ++r) if (seq_lens[r] < 0) return ORA_E_INVALID;
    for (int32_t d = 0; d < n_dir; ++d) {
        if (req[d] < 0 || req[d] >= n_req) return ORA_E_RANGE;
        if (start[d] < 0 || end[d] < start[d] || repl_len[d] < 0 || repl_row[d] < 0) return ORA_E_INVALID;
        if (semantic[d] != ORA_AMORTIZE && semantic[d] != ORA_FORGET) return ORA_E_INVALID;
        if (end[d] > seq_lens[req[d]]) return ORA_E_RANGE;
        if (d > 0) {
            if (req[d] < req[d - 1]) return ORA_E_UNSORTED;
            if (req[d] == req[d - 1]) {
                if (start[d] < start[d - 1]) return ORA_E_UNSORTED;
                if (start[d] < end[d - 1]) return ORA_E_OVERLAP;
            }
        }
    }
    return ORA_OK;
}

/* ------------------------------------------------------------------ O2 -------- */

/* Segments of ONE request, in new-position order.  Spans are in ORIGINAL token indices,
 * half-open [s,e) (reading G1; forced by Delta = |R| - (e - s) and the -46 example).
 *   running shift C starts at 0 ("running position shift carried over")
 *   KEEP   old [pos, s_j)        -> new [pos + C, s_j + C),  rotation C     (PAPER.md:127 step 3, :405(c))
 *   INSERT r_j replacement rows  -> new [s_j + C, s_j + C + r_j)            (PAPER.md:127 step 2, :405(b))
 *   C += r_j - (e_j - s_j); pos = e_j
 * A FORGET directive truncates the request at its start (new coordinates); nothing after it survives
 * (routed to prefix-trimmed re-prefill; DESIGN.md reading).  Empty segments are omitted.
 * Returns the number of segments; *L_new and *forget_trim (-1 if none) are set. */
int32_t ora_segments(int64_t L_old, int32_t k, const int64_t* start, const int64_t* end, const int64_t* repl_len,
                     const int64_t* repl_row, const int32_t* semantic, int32_t* kind, int64_t* src, int64_t* dst,
                     int64_t* len, int64_t* shift, int64_t* L_new, int64_t* forget_trim) {
    int32_t n = 0;
    int64_t C = 0, pos = 0;
    *forget_trim = -1;
    for (int32_t j = 0; j < k; ++j) {
        if (start[j] > pos) {
            kind[n] = ORA_KEEP; src[n] = pos; dst[n] = pos + C; len[n] = start[j] - pos; shift[n] = C; ++n;
        }
        if (semantic[j] == ORA_FORGET) {
            *L_new = start[j] + C;
            *forget_trim = start[j] + C;
            return n;
        }
        if (repl_len[j] > 0) {
            kind[n] = ORA_INSERT; src[n] = repl_row[j]; dst[n] = start[j] + C; len[n] = repl_len[j]; shift[n] = 0; ++n;
        }
        C += repl_len[j] - (end[j] - start[j]);
        pos = end[j];
    }
    if (L_old > pos) {
        kind[n] = ORA_KEEP; src[n] = pos; dst[n] = pos + C; len[n] = L_old - pos; shift[n] = C; ++n;
    }
    *L_new = L_old + C;
    return n;
}

/* ------------------------------------------------------------------ O3 -------- */

static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

/* First directive of a request, in order, that changes a byte or the running shift: AMORTIZE with a non-empty
 * span or a non-empty replacement.  No-op directives (start == end, |R| = 0) are skipped; a FORGET directive ends
 * the search (everything from its start on is dropped, nothing is rewritten in front of it).
 * Returns that directive's start, or -1 when there is none (DESIGN.md rule M1). */
int64_t ora_first_edit(int32_t k, const int64_t* start, const int64_t* end, const int64_t* repl_len,
                       const int32_t* semantic) {
    for (int32_t j = 0; j < k; ++j) {
        if (semantic[j] == ORA_FORGET) return -1;
        if (end[j] > start[j] || repl_len[j] > 0) return start[j];
    }
    return -1;
}

/* M1 FRESH (the paper's dst_slots path): s0 = ora_first_edit(...); k0 = floor(s0 / P); new
 * table = old pages [0,k0) by identity, then ceil(L_new/P) - k0 ids taken from the free list front to back; old
 * pages [k0, ceil(L_old/P)) are released in ascending logical order and never written.  A request that no directive
 * edits (s0 < 0: no directives, no-ops only, or a FORGET before any edit) keeps its first ceil(L_new/P) pages --
 * all of them unless a FORGET truncated it -- releases the rest, and consumes nothing.
 * Returns ORA_E_NOFREE when the free list is too short. */
int ora_map_fresh(int64_t P, int64_t L_old, int64_t L_new, int64_t s0, const int32_t* old_pages,
                  const int32_t* free_ids, int64_t n_free, int32_t* new_pages, int64_t* n_new_pages,
                  int64_t* n_consumed, int32_t* released, int64_t* n_released) {
    int64_t n_old = ceil_div(L_old, P);
    *n_consumed = 0; *n_released = 0;
    if (s0 < 0) {
        int64_t n_keep = ceil_div(L_new, P); /* L_new <= L_old here: nothing was inserted */
        for (int64_t p = 0; p < n_keep; ++p) new_pages[p] = old_pages[p];
        for (int64_t p = n_keep; p < n_old; ++p) released[(*n_released)++] = old_pages[p];
        *n_new_pages = n_keep;
        return ORA_OK;
    }
    int64_t k0 = s0 / P, n_new = ceil_div(L_new, P);
    if (n_new < k0) n_new = k0; /* cannot happen: L_new >= s0 >= k0*P */
    if (n_new - k0 > n_free) return ORA_E_NOFREE;
    for (int64_t p = 0; p < k0; ++p) new_pages[p] = old_pages[p];
    for (int64_t p = k0; p < n_new; ++p) new_pages[p] = free_ids[(*n_consumed)++];
    for (int64_t p = k0; p < n_old; ++p) released[(*n_released)++] = old_pages[p];
    *n_new_pages = n_new;
    return ORA_OK;
}

/* M2 INPLACE_MOVE: pages [0, min(n_old, n_new)) by identity; growth appends n_new - n_old free ids;
 * shrink releases the tail pages [n_new, n_old) ascending.  Logical position t lives at
 * table[t/P]*P + t%P before and after. */
int ora_map_inplace(int64_t P, int64_t L_old, int64_t L_new, const int32_t* old_pages, const int32_t* free_ids,
                    int64_t n_free, int32_t* new_pages, int64_t* n_new_pages, int64_t* n_consumed,
                    int32_t* released, int64_t* n_released) {
    int64_t n_old = ceil_div(L_old, P), n_new = ceil_div(L_new, P);
    *n_consumed = 0; *n_released = 0;
    if (n_new - n_old > n_free) return ORA_E_NOFREE;
    for (int64_t p = 0; p < n_new; ++p) {
        if (p < n_old) new_pages[p] = old_pages[p];
        else new_pages[p] = free_ids[(*n_consumed)++];
    }
    for (int64_t p = n_new; p < n_old; ++p) released[(*n_released)++] = old_pages[p];
    *n_new_pages = n_new;
    return ORA_OK;
}

/* token-level slot of logical position t under a page table */
int64_t ora_slot_of(int64_t P, const int32_t* pages, int64_t t) { return (int64_t)pages[t / P] * P + t % P; }

/* M3 ROTATE_ONLY (the paper's in-place DynamicCache path; index concat PAPER.md:135):
 * no row moves.  idx_new = for each segment in new-position order: KEEP -> idx_old[src..src+len),
 * INSERT -> the next len free SLOT ids.  Released = idx_old over every removed old position, in order
 * (spans, and everything from a FORGET directive's start).  Token-level even when P > 1. */
int ora_map_rotate_only(int64_t P, int64_t L_old, const int32_t* old_pages, int32_t n_seg, const int32_t* kind,
                        const int64_t* src, const int64_t* dst, const int64_t* len, const int32_t* free_ids,
                        int64_t n_free, int64_t* idx_new, int64_t* n_consumed, int32_t* released,
                        int64_t* n_released) {
    *n_consumed = 0; *n_released = 0;
    int64_t pos = 0; /* next old position not yet accounted for */
    for (int32_t g = 0; g < n_seg; ++g) {
        if (kind[g] == ORA_KEEP) {
            for (int64_t t = pos; t < src[g]; ++t) released[(*n_released)++] = (int32_t)ora_slot_of(P, old_pages, t);
            for (int64_t q = 0; q < len[g]; ++q) idx_new[dst[g] + q] = ora_slot_of(P, old_pages, src[g] + q);
            pos = src[g] + len[g];
        } else {
            if (*n_consumed + len[g] > n_free) return ORA_E_NOFREE;
            for (int64_t q = 0; q < len[g]; ++q) idx_new[dst[g] + q] = free_ids[(*n_consumed)++];
        }
    }
    for (int64_t t = pos; t < L_old; ++t) released[(*n_released)++] = (int32_t)ora_slot_of(P, old_pages, t);
    return ORA_OK;
}

/* ------------------------------------------------------------------ O4 -------- */

/* Standard RoPE rotation of one pair by angle phi (reading G8; Eq.(1) at :118):
 *   a' = a cos(phi) - b sin(phi),   b' = b cos(phi) + a sin(phi)      all in fp64. */
void ora_rotate_pair(double a, double b, double phi, double* a2, double* b2) {
    double c = cos(phi), s = sin(phi);
    *a2 = a * c - b * s;
    *b2 = b * c + a * s;
}

/* O4': brute-force re-RoPE of a pair cached at absolute old position p, moved to p + C:
 * un-rope with R(-p*theta), then rope afresh with R((p+C)*theta). */
void ora_rerope_pair(double a, double b, double p, double C, double theta, double* a2, double* b2) {
    double ra, rb;
    ora_rotate_pair(a, b, -p * theta, &ra, &rb);
    ora_rotate_pair(ra, rb, (p + C) * theta, a2, b2);
}

/* One layer.  old_pool is a pristine snapshot, new_pool a separate buffer (pre-filled by the caller),
 * so no ordering or hazard logic exists here.  slot_old[t] / slot_new[t'] are token-level slots of old /
 * new logical positions.  A row is Dc position-free elements followed by n_heads heads of Dr rotated elements:
 * n_heads = 1 is MLA's K_pe band; n_heads = kv_heads with Dc = 0 is the GQA / MHA degenerate case
 * "qk_nope_head_dim=0 ... rotates the full 128-dim K" ("the rotation must act across
 * all d_K dimensions per token"), every head using the same theta_i (RoPE is applied per head, Su et al.).
 * For every segment, for every token (explicit loop):
 *   latent  : Dc*E bytes copied verbatim, never decoded                     ("K_nope and V preserved")
 *   K_pe    : shift C == 0 -> n_heads*Dr*E bytes verbatim (G19: -0 must survive);
 *             else for every head h, for i in [0,H): pair (i, i+H) NeoX or (2i, 2i+1)
 *             interleaved inside the head,
 *             phi = (double)C * (double)inv_freq[i], rotate in fp64, encode by direct RNE.
 *             fp8: x = decode(byte)*scale, rotate, encode(x'/scale) saturating (G16).
 *   INSERT  : W*E bytes verbatim from the replacement buffer row repl_row+q (its K_pe is already roped
 *             at the final position, G12; PAPER.md:127 step 2).
 * Bytes of a row beyond W*E (row padding) are not touched. */
int ora_apply_layer(int dtype, int pairing, int32_t Dc, int32_t Dr, int32_t n_heads, int64_t stride,
                    const float* inv_freq, float scale_f, const uint8_t* old_pool, uint8_t* new_pool,
                    const uint8_t* repl, int32_t n_seg, const int32_t* kind, const int64_t* src, const int64_t* dst,
                    const int64_t* len, const int64_t* shift, const int64_t* slot_old, const int64_t* slot_new) {
    int E = elem_bytes(dtype);
    int32_t H = Dr / 2;
    double scale = (dtype == ORA_FP8_E4M3) ? (double)scale_f : 1.0;
    if (Dr % 2 != 0 || n_heads < 1) return ORA_E_UNSUPPORTED;
    for (int32_t g = 0; g < n_seg; ++g) {
        for (int64_t q = 0; q < len[g]; ++q) {
            uint8_t* out = new_pool + slot_new[dst[g] + q] * stride;
            if (kind[g] == ORA_INSERT) {
                memcpy(out, repl + (src[g] + q) * stride, (size_t)(Dc + (int64_t)n_heads * Dr) * E);
                continue;
            }
            const uint8_t* in = old_pool + slot_old[src[g] + q] * stride;
            memcpy(out, in, (size_t)Dc * E); /* latent */
            if (shift[g] == 0) {
                memcpy(out + (int64_t)Dc * E, in + (int64_t)Dc * E, (size_t)n_heads * Dr * E);
                continue;
            }
            for (int32_t h = 0; h < n_heads; ++h) {
                const uint8_t* kin = in + ((int64_t)Dc + (int64_t)h * Dr) * E;
                uint8_t* kout = out + ((int64_t)Dc + (int64_t)h * Dr) * E;
                for (int32_t i = 0; i < H; ++i) {
                    int64_t ia = (pairing == ORA_NEOX) ? i : 2 * i;
                    int64_t ib = (pairing == ORA_NEOX) ? i + H : 2 * i + 1;
                    double a = load_elem(dtype, kin, ia, scale), b = load_elem(dtype, kin, ib, scale);
                    double phi = (double)shift[g] * (double)inv_freq[i];
                    double a2, b2;
                    ora_rotate_pair(a, b, phi, &a2, &b2);
                    store_elem(dtype, kout, ia, a2, scale);
                    store_elem(dtype, kout, ib, b2, scale);
                }
            }
        }
    }
    return ORA_OK;
}

/* The RE-ANCHOR option of the in-place path (chained bf16 rotations drift,
 * "periodic re-prefill of the affected slots" is the paper's remedy).  DESIGN.md reading R1: next to the bf16 pool the
 * caller keeps an fp32 master of the rotated band, master[slot][n_heads*Dr]; a ROTATE_ONLY splice
 *   - rotates the master of every downstream token (shift C != 0): exact fp32 inputs, fp64 rotation with fresh libm
 *     sin/cos, ONE rounding to fp32 (the C cast, round-to-nearest-even);
 *   - re-derives the stored band from the NEW master: bf16 = RNE(fp32 value) -- the decision is taken on the fp32
 *     value, the precision both sides hold;
 *   - copies replacement rows into the pool and widens their band exactly into the master;
 *   - leaves C = 0 rows alone.
 * Rows do not move in this mode: slot_new[dst + q] == slot_old[src + q]. */
int ora_rotate_master_layer(int pairing, int32_t Dc, int32_t Dr, int32_t n_heads, int64_t stride, const float* inv_freq,
                            uint8_t* pool, float* master, const uint8_t* repl, int32_t n_seg, const int32_t* kind,
                            const int64_t* src, const int64_t* dst, const int64_t* len, const int64_t* shift,
                            const int64_t* slot_new) {
    int32_t H = Dr / 2;
    int64_t band = (int64_t)n_heads * Dr;
    if (Dr % 2 != 0 || n_heads < 1) return ORA_E_UNSUPPORTED;
    for (int32_t g = 0; g < n_seg; ++g) {
        for (int64_t q = 0; q < len[g]; ++q) {
            int64_t slot = slot_new[dst[g] + q];
            uint8_t* row = pool + slot * stride;
            float* m = master + slot * band;
            if (kind[g] == ORA_INSERT) {
                if (!repl) continue; /* the caller prefills pool and master */
                memcpy(row, repl + (src[g] + q) * stride, (size_t)(Dc + band) * 2);
                for (int64_t e = 0; e < band; ++e) m[e] = (float)load_elem(ORA_BF16, row + (int64_t)Dc * 2, e, 1.0);
                continue;
            }
            if (shift[g] == 0) continue;
            for (int32_t h = 0; h < n_heads; ++h) {
                float* mh = m + (int64_t)h * Dr;
                uint8_t* kout = row + ((int64_t)Dc + (int64_t)h * Dr) * 2;
                for (int32_t i = 0; i < H; ++i) {
                    int64_t ia = (pairing == ORA_NEOX) ? i : 2 * i;
                    int64_t ib = (pairing == ORA_NEOX) ? i + H : 2 * i + 1;
                    double phi = (double)shift[g] * (double)inv_freq[i];
                    double a2, b2;
                    ora_rotate_pair((double)mh[ia], (double)mh[ib], phi, &a2, &b2);
                    mh[ia] = (float)a2;
                    mh[ib] = (float)b2;
                    store_elem(ORA_BF16, kout, ia, (double)mh[ia], 1.0);
                    store_elem(ORA_BF16, kout, ib, (double)mh[ib], 1.0);
                }
            }
        }
    }
    return ORA_OK;
}

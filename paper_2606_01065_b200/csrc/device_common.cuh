/*
 * device_common.cuh -- device helpers shared by the Leyline kernels (sm_100a).
 *
 * The K_pe arithmetic is Eq. (1) of the paper: K_pe_new = R(C) K_pe, applied per RoPE pair
 *   a' = a cos(phi) - b sin(phi),  b' = b cos(phi) + a sin(phi),  phi = C * theta_i,
 * in fp32 with FMA and one round-to-nearest-even on store (the paper's default AKASHA_PIC_ROTATION_FP32=1,
 * PAPER.md:163, :650).  cos/sin come from the launch's table (fp64 product and trig, kept as an fp32 hi + lo pair); on
 * bf16 caches an output whose two products cancel is redone with compensated fp32 arithmetic (rot_comp), so every stored
 * code is within one of the exact result's.  No fast-math, no flush-to-zero.
 */
#ifndef LEYLINE_DEVICE_COMMON_CUH_
#define LEYLINE_DEVICE_COMMON_CUH_

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "plan_internal.h"

namespace leyline {

constexpr int kThreads = 256;
constexpr int kMaxLayers = LEYLINE_MAX_LAYERS_PER_LAUNCH;

struct MoveParams {
    const DevTile* tiles;
    const float* trig;
    const int32_t* tabs;
    unsigned long long* ticket;   /* work counter, zeroed before the launch */
    int32_t* flags;               /* INPLACE_MOVE "loaded" flags [move tile][layer], zeroed before the launch */
    long long n_items;            /* tiles in this launch * layers in this launch */
    long long n_copy_items;       /* k_rotate_band only: replacement-insert tiles * layers, handled after the rotations */
    int32_t copy_tile_begin;      /* k_rotate_band only: first insert tile */
    int32_t n_rot_tiles;          /* k_rotate_band_flat only: rotate tiles [tile_begin, tile_begin + n_rot_tiles) */
    const RotPass* passes;        /* k_rotate_band_flat only: one entry per pass; n_items = passes * layers */
    int64_t stride;               /* row stride in bytes */
    int32_t tile_begin;           /* first tile of this launch in the plan's list */
    int32_t n_layers;             /* layers in this launch */
    int32_t layer0;               /* first layer of this launch (flag index) */
    int32_t n_layers_total;
    int32_t page_shift;
    int32_t H;                    /* rope_dim / 2 */
    int32_t lat_chunks;           /* 16-byte chunks of latent per row */
    int32_t band_chunks;          /* 16-byte chunks of the rotated band per row = n_heads * head_chunks */
    int32_t n_heads;              /* heads in the rotated band (1 for MLA's K_pe; kv_heads for full-width K) */
    int32_t head_chunks;          /* 16-byte chunks per head (rope_dim * elem bytes / 16) */
    const uint8_t* src[kMaxLayers];
    uint8_t* dst[kMaxLayers];
    const uint8_t* repl[kMaxLayers];
};

struct IndexParams {
    const IdxRun* runs;
    const int32_t* tabs;
    int32_t* out;
    long long total;
    int32_t n_runs;
    int32_t page_shift;
};

/* The cos/sin table of the launch, evaluated on the device by the index kernel: row g = cos then sin of
 * shifts[g] * inv_freq[i], i in [0, H) -- fp64 product of the exact integer shift and the fp32 theta_i promoted exactly,
 * fp64 sincos (CUDA math library, <= 2 ulp of fp64, exact argument reduction for |x| up to ~1.3e5 rad here), rounded
 * once to fp32. */
struct TrigParams {
    const int64_t* shifts;
    const float* inv_freq;
    float* out;
    int32_t n_trig;
    int32_t H;
};

/* ---- global memory access ---- */

__device__ __forceinline__ int4 ld_stream(const void* p) { /* read-only for the whole kernel, read once */
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
/* the buffer is also written by this kernel.  HALF_LINE: ask L2 to fetch 64 bytes, not the 128-byte line, on a miss --
 * for bands that are half a line (fp8 MLA: 64 of every 576 bytes), where the other half is latent nobody reads
 * (measured on B200: a5 on config 5 2.86 -> 3.31 TB/s; SASS: LDG.E.NA.LTC64B.128) */
#ifndef LEYLINE_L2_HALF_LINE
#define LEYLINE_L2_HALF_LINE 1 /* 0: measurement builds only (the default 128-byte fetch on half-line bands) */
#endif
template <bool HALF_LINE = false>
__device__ __forceinline__ int4 ld_coherent(const void* p) {
    int4 r;
    if (HALF_LINE && LEYLINE_L2_HALF_LINE)
        asm volatile("ld.global.L1::no_allocate.L2::64B.v4.s32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p) : "memory");
    else
        asm volatile("ld.global.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st_stream(void* p, const int4& v) {
    asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}

/* slot of logical position `pos` through table `tab` of `tabs` (shift = log2 page size, 0 for token-level lists) */
__device__ __forceinline__ int64_t slot_of(const int32_t* __restrict__ tabs, int32_t tab, int64_t pos, int shift) {
    const int64_t page = __ldg(tabs + tab + (pos >> shift));
    return (page << shift) | (pos & ((int64_t(1) << shift) - 1));
}

/* ---- the rotation of one 16-byte chunk of the K_pe band ----
 * NeoX (pair i <-> i+H): `mine` holds elements of one half, `other` the same elements of the other half
 * (fetched from the partner lane); sgn = -1 for the first half (a' = a c - b s), +1 for the second
 * (b' = b c + a s).  cs / sn point at cos / sin of the first element of the chunk.
 * Interleaved (pair 2i <-> 2i+1): both elements of a pair sit in `mine`; cs / sn point at the first pair. */

template <int DT>
struct Codec;

template <>
struct Codec<LEYLINE_BF16> {
    static constexpr int kElems = 8; /* per 16-byte chunk */
    static __device__ __forceinline__ void unpack(const int4& v, float* f) {
        const uint32_t w[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) { /* bf16 -> fp32 is exact: the bits are the top half */
            f[2 * k] = __uint_as_float(w[k] << 16);
            f[2 * k + 1] = __uint_as_float(w[k] & 0xFFFF0000u);
        }
    }
    static __device__ __forceinline__ int4 pack(const float* f) {
        uint32_t w[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const __nv_bfloat162 h = __floats2bfloat162_rn(f[2 * k], f[2 * k + 1]); /* RNE */
            w[k] = *reinterpret_cast<const uint32_t*>(&h);
        }
        return make_int4((int)w[0], (int)w[1], (int)w[2], (int)w[3]);
    }
};

template <>
struct Codec<LEYLINE_FP8_E4M3> {
    static constexpr int kElems = 16;
    static __device__ __forceinline__ void unpack(const int4& v, float* f) {
        const uint32_t w[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
#pragma unroll
            for (int h = 0; h < 2; ++h) { /* e4m3 -> f16 is exact, f16 -> fp32 is exact */
                const __half2_raw r = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)((w[k] >> (16 * h)) & 0xFFFFu), __NV_E4M3);
                const float2 x = __half22float2(*reinterpret_cast<const __half2*>(&r));
                f[4 * k + 2 * h] = x.x;
                f[4 * k + 2 * h + 1] = x.y;
            }
        }
    }
    static __device__ __forceinline__ int4 pack(const float* f) {
        uint32_t w[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { /* RNE, saturate to +-448, never NaN from finite input (G16) */
            const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(f[4 * k], f[4 * k + 1]), __NV_SATFINITE, __NV_E4M3);
            const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(f[4 * k + 2], f[4 * k + 3]), __NV_SATFINITE, __NV_E4M3);
            w[k] = lo | (hi << 16);
        }
        return make_int4((int)w[0], (int)w[1], (int)w[2], (int)w[3]);
    }
};

__device__ __forceinline__ void load_floats(const float* __restrict__ p, float* out, int n) {
    /* p is 16-byte aligned and n a multiple of 4 by construction (H is a multiple of 4) */
#pragma unroll
    for (int k = 0; k < 16; k += 4) {
        if (k < n) {
            const float4 v = __ldg(reinterpret_cast<const float4*>(p + k));
            out[k] = v.x; out[k + 1] = v.y; out[k + 2] = v.z; out[k + 3] = v.w;
        }
    }
}

/* ---- the cos/sin table of a launch ----
 * Row g (one per distinct non-zero shift) = [cos_hi | sin_hi | cos_lo | sin_lo], H floats each: hi = the fp64 value
 * rounded to fp32, lo = (fp64 value - hi) rounded to fp32, so hi + lo carries ~48 bits of cos / sin (k_index writes it). */
constexpr int kTrigParts = 4;
__device__ __forceinline__ const float* trig_row_of(const float* __restrict__ trig, int32_t g, int H) {
    return trig + (int64_t)g * kTrigParts * H;
}

/* ---- THE rotation arithmetic: x*c + y*t, one output element (a' = a c + b (-s), b' = b c + a s) ----
 * The same function of (x, y, cos, sin) in every kernel, so every mode and mover stores the same bits:
 *   plain form   p = fl(x c_hi), r = fl(y t_hi + p) (fma): two fp32 roundings plus the roundings of cos / sin themselves,
 *                absolute error <= ~1.7 * 2^-24 * (|x c| + |y t|) whatever the size of the result;
 *   on bf16 caches, when |r| < 2^-12 |p| -- the two products cancel -- the compensated form instead:
 *                q = fl(y t_hi), e = y t_hi - q exactly (fma), r1 = fl(x c_hi + q) (one rounding of the exact sum), and
 *                the terms left out so far, e + x c_lo + y t_lo, are added last: error ~2^-24 |r| + 2^-47 (|x c| + |y t|).
 * Without cancellation the plain form's error is below 2^-11 |r|, so the stored bf16 code is at most one from the
 * oracle's single rounding of the exact value (the fp32 -> bf16 double rounding); with the fix-up the same holds where the
 * result cancels, and the tolerance needs no cancellation floor (DESIGN.md T).  About one output in 10^4 takes the
 * compensated form, so cos_lo / sin_lo are fetched only then.  e4m3 codes are 2^-3 apart in relative terms and 2^-9 in
 * absolute ones: there the plain form is already within one code. */
#ifndef LEYLINE_COMPENSATE
#define LEYLINE_COMPENSATE 1 /* 0: experiment builds only (what the tests report without the fix-up) */
#endif
template <int DT>
struct Comp { static constexpr bool value = DT == LEYLINE_BF16 && LEYLINE_COMPENSATE != 0; };

__device__ __forceinline__ bool cancels(float r, float p) { return fabsf(r) * 4096.0f < fabsf(p); }

__device__ __forceinline__ float rot_plain(float x, float ch, float y, float th, bool& any) {
    const float p = __fmul_rn(x, ch);
    const float r = __fmaf_rn(y, th, p);
    any |= cancels(r, p);
    return r;
}
__device__ __forceinline__ float rot_comp(float x, float ch, float cl, float y, float th, float tl) {
    const float q = __fmul_rn(y, th);
    const float e = __fmaf_rn(y, th, -q);
    const float r1 = __fmaf_rn(x, ch, q);
    return __fadd_rn(r1, __fmaf_rn(x, cl, __fmaf_rn(y, tl, e)));
}
/* the rare path for one output: r = the plain result already formed from (x, y); cl_at / tl_at -> the lo parts */
__device__ __forceinline__ float rot_fix(float r, float x, float ch, const float* __restrict__ cl_at, float y, float th,
                                         const float* __restrict__ tl_at, float tl_sign) {
    if (cancels(r, __fmul_rn(x, ch))) r = rot_comp(x, ch, __ldg(cl_at), y, th, tl_sign * __ldg(tl_at));
    return r;
}

/* cos / sin registers of one pair column (see rotate_chunk_pair): the hi parts, and the lo parts when LO */
template <int N, bool LO>
struct PairTrig {
    float c[N], s[N], cl[LO ? N : 1], sl[LO ? N : 1];
};

/* NeoX: elements [q*N, q*N+N) of the head's cos / sin.  Interleaved: c[0..N/2) / s[0..N/2) belong to chunk q (pairs
 * q*N/2 ..), c[N/2..N) / s[N/2..N) to chunk q + half (pairs (q+half)*N/2 ..). */
template <int PAIRING, int N>
__device__ __forceinline__ void load_pair_part(const float* __restrict__ cos_row, const float* __restrict__ sin_row, int q, int half,
                                               float* c, float* s) {
    if (PAIRING == LEYLINE_ROPE_NEOX) {
        load_floats(cos_row + q * N, c, N);
        load_floats(sin_row + q * N, s, N);
    } else {
        load_floats(cos_row + q * (N / 2), c, N / 2);
        load_floats(sin_row + q * (N / 2), s, N / 2);
        load_floats(cos_row + (q + half) * (N / 2), c + N / 2, N / 2);
        load_floats(sin_row + (q + half) * (N / 2), s + N / 2, N / 2);
    }
}
template <int PAIRING, int N, bool LO>
__device__ __forceinline__ void load_pair_trig(const float* __restrict__ trig_row, int H, int q, int half, PairTrig<N, LO>& t) {
    load_pair_part<PAIRING, N>(trig_row, trig_row + H, q, half, t.c, t.s);
    if (LO) load_pair_part<PAIRING, N>(trig_row + 2 * H, trig_row + 3 * H, q, half, t.cl, t.sl);
}

/* ---- the rotation of a PAIR of 16-byte chunks held by one thread (no lane exchange) ----
 * NeoX: `lo` = elements [q*N, q*N+N) of a head's first half, `hi` = the same elements of its second half (N pairs).
 * Interleaved: `lo` = chunk q of the head, `hi` = chunk q + half; each holds N/2 whole pairs.
 * t = the hi parts of the column's cos / sin; trig_row / q / half locate the lo parts for the rare compensated outputs.
 * lo_at / hi_at: where the INPUT chunks can be read again (the global or shared memory they were loaded from, not yet
 * overwritten): the rare path re-reads them instead of keeping eight more registers alive in every kernel's main loop. */
template <int DT, int PAIRING>
__device__ __forceinline__ bool rotate_chunk_pair_plain(int4& lo, int4& hi, const PairTrig<Codec<DT>::kElems, false>& t) {
    constexpr int N = Codec<DT>::kElems;
    float a[N], b[N];
    Codec<DT>::unpack(lo, a);
    Codec<DT>::unpack(hi, b);
    bool any = false;
    if (PAIRING == LEYLINE_ROPE_NEOX) {
#pragma unroll
        for (int e = 0; e < N; ++e) {
            const float x = a[e], y = b[e];
            a[e] = rot_plain(x, t.c[e], y, -t.s[e], any);
            b[e] = rot_plain(y, t.c[e], x, t.s[e], any);
        }
    } else {
#pragma unroll
        for (int k = 0; k < N / 2; ++k) {
            const float x0 = a[2 * k], y0 = a[2 * k + 1], x1 = b[2 * k], y1 = b[2 * k + 1];
            a[2 * k] = rot_plain(x0, t.c[k], y0, -t.s[k], any);
            a[2 * k + 1] = rot_plain(y0, t.c[k], x0, t.s[k], any);
            b[2 * k] = rot_plain(x1, t.c[N / 2 + k], y1, -t.s[N / 2 + k], any);
            b[2 * k + 1] = rot_plain(y1, t.c[N / 2 + k], x1, t.s[N / 2 + k], any);
        }
    }
    lo = Codec<DT>::pack(a);
    hi = Codec<DT>::pack(b);
    return any;
}

/* the rare path: the whole chunk pair again from its inputs, every output through the plain form and the fix-up; cos /
 * sin come from the table */
template <int DT, int PAIRING>
__device__ __forceinline__ void rotate_chunk_pair_careful(int4& lo, int4& hi, const float* __restrict__ trig_row, int H, int q, int half,
                                                          const int4 lo_in, const int4 hi_in) {
    constexpr int N = Codec<DT>::kElems;
    float x[N], y[N];
    Codec<DT>::unpack(lo_in, x);
    Codec<DT>::unpack(hi_in, y);
    const float* __restrict__ sn = trig_row + H;
    const float* __restrict__ cl = trig_row + 2 * H;
    const float* __restrict__ sl = trig_row + 3 * H;
    bool unused = false;
    float a[N], b[N];
    if (PAIRING == LEYLINE_ROPE_NEOX) {
#pragma unroll
        for (int e = 0; e < N; ++e) {
            const int i = q * N + e;
            const float c = __ldg(trig_row + i), s = __ldg(sn + i);
            a[e] = rot_fix(rot_plain(x[e], c, y[e], -s, unused), x[e], c, cl + i, y[e], -s, sl + i, -1.0f);
            b[e] = rot_fix(rot_plain(y[e], c, x[e], s, unused), y[e], c, cl + i, x[e], s, sl + i, 1.0f);
        }
    } else {
#pragma unroll
        for (int k = 0; k < N / 2; ++k) {
            const int i0 = q * (N / 2) + k, i1 = (q + half) * (N / 2) + k;
            const float c0 = __ldg(trig_row + i0), s0 = __ldg(sn + i0), c1 = __ldg(trig_row + i1), s1 = __ldg(sn + i1);
            a[2 * k] = rot_fix(rot_plain(x[2 * k], c0, x[2 * k + 1], -s0, unused), x[2 * k], c0, cl + i0, x[2 * k + 1], -s0, sl + i0, -1.0f);
            a[2 * k + 1] = rot_fix(rot_plain(x[2 * k + 1], c0, x[2 * k], s0, unused), x[2 * k + 1], c0, cl + i0, x[2 * k], s0, sl + i0, 1.0f);
            b[2 * k] = rot_fix(rot_plain(y[2 * k], c1, y[2 * k + 1], -s1, unused), y[2 * k], c1, cl + i1, y[2 * k + 1], -s1, sl + i1, -1.0f);
            b[2 * k + 1] = rot_fix(rot_plain(y[2 * k + 1], c1, y[2 * k], s1, unused), y[2 * k + 1], c1, cl + i1, y[2 * k], s1, sl + i1, 1.0f);
        }
    }
    lo = Codec<DT>::pack(a);
    hi = Codec<DT>::pack(b);
}

template <int DT, int PAIRING>
__device__ __forceinline__ void rotate_chunk_pair(int4& lo, int4& hi, const PairTrig<Codec<DT>::kElems, false>& t,
                                                  const float* __restrict__ trig_row, int H, int q, int half,
                                                  const int4* lo_at, const int4* hi_at) {
    if (rotate_chunk_pair_plain<DT, PAIRING>(lo, hi, t) && Comp<DT>::value)
        rotate_chunk_pair_careful<DT, PAIRING>(lo, hi, trig_row, H, q, half, *lo_at, *hi_at);
}

/* The fp32 master band (k_rotate_master): fp32 inputs, always the compensated form (N pairs as for rotate_chunk_pair). */
template <int PAIRING, int N>
__device__ __forceinline__ void rotate_pair_master(float* a, float* b, const PairTrig<N, true>& t) {
    if (PAIRING == LEYLINE_ROPE_NEOX) {
#pragma unroll
        for (int e = 0; e < N; ++e) {
            const float x = a[e], y = b[e];
            a[e] = rot_comp(x, t.c[e], t.cl[e], y, -t.s[e], -t.sl[e]);
            b[e] = rot_comp(y, t.c[e], t.cl[e], x, t.s[e], t.sl[e]);
        }
    } else {
#pragma unroll
        for (int k = 0; k < N / 2; ++k) {
            const float x0 = a[2 * k], y0 = a[2 * k + 1], x1 = b[2 * k], y1 = b[2 * k + 1];
            a[2 * k] = rot_comp(x0, t.c[k], t.cl[k], y0, -t.s[k], -t.sl[k]);
            a[2 * k + 1] = rot_comp(y0, t.c[k], t.cl[k], x0, t.s[k], t.sl[k]);
            b[2 * k] = rot_comp(x1, t.c[N / 2 + k], t.cl[N / 2 + k], y1, -t.s[N / 2 + k], -t.sl[N / 2 + k]);
            b[2 * k + 1] = rot_comp(y1, t.c[N / 2 + k], t.cl[N / 2 + k], x1, t.s[N / 2 + k], t.sl[N / 2 + k]);
        }
    }
}

/* ---- one 16-byte chunk per thread (k_move_rows, k_rotate_band_tma) ----
 * NeoX (pair i <-> i+H): `mine` holds N elements of one half, `other` the same elements of the other half (fetched from
 * the partner lane); sgn = -1 for the first half (a' = a c - b s), +1 for the second (b' = b c + a s).
 * `first` = index of the chunk's first pair in the head's cos / sin. */
template <int DT>
__device__ __forceinline__ int4 rotate_chunk_neox(const int4& mine, const int4& other, const float* __restrict__ trig_row, int H,
                                                  int first, float sgn) {
    constexpr int N = Codec<DT>::kElems;
    float m[N], o[N], c[N], s[N], r[N];
    Codec<DT>::unpack(mine, m);
    Codec<DT>::unpack(other, o);
    load_floats(trig_row + first, c, N);
    load_floats(trig_row + H + first, s, N);
    bool any = false;
#pragma unroll
    for (int e = 0; e < N; ++e) r[e] = rot_plain(m[e], c[e], o[e], sgn * s[e], any);
    if (Comp<DT>::value && any) {
#pragma unroll
        for (int e = 0; e < N; ++e)
            r[e] = rot_fix(r[e], m[e], c[e], trig_row + 2 * H + first + e, o[e], sgn * s[e], trig_row + 3 * H + first + e, sgn);
    }
    return Codec<DT>::pack(r);
}

/* Interleaved (pair 2i <-> 2i+1): both elements of a pair sit in `mine`; `first` = index of the chunk's first pair. */
template <int DT>
__device__ __forceinline__ int4 rotate_chunk_interleaved(const int4& mine, const float* __restrict__ trig_row, int H, int first) {
    constexpr int N = Codec<DT>::kElems;
    float m[N], c[N / 2], s[N / 2], r[N];
    Codec<DT>::unpack(mine, m);
    load_floats(trig_row + first, c, N / 2);
    load_floats(trig_row + H + first, s, N / 2);
    bool any = false;
#pragma unroll
    for (int k = 0; k < N / 2; ++k) {
        r[2 * k] = rot_plain(m[2 * k], c[k], m[2 * k + 1], -s[k], any);
        r[2 * k + 1] = rot_plain(m[2 * k + 1], c[k], m[2 * k], s[k], any);
    }
    if (Comp<DT>::value && any) {
#pragma unroll
        for (int k = 0; k < N / 2; ++k) {
            const float* cl = trig_row + 2 * H + first + k;
            const float* sl = trig_row + 3 * H + first + k;
            r[2 * k] = rot_fix(r[2 * k], m[2 * k], c[k], cl, m[2 * k + 1], -s[k], sl, -1.0f);
            r[2 * k + 1] = rot_fix(r[2 * k + 1], m[2 * k + 1], c[k], cl, m[2 * k], s[k], sl, 1.0f);
        }
    }
    return Codec<DT>::pack(r);
}

__device__ __forceinline__ int4 shfl_xor_int4(const int4& v, int lane_mask) {
    return make_int4(__shfl_xor_sync(0xFFFFFFFFu, v.x, lane_mask), __shfl_xor_sync(0xFFFFFFFFu, v.y, lane_mask),
                     __shfl_xor_sync(0xFFFFFFFFu, v.z, lane_mask), __shfl_xor_sync(0xFFFFFFFFu, v.w, lane_mask));
}

/* Rotate band chunk j (0 .. nb-1) of a row.  All 32 lanes of the warp must call this together (the NeoX
 * partner chunk j ^ nb/2 is held by lane ^ nb/2); lanes without a valid chunk pass active = false. */
template <int DT, int PAIRING>
__device__ __forceinline__ int4 rotate_band_chunk(const int4& mine, int j, int nb, const float* __restrict__ trig_row,
                                                  int H, bool active) {
    constexpr int N = Codec<DT>::kElems;
    if (PAIRING == LEYLINE_ROPE_NEOX) {
        const int half = nb >> 1;
        const int4 other = shfl_xor_int4(mine, half);
        if (!active) return mine;
        const int jj = j & (half - 1);
        return rotate_chunk_neox<DT>(mine, other, trig_row, H, jj * N, j < half ? -1.0f : 1.0f);
    } else {
        if (!active) return mine;
        return rotate_chunk_interleaved<DT>(mine, trig_row, H, j * (N / 2));
    }
}

}  // namespace leyline

#endif /* LEYLINE_DEVICE_COMMON_CUH_ */

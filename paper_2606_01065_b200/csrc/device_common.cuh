/*
 * device_common.cuh -- device helpers shared by the Leyline kernels (sm_100a).
 *
 * The K_pe arithmetic is Eq. (1) of the paper: K_pe_new = R(C) K_pe, applied per RoPE pair
 *   a' = a cos(phi) - b sin(phi),  b' = b cos(phi) + a sin(phi),  phi = C * theta_i,
 * in fp32 with FMA and one round-to-nearest-even on store (the paper's default AKASHA_PIC_ROTATION_FP32=1,
 * PAPER.md:163, :650).  cos/sin come from the plan's table (fp64 product and trig, rounded once to fp32).
 * No fast-math, no flush-to-zero.
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
    int32_t pad0_;
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
__device__ __forceinline__ int4 ld_coherent(const void* p) { /* the buffer is also written by this kernel */
    int4 r;
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

template <int DT>
__device__ __forceinline__ int4 rotate_chunk_neox(const int4& mine, const int4& other, const float* __restrict__ cs,
                                                  const float* __restrict__ sn, float sgn) {
    constexpr int N = Codec<DT>::kElems;
    float m[N], o[N], c[N], s[N];
    Codec<DT>::unpack(mine, m);
    Codec<DT>::unpack(other, o);
    load_floats(cs, c, N);
    load_floats(sn, s, N);
#pragma unroll
    for (int e = 0; e < N; ++e) m[e] = __fmaf_rn(o[e], sgn * s[e], m[e] * c[e]);
    return Codec<DT>::pack(m);
}

template <int DT>
__device__ __forceinline__ int4 rotate_chunk_interleaved(const int4& mine, const float* __restrict__ cs,
                                                         const float* __restrict__ sn) {
    constexpr int N = Codec<DT>::kElems;
    float m[N], c[N / 2], s[N / 2], r[N];
    Codec<DT>::unpack(mine, m);
    load_floats(cs, c, N / 2);
    load_floats(sn, s, N / 2);
#pragma unroll
    for (int q = 0; q < N / 2; ++q) {
        const float a = m[2 * q], b = m[2 * q + 1];
        r[2 * q] = __fmaf_rn(b, -s[q], a * c[q]);
        r[2 * q + 1] = __fmaf_rn(a, s[q], b * c[q]);
    }
    return Codec<DT>::pack(r);
}

/* ---- the rotation of a PAIR of 16-byte chunks held by one thread (no lane exchange) ----
 * NeoX: `lo` = elements [q*N, q*N+N) of a head's first half, `hi` = the same elements of its second half;
 *       c / s = cos / sin of those N pairs (trig_row + q*N, trig_row + H + q*N).
 * Interleaved: `lo` = chunk q of the head, `hi` = chunk q + half; each holds N/2 whole pairs;
 *       c[0..N/2) / s[0..N/2) belong to lo (pairs q*N/2 ..), c[N/2..N) / s[N/2..N) to hi (pairs (q+half)*N/2 ..).
 * Same fp32 expressions as rotate_chunk_neox / rotate_chunk_interleaved: a' = fma(b, -s, a*c), b' = fma(a, s, b*c). */
/* The fp32 arithmetic of one (lo, hi) chunk pair: N elements each, cos / sin as described above. */
template <int PAIRING, int N>
__device__ __forceinline__ void rotate_pair_f32(float* a, float* b, const float* c, const float* s) {
    if (PAIRING == LEYLINE_ROPE_NEOX) {
#pragma unroll
        for (int e = 0; e < N; ++e) {
            const float x = a[e], y = b[e];
            a[e] = __fmaf_rn(y, -s[e], x * c[e]);
            b[e] = __fmaf_rn(x, s[e], y * c[e]);
        }
    } else {
#pragma unroll
        for (int q = 0; q < N / 2; ++q) {
            const float x0 = a[2 * q], y0 = a[2 * q + 1], x1 = b[2 * q], y1 = b[2 * q + 1];
            a[2 * q] = __fmaf_rn(y0, -s[q], x0 * c[q]);
            a[2 * q + 1] = __fmaf_rn(x0, s[q], y0 * c[q]);
            b[2 * q] = __fmaf_rn(y1, -s[N / 2 + q], x1 * c[N / 2 + q]);
            b[2 * q + 1] = __fmaf_rn(x1, s[N / 2 + q], y1 * c[N / 2 + q]);
        }
    }
}

template <int DT, int PAIRING>
__device__ __forceinline__ void rotate_chunk_pair(int4& lo, int4& hi, const float* c, const float* s) {
    constexpr int N = Codec<DT>::kElems;
    float a[N], b[N];
    Codec<DT>::unpack(lo, a);
    Codec<DT>::unpack(hi, b);
    rotate_pair_f32<PAIRING, N>(a, b, c, s);
    lo = Codec<DT>::pack(a);
    hi = Codec<DT>::pack(b);
}

/* cos / sin registers for pair column q of a head (see rotate_chunk_pair): N floats each. */
template <int DT, int PAIRING>
__device__ __forceinline__ void load_pair_trig(const float* __restrict__ trig_row, int H, int q, int half, float* c, float* s) {
    constexpr int N = Codec<DT>::kElems;
    if (PAIRING == LEYLINE_ROPE_NEOX) {
        load_floats(trig_row + q * N, c, N);
        load_floats(trig_row + H + q * N, s, N);
    } else {
        load_floats(trig_row + q * (N / 2), c, N / 2);
        load_floats(trig_row + H + q * (N / 2), s, N / 2);
        load_floats(trig_row + (q + half) * (N / 2), c + N / 2, N / 2);
        load_floats(trig_row + H + (q + half) * (N / 2), s + N / 2, N / 2);
    }
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
        const float sgn = j < half ? -1.0f : 1.0f;
        return rotate_chunk_neox<DT>(mine, other, trig_row + jj * N, trig_row + H + jj * N, sgn);
    } else {
        if (!active) return mine;
        return rotate_chunk_interleaved<DT>(mine, trig_row + j * (N / 2), trig_row + H + j * (N / 2));
    }
}

}  // namespace leyline

#endif /* LEYLINE_DEVICE_COMMON_CUH_ */

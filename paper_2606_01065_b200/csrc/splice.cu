/*
 * splice.cu -- leyline_splice / leyline_rotate_inplace: upload the plan's tables once, then launch
 * the index rewrite (a2) and the fused gather -> rotate -> scatter (+ insert) kernels (a3, a4, a5) on the
 * caller's stream.  No synchronisation, no CPU fallback: every failure is a LEYLINE_E_CUDA status.
 */
#include <cstdio>
#include <algorithm>
#include <cstring>
#include <deque>
#include <mutex>
#include <string>
#include <vector>

#include <cudaTypedefs.h> /* PFN_cuTensorMapEncodeTiled */

#include "kernels_band_tma.cuh"
#include "kernels_bulk.cuh"
#include "kernels_rows.cuh"

using namespace leyline;

namespace {

thread_local std::string g_last_error;

bool cuda_ok(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return true;
    g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
    (void)cudaGetLastError(); /* clear the sticky-less error state */
    return false;
}
#define CU(call) do { if (!cuda_ok((call), #call)) return LEYLINE_E_CUDA; } while (0)

inline int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

struct DeviceInfo { int device = -1; int sms = 0; int smem_optin = 0; };
thread_local DeviceInfo g_dev; /* per host thread: callers may drive different devices from different threads */

/* ---- pinned staging for the plan upload ----
 * A pageable source makes the runtime stage the tables itself (an extra host copy, and a DMA that cannot start
 * before it); at 48 B per 32-row tile that upload is the largest fixed cost of a call.  Buffers are recycled: each
 * goes back to the pool right after its copy is enqueued, guarded by an event the next user checks. */
struct PinnedBuf { void* p = nullptr; size_t cap = 0; cudaEvent_t ev = nullptr; int device = -1; };
std::mutex g_pin_mu;
std::vector<PinnedBuf> g_pin_pool;
constexpr size_t kPinMinBytes = 256 << 10, kPinMaxPooled = 32;
constexpr int kPinPrefill = 5;
/* The pool is bounded in BYTES as well as in buffers: only small size classes are stocked ahead (a plan with tens of MB
 * of tables would otherwise pin six times that in one call, six device-stalling cudaHostAlloc calls back to back), the
 * pool keeps at most kPinMaxPooledBytes, and a buffer of more than kPinMaxKeptCap is freed when its copy is done. */
constexpr size_t kPinPrefillMaxCap = size_t(4) << 20, kPinMaxPooledBytes = size_t(256) << 20, kPinMaxKeptCap = size_t(64) << 20;
size_t g_pin_pool_bytes = 0; /* sum of cap over g_pin_pool, under g_pin_mu */

PinnedBuf pin_acquire(size_t bytes, int dev) {
    {
        std::lock_guard<std::mutex> lk(g_pin_mu);
        for (size_t i = 0; i < g_pin_pool.size(); ++i) {
            PinnedBuf b = g_pin_pool[i];
            if (b.cap >= bytes && b.device == dev && cudaEventQuery(b.ev) == cudaSuccess) {
                g_pin_pool.erase(g_pin_pool.begin() + (long)i);
                g_pin_pool_bytes -= b.cap;
                return b;
            }
        }
        (void)cudaGetLastError(); /* cudaErrorNotReady from a busy buffer is not an error */
    }
    size_t cap = kPinMinBytes;
    while (cap < bytes) cap <<= 1;
    auto make = [&](PinnedBuf& b) {
        if (cudaHostAlloc(&b.p, cap, cudaHostAllocDefault) != cudaSuccess ||
            cudaEventCreateWithFlags(&b.ev, cudaEventDisableTiming) != cudaSuccess) {
            (void)cudaGetLastError();
            if (b.p) cudaFreeHost(b.p);
            b = PinnedBuf{};
            return false;
        }
        b.cap = cap;
        b.device = dev;
        return true;
    };
    PinnedBuf b;
    if (!make(b)) return PinnedBuf{}; /* caller falls back to a pageable source */
    /* cudaHostAlloc waits for the device and takes milliseconds: when this size class runs dry, stock it for the calls
     * that follow (a server keeps a few plans in flight), so that the stall is paid once, not once per concurrent plan */
    for (int extra = 0; extra < kPinPrefill && cap <= kPinPrefillMaxCap; ++extra) {
        PinnedBuf e;
        if (!make(e)) break;
        std::lock_guard<std::mutex> lk(g_pin_mu);
        if (g_pin_pool.size() >= kPinMaxPooled || g_pin_pool_bytes + cap > kPinMaxPooledBytes) {
            cudaEventDestroy(e.ev);
            cudaFreeHost(e.p);
            break;
        }
        g_pin_pool.push_back(e);
        g_pin_pool_bytes += cap;
    }
    return b;
}

void pin_release(PinnedBuf b, cudaStream_t stream) {
    cudaEventRecord(b.ev, stream);
    {
        std::lock_guard<std::mutex> lk(g_pin_mu);
        if (g_pin_pool.size() < kPinMaxPooled && b.cap <= kPinMaxKeptCap && g_pin_pool_bytes + b.cap <= kPinMaxPooledBytes) {
            g_pin_pool.push_back(b);
            g_pin_pool_bytes += b.cap;
            return;
        }
    }
    /* over the bound, or an oversized buffer: freed once its copy has finished (outside the lock) */
    cudaEventSynchronize(b.ev);
    cudaEventDestroy(b.ev);
    cudaFreeHost(b.p);
}

/* ---- device memory for the plan tables ----
 * A pool of its own: allocations made on the copy stream (leyline_plan_prefetch) must never pick up a dependency
 * on the work of the stream that freed the previous plan's tables, which the default pool is allowed to insert. */
constexpr size_t kPlanPoolReserveBytes = 128u << 20;
struct PlanPool { int device = -1; cudaMemPool_t pool = nullptr; cudaStream_t copy_stream = nullptr; };
std::deque<PlanPool> g_plan_pools; /* deque: references stay valid as devices are added */

PlanPool* plan_pool(int dev) {
    std::lock_guard<std::mutex> lk(g_pin_mu);
    for (auto& pp : g_plan_pools)
        if (pp.device == dev) return &pp;
    PlanPool pp;
    pp.device = dev;
    cudaMemPoolProps props;
    std::memset(&props, 0, sizeof(props));
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    if (cudaMemPoolCreate(&pp.pool, &props) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
    int off = 0;
    unsigned long long keep = ~0ull; /* keep freed blocks cached: a plan per turn is the steady state */
    cudaMemPoolSetAttribute(pp.pool, cudaMemPoolReuseAllowInternalDependencies, &off);
    cudaMemPoolSetAttribute(pp.pool, cudaMemPoolAttrReleaseThreshold, &keep);
    if (cudaStreamCreateWithFlags(&pp.copy_stream, cudaStreamNonBlocking) != cudaSuccess) {
        (void)cudaGetLastError();
        cudaMemPoolDestroy(pp.pool);
        return nullptr;
    }
    /* Growing the pool (cuMemCreate + map) stalls every stream of the device for tens of ms, and it would happen at some
     * later call, whenever one more plan is in flight than ever before: reserve once, now.  The block goes straight back
     * to the pool, which keeps it (release threshold above) and carves the plans' tables out of it. */
    void* reserve = nullptr;
    if (cudaMallocFromPoolAsync(&reserve, kPlanPoolReserveBytes, pp.pool, pp.copy_stream) == cudaSuccess) {
        cudaFreeAsync(reserve, pp.copy_stream);
        cudaStreamSynchronize(pp.copy_stream);
    }
    (void)cudaGetLastError();
    g_plan_pools.push_back(pp);
    return &g_plan_pools.back();
}

leyline_status device_info(int* dev_out) {
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (g_dev.device != dev) {
        int sms = 0, optin = 0;
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        CU(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        g_dev.device = dev;
        g_dev.sms = sms;
        g_dev.smem_optin = optin;
    }
    *dev_out = dev;
    return LEYLINE_OK;
}

/* Allocate tables + scratch, copy the tables and zero the scratch, all stream-ordered on `stream`. */
leyline_status upload_tables(leyline_plan_s* pl, int dev, cudaStream_t stream) {
    /* one allocation: shifts | inv_freq | tiles | tabs | slot_runs | page_runs (uploaded) | trig (written by k_index) |
     * scratch, each 256-byte aligned */
    int64_t off = 0;
    auto place = [&](int64_t bytes) { int64_t o = off; off = align_up(off + bytes, 256); return o; };
    pl->off_shifts = place((int64_t)pl->trig_shifts.size() * sizeof(int64_t));
    pl->off_inv_freq = place((int64_t)pl->inv_freq.size() * sizeof(float));
    pl->off_tiles = place((int64_t)pl->tiles.size() * sizeof(DevTile));
    pl->off_tabs = place((int64_t)pl->tabs.size() * sizeof(int32_t));
    pl->off_slot_runs = place((int64_t)pl->slot_runs.size() * sizeof(IdxRun));
    pl->off_page_runs = place((int64_t)pl->page_runs.size() * sizeof(IdxRun));
    pl->off_rot_passes = place((int64_t)pl->rot_passes.size() * sizeof(leyline::RotPass));
    const int64_t upload_bytes = off > 0 ? off : 256;
    pl->off_trig = place((int64_t)pl->trig_shifts.size() * kTrigParts * (int64_t)pl->inv_freq.size() * sizeof(float)); /* cos, sin: hi and lo parts */
    pl->blob_bytes = off > 0 ? off : 256;
    const int64_t n_flags = pl->mode == LEYLINE_INPLACE_MOVE ? pl->info.n_tiles * pl->desc.n_layers : 0;
    pl->scratch_bytes = 256 + align_up(n_flags * (int64_t)sizeof(int32_t), 256);
    PinnedBuf pin = pin_acquire((size_t)upload_bytes, dev);
    std::string pageable;
    if (!pin.p) pageable.resize((size_t)upload_bytes);
    uint8_t* host = pin.p ? static_cast<uint8_t*>(pin.p) : reinterpret_cast<uint8_t*>(&pageable[0]);
    auto put = [&](int64_t o, const void* src, size_t bytes) { if (bytes) std::memcpy(host + o, src, bytes); };
    put(pl->off_shifts, pl->trig_shifts.data(), pl->trig_shifts.size() * sizeof(int64_t));
    put(pl->off_inv_freq, pl->inv_freq.data(), pl->inv_freq.size() * sizeof(float));
    put(pl->off_tiles, pl->tiles.data(), pl->tiles.size() * sizeof(DevTile));
    put(pl->off_tabs, pl->tabs.data(), pl->tabs.size() * sizeof(int32_t));
    put(pl->off_slot_runs, pl->slot_runs.data(), pl->slot_runs.size() * sizeof(IdxRun));
    put(pl->off_page_runs, pl->page_runs.data(), pl->page_runs.size() * sizeof(IdxRun));
    put(pl->off_rot_passes, pl->rot_passes.data(), pl->rot_passes.size() * sizeof(leyline::RotPass));
    PlanPool* pp = plan_pool(dev);
    const size_t total = (size_t)(pl->blob_bytes + pl->scratch_bytes);
    const cudaError_t e = pp ? cudaMallocFromPoolAsync(&pl->d_blob, total, pp->pool, stream) : cudaMallocAsync(&pl->d_blob, total, stream);
    if (!cuda_ok(e, "cudaMallocAsync(plan tables)")) {
        if (pin.p) pin_release(pin, stream);
        pl->d_blob = nullptr;
        return LEYLINE_E_CUDA;
    }
    pl->d_scratch = static_cast<uint8_t*>(pl->d_blob) + pl->blob_bytes;
    /* pinned source: a plain stream-ordered DMA; pageable fallback: the runtime stages it before returning */
    bool ok = cuda_ok(cudaMemcpyAsync(pl->d_blob, host, (size_t)upload_bytes, cudaMemcpyHostToDevice, stream),
                      "cudaMemcpyAsync(plan tables)");
    if (pin.p) pin_release(pin, stream);
    ok = ok && cuda_ok(cudaMemsetAsync(pl->d_scratch, 0, (size_t)pl->scratch_bytes, stream), "cudaMemsetAsync(scratch)");
    if (!ok) return LEYLINE_E_CUDA;
    pl->scratch_clean = true;
    pl->device = dev;
    return LEYLINE_OK;
}

leyline_status ensure_device(leyline_plan_s* pl, cudaStream_t stream) {
    int dev = 0;
    leyline_status st = device_info(&dev);
    if (st != LEYLINE_OK) return st;
    if (pl->d_blob || pl->device >= 0) {
        if (pl->device != dev) { g_last_error = "plan was uploaded on another device"; return LEYLINE_E_CUDA; }
        /* prefetched tables: order this stream after the copy (cheap once the event has completed) */
        if (pl->ev_uploaded) CU(cudaStreamWaitEvent(stream, static_cast<cudaEvent_t>(pl->ev_uploaded), 0));
        return LEYLINE_OK;
    }
    return upload_tables(pl, dev, stream);
}

template <class T>
const T* blob_at(const leyline_plan_s* pl, int64_t off) {
    return reinterpret_cast<const T*>(static_cast<const uint8_t*>(pl->d_blob) + off);
}

IndexParams index_params(const leyline_plan_s* pl, const std::vector<IdxRun>& runs, int64_t off, int32_t* out) {
    IndexParams ip;
    std::memset(&ip, 0, sizeof(ip));
    if (!out || runs.empty()) return ip;
    ip.runs = blob_at<IdxRun>(pl, off);
    ip.tabs = blob_at<int32_t>(pl, pl->off_tabs);
    ip.out = out;
    ip.total = runs.back().out_begin + runs.back().length;
    ip.n_runs = (int32_t)runs.size();
    ip.page_shift = pl->page_shift;
    return ip;
}

/* a2: page-table rows and token-level slot list (either output may be NULL), and the cos/sin table the data kernel
 * behind it reads, in ONE launch. */
leyline_status launch_index(leyline_plan_s* pl, int32_t* page_table_out, int32_t* slot_idx_out, cudaStream_t stream) {
    const IndexParams a = index_params(pl, pl->page_runs, pl->off_page_runs, page_table_out);
    const IndexParams b = index_params(pl, pl->slot_runs, pl->off_slot_runs, slot_idx_out);
    TrigParams tp;
    tp.shifts = blob_at<int64_t>(pl, pl->off_shifts);
    tp.inv_freq = blob_at<float>(pl, pl->off_inv_freq);
    tp.out = const_cast<float*>(blob_at<float>(pl, pl->off_trig));
    tp.n_trig = pl->trig_ready ? 0 : (int32_t)pl->trig_shifts.size(); /* a relaunched plan keeps its table */
    tp.H = (int32_t)pl->inv_freq.size();
    auto blocks_of = [](const IndexParams& ip) {
        long long n = (ip.total + kThreads - 1) / kThreads;
        return n > 4LL * g_dev.sms ? 4LL * g_dev.sms : n;
    };
    const long long na = blocks_of(a), nb = blocks_of(b), nt = ((long long)tp.n_trig * tp.H + kThreads - 1) / kThreads;
    if (na + nb + nt == 0) return LEYLINE_OK;
    k_index<<<(unsigned)(na + nb + nt), kThreads, 0, stream>>>(a, b, tp, (int)na, (int)nb);
    CU(cudaGetLastError());
    pl->trig_ready = true;
    return LEYLINE_OK;
}

using MoveKernel = void (*)(const MoveParams);

template <int DT, int PAIRING, bool HAZARD>
MoveKernel pick_move_geom(const leyline_plan_s* pl) {
    const int lc = pl->desc.latent_dim * pl->elem_bytes / 16, nb = pl->head_chunks; /* row kernel: one head */
    if (DT == LEYLINE_BF16 && lc == 64 && nb == 8) return k_move_rows<DT, PAIRING, HAZARD, 64, 8>;
    if (DT == LEYLINE_FP8_E4M3 && lc == 32 && nb == 4) return k_move_rows<DT, PAIRING, HAZARD, 32, 4>;
    return k_move_rows<DT, PAIRING, HAZARD, -1, -1>;
}
template <int DT, int PAIRING>
MoveKernel pick_move_hazard(const leyline_plan_s* pl, bool hazard) {
    return hazard ? pick_move_geom<DT, PAIRING, true>(pl) : pick_move_geom<DT, PAIRING, false>(pl);
}
MoveKernel pick_move(const leyline_plan_s* pl, int pairing, bool hazard) {
    const bool neox = pairing == LEYLINE_ROPE_NEOX;
    if (pl->desc.dtype == LEYLINE_BF16)
        return neox ? pick_move_hazard<LEYLINE_BF16, LEYLINE_ROPE_NEOX>(pl, hazard)
                    : pick_move_hazard<LEYLINE_BF16, LEYLINE_ROPE_INTERLEAVED>(pl, hazard);
    return neox ? pick_move_hazard<LEYLINE_FP8_E4M3, LEYLINE_ROPE_NEOX>(pl, hazard)
                : pick_move_hazard<LEYLINE_FP8_E4M3, LEYLINE_ROPE_INTERLEAVED>(pl, hazard);
}

using BulkKernel = void (*)(const MoveParams, int, int, int, int, int);

template <int DT>
BulkKernel pick_bulk_dt(int pairing, bool hazard) {
    const bool neox = pairing == LEYLINE_ROPE_NEOX;
    if (hazard) return neox ? k_move_bulk<DT, LEYLINE_ROPE_NEOX, true> : k_move_bulk<DT, LEYLINE_ROPE_INTERLEAVED, true>;
    return neox ? k_move_bulk<DT, LEYLINE_ROPE_NEOX, false> : k_move_bulk<DT, LEYLINE_ROPE_INTERLEAVED, false>;
}
BulkKernel pick_bulk(const leyline_plan_s* pl, int pairing, bool hazard) {
    return pl->desc.dtype == LEYLINE_BF16 ? pick_bulk_dt<LEYLINE_BF16>(pairing, hazard) : pick_bulk_dt<LEYLINE_FP8_E4M3>(pairing, hazard);
}

template <int DT>
MoveKernel pick_rotate_dt(int pairing, bool fixed) {
    const bool neox = pairing == LEYLINE_ROPE_NEOX;
    if (fixed) return neox ? k_rotate_band<DT, LEYLINE_ROPE_NEOX, true> : k_rotate_band<DT, LEYLINE_ROPE_INTERLEAVED, true>;
    return neox ? k_rotate_band<DT, LEYLINE_ROPE_NEOX, false> : k_rotate_band<DT, LEYLINE_ROPE_INTERLEAVED, false>;
}
/* a5.  FIXED when the pair columns of a row divide the block (a thread then keeps one column and its cos/sin). */
MoveKernel pick_rotate(const leyline_plan_s* pl, int pairing) {
    const int cols = pl->n_heads * (pl->head_chunks / 2);
    const bool fixed = cols <= kThreads && kThreads % cols == 0;
    return pl->desc.dtype == LEYLINE_BF16 ? pick_rotate_dt<LEYLINE_BF16>(pairing, fixed) : pick_rotate_dt<LEYLINE_FP8_E4M3>(pairing, fixed);
}
/* a5 on short segments (plan.cpp sets rotate_flat only for the FIXED geometry) */
MoveKernel pick_rotate_flat(const leyline_plan_s* pl, int pairing) {
    const bool neox = pairing == LEYLINE_ROPE_NEOX;
    if (pl->desc.dtype == LEYLINE_BF16)
        return neox ? k_rotate_band_flat<LEYLINE_BF16, LEYLINE_ROPE_NEOX> : k_rotate_band_flat<LEYLINE_BF16, LEYLINE_ROPE_INTERLEAVED>;
    return neox ? k_rotate_band_flat<LEYLINE_FP8_E4M3, LEYLINE_ROPE_NEOX> : k_rotate_band_flat<LEYLINE_FP8_E4M3, LEYLINE_ROPE_INTERLEAVED>;
}

}  // namespace

namespace {

struct OccCache { const void* fn; int smem; int blocks; };
thread_local OccCache g_occ[64];
thread_local int g_occ_n = 0;

int occupancy(const void* fn, int smem) {
    for (int i = 0; i < g_occ_n; ++i)
        if (g_occ[i].fn == fn && g_occ[i].smem == smem) return g_occ[i].blocks;
    int blocks = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks, fn, kThreads, (size_t)smem) != cudaSuccess || blocks < 1) {
        (void)cudaGetLastError();
        blocks = 1;
    }
    if (g_occ_n < 64) g_occ[g_occ_n++] = {fn, smem, blocks};
    return blocks;
}

/* Static shared memory of a kernel and the dynamic size it was last opted in for (per host thread and device): asking the
 * runtime for both on every launch cost ~8 us of a ~25 us call. */
struct SmemCache { const void* fn; int device; int static_bytes; int dyn_set; };  /* dyn_set: -1 until opted in */
thread_local SmemCache g_smem[32];
thread_local int g_smem_n = 0;

leyline_status smem_entry(const void* fn, SmemCache** out) {
    for (int i = 0; i < g_smem_n; ++i)
        if (g_smem[i].fn == fn && g_smem[i].device == g_dev.device) { *out = &g_smem[i]; return LEYLINE_OK; }
    cudaFuncAttributes fa;
    CU(cudaFuncGetAttributes(&fa, fn));
    if (g_smem_n == 32) g_smem_n = 0; /* more kernel variants than slots: start over */
    g_smem[g_smem_n] = {fn, g_dev.device, (int)fa.sharedSizeBytes, -1};
    *out = &g_smem[g_smem_n++];
    return LEYLINE_OK;
}
/* Opt the kernel in for ALL the dynamic shared memory the device allows, once: the attribute belongs to the function, not
 * to this thread, so a per-launch size cached here could be lowered behind our back by another thread's launch. */
leyline_status smem_opt_in(SmemCache* e) {
    const int dyn_bytes = g_dev.smem_optin - e->static_bytes;
    if (e->dyn_set == dyn_bytes) return LEYLINE_OK;
    CU(cudaFuncSetAttribute(e->fn, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_bytes));
    e->dyn_set = dyn_bytes;
    return LEYLINE_OK;
}

/* Layers that one launch can serve: same pairing convention ("per layer"; G20), at most kMaxLayers.
 * `flag_base` numbers the launch's layers uniquely inside the call (hazard-flag column). */
struct LayerChunk { int pairing; int flag_base; std::vector<int> layers; };

std::vector<LayerChunk> layer_chunks(const leyline_plan_s* pl, size_t kMaxLayers = leyline::kMaxLayers) {
    std::vector<LayerChunk> out;
    const int L = pl->desc.n_layers;
    int base = 0;
    for (int conv = 0; conv < 2; ++conv) {
        std::vector<int> mine;
        for (int l = 0; l < L; ++l)
            if ((pl->layer_pairing.empty() ? pl->desc.pairing : pl->layer_pairing[l]) == conv) mine.push_back(l);
        for (size_t i = 0; i < mine.size(); i += kMaxLayers) {
            const size_t n = std::min<size_t>(kMaxLayers, mine.size() - i);
            out.push_back({conv, base, std::vector<int>(mine.begin() + (long)i, mine.begin() + (long)(i + n))});
            base += (int)n;
        }
    }
    return out;
}

void fill_params(const leyline_plan_s* pl, MoveParams& mp, int32_t tile_begin, int64_t tile_count, const LayerChunk& lc,
                 void* const* layer_src, void* const* layer_dst, const void* const* layer_repl, int ticket_slot) {
    const int nl = (int)lc.layers.size(), l0 = lc.flag_base;
    std::memset(&mp, 0, sizeof(mp));
    mp.tiles = blob_at<DevTile>(pl, pl->off_tiles);
    mp.trig = blob_at<float>(pl, pl->off_trig);
    mp.tabs = blob_at<int32_t>(pl, pl->off_tabs);
    mp.ticket = reinterpret_cast<unsigned long long*>(pl->d_scratch) + ticket_slot;
    mp.flags = reinterpret_cast<int32_t*>(static_cast<uint8_t*>(pl->d_scratch) + 256);
    mp.n_items = (long long)tile_count * nl;
    mp.stride = pl->desc.row_stride_bytes;
    mp.tile_begin = tile_begin;
    mp.n_layers = nl;
    mp.layer0 = l0;
    mp.n_layers_total = pl->desc.n_layers;
    mp.page_shift = pl->page_shift;
    mp.H = pl->desc.rope_dim / 2;
    mp.lat_chunks = pl->desc.latent_dim * pl->elem_bytes / 16;
    mp.n_heads = pl->n_heads;
    mp.head_chunks = pl->head_chunks;
    mp.band_chunks = pl->n_heads * pl->head_chunks;
    for (int l = 0; l < nl; ++l) {
        mp.src[l] = static_cast<const uint8_t*>(layer_src ? layer_src[lc.layers[l]] : nullptr);
        mp.dst[l] = static_cast<uint8_t*>(layer_dst[lc.layers[l]]);
        mp.repl[l] = static_cast<const uint8_t*>(layer_repl ? layer_repl[lc.layers[l]] : nullptr);
    }
}

/* Launch `fn` over tiles [tile_begin, tile_begin + tile_count) x all layers (chunks of kMaxLayers). */
leyline_status run_tiles(leyline_plan_s* pl, bool hazard, int smem, int max_ctas_per_sm, int32_t tile_begin,
                         int64_t tile_count, void* const* layer_src, void* const* layer_dst,
                         const void* const* layer_repl, cudaStream_t stream, int* ticket_slot) {
    if (tile_count <= 0) return LEYLINE_OK;
    for (const LayerChunk& lc : layer_chunks(pl)) {
        if (*ticket_slot >= 32) { g_last_error = "too many launches for one plan"; return LEYLINE_E_UNSUPPORTED; }
        MoveKernel fn = pick_move(pl, lc.pairing, hazard);
        MoveParams mp;
        fill_params(pl, mp, tile_begin, tile_count, lc, layer_src, layer_dst, layer_repl, (*ticket_slot)++);
        int per_sm = occupancy(reinterpret_cast<const void*>(fn), smem);
        if (max_ctas_per_sm > 0 && per_sm > max_ctas_per_sm) per_sm = max_ctas_per_sm;
        long long grid = (long long)g_dev.sms * per_sm;
        if (grid > mp.n_items) grid = mp.n_items;
        fn<<<(unsigned)grid, kThreads, (size_t)smem, stream>>>(mp);
        CU(cudaGetLastError());
    }
    return LEYLINE_OK;
}

/* a5: k_rotate_band takes its (tile, layer) items round-robin; enough blocks that the hardware scheduler balances. */
leyline_status run_rotate(leyline_plan_s* pl, int32_t tile_begin, int64_t tile_count, int64_t insert_count,
                          void* const* layer_ptrs, const void* const* layer_repl, cudaStream_t stream, int* ticket_slot) {
    if (tile_count + insert_count <= 0) return LEYLINE_OK;
    const bool flat = pl->rotate_flat && tile_begin == 0 && tile_count == pl->info.n_move_tiles && tile_count > 0;
    for (const LayerChunk& lc : layer_chunks(pl)) {
        MoveKernel fn = flat ? pick_rotate_flat(pl, lc.pairing) : pick_rotate(pl, lc.pairing);
        MoveParams mp;
        fill_params(pl, mp, tile_begin, tile_count, lc, nullptr, layer_ptrs, layer_repl, *ticket_slot);
        mp.n_copy_items = insert_count * (long long)lc.layers.size();   /* a4 rides in the same launch */
        mp.copy_tile_begin = tile_begin + (int32_t)tile_count;
        const int per_sm = occupancy(reinterpret_cast<const void*>(fn), 0);
        long long grid = (long long)g_dev.sms * per_sm * 8;
        if (flat) {
            /* items are (pass, layer): full block passes.  Resident blocks only, each with an equal share of the items, so
             * that every block's look-ups for item n+1 run under the loads of item n (a block with ONE item has nothing
             * to hide its tile -> page table -> slot chain behind) */
            mp.passes = blob_at<leyline::RotPass>(pl, pl->off_rot_passes);
            mp.n_rot_tiles = (int32_t)tile_count;
            mp.n_items = (long long)pl->rot_passes.size() * (long long)lc.layers.size();
#ifndef LEYLINE_FLAT_OVERSUBSCRIBE
#define LEYLINE_FLAT_OVERSUBSCRIBE 0
#endif
            const long long resident = (long long)g_dev.sms * per_sm * (LEYLINE_FLAT_OVERSUBSCRIBE ? LEYLINE_FLAT_OVERSUBSCRIBE : 1);
            grid = mp.n_items;
            if (mp.n_items > resident) {
                const long long share = (mp.n_items + resident - 1) / resident;
                grid = (mp.n_items + share - 1) / share;
            }
            if (grid < 1) grid = 1;
        }
        const long long most = mp.n_items > mp.n_copy_items ? mp.n_items : mp.n_copy_items;
        if (grid > most) grid = most;
        fn<<<(unsigned)grid, kThreads, 0, stream>>>(mp);
        CU(cudaGetLastError());
    }
    return LEYLINE_OK;
}

/* ---- a5 with 2-D TMA boxes (k_rotate_band_tma) ----
 * One tensor map per layer pool: a [pool_slots x band] view of the pool (pitch = row stride, base = pool + latent bytes),
 * box = box_rows x band.  cuTensorMapEncodeTiled is host-only arithmetic (no driver call into the device); it is fetched
 * from the driver once, and encoded maps are kept per (pointer, geometry) since a serving pool's layer pointers are
 * stable. */
PFN_cuTensorMapEncodeTiled g_encode_tiled = nullptr;
std::once_flag g_encode_once;

struct MapKey {
    const void* base; int64_t stride, slots; int32_t band_bytes, box_rows;
    bool operator==(const MapKey& o) const {
        return base == o.base && stride == o.stride && slots == o.slots && band_bytes == o.band_bytes && box_rows == o.box_rows;
    }
};
struct MapEntry { MapKey key; CUtensorMap map; };
thread_local std::vector<MapEntry> g_maps; /* small: layers x pools in use by this thread */

leyline_status band_map(const leyline_plan_s* pl, void* pool, int box_rows, CUtensorMap* out) {
    const int64_t band0 = (int64_t)pl->desc.latent_dim * pl->elem_bytes;
    const int32_t band_bytes = pl->n_heads * pl->desc.rope_dim * pl->elem_bytes;
    const MapKey key{static_cast<uint8_t*>(pool) + band0, pl->desc.row_stride_bytes, pl->desc.pool_slots, band_bytes, box_rows};
    for (const MapEntry& e : g_maps)
        if (e.key == key) { *out = e.map; return LEYLINE_OK; }
    std::call_once(g_encode_once, [] {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            g_encode_tiled = reinterpret_cast<PFN_cuTensorMapEncodeTiled>(fn);
        (void)cudaGetLastError();
    });
    if (!g_encode_tiled) { g_last_error = "cuTensorMapEncodeTiled is not available from this driver"; return LEYLINE_E_CUDA; }
    /* elements are 32-bit words: the band is a multiple of 32 bytes, and a box edge holds at most 256 elements */
    const cuuint64_t dims[2] = {(cuuint64_t)(band_bytes / 4), (cuuint64_t)pl->desc.pool_slots};
    const cuuint64_t strides[1] = {(cuuint64_t)pl->desc.row_stride_bytes};
    const cuuint32_t box[2] = {(cuuint32_t)(band_bytes / 4), (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    MapEntry e;
    e.key = key;
    const CUresult r = g_encode_tiled(&e.map, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, const_cast<void*>(key.base), dims, strides, box, estr,
                                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { g_last_error = "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")"; return LEYLINE_E_CUDA; }
    if (g_maps.size() >= 4096) g_maps.clear();
    g_maps.push_back(e);
    *out = e.map;
    return LEYLINE_OK;
}

using BandKernel = void (*)(const MoveParams, const BandMaps, int, int, int, int, int);

template <int DT>
BandKernel pick_band_dt(int pairing) {
    return pairing == LEYLINE_ROPE_NEOX ? k_rotate_band_tma<DT, LEYLINE_ROPE_NEOX> : k_rotate_band_tma<DT, LEYLINE_ROPE_INTERLEAVED>;
}

leyline_status run_rotate_tma(leyline_plan_s* pl, int64_t tile_count, int64_t insert_count, void* const* layer_ptrs,
                              const void* const* layer_repl, cudaStream_t stream, int* ticket_slot) {
    if (tile_count + insert_count <= 0) return LEYLINE_OK;
    const int band_bytes = pl->n_heads * pl->desc.rope_dim * pl->elem_bytes;
    const int box_rows = pl->rot_tile_rows;
    const int stage_bytes = (int)align_up((int64_t)box_rows * band_bytes, 128);
    for (const LayerChunk& lc : layer_chunks(pl, kBandTmaLayers)) {
        const int nl = (int)lc.layers.size();
        BandKernel fn = pl->desc.dtype == LEYLINE_BF16 ? pick_band_dt<LEYLINE_BF16>(lc.pairing) : pick_band_dt<LEYLINE_FP8_E4M3>(lc.pairing);
        SmemCache* sc = nullptr;
        leyline_status sst = smem_entry(reinterpret_cast<const void*>(fn), &sc);
        if (sst != LEYLINE_OK) return sst;
        int stages = (g_dev.smem_optin - sc->static_bytes - 1024) / stage_bytes;
        if (pl->tuning.stages > 0 && stages > pl->tuning.stages) stages = pl->tuning.stages;
        if (stages > kBandMaxStages) stages = kBandMaxStages;
        if (stages < kBandStoresInFlight + 2) { g_last_error = "TMA band kernel: too few shared-memory stages"; return LEYLINE_E_UNSUPPORTED; }
        const int smem = stages * stage_bytes;
        if ((sst = smem_opt_in(sc)) != LEYLINE_OK) return sst;
        if (*ticket_slot >= 32) { g_last_error = "too many launches for one plan"; return LEYLINE_E_UNSUPPORTED; }
        MoveParams mp;
        fill_params(pl, mp, 0, tile_count, lc, nullptr, layer_ptrs, layer_repl, (*ticket_slot)++);
        BandMaps maps;
        std::memset(&maps, 0, sizeof(maps));
        for (int l = 0; l < nl; ++l) {
            leyline_status st = band_map(pl, layer_ptrs[lc.layers[l]], box_rows, &maps.m[l]);
            if (st != LEYLINE_OK) return st;
        }
        int group = pl->tuning.layer_group > 0 ? pl->tuning.layer_group : 8;
        if (group > nl) group = nl;
        mp.n_items = tile_count * ((nl + group - 1) / group);
        mp.n_copy_items = insert_count * (long long)nl;   /* a4 rides in the same launch */
        mp.copy_tile_begin = (int32_t)tile_count;
        long long grid = g_dev.sms;
        const long long most = mp.n_items > mp.n_copy_items ? mp.n_items : mp.n_copy_items;
        if (grid > most) grid = most;
        fn<<<(unsigned)grid, kBandThreads, (size_t)smem, stream>>>(mp, maps, stages, stage_bytes, box_rows, band_bytes, group);
        CU(cudaGetLastError());
    }
    return LEYLINE_OK;
}

/* Same, with the bulk kernel: one persistent CTA per SM, a ring of shared-memory stages of one tile each. */
leyline_status run_tiles_bulk(leyline_plan_s* pl, bool hazard, int32_t tile_begin, int64_t tile_count,
                              void* const* layer_src, void* const* layer_dst, const void* const* layer_repl,
                              cudaStream_t stream, int* ticket_slot) {
    if (tile_count <= 0) return LEYLINE_OK;
    const int row_bytes = (pl->desc.latent_dim + pl->n_heads * pl->desc.rope_dim) * pl->elem_bytes;
    const int stage_bytes = pl->tile_rows * row_bytes;
    /* consumer warps rotate the band in shared memory: 4 keep up with MLA's 1/9 of the bytes, a band that is most of
     * the row (full-width K) needs more issue slots */
    int cwarps = (int64_t)pl->n_heads * pl->desc.rope_dim * 4 <= (int64_t)pl->desc.latent_dim + (int64_t)pl->n_heads * pl->desc.rope_dim
                     ? kBulkConsumerWarps : kBulkWideConsumerWarps;
    if (pl->tuning.consumer_warps > 0) cwarps = pl->tuning.consumer_warps;
    if (cwarps > kBulkMaxConsumerWarps) cwarps = kBulkMaxConsumerWarps;
    for (const LayerChunk& lc : layer_chunks(pl)) {
        const int nl = (int)lc.layers.size();
        BulkKernel fn = pick_bulk(pl, lc.pairing, hazard);
        SmemCache* sc = nullptr;
        leyline_status sst = smem_entry(reinterpret_cast<const void*>(fn), &sc);
        if (sst != LEYLINE_OK) return sst;
        int stages = (g_dev.smem_optin - sc->static_bytes - 1024) / stage_bytes;
        if (pl->tuning.stages > 0 && stages > pl->tuning.stages) stages = pl->tuning.stages;
        if (stages > kBulkMaxStages) stages = kBulkMaxStages;
        if (stages < 3) { g_last_error = "bulk kernel: tile does not fit three shared-memory stages"; return LEYLINE_E_UNSUPPORTED; }
        const int smem = stages * stage_bytes;
        if ((sst = smem_opt_in(sc)) != LEYLINE_OK) return sst;
        if (*ticket_slot >= 32) { g_last_error = "too many launches for one plan"; return LEYLINE_E_UNSUPPORTED; }
        MoveParams mp;
        fill_params(pl, mp, tile_begin, tile_count, lc, layer_src, layer_dst, layer_repl, (*ticket_slot)++);
        int group = pl->tuning.layer_group > 0 ? pl->tuning.layer_group : 4;
        /* In-place moves whose dependencies sit only a few tiles back (small shifts, batched serving): with 4-layer
         * items the tile a store waits for is still in flight on another SM; items of 32 layers make neighbouring
         * tiles advance layer by layer in step, so the wait is over when the store is ready (measured on config 4:
         * 6.35 -> 6.56 TB/s; far dependencies, e.g. config 3, prefer the small items). */
        if (hazard && pl->tuning.layer_group == 0 && pl->dep_distance_median >= 0 &&
            (int64_t)pl->dep_distance_median * ((nl + 3) / 4) < 1024)
            group = 32;
        if (group > nl) group = nl;
        mp.n_items = (long long)tile_count * ((nl + group - 1) / group);
        long long grid = g_dev.sms;
        if (grid > mp.n_items) grid = mp.n_items;
        const int threads = 32 * (1 + cwarps + (hazard ? kBulkHazardWarps + 1 : 0));
        fn<<<(unsigned)grid, threads, (size_t)smem, stream>>>(mp, stages, stage_bytes, row_bytes, group, cwarps);
        CU(cudaGetLastError());
    }
    return LEYLINE_OK;
}

leyline_status check_layers(const leyline_plan_s* pl, const void* const* a, const char* what) {
    if (!a) { g_last_error = std::string(what) + " is NULL"; return LEYLINE_E_INVALID; }
    for (int l = 0; l < pl->desc.n_layers; ++l)
        if (!a[l] || (reinterpret_cast<uintptr_t>(a[l]) & 15)) {
            g_last_error = std::string(what) + ": NULL or not 16-byte aligned layer pointer";
            return LEYLINE_E_INVALID;
        }
    return LEYLINE_OK;
}

leyline_status begin_call(leyline_plan_s* pl, cudaStream_t stream) {
    leyline_status st = ensure_device(pl, stream);
    if (st != LEYLINE_OK) return st;
    pl->last_stream = stream;
    if (!pl->scratch_clean) CU(cudaMemsetAsync(pl->d_scratch, 0, (size_t)pl->scratch_bytes, stream));
    pl->scratch_clean = false; /* tickets and hazard flags are consumed by this launch */
    if (pl->tuning.profile && !pl->ev_start) {
        CU(cudaEventCreate(reinterpret_cast<cudaEvent_t*>(&pl->ev_start)));
        CU(cudaEventCreate(reinterpret_cast<cudaEvent_t*>(&pl->ev_stop)));
    }
    return LEYLINE_OK;
}

}  // namespace

extern "C" LEYLINE_API leyline_status leyline_splice(leyline_plan_t* pl, void* const* layer_src, void* const* layer_dst,
                                         const void* const* layer_repl, int32_t* dev_page_table_out,
                                         int32_t* dev_slot_idx_out, void* cuda_stream) try {
    g_last_error.clear();
    if (!pl || pl->mode == LEYLINE_ROTATE_ONLY) return LEYLINE_E_INVALID;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const bool inplace = pl->mode == LEYLINE_INPLACE_MOVE;
    /* layer_repl == NULL: the caller prefills the replacement slots itself (PAPER.md:405(b)); insert tiles are skipped */
    const int64_t n_move = pl->info.n_move_tiles, n_ins = layer_repl ? pl->info.n_tiles - n_move : 0;
    if (n_move + n_ins > 0) {
        leyline_status st = check_layers(pl, layer_dst, "layer_dst");
        if (st == LEYLINE_OK && n_move > 0) st = check_layers(pl, layer_src, "layer_src");
        if (st == LEYLINE_OK && n_ins > 0) st = check_layers(pl, layer_repl, "layer_repl");
        if (st != LEYLINE_OK) return st;
        if (inplace && n_move > 0)
            for (int l = 0; l < pl->desc.n_layers; ++l)
                if (layer_src[l] != layer_dst[l]) {
                    g_last_error = "INPLACE_MOVE needs layer_src == layer_dst";
                    return LEYLINE_E_INVALID;
                }
    }
    leyline_status st = begin_call(pl, stream);
    if (st != LEYLINE_OK) return st;
    /* a2: page-table rows and token-level slot list */
    st = launch_index(pl, dev_page_table_out, dev_slot_idx_out, stream);
    if (st != LEYLINE_OK) return st;
    if (pl->tuning.profile) CU(cudaEventRecord(static_cast<cudaEvent_t>(pl->ev_start), stream));
    int slot = 0;
    const int cps = pl->tuning.ctas_per_sm;
    if (pl->use_bulk) {
        /* bulk kernel (TMA 1-D copies through shared memory) */
        if (inplace) {
            /* one launch: the insert tiles hold the last tickets and wait for the move tiles that read their rows */
            st = run_tiles_bulk(pl, true, 0, n_move + n_ins, layer_src, layer_dst, layer_repl, stream, &slot);
        } else {
            st = run_tiles_bulk(pl, false, 0, n_move + n_ins, layer_src, layer_dst, layer_repl, stream, &slot);
        }
    } else if (inplace) {
        /* a3 under rule M2 ordering and a4 in one launch: insert tiles wait for the move tiles that read their rows */
        st = run_tiles(pl, true, 0, cps, 0, n_move + n_ins, layer_src, layer_dst, layer_repl, stream, &slot);
    } else {
        /* a3 + a4 in one launch: fresh pages alias nothing */
        st = run_tiles(pl, false, 0, cps, 0, n_move + n_ins, layer_src, layer_dst, layer_repl, stream,
                       &slot);
    }
    if (st != LEYLINE_OK) return st;
    if (pl->tuning.profile) CU(cudaEventRecord(static_cast<cudaEvent_t>(pl->ev_stop), stream));
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

extern "C" LEYLINE_API leyline_status leyline_rotate_inplace(leyline_plan_t* pl, void* const* layer_ptrs,
                                                 const void* const* layer_repl, int32_t* dev_slot_idx_out,
                                                 void* cuda_stream) try {
    g_last_error.clear();
    if (!pl || pl->mode != LEYLINE_ROTATE_ONLY) return LEYLINE_E_INVALID;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int64_t n_rot = pl->info.n_move_tiles, n_ins = layer_repl ? pl->info.n_tiles - n_rot : 0;
    if (n_rot + n_ins > 0) {
        leyline_status st = check_layers(pl, layer_ptrs, "layer_ptrs");
        if (st == LEYLINE_OK && n_ins > 0) st = check_layers(pl, layer_repl, "layer_repl");
        if (st != LEYLINE_OK) return st;
    }
    leyline_status st = begin_call(pl, stream);
    if (st != LEYLINE_OK) return st;
    st = launch_index(pl, nullptr, dev_slot_idx_out, stream);
    if (st != LEYLINE_OK) return st;
    if (pl->tuning.profile) CU(cudaEventRecord(static_cast<cudaEvent_t>(pl->ev_start), stream));
    int slot = 0;
    /* a5: rotate where the rows sit; a4: replacement rows go to the consumed free slots (disjoint from a5's) */
    if (pl->rotate_with_bulk) /* wide band: whole rows through the bulk mover, written back in place; inserts as usual */
        st = run_tiles_bulk(pl, false, 0, n_rot + n_ins, layer_ptrs, layer_ptrs, layer_repl, stream, &slot);
    else if (pl->rotate_with_tma) /* narrow band in pages: one 2-D TMA box per page and layer */
        st = run_rotate_tma(pl, n_rot, n_ins, layer_ptrs, layer_repl, stream, &slot);
    else
        st = run_rotate(pl, 0, n_rot, n_ins, layer_ptrs, layer_repl, stream, &slot);
    if (st != LEYLINE_OK) return st;
    if (pl->tuning.profile) CU(cudaEventRecord(static_cast<cudaEvent_t>(pl->ev_stop), stream));
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

extern "C" LEYLINE_API leyline_status leyline_rotate_inplace_master(leyline_plan_t* pl, void* const* layer_ptrs, void* const* layer_master,
                                                        const void* const* layer_repl, int32_t* dev_slot_idx_out,
                                                        void* cuda_stream) try {
    g_last_error.clear();
    if (!pl || pl->mode != LEYLINE_ROTATE_ONLY) return LEYLINE_E_INVALID;
    if (pl->desc.dtype != LEYLINE_BF16) { g_last_error = "the fp32 master option covers bf16 caches"; return LEYLINE_E_UNSUPPORTED; }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int64_t n_rot = pl->info.n_move_tiles, n_ins = layer_repl ? pl->info.n_tiles - n_rot : 0;
    if (n_rot + n_ins > 0) {
        leyline_status st = check_layers(pl, layer_ptrs, "layer_ptrs");
        if (st == LEYLINE_OK) st = check_layers(pl, layer_master, "layer_master");
        if (st == LEYLINE_OK && n_ins > 0) st = check_layers(pl, layer_repl, "layer_repl");
        if (st != LEYLINE_OK) return st;
    }
    leyline_status st = begin_call(pl, stream);
    if (st != LEYLINE_OK) return st;
    st = launch_index(pl, nullptr, dev_slot_idx_out, stream);
    if (st != LEYLINE_OK) return st;
    if (pl->tuning.profile) CU(cudaEventRecord(static_cast<cudaEvent_t>(pl->ev_start), stream));
    if (n_rot + n_ins > 0) {
        for (const LayerChunk& lc : layer_chunks(pl)) {
            MoveKernel fn = lc.pairing == LEYLINE_ROPE_NEOX ? k_rotate_master<LEYLINE_ROPE_NEOX> : k_rotate_master<LEYLINE_ROPE_INTERLEAVED>;
            MoveParams mp;
            /* the master pointers travel in the (otherwise unused) source slots of the parameter block */
            fill_params(pl, mp, 0, n_rot, lc, layer_master, layer_ptrs, layer_repl, 0);
            mp.n_copy_items = n_ins * (long long)lc.layers.size();
            mp.copy_tile_begin = (int32_t)n_rot;
            const int per_sm = occupancy(reinterpret_cast<const void*>(fn), 0);
            long long grid = (long long)g_dev.sms * per_sm * 8;
            const long long most = mp.n_items > mp.n_copy_items ? mp.n_items : mp.n_copy_items;
            if (grid > most) grid = most;
            fn<<<(unsigned)grid, kThreads, 0, stream>>>(mp);
            CU(cudaGetLastError());
        }
    }
    if (pl->tuning.profile) CU(cudaEventRecord(static_cast<cudaEvent_t>(pl->ev_stop), stream));
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

extern "C" LEYLINE_API leyline_status leyline_plan_prefetch(leyline_plan_t* pl) try {
    g_last_error.clear();
    if (!pl) return LEYLINE_E_INVALID;
    if (pl->d_blob || pl->device >= 0) return LEYLINE_OK;
    int dev = 0;
    leyline_status st = device_info(&dev);
    if (st != LEYLINE_OK) return st;
    PlanPool* pp = plan_pool(dev);
    if (!pp) { g_last_error = "could not create the plan-table pool / copy stream"; return LEYLINE_E_CUDA; }
    st = upload_tables(pl, dev, pp->copy_stream);
    if (st != LEYLINE_OK) return st;
    CU(cudaEventCreateWithFlags(reinterpret_cast<cudaEvent_t*>(&pl->ev_uploaded), cudaEventDisableTiming));
    CU(cudaEventRecord(static_cast<cudaEvent_t>(pl->ev_uploaded), pp->copy_stream));
    pl->last_stream = pp->copy_stream; /* until a launch replaces it: a never-launched plan frees its tables there */
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

extern "C" LEYLINE_API leyline_status leyline_plan_kernel_ms(const leyline_plan_t* pl, float* ms) try {
    g_last_error.clear();
    if (!pl || !ms || !pl->ev_start) return LEYLINE_E_INVALID;
    CU(cudaEventSynchronize(static_cast<cudaEvent_t>(pl->ev_stop))); /* returns at once when the launch has finished */
    CU(cudaEventElapsedTime(ms, static_cast<cudaEvent_t>(pl->ev_start), static_cast<cudaEvent_t>(pl->ev_stop)));
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

/* The device's own cos/sin table, for comparison with the host evaluation (tests / tooling). */
extern "C" LEYLINE_API leyline_status leyline_plan_trig_table_device(const leyline_plan_t* pl, float* out) try {
    g_last_error.clear();
    if (!pl || (!out && !pl->trig_shifts.empty()) || !pl->trig_ready || !pl->d_blob) return LEYLINE_E_INVALID;
    if (pl->trig_shifts.empty()) return LEYLINE_OK;
    /* the hi parts [cos | sin] of every row: the fp64 values rounded once to fp32, which is what the host query evaluates */
    const size_t row = 2 * pl->inv_freq.size() * sizeof(float);
    cudaStream_t stream = static_cast<cudaStream_t>(pl->last_stream);
    CU(cudaMemcpy2DAsync(out, row, blob_at<float>(pl, pl->off_trig), kTrigParts / 2 * row, row, pl->trig_shifts.size(),
                         cudaMemcpyDeviceToHost, stream));
    CU(cudaStreamSynchronize(stream));
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

/* Measurement aid (leyline.h): the a5 access pattern on a contiguous buffer, nothing else. */
extern "C" LEYLINE_API leyline_status leyline_probe_band_update(void* dev_buf, int64_t n_rows, int64_t row_stride_bytes,
                                                                int32_t band_offset_bytes, int32_t band_bytes,
                                                                int32_t ctas_per_sm, void* cuda_stream) try {
    g_last_error.clear();
    if (!dev_buf || n_rows < 0 || row_stride_bytes < 16 || (row_stride_bytes & 15) || band_offset_bytes < 0 ||
        (band_offset_bytes & 15) || band_bytes < 16 || (band_bytes & 15) || band_offset_bytes + (int64_t)band_bytes > row_stride_bytes ||
        (reinterpret_cast<uintptr_t>(dev_buf) & 15) || ctas_per_sm < 0 || ctas_per_sm > 32)
        return LEYLINE_E_INVALID;
    if (n_rows == 0) return LEYLINE_OK;
    int dev = 0;
    leyline_status st = device_info(&dev);
    if (st != LEYLINE_OK) return st;
    const int per_sm = ctas_per_sm > 0 ? ctas_per_sm : 8;
    const bool half_line = ((row_stride_bytes | band_offset_bytes | band_bytes) & 127) != 0; /* bands that share lines with bytes nobody reads */
    auto probe = half_line ? k_probe_band_update<8, true> : k_probe_band_update<8, false>;
    probe<<<(unsigned)(g_dev.sms * per_sm), kThreads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        static_cast<uint8_t*>(dev_buf), n_rows, row_stride_bytes, band_offset_bytes, band_bytes / 16);
    CU(cudaGetLastError());
    return LEYLINE_OK;
} LEYLINE_CATCH_STATUS

void leyline::plan_release_device(leyline_plan_s* pl) {
    if (pl->ev_start) cudaEventDestroy(static_cast<cudaEvent_t>(pl->ev_start));
    if (pl->ev_stop) cudaEventDestroy(static_cast<cudaEvent_t>(pl->ev_stop));
    if (pl->ev_uploaded) cudaEventDestroy(static_cast<cudaEvent_t>(pl->ev_uploaded));
    pl->ev_uploaded = nullptr;
    /* stream-ordered: freed after everything this plan launched on its stream, without a device sync */
    if (pl->d_blob) cudaFreeAsync(pl->d_blob, static_cast<cudaStream_t>(pl->last_stream)); /* tables + scratch */
    pl->d_blob = pl->d_scratch = nullptr;
    pl->ev_start = pl->ev_stop = nullptr;
    if (pl->device >= 0) (void)cudaGetLastError();
}

extern "C" LEYLINE_API const char* leyline_last_cuda_error(void) { return g_last_error.c_str(); }

// Context, options and the executor: uploads descriptors, launches kernel (a) per hazard phase on the copy stream and
// runs the reload pipeline (b) on the reload stream.  PAPER.md:162-166: "issuing host-to-device reloads alongside GPU P2P
// transfers, allowing the P2P portions to be hidden beneath the PCIe-bound reload time".
//
// Multi-device (SURVEY.md 8(e), 8(f) #1; PAPER.md:64 "P2P direct access over high-speed interconnects", :162-166): the work
// of a call is PARTITIONED BY DESTINATION - every logical device runs one launch of kernel (a) per hazard phase that writes
// only the slabs / pools of the ranks mapped to it and PULLS its incoming intervals through peer-mapped source pointers; its
// reloads go over its own host link.  No collective: the exchange is a sparse all-to-all of one-sided reads.  A ctx owns one
// DevState per logical device (streams, descriptor arenas, events); several logical devices may alias one physical GPU
// (that is how the path is exercised on a one-GPU box).  The default ctx has ONE logical device and runs on the caller's
// streams, exactly as before.
#include <algorithm>
#include <chrono>
#include <cstring>

#include "etp_copy.cuh"

using namespace etp;

namespace {
constexpr int kArenaSlots = 2;
constexpr int kCounterSlots = 256;   // pairs of work-queue heads available to one call (they live in the call's arena slot)

struct ArenaSlot {
    void* h = nullptr;
    void* d = nullptr;
    int64_t bytes = 0;
    cudaEvent_t done_copy = nullptr, done_reload = nullptr;
    bool busy = false;
};
struct DevState {
    int device = 0;                                  // physical CUDA device
    cudaStream_t copy = nullptr, reload = nullptr;   // library-owned streams (multi-device ctx only)
    ArenaSlot slot[kArenaSlots];
    int next = 0;
    cudaEvent_t uploaded = nullptr, join_copy = nullptr, join_reload = nullptr;
    std::vector<cudaEvent_t> phase_ev;               // "copy phase p of this device has finished"
    std::vector<cudaEvent_t> tev;                    // timing events (pairs) around its copy-stream launches
    int32_t n_timed = 0;
    etp_reshard_report rep{};                        // what the last call did on this device
};
struct CtxExtra {
    std::vector<DevState> dev;
    std::vector<int32_t> rank_dev;                   // rank -> logical device, -1 = a rank another process writes; empty = all on 0
    cudaEvent_t fork_copy = nullptr, fork_reload = nullptr;   // on the primary device: the caller's streams at call time
};
CtxExtra* extra(const etp_ctx* c) { return reinterpret_cast<CtxExtra*>(c->impl); }

double now_ms() {
    return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count();
}
}  // namespace

namespace etp {
void reset_device_timing(etp_ctx* c) {
    for (DevState& D : extra(c)->dev) D.n_timed = 0;
}
int n_logical_devices(const etp_ctx* c) { return (int)extra(c)->dev.size(); }
int device_of_rank(const etp_ctx* c, int32_t rank) {
    const CtxExtra* x = extra(c);
    if (x->rank_dev.empty()) return 0;
    return (rank >= 0 && rank < (int32_t)x->rank_dev.size()) ? x->rank_dev[rank] : 0;
}
}  // namespace etp

extern "C" etp_status etp_ctx_create_multi(const int32_t* devices, int32_t n_devices, etp_ctx** out) {
    if (!out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_create: out is NULL");
    *out = nullptr;
    if (!devices || n_devices < 1 || n_devices > 64) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_create_multi: 1..64 logical devices");
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess) n_dev = 0;
    cudaGetLastError();
    int n_sms = 0;
    for (int32_t i = 0; i < n_devices; ++i) {
        const int device = devices[i];
        if (device < 0 || device >= n_dev)
            ETP_FAIL(ETP_ERR_CUDA, "etp_ctx_create: CUDA device %d not available (%d devices); there is no CPU fallback", device, n_dev);
        cudaDeviceProp prop;
        ETP_CUDA_OK(cudaGetDeviceProperties(&prop, device));
        if (prop.major != 10) ETP_FAIL(ETP_ERR_CUDA, "etp_ctx_create: device %d is sm_%d%d; this library is built for sm_100a only", device, prop.major, prop.minor);
        if (i == 0) n_sms = prop.multiProcessorCount;
        n_sms = std::min(n_sms, prop.multiProcessorCount);
    }
    // every destination device reads its sources through peer-mapped pointers
    for (int32_t i = 0; i < n_devices; ++i)
        for (int32_t j = 0; j < n_devices; ++j) {
            if (devices[i] == devices[j]) continue;
            int can = 0;
            ETP_CUDA_OK(cudaDeviceCanAccessPeer(&can, devices[i], devices[j]));
            if (!can) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_ctx_create_multi: device %d cannot map the memory of device %d", devices[i], devices[j]);
            ETP_CUDA_OK(cudaSetDevice(devices[i]));
            const cudaError_t e = cudaDeviceEnablePeerAccess(devices[j], 0);
            if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) ETP_CUDA_OK(e);
            cudaGetLastError();
        }
    ETP_CUDA_OK(cudaSetDevice(devices[0]));
    etp_ctx* c = new (std::nothrow) etp_ctx();
    if (!c) ETP_FAIL(ETP_ERR_NOMEM, "etp_ctx_create: out of memory");
    c->device = devices[0];
    c->n_sms = n_sms;
    std::memset(c->opts, 0, sizeof(c->opts));
    c->opts[ETP_OPT_TMA_MIN_BYTES] = 32768;
    c->opts[ETP_OPT_LDG_STEALS_BULK] = 0;
    c->opts[ETP_OPT_RELOAD_CHUNK_BYTES] = 64 << 20;
    c->opts[ETP_OPT_GRID_CTAS] = 0;
    c->opts[ETP_OPT_GATHER_CTAS] = 16;
    c->opts[ETP_OPT_LINEAR_CTA_PAIR] = 1;
    c->opts[ETP_OPT_VALIDATE_INTERVALS] = 1;
    c->opts[ETP_OPT_LINEAR_PDL] = 1;
    c->opts[ETP_OPT_LINEAR_RING] = 2;
    c->opts[ETP_OPT_ONLY_PHASE] = 0;
    c->opts[ETP_OPT_MOE_CTA_PAIR] = 1;
    c->opts[ETP_OPT_SMALL_STAGED] = 1;
    CtxExtra* x = new (std::nothrow) CtxExtra();
    if (!x) { delete c; ETP_FAIL(ETP_ERR_NOMEM, "etp_ctx_create: out of memory"); }
    c->impl = x;
    x->dev.resize((size_t)n_devices);
    cudaError_t e = cudaEventCreateWithFlags(&x->fork_copy, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&x->fork_reload, cudaEventDisableTiming);
    for (int32_t i = 0; i < n_devices && e == cudaSuccess; ++i) {
        DevState& D = x->dev[i];
        D.device = devices[i];
        e = cudaSetDevice(D.device);
        if (e == cudaSuccess && n_devices > 1) e = cudaStreamCreateWithFlags(&D.copy, cudaStreamNonBlocking);
        if (e == cudaSuccess && n_devices > 1) e = cudaStreamCreateWithFlags(&D.reload, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&D.uploaded, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&D.join_copy, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&D.join_reload, cudaEventDisableTiming);
        for (int k = 0; k < kArenaSlots && e == cudaSuccess; ++k) {
            e = cudaEventCreateWithFlags(&D.slot[k].done_copy, cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&D.slot[k].done_reload, cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = configure_copy_kernel();   // a per-device function attribute
        if (e == cudaSuccess && !g_wait_fault_host) {          // once per process: the fault record of the bounded waits (etp_wait.cuh)
            void* rec = nullptr;
            e = cudaHostAlloc(&rec, 64, cudaHostAllocPortable | cudaHostAllocMapped);
            if (e == cudaSuccess) {
                std::memset(rec, 0, 64);
                g_wait_fault_host = static_cast<volatile unsigned long long*>(rec);
            }
        }
        unsigned long long* rec = const_cast<unsigned long long*>(g_wait_fault_host);   // UVA: the host address is the device address
        if (e == cudaSuccess) e = install_wait_fault_copy(rec);
        if (e == cudaSuccess) e = install_wait_fault_linear(rec);
        if (e == cudaSuccess) e = install_wait_fault_group(rec);
        if (e == cudaSuccess) e = install_wait_fault_moe(rec);
    }
    cudaSetDevice(devices[0]);
    if (e != cudaSuccess) {
        set_error("etp_ctx_create: %s", cudaGetErrorString(e));
        etp_ctx_destroy(c);
        return ETP_ERR_CUDA;
    }
    *out = c;
    return ETP_OK;
}

extern "C" etp_status etp_ctx_create(int device, int64_t staging_bytes, etp_ctx** out) {
    if (!out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_create: out is NULL");
    *out = nullptr;
    if (staging_bytes < 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_create: staging_bytes < 0");
    const int32_t d = device;
    return etp_ctx_create_multi(&d, 1, out);
}

extern "C" etp_status etp_ctx_set_rank_devices(etp_ctx* c, const int32_t* device_of_rank, int32_t n_ranks) {
    if (!c || n_ranks < 0 || (n_ranks > 0 && !device_of_rank)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_set_rank_devices: bad arguments");
    CtxExtra* x = extra(c);
    for (int32_t r = 0; r < n_ranks; ++r)
        if (device_of_rank[r] < -1 || device_of_rank[r] >= (int32_t)x->dev.size())
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_set_rank_devices: rank %d -> logical device %d, the ctx has %d", r, device_of_rank[r], (int)x->dev.size());
    x->rank_dev.assign(device_of_rank, device_of_rank + n_ranks);
    return ETP_OK;
}

extern "C" etp_status etp_ctx_device_report(etp_ctx* c, int32_t logical_device, etp_reshard_report* out) {
    if (!c || !out || logical_device < 0 || logical_device >= (int32_t)extra(c)->dev.size())
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_device_report: bad arguments");
    *out = extra(c)->dev[logical_device].rep;
    return ETP_OK;
}

extern "C" void etp_ctx_destroy(etp_ctx* c) {
    if (!c) return;
    CtxExtra* x = extra(c);
    if (x) {
        for (DevState& D : x->dev) {
            cudaSetDevice(D.device);
            cudaDeviceSynchronize();
            for (int i = 0; i < kArenaSlots; ++i) {
                if (D.slot[i].h) cudaFreeHost(D.slot[i].h);
                if (D.slot[i].d) cudaFree(D.slot[i].d);
                if (D.slot[i].done_copy) cudaEventDestroy(D.slot[i].done_copy);
                if (D.slot[i].done_reload) cudaEventDestroy(D.slot[i].done_reload);
            }
            for (cudaEvent_t e : {D.uploaded, D.join_copy, D.join_reload})
                if (e) cudaEventDestroy(e);
            for (cudaEvent_t e : D.phase_ev) cudaEventDestroy(e);
            for (cudaEvent_t e : D.tev) cudaEventDestroy(e);
            if (D.copy) cudaStreamDestroy(D.copy);
            if (D.reload) cudaStreamDestroy(D.reload);
        }
        cudaSetDevice(c->device);
        if (x->fork_copy) cudaEventDestroy(x->fork_copy);
        if (x->fork_reload) cudaEventDestroy(x->fork_reload);
    }
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    etp::free_interval_state(c);
    etp::lin_teardown(c);
    cudaGetLastError();
    delete x;
    delete c;
}

extern "C" etp_status etp_ctx_set_option(etp_ctx* c, etp_option key, int64_t value) {
    if (!c || key < 0 || key >= ETP_OPT__COUNT) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_set_option: bad ctx/key");
    if (value < 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_set_option: negative value");
    if (key == ETP_OPT_TMA_MIN_BYTES && value < 16) value = 16;
    if (key == ETP_OPT_RELOAD_CHUNK_BYTES && value < 4096) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_set_option: reload chunk < 4096");
    c->opts[key] = value;
    return ETP_OK;
}

extern "C" etp_status etp_ctx_get_option(const etp_ctx* c, etp_option key, int64_t* value) {
    if (!c || !value || key < 0 || key >= ETP_OPT__COUNT) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_get_option: bad ctx/key");
    *value = c->opts[key];
    return ETP_OK;
}

extern "C" etp_status etp_ctx_kernel_time(etp_ctx* c, double* ms_out, int32_t* n_out) {
    if (!c || !ms_out || !n_out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_kernel_time: NULL argument");
    double ms = 0;
    int32_t n = 0;
    for (DevState& D : extra(c)->dev) {
        for (int32_t i = 0; i < D.n_timed; ++i) {
            float t = 0;
            ETP_CUDA_OK(cudaEventSynchronize(D.tev[2 * i + 1]));
            ETP_CUDA_OK(cudaEventElapsedTime(&t, D.tev[2 * i], D.tev[2 * i + 1]));
            ms += t;
        }
        n += D.n_timed;
    }
    double iv_ms = 0;
    n += interval_timed_launches(c, &iv_ms);   // chunked launches of a device-lowered etp_copy_intervals
    *ms_out = ms + iv_ms;
    *n_out = n;
    return ETP_OK;
}

namespace etp {

namespace {
struct Off { int64_t bulk, bulk_items, vec, vec_items, small, small_first, gat, gat_items; };
struct DevPlan {                      // one device's share of a call, laid out in its arena slot
    std::vector<Off> off;
    int64_t off_counters = 0, off_pairs = 0, total = 0, n_jobs = 0, n_items = 0;
    int launches_needed = 0;
    ArenaSlot* slot = nullptr;
    char* d_base = nullptr;
    int counter_slot = 0;
};
inline int64_t pad256(int64_t b) { return (b + 255) & ~int64_t(255); }

// item table: the segment index of every work item, one fill per segment
void fill_items(uint32_t* items, uint32_t n_items_total, const uint32_t* firsts, size_t n_segs, size_t stride) {
    for (size_t i = 0; i < n_segs; ++i) {
        const uint32_t b = *(const uint32_t*)((const char*)firsts + i * stride);
        const uint32_t e = i + 1 < n_segs ? *(const uint32_t*)((const char*)firsts + (i + 1) * stride) : n_items_total;
        std::fill(items + b, items + e, (uint32_t)i);
    }
}

etp_status ensure_phase_event(DevState& D, size_t i) {
    while (D.phase_ev.size() <= i) {
        cudaEvent_t e;
        ETP_CUDA_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        D.phase_ev.push_back(e);
    }
    return ETP_OK;
}
}  // namespace

etp_status execute(etp_ctx* c, LoweredWork* w, void* copy_stream_v, void* reload_stream_v, etp_reshard_report* report) {
    const double t0 = now_ms();
    cudaStream_t caller_cs = (cudaStream_t)copy_stream_v, caller_rs = (cudaStream_t)reload_stream_v;
    CtxExtra* x = extra(c);
    reset_interval_timing(c);
    note_slab_write(c, copy_stream_v);     // the next small-token linear launch on these streams must not prefetch weights early
    note_slab_write(c, reload_stream_v);
    const size_t n_dev = x->dev.size();
    const bool multi = n_dev > 1;
    const bool skip_d2d = c->opts[ETP_OPT_SKIP_D2D] != 0, skip_reload = c->opts[ETP_OPT_SKIP_RELOAD] != 0;
    const int64_t only_phase = c->opts[ETP_OPT_ONLY_PHASE];   // 0 = every phase; k > 0 = phase k - 1 only (caller synchronises between)
    w->dev.resize(n_dev);
    size_t n_ph = 1;
    for (DeviceWork& dw : w->dev) {
        n_ph = std::max({n_ph, dw.phases.size(), dw.host_gather.size()});
        for (const DmaCopy& d : dw.dma) n_ph = std::max(n_ph, (size_t)d.phase + 1);   // a reload may be the last phase
    }
    for (DeviceWork& dw : w->dev) {
        dw.phases.resize(n_ph);
        dw.host_gather.resize(n_ph);
    }
    auto phase_on = [&](size_t p) { return only_phase == 0 || (int64_t)p == only_phase - 1; };

    // ---- per device: descriptor arena layout: work-queue heads (zero) | pairs | per phase: bulk segs, bulk items, vec segs,
    //      vec items, small segs, batch starts, gather segs, gather items.  The queue heads travel with the descriptors, so the
    //      done_copy / done_reload events that guard an arena slot also guard its counters: a call whose zero-copy gather is
    //      still queued behind GBs of DMA on the reload stream cannot have its heads reset by the next call.
    std::vector<DevPlan> plan(n_dev);
    for (size_t d = 0; d < n_dev; ++d) {
        DeviceWork& dw = w->dev[d];
        DevPlan& P = plan[d];
        P.off.resize(n_ph);
        for (size_t p = 0; p < n_ph; ++p) P.launches_needed += (!dw.phases[p].empty()) + (!dw.host_gather[p].vec.empty());
        if (P.launches_needed > kCounterSlots) ETP_FAIL(ETP_ERR_CAPACITY, "plan needs %d launches > %d", P.launches_needed, kCounterSlots);
        P.off_counters = 0;
        P.total = pad256((int64_t)P.launches_needed * 2 * sizeof(unsigned int));
        P.off_pairs = P.total;
        P.total += pad256((int64_t)w->pairs.size() * sizeof(int32_t));
        for (size_t p = 0; p < n_ph; ++p) {
            const JobList &jl = dw.phases[p], &gl = dw.host_gather[p];
            Off& o = P.off[p];
            o.bulk = P.total;        P.total += pad256((int64_t)jl.bulk.size() * sizeof(BulkSeg));
            o.bulk_items = P.total;  P.total += pad256((int64_t)jl.n_bulk_items * sizeof(uint32_t));
            o.vec = P.total;         P.total += pad256((int64_t)jl.vec.size() * sizeof(VecSeg));
            o.vec_items = P.total;   P.total += pad256((int64_t)jl.n_vec_items * sizeof(uint32_t));
            o.small = P.total;       P.total += pad256((int64_t)jl.small.size() * sizeof(SmallSeg));
            o.small_first = P.total; P.total += pad256((int64_t)(jl.small_first.size() + 1) * sizeof(uint32_t));
            o.gat = P.total;         P.total += pad256((int64_t)gl.vec.size() * sizeof(VecSeg));
            o.gat_items = P.total;   P.total += pad256((int64_t)gl.n_vec_items * sizeof(uint32_t));
            P.n_jobs += (int64_t)(jl.bulk.size() + jl.vec.size() + jl.small.size() + gl.vec.size());
            P.n_items += (int64_t)jl.n_bulk_items + jl.n_vec_items + (int64_t)jl.small_first.size() + gl.n_vec_items;
            if (jl.bulk.size() >= 0xFFFFFFF0ull || jl.vec.size() >= 0xFFFFFFF0ull || jl.small.size() >= 0xFFFFFFF0ull ||
                gl.vec.size() >= 0xFFFFFFF0ull || (uint64_t)jl.n_vec_items + jl.small_first.size() >= 0xFFFFFFF0ull)
                ETP_FAIL(ETP_ERR_CAPACITY, "too many segments in one phase");
        }
    }

    // ---- fork: the library's per-device streams start where the caller's streams are
    if (multi) {
        ETP_CUDA_OK(cudaSetDevice(c->device));
        ETP_CUDA_OK(cudaEventRecord(x->fork_copy, caller_cs));
        ETP_CUDA_OK(cudaEventRecord(x->fork_reload, caller_rs));
    }
    auto cs_of = [&](size_t d) { return multi ? x->dev[d].copy : caller_cs; };
    auto rs_of = [&](size_t d) { return multi ? x->dev[d].reload : caller_rs; };

    // ---- upload every device's descriptors
    for (size_t d = 0; d < n_dev; ++d) {
        DevState& D = x->dev[d];
        DeviceWork& dw = w->dev[d];
        DevPlan& P = plan[d];
        D.n_timed = 0;
        D.rep = etp_reshard_report{};
        ETP_CUDA_OK(cudaSetDevice(D.device));
        if (multi) {
            ETP_CUDA_OK(cudaStreamWaitEvent(D.copy, x->fork_copy, 0));
            ETP_CUDA_OK(cudaStreamWaitEvent(D.reload, x->fork_reload, 0));
        }
        if (P.n_jobs == 0) continue;
        ArenaSlot* slot = &D.slot[D.next];
        D.next = (D.next + 1) % kArenaSlots;
        if (slot->busy) {  // the call that used this slot two calls ago must have consumed its descriptors
            ETP_CUDA_OK(cudaEventSynchronize(slot->done_copy));
            ETP_CUDA_OK(cudaEventSynchronize(slot->done_reload));
            slot->busy = false;
        }
        if (slot->bytes < P.total) {
            if (slot->h) cudaFreeHost(slot->h);
            if (slot->d) cudaFree(slot->d);
            slot->h = slot->d = nullptr;
            slot->bytes = 0;
            const int64_t want = std::max<int64_t>(P.total + P.total / 4, 1 << 20);
            ETP_CUDA_OK(cudaMallocHost(&slot->h, want));
            ETP_CUDA_OK(cudaMalloc(&slot->d, want));
            slot->bytes = want;
        }
        char* h = (char*)slot->h;
        std::memset(h + P.off_counters, 0, (size_t)P.launches_needed * 2 * sizeof(unsigned int));
        if (!w->pairs.empty()) std::memcpy(h + P.off_pairs, w->pairs.data(), w->pairs.size() * sizeof(int32_t));
        for (size_t p = 0; p < n_ph; ++p) {
            const JobList &jl = dw.phases[p], &gl = dw.host_gather[p];
            const Off& o = P.off[p];
            if (!jl.bulk.empty()) {
                std::memcpy(h + o.bulk, jl.bulk.data(), jl.bulk.size() * sizeof(BulkSeg));
                fill_items((uint32_t*)(h + o.bulk_items), jl.n_bulk_items, &jl.bulk[0].first_item, jl.bulk.size(), sizeof(BulkSeg));
            }
            if (!jl.vec.empty()) {
                std::memcpy(h + o.vec, jl.vec.data(), jl.vec.size() * sizeof(VecSeg));
                fill_items((uint32_t*)(h + o.vec_items), jl.n_vec_items, &jl.vec[0].first_item, jl.vec.size(), sizeof(VecSeg));
            }
            if (!jl.small.empty()) {
                std::memcpy(h + o.small, jl.small.data(), jl.small.size() * sizeof(SmallSeg));
                uint32_t* f = (uint32_t*)(h + o.small_first);
                std::memcpy(f, jl.small_first.data(), jl.small_first.size() * sizeof(uint32_t));
                f[jl.small_first.size()] = (uint32_t)jl.small.size();
            }
            if (!gl.vec.empty()) {
                std::memcpy(h + o.gat, gl.vec.data(), gl.vec.size() * sizeof(VecSeg));
                fill_items((uint32_t*)(h + o.gat_items), gl.n_vec_items, &gl.vec[0].first_item, gl.vec.size(), sizeof(VecSeg));
            }
        }
        P.slot = slot;
        P.d_base = (char*)slot->d;
        ETP_CUDA_OK(cudaMemcpyAsync(P.d_base, h, P.total, cudaMemcpyHostToDevice, cs_of(d)));
        ETP_CUDA_OK(cudaEventRecord(D.uploaded, cs_of(d)));
    }

    // Hazard phases are global: phase p + 1 may overwrite what ANY device still reads in phase p, so every device publishes
    // "my copy phase p is done" and the others wait for it before their phase p + 1 (copy and reload streams alike).
    const bool publish = n_ph > 1 && only_phase == 0;
    const int grid = c->opts[ETP_OPT_GRID_CTAS] > 0 ? (int)c->opts[ETP_OPT_GRID_CTAS] : c->n_sms;
    const bool timed = c->opts[ETP_OPT_TIME_KERNELS] != 0;
    int launches = 0;
    // ---- kernel (a) on each device's copy stream, one launch per hazard phase
    for (size_t p = 0; p < n_ph; ++p) {
        for (size_t d = 0; d < n_dev; ++d) {
            DevState& D = x->dev[d];
            DevPlan& P = plan[d];
            const JobList& jl = w->dev[d].phases[p];
            cudaStream_t cs = cs_of(d);
            ETP_CUDA_OK(cudaSetDevice(D.device));
            if (multi && publish && p > 0)
                for (size_t o = 0; o < n_dev; ++o)
                    if (o != d) ETP_CUDA_OK(cudaStreamWaitEvent(cs, x->dev[o].phase_ev[p - 1], 0));
            if (!jl.empty() && !skip_d2d && phase_on(p)) {
                const Off& o = P.off[p];
                CopyArgs a;
                a.bulk = (const BulkSeg*)(P.d_base + o.bulk);
                a.vec = (const VecSeg*)(P.d_base + o.vec);
                a.bulk_items = (const uint32_t*)(P.d_base + o.bulk_items);
                a.vec_items = (const uint32_t*)(P.d_base + o.vec_items);
                a.pairs = (const int2*)(P.d_base + P.off_pairs);
                a.n_bulk_items = jl.n_bulk_items;
                a.n_vec_items = jl.n_vec_items;
                a.small = (const SmallSeg*)(P.d_base + o.small);
                a.small_first = (const uint32_t*)(P.d_base + o.small_first);
                a.n_small_batches = (unsigned int)jl.small_first.size();
                a.dev_counts = nullptr;
                a.counters = (unsigned int*)(P.d_base + P.off_counters) + 2 * P.counter_slot;
                a.flags = c->opts[ETP_OPT_LDG_STEALS_BULK] ? 1u : 0u;
                if (timed) {
                    while ((int)D.tev.size() < 2 * (D.n_timed + 1)) {
                        cudaEvent_t e;
                        ETP_CUDA_OK(cudaEventCreate(&e));
                        D.tev.push_back(e);
                    }
                    ETP_CUDA_OK(cudaEventRecord(D.tev[2 * D.n_timed], cs));
                }
                launch_copy_kernel(a, grid, cs, c->opts[ETP_OPT_SMALL_STAGED] && jl.n_bulk_items == 0 && !jl.small_first.empty());
                ETP_CUDA_OK(cudaGetLastError());
                if (timed) {
                    ETP_CUDA_OK(cudaEventRecord(D.tev[2 * D.n_timed + 1], cs));
                    ++D.n_timed;
                }
                ++launches;
                ++D.rep.n_kernel_launches;
            }
            if (!jl.empty()) ++P.counter_slot;
            if (publish) {
                ETP_TRY(ensure_phase_event(D, p));
                ETP_CUDA_OK(cudaEventRecord(D.phase_ev[p], cs));
            }
        }
    }

    // ---- pipeline (b) on each device's reload stream
    int64_t n_memcpys = 0;
    if (!skip_reload) {
        const int64_t chunk = c->opts[ETP_OPT_RELOAD_CHUNK_BYTES];
        for (size_t d = 0; d < n_dev; ++d) {
            DevState& D = x->dev[d];
            DevPlan& P = plan[d];
            DeviceWork& dw = w->dev[d];
            cudaStream_t cs = cs_of(d), rs = rs_of(d);
            ETP_CUDA_OK(cudaSetDevice(D.device));
            // DMAs in phase order so that a late-phase wait does not hold back hazard-free reloads
            std::stable_sort(dw.dma.begin(), dw.dma.end(), [](const DmaCopy& a, const DmaCopy& b) { return a.phase < b.phase; });
            bool gather_waited_upload = false;
            size_t di = 0;
            for (size_t p = 0; p < n_ph; ++p) {
                bool has_work = !dw.host_gather[p].vec.empty();
                for (size_t k = di; k < dw.dma.size() && !has_work; ++k) has_work = dw.dma[k].phase == (int32_t)p;
                if (p > 0 && has_work && publish)
                    for (size_t o = 0; o < n_dev; ++o)
                        if (o != d || cs != rs) ETP_CUDA_OK(cudaStreamWaitEvent(rs, x->dev[o].phase_ev[p - 1], 0));
                for (; di < dw.dma.size() && dw.dma[di].phase == (int32_t)p; ++di) {
                    if (!phase_on(p)) continue;
                    const DmaCopy& m = dw.dma[di];
                    for (int64_t o = 0; o < m.bytes; o += chunk) {
                        const int64_t n = std::min(chunk, m.bytes - o);
                        ETP_CUDA_OK(cudaMemcpyAsync((char*)m.dst + o, (const char*)m.src + o, n, cudaMemcpyHostToDevice, rs));
                        ++n_memcpys;
                        ++D.rep.n_memcpys;
                    }
                }
                const JobList& gl = dw.host_gather[p];
                if (!gl.vec.empty()) {
                    if (phase_on(p)) {
                        if (!gather_waited_upload && cs != rs) {
                            ETP_CUDA_OK(cudaStreamWaitEvent(rs, D.uploaded, 0));
                            gather_waited_upload = true;
                        }
                        const Off& o = P.off[p];
                        CopyArgs a;
                        a.bulk = nullptr;
                        a.bulk_items = nullptr;
                        a.vec = (const VecSeg*)(P.d_base + o.gat);
                        a.vec_items = (const uint32_t*)(P.d_base + o.gat_items);
                        a.pairs = (const int2*)(P.d_base + P.off_pairs);
                        a.n_bulk_items = 0;
                        a.small = nullptr;
                        a.small_first = nullptr;
                        a.n_small_batches = 0;
                        a.n_vec_items = gl.n_vec_items;
                        a.dev_counts = nullptr;
                        a.counters = (unsigned int*)(P.d_base + P.off_counters) + 2 * P.counter_slot;
                        a.flags = 0;
                        const int ggrid = (int)std::max<int64_t>(1, std::min<int64_t>(c->opts[ETP_OPT_GATHER_CTAS], c->n_sms));
                        launch_copy_kernel(a, ggrid, rs);
                        ETP_CUDA_OK(cudaGetLastError());
                        ++launches;
                        ++D.rep.n_kernel_launches;
                    }
                    ++P.counter_slot;
                }
            }
        }
    }

    // ---- arena bookkeeping and join: the caller's streams continue after every device has finished its share
    for (size_t d = 0; d < n_dev; ++d) {
        DevState& D = x->dev[d];
        DevPlan& P = plan[d];
        if (!P.slot && !multi) continue;
        ETP_CUDA_OK(cudaSetDevice(D.device));
        if (P.slot) {
            ETP_CUDA_OK(cudaEventRecord(P.slot->done_copy, cs_of(d)));
            ETP_CUDA_OK(cudaEventRecord(P.slot->done_reload, rs_of(d)));
            P.slot->busy = true;
        }
        if (multi) {
            ETP_CUDA_OK(cudaEventRecord(D.join_copy, D.copy));
            ETP_CUDA_OK(cudaEventRecord(D.join_reload, D.reload));
        }
    }
    ETP_CUDA_OK(cudaSetDevice(c->device));
    if (multi)
        for (size_t d = 0; d < n_dev; ++d) {
            ETP_CUDA_OK(cudaStreamWaitEvent(caller_cs, x->dev[d].join_copy, 0));
            ETP_CUDA_OK(cudaStreamWaitEvent(caller_rs, x->dev[d].join_reload, 0));
        }

    c->launches = launches;
    for (size_t d = 0; d < n_dev; ++d) {
        etp_reshard_report& r = x->dev[d].rep;
        const etp_reshard_report lowered = w->dev[d].rep;
        const int32_t kl = r.n_kernel_launches;
        const int64_t nm = r.n_memcpys;
        r = lowered;
        r.n_kernel_launches = kl;
        r.n_memcpys = nm;
        r.n_jobs = plan[d].n_jobs;
        r.n_units = plan[d].n_items;
        r.n_phases = w->rep.n_phases;
        w->rep.n_jobs += plan[d].n_jobs;
        w->rep.n_units += plan[d].n_items;
    }
    w->rep.n_memcpys = n_memcpys;
    w->rep.n_kernel_launches = launches;
    w->rep.lower_ms += now_ms() - t0;
    if (report) *report = w->rep;
    return ETP_OK;
}

}  // namespace etp

// ------------------------------------------------------------------------------------------------ C ABI device calls
extern "C" etp_status etp_reshard_params(etp_ctx* ctx, const etp_tensor* tensors, int32_t n_tensors,
                                         const etp_plan* const* plans, int32_t n_plans, void* copy_stream,
                                         void* reload_stream, etp_reshard_report* report) {
    if (!ctx) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_params: ctx is NULL");
    const double t0 = now_ms();
    ETP_CUDA_OK(cudaSetDevice(ctx->device));
    LoweredWork w;
    ETP_TRY(lower_params(ctx, tensors, n_tensors, plans, n_plans, &w));
    w.rep.lower_ms = now_ms() - t0;
    return execute(ctx, &w, copy_stream, reload_stream, report);
}

extern "C" etp_status etp_reshard_kv(etp_ctx* ctx, const etp_kv_geometry* geom, etp_page_table* pt,
                                     const etp_plan* head_plan, int32_t new_block_budget, int32_t* evicted_seqs_out,
                                     int32_t* n_evicted, void* copy_stream, void* reload_stream,
                                     etp_reshard_report* report) {
    if (!ctx || !geom || !pt || !head_plan || !n_evicted) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: NULL argument");
    const double t0 = now_ms();
    ETP_CUDA_OK(cudaSetDevice(ctx->device));
    if (new_block_budget < 0 || new_block_budget > geom->n_blocks)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: budget %d outside [0, n_blocks=%d]", new_block_budget, geom->n_blocks);
    if (head_plan->total_units < 1) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: empty head plan");
    if (geom->block_size < 1) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: block_size %d < 1", geom->block_size);
    if (pt->n_seqs < 0 || pt->max_blocks < 0 || (pt->n_seqs > 0 && (!pt->block_table || !pt->seq_lens || !pt->last_use)))
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: bad page table");
    // Nothing of the caller's is written before the whole call is known to succeed: the page-table rule runs on a PRIVATE
    // copy of the table, the plan is lowered (geometry, capacity, backup range, alignment, hazard analysis) against it, and
    // only then are the new table and the eviction list copied out and the work enqueued.
    int64_t max_pairs = 0;
    for (int32_t s = 0; s < pt->n_seqs; ++s) {
        if (pt->seq_lens[s] < 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: negative seq_len");
        const int32_t need = (pt->seq_lens[s] + geom->block_size - 1) / geom->block_size;
        max_pairs += need;
        for (int32_t i = 0; i < need && i < pt->max_blocks; ++i) {
            const int32_t b = pt->block_table[(int64_t)s * pt->max_blocks + i];
            if (b >= geom->n_blocks) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: block id %d >= n_blocks %d", b, geom->n_blocks);
        }
    }
    const size_t table_n = (size_t)pt->n_seqs * (size_t)pt->max_blocks;
    std::vector<int32_t> table(pt->block_table, pt->block_table + table_n);
    etp_page_table priv = *pt;
    priv.block_table = table.data();
    std::vector<int32_t> pairs((size_t)std::max<int64_t>(max_pairs, 1) * 2);
    std::vector<int32_t> ev((size_t)std::max(pt->n_seqs, 1));
    int64_t n_pairs = 0;
    int32_t n_ev = 0;
    ETP_TRY(etp_page_table_rewrite(&priv, geom->block_size, new_block_budget, ev.data(), &n_ev, pairs.data(), max_pairs, &n_pairs));
    bool needs_backup = false;
    for (const etp_task& t : head_plan->tasks) needs_backup = needs_backup || (t.kind == ETP_RELOAD && t.begin < t.end);
    if (needs_backup && !geom->host_backup) {
        // reading K4: without a backup the reloaded heads stay missing, so every surviving sequence is reported too.  Their
        // rows stay mapped and their TRANSFER / relocated heads are still moved: the surviving heads are valid where the new
        // table says, and a replay (out of scope) would only have to refill the missing heads.
        std::vector<char> gone((size_t)std::max(pt->n_seqs, 1), 0);
        for (int32_t i = 0; i < n_ev; ++i) gone[ev[i]] = 1;
        for (int32_t s = 0; s < pt->n_seqs; ++s)
            if (!gone[s] && pt->seq_lens[s] > 0) ev[n_ev++] = s;
    }
    LoweredWork w;
    ETP_TRY(lower_kv(ctx, geom, head_plan, pairs.data(), n_pairs, &w));
    w.rep.lower_ms = now_ms() - t0;
    ETP_TRY(execute(ctx, &w, copy_stream, reload_stream, report));   // capacity checks come before its first enqueue
    // Phase-by-phase runs (ETP_OPT_ONLY_PHASE = k > 0): every phase call must lower the SAME plan, i.e. see the ORIGINAL table - a
    // rewritten one would give identity {old, new} pairs and the later phases would read the source pools at the new block ids.  So
    // such a call leaves the caller's table alone (the eviction list, a pure function of the inputs, is still reported); the caller
    // applies etp_page_table_rewrite itself after the last phase (include/etp.h).
    if (table_n && ctx->opts[ETP_OPT_ONLY_PHASE] == 0) std::memcpy(pt->block_table, table.data(), table_n * sizeof(int32_t));
    *n_evicted = n_ev;
    if (evicted_seqs_out)
        for (int32_t i = 0; i < n_ev; ++i) evicted_seqs_out[i] = ev[i];
    return ETP_OK;
}

extern "C" etp_status etp_debug_starved_wait(etp_ctx* ctx, void* stream) {
    if (!ctx) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_debug_starved_wait: ctx is NULL");
    ETP_CUDA_OK(cudaSetDevice(ctx->device));
    launch_starved_wait_kernel((cudaStream_t)stream);
    ETP_CUDA_OK(cudaGetLastError());
    ETP_CUDA_OK(cudaStreamSynchronize((cudaStream_t)stream));   // returns the trap as a sticky error -> ETP_ERR_CUDA + the record
    ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_debug_starved_wait: the starved kernel returned without an error");
}

extern "C" etp_status etp_copy_intervals(etp_ctx* ctx, const etp_interval* host_descs, int64_t n, void* stream,
                                         etp_reshard_report* report) {
    if (!ctx || n < 0 || (n > 0 && !host_descs)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: bad arguments");
    const double t0 = now_ms();
    const bool device_path = n >= kDeviceLoweringMin;
    // the contract of include/etp.h (etp_validate.cpp): argument checks always on the host-lowered path, the disjointness check
    // unless the caller switched it off
    if (ctx->opts[ETP_OPT_VALIDATE_INTERVALS]) {
        ETP_TRY(validate_intervals(host_descs, n, true));
    } else if (!device_path) {
        ETP_TRY(validate_intervals(host_descs, n, false));
    }
    if (device_path) {
        // 10^5 .. 10^6 intervals: the raw records are uploaded in chunks and lowered by kernels while the previous chunk is being
        // copied (without the validation above, argument errors of a later chunk surface after earlier chunks were enqueued)
        ETP_TRY(copy_intervals_device(ctx, host_descs, n, stream, report));
        if (report) report->lower_ms = now_ms() - t0;
        return ETP_OK;
    }
    LoweredWork w;
    w.dev.resize(1);   // the intervals are raw addresses: everything runs on the ctx's first logical device
    w.dev[0].phases.resize(1);
    w.dev[0].phases[0].small.reserve((size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        const etp_interval& d = host_descs[i];
        if (d.bytes == 0) continue;
        push_contiguous(ctx, &w.dev[0].phases[0], d.src, d.dst, d.bytes);
        w.rep.d2d_bytes += d.bytes;
        w.dev[0].rep.d2d_bytes += d.bytes;
    }
    w.rep.n_phases = 1;
    w.rep.lower_ms = now_ms() - t0;
    return execute(ctx, &w, stream, stream, report);
}

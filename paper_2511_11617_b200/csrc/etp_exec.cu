// Context, options and the executor: uploads descriptors, launches kernel (a) per hazard phase on the copy stream and
// runs the reload pipeline (b) on the reload stream.  PAPER.md:162-166: "issuing host-to-device reloads alongside GPU P2P
// transfers, allowing the P2P portions to be hidden beneath the PCIe-bound reload time".
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
struct CtxExtra {
    ArenaSlot slot[kArenaSlots];
    int next = 0;
    cudaEvent_t uploaded = nullptr;
};
CtxExtra* extra(etp_ctx* c) { return reinterpret_cast<CtxExtra*>(c->impl); }

double now_ms() {
    return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count();
}
}  // namespace

extern "C" etp_status etp_ctx_create(int device, int64_t staging_bytes, etp_ctx** out) {
    if (!out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_create: out is NULL");
    *out = nullptr;
    if (staging_bytes < 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_ctx_create: staging_bytes < 0");
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) {
        cudaGetLastError();
        ETP_FAIL(ETP_ERR_CUDA, "etp_ctx_create: CUDA device %d not available (%d devices); there is no CPU fallback", device, n_dev);
    }
    cudaDeviceProp prop;
    ETP_CUDA_OK(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) ETP_FAIL(ETP_ERR_CUDA, "etp_ctx_create: device %d is sm_%d%d; this library is built for sm_100a only", device, prop.major, prop.minor);
    ETP_CUDA_OK(cudaSetDevice(device));
    etp_ctx* c = new (std::nothrow) etp_ctx();
    if (!c) ETP_FAIL(ETP_ERR_NOMEM, "etp_ctx_create: out of memory");
    c->device = device;
    c->n_sms = prop.multiProcessorCount;
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
    CtxExtra* x = new (std::nothrow) CtxExtra();
    if (!x) { delete c; ETP_FAIL(ETP_ERR_NOMEM, "etp_ctx_create: out of memory"); }
    c->impl = x;
    cudaError_t e = cudaEventCreateWithFlags(&x->uploaded, cudaEventDisableTiming);
    for (int i = 0; i < kArenaSlots && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&x->slot[i].done_copy, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&x->slot[i].done_reload, cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = configure_copy_kernel();
    if (e != cudaSuccess) {
        set_error("etp_ctx_create: %s", cudaGetErrorString(e));
        etp_ctx_destroy(c);
        return ETP_ERR_CUDA;
    }
    *out = c;
    return ETP_OK;
}

extern "C" void etp_ctx_destroy(etp_ctx* c) {
    if (!c) return;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    CtxExtra* x = extra(c);
    if (x) {
        for (int i = 0; i < kArenaSlots; ++i) {
            if (x->slot[i].h) cudaFreeHost(x->slot[i].h);
            if (x->slot[i].d) cudaFree(x->slot[i].d);
            if (x->slot[i].done_copy) cudaEventDestroy(x->slot[i].done_copy);
            if (x->slot[i].done_reload) cudaEventDestroy(x->slot[i].done_reload);
        }
        if (x->uploaded) cudaEventDestroy(x->uploaded);
        delete x;
    }
    for (cudaEvent_t e : c->events) cudaEventDestroy(e);
    for (cudaEvent_t e : c->tev) cudaEventDestroy(e);
    etp::lin_teardown(c);
    if (c->moe_items) cudaFree(c->moe_items);
    cudaGetLastError();
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
    for (int32_t i = 0; i < c->n_timed; ++i) {
        float t = 0;
        ETP_CUDA_OK(cudaEventSynchronize(c->tev[2 * i + 1]));
        ETP_CUDA_OK(cudaEventElapsedTime(&t, c->tev[2 * i], c->tev[2 * i + 1]));
        ms += t;
    }
    *ms_out = ms;
    *n_out = c->n_timed;
    return ETP_OK;
}

namespace etp {

static etp_status ensure_event(etp_ctx* c, size_t i) {
    while (c->events.size() <= i) {
        cudaEvent_t e;
        ETP_CUDA_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        c->events.push_back(e);
    }
    return ETP_OK;
}

etp_status execute(etp_ctx* c, LoweredWork* w, void* copy_stream_v, void* reload_stream_v, etp_reshard_report* report) {
    const double t0 = now_ms();
    cudaStream_t cs = (cudaStream_t)copy_stream_v, rs = (cudaStream_t)reload_stream_v;
    ETP_CUDA_OK(cudaSetDevice(c->device));
    CtxExtra* x = extra(c);
    const bool skip_d2d = c->opts[ETP_OPT_SKIP_D2D] != 0, skip_reload = c->opts[ETP_OPT_SKIP_RELOAD] != 0;
    size_t n_ph = std::max(w->phases.size(), w->host_gather.size());
    for (const DmaCopy& d : w->dma) n_ph = std::max(n_ph, (size_t)d.phase + 1);   // a reload may be the last phase
    w->phases.resize(n_ph);
    w->host_gather.resize(n_ph);

    // ---- descriptor arena layout: work-queue heads (zero) | pairs | per phase: bulk segs, bulk items, vec segs, vec items,
    //      small segs, batch starts, gather segs, gather items.  The queue heads travel with the descriptors, so the
    //      done_copy / done_reload events that guard an arena slot also guard its counters: a call whose zero-copy gather is
    //      still queued behind GBs of DMA on the reload stream cannot have its heads reset by the next call.
    int64_t total = 0, n_jobs = 0, n_items = 0;
    auto pad = [](int64_t b) { return (b + 255) & ~int64_t(255); };
    struct Off { int64_t bulk, bulk_items, vec, vec_items, small, small_first, gat, gat_items; };
    std::vector<Off> off(n_ph);
    int launches_needed = 0;
    for (size_t p = 0; p < n_ph; ++p) launches_needed += (!w->phases[p].empty()) + (!w->host_gather[p].vec.empty());
    const int64_t off_counters = 0;
    total += pad((int64_t)launches_needed * 2 * sizeof(unsigned int));
    const int64_t off_pairs = total;
    total += pad((int64_t)w->pairs.size() * sizeof(int32_t));
    for (size_t p = 0; p < n_ph; ++p) {
        const JobList &jl = w->phases[p], &gl = w->host_gather[p];
        off[p].bulk = total;        total += pad((int64_t)jl.bulk.size() * sizeof(BulkSeg));
        off[p].bulk_items = total;  total += pad((int64_t)jl.n_bulk_items * sizeof(uint32_t));
        off[p].vec = total;         total += pad((int64_t)jl.vec.size() * sizeof(VecSeg));
        off[p].vec_items = total;   total += pad((int64_t)jl.n_vec_items * sizeof(uint32_t));
        off[p].small = total;       total += pad((int64_t)jl.small.size() * sizeof(SmallSeg));
        off[p].small_first = total; total += pad((int64_t)(jl.small_first.size() + 1) * sizeof(uint32_t));
        off[p].gat = total;         total += pad((int64_t)gl.vec.size() * sizeof(VecSeg));
        off[p].gat_items = total;   total += pad((int64_t)gl.n_vec_items * sizeof(uint32_t));
        n_jobs += (int64_t)(jl.bulk.size() + jl.vec.size() + jl.small.size() + gl.vec.size());
        n_items += (int64_t)jl.n_bulk_items + jl.n_vec_items + (int64_t)jl.small_first.size() + gl.n_vec_items;
        if (jl.bulk.size() >= 0xFFFFFFF0ull || jl.vec.size() >= 0xFFFFFFF0ull || jl.small.size() >= 0xFFFFFFF0ull ||
            gl.vec.size() >= 0xFFFFFFF0ull || (uint64_t)jl.n_vec_items + jl.small_first.size() >= 0xFFFFFFF0ull)
            ETP_FAIL(ETP_ERR_CAPACITY, "too many segments in one phase");
    }
    if (launches_needed > kCounterSlots) ETP_FAIL(ETP_ERR_CAPACITY, "plan needs %d launches > %d", launches_needed, kCounterSlots);

    // item table: the segment index of every work item, one fill per segment
    auto fill_items = [](uint32_t* items, uint32_t n_items_total, const uint32_t* firsts, size_t n_segs, size_t stride) {
        for (size_t i = 0; i < n_segs; ++i) {
            const uint32_t b = *(const uint32_t*)((const char*)firsts + i * stride);
            const uint32_t e = i + 1 < n_segs ? *(const uint32_t*)((const char*)firsts + (i + 1) * stride) : n_items_total;
            std::fill(items + b, items + e, (uint32_t)i);
        }
    };

    char* d_base = nullptr;
    ArenaSlot* slot = nullptr;
    if (n_jobs > 0) {
        slot = &x->slot[x->next];
        x->next = (x->next + 1) % kArenaSlots;
        if (slot->busy) {  // the call that used this slot two calls ago must have consumed its descriptors
            ETP_CUDA_OK(cudaEventSynchronize(slot->done_copy));
            ETP_CUDA_OK(cudaEventSynchronize(slot->done_reload));
            slot->busy = false;
        }
        if (slot->bytes < total) {
            if (slot->h) cudaFreeHost(slot->h);
            if (slot->d) cudaFree(slot->d);
            slot->h = slot->d = nullptr;
            slot->bytes = 0;
            const int64_t want = std::max<int64_t>(total + total / 4, 1 << 20);
            ETP_CUDA_OK(cudaMallocHost(&slot->h, want));
            ETP_CUDA_OK(cudaMalloc(&slot->d, want));
            slot->bytes = want;
        }
        char* h = (char*)slot->h;
        std::memset(h + off_counters, 0, (size_t)launches_needed * 2 * sizeof(unsigned int));
        if (!w->pairs.empty()) std::memcpy(h + off_pairs, w->pairs.data(), w->pairs.size() * sizeof(int32_t));
        for (size_t p = 0; p < n_ph; ++p) {
            const JobList &jl = w->phases[p], &gl = w->host_gather[p];
            if (!jl.bulk.empty()) {
                std::memcpy(h + off[p].bulk, jl.bulk.data(), jl.bulk.size() * sizeof(BulkSeg));
                fill_items((uint32_t*)(h + off[p].bulk_items), jl.n_bulk_items, &jl.bulk[0].first_item, jl.bulk.size(), sizeof(BulkSeg));
            }
            if (!jl.vec.empty()) {
                std::memcpy(h + off[p].vec, jl.vec.data(), jl.vec.size() * sizeof(VecSeg));
                fill_items((uint32_t*)(h + off[p].vec_items), jl.n_vec_items, &jl.vec[0].first_item, jl.vec.size(), sizeof(VecSeg));
            }
            if (!jl.small.empty()) {
                std::memcpy(h + off[p].small, jl.small.data(), jl.small.size() * sizeof(SmallSeg));
                uint32_t* f = (uint32_t*)(h + off[p].small_first);
                std::memcpy(f, jl.small_first.data(), jl.small_first.size() * sizeof(uint32_t));
                f[jl.small_first.size()] = (uint32_t)jl.small.size();
            }
            if (!gl.vec.empty()) {
                std::memcpy(h + off[p].gat, gl.vec.data(), gl.vec.size() * sizeof(VecSeg));
                fill_items((uint32_t*)(h + off[p].gat_items), gl.n_vec_items, &gl.vec[0].first_item, gl.vec.size(), sizeof(VecSeg));
            }
        }
        d_base = (char*)slot->d;
        ETP_CUDA_OK(cudaMemcpyAsync(d_base, h, total, cudaMemcpyHostToDevice, cs));
        ETP_CUDA_OK(cudaEventRecord(x->uploaded, cs));
    }

    // which phases must publish an event for the reload stream
    std::vector<char> need_event(n_ph + 1, 0);
    if (!skip_reload) {
        for (const DmaCopy& d : w->dma)
            if (d.phase > 0) need_event[d.phase - 1] = 1;
        for (size_t p = 1; p < n_ph; ++p)
            if (!w->host_gather[p].vec.empty()) need_event[p - 1] = 1;
    }

    const int grid = c->opts[ETP_OPT_GRID_CTAS] > 0 ? (int)c->opts[ETP_OPT_GRID_CTAS] : c->n_sms;
    int counter_slot = 0, launches = 0;
    const bool timed = c->opts[ETP_OPT_TIME_KERNELS] != 0;
    c->n_timed = 0;
    // ---- kernel (a) on the copy stream, one launch per hazard phase
    for (size_t p = 0; p < n_ph; ++p) {
        const JobList& jl = w->phases[p];
        if (!jl.empty() && !skip_d2d) {
            CopyArgs a;
            a.bulk = (const BulkSeg*)(d_base + off[p].bulk);
            a.vec = (const VecSeg*)(d_base + off[p].vec);
            a.bulk_items = (const uint32_t*)(d_base + off[p].bulk_items);
            a.vec_items = (const uint32_t*)(d_base + off[p].vec_items);
            a.pairs = (const int2*)(d_base + off_pairs);
            a.n_bulk_items = jl.n_bulk_items;
            a.n_vec_items = jl.n_vec_items;
            a.small = (const SmallSeg*)(d_base + off[p].small);
            a.small_first = (const uint32_t*)(d_base + off[p].small_first);
            a.n_small_batches = (unsigned int)jl.small_first.size();
            a.counters = (unsigned int*)(d_base + off_counters) + 2 * counter_slot;
            a.flags = c->opts[ETP_OPT_LDG_STEALS_BULK] ? 1u : 0u;
            if (timed) {
                while ((int)c->tev.size() < 2 * (c->n_timed + 1)) {
                    cudaEvent_t e;
                    ETP_CUDA_OK(cudaEventCreate(&e));
                    c->tev.push_back(e);
                }
                ETP_CUDA_OK(cudaEventRecord(c->tev[2 * c->n_timed], cs));
            }
            launch_copy_kernel(a, grid, cs);
            ETP_CUDA_OK(cudaGetLastError());
            if (timed) {
                ETP_CUDA_OK(cudaEventRecord(c->tev[2 * c->n_timed + 1], cs));
                ++c->n_timed;
            }
            ++launches;
        }
        if (!jl.empty()) ++counter_slot;
        if (need_event[p]) {
            ETP_TRY(ensure_event(c, p));
            ETP_CUDA_OK(cudaEventRecord(c->events[p], cs));
        }
    }

    // ---- pipeline (b) on the reload stream
    int64_t n_memcpys = 0;
    if (!skip_reload) {
        const int64_t chunk = c->opts[ETP_OPT_RELOAD_CHUNK_BYTES];
        // DMAs in phase order so that a late-phase wait does not hold back hazard-free reloads
        std::stable_sort(w->dma.begin(), w->dma.end(), [](const DmaCopy& a, const DmaCopy& b) { return a.phase < b.phase; });
        bool gather_waited_upload = false;
        size_t di = 0;
        for (size_t p = 0; p < n_ph; ++p) {
            bool has_work = !w->host_gather[p].vec.empty();
            for (size_t k = di; k < w->dma.size() && !has_work; ++k) has_work = w->dma[k].phase == (int32_t)p;
            if (p > 0 && has_work && cs != rs) ETP_CUDA_OK(cudaStreamWaitEvent(rs, c->events[p - 1], 0));
            for (; di < w->dma.size() && w->dma[di].phase == (int32_t)p; ++di) {
                const DmaCopy& d = w->dma[di];
                for (int64_t o = 0; o < d.bytes; o += chunk) {
                    const int64_t n = std::min(chunk, d.bytes - o);
                    ETP_CUDA_OK(cudaMemcpyAsync((char*)d.dst + o, (const char*)d.src + o, n, cudaMemcpyHostToDevice, rs));
                    ++n_memcpys;
                }
            }
            const JobList& gl = w->host_gather[p];
            if (!gl.vec.empty()) {
                if (!gather_waited_upload && cs != rs) {
                    ETP_CUDA_OK(cudaStreamWaitEvent(rs, x->uploaded, 0));
                    gather_waited_upload = true;
                }
                CopyArgs a;
                a.bulk = nullptr;
                a.bulk_items = nullptr;
                a.vec = (const VecSeg*)(d_base + off[p].gat);
                a.vec_items = (const uint32_t*)(d_base + off[p].gat_items);
                a.pairs = (const int2*)(d_base + off_pairs);
                a.n_bulk_items = 0;
                a.small = nullptr;
                a.small_first = nullptr;
                a.n_small_batches = 0;
                a.n_vec_items = gl.n_vec_items;
                a.counters = (unsigned int*)(d_base + off_counters) + 2 * counter_slot;
                a.flags = 0;
                const int ggrid = (int)std::max<int64_t>(1, std::min<int64_t>(c->opts[ETP_OPT_GATHER_CTAS], c->n_sms));
                launch_copy_kernel(a, ggrid, rs);
                ETP_CUDA_OK(cudaGetLastError());
                ++launches;
                ++counter_slot;
            }
        }
    }
    if (slot) {
        ETP_CUDA_OK(cudaEventRecord(slot->done_copy, cs));
        ETP_CUDA_OK(cudaEventRecord(slot->done_reload, rs));
        slot->busy = true;
    }
    c->launches = launches;
    w->rep.n_jobs = n_jobs;
    w->rep.n_units = n_items;
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
    if (table_n) std::memcpy(pt->block_table, table.data(), table_n * sizeof(int32_t));
    *n_evicted = n_ev;
    if (evicted_seqs_out)
        for (int32_t i = 0; i < n_ev; ++i) evicted_seqs_out[i] = ev[i];
    return ETP_OK;
}

extern "C" etp_status etp_copy_intervals(etp_ctx* ctx, const etp_interval* host_descs, int64_t n, void* stream,
                                         etp_reshard_report* report) {
    if (!ctx || n < 0 || (n > 0 && !host_descs)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: bad arguments");
    const double t0 = now_ms();
    LoweredWork w;
    w.phases.resize(1);
    w.phases[0].small.reserve((size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        const etp_interval& d = host_descs[i];
        if (d.bytes < 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: interval %lld has negative size", (long long)i);
        if (d.bytes == 0) continue;
        if (!d.src || !d.dst) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: interval %lld has a NULL pointer", (long long)i);
        if (((uintptr_t)d.src | (uintptr_t)d.dst | (uint64_t)d.bytes) & 15)
            ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_copy_intervals: interval %lld is not 16-byte aligned", (long long)i);
        push_contiguous(ctx, &w.phases[0], d.src, d.dst, d.bytes);
        w.rep.d2d_bytes += d.bytes;
    }
    if (ctx->opts[ETP_OPT_VALIDATE_INTERVALS]) {
        // the contract of include/etp.h: destinations mutually disjoint and disjoint from every source (one launch, no order
        // between intervals).  Sort both sides by start address, then one sweep each.
        struct Iv { uint64_t b, e; int64_t i; };
        std::vector<Iv> dst, src;
        dst.reserve((size_t)n);
        src.reserve((size_t)n);
        for (int64_t i = 0; i < n; ++i) {
            const etp_interval& d = host_descs[i];
            if (d.bytes == 0) continue;
            dst.push_back({(uint64_t)(uintptr_t)d.dst, (uint64_t)(uintptr_t)d.dst + (uint64_t)d.bytes, i});
            src.push_back({(uint64_t)(uintptr_t)d.src, (uint64_t)(uintptr_t)d.src + (uint64_t)d.bytes, i});
        }
        auto by_start = [](const Iv& a, const Iv& b) { return a.b < b.b; };
        std::sort(dst.begin(), dst.end(), by_start);
        std::sort(src.begin(), src.end(), by_start);
        for (size_t k = 1; k < dst.size(); ++k)
            if (dst[k].b < dst[k - 1].e)
                ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: destinations of intervals %lld and %lld overlap", (long long)dst[k - 1].i, (long long)dst[k].i);
        size_t si = 0;
        uint64_t src_reach = 0;   // largest end among the sources that start below the current destination's end
        int64_t src_reach_i = -1;
        for (const Iv& d : dst) {   // destinations are disjoint and ascending, so one forward pass over the sources suffices
            while (si < src.size() && src[si].b < d.e) {
                if (src[si].e > src_reach) { src_reach = src[si].e; src_reach_i = src[si].i; }
                ++si;
            }
            if (src_reach > d.b)
                ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: destination of interval %lld overlaps the source of interval %lld", (long long)d.i, (long long)src_reach_i);
        }
    }
    w.rep.n_phases = 1;
    w.rep.lower_ms = now_ms() - t0;
    return execute(ctx, &w, stream, stream, report);
}

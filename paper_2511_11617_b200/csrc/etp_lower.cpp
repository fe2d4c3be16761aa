// S3 — lowering a CMM plan onto concrete memory: unit intervals x (tensor, src slab, dst slab) -> byte descriptors of the
// copy kernel and DMA requests of the reload pipeline, with write-after-read hazard phases.
// PAPER.md:164 ("a single pass pre-allocates all destination buffers"), :178 (Transfer / Reload tasks on interval
// boundaries, range reads of only the needed byte intervals); layout contract: DESIGN.md readings L1-L7, K1-K6.
#include <algorithm>
#include <cstring>
#include <map>

#include "etp_internal.h"

namespace etp {

MemKind classify_pointer(const void* p) {
    cudaPointerAttributes a;
    std::memset(&a, 0, sizeof(a));
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return MEM_HOST_PAGEABLE;
    }
    if (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) return MEM_DEVICE;
    if (a.type == cudaMemoryTypeHost) return MEM_HOST_PINNED;
    return MEM_HOST_PAGEABLE;
}

// One contiguous interval -> one segment.  Large intervals go to the cp.async.bulk queue, where the kernel cuts them into
// kBulkItem pieces (so that 148 SMs balance even on a single 130 MB embedding interval); small ones to the vector queue.
void push_contiguous(const etp_ctx* ctx, JobList* jl, const void* src, void* dst, int64_t bytes) {
    if (bytes <= 0) return;
    const int64_t tma_min = ctx->opts[ETP_OPT_TMA_MIN_BYTES];
    jl->bytes += bytes;
    if (bytes >= tma_min) {
        jl->bulk.push_back({(uint64_t)(uintptr_t)src, (uint64_t)(uintptr_t)dst, (uint64_t)bytes, jl->n_bulk_items, 0});
        jl->n_bulk_items += (uint32_t)((bytes + kBulkItem - 1) / kBulkItem);
    } else if (bytes <= kVecItem) {
        const bool open = !jl->small_first.empty() && jl->small.size() - jl->small_first.back() < (size_t)kSmallBatchSegs &&
                          jl->open_batch_bytes + bytes <= kVecItem;
        if (!open) {
            jl->small_first.push_back((uint32_t)jl->small.size());
            jl->open_batch_bytes = 0;
        }
        jl->small.push_back({(uint64_t)(uintptr_t)src, (uint64_t)(uintptr_t)dst, (uint32_t)bytes, 0, 0});
        jl->open_batch_bytes += bytes;
    } else {
        VecSeg v{};
        v.src = (uint64_t)(uintptr_t)src;
        v.dst = (uint64_t)(uintptr_t)dst;
        v.kind = VEC_LINEAR;
        v.first_item = jl->n_vec_items;
        v.s_plane = bytes;
        jl->vec.push_back(v);
        jl->n_vec_items += (uint32_t)((bytes + kVecItem - 1) / kVecItem);
    }
}

namespace {
inline int64_t pmod(int64_t a, int64_t m) {
    int64_t r = a % m;
    return r < 0 ? r + m : r;
}

struct SlotRun {
    int64_t first_unit, count, src_slot, dst_slot;
};

// Split units [b,e) into runs over which both the source slot and the destination slot advance without wrapping.
// src_cap == 0 means "no slot addressing on the source side" (host image).
void slot_runs(int64_t b, int64_t e, int64_t src_anchor, int64_t src_cap, int64_t dst_anchor, int64_t dst_cap,
               std::vector<SlotRun>* out) {
    out->clear();
    int64_t u = b;
    while (u < e) {
        int64_t n = e - u;
        int64_t ss = 0, ds = pmod(u - dst_anchor, dst_cap);
        n = std::min(n, dst_cap - ds);
        if (src_cap > 0) {
            ss = pmod(u - src_anchor, src_cap);
            n = std::min(n, src_cap - ss);
        }
        out->push_back({u, n, ss, ds});
        u += n;
    }
}

struct Range {
    int32_t rank;
    int64_t b, e;  // slots
};

// Hazard phases (reading L4): task k must run after every task j that READS bytes k OVERWRITES.
// phase(k) = 0 if nothing reads what k writes, else 1 + max phase of those readers.  A cycle is unsupported.
// Cost: the read ranges are sorted per rank with a running maximum of their ends, every write range finds its readers
// with one binary search and a backward scan that stops as soon as no earlier read can reach it (reads of one plan are
// disjoint, so that is the readers themselves), then one longest-path sweep in topological order:
// O((R + W) log R + edges) for R read and W write ranges, instead of testing every pair of tasks in every round.
etp_status assign_phases(const std::vector<std::vector<Range>>& reads, const std::vector<std::vector<Range>>& writes,
                         std::vector<int32_t>* phase) {
    const size_t n = reads.size();
    phase->assign(n, 0);
    struct Rd { int32_t rank; int64_t b, e; uint32_t task; int64_t max_e; };
    std::vector<Rd> rd;
    for (size_t j = 0; j < n; ++j)
        for (const Range& r : reads[j])
            if (r.b < r.e) rd.push_back({r.rank, r.b, r.e, (uint32_t)j, 0});
    if (rd.empty()) return ETP_OK;
    std::sort(rd.begin(), rd.end(), [](const Rd& a, const Rd& b) { return a.rank != b.rank ? a.rank < b.rank : a.b < b.b; });
    for (size_t i = 0; i < rd.size(); ++i)
        rd[i].max_e = (i > 0 && rd[i - 1].rank == rd[i].rank) ? std::max(rd[i - 1].max_e, rd[i].e) : rd[i].e;
    // edges reader j -> writer k
    std::vector<std::pair<uint32_t, uint32_t>> edges;
    for (size_t k = 0; k < n; ++k)
        for (const Range& w : writes[k]) {
            if (w.b >= w.e) continue;
            // first read (rank, begin) >= (w.rank, w.e): everything before it on this rank begins below w.e
            size_t hi = std::lower_bound(rd.begin(), rd.end(), w, [](const Rd& a, const Range& w) {
                            return a.rank != w.rank ? a.rank < w.rank : a.b < w.e;
                        }) - rd.begin();
            while (hi > 0 && rd[hi - 1].rank == w.rank && rd[hi - 1].max_e > w.b) {
                const Rd& r = rd[hi - 1];
                if (r.e > w.b && r.task != k) edges.push_back({r.task, (uint32_t)k});
                --hi;
            }
        }
    if (edges.empty()) return ETP_OK;
    std::sort(edges.begin(), edges.end());
    edges.erase(std::unique(edges.begin(), edges.end()), edges.end());
    std::vector<uint32_t> first(n + 1, 0), indeg(n, 0);
    for (const auto& e : edges) { ++first[e.first + 1]; ++indeg[e.second]; }
    for (size_t i = 0; i < n; ++i) first[i + 1] += first[i];
    std::vector<uint32_t> ready;
    for (size_t i = 0; i < n; ++i)
        if (!indeg[i]) ready.push_back((uint32_t)i);
    size_t done = 0;
    while (!ready.empty()) {
        const uint32_t j = ready.back();
        ready.pop_back();
        ++done;
        for (uint32_t x = first[j]; x < first[j + 1]; ++x) {
            const uint32_t k = edges[x].second;
            (*phase)[k] = std::max((*phase)[k], (*phase)[j] + 1);
            if (--indeg[k] == 0) ready.push_back(k);
        }
    }
    if (done != n) ETP_FAIL(ETP_ERR_UNSUPPORTED, "cyclic write-after-read hazard between tasks (needs a bounce buffer)");
    return ETP_OK;
}

JobList& phase_list(std::vector<JobList>& v, int32_t p) {
    if ((int32_t)v.size() <= p) v.resize(p + 1);
    return v[p];
}
}  // namespace

// ------------------------------------------------------------------------------------------------ parameters
etp_status lower_params(const etp_ctx* ctx, const etp_tensor* tensors, int32_t n_tensors, const etp_plan* const* plans,
                        int32_t n_plans, LoweredWork* out) {
    if (n_tensors < 0 || n_plans < 0 || (n_tensors > 0 && (!tensors || !plans)))
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_params: NULL tensors/plans");
    std::vector<SlotRun> runs;
    std::map<std::vector<int64_t>, std::vector<int32_t>> phase_cache;
    int32_t max_phase = 0;
    out->dev.resize((size_t)n_logical_devices(ctx));
    for (int32_t t = 0; t < n_tensors; ++t) {
        const etp_tensor& T = tensors[t];
        if (T.plan_index < 0 || T.plan_index >= n_plans || !plans[T.plan_index])
            ETP_FAIL(ETP_ERR_INVALID_ARG, "tensor %d: plan_index %d out of range", t, T.plan_index);
        const etp_plan& P = *plans[T.plan_index];
        if (T.unit_bytes <= 0 || T.total_units != P.total_units)
            ETP_FAIL(ETP_ERR_INVALID_ARG, "tensor %d: total_units %lld does not match its plan (%lld) or unit_bytes <= 0", t,
                     (long long)T.total_units, (long long)P.total_units);
        if (T.unit_bytes % 16) ETP_FAIL(ETP_ERR_ALIGNMENT, "tensor %d: unit_bytes %lld is not a multiple of 16", t, (long long)T.unit_bytes);
        if (!T.slabs || T.n_ranks < 1) ETP_FAIL(ETP_ERR_INVALID_ARG, "tensor %d: no slabs", t);
        auto slab_of = [&](int32_t rank) -> const etp_slab* {
            return (rank >= 0 && rank < T.n_ranks) ? &T.slabs[rank] : nullptr;
        };
        // capacity: every new shard must fit its slab
        for (const etp_shard& s : P.new_layout) {
            const etp_slab* sl = slab_of(s.rank);
            if (!sl || (s.end > s.begin && !sl->base)) ETP_FAIL(ETP_ERR_INVALID_ARG, "tensor %d: no slab for rank %d", t, s.rank);
            if (sl->cap_units < 1 || s.end - s.begin > sl->cap_units)
                ETP_FAIL(ETP_ERR_CAPACITY, "tensor %d rank %d: new shard of %lld units does not fit cap_units %lld", t, s.rank,
                         (long long)(s.end - s.begin), (long long)sl->cap_units);
            if ((uintptr_t)sl->base % 16) ETP_FAIL(ETP_ERR_ALIGNMENT, "tensor %d rank %d: slab base not 16-byte aligned", t, s.rank);
        }
        MemKind image_kind = MEM_HOST_PAGEABLE;
        bool image_checked = false;

        // read / write slot ranges per task for the hazard analysis.  Slot ranges are in UNITS, so every tensor of a
        // granularity class with the same per-rank (anchor, cap) shares one phase vector (config 2: 4 analyses, not 282).
        const size_t nt = P.tasks.size();
        std::vector<int64_t> key;
        key.reserve(2 + 2 * (size_t)T.n_ranks);
        key.push_back(T.plan_index);
        key.push_back(T.n_ranks);
        for (int32_t r = 0; r < T.n_ranks; ++r) {
            key.push_back(T.slabs[r].base ? T.slabs[r].anchor_unit : 0);
            key.push_back(T.slabs[r].base ? T.slabs[r].cap_units : 0);
        }
        for (size_t k = 0; k < nt; ++k) {
            const etp_task& K = P.tasks[k];
            if (K.kind != ETP_TRANSFER || K.begin >= K.end) continue;
            const etp_slab* S = slab_of(K.src_rank);
            if (!S || !S->base || S->cap_units < 1) ETP_FAIL(ETP_ERR_INVALID_ARG, "tensor %d: no slab for source rank %d", t, K.src_rank);
            if ((uintptr_t)S->base % 16) ETP_FAIL(ETP_ERR_ALIGNMENT, "tensor %d rank %d: slab base not 16-byte aligned", t, K.src_rank);
            if (K.end - K.begin > S->cap_units) ETP_FAIL(ETP_ERR_CAPACITY, "tensor %d: transfer wider than the source slab", t);
        }
        auto hit = phase_cache.find(key);
        if (hit == phase_cache.end()) {
            std::vector<std::vector<Range>> reads(nt), writes(nt);
            for (size_t k = 0; k < nt; ++k) {
                const etp_task& K = P.tasks[k];
                if (K.kind == ETP_KEEP || K.begin >= K.end) continue;
                const etp_slab* D = slab_of(K.dst_rank);
                const etp_slab* S = K.kind == ETP_TRANSFER ? slab_of(K.src_rank) : nullptr;
                slot_runs(K.begin, K.end, S ? S->anchor_unit : 0, S ? S->cap_units : 0, D->anchor_unit, D->cap_units, &runs);
                for (const SlotRun& r : runs) {
                    writes[k].push_back({K.dst_rank, r.dst_slot, r.dst_slot + r.count});
                    if (S) reads[k].push_back({K.src_rank, r.src_slot, r.src_slot + r.count});
                }
            }
            std::vector<int32_t> ph;
            ETP_TRY(assign_phases(reads, writes, &ph));
            hit = phase_cache.emplace(std::move(key), std::move(ph)).first;
        }
        const std::vector<int32_t>& phase = hit->second;

        for (size_t k = 0; k < nt; ++k) {
            const etp_task& K = P.tasks[k];
            const int64_t bytes = (K.end - K.begin) * T.unit_bytes;
            if (K.kind == ETP_KEEP) {
                out->rep.kept_bytes += bytes;
                continue;
            }
            if (K.begin >= K.end) continue;
            max_phase = std::max(max_phase, phase[k]);   // the phase structure is global: every process agrees on it
            const etp_slab* D = slab_of(K.dst_rank);
            const int dv = device_of_rank(ctx, K.dst_rank);
            if (dv < 0) {   // a rank whose memory another process writes (its own executor pulls these bytes)
                out->rep.remote_bytes += bytes;
                continue;
            }
            DeviceWork& W = out->dev[(size_t)dv];
            if (K.kind == ETP_TRANSFER) {
                const etp_slab* S = slab_of(K.src_rank);
                slot_runs(K.begin, K.end, S->anchor_unit, S->cap_units, D->anchor_unit, D->cap_units, &runs);
                for (const SlotRun& r : runs) {
                    push_contiguous(ctx, &phase_list(W.phases, phase[k]), (const char*)S->base + r.src_slot * T.unit_bytes,
                                    (char*)D->base + r.dst_slot * T.unit_bytes, r.count * T.unit_bytes);
                }
                out->rep.d2d_bytes += bytes;
                W.rep.d2d_bytes += bytes;
            } else {  // RELOAD
                if (!T.host_image || K.begin < T.host_unit0 || K.end > T.host_unit0 + T.host_units)
                    ETP_FAIL(ETP_ERR_NO_SOURCE, "tensor %d: RELOAD [%lld,%lld) not covered by the host image", t,
                             (long long)K.begin, (long long)K.end);
                if ((uintptr_t)T.host_image % 16) ETP_FAIL(ETP_ERR_ALIGNMENT, "tensor %d: host image not 16-byte aligned", t);
                if (!image_checked) {
                    image_kind = classify_pointer(T.host_image);
                    image_checked = true;
                }
                slot_runs(K.begin, K.end, 0, 0, D->anchor_unit, D->cap_units, &runs);
                for (const SlotRun& r : runs) {
                    const char* src = (const char*)T.host_image + (r.first_unit - T.host_unit0) * T.unit_bytes;
                    char* dst = (char*)D->base + r.dst_slot * T.unit_bytes;
                    if (image_kind == MEM_DEVICE) {
                        push_contiguous(ctx, &phase_list(W.phases, phase[k]), src, dst, r.count * T.unit_bytes);
                    } else {
                        W.dma.push_back({src, dst, r.count * T.unit_bytes, phase[k]});
                    }
                }
                if (image_kind == MEM_DEVICE) { out->rep.reload_dev_bytes += bytes; W.rep.reload_dev_bytes += bytes; }
                else { out->rep.h2d_bytes += bytes; W.rep.h2d_bytes += bytes; }
            }
        }
    }
    out->rep.n_phases = std::max<int32_t>(out->rep.n_phases, max_phase + 1);
    return ETP_OK;
}

// ------------------------------------------------------------------------------------------------ paged KV
namespace {
struct PoolShape {
    int64_t plane, block, row, slot;  // byte strides: (layer,K|V) plane, block, token row (token-major) and head slot
};
PoolShape pool_shape(const etp_kv_geometry& g, int64_t heads) {
    const int64_t frag = (int64_t)g.head_dim * g.elem_bytes;
    PoolShape s;
    s.block = (int64_t)g.block_size * heads * frag;
    s.plane = (int64_t)g.n_blocks * s.block;
    if (g.layout == ETP_KV_TOKEN_MAJOR) {
        s.row = heads * frag;  // [token][slot][dim]
        s.slot = frag;
    } else {
        s.row = frag;  // [slot][token][dim]
        s.slot = (int64_t)g.block_size * frag;
    }
    return s;
}
}  // namespace

etp_status lower_kv(const etp_ctx* ctx, const etp_kv_geometry* gp, const etp_plan* head_plan, const int32_t* pairs,
                    int64_t n_pairs, LoweredWork* out) {
    const etp_kv_geometry& g = *gp;
    const etp_plan& P = *head_plan;
    if (g.n_layers < 1 || g.n_blocks < 1 || g.block_size < 1 || g.head_cap < 1 || g.head_dim < 1 || g.elem_bytes < 1 || g.n_ranks < 1 ||
        !g.pools || !g.head_anchor)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: bad geometry");
    if (g.layout != ETP_KV_TOKEN_MAJOR && g.layout != ETP_KV_HEAD_MAJOR) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: unknown layout");
    const int64_t frag = (int64_t)g.head_dim * g.elem_bytes;
    if (frag % 16) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_reshard_kv: fragment of %lld bytes is not a multiple of 16", (long long)frag);
    for (const etp_shard& s : P.new_layout) {
        if (s.rank < 0 || s.rank >= g.n_ranks || (s.end > s.begin && !g.pools[s.rank]))
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: no pool for rank %d", s.rank);
        if (s.end - s.begin > g.head_cap)
            ETP_FAIL(ETP_ERR_CAPACITY, "etp_reshard_kv: rank %d gets %lld heads > head_cap %d", s.rank, (long long)(s.end - s.begin), g.head_cap);
        if ((uintptr_t)g.pools[s.rank] % 16) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_reshard_kv: pool of rank %d not 16-byte aligned", s.rank);
    }
    const PoolShape dev = pool_shape(g, g.head_cap);
    const PoolShape bak = pool_shape(g, g.host_heads > 0 ? g.host_heads : 1);
    const int64_t n_planes = 2 * (int64_t)g.n_layers;
    MemKind backup_kind = g.host_backup ? classify_pointer(g.host_backup) : MEM_DEVICE;
    if (g.host_backup && backup_kind == MEM_HOST_PAGEABLE)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: host_backup must be pinned host or device memory");

    // hazard analysis at (rank, slot) granularity; relocations of kept heads only touch free blocks -> phase 0
    const size_t nt = P.tasks.size();
    std::vector<std::vector<Range>> reads(nt), writes(nt);
    std::vector<SlotRun> runs;
    for (size_t k = 0; k < nt; ++k) {
        const etp_task& K = P.tasks[k];
        if (K.kind == ETP_KEEP || K.begin >= K.end) continue;
        if (K.kind == ETP_TRANSFER && (K.src_rank < 0 || K.src_rank >= g.n_ranks || !g.pools[K.src_rank]))
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_reshard_kv: no pool for source rank %d", K.src_rank);
        const bool dev_src = K.kind == ETP_TRANSFER;
        slot_runs(K.begin, K.end, dev_src ? g.head_anchor[K.src_rank] : 0, dev_src ? g.head_cap : 0, g.head_anchor[K.dst_rank], g.head_cap, &runs);
        for (const SlotRun& r : runs) {
            writes[k].push_back({K.dst_rank, r.dst_slot, r.dst_slot + r.count});
            if (dev_src) reads[k].push_back({K.src_rank, r.src_slot, r.src_slot + r.count});
        }
    }
    std::vector<int32_t> phase;
    ETP_TRY(assign_phases(reads, writes, &phase));
    int32_t max_phase = 0;
    out->dev.resize((size_t)n_logical_devices(ctx));

    // pair lists on the device: [0, n_pairs) every surviving live block, [n_pairs, n_pairs + n_reloc) the relocated ones
    out->pairs.assign(pairs, pairs + 2 * n_pairs);
    int64_t n_reloc = 0;
    for (int64_t p = 0; p < n_pairs; ++p)
        if (pairs[2 * p] != pairs[2 * p + 1]) {
            out->pairs.push_back(pairs[2 * p]);
            out->pairs.push_back(pairs[2 * p + 1]);
            ++n_reloc;
        }

    for (size_t k = 0; k < nt; ++k) {
        const etp_task& K = P.tasks[k];
        if (K.begin >= K.end) continue;
        const int64_t live_bytes = (K.end - K.begin) * frag * g.block_size * n_planes * n_pairs;
        const char* src_base;
        const PoolShape* ss;
        const int dv = device_of_rank(ctx, K.dst_rank);   // KV heads are written by the device that holds the destination pool
        if (dv < 0) {
            if (K.kind != ETP_KEEP) out->rep.remote_bytes += live_bytes;
            continue;
        }
        DeviceWork& W = out->dev[(size_t)dv];
        std::vector<JobList>* dest = &W.phases;
        int64_t *counter, *dev_counter;
        if (K.kind == ETP_KEEP) {
            src_base = (const char*)g.pools[K.dst_rank];
            ss = &dev;
            slot_runs(K.begin, K.end, g.head_anchor[K.dst_rank], g.head_cap, g.head_anchor[K.dst_rank], g.head_cap, &runs);
            counter = &out->rep.d2d_bytes;
            dev_counter = &W.rep.d2d_bytes;
        } else if (K.kind == ETP_TRANSFER) {
            src_base = (const char*)g.pools[K.src_rank];
            ss = &dev;
            slot_runs(K.begin, K.end, g.head_anchor[K.src_rank], g.head_cap, g.head_anchor[K.dst_rank], g.head_cap, &runs);
            counter = &out->rep.d2d_bytes;
            dev_counter = &W.rep.d2d_bytes;
        } else {
            if (!g.host_backup) continue;  // reading K4: fragments left untouched; the caller reports the sequences
            if (K.begin < g.host_head0 || K.end > g.host_head0 + g.host_heads)
                ETP_FAIL(ETP_ERR_NO_SOURCE, "etp_reshard_kv: RELOAD heads [%lld,%lld) not covered by the backup", (long long)K.begin, (long long)K.end);
            if ((uintptr_t)g.host_backup % 16) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_reshard_kv: host_backup not 16-byte aligned");
            src_base = (const char*)g.host_backup;
            ss = &bak;
            slot_runs(K.begin, K.end, 0, 0, g.head_anchor[K.dst_rank], g.head_cap, &runs);
            for (SlotRun& r : runs) r.src_slot = r.first_unit - g.host_head0;
            if (backup_kind == MEM_DEVICE) {
                counter = &out->rep.reload_dev_bytes;
                dev_counter = &W.rep.reload_dev_bytes;
            } else {
                counter = &out->rep.h2d_bytes;
                dev_counter = &W.rep.h2d_bytes;
                dest = &W.host_gather;
            }
        }
        const int32_t ph = K.kind == ETP_KEEP ? 0 : phase[k];
        int64_t moved = 0;
        char* dst_base = (char*)g.pools[K.dst_rank];
        // KEEP heads move only inside relocated blocks; every other task touches every surviving live block
        const int64_t np_task = K.kind == ETP_KEEP ? n_reloc : n_pairs;
        const uint32_t pairs_first = K.kind == ETP_KEEP ? (uint32_t)n_pairs : 0u;
        if (np_task == 0) {
            if (K.kind == ETP_KEEP) out->rep.kept_bytes += live_bytes;
            continue;
        }
        for (const SlotRun& r : runs) {
            VecSeg v{};
            v.kind = VEC_PAGED;
            if (g.layout == ETP_KV_TOKEN_MAJOR) {  // block_size rows of (run of heads) per plane
                v.row_bytes = (uint32_t)(r.count * frag);
                v.rows_per_plane = (uint32_t)g.block_size;
                v.s_row = ss->row;
                v.d_row = dev.row;
            } else {  // one contiguous run of block_size * heads fragments per plane
                v.row_bytes = (uint32_t)(r.count * g.block_size * frag);
                v.rows_per_plane = 1;
            }
            const int64_t plane_bytes = (int64_t)v.row_bytes * v.rows_per_plane;
            v.planes_per_item = (uint32_t)std::min<int64_t>(n_planes, std::max<int64_t>(1, kVecItem / plane_bytes));
            v.n_planes = (uint32_t)n_planes;
            v.items_per_pair = (uint32_t)((n_planes + v.planes_per_item - 1) / v.planes_per_item);
            v.pairs_first = pairs_first;
            v.src = (uint64_t)(uintptr_t)(src_base + r.src_slot * ss->slot);
            v.dst = (uint64_t)(uintptr_t)(dst_base + r.dst_slot * dev.slot);
            v.s_plane = ss->plane;
            v.d_plane = dev.plane;
            v.s_block = ss->block;
            v.d_block = dev.block;
            JobList& jl = phase_list(*dest, ph);
            const int64_t items = np_task * v.items_per_pair;
            if (items + jl.n_vec_items >= 0xFFFFFFF0ll) ETP_FAIL(ETP_ERR_CAPACITY, "etp_reshard_kv: too many work items in one phase");
            v.first_item = jl.n_vec_items;
            jl.n_vec_items += (uint32_t)items;
            jl.vec.push_back(v);
            jl.bytes += np_task * n_planes * plane_bytes;
            moved += np_task * n_planes * plane_bytes;
        }
        *counter += moved;
        *dev_counter += moved;
        if (K.kind == ETP_KEEP) out->rep.kept_bytes += live_bytes - moved;
        if (moved) max_phase = std::max(max_phase, ph);
    }
    out->rep.n_phases = std::max<int32_t>(out->rep.n_phases, max_phase + 1);
    return ETP_OK;
}

}  // namespace etp

// Device-side lowering for etp_copy_intervals (config 5b: 10^5 .. 10^6 intervals per plan).  SURVEY.md 8(a) S3 / 8(d) row 5b.
//
// Lowering 10^6 intervals on the host costs ~24 ms (23 ns each: classify, batch, fill item tables, copy into the pinned arena)
// against a 6.6-ms copy kernel.  Here the raw 24-byte etp_interval records are uploaded as they are, in chunks, and three small
// kernels per chunk build exactly the descriptors the host lowering would have built (etp_internal.h):
//   count    one thread per interval: class (bulk >= TMA threshold / small <= 32 KiB / linear between) and its item count;
//            per-block sums of {bulk segs, bulk items, vec segs, vec items, small segs, small bytes}
//   scan     one block: exclusive scan of the block sums -> block bases, chunk totals (read back by the host: 48 bytes - the
//            item tables are sized from them), argument errors
//   scatter  per-block exclusive scan + base -> every interval writes its segment descriptor and fills its items' table
//            entries; small intervals also record the byte offset at which they start in the concatenation of all small ones
//   batches  small intervals are batched by 32-KiB windows of that concatenation (an interval is <= 32 KiB, so no window is
//            empty and the window index IS the batch index): the first interval of every window writes the batch start
// Chunks are triple-buffered: the upload and the lowering of chunks k+1 and k+2 run on a library-owned stream while the copy
// kernel of chunk k runs on the caller's stream, so the call costs about the copy kernels plus the first chunk's upload.
#include <algorithm>
#include <chrono>
#include <cstring>
#include <vector>

#include "etp_copy.cuh"

using namespace etp;

namespace {

constexpr int kChunk = 1 << 18;       // intervals per chunk (a launch of the copy kernel per chunk: 64 MiB even at 256 B per interval)
constexpr int kBlock = 1024;
constexpr int kSlots = 3;         // descriptors of chunk k are copied while chunks k+1 and k+2 are uploaded and counted
enum { C_BULK_SEGS = 0, C_BULK_ITEMS, C_VEC_SEGS, C_VEC_ITEMS, C_SMALL_SEGS, C_SMALL_BYTES, C_ALL_BYTES, C_N };

struct Totals {            // written by the scan kernel, copied to pinned host memory
    unsigned long long v[C_N];
    unsigned int bad_align, bad_size;   // first offending interval index + 1 (0 = none)
};

struct Tuple {
    unsigned long long v[C_N];
};

__device__ __forceinline__ void classify(const etp_interval& d, long long tma_min, Tuple* t) {
#pragma unroll
    for (int k = 0; k < C_N; ++k) t->v[k] = 0;
    const long long b = d.bytes;
    if (b <= 0) return;
    t->v[C_ALL_BYTES] = (unsigned long long)b;
    if (b >= tma_min) {
        t->v[C_BULK_SEGS] = 1;
        t->v[C_BULK_ITEMS] = (unsigned long long)((b + kBulkItem - 1) / kBulkItem);
    } else if (b <= kVecItem) {
        t->v[C_SMALL_SEGS] = 1;
        t->v[C_SMALL_BYTES] = (unsigned long long)b;
    } else {
        t->v[C_VEC_SEGS] = 1;
        t->v[C_VEC_ITEMS] = (unsigned long long)((b + kVecItem - 1) / kVecItem);
    }
}

// exclusive scan of one Tuple per thread over a block of kBlock threads; returns the block total in *total (all threads)
__device__ void block_exclusive_scan(Tuple* t, Tuple* total, unsigned long long (*warp_sums)[C_N]) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    Tuple incl = *t;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1)
#pragma unroll
        for (int k = 0; k < C_N; ++k) {
            const unsigned long long o = __shfl_up_sync(0xffffffffu, incl.v[k], d);
            if (lane >= d) incl.v[k] += o;
        }
    if (lane == 31)
#pragma unroll
        for (int k = 0; k < C_N; ++k) warp_sums[warp][k] = incl.v[k];
    __syncthreads();
    Tuple base, tot;
#pragma unroll
    for (int k = 0; k < C_N; ++k) {
        base.v[k] = 0;
        tot.v[k] = 0;
    }
    for (int w = 0; w < kBlock / 32; ++w)
#pragma unroll
        for (int k = 0; k < C_N; ++k) {
            const unsigned long long s = warp_sums[w][k];
            if (w < warp) base.v[k] += s;
            tot.v[k] += s;
        }
#pragma unroll
    for (int k = 0; k < C_N; ++k) t->v[k] = base.v[k] + incl.v[k] - t->v[k];
    *total = tot;
    __syncthreads();
}

__global__ void __launch_bounds__(kBlock) etp_iv_count_kernel(const etp_interval* iv, int n, long long tma_min, unsigned long long* block_sums,
                                                               unsigned int* bad) {
    __shared__ unsigned long long warp_sums[kBlock / 32][C_N];
    const int i = blockIdx.x * kBlock + threadIdx.x;
    Tuple t;
#pragma unroll
    for (int k = 0; k < C_N; ++k) t.v[k] = 0;
    if (i < n) {
        const etp_interval d = iv[i];
        if (d.bytes < 0) atomicMin(&bad[1], (unsigned int)i);
        else if (d.bytes > 0 && (((unsigned long long)d.src | (unsigned long long)d.dst | (unsigned long long)d.bytes) & 15ull || !d.src || !d.dst))
            atomicMin(&bad[0], (unsigned int)i);
        classify(d, tma_min, &t);
    }
    Tuple tot;
    block_exclusive_scan(&t, &tot, warp_sums);
    if (threadIdx.x == 0)
#pragma unroll
        for (int k = 0; k < C_N; ++k) block_sums[(size_t)blockIdx.x * C_N + k] = tot.v[k];
}

// one block: exclusive scan over the (<= 256) block sums; also zeroes the copy kernel's work-queue heads for this chunk
__global__ void etp_iv_scan_kernel(unsigned long long* block_sums, int n_blocks, Totals* totals, const unsigned int* bad, unsigned int* counters) {
    const int k = threadIdx.x;   // one thread per counter
    if (k < C_N) {
        unsigned long long run = 0;
        for (int b = 0; b < n_blocks; ++b) {
            const unsigned long long s = block_sums[(size_t)b * C_N + k];
            block_sums[(size_t)b * C_N + k] = run;
            run += s;
        }
        totals->v[k] = run;
    }
    if (k == 0) {
        totals->bad_align = bad[0] == 0xffffffffu ? 0u : bad[0] + 1u;
        totals->bad_size = bad[1] == 0xffffffffu ? 0u : bad[1] + 1u;
        counters[0] = 0;
        counters[1] = 0;
    }
}

struct ScatterOut {
    BulkSeg* bulk;
    uint32_t* bulk_items;
    VecSeg* vec;
    uint32_t* vec_items;
    SmallSeg* small;
};

__global__ void __launch_bounds__(kBlock) etp_iv_scatter_kernel(const etp_interval* iv, int n, long long tma_min, const unsigned long long* block_base,
                                                                 ScatterOut o) {
    __shared__ unsigned long long warp_sums[kBlock / 32][C_N];
    const int i = blockIdx.x * kBlock + threadIdx.x;
    Tuple t, mine;
    etp_interval d{nullptr, nullptr, 0};
    if (i < n) d = iv[i];
    classify(d, tma_min, &mine);
    t = mine;
    Tuple tot;
    block_exclusive_scan(&t, &tot, warp_sums);
#pragma unroll
    for (int k = 0; k < C_N; ++k) t.v[k] += block_base[(size_t)blockIdx.x * C_N + k];
    if (mine.v[C_BULK_SEGS]) {
        const uint32_t seg = (uint32_t)t.v[C_BULK_SEGS], first = (uint32_t)t.v[C_BULK_ITEMS];
        o.bulk[seg] = BulkSeg{(uint64_t)d.src, (uint64_t)d.dst, (uint64_t)d.bytes, first, 0};
        for (unsigned long long k = 0; k < mine.v[C_BULK_ITEMS]; ++k) o.bulk_items[first + k] = seg;
    } else if (mine.v[C_VEC_SEGS]) {
        const uint32_t seg = (uint32_t)t.v[C_VEC_SEGS], first = (uint32_t)t.v[C_VEC_ITEMS];
        VecSeg v{};
        v.src = (uint64_t)d.src;
        v.dst = (uint64_t)d.dst;
        v.kind = VEC_LINEAR;
        v.first_item = first;
        v.s_plane = d.bytes;
        o.vec[seg] = v;
        for (unsigned long long k = 0; k < mine.v[C_VEC_ITEMS]; ++k) o.vec_items[first + k] = seg;
    } else if (mine.v[C_SMALL_SEGS]) {
        // pad1 = the byte offset at which this interval starts in the concatenation of all small intervals of the chunk
        o.small[t.v[C_SMALL_SEGS]] = SmallSeg{(uint64_t)d.src, (uint64_t)d.dst, (uint32_t)d.bytes, 0, (uint64_t)t.v[C_SMALL_BYTES]};
    }
}

// Batches of small intervals = 32-KiB windows of their concatenation.  counts = {n_bulk_items, n_vec_items, n_small_batches}.
__global__ void etp_iv_batches_kernel(const SmallSeg* small, const Totals* totals, uint32_t* small_first, unsigned int* counts) {
    const unsigned long long n_small = totals->v[C_SMALL_SEGS];
    const unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j == 0) {
        counts[0] = (unsigned int)totals->v[C_BULK_ITEMS];
        counts[1] = (unsigned int)totals->v[C_VEC_ITEMS];
        if (n_small == 0) counts[2] = 0;
    }
    if (j >= n_small) return;
    const uint64_t w = small[j].pad1 / (uint64_t)kVecItem;
    if (j == 0 || small[j - 1].pad1 / (uint64_t)kVecItem != w) small_first[w] = (uint32_t)j;
    if (j == n_small - 1) {
        small_first[w + 1] = (uint32_t)n_small;
        counts[2] = (unsigned int)(w + 1);
    }
}

struct Slot {
    etp_interval* h_raw = nullptr;   // pinned staging: the host copies the caller's (pageable) records here, the DMA is then truly asynchronous
    etp_interval* d_raw = nullptr;
    unsigned long long* d_block_sums = nullptr;
    Totals* d_totals = nullptr;
    Totals* h_totals = nullptr;      // pinned
    unsigned int* d_bad = nullptr;   // {min index with an alignment error, min index with a negative size}
    unsigned int* d_counts = nullptr;   // 3 queue lengths + 2 queue heads
    BulkSeg* d_bulk = nullptr;
    VecSeg* d_vec = nullptr;
    SmallSeg* d_small = nullptr;
    uint32_t* d_small_first = nullptr;
    uint32_t *d_bulk_items = nullptr, *d_vec_items = nullptr;
    int64_t bulk_items_cap = 0, vec_items_cap = 0;
    cudaEvent_t uploaded = nullptr, totals_ready = nullptr, lowered = nullptr, copied = nullptr;
    bool busy = false, staged = false;
};
struct IvState {
    cudaStream_t side = nullptr;     // upload + lowering stream
    Slot slot[kSlots];
    std::vector<cudaEvent_t> timing;   // pairs around the copy launches of the last call (ETP_OPT_TIME_KERNELS)
    int n_timed = 0;
};

double now_ms() {
    return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

etp_status ensure_state(etp_ctx* c, IvState** out) {
    if (c->iv_state) {
        *out = static_cast<IvState*>(c->iv_state);
        return ETP_OK;
    }
    IvState* S = new (std::nothrow) IvState();
    if (!S) ETP_FAIL(ETP_ERR_NOMEM, "etp_copy_intervals: out of memory");
    c->iv_state = S;
    ETP_CUDA_OK(cudaStreamCreateWithFlags(&S->side, cudaStreamNonBlocking));
    const int n_blocks = kChunk / kBlock;
    for (Slot& s : S->slot) {
        ETP_CUDA_OK(cudaMallocHost(&s.h_raw, sizeof(etp_interval) * kChunk));
        ETP_CUDA_OK(cudaMalloc(&s.d_raw, sizeof(etp_interval) * kChunk));
        ETP_CUDA_OK(cudaMalloc(&s.d_block_sums, sizeof(unsigned long long) * C_N * n_blocks));
        ETP_CUDA_OK(cudaMalloc(&s.d_totals, sizeof(Totals)));
        ETP_CUDA_OK(cudaMallocHost(&s.h_totals, sizeof(Totals)));
        ETP_CUDA_OK(cudaMalloc(&s.d_bad, 2 * sizeof(unsigned int)));
        ETP_CUDA_OK(cudaMalloc(&s.d_counts, 8 * sizeof(unsigned int)));
        ETP_CUDA_OK(cudaMalloc(&s.d_bulk, sizeof(BulkSeg) * kChunk));
        ETP_CUDA_OK(cudaMalloc(&s.d_vec, sizeof(VecSeg) * kChunk));
        ETP_CUDA_OK(cudaMalloc(&s.d_small, sizeof(SmallSeg) * kChunk));
        ETP_CUDA_OK(cudaMalloc(&s.d_small_first, sizeof(uint32_t) * (kChunk + 2)));
        for (cudaEvent_t* e : {&s.uploaded, &s.totals_ready, &s.lowered, &s.copied}) ETP_CUDA_OK(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    }
    *out = S;
    return ETP_OK;
}

}  // namespace

namespace etp {

void free_interval_state(etp_ctx* c) {
    if (!c->iv_state) return;
    IvState* S = static_cast<IvState*>(c->iv_state);
    for (Slot& s : S->slot) {
        for (void* p : {(void*)s.d_raw, (void*)s.d_block_sums, (void*)s.d_totals, (void*)s.d_bad, (void*)s.d_counts, (void*)s.d_bulk, (void*)s.d_vec,
                        (void*)s.d_small, (void*)s.d_small_first, (void*)s.d_bulk_items, (void*)s.d_vec_items})
            if (p) cudaFree(p);
        if (s.h_totals) cudaFreeHost(s.h_totals);
        if (s.h_raw) cudaFreeHost(s.h_raw);
        for (cudaEvent_t e : {s.uploaded, s.totals_ready, s.lowered, s.copied})
            if (e) cudaEventDestroy(e);
    }
    for (cudaEvent_t e : S->timing) cudaEventDestroy(e);
    if (S->side) cudaStreamDestroy(S->side);
    delete S;
    c->iv_state = nullptr;
}

int interval_timed_launches(etp_ctx* c, double* ms) {
    *ms = 0;
    if (!c->iv_state) return 0;
    IvState* S = static_cast<IvState*>(c->iv_state);
    for (int i = 0; i < S->n_timed; ++i) {
        float t = 0;
        if (cudaEventSynchronize(S->timing[2 * i + 1]) == cudaSuccess && cudaEventElapsedTime(&t, S->timing[2 * i], S->timing[2 * i + 1]) == cudaSuccess) *ms += t;
    }
    return S->n_timed;
}

void reset_interval_timing(etp_ctx* c) {
    if (c->iv_state) static_cast<IvState*>(c->iv_state)->n_timed = 0;
}

// host_descs: host memory (pageable or pinned).  Everything runs on logical device 0 of the ctx.
etp_status copy_intervals_device(etp_ctx* c, const etp_interval* host_descs, int64_t n, void* stream_v, etp_reshard_report* report) {
    const double t0 = now_ms();
    cudaStream_t user = (cudaStream_t)stream_v;
    ETP_CUDA_OK(cudaSetDevice(c->device));
    IvState* S = nullptr;
    ETP_TRY(ensure_state(c, &S));
    note_slab_write(c, stream_v);
    S->n_timed = 0;
    const long long tma_min = c->opts[ETP_OPT_TMA_MIN_BYTES];
    const int grid = c->opts[ETP_OPT_GRID_CTAS] > 0 ? (int)c->opts[ETP_OPT_GRID_CTAS] : c->n_sms;
    const bool timed = c->opts[ETP_OPT_TIME_KERNELS] != 0;
    etp_reshard_report rep{};
    rep.n_phases = 1;
    const int64_t n_chunks = (n + kChunk - 1) / kChunk;
    const bool pinned_input = classify_pointer(host_descs) == MEM_HOST_PINNED;

    // stage A of chunk k (side stream): upload the raw records, count, scan, totals -> pinned host
    auto stage_a = [&](int64_t k) -> etp_status {
        Slot& s = S->slot[k % kSlots];
        const int64_t b = k * kChunk, m = std::min<int64_t>(kChunk, n - b);
        if (s.busy) {   // the copy kernel that last used this slot's descriptors must be done before they are overwritten
            ETP_CUDA_OK(cudaStreamWaitEvent(S->side, s.copied, 0));
            s.busy = false;
        }
        if (pinned_input) {   // the caller's array is page-locked: the DMA reads it directly (it must stay valid until the stream is synchronised)
            ETP_CUDA_OK(cudaMemcpyAsync(s.d_raw, host_descs + b, sizeof(etp_interval) * (size_t)m, cudaMemcpyHostToDevice, S->side));
        } else {
            if (s.staged) {   // the DMA that last read this slot's staging buffer
                ETP_CUDA_OK(cudaEventSynchronize(s.uploaded));
                s.staged = false;
            }
            std::memcpy(s.h_raw, host_descs + b, sizeof(etp_interval) * (size_t)m);
            ETP_CUDA_OK(cudaMemcpyAsync(s.d_raw, s.h_raw, sizeof(etp_interval) * (size_t)m, cudaMemcpyHostToDevice, S->side));
            ETP_CUDA_OK(cudaEventRecord(s.uploaded, S->side));
            s.staged = true;
        }
        ETP_CUDA_OK(cudaMemsetAsync(s.d_bad, 0xff, 2 * sizeof(unsigned int), S->side));
        const int nb = int((m + kBlock - 1) / kBlock);
        etp_iv_count_kernel<<<nb, kBlock, 0, S->side>>>(s.d_raw, (int)m, tma_min, s.d_block_sums, s.d_bad);
        etp_iv_scan_kernel<<<1, 32, 0, S->side>>>(s.d_block_sums, nb, s.d_totals, s.d_bad, s.d_counts + 3);
        ETP_CUDA_OK(cudaGetLastError());
        ETP_CUDA_OK(cudaMemcpyAsync(s.h_totals, s.d_totals, sizeof(Totals), cudaMemcpyDeviceToHost, S->side));
        ETP_CUDA_OK(cudaEventRecord(s.totals_ready, S->side));
        return ETP_OK;
    };

    reset_device_timing(c);
    for (int64_t k = 0; k < std::min<int64_t>(n_chunks, kSlots - 1); ++k) ETP_TRY(stage_a(k));
    for (int64_t k = 0; k < n_chunks; ++k) {
        Slot& s = S->slot[k % kSlots];
        const int64_t b = k * kChunk, m = std::min<int64_t>(kChunk, n - b);
        const int nb = int((m + kBlock - 1) / kBlock);
        // the only host wait of the call: 48 bytes of totals, produced on the side stream while the previous chunk is being copied
        ETP_CUDA_OK(cudaEventSynchronize(s.totals_ready));
        const Totals T = *s.h_totals;
        if (T.bad_size) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: interval %lld has negative size", (long long)(b + T.bad_size - 1));
        if (T.bad_align) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_copy_intervals: interval %lld is not 16-byte aligned (or has a NULL pointer)", (long long)(b + T.bad_align - 1));
        if (T.v[C_BULK_ITEMS] >= 0xFFFFFFF0ull || T.v[C_VEC_ITEMS] + T.v[C_SMALL_SEGS] >= 0xFFFFFFF0ull) ETP_FAIL(ETP_ERR_CAPACITY, "too many work items in one chunk");
        if ((int64_t)T.v[C_BULK_ITEMS] > s.bulk_items_cap) {
            if (s.d_bulk_items) ETP_CUDA_OK(cudaFree(s.d_bulk_items));   // synchronises; rare (capacity only grows)
            s.bulk_items_cap = (int64_t)T.v[C_BULK_ITEMS] * 5 / 4 + 1024;
            ETP_CUDA_OK(cudaMalloc(&s.d_bulk_items, sizeof(uint32_t) * (size_t)s.bulk_items_cap));
        }
        if ((int64_t)T.v[C_VEC_ITEMS] > s.vec_items_cap) {
            if (s.d_vec_items) ETP_CUDA_OK(cudaFree(s.d_vec_items));
            s.vec_items_cap = (int64_t)T.v[C_VEC_ITEMS] * 5 / 4 + 1024;
            ETP_CUDA_OK(cudaMalloc(&s.d_vec_items, sizeof(uint32_t) * (size_t)s.vec_items_cap));
        }
        // stage B (side stream): scatter + batches
        ScatterOut o{s.d_bulk, s.d_bulk_items, s.d_vec, s.d_vec_items, s.d_small};
        etp_iv_scatter_kernel<<<nb, kBlock, 0, S->side>>>(s.d_raw, (int)m, tma_min, s.d_block_sums, o);
        const unsigned long long n_small = T.v[C_SMALL_SEGS];
        etp_iv_batches_kernel<<<(unsigned)std::max<unsigned long long>(1, (n_small + 255) / 256), 256, 0, S->side>>>(s.d_small, s.d_totals, s.d_small_first, s.d_counts);
        ETP_CUDA_OK(cudaGetLastError());
        ETP_CUDA_OK(cudaEventRecord(s.lowered, S->side));
        // stage C (caller's stream): the copy kernel on the device-built descriptors
        const unsigned long long moved_items = T.v[C_BULK_ITEMS] + T.v[C_VEC_ITEMS] + n_small;
        if (moved_items > 0) {
            ETP_CUDA_OK(cudaStreamWaitEvent(user, s.lowered, 0));
            CopyArgs a{};
            a.bulk = s.d_bulk;
            a.vec = s.d_vec;
            a.bulk_items = s.d_bulk_items;
            a.vec_items = s.d_vec_items;
            a.pairs = nullptr;
            a.small = s.d_small;
            a.small_first = s.d_small_first;
            a.dev_counts = s.d_counts;
            a.counters = s.d_counts + 3;
            a.flags = c->opts[ETP_OPT_LDG_STEALS_BULK] ? 1u : 0u;
            if (timed) {
                while ((int)S->timing.size() < 2 * (S->n_timed + 1)) {
                    cudaEvent_t e;
                    ETP_CUDA_OK(cudaEventCreate(&e));
                    S->timing.push_back(e);
                }
                ETP_CUDA_OK(cudaEventRecord(S->timing[2 * S->n_timed], user));
            }
            if (!c->opts[ETP_OPT_SKIP_D2D]) {
                launch_copy_kernel(a, grid, user, c->opts[ETP_OPT_SMALL_STAGED] && T.v[C_BULK_ITEMS] == 0 && n_small > 0);
                ETP_CUDA_OK(cudaGetLastError());
                ++rep.n_kernel_launches;
            }
            if (timed) {
                ETP_CUDA_OK(cudaEventRecord(S->timing[2 * S->n_timed + 1], user));
                ++S->n_timed;
            }
        }
        ETP_CUDA_OK(cudaEventRecord(s.copied, user));
        s.busy = true;
        // upload + count of chunk k + 2 (the slot chunk k - 1 used) while chunks k and k + 1 are copied / lowered; issued AFTER this
        // chunk's copy launch because the upload from pageable memory blocks the host
        if (k + kSlots - 1 < n_chunks) ETP_TRY(stage_a(k + kSlots - 1));
        rep.n_jobs += (int64_t)(T.v[C_BULK_SEGS] + T.v[C_VEC_SEGS] + T.v[C_SMALL_SEGS]);
        rep.n_units += (int64_t)moved_items;
        rep.d2d_bytes += (int64_t)T.v[C_ALL_BYTES];
    }
    if (report) {
        rep.lower_ms = now_ms() - t0;
        *report = rep;
    }
    c->launches = rep.n_kernel_launches;
    return ETP_OK;
}

}  // namespace etp

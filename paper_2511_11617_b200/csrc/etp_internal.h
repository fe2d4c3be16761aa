// Internal declarations of libetp.so (not part of the C ABI; see include/etp.h for the boundary).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "etp.h"

namespace etp {

// ---- error channel (thread-local message, PAPER-independent plumbing)
void set_error(const char* fmt, ...) __attribute__((format(printf, 1, 2)));
#define ETP_FAIL(code, ...)          \
    do {                             \
        ::etp::set_error(__VA_ARGS__); \
        return (code);               \
    } while (0)
#define ETP_CUDA_OK(call)                                                                     \
    do {                                                                                      \
        cudaError_t e__ = (call);                                                             \
        if (e__ != cudaSuccess) {                                                             \
            ::etp::set_error("%s:%d %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e__)); \
            return ETP_ERR_CUDA;                                                              \
        }                                                                                     \
    } while (0)
#define ETP_TRY(call)                        \
    do {                                     \
        etp_status s__ = (call);             \
        if (s__ != ETP_OK) return s__;       \
    } while (0)

// ---- device work descriptors of the interval-copy kernel (kernel (a))
// The host uploads O(#intervals) SEGMENT descriptors; the kernel expands them into fixed-size WORK ITEMS.  The k-th item
// of a queue is looked up through an item table (uint32 segment index per item, filled on the host with one fill_n per
// segment), so a claim costs one atomicAdd + two dependent loads and the host never touches per-block / per-chunk state.
//
// A BULK segment is one contiguous interval; its items are pieces of kBulkItem bytes moved global -> shared -> global
// with cp.async.bulk by the CTA's TMA thread.  32 B = one sector.
struct BulkSeg {
    uint64_t src, dst;
    uint64_t bytes;        // multiple of 16
    uint32_t first_item;   // index of this segment's first item in the bulk queue
    uint32_t pad;
};
// A VEC segment is moved by the vector-copy warps with 16-byte loads/stores, one item per warp at a time.
//   kind VEC_LINEAR: a contiguous interval below the TMA threshold; item k = bytes [k*kVecItem, (k+1)*kVecItem).
//   kind VEC_PAGED : head-strided KV fragments of every live block.  Item k = (pair p = k / items_per_pair, plane group
//                    g = k % items_per_pair): planes [g*planes_per_item, ...) of (layer, K|V); within a plane
//                    rows_per_plane rows of row_bytes contiguous bytes.  Block ids come from pairs[pairs_first + p]
//                    = {old id, new id}:  src = src + plane*s_plane + old*s_block + row*s_row (dst likewise).
struct VecSeg {
    uint64_t src, dst;
    uint32_t kind, first_item;
    uint32_t row_bytes;        // multiple of 16
    uint32_t rows_per_plane;   // >= 1
    uint32_t planes_per_item, n_planes;
    uint32_t items_per_pair, pairs_first;
    int64_t s_row, d_row;      // byte strides between rows of a plane
    int64_t s_plane, d_plane;  // byte strides between planes   (VEC_LINEAR: s_plane = total bytes of the interval)
    int64_t s_block, d_block;  // byte strides between blocks
};
enum { VEC_LINEAR = 0, VEC_PAGED = 1 };
// A SMALL segment is a contiguous interval of at most kVecItem bytes (below the TMA threshold).  Consecutive small segments
// are grouped on the host into BATCHES (<= kSmallBatchSegs segments, ~kVecItem bytes); one batch is one work item of the
// vector queue (indices n_vec_items .. n_vec_items + n_small_batches - 1), so that a queue claim moves tens of KiB even when
// every interval is 256 bytes.  32 B = one sector; batch k covers segments [small_first[k], small_first[k+1]).
struct SmallSeg {
    uint64_t src, dst;
    uint32_t bytes;        // multiple of 16, <= kVecItem
    uint32_t pad0;
    uint64_t pad1;
};
static_assert(sizeof(SmallSeg) == 32, "SmallSeg layout");
constexpr int kSmallBatchSegs = 128;
static_assert(sizeof(BulkSeg) == 32, "BulkSeg layout");
static_assert(sizeof(VecSeg) == 96, "VecSeg layout");

constexpr int64_t kBulkItem = 256 << 10;   // bytes per bulk work item (work-queue granularity)
constexpr int64_t kVecItem = 32 << 10;     // bytes per vector work item (target for paged items)

// One launch of the copy kernel = the segments of one hazard phase.
struct JobList {
    std::vector<BulkSeg> bulk;
    std::vector<VecSeg> vec;
    std::vector<SmallSeg> small;
    std::vector<uint32_t> small_first;   // first segment of every batch
    int64_t open_batch_bytes = 0;        // bytes in the last (still open) batch
    uint32_t n_bulk_items = 0, n_vec_items = 0;
    int64_t bytes = 0;
    bool empty() const { return bulk.empty() && vec.empty() && small.empty(); }
};

// A pinned-host -> device DMA of the reload pipeline (pipeline (b)).
struct DmaCopy {
    const void* src;
    void* dst;
    int64_t bytes;
    int32_t phase;
};

enum MemKind { MEM_HOST_PAGEABLE = 0, MEM_HOST_PINNED = 1, MEM_DEVICE = 2 };
MemKind classify_pointer(const void* p);

}  // namespace etp

// ---- opaque ABI objects
struct etp_plan {
    int mode = ETP_PLAN_CMM;
    int64_t total_units = 0;
    std::vector<etp_shard> old_layout;
    std::vector<etp_shard> new_layout;
    std::vector<etp_task> tasks;
    etp_plan_stats stats{};
};

struct etp_ctx {
    int device = 0;                     // physical CUDA device of logical device 0 (the caller's streams live there)
    int n_sms = 0;
    int64_t opts[ETP_OPT__COUNT];
    void* impl = nullptr;               // executor state (per logical device: streams, descriptor arenas, events), etp_exec.cu
    int32_t launches = 0;               // kernels launched by the last call
    void* iv_state = nullptr;           // device-side lowering of etp_copy_intervals (etp_lower_dev.cu)
    void* lin_state = nullptr;          // kernel (c): per-stream split-K workspaces + the cache of prepared groups (etp_linear_group.cu)
    // Streams on which a call of this library that WRITES slabs (reshard, EPLB replicas, interval copies) was enqueued since the last
    // <= 64-token shard-linear launch on that stream.  Such a launch prefetches weight tiles before griddepcontrol.wait when it carries
    // the programmatic-serialization attribute, and CUDA makes the previous kernel's writes visible only after that wait: the first
    // linear launch behind a slab write therefore goes out WITHOUT the attribute (plain stream order), see etp::take_slab_write.
    std::vector<void*> slab_write_streams;
};

namespace etp {
// lowering (host): etp_lower.cpp
// The work of one call, partitioned by DESTINATION device ("each GPU pulls its own incoming intervals").
struct DeviceWork {
    std::vector<JobList> phases;       // device-copy segments per hazard phase (copy stream)
    std::vector<JobList> host_gather;  // segments whose source is pinned host memory (zero-copy gather, reload stream), per phase
    std::vector<DmaCopy> dma;          // pinned host -> device DMAs (reload stream)
    etp_reshard_report rep{};          // bytes this device writes
};
struct LoweredWork {
    std::vector<DeviceWork> dev;       // indexed by logical device of the ctx
    std::vector<int32_t> pairs;        // {old block id, new block id} lists referenced by VEC_PAGED segments (uploaded to every device)
    etp_reshard_report rep{};          // totals
};
int n_logical_devices(const etp_ctx* ctx);
int device_of_rank(const etp_ctx* ctx, int32_t rank);   // logical device that WRITES the rank's memory; -1 = another process does
etp_status lower_params(const etp_ctx* ctx, const etp_tensor* tensors, int32_t n_tensors, const etp_plan* const* plans,
                        int32_t n_plans, LoweredWork* out);
etp_status lower_kv(const etp_ctx* ctx, const etp_kv_geometry* g, const etp_plan* head_plan, const int32_t* pairs,
                    int64_t n_pairs, LoweredWork* out);
void push_contiguous(const etp_ctx* ctx, JobList* jl, const void* src, void* dst, int64_t bytes);

// etp_copy_intervals above kDeviceLoweringMin intervals: descriptors are built by kernels from the raw records (etp_lower_dev.cu)
constexpr int64_t kDeviceLoweringMin = 32768;
// etp_validate.cpp: argument checks of every interval; with check_overlap also "destinations mutually disjoint and disjoint from every source"
etp_status validate_intervals(const etp_interval* descs, int64_t n, bool check_overlap);
etp_status copy_intervals_device(etp_ctx* ctx, const etp_interval* host_descs, int64_t n, void* stream, etp_reshard_report* report);
void free_interval_state(etp_ctx* ctx);
int interval_timed_launches(etp_ctx* ctx, double* ms);
void reset_interval_timing(etp_ctx* ctx);
void reset_device_timing(etp_ctx* ctx);   // forgets the timing events of the last executor call (etp_exec.cu)

inline void note_slab_write(etp_ctx* c, void* stream) {
    for (void* s : c->slab_write_streams)
        if (s == stream) return;
    c->slab_write_streams.push_back(stream);
}
// true (and forgets it) if a slab write is pending on `stream`, or on the legacy default stream (NULL), which orders against every
// blocking stream
inline bool take_slab_write(etp_ctx* c, void* stream) {
    bool hit = false;
    for (size_t i = 0; i < c->slab_write_streams.size();) {
        if (c->slab_write_streams[i] == stream || c->slab_write_streams[i] == nullptr) {
            hit = true;
            c->slab_write_streams.erase(c->slab_write_streams.begin() + (long)i);
        } else {
            ++i;
        }
    }
    return hit;
}

// Bounded waits (etp_wait.cuh): the fault record is 8 x u64 of host-mapped pinned memory, allocated once per process by the first
// etp_ctx_create and installed into every kernel translation unit on every device of a ctx.  set_error appends it to the message.
extern volatile unsigned long long* g_wait_fault_host;   // etp_plan.cpp; NULL until a ctx exists
cudaError_t install_wait_fault_copy(unsigned long long* rec);
cudaError_t install_wait_fault_linear(unsigned long long* rec);
cudaError_t install_wait_fault_group(unsigned long long* rec);
cudaError_t install_wait_fault_moe(unsigned long long* rec);
void launch_starved_wait_kernel(cudaStream_t stream);

// kernel (c): frees the ctx-owned cache of prepared groups and the split-K workspaces (etp_linear_group.cu)
void lin_teardown(etp_ctx* ctx);

// execution (device): etp_exec.cu
etp_status execute(etp_ctx* ctx, LoweredWork* w, void* copy_stream, void* reload_stream, etp_reshard_report* report);
}  // namespace etp

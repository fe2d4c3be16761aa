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
// A BULK job is one contiguous interval of at most kBulkJobMax bytes; it is moved global -> shared -> global with
// cp.async.bulk by the CTA's TMA thread.  32 B = one sector.
struct BulkJob {
    uint64_t src, dst;
    uint64_t bytes;   // multiple of 16
    uint64_t pad;
};
// A FRAG job is a two-level strided set of rows, each `row_bytes` contiguous (a KV (token, head-run) fragment, or a
// small contiguous interval when n_rows == 1).  Row i sits at  base + (i / rows_per_group) * grp_stride
// + (i % rows_per_group) * row_stride.  Moved by one warp with 16-byte vector loads/stores.  64 B.
struct FragJob {
    uint64_t src, dst;
    uint32_t row_bytes;        // multiple of 16
    uint32_t n_rows;
    uint32_t rows_per_group;   // >= 1
    uint32_t vec_shift;        // log2(row_bytes / 16) if row_bytes/16 is a power of two, else 0xFFFFFFFF
    int64_t s_row, d_row;      // byte strides between rows of a group
    int64_t s_grp, d_grp;      // byte strides between groups
};
static_assert(sizeof(BulkJob) == 32, "BulkJob layout");
static_assert(sizeof(FragJob) == 64, "FragJob layout");

constexpr int64_t kBulkJobMax = 256 << 10;   // bytes per bulk job (work-queue granularity)
constexpr int64_t kFragJobTarget = 32 << 10; // target bytes per frag job

// One launch of the copy kernel = the jobs of one hazard phase.
struct JobList {
    std::vector<BulkJob> bulk;
    std::vector<FragJob> frag;
    int64_t bytes = 0;
    bool empty() const { return bulk.empty() && frag.empty(); }
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
    int device = 0;
    int n_sms = 0;
    int64_t opts[ETP_OPT__COUNT];
    void* impl = nullptr;               // executor state (descriptor arenas, events), etp_exec.cu
    unsigned int* d_counters = nullptr; // work-queue heads (device), one pair per kernel launch of a call
    int n_counter_slots = 0;
    void* d_staging = nullptr;          // staging ring of the KV reload pipeline (allocated on first use)
    int64_t staging_bytes = 0;
    std::vector<cudaEvent_t> events;    // hazard-phase events
    int32_t launches = 0;               // kernels launched by the last call
    std::vector<cudaEvent_t> tev;       // timing events (pairs) around copy-stream launches, ETP_OPT_TIME_KERNELS
    int32_t n_timed = 0;                // pairs recorded by the last call
};

namespace etp {
// lowering (host): etp_lower.cpp
struct LoweredWork {
    std::vector<JobList> phases;       // device-copy jobs per hazard phase (copy stream)
    std::vector<JobList> host_gather;  // frag jobs whose source is pinned host memory (zero-copy gather, reload stream), per phase
    std::vector<DmaCopy> dma;          // pinned host -> device DMAs (reload stream)
    etp_reshard_report rep{};
};
etp_status lower_params(const etp_ctx* ctx, const etp_tensor* tensors, int32_t n_tensors, const etp_plan* const* plans,
                        int32_t n_plans, LoweredWork* out);
etp_status lower_kv(const etp_ctx* ctx, const etp_kv_geometry* g, const etp_plan* head_plan, const int32_t* pairs,
                    int64_t n_pairs, LoweredWork* out);
void push_contiguous(const etp_ctx* ctx, JobList* jl, const void* src, void* dst, int64_t bytes);

// execution (device): etp_exec.cu
etp_status execute(etp_ctx* ctx, LoweredWork* w, void* copy_stream, void* reload_stream, etp_reshard_report* report);
}  // namespace etp

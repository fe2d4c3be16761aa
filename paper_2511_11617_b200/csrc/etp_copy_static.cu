// etp_copy_intervals_static: kernel (a) for callers that must not allocate (include/etp.h has the contract).
//
// Who this is for.  A reshard runs at the worst moment for an allocator: a GPU has just died, the survivors' HBM is packed with
// weights and KV blocks up to the serving engine's memory budget, and the engine, not this library, owns what is left (its pool
// took the device's free memory at start-up, so a cudaMalloc from a library either fails or eats into what the engine promised its
// KV cache).  cudaMalloc / cudaFree also synchronise the whole device, which a recovery path that is overlapping reloads with
// decode steps on other streams cannot afford, and some hosts (a plugin running inside somebody else's CUDA context, a fault
// handler) are simply forbidden to create device memory.  Every other entry point of the library needs an etp_ctx, and creating
// one allocates descriptor arenas (pinned + device), events and streams.  This one needs no ctx and allocates nothing.
//
// How.  The persistent copy kernel needs global scratch next to its inputs and outputs: the segment descriptors, the item table
// that maps a work item to its segment, and the two work-queue heads its CTAs bump with atomicAdd.  Here that scratch is a fixed
// array in the library's own device image (g_scratch below, kScratchBytes = 410,112 bytes, about 0.4 MiB; every GPU that loads libetp.so carries it
// until the process exits).  The kernel is the same etp_interval_copy_kernel the ctx path launches; only where its descriptors
// live differs.
//
// The array's name is usable in device code only.  In host code `g_scratch` is the host-side shadow the runtime uses as a lookup
// key, NOT a device address; a kernel handed that value faults (or, where the GPU can reach host memory, scribbles on the wrong
// memory without an error).  The device address comes from cudaGetSymbolAddress, taken once per device with that device current.
#include <mutex>

#include <cstddef>
#include <cstring>

#include "etp_copy.cuh"

namespace etp {
namespace {

constexpr int64_t kStaticMaxIntervals = 4096;       // intervals per call
constexpr int64_t kStaticMaxBulkItems = 32768;      // 256-KiB pieces of the >= 32-KiB intervals of one call (8 GiB of them)
constexpr int64_t kStaticTmaMin = 32768;            // the ctx path's default ETP_OPT_TMA_MIN_BYTES; there is no option here
constexpr int kMaxDevices = 64;

// Layout of the scratch (device) and of its host image.  Only the used prefix of each array is uploaded.
struct Scratch {
    unsigned int heads[64];                          // [0] bulk-queue head, [1] vector-queue head; must be 0 at launch
    uint32_t small_first[kStaticMaxIntervals + 64];  // first segment of every batch of small intervals, + one end marker
    BulkSeg bulk[kStaticMaxIntervals];               // intervals >= 32 KiB
    SmallSeg small[kStaticMaxIntervals];             // intervals <= 32 KiB
    uint32_t bulk_items[kStaticMaxBulkItems];        // segment index of every bulk work item
};
constexpr size_t kScratchBytes = sizeof(Scratch);
static_assert(kScratchBytes == 410112, "the size stated in etp.h / README.md");
static_assert(offsetof(Scratch, bulk) % 32 == 0 && offsetof(Scratch, small) % 32 == 0, "descriptors are read as two uint4");

static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

std::mutex g_mu;                        // one host thread at a time builds and uploads (the array is shared anyway)
Scratch g_host;                         // host image the descriptors are built in (pageable; plain static storage, no allocation)
unsigned char* g_dev[kMaxDevices];      // device address of g_scratch on each device, filled by setup_device
int g_sms[kMaxDevices];

// Once per device, with that device current: resolve the array's device address, check the architecture, raise the kernel's
// dynamic shared-memory limit.  None of this allocates.
etp_status setup_device(int dev) {
    if (g_dev[dev]) return ETP_OK;
    int major = 0, sms = 0;
    ETP_CUDA_OK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) ETP_FAIL(ETP_ERR_CUDA, "etp_copy_intervals_static: device %d is sm_%dx; this library is built for sm_100a only", dev, major);
    ETP_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    void* p = nullptr;
    ETP_CUDA_OK(cudaGetSymbolAddress(&p, g_scratch));
    if (!p || ((uintptr_t)p & 255)) ETP_FAIL(ETP_ERR_CUDA, "etp_copy_intervals_static: cudaGetSymbolAddress returned %p", p);
    ETP_CUDA_OK(configure_copy_kernel());
    g_sms[dev] = sms;
    g_dev[dev] = (unsigned char*)p;
    return ETP_OK;
}

}  // namespace
}  // namespace etp

extern "C" etp_status etp_copy_intervals_static(const etp_interval* host_descs, int64_t n, void* stream) {
    using namespace etp;
    if (n < 0 || (n > 0 && !host_descs)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals_static: bad arguments");
    if (n > kStaticMaxIntervals)
        ETP_FAIL(ETP_ERR_CAPACITY, "etp_copy_intervals_static: %lld intervals, the static scratch holds at most %lld per call (split the call, "
                 "or use etp_copy_intervals with a ctx)", (long long)n, (long long)kStaticMaxIntervals);
    // same argument and disjointness contract as etp_copy_intervals (host-only check; n <= 4096, microseconds)
    ETP_TRY(validate_intervals(host_descs, n, true));
    int64_t bulk_items = 0;
    for (int64_t i = 0; i < n; ++i)
        if (host_descs[i].bytes >= kStaticTmaMin) bulk_items += (host_descs[i].bytes + kBulkItem - 1) / kBulkItem;
    if (bulk_items > kStaticMaxBulkItems)
        ETP_FAIL(ETP_ERR_CAPACITY, "etp_copy_intervals_static: the intervals of 32 KiB and more need %lld pieces of 256 KiB, the static scratch "
                 "holds %lld (8 GiB) per call", (long long)bulk_items, (long long)kStaticMaxBulkItems);

    int dev = -1;
    ETP_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) ETP_FAIL(ETP_ERR_CUDA, "etp_copy_intervals_static: current device %d", dev);
    std::lock_guard<std::mutex> lock(g_mu);
    ETP_TRY(setup_device(dev));

    // ---- lower into the host image: >= 32 KiB -> bulk segments (cp.async.bulk ring), the rest -> batches of small segments
    Scratch& h = g_host;
    uint32_t n_bulk = 0, n_bulk_items = 0, n_small = 0, n_batches = 0;
    int64_t open_bytes = 0;
    for (int64_t i = 0; i < n; ++i) {
        const etp_interval& d = host_descs[i];
        if (d.bytes == 0) continue;
        if (d.bytes >= kStaticTmaMin) {
            h.bulk[n_bulk] = {(uint64_t)(uintptr_t)d.src, (uint64_t)(uintptr_t)d.dst, (uint64_t)d.bytes, n_bulk_items, 0};
            const uint32_t k = (uint32_t)((d.bytes + kBulkItem - 1) / kBulkItem);
            for (uint32_t j = 0; j < k; ++j) h.bulk_items[n_bulk_items + j] = n_bulk;
            n_bulk_items += k;
            ++n_bulk;
        } else {
            const bool open = n_batches > 0 && n_small - h.small_first[n_batches - 1] < (uint32_t)kSmallBatchSegs && open_bytes + d.bytes <= kVecItem;
            if (!open) {
                h.small_first[n_batches++] = n_small;
                open_bytes = 0;
            }
            h.small[n_small++] = {(uint64_t)(uintptr_t)d.src, (uint64_t)(uintptr_t)d.dst, (uint32_t)d.bytes, 0, 0};
            open_bytes += d.bytes;
        }
    }
    if (n_bulk == 0 && n_small == 0) return ETP_OK;
    h.small_first[n_batches] = n_small;
    std::memset(h.heads, 0, sizeof(h.heads));

    // ---- upload.  The heads are rewritten to zero by every call: the array keeps whatever the last call (or last process-wide user)
    // left in it, and a non-zero head would make the kernel skip work items.  Stale descriptors beyond the counts are never read.
    // The sources are pageable host memory, so each cudaMemcpyAsync has consumed its source when it returns (the driver stages it),
    // and g_host can be rebuilt by the next call; the device-side copies are ordered on `stream` before the kernel.
    cudaStream_t s = (cudaStream_t)stream;
    unsigned char* d = g_dev[dev];
    ETP_CUDA_OK(cudaMemcpyAsync(d + offsetof(Scratch, heads), h.heads, offsetof(Scratch, small_first) + (size_t)(n_batches + 1) * sizeof(uint32_t),
                                cudaMemcpyHostToDevice, s));   // heads and small_first are adjacent
    if (n_bulk) {
        ETP_CUDA_OK(cudaMemcpyAsync(d + offsetof(Scratch, bulk), h.bulk, (size_t)n_bulk * sizeof(BulkSeg), cudaMemcpyHostToDevice, s));
        ETP_CUDA_OK(cudaMemcpyAsync(d + offsetof(Scratch, bulk_items), h.bulk_items, (size_t)n_bulk_items * sizeof(uint32_t), cudaMemcpyHostToDevice, s));
    }
    if (n_small) ETP_CUDA_OK(cudaMemcpyAsync(d + offsetof(Scratch, small), h.small, (size_t)n_small * sizeof(SmallSeg), cudaMemcpyHostToDevice, s));

    CopyArgs a{};
    a.bulk = (const BulkSeg*)(d + offsetof(Scratch, bulk));
    a.bulk_items = (const uint32_t*)(d + offsetof(Scratch, bulk_items));
    a.vec = nullptr;          // no mid-size class here: an interval is either >= 32 KiB (bulk) or <= 32 KiB (small)
    a.vec_items = nullptr;
    a.pairs = nullptr;
    a.small = (const SmallSeg*)(d + offsetof(Scratch, small));
    a.small_first = (const uint32_t*)(d + offsetof(Scratch, small_first));
    a.n_bulk_items = n_bulk_items;
    a.n_vec_items = 0;
    a.n_small_batches = n_batches;
    a.dev_counts = nullptr;
    a.counters = (unsigned int*)(d + offsetof(Scratch, heads));
    a.flags = 0;
    launch_copy_kernel(a, g_sms[dev], s, /*staged_small=*/n_bulk_items == 0 && n_batches > 0);
    ETP_CUDA_OK(cudaGetLastError());
    return ETP_OK;
}

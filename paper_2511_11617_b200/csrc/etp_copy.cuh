// Kernel (a): persistent, descriptor-driven interval copy for sm_100a.
// PAPER.md:96 / :146 (parameter re-assignment primitive, KV operators for variable-length shards), :166 (P2P transfers
// run beside the reloads).  One CTA per SM; two work queues with atomic heads; the queues hold WORK ITEMS that the kernel
// derives from O(#intervals) segment descriptors through an item table (etp_internal.h):
//   * BULK queue  - 256-KiB pieces of contiguous intervals.  Warp 0's elected thread drives a ring of shared-memory
//                   stages: cp.async.bulk global->shared (mbarrier complete_tx), then cp.async.bulk shared->global
//                   (bulk_group), kLookahead loads in flight, stores drained with wait_group.read.
//   * VEC queue   - ~32-KiB items: pieces of small intervals, or the head-strided KV fragments of one (live block, plane
//                   group).  Each of the other warps claims one item at a time and moves it with 16-byte ld.global.nc /
//                   st.global, 8 vectors in flight per lane, consecutive lanes on consecutive 16-byte words of a row.
//                   Intervals of <= 32 KiB are batched (<= 128 per item): the warp loads 32 descriptors at once, scans
//                   their lengths and walks the concatenated 16-byte words, finding each word's interval by a shuffle search.
#pragma once
#include "etp_internal.h"

namespace etp {

constexpr int kCopyThreads = 512;             // warp 0: TMA driver; warps 1..15: vector-copy warps
constexpr int kStageBytes = 32 << 10;         // bytes per ring stage
constexpr int kStages = 6;                    // ring depth (192 KiB of shared memory)
constexpr int kLookahead = 3;                 // bulk loads in flight ahead of the store front
constexpr int kCopySmemBytes = kStages * kStageBytes + 1024;

struct CopyArgs {
    const BulkSeg* bulk;
    const VecSeg* vec;
    const uint32_t* bulk_items;   // segment index of every bulk work item
    const uint32_t* vec_items;    // segment index of every vector work item
    const int2* pairs;            // {old block id, new block id} lists of the VEC_PAGED segments
    const SmallSeg* small;        // small contiguous intervals, batched: vector-queue items n_vec_items .. + n_small_batches
    const uint32_t* small_first;  // n_small_batches + 1 entries
    unsigned int n_bulk_items, n_vec_items, n_small_batches;
    const unsigned int* dev_counts;   // != NULL: {n_bulk_items, n_vec_items, n_small_batches} live on the device (descriptors
                                      // lowered by the device-side classifier, etp_lower_dev.cu) and override the three above
    unsigned int* counters;       // [0] bulk head, [1] vec head (zeroed before launch)
    unsigned int flags;           // bit 0: vector warps also drain the bulk queue when theirs is empty
};

// staged_small: the launch has small batches and NO bulk items and ETP_OPT_SMALL_STAGED is on -> the instantiation whose vector warps
// stage small batches through the (idle) ring
void launch_copy_kernel(const CopyArgs& a, int grid, cudaStream_t stream, bool staged_small = false);
cudaError_t configure_copy_kernel();

}  // namespace etp

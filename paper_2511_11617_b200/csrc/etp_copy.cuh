// Kernel (a): persistent, descriptor-driven interval copy for sm_100a.
// PAPER.md:96 / :146 (parameter re-assignment primitive, KV operators for variable-length shards), :166 (P2P transfers
// run beside the reloads).  One CTA per SM; two work queues with atomic heads:
//   * BULK queue  - contiguous intervals of up to 256 KiB.  Warp 0's elected thread drives a ring of shared-memory
//                   stages: cp.async.bulk global->shared (mbarrier complete_tx), then cp.async.bulk shared->global
//                   (bulk_group), kLookahead loads in flight, stores drained with wait_group.read.
//   * FRAG queue  - two-level strided rows (head-strided KV fragments) and small intervals.  Each of the other warps
//                   claims one job at a time and moves it with 16-byte ld.global.nc / st.global, 8 vectors in flight
//                   per lane, consecutive lanes on consecutive 16-byte words of a row (coalesced).
#pragma once
#include "etp_internal.h"

namespace etp {

constexpr int kCopyThreads = 512;             // warp 0: TMA driver; warps 1..15: vector-copy warps
constexpr int kStageBytes = 32 << 10;         // bytes per ring stage
constexpr int kStages = 6;                    // ring depth (192 KiB of shared memory)
constexpr int kLookahead = 3;                 // bulk loads in flight ahead of the store front
constexpr int kCopySmemBytes = kStages * kStageBytes + 1024;

struct CopyArgs {
    const BulkJob* bulk;
    const FragJob* frag;
    unsigned int n_bulk, n_frag;
    unsigned int* counters;   // [0] bulk head, [1] frag head (zeroed before launch)
    unsigned int flags;       // bit 0: vector warps also drain the bulk queue when the frag queue is empty
};

void launch_copy_kernel(const CopyArgs& a, int grid, cudaStream_t stream);
cudaError_t configure_copy_kernel();

}  // namespace etp

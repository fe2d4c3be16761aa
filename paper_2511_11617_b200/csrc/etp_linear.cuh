// Declarations shared by the two halves of kernel (c):
//   etp_linear.cu        the tensor-bound regime (> 64 tokens): 128 x 256 single-CTA tiles and CTA pairs (cta_group::2)
//   etp_linear_group.cu  the weight-streaming regime (<= 64 tokens): ONE persistent launch over a prepared, load-balanced item
//                        table that may span several linears of any mode (etp_linear_prepare / etp_linear_run)
#pragma once
#include <vector>

#include "etp_tc.cuh"

namespace etp {
namespace lin {

constexpr int kMaxLinRuns = 32;    // <= 2 contiguous runs per rank, 8 ranks, up to 3 fused linears (q|k|v) - capped at 32
constexpr int kMaxGroupLins = 8;   // linears of one prepared group

struct Run {          // one contiguous slot range of a rank's shard, runs sorted by (linear, global feature)
    int64_t feat0;    // first global feature of the run (out-feature: column-parallel, in-feature: row-parallel)
    int32_t n_feat;   // features in the run
    int32_t first;    // column-parallel: index of the run's first m tile; row-parallel: of its first K chunk entry
    void* y;          // column-parallel: output of the linear this run belongs to
    int32_t out_features, pad;   // ... and its row pitch
};
static_assert(sizeof(Run) == 32, "Run layout");

struct LinOut {   // one linear of a (possibly fused) legacy call
    const etp_tensor* w;
    int64_t out_features, features_per_unit;
    void* y;
};

// A shard layout checked and expanded into the contiguous slot runs of one weight tensor (L3), ascending unit order.
struct RunList {
    Run runs[kMaxLinRuns];
    const void* addr[kMaxLinRuns];
    int n = 0;
};
etp_status check_layout(const etp_shard* layout, int32_t n_shards, int64_t total_units, std::vector<etp_shard>* sorted);
etp_status append_runs(const etp_tensor* w, const std::vector<etp_shard>& sorted, int64_t features_per_unit, void* y,
                       int64_t out_features, RunList* out);
etp_status check_linear_shape(etp_linear_mode mode, int64_t in_features, int64_t out_features, int64_t features_per_unit,
                              const etp_tensor* w);

// > 64 tokens (etp_linear.cu): one launch per call; column-parallel linears that share X may be fused.
etp_status shard_linear_large(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x, int64_t tokens,
                              int64_t in_features, const LinOut* outs, int32_t n_outs, const etp_shard* layout,
                              int32_t n_shards, void* stream);

// <= 64 tokens (etp_linear_group.cu): the legacy entry points run through a ctx-owned cache of prepared groups.
etp_status shard_linear_small(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x, int64_t tokens,
                              int64_t in_features, const LinOut* outs, int32_t n_outs, const etp_shard* layout,
                              int32_t n_shards, void* stream);
void free_linear_cache(etp_ctx* ctx);

// per-stream split-K workspace of a ctx (fp32 partial tiles + arrival tickets); never shrinks, old blocks live until the ctx dies
struct LinWorkspace {
    cudaStream_t stream;
    float* partials;
    int64_t partial_bytes;
    unsigned int* tickets;
    int64_t n_tickets;
};
etp_status linear_workspace(etp_ctx* ctx, cudaStream_t stream, int64_t partial_bytes, int64_t n_tickets, LinWorkspace* out);
void free_linear_workspaces(etp_ctx* ctx);

}  // namespace lin
}  // namespace etp

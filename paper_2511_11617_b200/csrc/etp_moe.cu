// Grouped shard linear for MoE experts (reading G5): one launch computes, for every expert e
// with routed rows,  Y_perm[rows of e][out] = X_perm[rows of e][in] . W_e^T  on the expert matrices exactly where the
// expert-granularity reshard left them (the expert is the unit of the plan; slot-addressed slabs, L3).
//   ETP_COL_PARALLEL  W_e stored [out][in]  (gate, up):   A = K-major rows of W_e
//   ETP_ROW_PARALLEL  W_e stored [in][out]  (down_t):     A = MN-major, K loop over the expert's own in-features
// Same tcgen05 / TMEM / TMA pipeline as etp_shard_linear (etp_linear.cu): D[m = out feature][n = routed row] in TMEM,
// 128 x BN tiles, warp 0 TMA producer, warp 1 MMA issuer, warps 2-5 epilogue, two accumulator stages.  What differs is the
// work list: the host expands (expert, m tile, row tile) into 32-byte ITEM descriptors (the experts' row counts are ragged),
// uploaded with the call; a tile may over-read rows of the next expert (X) or of the next expert's matrix (W, column-parallel)
// - both only feed accumulator rows / columns that the epilogue masks.
#include <algorithm>
#include <cstring>
#include <vector>

#include "etp_tc.cuh"

using namespace etp;
using namespace etp::tc;

namespace {

struct MoeItem {       // 32 bytes
    int32_t run;       // tensor map of the contiguous slot run that holds the expert
    int32_t a_row;     // column-parallel: first weight row of the tile inside the run; row-parallel: the expert's first k row
    int32_t m0;        // first out feature of the tile (column offset in Y_perm)
    int32_t valid;     // out features of the tile that exist (<= 128)
    int32_t x_row;     // first routed row of the tile in X_perm / Y_perm
    int32_t n_rows;    // rows of the tile that belong to the expert (<= BN)
    int32_t pad[2];
};
static_assert(sizeof(MoeItem) == 32, "MoeItem layout");

struct alignas(64) MoeParams {
    CUtensorMap map_x;
    CUtensorMap map_w[kMaxRuns];
    const MoeItem* items;
    int32_t n_items, mode, dtype, n_chunks;   // n_chunks: K chunks of kBK per item
    int32_t out_features, n_runs;
    void* y;
};

template <int BN>
struct MoeCfg {
    static constexpr int kBBytes = BN * kBK * 2;
    static constexpr int kStageBytes = kABytes + kBBytes;
    static constexpr int kStages = (kSmemBudget / kStageBytes) > 12 ? 12 : (kSmemBudget / kStageBytes);
    static constexpr int kTmemCols = (2 * BN) < 32 ? 32 : 2 * BN;
    static constexpr int kSmemBytes = kStages * kStageBytes + 1024 + 256 + 4096;   // + per-warp epilogue transpose buffers
};

__device__ __forceinline__ MoeItem load_item(const MoeItem* items, int i) {
    const int4 a = __ldg(reinterpret_cast<const int4*>(items + i));
    const int4 b = __ldg(reinterpret_cast<const int4*>(items + i) + 1);
    MoeItem it;
    it.run = a.x; it.a_row = a.y; it.m0 = a.z; it.valid = a.w;
    it.x_row = b.x; it.n_rows = b.y;
    return it;
}

template <int BN, typename OutT>
__global__ void __launch_bounds__(kLinThreads, 1) etp_moe_linear_kernel(const __grid_constant__ MoeParams p) {
    using C = MoeCfg<BN>;
    constexpr int kXBox = BN < 64 ? BN : 64;   // rows per TMA box of the X tile
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + C::kStages * C::kStageBytes);
    uint64_t* empty_bar = full_bar + C::kStages;
    uint64_t* tmem_full = empty_bar + C::kStages;
    uint64_t* tmem_empty = tmem_full + 2;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(tmem_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool row_par = p.mode == ETP_ROW_PARALLEL;

    if (warp == 0 && lane == 1) {
        prefetch_tensormap(&p.map_x);
        for (int r = 0; r < p.n_runs; ++r) prefetch_tensormap(&p.map_w[r]);
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < C::kStages; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], 1);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&tmem_full[s], 1);
            mbar_init(&tmem_empty[s], 4);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_ptr)), "r"(uint32_t(C::kTmemCols))
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    if (warp == 0) {
        if (lane == 0) {   // ------------------------------------------------------------------ TMA producer
            int stage = 0;
            uint32_t phase = 0;
            for (int i = blockIdx.x; i < p.n_items; i += gridDim.x) {
                const MoeItem it = load_item(p.items, i);
                const int nb = (it.n_rows + kXBox - 1) / kXBox;
                for (int c = 0; c < p.n_chunks; ++c) {
                    uint8_t* sa = smem + stage * C::kStageBytes;
                    uint8_t* sb = sa + kABytes;
                    mbar_wait(&empty_bar[stage], phase ^ 1);
                    mbar_expect_tx(&full_bar[stage], uint32_t(kABytes + nb * kXBox * kBK * 2));
                    if (!row_par) {
                        tma_load_2d(sa, &p.map_w[it.run], &full_bar[stage], c * kBK, it.a_row);
                    } else {
                        tma_load_2d(sa, &p.map_w[it.run], &full_bar[stage], it.m0, it.a_row + c * kBK);
                        tma_load_2d(sa + kABytes / 2, &p.map_w[it.run], &full_bar[stage], it.m0 + 64, it.a_row + c * kBK);
                    }
                    for (int b = 0; b < nb; ++b)   // the X tile in 64-row boxes: a ragged last tile only fetches the boxes it has rows in
                        tma_load_2d(sb + b * kXBox * kBK * 2, &p.map_x, &full_bar[stage], c * kBK, it.x_row + b * kXBox);
                    if (++stage == C::kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        if (lane == 0) {   // ------------------------------------------------------------------ MMA issuer
            // UMMA_N per item: only the 64-row boxes of X that were fetched (a ragged last row tile of an expert runs a narrower MMA)
            const uint32_t a_lbo = row_par ? uint32_t(kABytes / 2) : 16u;
            const uint32_t a_kstep = row_par ? (uint32_t(kUmmaK) * 128u) >> 4 : (uint32_t(kUmmaK) * 2u) >> 4;
            int stage = 0;
            uint32_t phase = 0;
            int local = 0;
            for (int i = blockIdx.x; i < p.n_items; i += gridDim.x, ++local) {
                const int n_rows = __ldg(&p.items[i].n_rows);
                const uint32_t idesc = make_idesc(p.dtype == ETP_BF16 ? 1u : 0u, row_par ? 1u : 0u, uint32_t((n_rows + kXBox - 1) / kXBox * kXBox));
                const int as = local & 1;
                const uint32_t aph = (local >> 1) & 1;
                mbar_wait(&tmem_empty[as], aph ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + uint32_t(as * BN);
                for (int c = 0; c < p.n_chunks; ++c) {
                    uint8_t* sa = smem + stage * C::kStageBytes;
                    mbar_wait(&full_bar[stage], phase);
                    tc_fence_after();
                    const uint64_t a_desc = make_smem_desc(smem_u32(sa), a_lbo, 1024);
                    const uint64_t b_desc = make_smem_desc(smem_u32(sa + kABytes), 16, 1024);
#pragma unroll
                    for (int k = 0; k < kBK / kUmmaK; ++k)
                        tc_mma(d_tmem, a_desc + uint64_t(k) * a_kstep, b_desc + uint64_t(k) * 2u, idesc, (c > 0 || k > 0) ? 1u : 0u);
                    tc_commit(&empty_bar[stage]);
                    if (++stage == C::kStages) { stage = 0; phase ^= 1; }
                }
                tc_commit(&tmem_full[as]);
            }
        }
        __syncwarp();
    } else {               // ---------------------------------------------------------------------- epilogue warps 2..5
        const int q = warp & 3;
        OutT* y = reinterpret_cast<OutT*>(p.y);
        OutT* stage_t = reinterpret_cast<OutT*>(smem + C::kStages * C::kStageBytes + 256) + q * 512;   // [16 rows][32 features]
        int local = 0;
        for (int i = blockIdx.x; i < p.n_items; i += gridDim.x, ++local) {
            const MoeItem it = load_item(p.items, i);
            const int as = local & 1;
            const uint32_t aph = (local >> 1) & 1;
            mbar_wait(&tmem_full[as], aph);
            tc_fence_after();
            const uint32_t taddr = tmem_base + uint32_t(as * BN) + (uint32_t(q * 32) << 16);
            // up to 64 accumulator columns per tcgen05.wait::ld (four loads in flight hide the TMEM read latency); every 16
            // columns go through a 1-KiB per-warp transpose buffer so that the global stores are 16 bytes per lane (8 routed
            // rows x 64 contiguous bytes per instruction) instead of 2 - m0 and out_features are multiples of 8 by contract.
            for (int c64 = 0; c64 < it.n_rows; c64 += 64) {
                uint32_t v[4][16];
#pragma unroll
                for (int g = 0; g < 4; ++g)
                    if (BN >= 16 * (g + 1) && c64 + 16 * g < it.n_rows) tc_ld16(taddr + uint32_t(c64 + 16 * g), v[g]);
                tc_ld_wait();
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    if (BN >= 16 * (g + 1) && c64 + 16 * g < it.n_rows) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) stage_t[j * 32 + lane] = cvt16<OutT>(__uint_as_float(v[g][j]));
                        __syncwarp();
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int row = h * 8 + (lane >> 2), chunk = lane & 3;
                            const int tok = c64 + 16 * g + row;
                            const uint4 val = *reinterpret_cast<const uint4*>(stage_t + row * 32 + chunk * 8);
                            if (tok < it.n_rows && q * 32 + chunk * 8 < it.valid)
                                *reinterpret_cast<uint4*>(y + size_t(it.x_row + tok) * p.out_features + it.m0 + q * 32 + chunk * 8) = val;
                        }
                        __syncwarp();
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&tmem_empty[as]);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        __syncwarp();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(uint32_t(C::kTmemCols)) : "memory");
    }
}

template <int BN>
etp_status launch_moe(const MoeParams& p, int grid, cudaStream_t stream) {
    using C = MoeCfg<BN>;
    if (p.dtype == ETP_BF16) {
        auto k = etp_moe_linear_kernel<BN, __nv_bfloat16>;
        ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes));
        k<<<grid, kLinThreads, C::kSmemBytes, stream>>>(p);
    } else {
        auto k = etp_moe_linear_kernel<BN, __half>;
        ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes));
        k<<<grid, kLinThreads, C::kSmemBytes, stream>>>(p);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) ETP_FAIL(ETP_ERR_CUDA, "etp_moe_linear: launch failed: %s", cudaGetErrorString(e));
    return ETP_OK;
}

}  // namespace

extern "C" etp_status etp_moe_linear(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x_perm,
                                     const int64_t* row_offsets, int32_t n_experts, int64_t in_features, int64_t out_features,
                                     const etp_tensor* w, const etp_shard* layout, int32_t n_shards, void* y_perm, void* stream) {
    if (!ctx || !w || !layout || !w->slabs || !row_offsets) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: NULL argument");
    if (mode != ETP_COL_PARALLEL && mode != ETP_ROW_PARALLEL) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: bad mode %d", int(mode));
    if (dtype != ETP_BF16 && dtype != ETP_FP16) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_moe_linear: dtype %d is not bf16/fp16", int(dtype));
    if (n_experts <= 0 || in_features <= 0 || out_features <= 0 || n_shards <= 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: non-positive size");
    if (w->total_units != n_experts) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: the tensor has %lld units, n_experts = %d (one unit = one expert)", (long long)w->total_units, n_experts);
    if (w->unit_bytes != in_features * out_features * 2)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: unit_bytes %lld != in x out x 2 = %lld", (long long)w->unit_bytes, (long long)(in_features * out_features * 2));
    const bool row_par = mode == ETP_ROW_PARALLEL;
    const int64_t rows_per_expert = row_par ? in_features : out_features;   // rows of the stored expert matrix
    const int64_t row_len = row_par ? out_features : in_features;
    if ((in_features * 2) % 16 || (out_features * 2) % 16) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_moe_linear: feature counts must be multiples of 8");
    if (row_par && in_features % kBK)
        ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_moe_linear: row-parallel experts need in_features %% %d == 0 (a K chunk must not run into the next expert)", kBK);
    if (row_offsets[0] != 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: row_offsets[0] != 0");
    int64_t max_rows = 0;
    for (int32_t e = 0; e < n_experts; ++e) {
        if (row_offsets[e + 1] < row_offsets[e]) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: row_offsets decrease at expert %d", e);
        max_rows = std::max(max_rows, row_offsets[e + 1] - row_offsets[e]);
    }
    const int64_t n_rows = row_offsets[n_experts];
    if (n_rows >= (int64_t(1) << 31) || in_features >= (int64_t(1) << 31) || out_features >= (int64_t(1) << 31))
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: sizes must be below 2^31");
    if (n_rows == 0) return ETP_OK;
    if (!x_perm || !y_perm) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: x / y is NULL");
    if ((reinterpret_cast<uintptr_t>(x_perm) | reinterpret_cast<uintptr_t>(y_perm)) & 15) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_moe_linear: x / y not 16-byte aligned");

    // ---- shards must tile [0, n_experts); every shard is <= 2 contiguous slot runs of its slab (L3)
    std::vector<etp_shard> sh;
    for (int i = 0; i < n_shards; ++i)
        if (layout[i].alive && layout[i].end > layout[i].begin) sh.push_back(layout[i]);
    std::sort(sh.begin(), sh.end(), [](const etp_shard& a, const etp_shard& b) { return a.begin < b.begin; });
    int64_t cursor = 0;
    for (const etp_shard& s : sh) {
        if (s.begin != cursor) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: layout does not tile [0,%d): gap or overlap at expert %lld", n_experts, (long long)cursor);
        cursor = s.end;
    }
    if (cursor != n_experts) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: layout covers %lld of %d experts", (long long)cursor, n_experts);

    MoeParams p;
    std::memset(&p, 0, sizeof(p));
    struct RunInfo { int64_t first_expert, n, slot0; const char* base; };
    std::vector<RunInfo> runs;
    for (const etp_shard& s : sh) {
        if (s.rank < 0 || s.rank >= w->n_ranks) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: rank %d outside the tensor's %d slabs", s.rank, w->n_ranks);
        const etp_slab& sl = w->slabs[s.rank];
        if (!sl.base) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: rank %d has no slab", s.rank);
        if (reinterpret_cast<uintptr_t>(sl.base) & 15) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_moe_linear: slab of rank %d not 16-byte aligned", s.rank);
        const int64_t width = s.end - s.begin;
        if (sl.cap_units <= 0 || width > sl.cap_units) ETP_FAIL(ETP_ERR_CAPACITY, "etp_moe_linear: shard of rank %d (%lld experts) exceeds its slab (%lld)", s.rank, (long long)width, (long long)sl.cap_units);
        int64_t slot0 = (s.begin - sl.anchor_unit) % sl.cap_units;
        if (slot0 < 0) slot0 += sl.cap_units;
        const int64_t len1 = std::min(width, sl.cap_units - slot0);
        runs.push_back({s.begin, len1, slot0, static_cast<const char*>(sl.base)});
        if (width > len1) runs.push_back({s.begin + len1, width - len1, 0, static_cast<const char*>(sl.base)});
    }
    if ((int)runs.size() > kMaxRuns) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_moe_linear: more than %d contiguous runs", kMaxRuns);
    for (const RunInfo& r : runs)
        if (r.n * rows_per_expert >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: run too long");

    // ---- row tile BN: operand fetch into the SM bounds a tile (measured on kernel (c): 48 KiB per K chunk at BN = 256 is the
    // limit, the MMA is not), so an item costs (A tile + BN rows of X) bytes per K chunk; take the BN with the least total.
    int bn = 16;
    {
        int64_t best = INT64_MAX;
        for (int cand : {256, 128, 64, 16}) {
            int64_t cost = 0;
            const int box = std::min(cand, 64);
            for (int32_t e = 0; e < n_experts; ++e) {
                const int64_t c = row_offsets[e + 1] - row_offsets[e];
                const int64_t tiles = (c + cand - 1) / cand, boxes = (c + box - 1) / box;   // X is fetched in boxes of <= 64 rows
                cost += tiles * kABytes + boxes * box * kBK * 2;
            }
            if (cost < best) { best = cost; bn = cand; }
        }
    }

    // ---- items: (expert, m tile, row tile), m tiles of one expert adjacent so that its X tile stays in L2
    const int64_t m_extent = out_features;
    const int64_t m_tiles = (m_extent + kBM - 1) / kBM;
    std::vector<MoeItem> items;
    for (size_t ri = 0; ri < runs.size(); ++ri) {
        const RunInfo& r = runs[ri];
        for (int64_t k = 0; k < r.n; ++k) {
            const int64_t e = r.first_expert + k;
            const int64_t cnt = row_offsets[e + 1] - row_offsets[e];
            for (int64_t t = 0; t < cnt; t += bn)
                for (int64_t mt = 0; mt < m_tiles; ++mt) {
                    MoeItem it{};
                    it.run = int32_t(ri);
                    it.m0 = int32_t(mt * kBM);
                    it.valid = int32_t(std::min<int64_t>(kBM, m_extent - mt * kBM));
                    it.a_row = int32_t(row_par ? k * rows_per_expert : k * rows_per_expert + mt * kBM);
                    it.x_row = int32_t(row_offsets[e] + t);
                    it.n_rows = int32_t(std::min<int64_t>(bn, cnt - t));
                    items.push_back(it);
                }
        }
    }
    if (items.size() >= (size_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: too many work items");

    ETP_CUDA_OK(cudaSetDevice(ctx->device));
    const int64_t need = int64_t(items.size()) * int64_t(sizeof(MoeItem));
    if (need > ctx->moe_items_bytes) {   // ctx-owned, grown on demand (calls on one ctx must not overlap in time)
        if (ctx->moe_items) ETP_CUDA_OK(cudaFree(ctx->moe_items));
        ctx->moe_items = nullptr;
        ctx->moe_items_bytes = 0;
        const int64_t want = std::max<int64_t>(need + need / 2, 1 << 16);
        ETP_CUDA_OK(cudaMalloc(&ctx->moe_items, size_t(want)));
        ctx->moe_items_bytes = want;
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    ETP_CUDA_OK(cudaMemcpyAsync(ctx->moe_items, items.data(), size_t(need), cudaMemcpyHostToDevice, st));   // pageable source: staged before return

    p.items = static_cast<const MoeItem*>(ctx->moe_items);
    p.n_items = int32_t(items.size());
    p.mode = mode;
    p.dtype = dtype;
    p.n_chunks = int32_t((in_features + kBK - 1) / kBK);
    p.out_features = int32_t(out_features);
    p.n_runs = int32_t(runs.size());
    p.y = y_perm;
    ETP_TRY(encode_2d(&p.map_x, dtype, x_perm, n_rows, in_features, in_features, kBK, std::min(bn, 64)));
    for (size_t ri = 0; ri < runs.size(); ++ri) {
        const void* base = runs[ri].base + runs[ri].slot0 * w->unit_bytes;
        if (row_par) ETP_TRY(encode_2d(&p.map_w[ri], dtype, base, runs[ri].n * rows_per_expert, row_len, row_len, 64, kBK));
        else ETP_TRY(encode_2d(&p.map_w[ri], dtype, base, runs[ri].n * rows_per_expert, row_len, row_len, kBK, kBM));
    }
    const int grid = int(std::min<int64_t>(p.n_items, ctx->n_sms));
    ctx->launches = 1;
    if (bn == 16) return launch_moe<16>(p, grid, st);
    if (bn == 64) return launch_moe<64>(p, grid, st);
    if (bn == 128) return launch_moe<128>(p, grid, st);
    return launch_moe<256>(p, grid, st);
}

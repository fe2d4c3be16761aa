// Grouped shard linear for MoE experts (readings G5, E1): one launch computes, for every expert
// INSTANCE with routed rows,  Y_perm[rows][out] = X_perm[rows][in] . W_e^T  on the expert matrices exactly where the
// expert-granularity reshard (the expert is the unit of the plan; slot-addressed slabs, L3) or the EPLB-style
// replication (Fig. 4) left them.
//   ETP_COL_PARALLEL  W_e stored [out][in]  (gate, up):   A = K-major rows of W_e
//   ETP_ROW_PARALLEL  W_e stored [in][out]  (down_t):     A = MN-major, K loop over the expert's own in-features
//   FUSED gate | up   (etp_moe_gate_up): both projections of an item share the X tile; two TMEM accumulators per stage;
//                     the epilogue writes silu(gate x) . (up x) once, in 16 bit - X is read once and the two [rows][ffn]
//                     intermediates of the three-launch layer never exist.
// Same tcgen05 / TMEM / TMA pipeline as etp_shard_linear: D[m = out feature][n = routed row] in TMEM, 128 x BN tiles, warp 0
// TMA producer, warp 1 MMA issuer, warps 2-5 epilogue, two accumulator stages.  The work list is a table of 32-byte ITEM
// descriptors (instance, m tile, row tile) built on the host per call (the experts' row counts are ragged) and uploaded into a
// stream-ordered allocation, so calls on different streams of one ctx share nothing.  One tensor map per rank covers the whole
// slab; a tile may over-read rows of the next slot (W, column-parallel) or of the next expert (X) - both only feed accumulator
// rows / columns that the epilogue masks.
#include <algorithm>
#include <cstring>
#include <vector>

#define ETP_WAIT_TU 4
#include "etp_tc.cuh"

using namespace etp;
using namespace etp::tc;

namespace {

struct MoeItem {       // 32 bytes
    int32_t map;       // tensor map of the rank whose slab holds the instance
    int32_t a_row;     // column-parallel: first weight row of the tile inside the slab; row-parallel: the instance's first k row
    int32_t m0;        // first out feature of the tile (column offset in Y_perm)
    int32_t valid;     // out features of the tile that exist (<= 128)
    int32_t x_row;     // first routed row of the tile in X_perm / Y_perm
    int32_t n_rows;    // rows of the tile that belong to the instance (<= BN)
    int32_t pad[2];
};
static_assert(sizeof(MoeItem) == 32, "MoeItem layout");

struct alignas(64) MoeParams {
    CUtensorMap map_x;
    CUtensorMap map_xh[8];          // CTA-pair kernel: the same X with boxes of 16, 32, .. 128 rows (one TMA per half tile)
    CUtensorMap map_w[kMaxRuns];    // per rank (gate, in the fused kernel)
    CUtensorMap map_w2[kMaxRuns];   // fused kernel: up
    const MoeItem* items;
    const int32_t* first;                     // CTA-pair kernel: cluster c runs items [first[c], first[c + 1]) of `items`
    int32_t n_items, mode, dtype, n_chunks;   // n_chunks: K chunks of kBK per item
    int32_t out_features, n_maps;
    void* y;
};

template <int BN, bool FUSED>
struct MoeCfg {
    static constexpr int kAStage = FUSED ? 2 * kABytes : kABytes;
    static constexpr int kBBytes = BN * kBK * 2;
    static constexpr int kStageBytes = kAStage + kBBytes;
    static constexpr int kStages = (kSmemBudget / kStageBytes) > 12 ? 12 : (kSmemBudget / kStageBytes);
    static constexpr int kAccCols = FUSED ? 2 * BN : BN;                          // TMEM columns of one accumulator stage
    static constexpr int kTmemCols = (2 * kAccCols) < 32 ? 32 : 2 * kAccCols;      // two stages; a power of two >= 32
    static constexpr int kSmemBytes = kStages * kStageBytes + 1024 + 256 + 4096;   // + per-warp epilogue transpose buffers
    static_assert(kTmemCols <= 512, "TMEM has 512 columns");
};

__device__ __forceinline__ MoeItem load_item(const MoeItem* items, int i) {
    const int4 a = __ldg(reinterpret_cast<const int4*>(items + i));
    const int4 b = __ldg(reinterpret_cast<const int4*>(items + i) + 1);
    MoeItem it;
    it.map = a.x; it.a_row = a.y; it.m0 = a.z; it.valid = a.w;
    it.x_row = b.x; it.n_rows = b.y;
    return it;
}

__device__ __forceinline__ float silu_mul(float g, float u) { return __fdividef(g, 1.f + __expf(-g)) * u; }

template <int BN, typename OutT, bool FUSED>
__global__ void __launch_bounds__(kLinThreads, 1) etp_moe_linear_kernel(const __grid_constant__ MoeParams p) {
    using C = MoeCfg<BN, FUSED>;
    constexpr int kXBox = BN < 64 ? BN : 64;   // rows per TMA box of the X tile
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + C::kStages * C::kStageBytes);
    uint64_t* empty_bar = full_bar + C::kStages;
    uint64_t* tmem_full = empty_bar + C::kStages;
    uint64_t* tmem_empty = tmem_full + 2;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(tmem_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool row_par = !FUSED && p.mode == ETP_ROW_PARALLEL;

    if (warp == 0 && lane == 1) {
        prefetch_tensormap(&p.map_x);
        for (int r = 0; r < p.n_maps; ++r) {
            prefetch_tensormap(&p.map_w[r]);
            if (FUSED) prefetch_tensormap(&p.map_w2[r]);
        }
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
                    uint8_t* sb = sa + C::kAStage;
                    mbar_wait(&empty_bar[stage], phase ^ 1);
                    mbar_expect_tx(&full_bar[stage], uint32_t(C::kAStage + nb * kXBox * kBK * 2));
                    if (!row_par) {
                        tma_load_2d(sa, &p.map_w[it.map], &full_bar[stage], c * kBK, it.a_row);
                        if (FUSED) tma_load_2d(sa + kABytes, &p.map_w2[it.map], &full_bar[stage], c * kBK, it.a_row);
                    } else {
                        tma_load_2d(sa, &p.map_w[it.map], &full_bar[stage], it.m0, it.a_row + c * kBK);
                        tma_load_2d(sa + kABytes / 2, &p.map_w[it.map], &full_bar[stage], it.m0 + 64, it.a_row + c * kBK);
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
                const uint32_t d_tmem = tmem_base + uint32_t(as * C::kAccCols);
                for (int c = 0; c < p.n_chunks; ++c) {
                    uint8_t* sa = smem + stage * C::kStageBytes;
                    mbar_wait(&full_bar[stage], phase);
                    tc_fence_after();
                    const uint64_t a_desc = make_smem_desc(smem_u32(sa), a_lbo, 1024);
                    const uint64_t b_desc = make_smem_desc(smem_u32(sa + C::kAStage), 16, 1024);
#pragma unroll
                    for (int k = 0; k < kBK / kUmmaK; ++k)
                        tc_mma(d_tmem, a_desc + uint64_t(k) * a_kstep, b_desc + uint64_t(k) * 2u, idesc, (c > 0 || k > 0) ? 1u : 0u);
                    if (FUSED) {   // the up projection of the same rows into the second accumulator of the stage
                        const uint64_t a2_desc = make_smem_desc(smem_u32(sa + kABytes), a_lbo, 1024);
#pragma unroll
                        for (int k = 0; k < kBK / kUmmaK; ++k)
                            tc_mma(d_tmem + uint32_t(BN), a2_desc + uint64_t(k) * a_kstep, b_desc + uint64_t(k) * 2u, idesc, (c > 0 || k > 0) ? 1u : 0u);
                    }
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
            const uint32_t taddr = tmem_base + uint32_t(as * C::kAccCols) + (uint32_t(q * 32) << 16);
            // up to 64 accumulator columns per tcgen05.wait::ld (four loads in flight hide the TMEM read latency; the fused kernel
            // reads 32 columns of each of its two accumulators); every 16 columns go through a 1-KiB per-warp transpose buffer so
            // that the global stores are 16 bytes per lane (8 routed rows x 64 contiguous bytes per instruction) instead of 2 - m0
            // and out_features are multiples of 8 by contract.
            constexpr int kStep = FUSED ? 32 : 64;
            for (int c0 = 0; c0 < it.n_rows; c0 += kStep) {
                uint32_t v[4][16];
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    const int col = FUSED ? c0 + 16 * (g & 1) : c0 + 16 * g;   // fused: g = 0, 1 gate columns, g = 2, 3 the same columns of up
                    if (BN >= 16 * ((FUSED ? (g & 1) : g) + 1) && col < it.n_rows) tc_ld16(taddr + uint32_t(col) + (FUSED && g >= 2 ? uint32_t(BN) : 0u), v[g]);
                }
                tc_ld_wait();
#pragma unroll
                for (int g = 0; g < (FUSED ? 2 : 4); ++g) {
                    const int col = c0 + 16 * g;
                    if (BN >= 16 * (g + 1) && col < it.n_rows) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const float r = FUSED ? silu_mul(__uint_as_float(v[g][j]), __uint_as_float(v[g + 2][j])) : __uint_as_float(v[g][j]);
                            stage_t[j * 32 + lane] = cvt16<OutT>(r);
                        }
                        __syncwarp();
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int row = h * 8 + (lane >> 2), chunk = lane & 3;
                            const int tok = col + row;
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

// ------------------------------------------------------------------------------------------------ CTA-pair kernel
// Many routed rows per expert: the single-CTA kernel above is bound by what an SM can pull from L2 (the chip-wide L2 output of
// ~6300 B/clk is ~42 B/clk per SM; a fused item stages 32 KiB of weights + 16 KiB of X per K chunk for 2 x 128 x 128 x 64 MACs).
// Two CTAs of a cluster run ONE tcgen05.mma.cta_group::2 of M = 256 out features x N <= 256 routed rows: CTA rank c owns out
// feature tile 2 * pm + c (its A tile(s), its 128 TMEM lanes) and stages HALF of the X rows, so the same MACs need 48 KiB per CTA
// for twice the rows (fused: 171 flop per staged byte instead of 85).  N is the item's row count rounded up to 32; each CTA
// loads its N / 2 rows with ONE TMA (eight X maps with boxes of 16 .. 128 rows).  Protocol as etp_shard_linear_pair_kernel: both CTAs' TMA loads complete on the LEADER's full
// barrier, only the leader issues MMAs, tcgen05.commit multicasts "stage free" / "accumulator ready" to both CTAs, the epilogue
// warps of both arrive on the leader's "accumulator drained" barrier.  The fused kernel holds gate and up for 256 rows in all
// 512 TMEM columns (one accumulator stage: its epilogue is not overlapped with the next item's MMAs); the plain kernel keeps two
// stages of 256 columns.  Work: cluster c runs items [first[c], first[c + 1]) - a list schedule computed on the host from a cost
// model, in instance order so that the items sharing an X tile or an expert's weights run at about the same time (L2 hits).
template <bool FUSED>
struct MoePairCfg {
    static constexpr int kBN = 256;
    static constexpr int kAStage = FUSED ? 2 * kABytes : kABytes;
    static constexpr int kBBytes = (kBN / 2) * kBK * 2;
    static constexpr int kStageBytes = kAStage + kBBytes;
    static constexpr int kStages = (kSmemBudget / kStageBytes) > 8 ? 8 : (kSmemBudget / kStageBytes);
    static constexpr int kAccCols = FUSED ? 2 * kBN : kBN;
    static constexpr int kAccStages = FUSED ? 1 : 2;
    static constexpr int kTmemCols = 512;
    static constexpr int kThreads = 320;                             // TMA warp, MMA warp, 8 epilogue warps
    static constexpr int kSmemBytes = kStages * kStageBytes + 1024 + 256 + 8192;
};

#ifdef ETP_MOE_TIMING
// bring-up instrumentation (never in the product build): per cluster, sums of SM clocks
__device__ unsigned long long g_moe_t[128][8];
#define MOE_T(slot, expr) do { if (rank == 0) atomicAdd(&g_moe_t[cluster_id][slot], (unsigned long long)(expr)); } while (0)
#define MOE_CLK() clock64()
#else
#define MOE_T(slot, expr) do { } while (0)
#define MOE_CLK() 0ll
#endif

template <typename OutT, bool FUSED>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(MoePairCfg<FUSED>::kThreads, 1) etp_moe_pair_kernel(const __grid_constant__ MoeParams p) {
    using C = MoePairCfg<FUSED>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + C::kStages * C::kStageBytes);
    uint64_t* empty_bar = full_bar + C::kStages;
    uint64_t* tmem_full = empty_bar + C::kStages;
    uint64_t* tmem_empty = tmem_full + 2;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(tmem_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int cluster_id = blockIdx.x >> 1;
    const bool row_par = !FUSED && p.mode == ETP_ROW_PARALLEL;
    const int i_begin = __ldg(&p.first[cluster_id]), i_end = __ldg(&p.first[cluster_id + 1]);
    const long long t_kernel0 = MOE_CLK();
    (void)t_kernel0;

    if (warp == 0 && lane == 1) {
        for (int r = 0; r < 8; ++r) prefetch_tensormap(&p.map_xh[r]);
        for (int r = 0; r < p.n_maps; ++r) {
            prefetch_tensormap(&p.map_w[r]);
            if (FUSED) prefetch_tensormap(&p.map_w2[r]);
        }
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < C::kStages; ++s) {
            mbar_init(&full_bar[s], 1);      // used in the leader only: its own arrive.expect_tx of both CTAs' bytes
            mbar_init(&empty_bar[s], 1);     // one multicast commit per use
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&tmem_full[s], 1);     // one multicast commit per item
            mbar_init(&tmem_empty[s], 16);   // leader only: 8 epilogue warps of each CTA
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_ptr)), "r"(uint32_t(C::kTmemCols))
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();      // the peer's barriers exist before anything signals them
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    if (warp == 0) {
        if (lane == 0) {   // ------------------------------------------------------------------ TMA producer (one lane of each CTA)
            int stage = 0;
            uint32_t phase = 0;
            MoeItem nxt = i_begin < i_end ? load_item(p.items, i_begin) : MoeItem{};
            for (int i = i_begin; i < i_end; ++i) {
                const MoeItem it = nxt;
                if (i + 1 < i_end) nxt = load_item(p.items, i + 1);         // in flight while this item's tiles are requested
                const int h = ((it.n_rows + 31) >> 5) << 4;                 // N = 2 h (a multiple of 32); this CTA stages rows [x0, x0 + h)
                const int x0 = it.x_row + int(rank) * h;
                const CUtensorMap* mx = &p.map_xh[(h >> 4) - 1];
                const int a_row = row_par ? it.a_row : it.a_row + int(rank) * kBM;
                const int m0 = it.m0 + int(rank) * kBM;
                for (int c = 0; c < p.n_chunks; ++c) {
                    uint8_t* sa = smem + stage * C::kStageBytes;
                    uint8_t* sb = sa + C::kAStage;
                    const long long tp0 = MOE_CLK();
                    mbar_wait(&empty_bar[stage], phase ^ 1);
                    MOE_T(0, MOE_CLK() - tp0);
                    const uint32_t lbar = mapa_rank0(smem_u32(&full_bar[stage]));
                    if (rank == 0) mbar_expect_tx(&full_bar[stage], 2u * uint32_t(C::kAStage + h * kBK * 2));
                    if (!row_par) {
                        tma_load_2d_pair(sa, &p.map_w[it.map], lbar, c * kBK, a_row);
                        if (FUSED) tma_load_2d_pair(sa + kABytes, &p.map_w2[it.map], lbar, c * kBK, a_row);
                    } else {
                        tma_load_2d_pair(sa, &p.map_w[it.map], lbar, m0, a_row + c * kBK);
                        tma_load_2d_pair(sa + kABytes / 2, &p.map_w[it.map], lbar, m0 + 64, a_row + c * kBK);
                    }
                    tma_load_2d_pair(sb, mx, lbar, c * kBK, x0);
                    if (++stage == C::kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        if (lane == 0 && rank == 0) {   // ------------------------------------------------------ MMA issuer (one lane of the LEADER)
            const uint32_t a_lbo = row_par ? uint32_t(kABytes / 2) : 16u;
            const uint32_t a_kstep = row_par ? (uint32_t(kUmmaK) * 128u) >> 4 : (uint32_t(kUmmaK) * 2u) >> 4;
            int stage = 0;
            uint32_t phase = 0;
            int local = 0;
            int n_rows_next = i_begin < i_end ? __ldg(&p.items[i_begin].n_rows) : 0;
            for (int i = i_begin; i < i_end; ++i, ++local) {
                const int n_rows = n_rows_next;
                if (i + 1 < i_end) n_rows_next = __ldg(&p.items[i + 1].n_rows);   // in flight while this item's MMAs are issued
                const uint32_t idesc = make_idesc_pair(p.dtype == ETP_BF16 ? 1u : 0u, row_par ? 1u : 0u, uint32_t(((n_rows + 31) >> 5) << 5));
                const int as = local % C::kAccStages;
                const uint32_t aph = uint32_t(local / C::kAccStages) & 1u;
                const long long tm0 = MOE_CLK();
                mbar_wait(&tmem_empty[as], aph ^ 1);   // both CTAs' epilogues have drained this accumulator stage
                MOE_T(1, MOE_CLK() - tm0);
                MOE_T(4, 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + uint32_t(as * C::kAccCols);
                for (int c = 0; c < p.n_chunks; ++c) {
                    uint8_t* sa = smem + stage * C::kStageBytes;
                    const long long tm1 = MOE_CLK();
                    mbar_wait(&full_bar[stage], phase);
                    MOE_T(c < C::kStages ? 2 : 3, MOE_CLK() - tm1);
                    tc_fence_after();
                    const uint64_t a_desc = make_smem_desc(smem_u32(sa), a_lbo, 1024);
                    const uint64_t b_desc = make_smem_desc(smem_u32(sa + C::kAStage), 16, 1024);
#pragma unroll
                    for (int k = 0; k < kBK / kUmmaK; ++k)
                        tc_mma_pair(d_tmem, a_desc + uint64_t(k) * a_kstep, b_desc + uint64_t(k) * 2u, idesc, (c > 0 || k > 0) ? 1u : 0u);
                    if (FUSED) {
                        const uint64_t a2_desc = make_smem_desc(smem_u32(sa + kABytes), a_lbo, 1024);
#pragma unroll
                        for (int k = 0; k < kBK / kUmmaK; ++k)
                            tc_mma_pair(d_tmem + uint32_t(C::kBN), a2_desc + uint64_t(k) * a_kstep, b_desc + uint64_t(k) * 2u, idesc, (c > 0 || k > 0) ? 1u : 0u);
                    }
                    tc_commit_pair(&empty_bar[stage]);   // frees the stage in BOTH CTAs once these MMAs have read it
                    if (++stage == C::kStages) { stage = 0; phase ^= 1; }
                }
                tc_commit_pair(&tmem_full[as]);
            }
        }
        __syncwarp();
    } else {               // ---------------------------------------------------------------------- epilogue warps 2..9 of both CTAs
        // Two warps per TMEM lane quarter (a warp may only read lanes 32 * (warp % 4) ..): warp `half` of a quarter takes the column
        // blocks half, half + 2, ... of kStep routed rows.  The tcgen05.ld of the next block are in flight while the current one
        // goes through the activation, the transpose buffer and the 16-byte stores.
        const int q = warp & 3, half = (warp - 2) >> 2;
        OutT* y = reinterpret_cast<OutT*>(p.y);
        OutT* stage_t = reinterpret_cast<OutT*>(smem + C::kStages * C::kStageBytes + 256) + (warp - 2) * 512;   // [16 rows][32 features]
        const uint32_t drained = mapa_rank0(smem_u32(&tmem_empty[0]));
        constexpr int kStep = FUSED ? 32 : 64;
        int local = 0;
        for (int i = i_begin; i < i_end; ++i, ++local) {
            const MoeItem it = load_item(p.items, i);
            const int as = local % C::kAccStages;
            const uint32_t aph = uint32_t(local / C::kAccStages) & 1u;
            const int m0 = it.m0 + int(rank) * kBM;
            const int valid = it.valid - int(rank) * kBM;   // <= 0: this CTA's tile lies past the last out feature
            mbar_wait(&tmem_full[as], aph);
            const long long te0 = MOE_CLK();
            tc_fence_after();
            const uint32_t taddr = tmem_base + uint32_t(as * C::kAccCols) + (uint32_t(q * 32) << 16);
            auto load_blk = [&](int c0, uint32_t (&v)[4][16]) {
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    const int col = FUSED ? c0 + 16 * (g & 1) : c0 + 16 * g;   // fused: g = 0, 1 gate columns, g = 2, 3 the same columns of up
                    if (col < it.n_rows) tc_ld16(taddr + uint32_t(col) + (FUSED && g >= 2 ? uint32_t(C::kBN) : 0u), v[g]);
                }
            };
            auto emit_blk = [&](int c0, const uint32_t (&v)[4][16]) {
#pragma unroll
                for (int g = 0; g < (FUSED ? 2 : 4); ++g) {
                    const int col = c0 + 16 * g;
                    if (col < it.n_rows) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const float r = FUSED ? silu_mul(__uint_as_float(v[g][j]), __uint_as_float(v[g + 2][j])) : __uint_as_float(v[g][j]);
                            stage_t[j * 32 + lane] = cvt16<OutT>(r);
                        }
                        __syncwarp();
#pragma unroll
                        for (int hh = 0; hh < 2; ++hh) {
                            const int row = hh * 8 + (lane >> 2), chunk = lane & 3;
                            const int tok = col + row;
                            const uint4 val = *reinterpret_cast<const uint4*>(stage_t + row * 32 + chunk * 8);
                            if (tok < it.n_rows && q * 32 + chunk * 8 < valid)
                                *reinterpret_cast<uint4*>(y + size_t(it.x_row + tok) * p.out_features + m0 + q * 32 + chunk * 8) = val;
                        }
                        __syncwarp();
                    }
                }
            };
            int c0 = half * kStep;
            if (q * 32 < valid && c0 < it.n_rows) {
                uint32_t va[4][16], vb[4][16];
                load_blk(c0, va);
                tc_ld_wait();
                for (;;) {
                    const int c1 = c0 + 2 * kStep;
                    if (c1 < it.n_rows) load_blk(c1, vb);
                    emit_blk(c0, va);
                    if (c1 >= it.n_rows) break;
                    tc_ld_wait();
                    c0 = c1 + 2 * kStep;
                    if (c0 < it.n_rows) load_blk(c0, va);
                    emit_blk(c1, vb);
                    if (c0 >= it.n_rows) break;
                    tc_ld_wait();
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(drained + uint32_t(as) * 8u);
            if (warp == 2 && lane == 0) MOE_T(5, MOE_CLK() - te0);
        }
    }
    if (threadIdx.x == 0) MOE_T(6, MOE_CLK() - t_kernel0);

    tc_fence_before();
    __syncthreads();
    cluster_sync_all();      // the leader's MMAs read the peer's shared memory and both CTAs free the paired TMEM
    if (warp == 1) {
        __syncwarp();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(uint32_t(C::kTmemCols)) : "memory");
    }
}

template <typename OutT, bool FUSED>
etp_status launch_moe_pair_t(const MoeParams& p, int grid, cudaStream_t stream) {
    using C = MoePairCfg<FUSED>;
    auto k = etp_moe_pair_kernel<OutT, FUSED>;
    static bool configured = false;
    if (!configured) {
        ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes));
        configured = true;
    }
    k<<<grid, C::kThreads, C::kSmemBytes, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) ETP_FAIL(ETP_ERR_CUDA, "etp_moe_linear: pair launch failed: %s", cudaGetErrorString(e));
    return ETP_OK;
}
template <bool FUSED>
etp_status launch_moe_pair(const MoeParams& p, int grid, cudaStream_t st) {
    return p.dtype == ETP_BF16 ? launch_moe_pair_t<__nv_bfloat16, FUSED>(p, grid, st) : launch_moe_pair_t<__half, FUSED>(p, grid, st);
}

template <int BN, typename OutT, bool FUSED>
etp_status launch_moe_t(const MoeParams& p, int grid, cudaStream_t stream) {
    using C = MoeCfg<BN, FUSED>;
    auto k = etp_moe_linear_kernel<BN, OutT, FUSED>;
    static bool configured = false;
    if (!configured) {
        ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes));
        configured = true;
    }
    k<<<grid, kLinThreads, C::kSmemBytes, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) ETP_FAIL(ETP_ERR_CUDA, "etp_moe_linear: launch failed: %s", cudaGetErrorString(e));
    return ETP_OK;
}

template <bool FUSED>
etp_status launch_moe(const MoeParams& p, int bn, int grid, cudaStream_t st) {
    const bool bf = p.dtype == ETP_BF16;
    if (bn == 16) return bf ? launch_moe_t<16, __nv_bfloat16, FUSED>(p, grid, st) : launch_moe_t<16, __half, FUSED>(p, grid, st);
    if (bn == 64) return bf ? launch_moe_t<64, __nv_bfloat16, FUSED>(p, grid, st) : launch_moe_t<64, __half, FUSED>(p, grid, st);
    if (bn == 128) return bf ? launch_moe_t<128, __nv_bfloat16, FUSED>(p, grid, st) : launch_moe_t<128, __half, FUSED>(p, grid, st);
    if constexpr (FUSED) {   // two accumulators of 256 columns x two stages would exceed the 512 TMEM columns
        ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_moe_gate_up: no 256-row tile");
    } else {
        return bf ? launch_moe_t<256, __nv_bfloat16, false>(p, grid, st) : launch_moe_t<256, __half, false>(p, grid, st);
    }
}

// ------------------------------------------------------------------------------------------------ host side
struct Inst {   // one expert instance with routed rows
    int32_t rank;
    int64_t slot, row_b, row_e;
};

// Slot of unit u in rank r's slab (L3) if the layout says r holds u, else -1.
etp_status home_of(const etp_tensor* w, const std::vector<etp_shard>& sh, int64_t u, int32_t* rank, int64_t* slot) {
    for (const etp_shard& s : sh)
        if (s.begin <= u && u < s.end) {
            if (s.rank < 0 || s.rank >= w->n_ranks || !w->slabs[s.rank].base) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: rank %d has no slab", s.rank);
            const etp_slab& sl = w->slabs[s.rank];
            if (sl.cap_units <= 0 || s.end - s.begin > sl.cap_units)
                ETP_FAIL(ETP_ERR_CAPACITY, "etp_moe_linear: shard of rank %d (%lld experts) exceeds its slab (%lld)", s.rank, (long long)(s.end - s.begin), (long long)sl.cap_units);
            int64_t v = (u - sl.anchor_unit) % sl.cap_units;
            *slot = v < 0 ? v + sl.cap_units : v;
            *rank = s.rank;
            return ETP_OK;
        }
    ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: expert %lld is in no shard of the layout", (long long)u);
}

etp_status sorted_layout(const etp_shard* layout, int32_t n_shards, int64_t n_units, std::vector<etp_shard>* sh) {
    sh->clear();
    if (!layout || n_shards <= 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: empty layout");
    for (int i = 0; i < n_shards; ++i)
        if (layout[i].alive && layout[i].end > layout[i].begin) sh->push_back(layout[i]);
    std::sort(sh->begin(), sh->end(), [](const etp_shard& a, const etp_shard& b) { return a.begin < b.begin; });
    int64_t cursor = 0;
    for (const etp_shard& s : *sh) {
        if (s.begin != cursor) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: layout does not tile [0,%lld): gap or overlap at expert %lld", (long long)n_units, (long long)cursor);
        cursor = s.end;
    }
    if (cursor != n_units) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: layout covers %lld of %lld experts", (long long)cursor, (long long)n_units);
    return ETP_OK;
}

// w2 != NULL: fused gate | up (column-parallel, silu(w x) . (w2 x)); its slabs must mirror w's geometry rank by rank.
etp_status moe_run(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x_perm, int64_t n_rows, const std::vector<Inst>& insts,
                   int64_t in_features, int64_t out_features, const etp_tensor* w, const etp_tensor* w2, void* y_perm, void* stream) {
    const bool fused = w2 != nullptr;
    const bool row_par = mode == ETP_ROW_PARALLEL;
    const int64_t rows_per_expert = row_par ? in_features : out_features;   // rows of the stored expert matrix
    const int64_t row_len = row_par ? out_features : in_features;
    if (n_rows == 0 || insts.empty()) return ETP_OK;
    if (!x_perm || !y_perm) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: x / y is NULL");
    if ((reinterpret_cast<uintptr_t>(x_perm) | reinterpret_cast<uintptr_t>(y_perm)) & 15) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_moe_linear: x / y not 16-byte aligned");

    MoeParams p;
    std::memset(&p, 0, sizeof(p));
    // ---- one tensor map per rank over its whole slab
    std::vector<int32_t> map_of(size_t(w->n_ranks), -1);
    int n_maps = 0;
    for (const Inst& in : insts) {
        if (in.rank < 0 || in.rank >= w->n_ranks) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: instance on rank %d, the tensor has %d slabs", in.rank, w->n_ranks);
        const etp_slab& sl = w->slabs[in.rank];
        if (!sl.base) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: rank %d has no slab", in.rank);
        if (in.slot < 0 || in.slot >= sl.cap_units) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: slot %lld outside the slab of rank %d (%lld slots)", (long long)in.slot, in.rank, (long long)sl.cap_units);
        if (map_of[in.rank] >= 0) continue;
        if (reinterpret_cast<uintptr_t>(sl.base) & 15) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_moe_linear: slab of rank %d not 16-byte aligned", in.rank);
        if (n_maps == kMaxRuns) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_moe_linear: more than %d ranks", kMaxRuns);
        if (sl.cap_units * rows_per_expert >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: slab too long");
        const int bc = row_par ? 64 : kBK, br = row_par ? kBK : kBM;
        ETP_TRY(encode_2d(&p.map_w[n_maps], dtype, sl.base, sl.cap_units * rows_per_expert, row_len, row_len, bc, br));
        if (fused) {
            if (in.rank >= w2->n_ranks || !w2->slabs[in.rank].base || w2->slabs[in.rank].cap_units != sl.cap_units || w2->slabs[in.rank].anchor_unit != sl.anchor_unit)
                ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_gate_up: the slabs of gate and up must have the same geometry (rank %d)", in.rank);
            if (reinterpret_cast<uintptr_t>(w2->slabs[in.rank].base) & 15) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_moe_gate_up: slab of rank %d not 16-byte aligned", in.rank);
            ETP_TRY(encode_2d(&p.map_w2[n_maps], dtype, w2->slabs[in.rank].base, sl.cap_units * rows_per_expert, row_len, row_len, bc, br));
        }
        map_of[in.rank] = n_maps++;
    }

    // ---- row tile BN: operand fetch into the SM bounds a tile (measured on kernel (c): 48 KiB per K chunk at BN = 256 is the
    // limit, the MMA is not), so an item costs (A tile(s) + BN rows of X) bytes per K chunk; take the BN with the least total.
    int bn = 16;
    {
        int64_t best = INT64_MAX;
        const int64_t a_bytes = fused ? 2 * kABytes : kABytes;
        for (int cand : {256, 128, 64, 16}) {
            if (fused && cand == 256) continue;
            int64_t cost = 0;
            const int box = std::min(cand, 64);
            for (const Inst& in : insts) {
                const int64_t c = in.row_e - in.row_b;
                const int64_t tiles = (c + cand - 1) / cand, boxes = (c + box - 1) / box;   // X is fetched in boxes of <= 64 rows
                cost += tiles * a_bytes + boxes * box * kBK * 2;
            }
            if (cost < best) { best = cost; bn = cand; }
        }
    }

    // ---- CTA pairs when the row tiles are large (ETP_OPT_MOE_CTA_PAIR: 1 = when the cost model above picked >= 128 rows,
    // 2 = always, 0 = never)
    const int64_t pair_opt = ctx->opts[ETP_OPT_MOE_CTA_PAIR];
    const bool pair = ctx->n_sms >= 2 && (pair_opt == 2 || (pair_opt == 1 && bn >= 128));

    // ---- items: (instance, row tile, m tile), m tiles of one row tile adjacent so that its X tile stays in L2
    // Pair kernel: an instance with c rows gets ceil(c / 256) row tiles of EQUAL size (rounded up to 32 rows) - a 296-row expert
    // runs 160 + 136 rows, not 256 + 40: every tile re-streams the expert's weights, and a 40-row tile would do so for a quarter of
    // the MMA work of a full one (it is bound by the weight fetch, not by the MMA).
    const int m_step = pair ? 2 * kBM : kBM;
    const int64_t m_tiles = (out_features + m_step - 1) / m_step;
    std::vector<MoeItem> items;
    for (const Inst& in : insts) {
        const int64_t c_rows = in.row_e - in.row_b;
        int64_t row_step = bn;
        if (pair) {
            const int64_t tiles = (c_rows + 255) / 256;
            row_step = ((c_rows + tiles - 1) / tiles + 31) / 32 * 32;
        }
        for (int64_t t = in.row_b; t < in.row_e; t += row_step)
            for (int64_t mt = 0; mt < m_tiles; ++mt) {
                MoeItem it{};
                it.map = map_of[in.rank];
                it.m0 = int32_t(mt * m_step);
                it.valid = int32_t(std::min<int64_t>(m_step, out_features - mt * m_step));
                it.a_row = int32_t(row_par ? in.slot * rows_per_expert : in.slot * rows_per_expert + mt * m_step);
                it.x_row = int32_t(t);
                it.n_rows = int32_t(std::min<int64_t>(row_step, in.row_e - t));
                items.push_back(it);
            }
    }
    if (items.empty()) return ETP_OK;
    if (items.size() >= (size_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: too many work items");
    const int32_t n_chunks = int32_t((in_features + kBK - 1) / kBK);

    // ---- pair kernel: list schedule.  Items are dealt in order to the cluster with the least accumulated cost (what a work queue
    // would do, decided here so that the two CTAs of a cluster need no exchange); cost of an item in SM clocks = the larger of its
    // operand fetch (~55 B/clk per SM sustained from L2, measured on kernel (c)'s pair kernel) and its MMA time (N / 2 clk per
    // UMMA_K step), plus the epilogue where it is not overlapped (fused: one accumulator stage; ~22 clk per row, from ncu's
    // tensor-pipe-active share), plus a fixed per-item cost (pipeline refill, descriptor fetch).
    std::vector<int32_t> first;
    int n_clusters = 0;
    if (pair) {
        n_clusters = int(std::min<int64_t>(int64_t(items.size()), ctx->n_sms / 2));
        std::vector<int64_t> load(size_t(n_clusters), 0);
        std::vector<int32_t> owner(items.size());
        const int64_t a_stage = fused ? 2 * kABytes : kABytes;
        std::vector<int64_t> cost(items.size());
        for (size_t i = 0; i < items.size(); ++i) {
            const int64_t h = (items[i].n_rows + 31) / 32 * 16;   // rows staged per CTA; UMMA_N = 2 h
            const int64_t fetch = (a_stage + h * kBK * 2) * n_chunks / 55;
            const int64_t mma = int64_t(n_chunks) * (kBK / kUmmaK) * (fused ? 2 : 1) * h;
            const int64_t epi = int64_t(items[i].n_rows) * (fused ? 22 : 11);
            cost[i] = (fused ? std::max(fetch, mma) + epi : std::max(std::max(fetch, mma), epi)) + 1000;
        }
        // in instance order, NOT longest-first: dealing the items by descending cost (measured) takes the fused launch from 195 to
        // 233 us - the items that share an X tile or an expert's weights no longer run together and miss in L2
        for (size_t i = 0; i < items.size(); ++i) {
            int best = 0;
            for (int c = 1; c < n_clusters; ++c)
                if (load[size_t(c)] < load[size_t(best)]) best = c;
            owner[i] = best;
            load[size_t(best)] += cost[i];
        }
        first.assign(size_t(n_clusters) + 1, 0);
        for (size_t i = 0; i < items.size(); ++i) ++first[size_t(owner[i]) + 1];
        for (int c = 0; c < n_clusters; ++c) first[size_t(c) + 1] += first[size_t(c)];
        std::vector<int32_t> cursor(first.begin(), first.end() - 1);
        std::vector<MoeItem> sorted(items.size());
        for (size_t i = 0; i < items.size(); ++i) sorted[size_t(cursor[size_t(owner[i])]++)] = items[i];
        items.swap(sorted);
    }

    ETP_CUDA_OK(cudaSetDevice(ctx->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // table = [first[] padded to 32 bytes][items]; one stream-ordered allocation, one upload
    const size_t head = (first.size() * sizeof(int32_t) + 31) / 32 * 32;
    const size_t need = head + items.size() * sizeof(MoeItem);
    std::vector<uint8_t> table(need, 0);
    if (!first.empty()) std::memcpy(table.data(), first.data(), first.size() * sizeof(int32_t));
    std::memcpy(table.data() + head, items.data(), items.size() * sizeof(MoeItem));
    void* d_items = nullptr;
    ETP_CUDA_OK(cudaMallocAsync(&d_items, need, st));   // stream-ordered: nothing is shared between calls or streams
    cudaError_t e = cudaMemcpyAsync(d_items, table.data(), need, cudaMemcpyHostToDevice, st);   // pageable source: staged before return
    if (e != cudaSuccess) {
        cudaFreeAsync(d_items, st);
        ETP_FAIL(ETP_ERR_CUDA, "etp_moe_linear: uploading the item table failed: %s", cudaGetErrorString(e));
    }
    p.first = static_cast<const int32_t*>(d_items);
    p.items = reinterpret_cast<const MoeItem*>(static_cast<const uint8_t*>(d_items) + head);
    p.n_items = int32_t(items.size());
    p.mode = mode;
    p.dtype = dtype;
    p.n_chunks = n_chunks;
    p.out_features = int32_t(out_features);
    p.n_maps = n_maps;
    p.y = y_perm;
    etp_status s = ETP_OK;
    if (pair) {
        for (int r = 0; r < 8 && s == ETP_OK; ++r) s = encode_2d(&p.map_xh[r], dtype, x_perm, n_rows, in_features, in_features, kBK, 16 * (r + 1));
    } else {
        s = encode_2d(&p.map_x, dtype, x_perm, n_rows, in_features, in_features, kBK, std::min(bn, 64));
    }
    ctx->launches = 1;
    if (s == ETP_OK) {
        if (pair) {
            s = fused ? launch_moe_pair<true>(p, 2 * n_clusters, st) : launch_moe_pair<false>(p, 2 * n_clusters, st);
        } else {
            const int grid = int(std::min<int64_t>(p.n_items, ctx->n_sms));
            s = fused ? launch_moe<true>(p, bn, grid, st) : launch_moe<false>(p, bn, grid, st);
        }
    }
    cudaFreeAsync(d_items, st);
    return s;
}

etp_status check_moe_shapes(const char* who, etp_ctx* ctx, int mode, etp_dtype dtype, int32_t n_experts, int64_t in_features,
                            int64_t out_features, const etp_tensor* w) {
    if (!ctx || !w || !w->slabs) ETP_FAIL(ETP_ERR_INVALID_ARG, "%s: NULL argument", who);
    if (mode != ETP_COL_PARALLEL && mode != ETP_ROW_PARALLEL) ETP_FAIL(ETP_ERR_INVALID_ARG, "%s: bad mode %d", who, mode);
    if (dtype != ETP_BF16 && dtype != ETP_FP16) ETP_FAIL(ETP_ERR_UNSUPPORTED, "%s: dtype %d is not bf16/fp16", who, int(dtype));
    if (n_experts <= 0 || in_features <= 0 || out_features <= 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "%s: non-positive size", who);
    if (w->total_units != n_experts) ETP_FAIL(ETP_ERR_INVALID_ARG, "%s: the tensor has %lld units, n_experts = %d (one unit = one expert)", who, (long long)w->total_units, n_experts);
    if (w->unit_bytes != in_features * out_features * 2)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "%s: unit_bytes %lld != in x out x 2 = %lld", who, (long long)w->unit_bytes, (long long)(in_features * out_features * 2));
    if ((in_features * 2) % 16 || (out_features * 2) % 16) ETP_FAIL(ETP_ERR_ALIGNMENT, "%s: feature counts must be multiples of 8", who);
    if (mode == ETP_ROW_PARALLEL && in_features % kBK)
        ETP_FAIL(ETP_ERR_UNSUPPORTED, "%s: row-parallel experts need in_features %% %d == 0 (a K chunk must not run into the next expert)", who, kBK);
    if (in_features >= (int64_t(1) << 31) || out_features >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "%s: sizes must be below 2^31", who);
    return ETP_OK;
}

// rows [row_offsets[e], row_offsets[e+1]) of every expert on the rank / slot where the layout holds it
etp_status instances_from_layout(const int64_t* row_offsets, int32_t n_experts, const etp_tensor* w, const etp_shard* layout,
                                 int32_t n_shards, std::vector<Inst>* out, int64_t* n_rows) {
    if (!row_offsets || !layout) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: NULL argument");
    if (row_offsets[0] != 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: row_offsets[0] != 0");
    for (int32_t e = 0; e < n_experts; ++e)
        if (row_offsets[e + 1] < row_offsets[e]) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: row_offsets decrease at expert %d", e);
    *n_rows = row_offsets[n_experts];
    if (*n_rows >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear: sizes must be below 2^31");
    std::vector<etp_shard> sh;
    ETP_TRY(sorted_layout(layout, n_shards, n_experts, &sh));
    for (int32_t e = 0; e < n_experts; ++e) {
        int32_t r;
        int64_t slot;
        ETP_TRY(home_of(w, sh, e, &r, &slot));   // also validates every shard's slab, routed rows or not
        if (row_offsets[e + 1] > row_offsets[e]) out->push_back({r, slot, row_offsets[e], row_offsets[e + 1]});
    }
    return ETP_OK;
}

etp_status instances_from_list(const etp_moe_instance* inst, int32_t n_inst, int64_t n_rows, std::vector<Inst>* out) {
    if (n_inst < 0 || (n_inst > 0 && !inst) || n_rows < 0 || n_rows >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear_instances: bad arguments");
    std::vector<std::pair<int64_t, int64_t>> ranges;
    for (int32_t i = 0; i < n_inst; ++i) {
        if (inst[i].row_begin < 0 || inst[i].row_end < inst[i].row_begin || inst[i].row_end > n_rows)
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear_instances: instance %d has rows [%lld,%lld) outside [0,%lld)", i, (long long)inst[i].row_begin, (long long)inst[i].row_end, (long long)n_rows);
        if (inst[i].row_end == inst[i].row_begin) continue;
        out->push_back({inst[i].rank, inst[i].slot, inst[i].row_begin, inst[i].row_end});
        ranges.push_back({inst[i].row_begin, inst[i].row_end});
    }
    std::sort(ranges.begin(), ranges.end());
    for (size_t k = 1; k < ranges.size(); ++k)
        if (ranges[k].first < ranges[k - 1].second) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_linear_instances: two instances share row %lld", (long long)ranges[k].first);
    return ETP_OK;
}

}  // namespace

extern "C" etp_status etp_moe_linear(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x_perm,
                                     const int64_t* row_offsets, int32_t n_experts, int64_t in_features, int64_t out_features,
                                     const etp_tensor* w, const etp_shard* layout, int32_t n_shards, void* y_perm, void* stream) {
    ETP_TRY(check_moe_shapes("etp_moe_linear", ctx, mode, dtype, n_experts, in_features, out_features, w));
    std::vector<Inst> insts;
    int64_t n_rows = 0;
    ETP_TRY(instances_from_layout(row_offsets, n_experts, w, layout, n_shards, &insts, &n_rows));
    return moe_run(ctx, mode, dtype, x_perm, n_rows, insts, in_features, out_features, w, nullptr, y_perm, stream);
}

extern "C" etp_status etp_moe_linear_instances(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x_perm,
                                               const etp_moe_instance* instances, int32_t n_instances, int64_t n_rows,
                                               int32_t n_experts, int64_t in_features, int64_t out_features, const etp_tensor* w,
                                               void* y_perm, void* stream) {
    ETP_TRY(check_moe_shapes("etp_moe_linear_instances", ctx, mode, dtype, n_experts, in_features, out_features, w));
    std::vector<Inst> insts;
    ETP_TRY(instances_from_list(instances, n_instances, n_rows, &insts));
    return moe_run(ctx, mode, dtype, x_perm, n_rows, insts, in_features, out_features, w, nullptr, y_perm, stream);
}

extern "C" etp_status etp_moe_gate_up(etp_ctx* ctx, etp_dtype dtype, const void* x_perm, const int64_t* row_offsets,
                                      const etp_moe_instance* instances, int32_t n_instances, int64_t n_rows, int32_t n_experts,
                                      int64_t in_features, int64_t ffn, const etp_tensor* w_gate, const etp_tensor* w_up,
                                      const etp_shard* layout, int32_t n_shards, void* h_perm, void* stream) {
    ETP_TRY(check_moe_shapes("etp_moe_gate_up", ctx, ETP_COL_PARALLEL, dtype, n_experts, in_features, ffn, w_gate));
    ETP_TRY(check_moe_shapes("etp_moe_gate_up", ctx, ETP_COL_PARALLEL, dtype, n_experts, in_features, ffn, w_up));
    if (w_gate->n_ranks != w_up->n_ranks) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_moe_gate_up: gate and up have different rank counts");
    std::vector<Inst> insts;
    if (instances) {
        ETP_TRY(instances_from_list(instances, n_instances, n_rows, &insts));
    } else {
        ETP_TRY(instances_from_layout(row_offsets, n_experts, w_gate, layout, n_shards, &insts, &n_rows));
    }
    return moe_run(ctx, ETP_COL_PARALLEL, dtype, x_perm, n_rows, insts, in_features, ffn, w_gate, w_up, h_perm, stream);
}

// ------------------------------------------------------------------------------------------------ EPLB: materialise replicas
extern "C" etp_status etp_eplb_apply(etp_ctx* ctx, const etp_tensor* tensors, int32_t n_tensors, const etp_shard* layout,
                                     int32_t n_shards, const etp_replica* replicas, int32_t n_replicas, int64_t* slots_out,
                                     void* stream) {
    if (!ctx || !tensors || n_tensors < 1 || !layout || n_replicas < 0 || (n_replicas > 0 && (!replicas || !slots_out)))
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_apply: bad arguments");
    const etp_tensor& T0 = tensors[0];
    std::vector<etp_shard> sh;
    ETP_TRY(sorted_layout(layout, n_shards, T0.total_units, &sh));
    for (int32_t t = 0; t < n_tensors; ++t) {
        const etp_tensor& T = tensors[t];
        if (!T.slabs || T.n_ranks != T0.n_ranks || T.total_units != T0.total_units || T.unit_bytes <= 0 || T.unit_bytes % 16)
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_apply: tensor %d does not belong to the class of tensor 0 (or unit_bytes not a multiple of 16)", t);
        for (int32_t r = 0; r < T.n_ranks; ++r)
            if ((T.slabs[r].base != nullptr) != (T0.slabs[r].base != nullptr) ||
                (T.slabs[r].base && (T.slabs[r].cap_units != T0.slabs[r].cap_units || T.slabs[r].anchor_unit != T0.slabs[r].anchor_unit)))
                ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_apply: tensor %d, rank %d: slab geometry differs from tensor 0 (a replica takes the same slot in every tensor)", t, r);
    }
    // free slots of every rank: not holding a unit of its current shard, not given to an earlier replica; lowest slot first
    std::vector<std::vector<char>> taken((size_t)T0.n_ranks);
    for (int32_t r = 0; r < T0.n_ranks; ++r)
        if (T0.slabs[r].base && T0.slabs[r].cap_units > 0) taken[r].assign((size_t)T0.slabs[r].cap_units, 0);
    for (const etp_shard& s : sh)
        for (int64_t u = s.begin; u < s.end; ++u) {
            int32_t r;
            int64_t slot;
            ETP_TRY(home_of(&T0, sh, u, &r, &slot));
            taken[r][(size_t)slot] = 1;
        }
    // the same (expert, rank) twice would burn a second slot for a copy no routing convention can address
    {
        std::vector<std::pair<int32_t, int32_t>> seen((size_t)n_replicas);
        for (int32_t i = 0; i < n_replicas; ++i) seen[(size_t)i] = {replicas[i].expert, replicas[i].rank};
        std::sort(seen.begin(), seen.end());
        for (int32_t i = 1; i < n_replicas; ++i)
            if (seen[(size_t)i] == seen[(size_t)i - 1])
                ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_apply: replica (expert %d, rank %d) is listed twice", seen[(size_t)i].first, seen[(size_t)i].second);
    }
    LoweredWork w;
    w.dev.resize((size_t)n_logical_devices(ctx));
    for (int32_t i = 0; i < n_replicas; ++i) {
        const int32_t e = replicas[i].expert, d = replicas[i].rank;
        if (e < 0 || e >= T0.total_units || d < 0 || d >= T0.n_ranks || taken[d].empty())
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_apply: replica %d: expert %d / rank %d out of range", i, e, d);
        int32_t hr;
        int64_t hslot;
        ETP_TRY(home_of(&T0, sh, e, &hr, &hslot));
        if (hr == d) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_apply: replica %d: rank %d already holds expert %d", i, d, e);
        int64_t slot = -1;
        for (size_t s = 0; s < taken[d].size(); ++s)
            if (!taken[d][s]) { slot = (int64_t)s; break; }
        if (slot < 0) ETP_FAIL(ETP_ERR_CAPACITY, "etp_eplb_apply: replica %d: rank %d has no spare slot", i, d);
        taken[d][(size_t)slot] = 1;
        slots_out[i] = slot;
        const int dv = device_of_rank(ctx, d);
        if (dv < 0) continue;   // another process materialises it
        DeviceWork& W = w.dev[(size_t)dv];
        if (W.phases.empty()) W.phases.resize(1);
        for (int32_t t = 0; t < n_tensors; ++t) {
            const etp_tensor& T = tensors[t];
            push_contiguous(ctx, &W.phases[0], (const char*)T.slabs[hr].base + hslot * T.unit_bytes, (char*)T.slabs[d].base + slot * T.unit_bytes, T.unit_bytes);
            w.rep.d2d_bytes += T.unit_bytes;
            W.rep.d2d_bytes += T.unit_bytes;
        }
    }
    w.rep.n_phases = 1;
    return execute(ctx, &w, stream, stream, nullptr);
}

#ifdef ETP_MOE_TIMING
extern "C" void etp_moe_timing_dump(unsigned long long* out, int reset) {
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(out, g_moe_t, sizeof(unsigned long long) * 128 * 8);
    if (reset) {
        static unsigned long long z[128 * 8];
        cudaMemcpyToSymbol(g_moe_t, z, sizeof(z));
    }
}
#endif

namespace etp {
cudaError_t install_wait_fault_moe(unsigned long long* rec) { return wait_fault_install(rec); }
}  // namespace etp

// Kernel (c), tensor-bound regime (> 64 tokens): unequal-width column/row-parallel shard linear on the 5th-gen tensor cores
// (tcgen05 + TMEM, fed by TMA).  PAPER.md:45 ("unequal-width partitioning ... for attention and linear layers"), :92-94 (shard
// widths floor/ceil of S/g_t).  The weight-streaming regime (<= 64 tokens) lives in etp_linear_group.cu.
//
//   Y[tokens][out] = X[tokens][in] . W^T        fp32 accumulation, one round-to-nearest-even cast to 16 bit (G2)
//
// computed on the weight exactly as it sits in the simulated ranks' slabs after a reshard (slot-addressed, L3):
//   ETP_COL_PARALLEL  W is cut along out-features, stored [out][in]; a rank's shard is <= 2 contiguous row runs.
//   ETP_ROW_PARALLEL  W is cut along in-features, stored transposed [in][out]; the rank partial sums are accumulated in
//                     ONE TMEM accumulator by walking the K loop over the ranks' runs in ascending unit order.
//
// Mapping onto the MMA (the roles of the operands are swapped so the wide weight dimension fills the 128 MMA rows):
//   D[m = out feature (128 TMEM lanes)][n = token (256 fp32 columns)] += A[m][k] . B[n][k]
//   A = weight tile: K-major for column-parallel (rows of W), MN-major for row-parallel (rows of W^T are K, out is contiguous)
//   B = X tile [256 tokens][64 k], always K-major.
// Ragged shard edges never need a special path: every run has its own TMA tensor map, so rows past the end of a run are
// zero-filled by the TMA unit (out-of-bounds fill) and the epilogue masks them.
//
// CTA = 6 warps: warp 0 TMA producer, warp 1 MMA issuer (+ TMEM allocation), warps 2-5 epilogue (tcgen05.ld -> 16-bit stores).
// Persistent grid, static round-robin over (m tile, token tile) items; two TMEM accumulator stages so the epilogue of item i
// overlaps the MMAs of item i+1.  CTA pairs (cta_group::2) are the default above 64 tokens (second kernel below).

#include <algorithm>
#include <cstring>
#include <vector>

#define ETP_WAIT_TU 2
#include "etp_linear.cuh"

using namespace etp;
using namespace etp::tc;
using namespace etp::lin;

namespace {

struct alignas(64) LinearParams {
    CUtensorMap map_x;
    CUtensorMap map_w[kMaxLinRuns];
    Run runs[kMaxLinRuns];
    int32_t n_runs, mode, dtype;
    int32_t tokens, in_features, out_features;
    int32_t n_m_tiles, n_n_tiles, n_chunks, pad0;   // n_chunks: K chunks of kBK per output tile
    void* y;
    float* partials;          // CTA-pair tail split: fp32 partial tiles [(tail item * 2 + CTA rank) * tail_splits + split][256][128]
    unsigned int* tickets;    // ... one arrival ticket per (tail item, CTA rank), zero between launches
    int32_t tail_first, tail_splits;   // CTA-pair kernel: items >= tail_first (the grid's last, partial round) are cut into
                                       // tail_splits K ranges, one per CTA pair (0 / 1 = no split)
};

template <int BN>
struct Cfg {
    static constexpr int kBBytes = BN * kBK * 2;
    static constexpr int kStageBytes = kABytes + kBBytes;
    static constexpr int kStages = (kSmemBudget / kStageBytes) > 12 ? 12 : (kSmemBudget / kStageBytes);
    static constexpr int kTmemCols = (2 * BN) < 32 ? 32 : 2 * BN;   // two accumulator stages; a power of two >= 32
    static constexpr int kSmemBytes = kStages * kStageBytes + 1024 /* alignment slack */ + 256 /* barriers */ + kStageTileBytes /* epilogue transpose */;
};

struct Item {
    int m, n, c0, c1;
};
__device__ __forceinline__ Item decode_item(const LinearParams& p, int item) {
    Item it;
    it.n = item % p.n_n_tiles;
    it.m = item / p.n_n_tiles;
    it.c0 = 0;
    it.c1 = p.n_chunks;
    return it;
}
__device__ __forceinline__ int find_run(const LinearParams& p, int key) {   // last run with first <= key
    int r = 0;
    while (r + 1 < p.n_runs && p.runs[r + 1].first <= key) ++r;
    return r;
}
// ------------------------------------------------------------------------------------------------ the kernel
template <int BN, typename OutT>
__global__ void __launch_bounds__(kLinThreads, 1) etp_shard_linear_kernel(const __grid_constant__ LinearParams p) {
    using C = Cfg<BN>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // 128B swizzle atoms need 1024-B alignment
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + C::kStages * C::kStageBytes);
    uint64_t* empty_bar = full_bar + C::kStages;
    uint64_t* tmem_full = empty_bar + C::kStages;
    uint64_t* tmem_empty = tmem_full + 2;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(tmem_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_items = p.n_m_tiles * p.n_n_tiles;
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
            mbar_init(&tmem_empty[s], 4);   // one arrival per epilogue warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {   // whole warp: allocate the TMEM columns of the two accumulator stages
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_ptr)), "r"(uint32_t(C::kTmemCols))
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    if (warp == 0) {
        // ===================================================================== TMA producer (one elected lane)
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
                const Item it = decode_item(p, item);
                const int t0 = it.n * BN;
                int r = row_par ? 0 : find_run(p, it.m);
                const int row = row_par ? 0 : (it.m - p.runs[r].first) * kBM;
                for (int c = it.c0; c < it.c1; ++c) {
                    uint8_t* sa = smem + stage * C::kStageBytes;
                    uint8_t* sb = sa + kABytes;
                    mbar_wait(&empty_bar[stage], phase ^ 1);
                    mbar_expect_tx(&full_bar[stage], C::kStageBytes);
                    if (!row_par) {
                        tma_load_2d(sa, &p.map_w[r], &full_bar[stage], c * kBK, row);
                        tma_load_2d(sb, &p.map_x, &full_bar[stage], c * kBK, t0);
                    } else {
                        while (r + 1 < p.n_runs && p.runs[r + 1].first <= c) ++r;
                        // K chunks are aligned to multiples of 64 GLOBAL in-features (TMA needs 16-byte aligned box starts in X);
                        // a chunk that straddles two runs is issued once per run, the rows outside the run (negative or past
                        // its end) being zero-filled by TMA.
                        const int feat0 = int(p.runs[r].feat0);
                        const int xk = (feat0 / kBK + (c - p.runs[r].first)) * kBK;
                        const int kin = xk - feat0;
                        tma_load_2d(sa, &p.map_w[r], &full_bar[stage], it.m * kBM, kin);              // out features m0 .. m0+63
                        tma_load_2d(sa + kABytes / 2, &p.map_w[r], &full_bar[stage], it.m * kBM + 64, kin);   // m0+64 .. m0+127
                        tma_load_2d(sb, &p.map_x, &full_bar[stage], xk, t0);
                    }
                    if (++stage == C::kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        // ===================================================================== MMA issuer (one elected lane)
        if (lane == 0) {
            const bool a_mn = row_par;
            const uint32_t idesc = make_idesc(p.dtype == ETP_BF16 ? 1u : 0u, a_mn ? 1u : 0u, uint32_t(BN));
            // A, K-major  : rows of 128 B, 8-row groups 1024 B apart (SBO); LBO unused with 128B swizzle; +32 B per UMMA_K.
            // A, MN-major : k rows of 128 B (64 out features), 8-k groups 1024 B apart (SBO), the second 64 out features
            //               8192 B further (LBO); +16 k rows = 2048 B per UMMA_K.
            const uint32_t a_lbo = a_mn ? uint32_t(kABytes / 2) : 16u;
            const uint32_t a_kstep = a_mn ? (uint32_t(kUmmaK) * 128u) >> 4 : (uint32_t(kUmmaK) * 2u) >> 4;
            int stage = 0;
            uint32_t phase = 0;
            int local = 0;
            for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++local) {
                const Item it = decode_item(p, item);
                const int as = local & 1;
                const uint32_t aph = (local >> 1) & 1;
                mbar_wait(&tmem_empty[as], aph ^ 1);   // the epilogue has drained this accumulator stage
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + uint32_t(as * BN);
                for (int c = it.c0; c < it.c1; ++c) {
                    uint8_t* sa = smem + stage * C::kStageBytes;
                    mbar_wait(&full_bar[stage], phase);
                    tc_fence_after();
                    const uint64_t a_desc = make_smem_desc(smem_u32(sa), a_lbo, 1024);
                    const uint64_t b_desc = make_smem_desc(smem_u32(sa + kABytes), 16, 1024);
#pragma unroll
                    for (int k = 0; k < kBK / kUmmaK; ++k)
                        tc_mma(d_tmem, a_desc + uint64_t(k) * a_kstep, b_desc + uint64_t(k) * 2u, idesc, (c > it.c0 || k > 0) ? 1u : 0u);
                    tc_commit(&empty_bar[stage]);   // frees the smem stage once these MMAs have read it
                    if (++stage == C::kStages) { stage = 0; phase ^= 1; }
                }
                tc_commit(&tmem_full[as]);          // accumulator complete -> epilogue
            }
        }
        __syncwarp();
    } else {
        // ===================================================================== epilogue warps 2..5
        const int q = warp & 3;                 // a warp may only touch TMEM lanes 32*(warp % 4) .. +31
        const int m_local = q * 32 + lane;
        OutT* y = reinterpret_cast<OutT*>(p.y);
        int64_t outf = p.out_features;          // column-parallel: per run (a fused launch carries several linears)
        OutT* stage_t = reinterpret_cast<OutT*>(smem + C::kStages * C::kStageBytes + 256);
        bool vec_out = (p.out_features & 7) == 0;     // 16-byte epilogue stores need 16-byte aligned Y rows
        int local = 0;
        for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++local) {
            const Item it = decode_item(p, item);
            const int as = local & 1;
            const uint32_t aph = (local >> 1) & 1;
            const int t0 = it.n * BN;
            const int n_tok = min(BN, p.tokens - t0);
            int64_t gm0;
            int valid;
            if (!row_par) {
                const int r = find_run(p, it.m);
                const int row = (it.m - p.runs[r].first) * kBM;
                gm0 = p.runs[r].feat0 + row;
                valid = min(kBM, p.runs[r].n_feat - row);
                y = reinterpret_cast<OutT*>(p.runs[r].y);
                outf = p.runs[r].out_features;
                vec_out = (outf & 7) == 0;
            } else {
                gm0 = int64_t(it.m) * kBM;
                valid = min(kBM, int(outf) - it.m * kBM);
            }
            mbar_wait(&tmem_full[as], aph);
            tc_fence_after();
            const uint32_t taddr = tmem_base + uint32_t(as * BN) + (uint32_t(q * 32) << 16);
            for (int c16 = 0; c16 < n_tok; c16 += 16) {
                uint32_t v[16];
                tc_ld16(taddr + uint32_t(c16), v);
                tc_ld_wait();
                if (vec_out) {
                    store_block16(stage_t, v, m_local, y, size_t(t0 + c16), min(16, n_tok - c16), outf, gm0, valid);
                } else if (m_local < valid) {
#pragma unroll
                    for (int j = 0; j < 16; ++j)
                        if (c16 + j < n_tok) y[size_t(t0 + c16 + j) * outf + gm0 + m_local] = cvt16<OutT>(__uint_as_float(v[j]));
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
// Large token counts (BN = 256): two CTAs of a cluster (one TPC) run ONE tcgen05.mma.cta_group::2 of M = 256 out features x
// N = 256 tokens.  CTA rank c owns out-feature tile 2*pair + c (its own A tile and its own 128 TMEM lanes x 256 columns)
// and stages HALF of the X tile (tokens t0 + 128*c ..), so every SM reads 16 + 16 KiB of shared memory per K chunk
// instead of 16 + 32 KiB.  Only the leader (rank 0) issues MMAs; both CTAs issue TMA loads that complete on the
// LEADER's full barrier; tcgen05.commit multicasts the "stage free" and "accumulator ready" arrivals to both CTAs; the
// epilogue warps of both CTAs arrive on the leader's "accumulator drained" barrier.
// PBN = tokens per pair tile (UMMA_N): 256, or 128 when that fills the 74 CTA pairs more evenly (host heuristic).
template <int PBN>
struct PairCfg {
    static constexpr int kBBytes = (PBN / 2) * kBK * 2;   // this CTA's half of the X tile
    static constexpr int kStageBytes = kABytes + kBBytes;
    static constexpr int kStages = kSmemBudget / kStageBytes > 8 ? 8 : kSmemBudget / kStageBytes;
    static constexpr int kTmemCols = 2 * PBN;             // two accumulator stages of PBN fp32 columns
    static constexpr int kSmemBytes = kStages * kStageBytes + 1024 + 256 + kStageTileBytes;
};

// The k-th piece of work of a CTA pair.  Full rounds: item = cluster + k * n_clusters over all K chunks.  Then, if the last round
// is partial (tail_splits > 1), ONE K range [c0, c1) of a tail item, so that round costs ~1/tail_splits of a full one; its fp32
// partial tile goes through the split-K workspace and the last pair to arrive sums the ranges in order 0..S-1 (deterministic).
struct PairWork {
    int item, c0, c1, split;   // split < 0: the whole K range, written straight to Y
};
__device__ __forceinline__ bool pair_work(const LinearParams& p, int cluster_id, int n_clusters, int k, PairWork* w) {
    const int n_items = p.n_m_tiles * p.n_n_tiles;
    const int full = p.tail_splits > 1 ? p.tail_first : n_items;
    const int item = cluster_id + k * n_clusters;
    if (item < full) {
        *w = {item, 0, p.n_chunks, -1};
        return true;
    }
    if (p.tail_splits > 1 && k == full / n_clusters && cluster_id < (n_items - full) * p.tail_splits) {
        const int split = cluster_id % p.tail_splits;
        *w = {full + cluster_id / p.tail_splits, int(int64_t(split) * p.n_chunks / p.tail_splits),
              int(int64_t(split + 1) * p.n_chunks / p.tail_splits), split};
        return true;
    }
    return false;
}

// Items are (pair of m tiles, token tile); p.n_m_tiles counts PAIRS and runs[].first indexes pairs (column-parallel).
template <int PBN, typename OutT>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kLinThreads, 1) etp_shard_linear_pair_kernel(const __grid_constant__ LinearParams p) {
    constexpr int kPairBN = PBN, kPairStages = PairCfg<PBN>::kStages, kPairStageBytes = PairCfg<PBN>::kStageBytes;
    constexpr int kPairTmemCols = PairCfg<PBN>::kTmemCols;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + kPairStages * kPairStageBytes);
    uint64_t* empty_bar = full_bar + kPairStages;
    uint64_t* tmem_full = empty_bar + kPairStages;
    uint64_t* tmem_empty = tmem_full + 2;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(tmem_empty + 2);
    uint32_t* last_flag = tmem_ptr + 1;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int cluster_id = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;
    const bool row_par = p.mode == ETP_ROW_PARALLEL;

    if (warp == 0 && lane == 1) {
        prefetch_tensormap(&p.map_x);
        for (int r = 0; r < p.n_runs; ++r) prefetch_tensormap(&p.map_w[r]);
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < kPairStages; ++s) {
            mbar_init(&full_bar[s], 1);      // used in the leader only: its own arrive.expect_tx of both CTAs' bytes
            mbar_init(&empty_bar[s], 1);     // one multicast commit per use
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&tmem_full[s], 1);     // one multicast commit per item
            mbar_init(&tmem_empty[s], 8);    // leader only: 4 epilogue warps of each CTA
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {   // one warp of EACH CTA, same warp id, same destination offset
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_ptr)), "r"(uint32_t(kPairTmemCols))
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();      // the peer's barriers exist before anything signals them
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    if (warp == 0) {
        // ===================================================================== TMA producer (one lane of each CTA)
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            PairWork w;
            for (int kk = 0; pair_work(p, cluster_id, n_clusters, kk, &w); ++kk) {
                const int pn = w.item % p.n_n_tiles, pm = w.item / p.n_n_tiles;
                const int t0 = pn * kPairBN + int(rank) * (kPairBN / 2);
                int r = row_par ? 0 : find_run(p, pm);
                const int row = row_par ? 0 : ((pm - p.runs[r].first) * 2 + int(rank)) * kBM;   // may lie past the run: zero-filled
                const int m0 = (pm * 2 + int(rank)) * kBM;                                      // row-parallel: out features
                for (int c = w.c0; c < w.c1; ++c) {
                    uint8_t* sa = smem + stage * kPairStageBytes;
                    uint8_t* sb = sa + kABytes;
                    mbar_wait(&empty_bar[stage], phase ^ 1);
                    const uint32_t lbar = mapa_rank0(smem_u32(&full_bar[stage]));
                    if (rank == 0) mbar_expect_tx(&full_bar[stage], 2 * kPairStageBytes);
                    if (!row_par) {
                        tma_load_2d_pair(sa, &p.map_w[r], lbar, c * kBK, row);
                        tma_load_2d_pair(sb, &p.map_x, lbar, c * kBK, t0);
                    } else {
                        while (r + 1 < p.n_runs && p.runs[r + 1].first <= c) ++r;
                        const int feat0 = int(p.runs[r].feat0);
                        const int xk = (feat0 / kBK + (c - p.runs[r].first)) * kBK;
                        const int kin = xk - feat0;
                        tma_load_2d_pair(sa, &p.map_w[r], lbar, m0, kin);
                        tma_load_2d_pair(sa + kABytes / 2, &p.map_w[r], lbar, m0 + 64, kin);
                        tma_load_2d_pair(sb, &p.map_x, lbar, xk, t0);
                    }
                    if (++stage == kPairStages) { stage = 0; phase ^= 1; }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        // ===================================================================== MMA issuer (one lane of the LEADER)
        if (lane == 0 && rank == 0) {
            const bool a_mn = row_par;
            const uint32_t idesc = make_idesc_pair(p.dtype == ETP_BF16 ? 1u : 0u, a_mn ? 1u : 0u, uint32_t(kPairBN));
            const uint32_t a_lbo = a_mn ? uint32_t(kABytes / 2) : 16u;
            const uint32_t a_kstep = a_mn ? (uint32_t(kUmmaK) * 128u) >> 4 : (uint32_t(kUmmaK) * 2u) >> 4;
            int stage = 0;
            uint32_t phase = 0;
            int local = 0;
            PairWork w;
            for (; pair_work(p, cluster_id, n_clusters, local, &w); ++local) {
                const int as = local & 1;
                const uint32_t aph = (local >> 1) & 1;
                mbar_wait(&tmem_empty[as], aph ^ 1);   // both CTAs' epilogues have drained this accumulator stage
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + uint32_t(as * kPairBN);
                for (int c = w.c0; c < w.c1; ++c) {
                    uint8_t* sa = smem + stage * kPairStageBytes;
                    mbar_wait(&full_bar[stage], phase);
                    tc_fence_after();
                    const uint64_t a_desc = make_smem_desc(smem_u32(sa), a_lbo, 1024);
                    const uint64_t b_desc = make_smem_desc(smem_u32(sa + kABytes), 16, 1024);
#pragma unroll
                    for (int k = 0; k < kBK / kUmmaK; ++k)
                        tc_mma_pair(d_tmem, a_desc + uint64_t(k) * a_kstep, b_desc + uint64_t(k) * 2u, idesc, (c > w.c0 || k > 0) ? 1u : 0u);
                    tc_commit_pair(&empty_bar[stage]);   // frees the stage in BOTH CTAs once these MMAs have read it
                    if (++stage == kPairStages) { stage = 0; phase ^= 1; }
                }
                tc_commit_pair(&tmem_full[as]);
            }
        }
        __syncwarp();
    } else {
        // ===================================================================== epilogue warps 2..5 of both CTAs
        const int q = warp & 3;
        const int m_local = q * 32 + lane;
        OutT* y = reinterpret_cast<OutT*>(p.y);
        int64_t outf = p.out_features;          // column-parallel: per run (a fused launch carries several linears)
        const uint32_t drained = mapa_rank0(smem_u32(&tmem_empty[0]));
        OutT* stage_t = reinterpret_cast<OutT*>(smem + kPairStages * kPairStageBytes + 256);
        bool vec_out = (p.out_features & 7) == 0;
        int local = 0;
        PairWork w;
        for (; pair_work(p, cluster_id, n_clusters, local, &w); ++local) {
            const int pn = w.item % p.n_n_tiles, pm = w.item / p.n_n_tiles;
            const int as = local & 1;
            const uint32_t aph = (local >> 1) & 1;
            const int t0 = pn * kPairBN;
            const int n_tok = min(kPairBN, p.tokens - t0);
            int64_t gm0;
            int valid;
            if (!row_par) {
                const int r = find_run(p, pm);
                const int row = ((pm - p.runs[r].first) * 2 + int(rank)) * kBM;
                gm0 = p.runs[r].feat0 + row;
                valid = min(kBM, p.runs[r].n_feat - row);
                y = reinterpret_cast<OutT*>(p.runs[r].y);
                outf = p.runs[r].out_features;
                vec_out = (outf & 7) == 0;
            } else {
                gm0 = int64_t(pm * 2 + int(rank)) * kBM;
                valid = int(min(int64_t(kBM), outf - gm0));
            }
            mbar_wait(&tmem_full[as], aph);
            tc_fence_after();
            const uint32_t taddr = tmem_base + uint32_t(as * kPairBN) + (uint32_t(q * 32) << 16);
            for (int c16 = 0; c16 < n_tok; c16 += 16) {
                uint32_t v[16];
                tc_ld16(taddr + uint32_t(c16), v);
                tc_ld_wait();
                if (w.split >= 0) {
                    float* ws = p.partials + ((size_t(w.item - p.tail_first) * 2 + rank) * p.tail_splits + w.split) * size_t(kPairBN) * kBM;
#pragma unroll
                    for (int j = 0; j < 16; ++j)
                        if (c16 + j < n_tok) ws[(c16 + j) * kBM + m_local] = __uint_as_float(v[j]);
                } else if (vec_out) {
                    store_block16(stage_t, v, m_local, y, size_t(t0 + c16), min(16, n_tok - c16), outf, gm0, valid);
                } else if (m_local < valid) {
#pragma unroll
                    for (int j = 0; j < 16; ++j)
                        if (c16 + j < n_tok) y[size_t(t0 + c16 + j) * outf + gm0 + m_local] = cvt16<OutT>(__uint_as_float(v[j]));
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(drained + uint32_t(as) * 8u);
            if (w.split >= 0) {
                // the last of the tail_splits pairs to arrive at this (tile, CTA rank) sums the partials in range order
                unsigned int* ticket = p.tickets + (w.item - p.tail_first) * 2 + rank;
                __threadfence();
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (threadIdx.x == 64) *last_flag = (atomicAdd(ticket, 1u) == uint32_t(p.tail_splits - 1)) ? 1u : 0u;
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (*last_flag) {
                    __threadfence();
                    const float* w0 = p.partials + (size_t(w.item - p.tail_first) * 2 + rank) * p.tail_splits * size_t(kPairBN) * kBM;
                    // 32 threads x float4 cover the 128 features of one token, the four warps take tokens j, j+1, j+2, j+3; eight
                    // tokens per thread in flight.  Row-parallel only: gm0 is a multiple of 128 and out_features of 8, so the
                    // four 16-bit results of a thread are one aligned 8-byte store and `valid` is a multiple of 8.
                    const int col4 = lane * 4;
                    for (int j0 = q; j0 < n_tok; j0 += 32) {
                        float4 acc[8];
#pragma unroll
                        for (int u = 0; u < 8; ++u) acc[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                        for (int sp = 0; sp < p.tail_splits; ++sp) {
#pragma unroll
                            for (int u = 0; u < 8; ++u) {
                                const int j = j0 + 4 * u;
                                if (j < n_tok) {
                                    const float4 t = __ldcg(reinterpret_cast<const float4*>(w0 + (size_t(sp) * kPairBN + j) * kBM + col4));
                                    acc[u].x += t.x; acc[u].y += t.y; acc[u].z += t.z; acc[u].w += t.w;
                                }
                            }
                        }
#pragma unroll
                        for (int u = 0; u < 8; ++u) {
                            const int j = j0 + 4 * u;
                            if (j < n_tok && col4 < valid) {
                                OutT o[4] = {cvt16<OutT>(acc[u].x), cvt16<OutT>(acc[u].y), cvt16<OutT>(acc[u].z), cvt16<OutT>(acc[u].w)};
                                *reinterpret_cast<uint2*>(y + size_t(t0 + j) * outf + gm0 + col4) = *reinterpret_cast<const uint2*>(o);
                            }
                        }
                    }
                    if (threadIdx.x == 64) *ticket = 0;
                }
                asm volatile("bar.sync 1, 128;" ::: "memory");
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    cluster_sync_all();      // the leader's MMAs read the peer's shared memory and both CTAs free the paired TMEM
    if (warp == 1) {
        __syncwarp();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(uint32_t(kPairTmemCols)) : "memory");
    }
}

// ------------------------------------------------------------------------------------------------ host side
template <int BN>
etp_status launch_linear(const LinearParams& p, int grid, cudaStream_t stream) {
    using C = Cfg<BN>;
    static bool configured[2] = {false, false};   // the attribute belongs to the function: set once per process
    if (p.dtype == ETP_BF16) {
        auto k = etp_shard_linear_kernel<BN, __nv_bfloat16>;
        if (!configured[0]) { ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes)); configured[0] = true; }
        k<<<grid, kLinThreads, C::kSmemBytes, stream>>>(p);
    } else {
        auto k = etp_shard_linear_kernel<BN, __half>;
        if (!configured[1]) { ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes)); configured[1] = true; }
        k<<<grid, kLinThreads, C::kSmemBytes, stream>>>(p);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) ETP_FAIL(ETP_ERR_CUDA, "etp_shard_linear: launch failed: %s", cudaGetErrorString(e));
    return ETP_OK;
}

template <int PBN>
etp_status launch_linear_pair(const LinearParams& p, int grid, cudaStream_t stream) {
    constexpr int kPairSmemBytes = PairCfg<PBN>::kSmemBytes;
    static bool configured[2] = {false, false};
    if (p.dtype == ETP_BF16) {
        auto k = etp_shard_linear_pair_kernel<PBN, __nv_bfloat16>;
        if (!configured[0]) { ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, kPairSmemBytes)); configured[0] = true; }
        k<<<grid, kLinThreads, kPairSmemBytes, stream>>>(p);
    } else {
        auto k = etp_shard_linear_pair_kernel<PBN, __half>;
        if (!configured[1]) { ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, kPairSmemBytes)); configured[1] = true; }
        k<<<grid, kLinThreads, kPairSmemBytes, stream>>>(p);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) ETP_FAIL(ETP_ERR_CUDA, "etp_shard_linear: pair launch failed: %s", cudaGetErrorString(e));
    return ETP_OK;
}

}  // namespace

namespace etp {
namespace lin {

etp_status check_linear_shape(etp_linear_mode mode, int64_t in_features, int64_t out_features, int64_t features_per_unit,
                              const etp_tensor* w) {
    if (in_features <= 0 || out_features <= 0 || features_per_unit <= 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: non-positive size");
    if (in_features >= (int64_t(1) << 31) || out_features >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: sizes must be below 2^31");
    const bool row_par = mode == ETP_ROW_PARALLEL;
    const int64_t sharded = row_par ? in_features : out_features;   // the dimension the weight is cut along
    const int64_t row_len = row_par ? out_features : in_features;   // contiguous elements per feature row of the stored weight
    if (w->total_units * features_per_unit != sharded)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: total_units %lld x features_per_unit %lld != sharded dimension %lld",
                 (long long)w->total_units, (long long)features_per_unit, (long long)sharded);
    if (w->unit_bytes != features_per_unit * row_len * 2)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: unit_bytes %lld != features_per_unit x row length x 2 = %lld",
                 (long long)w->unit_bytes, (long long)(features_per_unit * row_len * 2));
    if ((in_features * 2) % 16 || (row_len * 2) % 16)
        ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_shard_linear: row pitches must be multiples of 16 bytes (in %lld, stored row %lld elements)",
                 (long long)in_features, (long long)row_len);
    return ETP_OK;
}

// the shards in ascending unit order must tile [0, total_units)
etp_status check_layout(const etp_shard* layout, int32_t n_shards, int64_t total_units, std::vector<etp_shard>* sh) {
    sh->clear();
    if (!layout || n_shards <= 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: empty layout");
    for (int i = 0; i < n_shards; ++i)
        if (layout[i].alive && layout[i].end > layout[i].begin) sh->push_back(layout[i]);
    std::sort(sh->begin(), sh->end(), [](const etp_shard& a, const etp_shard& b) { return a.begin < b.begin; });
    int64_t cursor = 0;
    for (const etp_shard& s : *sh) {
        if (s.begin != cursor) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: layout does not tile [0,%lld): gap or overlap at unit %lld", (long long)total_units, (long long)cursor);
        cursor = s.end;
    }
    if (cursor != total_units) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: layout covers %lld of %lld units", (long long)cursor, (long long)total_units);
    return ETP_OK;
}

// contiguous runs of every shard inside its slot-addressed slab (L3), appended in ascending unit order
etp_status append_runs(const etp_tensor* w, const std::vector<etp_shard>& sh, int64_t features_per_unit, void* y, int64_t out_features,
                       RunList* out) {
    for (const etp_shard& s : sh) {
        if (s.rank < 0 || s.rank >= w->n_ranks) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: rank %d outside the tensor's %d slabs", s.rank, w->n_ranks);
        const etp_slab& sl = w->slabs[s.rank];
        if (!sl.base) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: rank %d has no slab", s.rank);
        if (reinterpret_cast<uintptr_t>(sl.base) & 15) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_shard_linear: slab of rank %d not 16-byte aligned", s.rank);
        const int64_t width = s.end - s.begin;
        if (sl.cap_units <= 0 || width > sl.cap_units) ETP_FAIL(ETP_ERR_CAPACITY, "etp_shard_linear: shard of rank %d (%lld units) exceeds its slab (%lld)", s.rank, (long long)width, (long long)sl.cap_units);
        int64_t slot0 = (s.begin - sl.anchor_unit) % sl.cap_units;
        if (slot0 < 0) slot0 += sl.cap_units;
        const int64_t len1 = std::min(width, sl.cap_units - slot0);
        const int64_t piece_b[2] = {s.begin, s.begin + len1};
        const int64_t piece_n[2] = {len1, width - len1};
        const int64_t piece_slot[2] = {slot0, 0};
        for (int k = 0; k < 2; ++k) {
            if (piece_n[k] == 0) continue;
            if (out->n == kMaxLinRuns) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_shard_linear: more than %d contiguous runs", kMaxLinRuns);
            if (piece_n[k] * features_per_unit >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: run too long");
            Run& R = out->runs[out->n];
            R.feat0 = piece_b[k] * features_per_unit;
            R.n_feat = int32_t(piece_n[k] * features_per_unit);
            R.first = 0;
            R.y = y;
            R.out_features = int32_t(out_features);
            R.pad = 0;
            out->addr[out->n] = static_cast<const char*>(sl.base) + piece_slot[k] * w->unit_bytes;
            ++out->n;
        }
    }
    return ETP_OK;
}

// > 64 tokens.  Column-parallel: n_outs >= 1 linears that share X, in_features and the shard layout of their class (q|k|v, gate|up)
// in ONE launch - the runs of all of them are concatenated and every run carries its own Y.  Row-parallel: n_outs == 1.
etp_status shard_linear_large(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x, int64_t tokens, int64_t in_features,
                              const LinOut* outs, int32_t n_outs, const etp_shard* layout, int32_t n_shards, void* stream) {
    const bool row_par = mode == ETP_ROW_PARALLEL;
    const int64_t out_features = outs[0].out_features;   // row-parallel: the one linear's width
    std::vector<etp_shard> sh;
    ETP_TRY(check_layout(layout, n_shards, outs[0].w->total_units, &sh));
    RunList rl;
    for (int32_t o = 0; o < n_outs; ++o) ETP_TRY(append_runs(outs[o].w, sh, outs[o].features_per_unit, outs[o].y, outs[o].out_features, &rl));
    LinearParams p;
    std::memset(&p, 0, sizeof(p));
    const int n_runs = rl.n;
    for (int r = 0; r < n_runs; ++r) p.runs[r] = rl.runs[r];

    // ---- tiling: CTA pairs (256 out features x 256 tokens per pair) unless single-CTA 128 x 256 tiles need fewer rounds of the
    // persistent grid (few, ragged m tiles: e.g. 1024 out features in runs of 384/384/256).  Per item a pair takes ~0.93 of the
    // single-CTA time (it stages 32 KiB instead of 48 KiB per K chunk and SM; measured on the config-2 shapes).
    constexpr int bn = 256;
    const int64_t pair_opt = ctx->opts[ETP_OPT_LINEAR_CTA_PAIR];
    bool pair = pair_opt != 0 && ctx->n_sms >= 2;
    const int pbn = pair_opt == 128 ? 128 : 256;
    if (pair && pair_opt == 1) {
        int64_t mt_single = 0, mt_pair = 0;
        if (row_par) {
            mt_single = (out_features + kBM - 1) / kBM;
            mt_pair = (out_features + 2 * kBM - 1) / (2 * kBM);
        } else {
            for (int r = 0; r < n_runs; ++r) {
                mt_single += (p.runs[r].n_feat + kBM - 1) / kBM;
                mt_pair += (p.runs[r].n_feat + 2 * kBM - 1) / (2 * kBM);
            }
        }
        const int64_t tt = (tokens + 255) / 256, units = ctx->n_sms / 2;
        const int64_t rounds_single = (mt_single * tt + ctx->n_sms - 1) / ctx->n_sms, rounds_pair = (mt_pair * tt + units - 1) / units;
        pair = double(rounds_pair) * 0.93 <= double(rounds_single);
    }
    const int m_tile = pair ? 2 * kBM : kBM;
    const int tile_n = pair ? pbn : bn;
    p.n_runs = n_runs;
    p.mode = mode;
    p.dtype = dtype;
    p.tokens = int32_t(tokens);
    p.in_features = int32_t(in_features);
    p.out_features = int32_t(out_features);
    p.n_n_tiles = int32_t((tokens + tile_n - 1) / tile_n);
    p.y = outs[0].y;
    int32_t acc = 0;
    for (int r = 0; r < n_runs; ++r) {
        p.runs[r].first = acc;
        if (row_par) acc += int32_t((p.runs[r].feat0 + p.runs[r].n_feat + kBK - 1) / kBK - p.runs[r].feat0 / kBK);   // 64-aligned global K chunks it touches
        else acc += (p.runs[r].n_feat + m_tile - 1) / m_tile;
    }
    if (row_par) {
        p.n_chunks = acc;
        p.n_m_tiles = int32_t((out_features + m_tile - 1) / m_tile);
    } else {
        p.n_m_tiles = acc;
        p.n_chunks = int32_t((in_features + kBK - 1) / kBK);
    }
    const int64_t n_items = int64_t(p.n_m_tiles) * p.n_n_tiles;
    if (n_items >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: too many work items");

    // CTA pairs, row-parallel: a partial last round of the persistent grid is cut along K over the idle pairs (row-parallel only:
    // its items depend on the nominal shapes alone, and reading G3 keeps column-parallel outputs independent of the layout)
    ETP_CUDA_OK(cudaSetDevice(ctx->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (pair && row_par && pbn == 256 && pair_opt != 256) {
        const int64_t units = ctx->n_sms / 2, tail = n_items % units;
        if (n_items > units && tail > 0) {
            const int64_t S = std::min<int64_t>({units / tail, 8, int64_t(p.n_chunks)});
            if (S >= 2) {
                p.tail_first = int32_t(n_items - tail);
                p.tail_splits = int32_t(S);
                LinWorkspace w;   // per stream: calls on different streams of one ctx never share partial tiles or tickets
                ETP_TRY(linear_workspace(ctx, st, tail * 2 * S * pbn * kBM * int64_t(sizeof(float)), tail * 2, &w));
                p.partials = w.partials;
                p.tickets = w.tickets;
            }
        }
    }

    // ---- tensor maps: X [tokens][in]; one map per run so that TMA zero-fills everything past a run's end
    ETP_TRY(encode_2d(&p.map_x, dtype, x, tokens, in_features, in_features, kBK, pair ? pbn / 2 : bn));
    for (int r = 0; r < n_runs; ++r) {
        if (row_par) ETP_TRY(encode_2d(&p.map_w[r], dtype, rl.addr[r], p.runs[r].n_feat, out_features, out_features, 64, kBK));
        else ETP_TRY(encode_2d(&p.map_w[r], dtype, rl.addr[r], p.runs[r].n_feat, in_features, in_features, kBK, kBM));
    }

    ctx->launches = 1;
    if (pair) {
        const int pgrid = 2 * int(std::min<int64_t>(n_items, ctx->n_sms / 2));
        return pbn == 128 ? launch_linear_pair<128>(p, pgrid, st) : launch_linear_pair<256>(p, pgrid, st);
    }
    return launch_linear<256>(p, int(std::min<int64_t>(n_items, ctx->n_sms)), st);
}

}  // namespace lin
}  // namespace etp

// argument checks shared by the two legacy entry points, then the regime split
static etp_status shard_linear_impl(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x, int64_t tokens,
                                    int64_t in_features, const LinOut* outs, int32_t n_outs, const etp_shard* layout,
                                    int32_t n_shards, void* stream) {
    if (!ctx || !outs || !layout || n_outs < 1) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: NULL argument");
    if (mode != ETP_COL_PARALLEL && mode != ETP_ROW_PARALLEL) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: bad mode %d", int(mode));
    if (dtype != ETP_BF16 && dtype != ETP_FP16) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_shard_linear: dtype %d is not bf16/fp16", int(dtype));
    const bool row_par = mode == ETP_ROW_PARALLEL;
    if (row_par && n_outs != 1) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_shard_linear_multi: only column-parallel linears can be fused");
    if (tokens < 0 || in_features <= 0 || n_shards <= 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: non-positive size");
    if (tokens >= (int64_t(1) << 31) || in_features >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: sizes must be below 2^31");
    for (int32_t o = 0; o < n_outs; ++o) {
        const etp_tensor* w = outs[o].w;
        if (!w || !w->slabs) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: NULL argument");
        ETP_TRY(check_linear_shape(mode, in_features, outs[o].out_features, outs[o].features_per_unit, w));
        if (w->total_units != outs[0].w->total_units)
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear_multi: fused linears must belong to one granularity class (%lld vs %lld units)",
                     (long long)w->total_units, (long long)outs[0].w->total_units);
    }
    if (tokens == 0) return ETP_OK;
    if (!x) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: x / y is NULL");
    if (reinterpret_cast<uintptr_t>(x) & 15) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_shard_linear: x / y not 16-byte aligned");
    for (int32_t o = 0; o < n_outs; ++o) {
        if (!outs[o].y) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: x / y is NULL");
        if (reinterpret_cast<uintptr_t>(outs[o].y) & 15) ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_shard_linear: x / y not 16-byte aligned");
    }
    if (tokens <= 64) return shard_linear_small(ctx, mode, dtype, x, tokens, in_features, outs, n_outs, layout, n_shards, stream);
    return shard_linear_large(ctx, mode, dtype, x, tokens, in_features, outs, n_outs, layout, n_shards, stream);
}

extern "C" etp_status etp_shard_linear(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x, int64_t tokens,
                                       int64_t in_features, int64_t out_features, const etp_tensor* w, const etp_shard* layout,
                                       int32_t n_shards, int64_t features_per_unit, void* y, void* stream) {
    const LinOut one{w, out_features, features_per_unit, y};
    return shard_linear_impl(ctx, mode, dtype, x, tokens, in_features, &one, 1, layout, n_shards, stream);
}

extern "C" etp_status etp_shard_linear_multi(etp_ctx* ctx, etp_dtype dtype, const void* x, int64_t tokens, int64_t in_features,
                                             const etp_linear_out* outs, int32_t n_outs, const etp_shard* layout, int32_t n_shards,
                                             void* stream) {
    if (!outs || n_outs < 1 || n_outs > 8) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear_multi: 1..8 linears");
    LinOut lo[8];
    for (int32_t o = 0; o < n_outs; ++o) lo[o] = {outs[o].w, outs[o].out_features, outs[o].features_per_unit, outs[o].y};
    return shard_linear_impl(ctx, ETP_COL_PARALLEL, dtype, x, tokens, in_features, lo, n_outs, layout, n_shards, stream);
}

namespace etp {
cudaError_t install_wait_fault_linear(unsigned long long* rec) { return wait_fault_install(rec); }
}  // namespace etp

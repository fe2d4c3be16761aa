// Kernel (c), weight-streaming regime (<= 64 tokens): a PREPARED GROUP of shard linears in one persistent launch.
// PAPER.md:45, :92-94 (unequal-width sharding of attention and linear layers); DESIGN.md 5.3.
//
// At a handful of tokens a linear is a pure weight stream: 2 K N bytes of HBM traffic and almost no arithmetic.  What kept the
// per-linear launches of round 1 at 0.57 (0.71 fused) of the HBM peak was not traffic (ncu: 1.02 x algorithmic) but fixed cost:
// a launch needs ~6.5 us before its first byte arrives (TMEM allocation, barrier init, tensor-map fetch, first TMA round trip),
// a 10-MB projection therefore runs at 0.11 of peak, and the split-K tail of a static round-robin grid left SMs idle.  Here:
//   * etp_linear_prepare() does everything that depends only on the weights once: layout check, slot runs, one TMA tensor map
//     per run, the K split of every linear and a LOAD-BALANCED assignment of (linear, m tile, K range) items to the 148 CTAs
//     (longest-processing-time-first on the number of 16-KiB weight chunks per item), uploaded as a device table the plan owns.
//   * etp_linear_run() encodes at most the X maps (cached per (pointer, tokens)) and launches ONE kernel for the whole group:
//     column- and row-parallel linears mix freely (the instruction descriptor, the smem descriptors and the TMA boxes are
//     chosen per item), each linear has its own X and Y.
//   * launches carry the programmatic-stream-serialization attribute: the kernel signals griddepcontrol.launch_dependents
//     right after its prologue and executes griddepcontrol.wait only before it first touches X, Y or the split-K workspace,
//     so the prologue AND the first ring of weight tiles of launch i+1 overlap the tail of launch i (weights are not produced
//     by the previous kernel; X may be).
// Same tcgen05 / TMEM / TMA data path as the large-token kernels: D[m = out feature][n = token] in TMEM, 128 x BN tiles (BN = 16
// or 64 tokens), BLOCK_K = 64, 128B swizzle, warp 0 TMA producer, warp 1 MMA issuer, warps 2-5 epilogue, two accumulator stages.
// Split-K partials are fp32 tiles in a per-stream workspace; the last split to arrive at a tile sums them in split order.
#include <algorithm>
#include <cstring>
#include <memory>
#include <queue>
#include <string>
#include <unordered_map>
#include <vector>

#define ETP_WAIT_TU 3
#include "etp_linear.cuh"

using namespace etp;
using namespace etp::tc;
using namespace etp::lin;

namespace {

struct GroupItem {   // 16 bytes: K chunks [c0, c1) of m tile `m` of linear `lin`, split index `split`
    int16_t lin, split;
    int32_t m, c0, c1;
};
static_assert(sizeof(GroupItem) == 16, "GroupItem layout");

struct GroupLin {
    int32_t mode, run0, n_runs, out_features;
    int32_t n_chunks, n_splits, tile0, pad;   // tile0: first output tile of this linear in the group's ticket numbering
    int64_t ws0;                              // index of its first fp32 partial tile in the workspace
    void* y;                                  // row-parallel output (column-parallel: per run)
};

constexpr int kMaxGroupRuns = 64;   // contiguous slot runs of a whole group (8 KiB of tensor maps in the kernel parameters)

struct alignas(64) GroupParams {
    CUtensorMap map_x[kMaxGroupLins];
    CUtensorMap map_w[kMaxGroupRuns];
    Run runs[kMaxGroupRuns];
    GroupLin lin[kMaxGroupLins];
    const GroupItem* items;     // CTA-major item lists
    const int32_t* cta_first;   // [grid + 1]
    float* partials;            // [partial tile][BN][128]
    unsigned int* tickets;      // one per output tile, zero between launches
    int32_t n_lins, tokens, dtype, pad;
};

constexpr int kMaxCtaItems = 96;   // items of one CTA staged in shared memory

// HALF = false: one CTA per SM with a deep ring (10 / 8 stages of 18 / 24 KiB).  HALF = true: half the ring (5 / 4 stages,
// < 100 KiB) and TWO CTAs per SM (grid = 2 x SMs), see etp_linear_prepare.
template <int BN, bool HALF>
struct GCfg {
    static constexpr int kBBytes = BN * kBK * 2;
    static constexpr int kStageBytes = kABytes + kBBytes;
    static constexpr int kFull = (kSmemBudget / kStageBytes) > 10 ? 10 : (kSmemBudget / kStageBytes);
    static constexpr int kStages = HALF ? kFull / 2 : kFull;
    static constexpr int kMinCtas = HALF ? 2 : 1;
    static constexpr int kTmemCols = (2 * BN) < 32 ? 32 : 2 * BN;
    static constexpr int kSmemBytes = kStages * kStageBytes + 1024 + 256 + kStageTileBytes + kMaxCtaItems * int(sizeof(GroupItem));
};

__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ int find_run_in(const GroupParams& p, const GroupLin& L, int key) {   // last run of L with first <= key
    int r = L.run0;
    const int end = L.run0 + L.n_runs;
    while (r + 1 < end && p.runs[r + 1].first <= key) ++r;
    return r;
}

template <int BN, typename OutT, bool HALF>
__global__ void __launch_bounds__(kLinThreads, GCfg<BN, HALF>::kMinCtas) etp_linear_group_kernel(const __grid_constant__ GroupParams p) {
    using C = GCfg<BN, HALF>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + C::kStages * C::kStageBytes);
    uint64_t* empty_bar = full_bar + C::kStages;
    uint64_t* tmem_full = empty_bar + C::kStages;
    uint64_t* tmem_empty = tmem_full + 2;
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(tmem_empty + 2);
    uint32_t* last_flag = tmem_ptr + 1;
    OutT* stage_t = reinterpret_cast<OutT*>(smem + C::kStages * C::kStageBytes + 256);
    GroupItem* s_items = reinterpret_cast<GroupItem*>(smem + C::kStages * C::kStageBytes + 256 + kStageTileBytes);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i0 = __ldg(&p.cta_first[blockIdx.x]);
    const int n_my = __ldg(&p.cta_first[blockIdx.x + 1]) - i0;

    // ---- prologue: nothing here depends on the previous kernel of the stream (the item table and the tensor maps are the plan's)
    if (warp == 0 && lane == 1) {
        for (int l = 0; l < p.n_lins; ++l) prefetch_tensormap(&p.map_x[l]);
        int n_runs = 0;
        for (int l = 0; l < p.n_lins; ++l) n_runs = max(n_runs, p.lin[l].run0 + p.lin[l].n_runs);
        for (int r = 0; r < n_runs; ++r) prefetch_tensormap(&p.map_w[r]);
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
    if (warp >= 2)
        for (int i = threadIdx.x - 64; i < n_my && i < kMaxCtaItems; i += 128)
            reinterpret_cast<int4*>(s_items)[i] = __ldg(reinterpret_cast<const int4*>(p.items + i0) + i);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    griddep_launch_dependents();   // the next kernel of the stream may start its own prologue and weight ring
    const uint32_t tmem_base = *tmem_ptr;
    auto item_at = [&](int i) -> GroupItem {
        if (i < kMaxCtaItems) return s_items[i];
        const int4 v = __ldg(reinterpret_cast<const int4*>(p.items + i0) + i);
        GroupItem it;
        it.lin = int16_t(v.x & 0xffff);
        it.split = int16_t(v.x >> 16);
        it.m = v.y;
        it.c0 = v.z;
        it.c1 = v.w;
        return it;
    };

    if (warp == 0) {
        // ===================================================================== TMA producer (one elected lane)
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            // X may be written by the previous kernel of the stream, the weights are not: the weight tiles of the first ring
            // are requested at once, their X tiles only after griddepcontrol.wait (both complete the same full barrier).
            bool waited = false;
            int n_pend = 0;
            struct Pend { uint8_t* sb; const CUtensorMap* mx; uint64_t* bar; int xk; } pend[C::kStages];
            auto flush = [&]() {
                griddep_wait();
                for (int k = 0; k < n_pend; ++k) tma_load_2d(pend[k].sb, pend[k].mx, pend[k].bar, pend[k].xk, 0);
                n_pend = 0;
                waited = true;
            };
            for (int i = 0; i < n_my; ++i) {
                const GroupItem it = item_at(i);
                const GroupLin& L = p.lin[it.lin];
                const bool row_par = L.mode == ETP_ROW_PARALLEL;
                int r = row_par ? L.run0 : find_run_in(p, L, it.m);
                const int row = row_par ? 0 : (it.m - p.runs[r].first) * kBM;
                for (int c = it.c0; c < it.c1; ++c) {
                    uint8_t* sa = smem + stage * C::kStageBytes;
                    uint8_t* sb = sa + kABytes;
                    mbar_wait(&empty_bar[stage], phase ^ 1);
                    mbar_expect_tx(&full_bar[stage], C::kStageBytes);
                    int xk;
                    if (!row_par) {
                        tma_load_2d(sa, &p.map_w[r], &full_bar[stage], c * kBK, row);
                        xk = c * kBK;
                    } else {
                        while (r + 1 < L.run0 + L.n_runs && p.runs[r + 1].first <= c) ++r;
                        // K chunks are aligned to multiples of 64 GLOBAL in-features (TMA needs 16-byte aligned box starts in X); a
                        // chunk that straddles two runs is issued once per run, rows outside the run being zero-filled by TMA.
                        const int feat0 = int(p.runs[r].feat0);
                        xk = (feat0 / kBK + (c - p.runs[r].first)) * kBK;
                        const int kin = xk - feat0;
                        tma_load_2d(sa, &p.map_w[r], &full_bar[stage], it.m * kBM, kin);
                        tma_load_2d(sa + kABytes / 2, &p.map_w[r], &full_bar[stage], it.m * kBM + 64, kin);
                    }
                    if (waited) {
                        tma_load_2d(sb, &p.map_x[it.lin], &full_bar[stage], xk, 0);
                    } else {
                        pend[n_pend++] = {sb, &p.map_x[it.lin], &full_bar[stage], xk};
                        if (n_pend == C::kStages) flush();
                    }
                    if (++stage == C::kStages) { stage = 0; phase ^= 1; }
                }
            }
            if (!waited) flush();
        }
        __syncwarp();
    } else if (warp == 1) {
        // ===================================================================== MMA issuer (one elected lane)
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int i = 0; i < n_my; ++i) {
                const GroupItem it = item_at(i);
                const bool a_mn = p.lin[it.lin].mode == ETP_ROW_PARALLEL;
                const uint32_t idesc = make_idesc(p.dtype == ETP_BF16 ? 1u : 0u, a_mn ? 1u : 0u, uint32_t(BN));
                const uint32_t a_lbo = a_mn ? uint32_t(kABytes / 2) : 16u;
                const uint32_t a_kstep = a_mn ? (uint32_t(kUmmaK) * 128u) >> 4 : (uint32_t(kUmmaK) * 2u) >> 4;
                const int as = i & 1;
                const uint32_t aph = (i >> 1) & 1;
                mbar_wait(&tmem_empty[as], aph ^ 1);
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
                    tc_commit(&empty_bar[stage]);
                    if (++stage == C::kStages) { stage = 0; phase ^= 1; }
                }
                tc_commit(&tmem_full[as]);
            }
        }
        __syncwarp();
    } else {
        // ===================================================================== epilogue warps 2..5
        const int q = warp & 3;
        const int m_local = q * 32 + lane;
        const int n_tok = p.tokens;
        griddep_wait();   // Y and the split-K workspace may still be in use by the previous kernel of the stream
        for (int i = 0; i < n_my; ++i) {
            const GroupItem it = item_at(i);
            const GroupLin& L = p.lin[it.lin];
            const bool row_par = L.mode == ETP_ROW_PARALLEL;
            const int as = i & 1;
            const uint32_t aph = (i >> 1) & 1;
            OutT* y;
            int64_t outf, gm0;
            int valid;
            if (!row_par) {
                const int r = find_run_in(p, L, it.m);
                const int row = (it.m - p.runs[r].first) * kBM;
                gm0 = p.runs[r].feat0 + row;
                valid = min(kBM, p.runs[r].n_feat - row);
                y = reinterpret_cast<OutT*>(p.runs[r].y);
                outf = p.runs[r].out_features;
            } else {
                y = reinterpret_cast<OutT*>(L.y);
                outf = L.out_features;
                gm0 = int64_t(it.m) * kBM;
                valid = min(kBM, int(outf) - it.m * kBM);
            }
            const bool vec_out = (outf & 7) == 0;
            mbar_wait(&tmem_full[as], aph);
            tc_fence_after();
            const uint32_t taddr = tmem_base + uint32_t(as * BN) + (uint32_t(q * 32) << 16);
            float* ws = p.partials + size_t(L.ws0 + int64_t(it.m) * L.n_splits + it.split) * size_t(BN) * kBM;
            for (int c16 = 0; c16 < n_tok; c16 += 16) {
                uint32_t v[16];
                tc_ld16(taddr + uint32_t(c16), v);
                tc_ld_wait();
                if (L.n_splits == 1 && vec_out) {
                    store_block16(stage_t, v, m_local, y, size_t(c16), min(16, n_tok - c16), outf, gm0, valid);
                } else if (L.n_splits == 1) {
                    if (m_local < valid) {
#pragma unroll
                        for (int j = 0; j < 16; ++j)
                            if (c16 + j < n_tok) y[size_t(c16 + j) * outf + gm0 + m_local] = cvt16<OutT>(__uint_as_float(v[j]));
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < 16; ++j)
                        if (c16 + j < n_tok) ws[(c16 + j) * kBM + m_local] = __uint_as_float(v[j]);
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&tmem_empty[as]);
            if (L.n_splits > 1) {
                // split-K: the last split to arrive at this tile sums the fp32 partials in split order 0..S-1 (deterministic)
                unsigned int* ticket = p.tickets + L.tile0 + it.m;
                __threadfence();
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (threadIdx.x == 64) *last_flag = (atomicAdd(ticket, 1u) == uint32_t(L.n_splits - 1)) ? 1u : 0u;
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (*last_flag) {
                    __threadfence();
                    const float* w0 = p.partials + size_t(L.ws0 + int64_t(it.m) * L.n_splits) * size_t(BN) * kBM;
                    // 32 threads x float4 cover the 128 features of one token, the four warps take tokens q, q+4, ...; the partials
                    // of four splits are loaded together (independent L2 round trips) and added in split order 0..S-1.
                    const int col4 = lane * 4;
                    const bool vec8 = ((gm0 | outf) & 3) == 0;
                    for (int j = q; j < n_tok; j += 4) {
                        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
                        for (int s0 = 0; s0 < L.n_splits; s0 += 4) {
                            float4 t[4];
#pragma unroll
                            for (int u = 0; u < 4; ++u)
                                t[u] = s0 + u < L.n_splits ? __ldcg(reinterpret_cast<const float4*>(w0 + (size_t(s0 + u) * BN + j) * kBM + col4))
                                                           : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                            for (int u = 0; u < 4; ++u)
                                if (s0 + u < L.n_splits) { acc.x += t[u].x; acc.y += t[u].y; acc.z += t[u].z; acc.w += t[u].w; }
                        }
                        OutT o[4] = {cvt16<OutT>(acc.x), cvt16<OutT>(acc.y), cvt16<OutT>(acc.z), cvt16<OutT>(acc.w)};
                        OutT* dst = y + size_t(j) * outf + gm0 + col4;
                        if (vec8 && col4 + 4 <= valid) {
                            *reinterpret_cast<uint2*>(dst) = *reinterpret_cast<const uint2*>(o);
                        } else {
#pragma unroll
                            for (int e = 0; e < 4; ++e)
                                if (col4 + e < valid) dst[e] = o[e];
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
    if (warp == 1) {
        __syncwarp();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(uint32_t(C::kTmemCols)) : "memory");
    }
}

template <int BN, typename OutT, bool HALF>
etp_status launch_group_t(const GroupParams& p, int grid, cudaStream_t stream, bool pdl) {
    using C = GCfg<BN, HALF>;
    auto k = etp_linear_group_kernel<BN, OutT, HALF>;
    static bool configured = false;   // per instantiation; the attribute is a property of the function, set once per process
    if (!configured) {
        ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes));
        if (HALF) ETP_CUDA_OK(cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        configured = true;
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(unsigned(grid));
    cfg.blockDim = dim3(kLinThreads);
    cfg.dynamicSmemBytes = C::kSmemBytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    cudaError_t e = cudaLaunchKernelEx(&cfg, k, p);
    if (e != cudaSuccess) ETP_FAIL(ETP_ERR_CUDA, "etp_linear_run: launch failed: %s", cudaGetErrorString(e));
    return ETP_OK;
}

template <bool HALF>
etp_status launch_group_h(const GroupParams& p, int bn, int grid, cudaStream_t stream, bool pdl) {
    const bool bf = p.dtype == ETP_BF16;
    if (bn == 16) return bf ? launch_group_t<16, __nv_bfloat16, HALF>(p, grid, stream, pdl) : launch_group_t<16, __half, HALF>(p, grid, stream, pdl);
    return bf ? launch_group_t<64, __nv_bfloat16, HALF>(p, grid, stream, pdl) : launch_group_t<64, __half, HALF>(p, grid, stream, pdl);
}
etp_status launch_group(const GroupParams& p, int bn, int grid, cudaStream_t stream, bool pdl, bool half_ring) {
    return half_ring ? launch_group_h<true>(p, bn, grid, stream, pdl) : launch_group_h<false>(p, bn, grid, stream, pdl);
}

// ------------------------------------------------------------------------------------------------ ctx-owned linear state
struct LinState {
    std::vector<LinWorkspace> ws;
    std::vector<void*> retired;   // outgrown workspace blocks: kernels in flight may still use them, freed with the ctx
    std::unordered_map<std::string, etp_linear_plan*> cache;
};
LinState* lin_state(etp_ctx* c) {
    if (!c->lin_state) c->lin_state = new LinState();
    return static_cast<LinState*>(c->lin_state);
}

}  // namespace

// ------------------------------------------------------------------------------------------------ the plan object
struct etp_linear_plan {
    etp_ctx* ctx = nullptr;
    int device = 0;                         // CUDA device of d_table (kept here so that etp_linear_free never dereferences ctx)
    etp_dtype dtype = ETP_BF16;
    int n_lins = 0;
    struct Lin {
        etp_linear_mode mode;
        int64_t in_features, out_features, features_per_unit;
        etp_tensor w;                       // copy of the descriptor; slabs points into `slabs`
        std::vector<etp_slab> slabs;
        std::vector<etp_shard> layout;
        const void* x_cached = nullptr;     // what map_x[l] was last encoded for
        int64_t tokens_cached = -1;
        int bn_cached = 0;
    } lin[kMaxGroupLins];
    GroupParams p;
    void* d_table = nullptr;                // items + cta_first
    int grid = 0;
    bool half_ring = false;
    int64_t n_partial_tiles = 0, n_tiles = 0;
    int64_t n_items = 0, max_cta_chunks = 0, total_chunks = 0;
};

namespace etp {
namespace lin {

etp_status linear_workspace(etp_ctx* ctx, cudaStream_t stream, int64_t partial_bytes, int64_t n_tickets, LinWorkspace* out) {
    LinState* S = lin_state(ctx);
    LinWorkspace* w = nullptr;
    for (LinWorkspace& e : S->ws)
        if (e.stream == stream) { w = &e; break; }
    if (!w) {
        S->ws.push_back({stream, nullptr, 0, nullptr, 0});
        w = &S->ws.back();
    }
    if (partial_bytes > w->partial_bytes) {   // a new, larger block; the old one may still be read by kernels in flight
        if (w->partials) S->retired.push_back(w->partials);
        w->partials = nullptr;
        w->partial_bytes = 0;
        const int64_t want = std::max<int64_t>(partial_bytes + partial_bytes / 4, 1 << 20);
        ETP_CUDA_OK(cudaMalloc(&w->partials, size_t(want)));
        w->partial_bytes = want;
    }
    if (n_tickets > w->n_tickets) {
        if (w->tickets) S->retired.push_back(w->tickets);
        w->tickets = nullptr;
        w->n_tickets = 0;
        const int64_t n = std::max<int64_t>(n_tickets + n_tickets / 4, 4096);
        ETP_CUDA_OK(cudaMalloc(&w->tickets, size_t(n) * sizeof(unsigned int)));
        ETP_CUDA_OK(cudaMemsetAsync(w->tickets, 0, size_t(n) * sizeof(unsigned int), stream));   // ordered before the first use
        w->n_tickets = n;
    }
    *out = *w;
    return ETP_OK;
}

void free_linear_workspaces(etp_ctx* ctx) {
    if (!ctx->lin_state) return;
    LinState* S = static_cast<LinState*>(ctx->lin_state);
    for (LinWorkspace& e : S->ws) {
        if (e.partials) cudaFree(e.partials);
        if (e.tickets) cudaFree(e.tickets);
    }
    for (void* p : S->retired) cudaFree(p);
    S->ws.clear();
    S->retired.clear();
}

void free_linear_cache(etp_ctx* ctx) {
    if (!ctx->lin_state) return;
    LinState* S = static_cast<LinState*>(ctx->lin_state);
    for (auto& kv : S->cache) etp_linear_free(kv.second);
    S->cache.clear();
    free_linear_workspaces(ctx);
    delete S;
    ctx->lin_state = nullptr;
}

}  // namespace lin

void lin_teardown(etp_ctx* ctx) { lin::free_linear_cache(ctx); }
}  // namespace etp

namespace {

// K splits per linear and the CTA assignment.  The split counts are a function of the NOMINAL shapes only (never of the shard
// layout), so a column-parallel output is bit-identical before and after a reshard (G3).  `c` = target chunks per item.
struct Nominal { int64_t tiles, chunks; };
int splits_for(const Nominal& n, int c) { return int(std::max<int64_t>(1, std::min<int64_t>({(n.chunks + c / 2) / c, n.chunks, 32}))); }

// makespan (in 16-KiB weight chunks) of a longest-processing-time-first assignment of the items to n_ctas CTAs
int64_t lpt_makespan(std::vector<int64_t> costs, int n_ctas) {
    std::sort(costs.begin(), costs.end(), std::greater<int64_t>());
    std::priority_queue<int64_t, std::vector<int64_t>, std::greater<int64_t>> load;
    for (int i = 0; i < n_ctas; ++i) load.push(0);
    int64_t mk = 0;
    for (int64_t c : costs) {
        const int64_t l = load.top() + c;
        load.pop();
        load.push(l);
        mk = std::max(mk, l);
    }
    return mk;
}

// Cost of an item in QUARTER chunks (one chunk = 16 KiB of weights = 0.37 us of one SM's share of the HBM stream): its weight
// chunks, plus - for an item of a split tile - the fp32 partial tile it writes and the last arriver reads back (2 x 8 KiB at 16
// tokens ~ one chunk), plus a small hand-over cost (the ring keeps streaming across items; the epilogue overlaps the next MMAs).
constexpr int64_t item_cost(int64_t chunks, int splits) { return 4 * chunks + (splits > 1 ? 4 : 1); }

}  // namespace

extern "C" etp_status etp_linear_prepare(etp_ctx* ctx, etp_dtype dtype, const etp_linear_spec* lins, int32_t n_lins,
                                         etp_linear_plan** out) {
    if (!out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_prepare: out is NULL");
    *out = nullptr;
    if (!ctx || !lins) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_prepare: NULL argument");
    if (n_lins < 1 || n_lins > kMaxGroupLins) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_prepare: 1..%d linears per group", kMaxGroupLins);
    if (dtype != ETP_BF16 && dtype != ETP_FP16) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_linear_prepare: dtype %d is not bf16/fp16", int(dtype));
    std::unique_ptr<etp_linear_plan> P(new (std::nothrow) etp_linear_plan());
    if (!P) ETP_FAIL(ETP_ERR_NOMEM, "etp_linear_prepare: out of memory");
    P->ctx = ctx;
    P->device = ctx->device;
    P->dtype = dtype;
    P->n_lins = n_lins;
    std::memset(&P->p, 0, sizeof(P->p));
    GroupParams& p = P->p;
    p.n_lins = n_lins;
    p.dtype = dtype;

    int n_runs = 0;
    std::vector<Nominal> nominal(n_lins);
    std::vector<int> m_tiles(n_lins), n_chunks(n_lins);
    for (int l = 0; l < n_lins; ++l) {
        const etp_linear_spec& s = lins[l];
        if (s.mode != ETP_COL_PARALLEL && s.mode != ETP_ROW_PARALLEL) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_prepare: linear %d: bad mode %d", l, int(s.mode));
        if (!s.w || !s.w->slabs || !s.layout) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_prepare: linear %d: NULL argument", l);
        ETP_TRY(check_linear_shape(etp_linear_mode(s.mode), s.in_features, s.out_features, s.features_per_unit, s.w));
        etp_linear_plan::Lin& L = P->lin[l];
        L.mode = etp_linear_mode(s.mode);
        L.in_features = s.in_features;
        L.out_features = s.out_features;
        L.features_per_unit = s.features_per_unit;
        L.w = *s.w;
        L.slabs.assign(s.w->slabs, s.w->slabs + s.w->n_ranks);
        L.w.slabs = L.slabs.data();
        L.layout.assign(s.layout, s.layout + s.n_shards);
        std::vector<etp_shard> sorted;
        ETP_TRY(check_layout(s.layout, s.n_shards, s.w->total_units, &sorted));
        RunList rl;
        ETP_TRY(append_runs(&L.w, sorted, s.features_per_unit, nullptr, s.out_features, &rl));
        if (n_runs + rl.n > kMaxGroupRuns) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_linear_prepare: more than %d contiguous runs in the group", kMaxGroupRuns);
        const bool row_par = L.mode == ETP_ROW_PARALLEL;
        GroupLin& G = p.lin[l];
        G.mode = L.mode;
        G.run0 = n_runs;
        G.n_runs = rl.n;
        G.out_features = int32_t(s.out_features);
        int32_t acc = 0;
        for (int r = 0; r < rl.n; ++r) {
            Run& R = p.runs[n_runs + r];
            R = rl.runs[r];
            R.first = acc;
            if (row_par) {
                acc += int32_t((R.feat0 + R.n_feat + kBK - 1) / kBK - R.feat0 / kBK);   // 64-aligned global K chunks the run touches
                ETP_TRY(encode_2d(&p.map_w[n_runs + r], dtype, rl.addr[r], R.n_feat, s.out_features, s.out_features, 64, kBK));
            } else {
                acc += (R.n_feat + kBM - 1) / kBM;
                ETP_TRY(encode_2d(&p.map_w[n_runs + r], dtype, rl.addr[r], R.n_feat, s.in_features, s.in_features, kBK, kBM));
            }
        }
        n_runs += rl.n;
        m_tiles[l] = row_par ? int((s.out_features + kBM - 1) / kBM) : acc;
        n_chunks[l] = row_par ? acc : int((s.in_features + kBK - 1) / kBK);
        G.n_chunks = n_chunks[l];
        nominal[l] = {(s.out_features + kBM - 1) / kBM, (s.in_features + kBK - 1) / kBK};
    }

    // ---- K splits: the target item size c (in chunks) that minimises the LPT makespan of the NOMINAL group plus the
    // split-K partial traffic it causes (one fp32 tile written and read back per split item, ~BN/16 chunks, spread over the CTAs)
    // Two CTAs per SM with half the ring each (the same bytes in flight per SM): while one CTA of an SM is in its tail (last MMAs,
    // epilogue, split-K reduction) or a CTA of the NEXT launch is in its prologue, the other keeps streaming.  Measured on the
    // config-2 layer at 4 tokens (profiles/r2_linear.md): every single launch of a layer is faster this way (o_t 25.3 -> 19.4 us,
    // gate|up 64.5 -> 62.4 us, the 4-launch chain 121 -> 117 us per layer); the 7-linear group launch is not (103.5 -> 108.2 us:
    // twice as many CTAs want twice as many items, i.e. more split-K partial traffic).  ETP_OPT_LINEAR_RING: 0 / 1 force, 2 = by size.
    int64_t nominal_chunks = 0;
    for (int l = 0; l < n_lins; ++l) nominal_chunks += nominal[l].tiles * nominal[l].chunks;
    const int64_t ring_opt = ctx->opts[ETP_OPT_LINEAR_RING];
    P->half_ring = ring_opt == 1 || (ring_opt == 2 && nominal_chunks < int64_t(200) * ctx->n_sms);
    const int n_ctas = ctx->n_sms * (P->half_ring ? 2 : 1);
    int best_c = 64;
    {
        int64_t best = INT64_MAX;
        for (int c = 2; c <= 96; c += (c < 24 ? 1 : 4)) {
            std::vector<int64_t> costs;
            for (int l = 0; l < n_lins; ++l) {
                const int S = splits_for(nominal[l], c);
                for (int64_t t = 0; t < nominal[l].tiles; ++t)
                    for (int s = 0; s < S; ++s)
                        costs.push_back(item_cost(int64_t(s + 1) * nominal[l].chunks / S - int64_t(s) * nominal[l].chunks / S, S));
            }
            const int64_t cost = lpt_makespan(std::move(costs), n_ctas);
            if (cost < best) { best = cost; best_c = c; }
        }
    }

    // ---- items of the ACTUAL runs, assigned longest first to the least loaded CTA
    std::vector<GroupItem> items;
    int64_t tile0 = 0, ws0 = 0;
    for (int l = 0; l < n_lins; ++l) {
        GroupLin& G = p.lin[l];
        const int S = std::min(splits_for(nominal[l], best_c), std::max(n_chunks[l], 1));
        G.n_splits = S;
        G.tile0 = int32_t(tile0);
        G.ws0 = ws0;
        tile0 += m_tiles[l];
        if (S > 1) ws0 += int64_t(m_tiles[l]) * S;
        if (m_tiles[l] > 0x7fff0000 / std::max(S, 1)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_prepare: too many work items");
        for (int m = 0; m < m_tiles[l]; ++m)
            for (int s = 0; s < S; ++s)
                items.push_back({int16_t(l), int16_t(s), m, int32_t(int64_t(s) * n_chunks[l] / S), int32_t(int64_t(s + 1) * n_chunks[l] / S)});
    }
    P->n_tiles = tile0;
    P->n_partial_tiles = ws0;
    P->n_items = int64_t(items.size());
    const int grid = int(std::min<int64_t>(std::max<int64_t>(P->n_items, 1), n_ctas));
    P->grid = grid;
    std::vector<size_t> order(items.size());
    for (size_t i = 0; i < order.size(); ++i) order[i] = i;
    auto cost_of = [&](const GroupItem& it) { return item_cost(it.c1 - it.c0, p.lin[it.lin].n_splits); };
    std::stable_sort(order.begin(), order.end(), [&](size_t a, size_t b) { return cost_of(items[a]) > cost_of(items[b]); });
    std::vector<std::vector<GroupItem>> per_cta(grid);
    using Load = std::pair<int64_t, int>;
    std::priority_queue<Load, std::vector<Load>, std::greater<Load>> load;
    for (int i = 0; i < grid; ++i) load.push({0, i});
    for (size_t k : order) {
        Load t = load.top();
        load.pop();
        per_cta[t.second].push_back(items[k]);
        t.first += cost_of(items[k]);
        load.push(t);
        P->total_chunks += items[k].c1 - items[k].c0;
    }
    std::vector<int32_t> cta_first(grid + 1, 0);
    std::vector<GroupItem> table;
    table.reserve(items.size());
    for (int i = 0; i < grid; ++i) {
        int64_t chunks = 0;
        for (const GroupItem& it : per_cta[i]) {
            table.push_back(it);
            chunks += it.c1 - it.c0;
        }
        P->max_cta_chunks = std::max(P->max_cta_chunks, chunks);
        cta_first[i + 1] = int32_t(table.size());
    }
    ETP_CUDA_OK(cudaSetDevice(ctx->device));
    const size_t items_bytes = (table.size() * sizeof(GroupItem) + 255) & ~size_t(255);
    ETP_CUDA_OK(cudaMalloc(&P->d_table, items_bytes + cta_first.size() * sizeof(int32_t) + 256));
    cudaError_t e = cudaSuccess;
    if (!table.empty()) e = cudaMemcpy(P->d_table, table.data(), table.size() * sizeof(GroupItem), cudaMemcpyHostToDevice);
    if (e == cudaSuccess)
        e = cudaMemcpy(static_cast<char*>(P->d_table) + items_bytes, cta_first.data(), cta_first.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(P->d_table);
        ETP_FAIL(ETP_ERR_CUDA, "etp_linear_prepare: uploading the item table failed: %s", cudaGetErrorString(e));
    }
    p.items = static_cast<const GroupItem*>(P->d_table);
    p.cta_first = reinterpret_cast<const int32_t*>(static_cast<char*>(P->d_table) + items_bytes);
    *out = P.release();
    return ETP_OK;
}

extern "C" void etp_linear_free(etp_linear_plan* plan) {
    if (!plan) return;
    if (plan->d_table) {
        cudaSetDevice(plan->device);   // not plan->ctx->device: a plan may outlive its ctx up to this call
        cudaFree(plan->d_table);   // synchronises with the kernels that may still read the table
    }
    delete plan;
}

extern "C" etp_status etp_linear_plan_info(const etp_linear_plan* plan, etp_linear_plan_stats* out) {
    if (!plan || !out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_plan_info: NULL argument");
    out->n_linears = plan->n_lins;
    out->n_ctas = plan->grid;
    out->n_items = plan->n_items;
    out->total_chunks = plan->total_chunks;
    out->max_cta_chunks = plan->max_cta_chunks;
    out->n_split_tiles = plan->n_partial_tiles;
    for (int l = 0; l < kMaxGroupLins; ++l) out->n_splits[l] = l < plan->n_lins ? plan->p.lin[l].n_splits : 0;
    return ETP_OK;
}

extern "C" etp_status etp_linear_run(etp_linear_plan* P, const void* const* x, int64_t tokens, void* const* y, void* stream) {
    if (!P || !x || !y) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_run: NULL argument");
    if (tokens < 0 || tokens >= (int64_t(1) << 31)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_run: tokens out of range");
    if (tokens == 0) return ETP_OK;
    for (int l = 0; l < P->n_lins; ++l) {
        if (!x[l] || !y[l]) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_linear_run: x / y of linear %d is NULL", l);
        if ((reinterpret_cast<uintptr_t>(x[l]) | reinterpret_cast<uintptr_t>(y[l])) & 15)
            ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_linear_run: x / y of linear %d not 16-byte aligned", l);
    }
    etp_ctx* ctx = P->ctx;
    if (tokens > 64) {   // tensor-bound regime: one launch per linear (etp_linear.cu); launch overhead no longer matters there
        for (int l = 0; l < P->n_lins; ++l) {
            etp_linear_plan::Lin& L = P->lin[l];
            const LinOut one{&L.w, L.out_features, L.features_per_unit, y[l]};
            ETP_TRY(shard_linear_large(ctx, L.mode, P->dtype, x[l], tokens, L.in_features, &one, 1, L.layout.data(), int32_t(L.layout.size()), stream));
        }
        ctx->launches = P->n_lins;
        return ETP_OK;
    }
    const int bn = tokens <= 16 ? 16 : 64;
    GroupParams& p = P->p;
    for (int l = 0; l < P->n_lins; ++l) {
        etp_linear_plan::Lin& L = P->lin[l];
        if (L.x_cached != x[l] || L.tokens_cached != tokens || L.bn_cached != bn) {
            ETP_TRY(encode_2d(&p.map_x[l], P->dtype, x[l], tokens, L.in_features, L.in_features, kBK, bn));
            L.x_cached = x[l];
            L.tokens_cached = tokens;
            L.bn_cached = bn;
        }
        GroupLin& G = p.lin[l];
        G.y = y[l];
        for (int r = G.run0; r < G.run0 + G.n_runs; ++r) p.runs[r].y = y[l];
    }
    p.tokens = int32_t(tokens);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (P->n_partial_tiles > 0) {
        LinWorkspace w;
        ETP_TRY(linear_workspace(ctx, st, P->n_partial_tiles * int64_t(bn) * kBM * int64_t(sizeof(float)), P->n_tiles, &w));
        p.partials = w.partials;
        p.tickets = w.tickets;
    }
    ctx->launches = 1;
    // behind a slab write of this library on the same stream the launch keeps plain stream order once (etp_internal.h)
    const bool pdl = !etp::take_slab_write(ctx, stream) && ctx->opts[ETP_OPT_LINEAR_PDL] != 0;
    return launch_group(p, bn, P->grid, st, pdl, P->half_ring);
}

// ------------------------------------------------------------------------------------------------ legacy entry points, <= 64 tokens
// etp_shard_linear / etp_shard_linear_multi keep their per-call signatures; below 65 tokens they run through a ctx-owned cache of
// prepared groups keyed by EVERYTHING the preparation reads (mode, dtype, shapes, every slab's base / capacity / anchor, the
// layout), so an entry can never be stale - only unused.  A fused call (q|k|v, gate|up) is one group whose linears share X.
namespace etp {
namespace lin {

etp_status shard_linear_small(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x, int64_t tokens, int64_t in_features,
                              const LinOut* outs, int32_t n_outs, const etp_shard* layout, int32_t n_shards, void* stream) {
    if (n_outs > kMaxGroupLins) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear_multi: at most %d linears", kMaxGroupLins);
    std::string key;
    auto put = [&key](const void* p, size_t n) { key.append(static_cast<const char*>(p), n); };
    const int32_t head[4] = {int32_t(mode), int32_t(dtype), n_outs, n_shards};
    put(head, sizeof(head));
    put(&in_features, sizeof(in_features));
    for (int32_t o = 0; o < n_outs; ++o) {
        const etp_tensor* w = outs[o].w;
        if (!w || !w->slabs || w->n_ranks < 1) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_shard_linear: NULL argument");
        put(&outs[o].out_features, sizeof(int64_t));
        put(&outs[o].features_per_unit, sizeof(int64_t));
        put(&w->total_units, sizeof(int64_t));
        put(&w->unit_bytes, sizeof(int64_t));
        put(&w->n_ranks, sizeof(int32_t));
        put(w->slabs, sizeof(etp_slab) * size_t(w->n_ranks));
    }
    put(layout, sizeof(etp_shard) * size_t(n_shards));
    LinState* S = lin_state(ctx);
    auto it = S->cache.find(key);
    if (it == S->cache.end()) {
        if (S->cache.size() >= 1024) {   // bounded: drop everything (frees synchronise with kernels in flight)
            for (auto& kv : S->cache) etp_linear_free(kv.second);
            S->cache.clear();
        }
        etp_linear_spec specs[kMaxGroupLins];
        for (int32_t o = 0; o < n_outs; ++o)
            specs[o] = {int32_t(mode), 0, in_features, outs[o].out_features, outs[o].w, layout, n_shards, 0, outs[o].features_per_unit};
        etp_linear_plan* plan = nullptr;
        ETP_TRY(etp_linear_prepare(ctx, dtype, specs, n_outs, &plan));
        it = S->cache.emplace(std::move(key), plan).first;
    }
    const void* xs[kMaxGroupLins];
    void* ys[kMaxGroupLins];
    for (int32_t o = 0; o < n_outs; ++o) {
        xs[o] = x;
        ys[o] = outs[o].y;
    }
    return etp_linear_run(it->second, xs, tokens, ys, stream);
}

}  // namespace lin
}  // namespace etp

namespace etp {
cudaError_t install_wait_fault_group(unsigned long long* rec) { return wait_fault_install(rec); }
}  // namespace etp

#define ETP_WAIT_TU 1
#include "etp_copy.cuh"
#include "etp_wait.cuh"

namespace etp {
namespace {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// bounded (etp_wait.cuh): 65536 inline tries, then a slow path that records and traps after kWaitBudgetNs instead of spinning forever
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) { mbar_wait_bounded(bar, parity); }
// global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, uint64_t src_gmem, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_smem),
                 "l"(src_gmem), "r"(bytes), "r"(bar)
                 : "memory");
}
// shared -> global, completion tracked by the thread's bulk async-group
__device__ __forceinline__ void bulk_s2g(uint64_t dst_gmem, uint32_t src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(src_smem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ uint4 ld_stream(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(void* p, const uint4& v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// work item idx of the bulk queue -> (src, dst, bytes): piece (idx - first_item) of its segment
__device__ __forceinline__ void load_bulk_item(const CopyArgs& a, unsigned int idx, uint64_t* src, uint64_t* dst, uint64_t* bytes) {
    const BulkSeg* sg = a.bulk + __ldg(a.bulk_items + idx);
    const uint4 lo = __ldg(reinterpret_cast<const uint4*>(sg));
    const uint4 hi = __ldg(reinterpret_cast<const uint4*>(sg) + 1);
    const uint64_t total = (uint64_t)hi.x | ((uint64_t)hi.y << 32);
    const uint64_t off = (uint64_t)(idx - hi.z) * (uint64_t)kBulkItem;
    *src = ((uint64_t)lo.x | ((uint64_t)lo.y << 32)) + off;
    *dst = ((uint64_t)lo.z | ((uint64_t)lo.w << 32)) + off;
    *bytes = total - off < (uint64_t)kBulkItem ? total - off : (uint64_t)kBulkItem;
}

// ---------------------------------------------------------------------------------------------- bulk (TMA) driver
// One thread.  Chunks (<= kStageBytes) of successive jobs flow through the ring; `loaded - stored <= kLookahead`.
__device__ void tma_driver(const CopyArgs& a, uint8_t* ring, uint64_t* full_bar, uint64_t* s_dst, uint32_t* s_bytes) {
    uint32_t loaded = 0, stored = 0;
    uint64_t cur_src = 0, cur_dst = 0, cur_left = 0;
    bool exhausted = a.n_bulk_items == 0;
    for (;;) {
        bool progressed = false;
        if (!exhausted) {
            if (cur_left == 0) {
                const unsigned int idx = atomicAdd(&a.counters[0], 1u);
                if (idx < a.n_bulk_items) {
                    load_bulk_item(a, idx, &cur_src, &cur_dst, &cur_left);
                } else {
                    exhausted = true;
                }
            }
            if (cur_left != 0) {
                const uint32_t n = cur_left > (uint64_t)kStageBytes ? (uint32_t)kStageBytes : (uint32_t)cur_left;
                const uint32_t st = loaded % kStages;
                // the stage was last used by chunk loaded-kStages; its store is one of the committed groups and at most
                // kStages-1-kLookahead younger groups may still be reading shared memory
                if (loaded >= (uint32_t)kStages) bulk_wait_read<kStages - 1 - kLookahead>();
                const uint32_t bar = smem_u32(&full_bar[st]);
                mbar_arrive_expect_tx(bar, n);
                bulk_g2s(smem_u32(ring + (size_t)st * kStageBytes), cur_src, n, bar);
                s_dst[st] = cur_dst;
                s_bytes[st] = n;
                cur_src += n;
                cur_dst += n;
                cur_left -= n;
                ++loaded;
                progressed = true;
            }
        }
        if (stored < loaded && (loaded - stored > (uint32_t)kLookahead || exhausted)) {
            const uint32_t st = stored % kStages;
            mbar_wait(smem_u32(&full_bar[st]), (stored / kStages) & 1u);
            bulk_s2g(s_dst[st], smem_u32(ring + (size_t)st * kStageBytes), s_bytes[st]);
            bulk_commit();
            ++stored;
            progressed = true;
        }
        if (!progressed) break;
    }
    bulk_wait_all();
}

// ---------------------------------------------------------------------------------------------- vector-copy warps
constexpr int kUnroll = 8;

__device__ __forceinline__ void copy_linear(const char* __restrict__ src, char* __restrict__ dst, uint32_t n_vec, int lane) {
    uint32_t v = lane;
    for (; v + 32 * (kUnroll - 1) < n_vec; v += 32 * kUnroll) {
        uint4 buf[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) buf[u] = ld_stream(src + (size_t)(v + 32 * u) * 16);
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) st_stream(dst + (size_t)(v + 32 * u) * 16, buf[u]);
    }
    for (; v < n_vec; v += 32) st_stream(dst + (size_t)v * 16, ld_stream(src + (size_t)v * 16));
}

// a strided set of rows seen by one warp: row i sits at base + (i / rows_per_group) * grp + (i % rows_per_group) * row
struct RowSet {
    const char* src;
    char* dst;
    uint32_t row_bytes, n_rows, rows_per_group;
    int64_t s_row, d_row, s_grp, d_grp;
};

__device__ __forceinline__ void row_offsets(const RowSet& j, uint32_t v, int vs, int gs, uint32_t vpr, int64_t* so, int64_t* d_o) {
    uint32_t row, col;
    if (vs >= 0) {
        row = v >> vs;
        col = v & (vpr - 1);
    } else {
        row = v / vpr;
        col = v - row * vpr;
    }
    uint32_t grp, r;
    if (gs >= 0) {
        grp = row >> gs;
        r = row & (j.rows_per_group - 1);
    } else {
        grp = row / j.rows_per_group;
        r = row - grp * j.rows_per_group;
    }
    *so = (int64_t)grp * j.s_grp + (int64_t)r * j.s_row + (int64_t)col * 16;
    *d_o = (int64_t)grp * j.d_grp + (int64_t)r * j.d_row + (int64_t)col * 16;
}

__device__ __forceinline__ int log2_exact(uint32_t v) { return (v & (v - 1)) ? -1 : 31 - __clz(v); }

__device__ void copy_rows(const RowSet& j, int lane) {
    const uint32_t vpr = j.row_bytes >> 4;
    const int vs = log2_exact(vpr), gs = log2_exact(j.rows_per_group);
    const uint32_t total = j.n_rows * vpr;
    uint32_t v = lane;
    for (; v + 32 * (kUnroll - 1) < total; v += 32 * kUnroll) {
        uint4 buf[kUnroll];
        int64_t d_o[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            int64_t so;
            row_offsets(j, v + 32 * u, vs, gs, vpr, &so, &d_o[u]);
            buf[u] = ld_stream(j.src + so);
        }
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) st_stream(j.dst + d_o[u], buf[u]);
    }
    for (; v < total; v += 32) {
        int64_t so, d_o;
        row_offsets(j, v, vs, gs, vpr, &so, &d_o);
        st_stream(j.dst + d_o, ld_stream(j.src + so));
    }
}

__device__ __forceinline__ uint64_t u64_of(uint32_t lo, uint32_t hi) { return (uint64_t)lo | ((uint64_t)hi << 32); }

// work item idx of the vector queue: look up its segment, derive the item's addresses, copy it
__device__ void copy_vec_item(const CopyArgs& a, unsigned int idx, int lane) {
    const uint4* p = reinterpret_cast<const uint4*>(a.vec + __ldg(a.vec_items + idx));
    const uint4 q0 = __ldg(p), q1 = __ldg(p + 1);
    const char* src = reinterpret_cast<const char*>(u64_of(q0.x, q0.y));
    char* dst = reinterpret_cast<char*>(u64_of(q0.z, q0.w));
    const uint32_t k = idx - q1.y;   // item within the segment
    if (q1.x == VEC_LINEAR) {
        const uint4 q4 = __ldg(p + 4);
        const uint64_t total = u64_of(q4.x, q4.y), off = (uint64_t)k * (uint64_t)kVecItem;
        const uint64_t n = total - off < (uint64_t)kVecItem ? total - off : (uint64_t)kVecItem;
        copy_linear(src + off, dst + off, (uint32_t)(n >> 4), lane);
        return;
    }
    const uint4 q2 = __ldg(p + 2), q3 = __ldg(p + 3), q4 = __ldg(p + 4), q5 = __ldg(p + 5);
    const uint32_t planes_per_item = q2.x, n_planes = q2.y, items_per_pair = q2.z, pairs_first = q2.w;
    const uint32_t pr = k / items_per_pair, grp = k - pr * items_per_pair;
    const uint32_t pl0 = grp * planes_per_item;
    const uint32_t np = n_planes - pl0 < planes_per_item ? n_planes - pl0 : planes_per_item;
    const int2 ids = __ldg(a.pairs + pairs_first + pr);
    RowSet j;
    j.row_bytes = q1.z;
    j.rows_per_group = q1.w;
    j.n_rows = np * q1.w;
    j.s_row = (int64_t)u64_of(q3.x, q3.y);
    j.d_row = (int64_t)u64_of(q3.z, q3.w);
    j.s_grp = (int64_t)u64_of(q4.x, q4.y);
    j.d_grp = (int64_t)u64_of(q4.z, q4.w);
    j.src = src + (int64_t)pl0 * j.s_grp + (int64_t)ids.x * (int64_t)u64_of(q5.x, q5.y);
    j.dst = dst + (int64_t)pl0 * j.d_grp + (int64_t)ids.y * (int64_t)u64_of(q5.z, q5.w);
    copy_rows(j, lane);
}

// One batch of small contiguous intervals: 32 descriptors per round, one per lane.  Their lengths (in
// 16-byte words) are prefix-summed across the warp, then the warp walks the concatenated words with consecutive lanes on
// consecutive words; the interval of word w is the largest j with excl[j] <= w, found by a 5-step shuffle search, and its
// addresses come from lane j (pre-biased by -excl[j]*16 so that address = base + w*16).
__device__ void copy_small_batch(const CopyArgs& a, unsigned int k, int lane) {
    const uint32_t s0 = __ldg(a.small_first + k), s1 = __ldg(a.small_first + k + 1);
    // the descriptors of round r + 1 are requested before round r is walked, so their latency hides under the round's copies
    uint4 n0 = make_uint4(0, 0, 0, 0), n1 = make_uint4(0, 0, 0, 0);
    if (s0 + lane < s1) {
        const uint4* p = reinterpret_cast<const uint4*>(a.small + s0 + lane);
        n0 = __ldg(p);
        n1 = __ldg(p + 1);
    }
    for (uint32_t s = s0; s < s1; s += 32) {
        uint64_t sb = 0, db = 0;
        uint32_t nv = 0;
        if (s + lane < s1) {
            sb = u64_of(n0.x, n0.y);
            db = u64_of(n0.z, n0.w);
            nv = n1.x >> 4;
        }
        if (s + 32 + lane < s1) {
            const uint4* p = reinterpret_cast<const uint4*>(a.small + s + 32 + lane);
            n0 = __ldg(p);
            n1 = __ldg(p + 1);
        }
        uint32_t incl = nv;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        const uint32_t excl = incl - nv;
        const uint32_t total = __shfl_sync(0xffffffffu, incl, 31);
        sb -= (uint64_t)excl * 16;
        db -= (uint64_t)excl * 16;
        for (uint32_t w0 = 0; w0 < total; w0 += 32 * kUnroll) {   // uniform trip count: every lane joins the shuffles
            uint4 buf[kUnroll];
            uint64_t da[kUnroll];
            // the interval of the block's first and of its last word (warp-uniform): when they coincide - every interval of
            // 4 KiB and more, block after block - the whole block takes its addresses from one lane and skips the per-word search
            const uint32_t w_last = min(w0 + 32 * kUnroll, total) - 1;
            int j_lo = 0, j_hi = 0;
#pragma unroll
            for (int step = 16; step >= 1; step >>= 1) {
                const uint32_t e_lo = __shfl_sync(0xffffffffu, excl, j_lo + step), e_hi = __shfl_sync(0xffffffffu, excl, j_hi + step);
                if (e_lo <= w0) j_lo += step;
                if (e_hi <= w_last) j_hi += step;
            }
            if (j_lo == j_hi) {
                const uint64_t sj = __shfl_sync(0xffffffffu, sb, j_lo), dj = __shfl_sync(0xffffffffu, db, j_lo);
#pragma unroll
                for (int u = 0; u < kUnroll; ++u) {
                    const uint32_t w = w0 + 32 * u + lane;
                    da[u] = dj + (uint64_t)w * 16;
                    if (w < total) buf[u] = ld_stream(reinterpret_cast<const char*>(sj + (uint64_t)w * 16));
                }
            } else {
                // the 8 rows' searches are interleaved step by step: 8 independent shuffles per step instead of 8 serial
                // chains of 5 dependent ones (the warp was stalled on its own shuffle latency, not on memory)
                int j[kUnroll];
#pragma unroll
                for (int u = 0; u < kUnroll; ++u) j[u] = 0;
#pragma unroll
                for (int step = 16; step >= 1; step >>= 1) {
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) {
                        const uint32_t e = __shfl_sync(0xffffffffu, excl, j[u] + step);
                        if (e <= w0 + 32 * u + lane) j[u] += step;
                    }
                }
                uint64_t sa[kUnroll];
#pragma unroll
                for (int u = 0; u < kUnroll; ++u) {
                    sa[u] = __shfl_sync(0xffffffffu, sb, j[u]);
                    da[u] = __shfl_sync(0xffffffffu, db, j[u]) + (uint64_t)(w0 + 32 * u + lane) * 16;
                }
#pragma unroll
                for (int u = 0; u < kUnroll; ++u) {
                    const uint32_t w = w0 + 32 * u + lane;
                    if (w < total) buf[u] = ld_stream(reinterpret_cast<const char*>(sa[u] + (uint64_t)w * 16));
                }
            }
#pragma unroll
            for (int u = 0; u < kUnroll; ++u)
                if (w0 + 32 * u + lane < total) st_stream(reinterpret_cast<char*>(da[u]), buf[u]);
        }
    }
}

// ---------------------------------------------------------------------------------------------- small batches, staged
// The register path above keeps one block (8 x 32 words = 4 KiB) per warp in flight: a block's stores wait for its loads, the next
// block's loads are issued after them, and 126 registers per thread leave no room for a second buffer - at 256 B per interval the
// walk runs at 0.4-0.5 of the copy peak, latency-bound.  When a launch has NO bulk items the 192-KiB ring is idle, and every vector
// warp takes 12 KiB of it as kSmStages stages of 2 KiB.  A batch is then a sequence of BLOCKS of 128 words (rounds of 32 descriptors,
// prefix-summed as above); for every block each lane intersects ITS OWN interval with the block's word range and issues at most one
// cp.async.bulk global -> shared for that piece (completion in bytes on the stage's mbarrier) and, kSmLag blocks later, at most one
// cp.async.bulk shared -> global for the same piece.  No per-word search, no data in registers: the bytes in flight are bounded by
// shared memory (kSmLag blocks per warp), and 32 lanes issue the tensor-less bulk copies in parallel.  1-GiB buckets: 256 B 0.41 ->
// 0.47, 512 B 0.53 -> 0.64, 1 KiB 0.64 -> 0.77, 2 KiB 0.76 -> 0.87, 4 KiB 0.89 -> 0.96 of the copy peak; what is left is a cost of
// ~92 ps per interval (whole chip) on top of bytes / bandwidth that does not move with the depth of the pipeline or the path.
constexpr int kSmBlockWords = 128;   // measured: 128 x 6 stages (lag 4 or 5), 256 x 3 (lag 1 or 2) and 8 / 11 / 15 staged warps beside
constexpr int kSmStages = 6;         // register-path warps all land within 2 % of each other - the walk is no longer latency-bound
constexpr int kSmLag = 4;
constexpr int kSmWarpBytes = kSmStages * kSmBlockWords * 16;
static_assert(15 * kSmWarpBytes <= kStages * kStageBytes, "staged small path must fit the ring");

struct SmallGen {        // walks the blocks of one batch; every lane runs it (it shuffles)
    uint32_t s, s1;      // next round's first descriptor, batch end
    uint64_t base;       // this lane's src (or dst) address, pre-biased by -excl * 16
    uint32_t excl, nv, total, w0;
    uint64_t pf_base;    // the next round's descriptor of this lane, requested one round ahead
    uint32_t pf_bytes;
    bool valid;
};

__device__ __forceinline__ void gen_prefetch(SmallGen& g, const SmallSeg* small, int lane, bool use_dst) {
    g.pf_base = 0;
    g.pf_bytes = 0;
    if (g.s + lane < g.s1) {
        const uint4* p = reinterpret_cast<const uint4*>(small + g.s + lane);
        const uint4 q0 = __ldg(p);
        g.pf_bytes = __ldg(reinterpret_cast<const uint32_t*>(p + 1));
        g.pf_base = use_dst ? u64_of(q0.z, q0.w) : u64_of(q0.x, q0.y);
    }
}

__device__ __forceinline__ void gen_advance(SmallGen& g, const SmallSeg* small, int lane, bool use_dst) {
    g.w0 += kSmBlockWords;
    while (g.w0 >= g.total) {
        if (g.s >= g.s1) {
            g.valid = false;
            return;
        }
        const uint64_t b = g.pf_base;
        const uint32_t nv = g.pf_bytes >> 4;
        g.s += 32;
        gen_prefetch(g, small, lane, use_dst);      // in flight while this round's blocks are copied
        uint32_t incl = nv;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        g.nv = nv;
        g.excl = incl - nv;
        g.total = __shfl_sync(0xffffffffu, incl, 31);
        g.base = b - (uint64_t)g.excl * 16;
        g.w0 = 0;
    }
    g.valid = true;
}

__device__ uint32_t copy_small_batch_staged(const CopyArgs& a, unsigned int k, int lane, uint8_t* stage_mem, uint64_t* bars, uint32_t gb) {
    SmallGen lead, lag;
    lead.s = lag.s = __ldg(a.small_first + k);
    lead.s1 = lag.s1 = __ldg(a.small_first + k + 1);
    lead.total = lag.total = 0;
    lead.w0 = lag.w0 = 0;
    lead.nv = lag.nv = lead.excl = lag.excl = 0;
    lead.base = lag.base = 0;
    gen_prefetch(lead, a.small, lane, false);
    gen_prefetch(lag, a.small, lane, true);
    gen_advance(lead, a.small, lane, false);
    gen_advance(lag, a.small, lane, true);
    uint32_t issued = 0, stored = 0;
    for (;;) {
        bool did = false;
        if (lead.valid && issued - stored < (uint32_t)kSmLag) {
            const uint32_t g = gb + issued, st = g % kSmStages;
            // the stage's previous block (g - kSmStages) was stored at least kSmStages - kSmLag store groups ago
            bulk_wait_read<kSmStages - kSmLag>();
            __syncwarp();
            const uint32_t bar = smem_u32(&bars[st]);
            const uint32_t blk = min((uint32_t)kSmBlockWords, lead.total - lead.w0);
            if (lane == 0) mbar_arrive_expect_tx(bar, blk * 16);
            const uint32_t lo = max(lead.excl, lead.w0), hi = min(lead.excl + lead.nv, lead.w0 + blk);
            if (lo < hi)
                bulk_g2s(smem_u32(stage_mem + (size_t)st * (kSmBlockWords * 16) + (size_t)(lo - lead.w0) * 16), lead.base + (uint64_t)lo * 16, (hi - lo) * 16, bar);
            ++issued;
            gen_advance(lead, a.small, lane, false);
            did = true;
        }
        if (stored < issued && (issued - stored == (uint32_t)kSmLag || !lead.valid)) {
            const uint32_t g = gb + stored, st = g % kSmStages;
            mbar_wait(smem_u32(&bars[st]), (g / kSmStages) & 1u);
            const uint32_t blk = min((uint32_t)kSmBlockWords, lag.total - lag.w0);
            const uint32_t lo = max(lag.excl, lag.w0), hi = min(lag.excl + lag.nv, lag.w0 + blk);
            if (lo < hi)
                bulk_s2g(lag.base + (uint64_t)lo * 16, smem_u32(stage_mem + (size_t)st * (kSmBlockWords * 16) + (size_t)(lo - lag.w0) * 16), (hi - lo) * 16);
            bulk_commit();
            ++stored;
            gen_advance(lag, a.small, lane, true);
            did = true;
        }
        if (!did) break;
    }
    return gb + issued;
}

template <bool STAGED>
__device__ void vector_warp(const CopyArgs& a, int lane, uint8_t* stage_mem, uint64_t* bars) {
    const unsigned int n_items = a.n_vec_items + a.n_small_batches;
    constexpr bool staged = STAGED;             // the host launches this instantiation only when the ring is idle (no bulk items)
    uint32_t gb = 0;                            // blocks this warp has pushed through its stages (stage = gb % kSmStages)
    if (staged) {
        if (lane == 0) {
            for (int s = 0; s < kSmStages; ++s) mbar_init(smem_u32(&bars[s]), 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        __syncwarp();
    }
    for (;;) {
        unsigned int idx = 0;
        if (lane == 0) idx = atomicAdd(&a.counters[1], 1u);
        idx = __shfl_sync(0xffffffffu, idx, 0);
        if (idx >= n_items) break;
        if (idx < a.n_vec_items)
            copy_vec_item(a, idx, lane);
        else if constexpr (staged)
            gb = copy_small_batch_staged(a, idx - a.n_vec_items, lane, stage_mem, bars, gb);
        else
            copy_small_batch(a, idx - a.n_vec_items, lane);
    }
    if (staged) bulk_wait_all();
    if (a.flags & 1u) {
        // drain the bulk queue too (one item per warp at a time)
        for (;;) {
            unsigned int idx = 0;
            if (lane == 0) idx = atomicAdd(&a.counters[0], 1u);
            idx = __shfl_sync(0xffffffffu, idx, 0);
            if (idx >= a.n_bulk_items) break;
            uint64_t src, dst, bytes;
            load_bulk_item(a, idx, &src, &dst, &bytes);
            copy_linear(reinterpret_cast<const char*>(src), reinterpret_cast<char*>(dst), (uint32_t)(bytes >> 4), lane);
        }
    }
}

// STAGED = false is the kernel of the reshard path (and of every launch with bulk intervals); STAGED = true is launched by the host when
// a launch has small batches and NO bulk items: the ring belongs to the vector warps (copy_small_batch_staged).  Two instantiations, so
// that the staged code does not perturb the register allocation of the head-strided KV path (it cost that launch 5 % when inlined).
template <bool STAGED>
__global__ void __launch_bounds__(kCopyThreads, 1) etp_interval_copy_kernel(const CopyArgs args) {
    extern __shared__ __align__(1024) uint8_t smem[];
    CopyArgs a = args;
    if (args.dev_counts) {   // queue lengths computed on the device by the classifier kernels that ran before this launch
        a.n_bulk_items = __ldg(args.dev_counts);
        a.n_vec_items = __ldg(args.dev_counts + 1);
        a.n_small_batches = __ldg(args.dev_counts + 2);
    }
    uint8_t* ring = smem;
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + (size_t)kStages * kStageBytes);
    uint64_t* s_dst = full_bar + kStages;
    uint32_t* s_bytes = reinterpret_cast<uint32_t*>(s_dst + kStages);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp == 0) {
        if (!STAGED && lane == 0) {
            for (int s = 0; s < kStages; ++s) mbar_init(smem_u32(&full_bar[s]), 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            tma_driver(a, ring, full_bar, s_dst, s_bytes);
        }
    } else {
        uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)kStages * kStageBytes + 128) + (warp - 1) * kSmStages;
        vector_warp<STAGED>(a, lane, STAGED ? ring + (size_t)(warp - 1) * kSmWarpBytes : nullptr, bars);
    }
}

// debug: a barrier nobody arrives on, waited for with the same mbar_wait as the kernels (etp_debug_starved_wait)
__global__ void etp_starved_wait_kernel() {
    __shared__ uint64_t bar;
    if (threadIdx.x == 0) {
        mbar_init(smem_u32(&bar), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        mbar_wait(smem_u32(&bar), 0);
    }
}
}  // namespace

cudaError_t install_wait_fault_copy(unsigned long long* rec) { return wait_fault_install(rec); }
void launch_starved_wait_kernel(cudaStream_t stream) { etp_starved_wait_kernel<<<3, 64, 0, stream>>>(); }

cudaError_t configure_copy_kernel() {
    cudaError_t e = cudaFuncSetAttribute(etp_interval_copy_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCopySmemBytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(etp_interval_copy_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCopySmemBytes);
}

void launch_copy_kernel(const CopyArgs& a, int grid, cudaStream_t stream, bool staged_small) {
    if (staged_small)
        etp_interval_copy_kernel<true><<<grid, kCopyThreads, kCopySmemBytes, stream>>>(a);
    else
        etp_interval_copy_kernel<false><<<grid, kCopyThreads, kCopySmemBytes, stream>>>(a);
}

}  // namespace etp

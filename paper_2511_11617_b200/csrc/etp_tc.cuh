// tcgen05 / TMEM / TMA building blocks shared by kernel (c) (etp_linear.cu) and its grouped MoE variant (etp_moe.cu):
// tile constants, PTX wrappers, shared-memory / instruction descriptors and the host-side tensor-map encoder.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "etp_internal.h"
#include "etp_wait.cuh"

namespace etp {
namespace tc {

constexpr int kBM = 128;          // out features per tile = UMMA_M
constexpr int kBK = 64;           // K elements per pipeline stage: 128 bytes = one 128B-swizzle atom
constexpr int kUmmaK = 16;        // K per tcgen05.mma for 16-bit inputs
constexpr int kMaxRuns = 16;      // <= 2 contiguous runs per rank, 8 ranks
constexpr int kLinThreads = 192;  // 6 warps
constexpr int kABytes = kBM * kBK * 2;
constexpr int kSmemBudget = 200 << 10;


// ------------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// etp_wait.cuh: the plain try_wait loop, or (builds with ETP_BOUNDED_WAITS=1) the bounded wait that records and traps after kWaitBudgetNs
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) { etp::mbar_wait_bounded(smem_u32(bar), parity); }
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, uint64_t* bar, int32_t c0, int32_t c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            smem_u32(smem_dst)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void prefetch_tensormap(const CUtensorMap* map) {   // descriptor into the TMA unit's cache before first use
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void tc_ld16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
          "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tc_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor (tcgen05 "smem descriptor"): start address, leading / stride byte offsets (all >> 4),
// descriptor version 1 (Blackwell) at bit 46, layout type SWIZZLE_128B (= 2) at bits 61-63.
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return uint64_t((saddr & 0x3FFFFu) >> 4) | (uint64_t(lbo_bytes >> 4) << 16) | (uint64_t(sbo_bytes >> 4) << 32) |
           (uint64_t(1) << 46) | (uint64_t(2) << 61);
}
// Instruction descriptor of kind::f16: D = fp32 (bits 4-5 = 1), A/B format (0 = fp16, 1 = bf16) at bits 7-9 / 10-12,
// A/B major (0 = K, 1 = MN) at bits 15 / 16, N >> 3 at bits 17-22, M >> 4 at bits 24-28.
__host__ __device__ constexpr uint32_t make_idesc(uint32_t fmt, uint32_t a_mn_major, uint32_t n) {
    return (1u << 4) | (fmt << 7) | (fmt << 10) | (a_mn_major << 15) | ((n >> 3) << 17) | ((uint32_t(kBM) >> 4) << 24);
}

// ---- CTA pairs (cluster of 2, tcgen05 cta_group::2): shared by kernel (c)'s pair kernel and the grouped MoE pair kernel
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t mapa_rank0(uint32_t saddr) {   // the same shared-memory offset in CTA 0 of the cluster
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, 0;" : "=r"(r) : "r"(saddr));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void tma_load_2d_pair(void* smem_dst, const CUtensorMap* map, uint32_t leader_bar, int32_t c0, int32_t c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            smem_u32(smem_dst)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(leader_bar), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void tc_commit_pair(uint64_t* bar) {   // arrives on `bar` at the same offset in BOTH CTAs
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)),
                 "h"(uint16_t(3))
                 : "memory");
}
__device__ __forceinline__ void tc_mma_pair(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__host__ __device__ constexpr uint32_t make_idesc_pair(uint32_t fmt, uint32_t a_mn_major, uint32_t n) {
    return (1u << 4) | (fmt << 7) | (fmt << 10) | (a_mn_major << 15) | ((n >> 3) << 17) | ((uint32_t(2 * kBM) >> 4) << 24);
}

template <typename T>
__device__ __forceinline__ T cvt16(float v);
template <>
__device__ __forceinline__ __nv_bfloat16 cvt16<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }
template <>
__device__ __forceinline__ __half cvt16<__half>(float v) { return __float2half_rn(v); }


// Epilogue store of one [128 out features][16 tokens] fp32 block held by the four epilogue warps (thread = out feature
// m_local = 32 * (warp % 4) + lane, v[j] = token j) into row-major Y[token][out_features] as 16-BYTE stores.  The block is
// transposed through a [16][kStagePitch] 16-bit shared buffer written at column (gm0 mod 8) + m_local, so that column c of the
// buffer is global feature (gm0 - gm0 mod 8) + c and every aligned 8-element chunk of the buffer is an aligned 16-byte chunk
// of Y (out_features % 8 == 0 required); the <= 2 ragged chunks of a row fall back to 2-byte stores.  128 threads, named
// barrier 1.  `valid` may be <= 0 (nothing stored).
constexpr int kStagePitch = kBM + 8;                       // elements
constexpr int kStageTileBytes = 16 * kStagePitch * 2 + 256;  // rounded up
template <typename OutT>
__device__ __forceinline__ void store_block16(OutT* stage, const uint32_t (&v)[16], int m_local, OutT* y, size_t row0, int n_tok,
                                              int64_t out_features, int64_t gm0, int valid) {
    const int a = int(gm0 & 7);
#pragma unroll
    for (int j = 0; j < 16; ++j) stage[j * kStagePitch + a + m_local] = cvt16<OutT>(__uint_as_float(v[j]));
    asm volatile("bar.sync 1, 128;" ::: "memory");
    constexpr int kChunks = kStagePitch / 8;               // 17
    for (int id = m_local; id < 16 * kChunks; id += 128) {
        const int row = id / kChunks, ch = id - row * kChunks;
        if (row >= n_tok) break;
        const int c0 = ch * 8 - a;                         // feature of the chunk's first element, relative to gm0
        OutT* dst = y + (row0 + size_t(row)) * size_t(out_features) + gm0 + c0;
        const OutT* src = stage + row * kStagePitch + ch * 8;
        if (c0 >= 0 && c0 + 8 <= valid) {
            *reinterpret_cast<uint4*>(dst) = *reinterpret_cast<const uint4*>(src);
        } else {
#pragma unroll
            for (int e = 0; e < 8; ++e)
                if (c0 + e >= 0 && c0 + e < valid) dst[e] = src[e];
        }
    }
    asm volatile("bar.sync 1, 128;" ::: "memory");
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            p = nullptr;
        }
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

// 2-D row-major 16-bit tensor [rows][cols] at `base`, box {box_cols (= 64 elements = 128 B), box_rows}, 128B swizzle,
// out-of-bounds elements read as zero.
inline etp_status encode_2d(CUtensorMap* map, etp_dtype dtype, const void* base, int64_t rows, int64_t cols, int64_t pitch_elems,
                     int box_cols, int box_rows) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) ETP_FAIL(ETP_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
    cuuint64_t dims[2] = {cuuint64_t(cols), cuuint64_t(rows)};
    cuuint64_t strides[1] = {cuuint64_t(pitch_elems) * 2};
    cuuint32_t box[2] = {cuuint32_t(box_cols), cuuint32_t(box_rows)};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(map, dtype == ETP_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2,
                    const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS)
        ETP_FAIL(ETP_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d) for [%lld][%lld] pitch %lld box {%d,%d}", int(r),
                 (long long)rows, (long long)cols, (long long)pitch_elems, box_cols, box_rows);
    return ETP_OK;
}


}  // namespace tc
}  // namespace etp

// Bounded mbarrier waits: a starved barrier becomes an ERROR within seconds instead of a kernel that spins until the pool is reset.
//
// Every hand-rolled wait of this library is an mbarrier parity wait (TMA complete_tx, tcgen05.commit, consumer-release arrivals); a
// lost arrival or a wrong expect_tx count would leave a persistent kernel spinning forever.  mbar_wait_bounded spins inline for 65536 attempts (the
// old PTX loop plus one counter) and then enters a non-inlined slow path that keeps trying with
// %globaltimer as its clock; after kWaitBudgetNs it writes a record {kernel family, block, thread, barrier, parity, waited ns} to a
// host-mapped pinned buffer (it survives the death of the CUDA context) and executes trap.  The launch then fails with a sticky
// CUDA error, every later call of the library returns ETP_ERR_CUDA, and etp_last_error() carries the record (etp::set_error).
//
// `g_wait_fault` has internal linkage: each translation unit that includes this header has its own copy and exports a one-line
// installer (wait_fault_install); etp_ctx_create installs the record's address on every device of the ctx.  A kernel launched without
// a ctx (etp_copy_intervals_static) finds NULL there and traps without a record.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#ifndef ETP_WAIT_TU
#define ETP_WAIT_TU 0   // 1 = etp_copy.cu, 2 = etp_linear.cu, 3 = etp_linear_group.cu, 4 = etp_moe.cu
#endif

namespace etp {

constexpr unsigned long long kWaitBudgetNs = 10ull * 1000ull * 1000ull * 1000ull;   // 10 s: far above any legitimate wait (the longest
                                                                                   // is a tile load over the host link, milliseconds)
constexpr unsigned long long kWaitFaultMagic = 0x4554504641554c54ull;               // "ETPFAULT"
constexpr int kWaitFaultWords = 8;   // [0] magic  [1] family  [2] blockIdx.x  [3] threadIdx.x  [4] barrier (shared address)  [5] parity  [6] waited ns

static __device__ unsigned long long* g_wait_fault = nullptr;
static inline cudaError_t wait_fault_install(unsigned long long* p) { return cudaMemcpyToSymbol(g_wait_fault, &p, sizeof(p)); }

__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}

__device__ __forceinline__ unsigned long long wait_clock_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

[[maybe_unused]] static __device__ __noinline__ void mbar_wait_slow(uint32_t bar, uint32_t parity) {
    const unsigned long long t0 = wait_clock_ns();
    for (;;) {
#pragma unroll 1
        for (int i = 0; i < 64; ++i)
            if (mbar_try_wait(bar, parity)) return;
        const unsigned long long waited = wait_clock_ns() - t0;
        if (waited > kWaitBudgetNs) {
            volatile unsigned long long* r = g_wait_fault;
            if (r) {
                r[1] = ETP_WAIT_TU;
                r[2] = blockIdx.x;
                r[3] = threadIdx.x;
                r[4] = bar;
                r[5] = parity;
                r[6] = waited;
                __threadfence_system();
                r[0] = kWaitFaultMagic;
                __threadfence_system();
                while (r[0] != kWaitFaultMagic) {}   // a read round trip: the record is in host memory before the context dies
            }
            asm volatile("trap;");
        }
    }
}

// The common case - a producer / consumer pair of a pipeline waiting microseconds for each other - must cost what the plain try_wait
// loop cost.  Entering the slow path on every failed first try cost the tcgen05 kernels 3-12 % (measured), and so did a C++ loop
// around mbar_try_wait (the compiler's selp / setp / branch sequence sits between the barrier flipping and the MMA issue).  So the
// first kInlineTries attempts are the old two-instruction PTX loop plus a counter, in one asm block whose success path branches
// straight out; only a wait that outlasts them (>= ~1 ms) pays for the call and the %globaltimer reads.
//
// Where it is on.  Kernel (a) (etp_copy.cu, the hot path) always: its cost there is nil (config 2: 1.0032 vs 1.0028 of the copy peak, TRANSFER-only
// launch 0.6046 vs 0.6051 ms, profiles/r3_liveness.md).  The tcgen05 kernels (shard linear, grouped linear, MoE) only in a build with
// ETP_BOUNDED_WAITS=1 (environment variable read by _build.py -> -DETP_BOUNDED_WAITS=1): even in this form they lose 5-8 % (config 2 layer at
// 4096 tokens 1993 -> 2146 us, 4-token group launch 103.2 -> 108.7 us; the kernels become non-leaf functions and the waits sit on the
// MMA-issue / TMA-issue critical path), which is too much to pay in production for a check that only fires on a bug.
#ifndef ETP_BOUNDED_WAITS
#define ETP_BOUNDED_WAITS (ETP_WAIT_TU == 1)
#endif
constexpr uint32_t kInlineTries = 1u << 16;
__device__ __forceinline__ void mbar_wait_bounded(uint32_t bar, uint32_t parity) {
#if !ETP_BOUNDED_WAITS
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(bar), "r"(parity)
        : "memory");
#else
    uint32_t expired;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        ".reg .u32 n;\n\t"
        "mov.u32 n, %3;\n\t"
        "mov.u32 %0, 0;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "@p bra DONE_%=;\n\t"
        "sub.u32 n, n, 1;\n\t"
        "setp.ne.u32 p, n, 0;\n\t"
        "@p bra WAIT_%=;\n\t"
        "mov.u32 %0, 1;\n\t"
        "DONE_%=:\n\t"
        "}"
        : "=&r"(expired)
        : "r"(bar), "r"(parity), "n"(kInlineTries)
        : "memory");
    if (expired) mbar_wait_slow(bar, parity);
#endif
}

}  // namespace etp

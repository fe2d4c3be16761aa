// Host-only contract check of etp_copy_intervals (include/etp.h): every interval 16-byte aligned with a non-negative size, the
// destinations mutually disjoint and disjoint from every source (the intervals of one call are unordered, so a destination that
// overlapped another interval's source would race).  O(n) work apart from small per-bucket sorts, on up to 16 threads:
//   1. records -> (start, end, index) keys of both sides, argument checks on the way (parallel over index ranges);
//   2. keys are scattered into address buckets (uniform cuts of [min start, max start], per-thread histograms) and every bucket
//      is sorted on its own (std::sort, buckets handed out dynamically) - the concatenation is the sorted array;
//   3. destinations: adjacent pairs must not overlap (parallel);  sources vs destinations: prefix maximum of the source ends in
//      start order, then for every destination d the sources that start below d.end are a prefix - d overlaps one of them iff the
//      prefix maximum exceeds d.begin (binary search per destination, parallel).
// The first violation in address order is reported with the two interval indices.
#include <algorithm>
#include <atomic>
#include <cstdint>
#include <cstring>
#include <memory>
#include <thread>
#include <vector>

#include "etp_internal.h"

namespace {

struct Key {
    uint64_t b, e, i;
};

int n_threads_for(int64_t n) {
    if (n < 65536) return 1;
    unsigned hw = std::thread::hardware_concurrency();
    return int(std::max(1u, std::min(16u, hw ? hw : 1u)));
}

template <typename F>
void parallel_for(int T, F&& f) {   // f(t) for t in [0, T)
    if (T == 1) {
        f(0);
        return;
    }
    std::vector<std::thread> th;
    th.reserve(size_t(T) - 1);
    for (int t = 1; t < T; ++t) th.emplace_back([&f, t] { f(t); });
    f(0);
    for (std::thread& x : th) x.join();
}

// Sorts the n keys of v by start address; returns the array that holds the result (v, or scratch - n entries - when the bucket
// path ran: no copy back).
Key* bucket_sort(Key* v, size_t n, Key* scratch, int T) {
    if (n < 2) return v;
    if (T == 1 || n < 65536) {
        std::sort(v, v + n, [](const Key& a, const Key& b) { return a.b < b.b; });
        return v;
    }
    uint64_t lo = UINT64_MAX, hi = 0;
    {
        std::vector<uint64_t> los(size_t(T), UINT64_MAX), his(size_t(T), 0);
        parallel_for(T, [&](int t) {
            uint64_t l = UINT64_MAX, h = 0;
            for (size_t j = n * size_t(t) / size_t(T); j < n * size_t(t + 1) / size_t(T); ++j) {
                l = std::min(l, v[j].b);
                h = std::max(h, v[j].b);
            }
            los[size_t(t)] = l;
            his[size_t(t)] = h;
        });
        for (int t = 0; t < T; ++t) {
            lo = std::min(lo, los[size_t(t)]);
            hi = std::max(hi, his[size_t(t)]);
        }
    }
    const int B = 64 * T;                                   // buckets: uniform cuts of the start range
    const uint64_t width = (hi - lo) / uint64_t(B) + 1;
    std::vector<size_t> hist(size_t(T) * size_t(B), 0);
    auto range = [&](int t, size_t* a, size_t* b) {
        *a = n * size_t(t) / size_t(T);
        *b = n * size_t(t + 1) / size_t(T);
    };
    parallel_for(T, [&](int t) {
        size_t a, b;
        range(t, &a, &b);
        size_t* h = &hist[size_t(t) * size_t(B)];
        for (size_t j = a; j < b; ++j) ++h[(v[j].b - lo) / width];
    });
    std::vector<size_t> start(size_t(B) + 1, 0);
    {   // offsets: bucket-major, thread-minor, so that every thread scatters into its own sub-range of a bucket
        size_t acc = 0;
        for (int k = 0; k < B; ++k) {
            start[size_t(k)] = acc;
            for (int t = 0; t < T; ++t) {
                const size_t c = hist[size_t(t) * size_t(B) + size_t(k)];
                hist[size_t(t) * size_t(B) + size_t(k)] = acc;
                acc += c;
            }
        }
        start[size_t(B)] = acc;
    }
    parallel_for(T, [&](int t) {
        size_t a, b;
        range(t, &a, &b);
        size_t* h = &hist[size_t(t) * size_t(B)];
        for (size_t j = a; j < b; ++j) scratch[h[(v[j].b - lo) / width]++] = v[j];
    });
    std::atomic<int> next{0};
    parallel_for(T, [&](int) {
        for (;;) {
            const int k = next.fetch_add(1);
            if (k >= B) break;
            std::sort(scratch + start[size_t(k)], scratch + start[size_t(k) + 1], [](const Key& a, const Key& b) { return a.b < b.b; });
        }
    });
    return scratch;
}

}  // namespace

namespace etp {

etp_status validate_intervals(const etp_interval* d, int64_t n, bool check_overlap) {
    if (n < 0 || (n > 0 && !d)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: bad arguments");
    const int T = n_threads_for(n);
    // ---- 1. argument checks + keys
    std::vector<int64_t> first_bad(size_t(T), -1);
    std::vector<size_t> cnt(size_t(T) + 1, 0);
    auto irange = [&](int t, int64_t* a, int64_t* b) {
        *a = n * t / T;
        *b = n * (t + 1) / T;
    };
    parallel_for(T, [&](int t) {
        int64_t a, b;
        irange(t, &a, &b);
        size_t c = 0;
        for (int64_t i = a; i < b; ++i) {
            const etp_interval& x = d[i];
            if (x.bytes == 0) continue;
            ++c;
            if (first_bad[size_t(t)] < 0 &&
                (x.bytes < 0 || !x.src || !x.dst || (((uintptr_t)x.src | (uintptr_t)x.dst | (uint64_t)x.bytes) & 15)))
                first_bad[size_t(t)] = i;
        }
        cnt[size_t(t) + 1] = c;
    });
    for (int t = 0; t < T; ++t)
        if (first_bad[size_t(t)] >= 0) {
            const int64_t i = first_bad[size_t(t)];
            const etp_interval& x = d[i];
            if (x.bytes < 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: interval %lld has negative size", (long long)i);
            if (!x.src || !x.dst) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: interval %lld has a NULL pointer", (long long)i);
            ETP_FAIL(ETP_ERR_ALIGNMENT, "etp_copy_intervals: interval %lld is not 16-byte aligned", (long long)i);
        }
    if (!check_overlap) return ETP_OK;
    for (int t = 0; t < T; ++t) cnt[size_t(t) + 1] += cnt[size_t(t)];
    const size_t m = cnt[size_t(T)];
    if (m < 1) return ETP_OK;
    // uninitialised arrays (every entry is written below); two scratch arrays so that neither sort copies back
    std::unique_ptr<Key[]> dst_a(new Key[m]), src_a(new Key[m]), dst_s(new Key[m]), src_s(new Key[m]);
    Key *dst = dst_a.get(), *src = src_a.get();
    parallel_for(T, [&](int t) {
        int64_t a, b;
        irange(t, &a, &b);
        size_t o = cnt[size_t(t)];
        for (int64_t i = a; i < b; ++i) {
            const etp_interval& x = d[i];
            if (x.bytes == 0) continue;
            dst[o] = {(uint64_t)(uintptr_t)x.dst, (uint64_t)(uintptr_t)x.dst + (uint64_t)x.bytes, (uint64_t)i};
            src[o] = {(uint64_t)(uintptr_t)x.src, (uint64_t)(uintptr_t)x.src + (uint64_t)x.bytes, (uint64_t)i};
            ++o;
        }
    });
    // ---- 2. both sides in start order
    dst = bucket_sort(dst, m, dst_s.get(), T);
    src = bucket_sort(src, m, src_s.get(), T);
    // ---- 3a. destinations mutually disjoint (first violation in address order)
    std::vector<size_t> bad(size_t(T), SIZE_MAX);
    parallel_for(T, [&](int t) {
        const size_t a = std::max<size_t>(1, m * size_t(t) / size_t(T)), b = m * size_t(t + 1) / size_t(T);
        for (size_t k = a; k < b; ++k)
            if (dst[k].b < dst[k - 1].e) {
                bad[size_t(t)] = k;
                break;
            }
    });
    for (int t = 0; t < T; ++t)
        if (bad[size_t(t)] != SIZE_MAX) {
            const size_t k = bad[size_t(t)];
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: destinations of intervals %lld and %lld overlap", (long long)dst[k - 1].i, (long long)dst[k].i);
        }
    // ---- 3b. no destination overlaps a source: prefix maximum of the source ends (and who attains it) in start order
    std::vector<uint64_t> pmax(m);
    std::vector<uint64_t> parg(m);
    {
        uint64_t best = 0, who = 0;
        for (size_t k = 0; k < m; ++k) {
            if (src[k].e > best) {
                best = src[k].e;
                who = src[k].i;
            }
            pmax[k] = best;
            parg[k] = who;
        }
    }
    std::fill(bad.begin(), bad.end(), SIZE_MAX);
    parallel_for(T, [&](int t) {
        const size_t a = m * size_t(t) / size_t(T), b = m * size_t(t + 1) / size_t(T);
        size_t hint = 0;
        for (size_t k = a; k < b; ++k) {
            // number of sources that start below this destination's end (destinations ascend, so the count is monotone within a range)
            size_t lo = hint, hi = m;
            while (lo < hi) {
                const size_t mid = (lo + hi) >> 1;
                if (src[mid].b < dst[k].e) lo = mid + 1;
                else hi = mid;
            }
            hint = lo;
            if (lo > 0 && pmax[lo - 1] > dst[k].b) {
                bad[size_t(t)] = k;
                break;
            }
        }
    });
    for (int t = 0; t < T; ++t)
        if (bad[size_t(t)] != SIZE_MAX) {
            const size_t k = bad[size_t(t)];
            size_t lo = 0, hi = m;
            while (lo < hi) {
                const size_t mid = (lo + hi) >> 1;
                if (src[mid].b < dst[k].e) lo = mid + 1;
                else hi = mid;
            }
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_copy_intervals: destination of interval %lld overlaps the source of interval %lld", (long long)dst[k].i,
                     (long long)parg[lo - 1]);
        }
    return ETP_OK;
}

}  // namespace etp

// include/etp.h: the same check without a context or a device (what etp_copy_intervals runs first unless ETP_OPT_VALIDATE_INTERVALS is 0)
extern "C" etp_status etp_intervals_validate(const etp_interval* host_descs, int64_t n) { return etp::validate_intervals(host_descs, n, true); }

// EPLB-style expert replica placement after an elastic reshard (host-only).  PAPER.md:172-174, Fig. 4: "replicating hot-spot
// experts and adjusting routing ... schedules more expert replicas to the under-utilized GPU"; :235 (+29 % throughput with
// EPLB after an 8 -> 7 recovery); :249.  The paper names the strategy and gives no algorithm: the rule is DESIGN.md reading E1.
//
// Exact integer arithmetic: an expert with k <= 8 instances sends load / k to each, so every share is an integer multiple of
// 1/840 (840 = lcm(1..8)); rank loads are kept as integers in units of 1/840 token and updated incrementally, normalised
// loads S[r] / capacity[r] are compared by cross-multiplication in 128 bits.
#include <algorithm>
#include <vector>

#include "etp_internal.h"

namespace {
constexpr int kMaxInstances = 8;
constexpr int64_t kScale = 840;
typedef __int128 i128;

struct Frac {   // S / c with c > 0
    int64_t s, c;
};
inline bool less(const Frac& a, const Frac& b) { return (i128)a.s * b.c < (i128)b.s * a.c; }

struct State {
    int32_t E, R;
    const int64_t *load, *cap;
    std::vector<std::vector<int32_t>> inst;   // ranks per expert, home first
    std::vector<int64_t> S;                   // scaled load per rank
    std::vector<int32_t> free_slots;

    Frac worst(int32_t* where) const {
        Frac m{0, 1};
        int32_t at = -1;
        for (int32_t r = 0; r < R; ++r) {
            if (cap[r] <= 0) continue;
            const Frac f{S[r], cap[r]};
            if (at < 0 || less(m, f)) { m = f; at = r; }
        }
        if (where) *where = at;
        return m;
    }
    // move expert e from k to k + 1 instances, the new one on rank d (sign = +1), or back (sign = -1)
    void add_instance(int32_t e, int32_t d) {
        const int64_t k = (int64_t)inst[e].size();
        const int64_t before = k ? load[e] * kScale / k : 0, after = load[e] * kScale / (k + 1);
        for (int32_t r : inst[e]) S[r] += after - before;
        S[d] += after;
        inst[e].push_back(d);
        --free_slots[d];
    }
    void drop_last_instance(int32_t e) {
        const int32_t d = inst[e].back();
        inst[e].pop_back();
        const int64_t k = (int64_t)inst[e].size();
        const int64_t with = load[e] * kScale / (k + 1), without = k ? load[e] * kScale / k : 0;
        S[d] -= with;
        for (int32_t r : inst[e]) S[r] += without - with;
        ++free_slots[d];
    }
};
}  // namespace

extern "C" etp_status etp_eplb_place(const int64_t* expert_load, const int32_t* home_rank, int32_t n_experts,
                                     const int64_t* rank_capacity, const int32_t* spare_slots, int32_t n_ranks,
                                     etp_replica* replicas_out, int32_t cap, int32_t* n_replicas) {
    if (!expert_load || !home_rank || !rank_capacity || !spare_slots || !n_replicas || n_experts < 0 || n_ranks < 1)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_place: bad arguments");
    if (cap > 0 && !replicas_out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_place: replicas_out is NULL");
    State st{n_experts, n_ranks, expert_load, rank_capacity, {}, {}, {}};
    st.inst.resize((size_t)n_experts);
    st.S.assign((size_t)n_ranks, 0);
    st.free_slots.assign(spare_slots, spare_slots + n_ranks);
    int64_t total = 0;
    for (int32_t r = 0; r < n_ranks; ++r)
        if (rank_capacity[r] < 0 || rank_capacity[r] > (int64_t(1) << 30) || spare_slots[r] < 0)
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_place: capacity in [0, 2^30] and spare_slots >= 0 (rank %d)", r);
    for (int32_t e = 0; e < n_experts; ++e) {
        if (expert_load[e] < 0 || expert_load[e] > (int64_t(1) << 40)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_place: load of expert %d outside [0, 2^40]", e);
        total += expert_load[e];
        const int32_t h = home_rank[e];
        if (h == -1) continue;
        if (h < 0 || h >= n_ranks || rank_capacity[h] <= 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_place: expert %d: home %d is not a usable rank", e, h);
        st.inst[e].push_back(h);
        st.S[h] += expert_load[e] * kScale;
    }
    if (total > (int64_t(1) << 50)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_eplb_place: total load too large");
    std::vector<etp_replica> made;

    // step 1: experts without a holder, hottest first, to the rank that is least loaded after taking them
    std::vector<int32_t> homeless;
    for (int32_t e = 0; e < n_experts; ++e)
        if (home_rank[e] == -1) homeless.push_back(e);
    std::stable_sort(homeless.begin(), homeless.end(), [&](int32_t a, int32_t b) { return expert_load[a] > expert_load[b]; });
    for (int32_t e : homeless) {
        int32_t best = -1;
        Frac bf{0, 1};
        for (int32_t d = 0; d < n_ranks; ++d) {
            if (rank_capacity[d] <= 0 || st.free_slots[d] <= 0) continue;
            const Frac f{st.S[d] + expert_load[e] * kScale, rank_capacity[d]};
            if (best < 0 || less(f, bf)) { best = d; bf = f; }
        }
        if (best < 0) ETP_FAIL(ETP_ERR_CAPACITY, "etp_eplb_place: no spare slot for expert %d, which has no holder", e);
        st.add_instance(e, best);
        made.push_back({e, best});
    }

    // step 2: replicate what sits on the hottest rank while that lowers the maximum normalised load
    for (;;) {
        int32_t hot = -1;
        const Frac cur = st.worst(&hot);
        if (hot < 0) break;
        int32_t be = -1, bd = -1;
        Frac bf = cur;
        for (int32_t e = 0; e < n_experts; ++e) {
            const std::vector<int32_t>& in = st.inst[e];
            if ((int)in.size() >= kMaxInstances || std::find(in.begin(), in.end(), hot) == in.end()) continue;
            for (int32_t d = 0; d < n_ranks; ++d) {
                if (rank_capacity[d] <= 0 || st.free_slots[d] <= 0 || std::find(in.begin(), in.end(), d) != in.end()) continue;
                st.add_instance(e, d);
                const Frac f = st.worst(nullptr);
                st.drop_last_instance(e);
                if (less(f, bf)) { bf = f; be = e; bd = d; }   // strict: the first (lowest e, then lowest d) minimum wins
            }
        }
        if (be < 0) break;   // nothing lowers the maximum
        st.add_instance(be, bd);
        made.push_back({be, bd});
    }
    *n_replicas = (int32_t)made.size();
    for (int32_t i = 0; i < std::min<int32_t>(cap, *n_replicas); ++i) replicas_out[i] = made[i];
    if (cap > 0 && *n_replicas > cap) ETP_FAIL(ETP_ERR_CAPACITY, "etp_eplb_place: %d replicas, room for %d", *n_replicas, cap);
    return ETP_OK;
}

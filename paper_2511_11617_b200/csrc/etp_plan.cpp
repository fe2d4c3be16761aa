// Host side of S1 (partition), S2 (Continuous Minimal Migration plan) and S6 (page-table rule).
// PAPER.md:94 (floor/ceil shard widths), Algorithm 1 (:98-140), Fig. 3 (:144), Eq. 1 (:154-160), :204 (Greedy / Full
// Reload comparison planners), :86 (LRU eviction).  Readings of garbled passages: DESIGN.md "Readings" C1-C7, K5.
#include <stdarg.h>
#include <stdio.h>

#include <algorithm>
#include <map>
#include <set>

#include "etp_internal.h"

namespace etp {
static thread_local char g_err[512] = "";
volatile unsigned long long* g_wait_fault_host = nullptr;
void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    int n = vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    // a kernel that gave up on a starved barrier left a record in host memory (etp_wait.cuh): every error after it says so
    volatile unsigned long long* r = g_wait_fault_host;
    if (r && r[0] == 0x4554504641554c54ull && n >= 0 && n < (int)sizeof(g_err) - 1) {
        static const char* const family[] = {"?", "interval copy (etp_copy.cu)", "shard linear (etp_linear.cu)", "grouped linear (etp_linear_group.cu)",
                                             "MoE (etp_moe.cu)"};
        snprintf(g_err + n, sizeof(g_err) - (size_t)n,
                 " [device wait starved: %s kernel, block %llu thread %llu gave up on mbarrier 0x%llx parity %llu after %.1f s and trapped; the "
                 "CUDA context is lost]",
                 family[r[1] <= 4 ? r[1] : 0], r[2], r[3], r[4], r[5], (double)r[6] * 1e-9);
    }
}
}  // namespace etp

extern "C" const char* etp_last_error(void) { return etp::g_err; }
extern "C" const char* etp_version(void) { return "etp 0.1 sm_100a"; }

// ------------------------------------------------------------------------------------------------ S1
extern "C" etp_status etp_partition(etp_granularity g, int64_t total_units, int32_t parts, etp_split_policy policy,
                                    int64_t align_units, int64_t* bounds_out) {
    (void)g;  // label only
    if (!bounds_out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_partition: bounds_out is NULL");
    if (parts < 1 || total_units < 0 || align_units < 1)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_partition: parts=%d total_units=%lld align_units=%lld", parts,
                 (long long)total_units, (long long)align_units);
    if (total_units > (int64_t(1) << 40) || parts > (1 << 20))
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_partition: total_units <= 2^40 and parts <= 2^20 (64-bit product)");
    // widths are counted in groups of align_units; the last group may be short
    const int64_t groups = (total_units + align_units - 1) / align_units;
    if (groups < parts)
        ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_partition: %lld units (align %lld) over %d shards needs replication",
                 (long long)total_units, (long long)align_units, parts);
    int64_t edge = 0;  // in groups
    for (int32_t j = 0; j <= parts; ++j) {
        if (policy == ETP_SPLIT_FLOOR_BOUNDARY) {
            edge = (int64_t(j) * groups) / parts;  // Alg. 1 l.3-4: floor(j*H/M)
        } else if (policy == ETP_SPLIT_CEIL_FIRST) {
            // the first (groups mod parts) shards are one group wider
            const int64_t q = groups / parts, r = groups % parts;
            edge = int64_t(j) * q + std::min<int64_t>(j, r);
        } else {
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_partition: unknown policy %d", (int)policy);
        }
        bounds_out[j] = std::min(edge * align_units, total_units);
    }
    return ETP_OK;
}

// ------------------------------------------------------------------------------------------------ S2
namespace {
struct Span {
    int64_t b, e;
};

// Remove [b,e) from a sorted disjoint span list.
void carve(std::vector<Span>& open, int64_t b, int64_t e) {
    std::vector<Span> next;
    next.reserve(open.size() + 1);
    for (const Span& s : open) {
        if (e <= s.b || s.e <= b) {
            next.push_back(s);
        } else {
            if (s.b < b) next.push_back({s.b, b});
            if (e < s.e) next.push_back({e, s.e});
        }
    }
    open.swap(next);
}

void finish_stats(etp_plan* p, const std::vector<int64_t>& tb) {
    etp_plan_stats st{};
    for (const etp_task& t : p->tasks) {
        const int64_t n = t.end - t.begin;
        if (t.kind == ETP_KEEP) st.keep_units += n;
        else if (t.kind == ETP_TRANSFER) st.transfer_units += n;
        else st.reload_units += n;
    }
    st.total_units = p->total_units;
    st.n_tasks = (int64_t)p->tasks.size();
    // Eq. 1: Reload* = H - sum_{i alive} sum_j |[s_i,e_i) ∩ [u_j,v_j)|.  For overlapping (replicated)
    // sources the union is what can be reused, so count covered units once.
    std::vector<Span> covered;
    for (const etp_shard& s : p->old_layout)
        if (s.alive && s.begin < s.end) covered.push_back({s.begin, s.end});
    std::sort(covered.begin(), covered.end(), [](const Span& a, const Span& b) { return a.b < b.b; });
    int64_t reuse = 0, hi = 0;
    for (const Span& c : covered) {
        const int64_t b = std::max(c.b, hi), e = std::min(c.e, tb.back());
        if (b < e) reuse += e - b;
        hi = std::max(hi, c.e);
    }
    st.reload_lower_bound = p->total_units - reuse;
    p->stats = st;
}

// One target of Algorithm 1 for a given owner: intersect with the sources in the order of reading C7 (the owner itself, then
// ascending rank id) - or, with link costs (reading M2), ascending (cost of the link to the owner, rank id) - and subtract;
// what stays open is reloaded.  Appends the tasks when `tasks` is given; returns the weighted transfer cost of the target.
struct LinkCost {
    const int64_t* m = nullptr;   // [n][n], m[src * n + dst] per unit; NULL = every link costs 1
    int32_t n = 0;
    int64_t at(int32_t src, int32_t dst) const { return m ? m[(int64_t)src * n + dst] : 1; }
};

int64_t plan_target(etp_plan_mode mode, const std::vector<etp_shard>& alive, const etp_shard& own, int64_t tb0, int64_t tb1,
                    const LinkCost& lc, std::vector<etp_task>* tasks) {
    const int32_t owner = own.rank;
    std::vector<Span> open;
    if (tb0 < tb1) open.push_back({tb0, tb1});
    int64_t cost = 0;
    if (mode != ETP_PLAN_FULL_RELOAD) {
        std::vector<const etp_shard*> order;
        for (const etp_shard& s : alive)
            if (s.rank != owner) order.push_back(&s);
        if (lc.m)
            std::stable_sort(order.begin(), order.end(), [&](const etp_shard* a, const etp_shard* b) { return lc.at(a->rank, owner) < lc.at(b->rank, owner); });
        order.insert(order.begin(), &own);
        for (const etp_shard* s : order) {
            const bool self = s->rank == owner;
            if (mode == ETP_PLAN_GREEDY && !self) continue;  // no cross-device transfer for gaps
            std::vector<Span> hits;
            for (const Span& o : open) {
                const int64_t b = std::max(o.b, s->begin), e = std::min(o.e, s->end);  // Alg. 1 l.10
                if (b < e) hits.push_back({b, e});
            }
            for (const Span& h : hits) {
                if (tasks) tasks->push_back({self ? ETP_KEEP : ETP_TRANSFER, s->rank, owner, 0, h.b, h.e});  // l.11-12, C1, C4
                if (!self) cost += (h.e - h.b) * lc.at(s->rank, owner);
                carve(open, h.b, h.e);                                                                     // l.13
            }
        }
    }
    if (tasks)
        for (const Span& o : open) tasks->push_back({ETP_RELOAD, -1, owner, 0, o.b, o.e});  // l.17-18, C2, C5
    return cost;
}

// ETP_PLAN_MIGRATION_AWARE (readings M1, M2; an extension, PAPER.md:160 minimises only the reload volume and
// :247/:257 leave transfer cost and "link reachability and cost weighting" to future work).  The reload volume does not depend
// on who owns what, so the search minimises the (link-weighted) TRANSFER cost  sum_j cost(target j owned by owner(j))  over
// injective owner choices and, when the bounds are free, over every placement of the ceil(H/M)-wide shards.  Assignment by
// dynamic programming over subsets of alive ranks (f[mask] = least cost of targets popcount(mask).. with the ranks in mask
// taken); ties go to the lexicographically smallest (bounds, owners) - bounds vectors are visited in lexicographic order and
// an equal score never replaces the incumbent; the owners are rebuilt front to back taking the smallest rank that still reaches f.
constexpr int kMaxAliveMigrationAware = 10;
constexpr int64_t kNoAssignment = INT64_MAX;

int64_t best_owners(const std::vector<etp_shard>& alive, const std::vector<int64_t>& tb, int M, const LinkCost& lc, std::vector<int>* owners) {
    const int n = (int)alive.size();
    std::vector<int64_t> cost((size_t)M * n);
    for (int j = 0; j < M; ++j)
        for (int i = 0; i < n; ++i) cost[(size_t)j * n + i] = plan_target(ETP_PLAN_CMM, alive, alive[i], tb[j], tb[j + 1], lc, nullptr);
    std::vector<int64_t> f(size_t(1) << n, kNoAssignment);
    for (int64_t mask = (int64_t(1) << n) - 1; mask >= 0; --mask) {
        const int j = __builtin_popcountll((unsigned long long)mask);
        if (j > M) continue;
        if (j == M) { f[mask] = 0; continue; }
        int64_t best = kNoAssignment;
        for (int i = 0; i < n; ++i)
            if (!(mask >> i & 1) && f[mask | (int64_t(1) << i)] != kNoAssignment)
                best = std::min(best, cost[(size_t)j * n + i] + f[mask | (int64_t(1) << i)]);
        f[mask] = best;
    }
    owners->assign(M, 0);
    int64_t mask = 0;
    for (int j = 0; j < M; ++j)
        for (int i = 0; i < n; ++i)
            if (!(mask >> i & 1) && f[mask | (int64_t(1) << i)] != kNoAssignment && cost[(size_t)j * n + i] + f[mask | (int64_t(1) << i)] == f[mask]) {
                (*owners)[j] = i;
                mask |= int64_t(1) << i;
                break;
            }
    return f[0];
}

etp_status choose_layout(const std::vector<etp_shard>& alive, int64_t H, int M, bool bounds_fixed, const LinkCost& lc,
                         std::vector<int64_t>* tb, std::vector<int>* owner_idx) {
    if ((int)alive.size() > kMaxAliveMigrationAware)
        ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_plan_create: the migration-aware search is limited to %d alive ranks", kMaxAliveMigrationAware);
    if (bounds_fixed) {
        best_owners(alive, *tb, M, lc, owner_idx);
        return ETP_OK;
    }
    if (H < M) ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_plan_create: %lld units over %d shards needs replication", (long long)H, M);
    const int64_t q = H / M;
    const int r = int(H % M);
    // width vectors with exactly r wide shards in lexicographic order (narrow before wide at the first difference)
    std::vector<int> wide(M, 0);
    for (int j = M - r; j < M; ++j) wide[j] = 1;   // lexicographically smallest: the wide shards last
    int64_t best_cost = kNoAssignment;
    std::vector<int64_t> cand(M + 1);
    std::vector<int> own;
    do {
        cand[0] = 0;
        for (int j = 0; j < M; ++j) cand[j + 1] = cand[j] + q + wide[j];
        const int64_t k = best_owners(alive, cand, M, lc, &own);
        if (k < best_cost) {
            best_cost = k;
            *tb = cand;
            *owner_idx = own;
        }
    } while (std::next_permutation(wide.begin(), wide.end()));
    return ETP_OK;
}
}  // namespace

extern "C" etp_status etp_plan_create(etp_plan_mode mode, const etp_shard* old_layout, int32_t n_old,
                                      const int64_t* target_bounds, int32_t M, etp_plan** out) {
    return etp_plan_create_weighted(mode, old_layout, n_old, target_bounds, M, nullptr, 0, out);
}

extern "C" etp_status etp_plan_create_weighted(etp_plan_mode mode, const etp_shard* old_layout, int32_t n_old,
                                               const int64_t* target_bounds, int32_t M, const int64_t* link_cost,
                                               int32_t n_cost_ranks, etp_plan** out) {
    if (!out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create: out is NULL");
    *out = nullptr;
    if (!old_layout || n_old < 1) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create: empty old layout");
    if (mode != ETP_PLAN_CMM && mode != ETP_PLAN_GREEDY && mode != ETP_PLAN_FULL_RELOAD && mode != ETP_PLAN_MIGRATION_AWARE)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create: unknown mode %d", (int)mode);
    int64_t H = 0;
    std::set<int32_t> seen;
    std::vector<etp_shard> alive;
    for (int32_t i = 0; i < n_old; ++i) {
        const etp_shard& s = old_layout[i];
        if (s.begin < 0 || s.end < s.begin)
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create: shard %d has interval [%lld,%lld)", i, (long long)s.begin,
                     (long long)s.end);
        if (s.rank < 0 || !seen.insert(s.rank).second)
            ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create: rank id %d negative or repeated", s.rank);
        H = std::max(H, s.end);  // Alg. 1 l.1: H over ALL shards, alive or not
        if (s.alive) alive.push_back(s);
    }
    std::sort(alive.begin(), alive.end(), [](const etp_shard& a, const etp_shard& b) { return a.rank < b.rank; });
    if (M < 1 || M > (int32_t)alive.size())
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create: M=%d must be in 1..%d (number of alive ranks)", M,
                 (int)alive.size());
    std::vector<int64_t> tb(M + 1);
    if (target_bounds) {
        for (int32_t j = 0; j <= M; ++j) tb[j] = target_bounds[j];
        bool ok = tb[0] == 0 && tb[M] == H;
        for (int32_t j = 0; j < M && ok; ++j) ok = tb[j] <= tb[j + 1];
        if (!ok) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create: target bounds must tile [0,%lld)", (long long)H);
    } else {
        for (int32_t j = 0; j <= M; ++j) tb[j] = (int64_t(j) * H) / M;  // Alg. 1 l.2-5
    }

    // owner_idx[j] = index into `alive` of the rank that holds target j.  Reading C3: the j-th alive rank in ascending id.
    std::vector<int> owner_idx(M);
    for (int32_t j = 0; j < M; ++j) owner_idx[j] = j;
    LinkCost lc;
    if (link_cost) {
        if (mode != ETP_PLAN_MIGRATION_AWARE) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create_weighted: link costs belong to ETP_PLAN_MIGRATION_AWARE");
        for (const etp_shard& s : alive)
            if (s.rank >= n_cost_ranks) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create_weighted: rank %d outside the %d x %d cost matrix", s.rank, n_cost_ranks, n_cost_ranks);
        for (int64_t k = 0; k < (int64_t)n_cost_ranks * n_cost_ranks; ++k)
            if (link_cost[k] < 0 || link_cost[k] > (int64_t(1) << 20)) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_create_weighted: link costs must be in [0, 2^20]");
        lc.m = link_cost;
        lc.n = n_cost_ranks;
    }
    if (mode == ETP_PLAN_MIGRATION_AWARE) ETP_TRY(choose_layout(alive, H, M, target_bounds != nullptr, lc, &tb, &owner_idx));

    etp_plan* p = new (std::nothrow) etp_plan();
    if (!p) ETP_FAIL(ETP_ERR_NOMEM, "etp_plan_create: out of memory");
    p->mode = mode;
    p->total_units = H;
    p->old_layout.assign(old_layout, old_layout + n_old);
    for (int32_t j = 0; j < M; ++j) {
        const etp_shard& own = alive[owner_idx[j]];
        p->new_layout.push_back({own.rank, 1, tb[j], tb[j + 1]});
        plan_target(mode, alive, own, tb[j], tb[j + 1], lc, &p->tasks);
    }
    std::stable_sort(p->tasks.begin(), p->tasks.end(), [](const etp_task& a, const etp_task& b) {
        return a.dst_rank != b.dst_rank ? a.dst_rank < b.dst_rank : a.begin < b.begin;
    });
    finish_stats(p, tb);
    *out = p;
    return ETP_OK;
}

extern "C" etp_status etp_cmm_plan(const etp_shard* old_layout, int32_t n_old, const int64_t* target_bounds, int32_t M,
                                   etp_plan** out) {
    return etp_plan_create(ETP_PLAN_CMM, old_layout, n_old, target_bounds, M, out);
}

extern "C" etp_status etp_plan_tasks(const etp_plan* plan, etp_task* out, int64_t cap, int64_t* n_out) {
    if (!plan || !n_out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_tasks: NULL argument");
    *n_out = (int64_t)plan->tasks.size();
    if (cap > 0 && !out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_tasks: out is NULL");
    const int64_t n = std::min<int64_t>(cap, *n_out);
    for (int64_t i = 0; i < n; ++i) out[i] = plan->tasks[i];
    return ETP_OK;
}

extern "C" etp_status etp_plan_new_layout(const etp_plan* plan, etp_shard* out, int32_t cap, int32_t* n_out) {
    if (!plan || !n_out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_new_layout: NULL argument");
    *n_out = (int32_t)plan->new_layout.size();
    if (cap > 0 && !out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_new_layout: out is NULL");
    for (int32_t i = 0; i < std::min(cap, *n_out); ++i) out[i] = plan->new_layout[i];
    return ETP_OK;
}

extern "C" etp_status etp_plan_get_stats(const etp_plan* plan, etp_plan_stats* out) {
    if (!plan || !out) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_get_stats: NULL argument");
    *out = plan->stats;
    return ETP_OK;
}

extern "C" etp_status etp_plan_slab_span(const etp_plan* plan, int32_t rank, int64_t* first_unit, int64_t* span_units) {
    if (!plan || !first_unit || !span_units) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_slab_span: NULL argument");
    bool found = false, any = false;
    int64_t lo = 0, hi = 0;
    auto take = [&](const etp_shard& s) {
        if (s.rank != rank) return;
        found = true;
        if (s.begin >= s.end) return;
        lo = any ? std::min(lo, s.begin) : s.begin;
        hi = any ? std::max(hi, s.end) : s.end;
        any = true;
    };
    for (const etp_shard& s : plan->old_layout) take(s);
    for (const etp_shard& s : plan->new_layout) take(s);
    if (!found) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_plan_slab_span: rank %d is in neither layout", rank);
    *first_unit = lo;
    *span_units = hi - lo;
    return ETP_OK;
}

extern "C" void etp_plan_free(etp_plan* plan) { delete plan; }

// ------------------------------------------------------------------------------------------------ S6 page table
extern "C" etp_status etp_page_table_rewrite(etp_page_table* pt, int32_t block_size, int32_t new_block_budget,
                                             int32_t* evicted_out, int32_t* n_evicted, int32_t* pairs_out,
                                             int64_t pairs_cap, int64_t* n_pairs) {
    if (!pt || !n_evicted || !n_pairs) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_page_table_rewrite: NULL argument");
    if (block_size < 1 || new_block_budget < 0 || pt->n_seqs < 0 || pt->max_blocks < 0)
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_page_table_rewrite: bad sizes");
    if (pt->n_seqs > 0 && (!pt->block_table || !pt->seq_lens || !pt->last_use))
        ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_page_table_rewrite: NULL table");
    const int32_t S = pt->n_seqs, W = pt->max_blocks;
    std::vector<int32_t> need(S);
    int64_t live = 0;
    for (int32_t s = 0; s < S; ++s) {
        if (pt->seq_lens[s] < 0) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_page_table_rewrite: negative seq_len");
        need[s] = (pt->seq_lens[s] + block_size - 1) / block_size;
        if (need[s] > W) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_page_table_rewrite: seq %d needs %d blocks > max_blocks %d", s, need[s], W);
        for (int32_t i = 0; i < need[s]; ++i)
            if (pt->block_table[(int64_t)s * W + i] < 0)
                ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_page_table_rewrite: seq %d logical block %d unmapped", s, i);
        live += need[s];
    }
    // (i) LRU eviction: coldest first (smallest last_use, tie -> smaller index)
    std::vector<int32_t> by_age;
    for (int32_t s = 0; s < S; ++s)
        if (need[s] > 0) by_age.push_back(s);
    std::stable_sort(by_age.begin(), by_age.end(),
                     [&](int32_t a, int32_t b) { return pt->last_use[a] < pt->last_use[b]; });
    std::vector<char> gone(S, 0);
    int32_t n_ev = 0;
    for (size_t k = 0; k < by_age.size() && live > new_block_budget; ++k) {
        const int32_t v = by_age[k];
        gone[v] = 1;
        live -= need[v];
        if (evicted_out) evicted_out[n_ev] = v;
        ++n_ev;
    }
    *n_evicted = n_ev;
    // (ii) relocation of surviving blocks with id >= budget to the smallest free ids
    std::vector<char> taken((size_t)std::max<int32_t>(new_block_budget, 0), 0);
    for (int32_t s = 0; s < S; ++s) {
        if (gone[s]) continue;
        for (int32_t i = 0; i < need[s]; ++i) {
            const int32_t b = pt->block_table[(int64_t)s * W + i];
            if (b < new_block_budget) {
                if (taken[b]) ETP_FAIL(ETP_ERR_INVALID_ARG, "etp_page_table_rewrite: block %d mapped twice", b);
                taken[b] = 1;
            }
        }
    }
    int32_t cursor = 0;
    int64_t np = 0;
    for (int32_t s = 0; s < S; ++s) {
        int32_t* row = pt->block_table + (int64_t)s * W;
        if (gone[s]) {
            for (int32_t i = 0; i < W; ++i) row[i] = -1;
            continue;
        }
        for (int32_t i = 0; i < need[s]; ++i) {
            const int32_t old_id = row[i];
            int32_t new_id = old_id;
            if (old_id >= new_block_budget) {
                while (cursor < new_block_budget && taken[cursor]) ++cursor;
                if (cursor >= new_block_budget) ETP_FAIL(ETP_ERR_CAPACITY, "etp_page_table_rewrite: no free block below the budget");
                new_id = cursor;
                taken[cursor] = 1;
                row[i] = new_id;
            }
            if (pairs_out && np < pairs_cap) {
                pairs_out[2 * np] = old_id;
                pairs_out[2 * np + 1] = new_id;
            }
            ++np;
        }
    }
    *n_pairs = np;
    if (pairs_out && np > pairs_cap) ETP_FAIL(ETP_ERR_CAPACITY, "etp_page_table_rewrite: pairs_out too small (%lld > %lld)", (long long)np, (long long)pairs_cap);
    return ETP_OK;
}

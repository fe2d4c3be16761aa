/* CPU ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Shares nothing with the CUDA library.
 *
 * Element-by-element application of a migration plan ("parameter re-assignment/reloading
 * primitive" and "KV-cache operators that support variable-length shards"; :152 Transfer / Reload tasks).
 * Plain C, no intrinsics, no blocking, one byte at a time, in the order DESIGN.md "O-A" states:
 *     TRANSFER: out[dst][slot_dst(u)][e] = snap[src][slot_src(u)][e]
 *     RELOAD  : out[dst][slot_dst(u)][e] = host_image[u - host_unit0][e]
 *     KEEP    : nothing
 * Sources are always read from the pre-reshard snapshot (snapshot semantics, reading L4).
 * Slot addressing (reading L3): unit u of a rank lives at slot (u - anchor) mod cap of that rank's slab.
 */
#include <stdint.h>

#define ORACLE_KEEP 0
#define ORACLE_TRANSFER 1
#define ORACLE_RELOAD 2

static int64_t slot_of(int64_t u, int64_t anchor, int64_t cap) {
    int64_t d = (u - anchor) % cap;
    if (d < 0) d += cap;
    return d;
}

int64_t oracle_slot(int64_t u, int64_t anchor, int64_t cap) { return slot_of(u, anchor, cap); }

/* One parameter task over units [begin,end).  Returns bytes written. */
int64_t oracle_apply_param_task(int kind, int64_t begin, int64_t end, int64_t unit_bytes,
                                const uint8_t* snap_src, int64_t src_anchor, int64_t src_cap,
                                uint8_t* out_dst, int64_t dst_anchor, int64_t dst_cap,
                                const uint8_t* host_image, int64_t host_unit0) {
    int64_t written = 0;
    if (kind == ORACLE_KEEP) return 0;
    for (int64_t u = begin; u < end; ++u) {
        int64_t sd = slot_of(u, dst_anchor, dst_cap);
        if (kind == ORACLE_TRANSFER) {
            int64_t ss = slot_of(u, src_anchor, src_cap);
            for (int64_t e = 0; e < unit_bytes; ++e)
                out_dst[sd * unit_bytes + e] = snap_src[ss * unit_bytes + e];
        } else {
            for (int64_t e = 0; e < unit_bytes; ++e)
                out_dst[sd * unit_bytes + e] = host_image[(u - host_unit0) * unit_bytes + e];
        }
        written += unit_bytes;
    }
    return written;
}

/* Paged KV pool of one rank: [layer][K|V][block][token][slot][dim] (token-major, layout 0, reading K1)
 * or [layer][K|V][block][slot][token][dim] (head-major, layout 1).  Byte offset of one (token, head) fragment. */
static int64_t kv_off(int layout, int64_t l, int64_t c, int64_t b, int64_t t, int64_t slot,
                      int64_t n_blocks, int64_t block_size, int64_t heads, int64_t frag_bytes) {
    int64_t lcb = (l * 2 + c) * n_blocks + b;
    if (layout == 0) return ((lcb * block_size + t) * heads + slot) * frag_bytes;
    return ((lcb * heads + slot) * block_size + t) * frag_bytes;
}

/* One head task over heads [h_begin,h_end) and a list of live (old block id, new block id) pairs.
 * KEEP: same pool, copies only pairs whose id changed (relocation of kept heads, reading K5).
 * TRANSFER: snap_src pool (old id) -> out_dst pool (new id).
 * RELOAD: host backup = the dead rank's pool in the same layout with host_heads slots (slot = h - host_head0),
 *         indexed by the OLD block id (reading K4). */
int64_t oracle_apply_kv_task(int kind, int64_t h_begin, int64_t h_end, int layout,
                             int64_t n_layers, int64_t n_blocks, int64_t block_size, int64_t head_cap,
                             int64_t frag_bytes,
                             const uint8_t* snap_src, int64_t src_anchor,
                             uint8_t* out_dst, int64_t dst_anchor,
                             const uint8_t* host_backup, int64_t host_heads, int64_t host_head0,
                             const int32_t* old_ids, const int32_t* new_ids, int64_t n_pairs) {
    int64_t written = 0;
    for (int64_t p = 0; p < n_pairs; ++p) {
        int64_t bo = old_ids[p], bn = new_ids[p];
        if (kind == ORACLE_KEEP && bo == bn) continue;
        for (int64_t l = 0; l < n_layers; ++l)
            for (int64_t c = 0; c < 2; ++c)
                for (int64_t t = 0; t < block_size; ++t)
                    for (int64_t h = h_begin; h < h_end; ++h) {
                        int64_t d = kv_off(layout, l, c, bn, t, slot_of(h, dst_anchor, head_cap),
                                           n_blocks, block_size, head_cap, frag_bytes);
                        if (kind == ORACLE_RELOAD) {
                            int64_t s = kv_off(layout, l, c, bo, t, h - host_head0, n_blocks, block_size,
                                               host_heads, frag_bytes);
                            for (int64_t e = 0; e < frag_bytes; ++e) out_dst[d + e] = host_backup[s + e];
                        } else {
                            int64_t s = kv_off(layout, l, c, bo, t, slot_of(h, src_anchor, head_cap),
                                               n_blocks, block_size, head_cap, frag_bytes);
                            for (int64_t e = 0; e < frag_bytes; ++e) out_dst[d + e] = snap_src[s + e];
                        }
                        written += frag_bytes;
                    }
    }
    return written;
}

/* ---------------------------------------------------------------------------------------------------------------
 * All-cores leg of the CPU baseline (SURVEY.md 8(d) "Oracle timing": once on 1 core, once with an OpenMP parallel for
 * over tasks on all cores).  The SAME element-by-element functions above, called from a parallel loop over a job list
 * (one job = one task, or a sub-range of a task's units / live blocks so that the loop balances); jobs write disjoint
 * bytes (targets tile the unit space, live blocks are distinct), and sources are read from the snapshot only.
 * Built twice from this file: libetp_oracle.so (-O2; the pragma is ignored) and libetp_oracle_omp.so (-O2 -fopenmp). */
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

typedef struct {
    int64_t kind, begin, end, unit_bytes;
    const uint8_t* snap_src; int64_t src_anchor, src_cap;
    uint8_t* out_dst; int64_t dst_anchor, dst_cap;
    const uint8_t* host_image; int64_t host_unit0;
} oracle_param_job;

int64_t oracle_apply_param_jobs(const oracle_param_job* jobs, int64_t n_jobs) {
    int64_t written = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : written)
    for (int64_t j = 0; j < n_jobs; ++j) {
        const oracle_param_job* q = &jobs[j];
        written += oracle_apply_param_task((int)q->kind, q->begin, q->end, q->unit_bytes, q->snap_src, q->src_anchor, q->src_cap,
                                           q->out_dst, q->dst_anchor, q->dst_cap, q->host_image, q->host_unit0);
    }
    return written;
}

typedef struct {
    int64_t kind, h_begin, h_end, layout, n_layers, n_blocks, block_size, head_cap, frag_bytes;
    const uint8_t* snap_src; int64_t src_anchor;
    uint8_t* out_dst; int64_t dst_anchor;
    const uint8_t* host_backup; int64_t host_heads, host_head0;
    const int32_t* old_ids; const int32_t* new_ids; int64_t n_pairs;
} oracle_kv_job;

int64_t oracle_apply_kv_jobs(const oracle_kv_job* jobs, int64_t n_jobs) {
    int64_t written = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : written)
    for (int64_t j = 0; j < n_jobs; ++j) {
        const oracle_kv_job* q = &jobs[j];
        written += oracle_apply_kv_task((int)q->kind, q->h_begin, q->h_end, (int)q->layout, q->n_layers, q->n_blocks, q->block_size,
                                        q->head_cap, q->frag_bytes, q->snap_src, q->src_anchor, q->out_dst, q->dst_anchor,
                                        q->host_backup, q->host_heads, q->host_head0, q->old_ids, q->new_ids, q->n_pairs);
    }
    return written;
}

/* etp.h — C ABI of the B200-native Elastic-TP reshard library (libetp.so).
 *
 * The hot path of AnchorTP's state-preserving recovery (arxiv 2511.11617; citations are PAPER.md:line):
 * apply a Continuous Minimal Migration (CMM) plan — rewrite model parameters and a paged KV cache from an
 * N-rank unequal-width Elastic-TP layout into an M-rank one, moving only the intervals the plan says move,
 * with the host reload of the failed rank's bytes pipelined beside the device copies.
 * Every simulated TP rank is a separate allocation on ONE GPU; P2P is an intra-HBM copy.
 *
 * Conventions
 *  - plain C, no exceptions or aborts cross this boundary; every call returns etp_status (0 = OK) and
 *    etp_last_error() returns a thread-local message for the last failure on the calling thread.
 *  - the CALLER owns every data buffer (device slabs, KV pools, host image, page table, X/Y); pointers are raw
 *    (torch.Tensor.data_ptr()) and streams are raw cudaStream_t (torch.cuda.Stream.cuda_stream), passed as void*.
 *    "device" / "host" / "pinned host" is stated per argument.
 *  - the LIBRARY owns plan objects, descriptor arenas (pinned + device) and its events; they
 *    live in an etp_ctx / etp_plan and are freed by the matching _destroy / _free.
 *  - device calls are ASYNCHRONOUS: work is enqueued on the given streams and is complete when the caller has
 *    synchronised BOTH streams.  Data buffers must stay valid until then.  A ctx may be used from one host
 *    thread at a time.
 *  - all byte sizes are int64_t; every base pointer and unit_bytes must be a multiple of 16 (else
 *    ETP_ERR_ALIGNMENT).  Rank ids are 0-based (Fig. 3 of the paper is 1-based).
 *  - there is no CPU fallback: without a CUDA device every device call fails with ETP_ERR_CUDA.
 */
#ifndef ETP_H_
#define ETP_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    ETP_OK = 0,
    ETP_ERR_INVALID_ARG = 1,
    ETP_ERR_ALIGNMENT = 2,
    ETP_ERR_CAPACITY = 3,     /* a new shard does not fit its slab (width > cap_units) / output array too small */
    ETP_ERR_NO_SOURCE = 4,    /* a RELOAD task but no host image / backup covering it */
    ETP_ERR_UNSUPPORTED = 5,  /* fewer units than shards; cyclic write-after-read hazard; bad dtype */
    ETP_ERR_CUDA = 6,
    ETP_ERR_NOMEM = 7
} etp_status;

typedef struct etp_ctx etp_ctx;
typedef struct etp_plan etp_plan;

/* ------------------------------------------------------------------------------------------------ context */

/* Create a context on CUDA device `device`.  `staging_bytes` must be >= 0 and is otherwise RESERVED: the KV reload
 * pipeline needs no device staging ring (the copy kernel reads the pinned backup over the host link and writes the
 * head-strided fragments in place), so nothing is allocated for it.  Fails with ETP_ERR_CUDA if the
 * device is missing or is not compute capability 10.x. */
etp_status etp_ctx_create(int device, int64_t staging_bytes, etp_ctx** out);
void etp_ctx_destroy(etp_ctx* ctx);

/* Multi-device (SURVEY.md 8(e), 8(f) #1; PAPER.md:64 "P2P direct access over high-speed interconnects", :162-166 execution
 * scheduler).  A ctx over n_devices LOGICAL devices: devices[i] is the CUDA device of logical device i; several logical
 * devices may name the same CUDA device (that is how the partitioned path is exercised on a one-GPU box).  Peer access is
 * enabled between every pair of distinct CUDA devices (ETP_ERR_UNSUPPORTED if the hardware cannot).  etp_reshard_params and
 * etp_reshard_kv then PARTITION THEIR WORK BY DESTINATION: logical device d runs, on its own library-owned streams, one launch
 * of the copy kernel per hazard phase that writes only memory of the ranks mapped to d and pulls its incoming intervals
 * through peer-mapped source pointers, plus the reloads of those ranks over its own host link; hazard phases are ordered
 * across devices with events; the caller's copy / reload streams (streams of devices[0]) are forked from and joined back
 * to, so "complete when both streams are synchronised" still holds.  No collective is involved.
 *
 * etp_ctx_set_rank_devices: device_of_rank[r] = the logical device whose memory holds rank r's slabs and KV pool, or -1 for
 * a rank that ANOTHER PROCESS writes (one process per GPU: its slabs are still valid SOURCES here if the caller passes
 * pointers this process can read, e.g. CUDA-IPC mappings, but no byte of it is written by this ctx; those bytes are counted
 * in etp_reshard_report.remote_bytes).  Every process lowers the same plan and therefore sees the same hazard phases; with
 * more than one phase in a multi-process job the caller runs the phases one by one (ETP_OPT_ONLY_PHASE) with a barrier of
 * its own in between.  Default (never called, or n_ranks = 0): every rank on logical device 0.
 * etp_ctx_device_report: what the last call enqueued on one logical device (bytes by destination, launches, memcpys). */
etp_status etp_ctx_create_multi(const int32_t* devices, int32_t n_devices, etp_ctx** out);
etp_status etp_ctx_set_rank_devices(etp_ctx* ctx, const int32_t* device_of_rank, int32_t n_ranks);
const char* etp_last_error(void);
/* library version string, e.g. "etp 0.1 sm_100a" (static storage) */
const char* etp_version(void);

typedef enum {
    ETP_OPT_SKIP_D2D = 0,        /* 1: do not launch the device-copy kernel (time pipeline (b) alone)            */
    ETP_OPT_SKIP_RELOAD = 1,     /* 1: do not issue reloads (time kernel (a) alone)                              */
    ETP_OPT_TMA_MIN_BYTES = 2,   /* contiguous intervals >= this go to the cp.async.bulk path (default 32768);
                                    INT64_MAX disables the TMA path, 0 sends everything 16-B aligned to it       */
    ETP_OPT_LDG_STEALS_BULK = 3, /* 1 (default 0): vector-copy warps also drain the bulk queue when theirs is empty */
    ETP_OPT_RELOAD_CHUNK_BYTES = 4, /* max bytes per cudaMemcpyAsync of the reload pipeline (default 64 MiB)     */
    ETP_OPT_RESERVED_5 = 5,      /* ignored (round 1 reserved it for a staged KV reload that was never built: the
                                    zero-copy gather already runs at the speed of the host link)                   */
    ETP_OPT_GRID_CTAS = 6,       /* persistent grid size; 0 (default) = number of SMs                            */
    ETP_OPT_GATHER_CTAS = 7,     /* CTAs of the zero-copy gather launch on the reload stream (default 16)        */
    ETP_OPT_TIME_KERNELS = 8,    /* 1 (default 0): bracket every launch of the copy kernel on the copy stream with CUDA
                                    events (on that stream) so that etp_ctx_kernel_time can report device durations   */
    ETP_OPT_LINEAR_CTA_PAIR = 9, /* 1 (default): etp_shard_linear at > 64 tokens runs CTA pairs (tcgen05 cta_group::2,
                                    256 out features x 256 tokens per pair) unless single-CTA tiles need fewer rounds of
                                    the persistent grid, and a partial last round of a row-parallel linear is cut along
                                    K over the idle pairs (fp32 partials summed in range order); 256 / 128: always
                                    pairs, with that token tile, no tail split; 0: always single-CTA 128 x 256 tiles  */
    ETP_OPT_VALIDATE_INTERVALS = 10, /* 1 (default): etp_copy_intervals checks on the host that the destinations are mutually
                                    disjoint and disjoint from every source (radix sorts of both sides, O(n)) and returns
                                    ETP_ERR_INVALID_ARG before anything is enqueued; 0: trust the caller                   */
    ETP_OPT_LINEAR_PDL = 11,     /* 1 (default): launches of the <= 64-token shard-linear kernel carry the programmatic-stream-
                                    serialization attribute: their prologue and first ring of weight tiles overlap the tail of the
                                    previous kernel of the stream (griddepcontrol; X, Y and the workspace are only touched after
                                    griddepcontrol.wait, the WEIGHT tiles before it); 0: plain stream order.  The first such launch
                                    after a call of this library that writes slabs on the same stream (etp_reshard_params / _kv,
                                    etp_eplb_apply, etp_copy_intervals) is sent without the attribute, so it sees the new weights.
                                    A caller that writes slabs by other means (its own kernels, cudaMemcpyAsync) directly before a
                                    <= 64-token linear on the same stream must set this option to 0 for that launch or put an
                                    event / another kernel in between                                                      */
    ETP_OPT_LINEAR_RING = 12,    /* read by etp_linear_prepare: 0 = one CTA per SM with the full shared-memory ring; 1 = two CTAs per SM
                                    with half the ring each (one keeps streaming while the other is in its prologue or tail);
                                    2 (default) = two per SM unless the group streams >= 200 weight chunks (3.2 MiB) per SM      */
    ETP_OPT_ONLY_PHASE = 13,     /* 0 (default): a call runs every hazard phase, ordered by events; k > 0: only phase k - 1 is
                                    enqueued (multi-process jobs: the caller puts its own barrier between the phases).  Every
                                    phase call must be given the same arguments; etp_reshard_kv therefore does NOT rewrite
                                    pt->block_table when k > 0 (see there)                                                    */
    ETP_OPT_MOE_CTA_PAIR = 14,   /* 1 (default): the grouped MoE kernels run CTA pairs (tcgen05 cta_group::2, 256 out features x up to
                                    256 routed rows per pair, each CTA staging half of the rows) when the instances carry enough rows
                                    for >= 128-row tiles; 2: always; 0: never (single-CTA 128-feature tiles)                  */
    ETP_OPT_SMALL_STAGED = 15,   /* 1 (default): in a launch of the copy kernel without bulk (>= TMA_MIN_BYTES) intervals, batches of small
                                    intervals are staged through the idle shared-memory ring with per-lane cp.async.bulk copies (more
                                    bytes in flight than the register path allows); 0: always the register path                    */
    ETP_OPT__COUNT
} etp_option;
etp_status etp_ctx_set_option(etp_ctx* ctx, etp_option key, int64_t value);
etp_status etp_ctx_get_option(const etp_ctx* ctx, etp_option key, int64_t* value);
/* With ETP_OPT_TIME_KERNELS = 1: blocks until the copy-stream kernels of the LAST device call have finished and writes
 * the sum of their device durations (CUDA events recorded on the launching stream, milliseconds) and their count.
 * ms_out / n_out: host.  Without the option (or before any call) both are 0. */
etp_status etp_ctx_kernel_time(etp_ctx* ctx, double* ms_out, int32_t* n_out);

/* ------------------------------------------------------------------------------------------------ S1 partition
 * "some GPUs hold shard size floor(S/g_t) while others hold ceil(S/g_t)"; Algorithm 1 l.2-5
 * (PAPER.md:107-110): s_j = floor((j-1)H/M), e_j = floor(jH/M); Fig. 3 (:144): 1024 over 3 -> 0/341/682/1024. */
typedef enum {
    ETP_SPLIT_FLOOR_BOUNDARY = 0, /* bounds[j] = floor(j*S/M)  (the paper's formula; wide shards last) */
    ETP_SPLIT_CEIL_FIRST = 1      /* first S mod M shards get ceil(S/M)  (BASELINE.json config 2: heads 3/3/2) */
} etp_split_policy;
typedef enum { ETP_GRAN_HEAD = 0, ETP_GRAN_FFN = 1, ETP_GRAN_EXPERT = 2, ETP_GRAN_VOCAB = 3 } etp_granularity; /* label only */

/* Host-only.  Writes parts+1 non-decreasing bounds, bounds[0] = 0, bounds[parts] = total_units, into bounds_out
 * (host, caller-owned, parts+1 entries).  align_units >= 1: every interior bound is a multiple of it.
 * ETP_ERR_UNSUPPORTED if ceil(total_units/align_units) < parts (replication is out of scope). */
etp_status etp_partition(etp_granularity g, int64_t total_units, int32_t parts, etp_split_policy policy,
                         int64_t align_units, int64_t* bounds_out);

/* ------------------------------------------------------------------------------------------------ S2 CMM plan
 * Algorithm 1: Require {(gpu_i, s_i, e_i, alive_i)}, target GPU count M;
 * Ensure {(gpu_j, sources_j)}.  Intersections with surviving sources become Transfer tasks (Keep when the
 * source is the owner itself, Fig. 3 "keeps"); uncovered gaps become Reload tasks. */
typedef struct { int32_t rank; int32_t alive; int64_t begin, end; } etp_shard;   /* (gpu_i, alive_i, s_i, e_i) */
typedef enum { ETP_KEEP = 0, ETP_TRANSFER = 1, ETP_RELOAD = 2 } etp_task_kind;
typedef struct { int32_t kind; int32_t src_rank /* -1 for RELOAD */; int32_t dst_rank; int32_t reserved;
                 int64_t begin, end; } etp_task;
typedef struct { int64_t total_units, keep_units, transfer_units, reload_units,
                 reload_lower_bound /* Eq. 1 */, n_tasks; } etp_plan_stats;
typedef enum { ETP_PLAN_CMM = 0, ETP_PLAN_GREEDY = 1, ETP_PLAN_FULL_RELOAD = 2,
               ETP_PLAN_MIGRATION_AWARE = 3 /* Algorithm 1 with the owner of every target (and, when target_bounds is NULL,
                  the placement of the ceil(H/M)-wide shards) chosen to minimise the transferred units at the same minimal
                  reload volume; ties -> lexicographically smallest (bounds, owner ranks).  An extension (PAPER.md:160, :247:
                  the paper minimises reload only).  <= 10 alive ranks, else ETP_ERR_UNSUPPORTED.  The new layout is in
                  target order, not rank order. */ } etp_plan_mode;

/* Host-only.  old_layout: n_old entries (host), distinct rank ids, arbitrary intervals.  target_bounds: M+1 bounds
 * tiling [0,H), H = max end over ALL entries, or NULL for the floor formula.  Target j is owned by the j-th alive
 * rank in ascending rank id; M must be in 1..#alive.  Tasks are sorted by (dst_rank, begin).  *out is owned by the
 * library: release with etp_plan_free. */
etp_status etp_cmm_plan(const etp_shard* old_layout, int32_t n_old, const int64_t* target_bounds, int32_t M,
                        etp_plan** out);
/* same with the comparison planners of PAPER.md:204 / Table II (Greedy: no P2P for gaps; Full Reload: no reuse) and the
 * migration-aware extension */
etp_status etp_plan_create(etp_plan_mode mode, const etp_shard* old_layout, int32_t n_old,
                           const int64_t* target_bounds, int32_t M, etp_plan** out);
/* ETP_PLAN_MIGRATION_AWARE with a price per link (reading M2; "requires incorporating link
 * reachability and cost weighting into planning", :257): link_cost is a host array [n_cost_ranks][n_cost_ranks] of integers
 * in [0, 2^20], link_cost[src * n_cost_ranks + dst] = cost of moving ONE unit from rank src to rank dst (indexed by rank id).
 * The planner minimises sum(transferred units x link cost) at the same minimal reload volume; a unit held by several alive
 * ranks is taken from the cheapest link (tie: lower rank id).  link_cost = NULL is etp_plan_create (every link costs 1; on one
 * NVSwitch node the matrix is uniform and the plan is the unweighted one). */
etp_status etp_plan_create_weighted(etp_plan_mode mode, const etp_shard* old_layout, int32_t n_old,
                                    const int64_t* target_bounds, int32_t M, const int64_t* link_cost,
                                    int32_t n_cost_ranks, etp_plan** out);
/* copies up to cap tasks into out (host); *n_out = total number of tasks (call with cap = 0 to size) */
etp_status etp_plan_tasks(const etp_plan* plan, etp_task* out, int64_t cap, int64_t* n_out);
/* writes the M new shards (host, M entries), alive = 1 */
etp_status etp_plan_new_layout(const etp_plan* plan, etp_shard* out, int32_t cap, int32_t* n_out);
etp_status etp_plan_get_stats(const etp_plan* plan, etp_plan_stats* out);
/* PAPER.md:164 "a single pass pre-allocates all destination buffers": the union span of `rank`'s old and new interval
 * under this plan, [*first_unit, *first_unit + *span_units).  A slab with cap_units >= span_units (any anchor) holds both
 * without wrap-around collisions, so the plan lowers to a single hazard phase (L4/L5).  A rank that holds
 * nothing before and after gives span 0.  ETP_ERR_INVALID_ARG if the rank is in neither layout. */
etp_status etp_plan_slab_span(const etp_plan* plan, int32_t rank, int64_t* first_unit, int64_t* span_units);
void etp_plan_free(etp_plan* plan);

/* ------------------------------------------------------------------------------------------------ S3-S5 parameters
 * PAPER.md:96 "parameter re-assignment/reloading primitive"; :164-166 pre-allocation, overlap of reloads with P2P.
 *
 * Layout contract (L1-L7): a sharded tensor is [total_units][unit_bytes], each unit contiguous.  Rank r keeps
 * unit u at  slabs[r].base + ((u - anchor_unit) mod cap_units) * unit_bytes ; kept units never change address, a shard
 * may wrap.  Sources are read with SNAPSHOT semantics (as if every read happened before every write); when a write
 * would land on bytes another task still has to read, the library orders the copies in hazard phases.
 * Only bytes of TRANSFER and RELOAD tasks are written; everything else in a slab is left untouched. */
typedef struct { void* base /* device, 16-B aligned; NULL for a dead rank */; int64_t cap_units; int64_t anchor_unit; } etp_slab;
typedef struct {
    int64_t total_units, unit_bytes;
    const etp_slab* slabs;      /* host array indexed by rank id, n_ranks entries                                   */
    int32_t n_ranks;
    int32_t plan_index;         /* which of `plans` drives this tensor (one plan per granularity class)             */
    const void* host_image;     /* reload source, addressed by global unit: host_image + (u - host_unit0)*unit_bytes.
                                   PINNED HOST memory (copied by DMA on the reload stream) or DEVICE memory (then
                                   reloads are lowered into the device-copy kernel).  NULL only if no RELOAD task.  */
    int64_t host_unit0, host_units;
} etp_tensor;
typedef struct {
    int64_t d2d_bytes;          /* bytes moved device-to-device by TRANSFER tasks (and same-rank KV relocations)   */
    int64_t h2d_bytes;          /* bytes reloaded from pinned host memory                                          */
    int64_t reload_dev_bytes;   /* bytes reloaded from a device-resident image (moved by the copy kernel)          */
    int64_t kept_bytes;         /* bytes of KEEP tasks (never touched)                                             */
    int64_t n_jobs, n_units;    /* segment descriptors uploaded / work items the kernels derived from them         */
    int64_t n_memcpys;          /* cudaMemcpyAsync calls issued by the reload pipeline                             */
    int32_t n_phases;           /* hazard phases (1 = hazard-free)                                                 */
    int32_t n_kernel_launches;  /* launches of this library's kernels                                              */
    double lower_ms;            /* host time spent lowering + enqueueing                                           */
    int64_t remote_bytes;       /* TRANSFER + RELOAD bytes whose destination rank another process writes (rank map -1) */
} etp_reshard_report;
etp_status etp_ctx_device_report(etp_ctx* ctx, int32_t logical_device, etp_reshard_report* out);

/* tensors: host array.  plans: host array of n_plans plan handles.  copy_stream / reload_stream: cudaStream_t of the
 * ctx device (may be the same stream; NULL = legacy default stream).  report: host, may be NULL. */
etp_status etp_reshard_params(etp_ctx* ctx, const etp_tensor* tensors, int32_t n_tensors,
                              const etp_plan* const* plans, int32_t n_plans,
                              void* copy_stream, void* reload_stream, etp_reshard_report* report);

/* ------------------------------------------------------------------------------------------------ S3-S6 paged KV
 * PAPER.md:96 "the KV cache is localized by attention head-groups per token block ... KV-cache operators that support
 * variable-length shards"; :166 "the runtime KV cache and parameters share the same planning and task generation";
 * :86 LRU eviction when KV demand exceeds the budget. */
typedef enum { ETP_KV_TOKEN_MAJOR = 0 /* [block][token][slot][dim] */, ETP_KV_HEAD_MAJOR = 1 /* [block][slot][token][dim] */ } etp_kv_layout;
typedef struct {
    int32_t n_layers, n_blocks, block_size, head_cap /* slots per token */, head_dim, elem_bytes;
    int32_t layout;             /* etp_kv_layout                                                                    */
    int32_t n_ranks;
    void* const* pools;         /* host array [n_ranks] of device pointers (NULL for a dead rank);
                                   pool[r] = [layer][K|V][n_blocks][...layout...], head h at slot (h - head_anchor[r]) mod head_cap */
    const int64_t* head_anchor; /* host array [n_ranks]                                                             */
    const void* host_backup;    /* the dead rank's pool compacted to host_heads slots (slot = h - host_head0), same
                                   layout, indexed by the OLD physical block id.  Pinned host or device memory; NULL =>
                                   reload heads are left untouched and every live sequence is reported evicted.     */
    int32_t host_heads; int64_t host_head0;
} etp_kv_geometry;
typedef struct {
    int32_t n_seqs, max_blocks;
    int32_t* block_table;       /* host [n_seqs][max_blocks], in/out, -1 = none                                     */
    const int32_t* seq_lens;    /* host [n_seqs]                                                                    */
    const int64_t* last_use;    /* host [n_seqs], larger = more recent                                              */
} etp_page_table;

/* Host-only page-table rule (K5): (i) while live blocks > budget evict the sequence with the smallest last_use
 * (tie: smaller index), its row becomes -1; (ii) every surviving block with id >= budget moves, in ascending (seq, logical
 * index), to the smallest id < budget not used by a surviving block.  pairs_out (host, may be NULL, cap entries of
 * {old id, new id}) receives every surviving live block.  evicted_out: host [n_seqs]. */
etp_status etp_page_table_rewrite(etp_page_table* pt, int32_t block_size, int32_t new_block_budget,
                                  int32_t* evicted_out, int32_t* n_evicted,
                                  int32_t* pairs_out, int64_t pairs_cap, int64_t* n_pairs);

/* Rewrites the page table (above), then moves KV-head slices of every surviving live block according to head_plan
 * (unit = KV head): TRANSFER heads between pools, RELOAD heads from the backup, KEEP heads only when their block was
 * relocated.  Free blocks are never copied.
 * With ETP_OPT_ONLY_PHASE = k > 0 (phase-by-phase runs of a multi-process job) the call reports the evicted sequences but
 * leaves pt->block_table as it was: every phase call has to lower the plan from the ORIGINAL table (the {old, new} block
 * pairs come from it), and n_phases of the report tells how many calls there are.  After the last phase the caller obtains
 * the new table with etp_page_table_rewrite(pt, block_size, new_block_budget, ...), the same host-only rule this call applies. */
etp_status etp_reshard_kv(etp_ctx* ctx, const etp_kv_geometry* geom, etp_page_table* pt, const etp_plan* head_plan,
                          int32_t new_block_budget, int32_t* evicted_seqs_out, int32_t* n_evicted,
                          void* copy_stream, void* reload_stream, etp_reshard_report* report);

/* ------------------------------------------------------------------------------------------------ S7 shard linear
 * unequal-width sharding for linear layers.  Computes, on the sharded weight as it sits in the
 * slabs, Y[tokens][out_features] = X[tokens][in_features] · W^T with fp32 accumulation and one rounding to 16 bit:
 *   ETP_COL_PARALLEL: the weight is cut along out-features; w is stored [out][in]; rank r produces its columns of Y.
 *   ETP_ROW_PARALLEL: the weight is cut along in-features; w is stored transposed [in][out]; the rank partial sums
 *                     are accumulated in one fp32 accumulator in ascending unit order (no second pass).
 * w->unit_bytes = features_per_unit * (row length) * 2.  x, y: device, 16-B aligned, row-major, same dtype as w. */
typedef enum { ETP_COL_PARALLEL = 0, ETP_ROW_PARALLEL = 1 } etp_linear_mode;
typedef enum { ETP_BF16 = 0, ETP_FP16 = 1 } etp_dtype;
etp_status etp_shard_linear(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype,
                            const void* x, int64_t tokens, int64_t in_features, int64_t out_features,
                            const etp_tensor* w, const etp_shard* layout, int32_t n_shards,
                            int64_t features_per_unit, void* y, void* stream);

/* Several COLUMN-parallel linears that share X, in_features and the shard layout of their granularity class (q | k | v of the
 * attention class, gate | up of the FFN class) in ONE launch: at a few tokens a linear is a weight stream with a fixed cost of
 * several microseconds per launch, and a serving engine runs these projections as one GEMM anyway.  Every
 * linear keeps its own slabs and its own output y [tokens][out_features]; results are bitwise those of separate
 * etp_shard_linear calls only when no K split is chosen (the split count depends on the total width).  n_outs in 1..8, all
 * w->total_units equal; the rest as etp_shard_linear.  (At <= 64 tokens both calls run through a ctx-owned cache of prepared
 * groups, see etp_linear_prepare below.) */
typedef struct { const etp_tensor* w; int64_t out_features; int64_t features_per_unit; void* y; } etp_linear_out;
etp_status etp_shard_linear_multi(etp_ctx* ctx, etp_dtype dtype, const void* x, int64_t tokens, int64_t in_features,
                                  const etp_linear_out* outs, int32_t n_outs, const etp_shard* layout, int32_t n_shards,
                                  void* stream);

/* Prepared groups.  At a few tokens a shard linear is a weight stream whose cost is dominated by what does NOT
 * scale with the bytes: argument checks, tensor-map encoding, the launch ramp and the tail of a static grid.  etp_linear_prepare
 * does everything that depends only on the weights and the layout once (slot runs, TMA tensor maps, the K split of every linear,
 * a load-balanced assignment of work items to the SMs) and returns a plan; etp_linear_run then costs one kernel launch for the
 * WHOLE group at <= 64 tokens - the linears of a group are independent of each other (none reads another's output), may mix
 * column- and row-parallel modes and have their own x and y each - and one launch per linear above 64 tokens.  The plan keeps
 * copies of the descriptors (not of the weights): the slabs must stay where they were.  Results equal etp_shard_linear's up to
 * the fp32 summation order of the K split (column-parallel outputs stay bitwise independent of the shard layout, reading G3).
 * A plan belongs to its ctx and is used from one host thread at a time; runs on different streams may overlap (the split-K
 * workspace is per stream).  etp_linear_run needs the ctx alive; etp_linear_free is also safe after etp_ctx_destroy (it touches
 * only the plan's own device table). */
typedef struct etp_linear_plan etp_linear_plan;
typedef struct {
    int32_t mode;               /* etp_linear_mode                                                                    */
    int32_t reserved0;
    int64_t in_features, out_features;
    const etp_tensor* w;        /* as etp_shard_linear                                                                */
    const etp_shard* layout;    /* host array of n_shards entries                                                     */
    int32_t n_shards;
    int32_t reserved1;
    int64_t features_per_unit;
} etp_linear_spec;
typedef struct {
    int32_t n_linears, n_ctas;
    int64_t n_items;            /* (linear, 128-feature tile, K range) work items of the <= 64-token launch              */
    int64_t total_chunks;       /* 16-KiB weight chunks of the whole group                                              */
    int64_t max_cta_chunks;     /* ... of the most loaded CTA (balance = total_chunks / n_ctas / max_cta_chunks)          */
    int64_t n_split_tiles;      /* fp32 partial tiles of the K split                                                    */
    int32_t n_splits[8];        /* K splits per linear                                                                  */
} etp_linear_plan_stats;
/* lins: host array of n_lins (1..8) specs.  *out is owned by the library. */
etp_status etp_linear_prepare(etp_ctx* ctx, etp_dtype dtype, const etp_linear_spec* lins, int32_t n_lins, etp_linear_plan** out);
/* x, y: host arrays of n_lins device pointers (16-B aligned; x[l] is [tokens][in_features of l], y[l] is [tokens][out_features
 * of l]); several linears may share an x.  Asynchronous on `stream`. */
etp_status etp_linear_run(etp_linear_plan* plan, const void* const* x, int64_t tokens, void* const* y, void* stream);
etp_status etp_linear_plan_info(const etp_linear_plan* plan, etp_linear_plan_stats* out);
void etp_linear_free(etp_linear_plan* plan);

/* ------------------------------------------------------------------------------------------------ grouped MoE linear
 * SURVEY.md 8(f) #3, reading G5; PAPER.md:172-174 (experts are the unit of the expert-granularity plan).  One
 * launch computes, for every expert e,  Y_perm[r][:] = X_perm[r][:] . W_e^T  for its routed rows r in
 * [row_offsets[e], row_offsets[e+1]) on the expert matrices where the reshard left them.  w: total_units = n_experts, one
 * unit = one expert matrix of in_features x out_features 16-bit elements (unit_bytes = in x out x 2):
 *   ETP_COL_PARALLEL: stored [out][in] (gate, up);  ETP_ROW_PARALLEL: stored transposed [in][out] (down), in % 64 == 0.
 * x_perm [n_rows][in_features], y_perm [n_rows][out_features]: device, 16-B aligned, row-major, rows grouped by expert in
 * ascending expert id; row_offsets: HOST array of n_experts + 1 non-decreasing offsets starting at 0.  Routing, activation
 * and the weighted combine are the caller's.  fp32 accumulation, one rounding to 16 bit.  Asynchronous on `stream`; the work-item
 * table lives in a stream-ordered allocation, so calls on different streams of one ctx may overlap. */
etp_status etp_moe_linear(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x_perm,
                          const int64_t* row_offsets, int32_t n_experts, int64_t in_features, int64_t out_features,
                          const etp_tensor* w, const etp_shard* layout, int32_t n_shards, void* y_perm, void* stream);

/* The same with explicit expert INSTANCES (reading E1): after etp_eplb_place / etp_eplb_apply an expert may exist on
 * several ranks, each instance serving a slice of the expert's routed rows.  instances: host array; instance i multiplies rows
 * [row_begin, row_end) of x_perm by the expert matrix that sits in slot `slot` of rank `rank`'s slab (for the home instance
 * slot = (expert - anchor_unit) mod cap_units, for a replica the slot etp_eplb_apply returned).  Row ranges must be disjoint
 * and inside [0, n_rows); rows no instance covers are left untouched.  `expert` is informational. */
typedef struct { int32_t expert, rank; int64_t slot; int64_t row_begin, row_end; } etp_moe_instance;
etp_status etp_moe_linear_instances(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x_perm,
                                    const etp_moe_instance* instances, int32_t n_instances, int64_t n_rows, int32_t n_experts,
                                    int64_t in_features, int64_t out_features, const etp_tensor* w, void* y_perm, void* stream);
/* gate | up of a SwiGLU expert layer in ONE launch (reading G5): h_perm[r][:] = silu(W_gate,e x_perm[r]) * (W_up,e x_perm[r]),
 * fp32 accumulation, the activation in fp32, ONE rounding to 16 bit; X is read once and the two [rows][ffn] intermediates of
 * the separate launches never exist.  Both tensors column-parallel [ffn][in] per expert, slabs of the same geometry rank by
 * rank.  Either instances != NULL (as etp_moe_linear_instances; row_offsets / layout ignored) or row_offsets + layout (as
 * etp_moe_linear; n_rows ignored). */
etp_status etp_moe_gate_up(etp_ctx* ctx, etp_dtype dtype, const void* x_perm, const int64_t* row_offsets,
                           const etp_moe_instance* instances, int32_t n_instances, int64_t n_rows, int32_t n_experts,
                           int64_t in_features, int64_t ffn, const etp_tensor* w_gate, const etp_tensor* w_up,
                           const etp_shard* layout, int32_t n_shards, void* h_perm, void* stream);

/* ------------------------------------------------------------------------------------------------ EPLB-style placement
 * PAPER.md:172-174, Fig. 4, :235, :249 - "replicating hot-spot experts and adjusting routing"; after an unequal-width reshard
 * one GPU holds a smaller shard and "more idle compute capacity", and the planner "schedules more expert replicas to the
 * under-utilized GPU".  The rule is DESIGN.md reading E1 (the paper gives none).  Host-only, exact integer arithmetic.
 *   expert_load[e]   tokens routed to expert e (0 .. 2^40);  home_rank[e]: the rank that holds e (the expert plan), or -1 for
 *                    an expert without a holder (Fig. 4's recovered expert);
 *   rank_capacity[r] compute available for expert work on rank r (0 = dead rank, <= 2^30);  spare_slots[r]: free expert slots.
 * An expert with k instances (<= 8) serves load / k on each; L(r) = (sum of the shares on r) / capacity[r].  Step 1: holderless
 * experts, hottest first, go to the usable rank with a spare slot that is least loaded after taking them.  Step 2: while it
 * strictly lowers max L, add the instance (expert on the hottest rank -> rank with a spare slot) that minimises the new max L
 * (ties: lower expert id, then lower rank id).  replicas_out receives the new instances in creation order (call with cap = 0
 * to size).  Routing convention for etp_moe_linear_instances: instance j of k gets rows [floor(j n / k), floor((j+1) n / k))
 * of the expert's n routed rows, instances ordered home first, then replicas in creation order. */
typedef struct { int32_t expert, rank; } etp_replica;
etp_status etp_eplb_place(const int64_t* expert_load, const int32_t* home_rank, int32_t n_experts,
                          const int64_t* rank_capacity, const int32_t* spare_slots, int32_t n_ranks,
                          etp_replica* replicas_out, int32_t cap, int32_t* n_replicas);

/* Materialises replicas: for every replica (expert e -> rank d) the lowest spare slot of rank d's slab (a slot that holds no
 * unit of d's shard under `layout` and was not given to an earlier replica of this call) receives a copy of e's unit from its
 * home rank, in EVERY tensor of the class (e.g. gate, up, down of a layer; all must share total_units and, rank by rank, the
 * slab geometry, so a replica has ONE slot).  One launch of the interval-copy kernel on `stream`; slots_out[i] (host) = the
 * slot of replica i.  ETP_ERR_CAPACITY if a rank has no spare slot; ETP_ERR_INVALID_ARG if an (expert, rank) pair is listed twice or
 * the rank is the expert's home.  The spare slots are derived from `layout` alone: the call does not know what an EARLIER call put
 * into them, so pass ALL replicas of a layout in ONE call (a second call on the same layout reuses, i.e. overwrites, the same slots). */
etp_status etp_eplb_apply(etp_ctx* ctx, const etp_tensor* tensors, int32_t n_tensors, const etp_shard* layout, int32_t n_shards,
                          const etp_replica* replicas, int32_t n_replicas, int64_t* slots_out, void* stream);

/* ------------------------------------------------------------------------------------------------ microbenchmark entry
 * Copies n arbitrary intervals with the same persistent kernel (config 5b).  host_descs: host array (pageable: consumed before
 * the call returns; page-locked: read by DMA, must stay valid until `stream` is synchronised); src/dst: device, 16-B aligned;
 * bytes: multiple of 16.  From 32768 intervals on, the raw records are uploaded in chunks and lowered to work descriptors by
 * kernels on a library-owned stream while earlier chunks are being copied (one kernel launch per 262144 intervals).  Destinations must be mutually disjoint and disjoint from every source (the
 * intervals of one call are unordered); checked unless ETP_OPT_VALIDATE_INTERVALS is 0 -> ETP_ERR_INVALID_ARG, nothing
 * enqueued.  Sources may overlap each other. */
typedef struct { const void* src; void* dst; int64_t bytes; } etp_interval;
etp_status etp_copy_intervals(etp_ctx* ctx, const etp_interval* host_descs, int64_t n, void* stream,
                              etp_reshard_report* report);
/* Host-only, no context: the check etp_copy_intervals runs first (unless ETP_OPT_VALIDATE_INTERVALS is 0).  ETP_ERR_INVALID_ARG for a
 * negative size, a NULL pointer, two overlapping destinations or a destination that overlaps any source (the message names the two
 * intervals); ETP_ERR_ALIGNMENT for an address or size that is not a multiple of 16.  Zero-byte intervals are ignored.  O(n) plus
 * small sorts, on up to 16 threads from 65536 intervals. */
etp_status etp_intervals_validate(const etp_interval* host_descs, int64_t n);

/* ------------------------------------------------------------------------------------------------ liveness (debug entry)
 * Every spin wait inside the kernels of this library is an mbarrier wait with a deadline: a wait that is still unsatisfied after
 * 10 s (a lost arrival, a wrong byte count: a bug, not a load condition) writes {kernel family, block, thread, barrier, parity, time
 * waited} to host memory and traps.  The launch fails with a sticky CUDA error, so the next synchronising call of the caller and every
 * later call of this library fail (ETP_ERR_CUDA) instead of hanging, and etp_last_error() carries the record.  The CUDA context is
 * lost after a trap: the process has to be restarted, as after any device-side fault.
 * etp_debug_starved_wait proves the mechanism: it launches a kernel that waits, with the very wait routine the copy kernel uses, on a
 * barrier nobody arrives on, and synchronises `stream`.  Expected result: ETP_ERR_CUDA after about 10 s with the record in
 * etp_last_error().  It POISONS THE PROCESS'S CUDA CONTEXT: call it from a throw-away process only (tests/test_gpu_stress.py). */
etp_status etp_debug_starved_wait(etp_ctx* ctx, void* stream);

/* ------------------------------------------------------------------------------------------------ no-allocation entry
 * etp_copy_intervals for a caller that cannot allocate device memory.  Such callers are the normal case on the recovery path this
 * library serves ("a single pass pre-allocates all destination buffers"): when a rank dies the survivors' HBM is already
 * committed to weights and KV blocks and the serving engine's pool owns the remainder, so a cudaMalloc issued from inside a library
 * may fail, or shrink what the engine promised its KV cache; cudaMalloc / cudaFree also stall every stream of the device, which hurts
 * a recovery that overlaps with decode steps; and code that runs inside another component's CUDA context (a plugin, a fault handler)
 * is often not allowed to create memory at all.  Every other device call here needs an etp_ctx, and etp_ctx_create allocates
 * (descriptor arenas, events, streams).  This call needs no ctx: it calls no cudaMalloc / cudaFree / cudaHostAlloc, creates no
 * stream or event, and uses no allocating library routine.
 *
 * It launches the same persistent copy kernel; the kernel's scratch (segment descriptors, item table, the two work-queue heads) lives
 * in a fixed array inside the library's device image: 410,112 bytes (0.4 MiB) that every GPU which loads libetp.so holds until the
 * process exits, whether or not this call is ever made.
 *
 *  - host_descs: host array (pageable is fine; consumed before the call returns); src / dst: device memory of the CURRENT device,
 *    16-B aligned; bytes: multiple of 16.  Same disjointness contract as etp_copy_intervals, always checked (ETP_ERR_INVALID_ARG /
 *    ETP_ERR_ALIGNMENT, nothing enqueued).  Runs on the current CUDA device, asynchronously on `stream` (a stream of that device; NULL
 *    = legacy default stream): the data is in place once the caller has synchronised `stream`.  Intervals of >= 32 KiB take the
 *    cp.async.bulk ring, smaller ones are batched, as in etp_copy_intervals with default options; there are no options here.
 *  - Limits, both per call: n <= 4096 intervals, and the intervals of >= 32 KiB together at most 32768 pieces of 256 KiB (8 GiB when
 *    they are multiples of 256 KiB).  Beyond either -> ETP_ERR_CAPACITY with a message that names the limit; nothing is enqueued.
 *    Split a larger job into several calls on one stream.
 *  - The FIRST call on each device does a one-time set-up (looks up the array's device address, raises the kernel's shared-memory
 *    limit).  Make that first call before any stream capture is begun.
 *  - All calls on a device share the one array, and it keeps the previous call's contents.  The queue heads are rewritten to zero by
 *    every call and stale descriptors are never read, so back-to-back calls ON ONE STREAM are safe.  Two calls whose GPU work can
 *    overlap (different streams without an event between them, or two host threads on different streams) RACE on the array and
 *    copy wrong bytes: order them yourself.  The host side is serialised by a library mutex. */
etp_status etp_copy_intervals_static(const etp_interval* host_descs, int64_t n, void* stream);


#ifdef __cplusplus
}
#endif
#endif /* ETP_H_ */

/*
 * reshard.h -- C ABI of the B200-native cross-mesh resharding hot path (arXiv 2211.05322).
 *
 * One shared library, paper_2211_05322_b200/libreshard.so, exports exactly the symbols declared
 * here.  No torch types, no C++ types: plain pointers and sizes.  Every pointer argument says
 * whether it is a HOST or a DEVICE pointer.  Citations are PAPER.md:<line> (section).
 *
 * The operation (S2.2 "Cross-mesh resharding"): a tensor D of shape l[0..N) is held
 * by the devices of a source mesh Mesh_A under sharding spec X_A; materialise it on a disjoint
 * destination mesh Mesh_B under spec X_B.  Both meshes are VIRTUAL here: every virtual device is
 * one dense row-major shard buffer in the one GPU's HBM.
 *
 *   device mesh     PAPER.md:78-82  n-D array of devices, row-major ids: (2,2) = [[0,1],[2,3]]
 *   sharding spec   PAPER.md:84     one entry per tensor dim: R, or S followed by the mesh axes the
 *                                   dim is sharded over ("S0", "S1", "S01"); first listed axis is
 *                                   the most significant digit of the shard index (R2)
 *   data slice      PAPER.md:86     device r holds the box [p_i*c_i, (p_i+1)*c_i) of D, c_i = l_i/k_i,
 *                                   dense row-major (R11)
 *   uneven split    PAPER.md:259, 263 ("tiling, padding", "pad it in case 6"; R5): when k_i
 *                                   does not divide l_i, c_i = ceil(l_i/k_i) and the box is clipped to
 *                                   D: the last shard is short, later ones may be empty.  EVERY shard
 *                                   buffer is dense row-major of the padded local shape (c_0..c_{N-1}),
 *                                   the box at its origin; padding is never read, and its content after
 *                                   a call is unspecified (execute/pack/unpack leave it untouched,
 *                                   reshard_execute_host may overwrite it)
 *   unit task       PAPER.md:90, 482-492 (App. B.2): slices = product of the per-dim intervals cut
 *                                   at every source and destination shard boundary; senders N_i =
 *                                   source devices holding the slice, receivers M_i = destination
 *                                   devices requiring it.  Slice id = row-major rank in
 *                                   I_0 x ... x I_{N-1} (dim 0 slowest).
 *   sender choice   PAPER.md:163 (naive: lowest-indexed device), Eq. 4 (load
 *                                   balance: minimise the maximum per-sender bytes)
 *   broadcast       PAPER.md:137    one sender, all receivers; here: slice read ONCE from the
 *                                   chosen sender's shard and written to EVERY receiver shard
 *
 * Spec text accepted: entries 'R' or 'S<axes>' separated by optional commas/spaces/parentheses,
 * '^', '{', '}', '_' ignored after 'S': "S0,R,S1", "(S01, R, R)", "RRR", "RS^{01}R".
 *
 * Threading: a plan is immutable after reshard_plan returns; any number of host threads may
 * execute the same plan concurrently on different streams.  reshard_last_error is thread-local.
 */
#ifndef RESHARD_H_
#define RESHARD_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define RS_API __attribute__((visibility("default")))
#else
#define RS_API
#endif

#define RS_MAX_NDIM       8     /* tensor dims                                              */
#define RS_MAX_MESH_NDIM  4     /* mesh dims (the paper uses the 2-D view)      */
#define RS_MAX_DEVICES    128   /* virtual devices per mesh                                  */

typedef struct rs_plan rs_plan; /* opaque; owns its host tables and ONE device allocation    */

typedef enum rs_status {
    RS_OK = 0,
    RS_EINVAL = 1,        /* null pointer, non-positive extent, bad elem_bytes, bad index      */
    RS_ESPEC = 2,         /* unparsable spec, wrong entry count, mesh axis out of range or used
                             by two tensor dims (R3)                                 */
    RS_EDIVIS = 3,        /* l_i not divisible by the sharding degree k_i, with RS_EVEN_ONLY    */
    RS_EUNSUPPORTED = 4,  /* more than RS_MAX_DEVICES devices, > 2^31-1 rows per slice, ...     */
    RS_ENOMEM = 5,
    RS_ECUDA = 6          /* a CUDA runtime call failed; text via reshard_last_error()          */
} rs_status;

/* flags of reshard_plan (OR together) */
enum {
    RS_LB_GREEDY   = 0x0,   /* Eq. 4 load balance: tasks by descending bytes, each
                               to the lightest candidate; groups of <= 16 tasks are finished by an
                               exact branch-and-bound (R9).  Default.                  */
    RS_LB_NAIVE    = 0x1,   /* always the lowest-indexed candidate                  */
    RS_PATH_AUTO   = 0x00,  /* executor chosen per operation from alignment, run length and size  */
    RS_PATH_LSU    = 0x10,  /* force the register paths: 128-bit ld.global -> st.global x k (AUTO:
                               runs < 512 B, operations moving <= 32 MiB, write-heavy ones <= 10 MiB) */
    RS_PATH_BULK   = 0x20,  /* force the TMA path: cp.async.bulk global->smem ring->global x k    */
    RS_PATH_BULK_SHIFT = 0x30, /* force TMA loads + byte-shifted stores (any alignment; what AUTO picks for runs
                               >= 512 B that are not 16-byte aligned): rows >= 4 KiB are realigned in shared memory
                               and stored with cp.async.bulk, shorter ones with 128-bit register stores        */
    RS_PATH_TMAP   = 0x40,  /* force the tensor-map TMA path: like RS_PATH_BULK, but a tile of several short rows
                               (<= 2 KiB each) moves with ONE cp.async.bulk.tensor load and one store per receiver
                               instead of one bulk copy per row; tensor maps are encoded at execute time from the
                               caller's pointers.  Needs <= 16 shards per side and 16-byte aligned layouts, else it is
                               RS_PATH_BULK.  AUTO picks it for operations of 32-320 MiB whose rows are at most 2 KiB
                               long (profiles/r02_tmap.md)                                                    */
    RS_HOST_ONLY   = 0x100, /* build host tables only: no CUDA call, execute/pack/unpack refuse   */
    RS_WITH_STRATEGIES = 0x400, /* also build the tables of RS_STRATEGY_SENDRECV / RS_STRATEGY_ALLGATHER
                               (reshard_execute_strategy): the comparison of PAPER.md S3.1, S5.1         */
    RS_EVEN_ONLY   = 0x200  /* reject l_i not divisible by k_i with RS_EDIVIS ("evenly sharded",
                               PAPER.md:64) instead of padding the last shard (R5)      */
};
#define RS_PATH_MASK 0xF0

/* load balance + ORDER of the unit tasks at host level (S3.2) */
enum {
    RS_SCHED_NONE = 0,          /* Eq. 4 per device, tables in slice-id order (reshard_plan's behaviour)   */
    RS_SCHED_NAIVE = 1,         /* lowest-indexed sender, slice-id order                      */
    RS_SCHED_LOAD_BALANCE = 2,  /* Eq. 4 greedy over hosts, order = the greedy's order   */
    RS_SCHED_DFS = 3,           /* DFS over (next task, sender host), pruned, node budget */
    RS_SCHED_GREEDY = 4,        /* rounds of non-overlapping tasks covering the most hosts,
                                   found by `trials` random orderings (R24)                       */
    RS_SCHED_ENSEMBLE = 5       /* DFS and greedy, the better one (ties: DFS)                 */
};

/* Launch-shape overrides for tests and tuning sweeps (rs_plan_opts.tuning).  Every field: 0 = the library's
 * choice.  They change how an operation is tiled and launched, never its result.  The plan copies the struct. */
typedef struct rs_tuning {
    int32_t bulk_warps, bulk_stages, bulk_lookahead;   /* rs_copy_bulk: warps (pipelines) per CTA, ring slots per warp,
                                                          loads in flight per warp                                   */
    int32_t bulk_tile_bytes;                           /* bytes per ring slot = tile size (multiple of 128)          */
    int32_t bulk_ctas, bulk_ctas_mcast;                /* CTAs for 1 : 1 / for write-heavy (multicast) operations    */
    int32_t shift_warps, shift_stages, shift_lookahead, shift_tile_bytes;   /* the same for rs_copy_bulk_shift       */
    int32_t lsu_tile_bytes, lsu_ctas_per_sm;           /* register kernels                                           */
    int32_t task_order;                                /* 1: walk tiles task by task even where slices share
                                                          destination rows (default: destination address order)     */
    int32_t small_op_bytes_mib;                        /* AUTO takes the register path for aligned operations moving
                                                          at most this many MiB (-1: never); 0 = library default     */
    int32_t tiles_per_worker;                          /* small operations: tiles shrink (to 2 KiB at least) until every
                                                          worker (warp) has this many; 0 = library default          */
    int32_t pace_permille;                             /* rs_copy_bulk rate matching: offered load in permille of the DRAM
                                                          peak (2 x memory clock x bus width); -1: unpaced; 0 = default */
    int32_t no_pdl;                                    /* 1: launch without programmatic dependent launch (a kernel then
                                                          starts only after the previous kernel of the stream has ended) */
    int32_t pace_burst;                                /* rate matching: tiles of credit a warp that fell behind may catch up with; 0 = default (2) */
    int32_t pace_adapt;                                /* rate matching: 1 = the interval backs off while ring slots come back late (HBM behind the
                                                          offered load) and returns to the target afterwards; 0 = default: fixed interval */
    int32_t ring_min_smem;                             /* ring kernels request at least this many bytes of shared memory (0 = default, 116 KiB:
                                                          never two ring CTAs on one SM; 1 = only what the ring needs) */
    int32_t lsu_narrow;                                /* register path on layouts that are not 16-byte aligned: 1 = always at the layout's own vector
                                                          width, -1 = always the 16-byte shift kernel, 0 = library default (by row length) */
    int32_t shift_mode;                                /* rs_copy_bulk_shift, rows >= 1 KiB: 0 = library default (= 1); 1: windows
                                                          assembled in registers and stored with st.global; 2: row bodies
                                                          realigned in shared memory and stored with cp.async.bulk      */
} rs_tuning;

typedef struct rs_plan_opts {
    uint32_t flags;                  /* as reshard_plan; RS_LB_* is ignored when schedule != RS_SCHED_NONE  */
    int32_t schedule;                /* RS_SCHED_*                                                          */
    int32_t src_devices_per_host;    /* host = device id / this (R8); 0 or 1: every device a host */
    int32_t dst_devices_per_host;
    int32_t trials;                  /* random orderings per round of RS_SCHED_GREEDY; 0 = 32               */
    int32_t max_ctas;                /* 0 = launch shape chosen by the library; > 0: never more than this many
                                        CTAs (one per SM) per launch, leaving the other SMs to kernels of other
                                        streams -- overlapping a resharding with compute (PAPER.md S4) on chip  */
    int64_t node_budget;             /* DFS nodes before giving up with the best found; 0 = 200000          */
    uint64_t seed;                   /* of the counter-based generator the greedy search draws from         */
    const rs_tuning *tuning;         /* [HOST] may be NULL: launch shapes chosen by the library             */
    const int32_t *src_owner;        /* [HOST, n_src] may be NULL.  Multi-process executor (one process per GPU): the
                                        rank that holds source shard r.  With it the plan's execute table lists only
                                        the unit tasks whose chosen sender `rank` holds (unit tasks are independent,
                                        PAPER.md:90, 100); every rank builds the same plan with its own `rank`, and the
                                        union of their launches is the whole task.  Such a plan supports
                                        reshard_execute and the queries; pack / unpack / execute_host / strategies /
                                        groups return RS_EINVAL                                             */
    int32_t rank;                    /* this process, with src_owner                                        */
    int32_t reserved;
} rs_plan_opts;

typedef struct rs_schedule_info {
    int32_t algorithm;               /* RS_SCHED_* the plan was built with                                  */
    int32_t winner;                  /* ensemble: RS_SCHED_DFS or RS_SCHED_GREEDY; else = algorithm         */
    int32_t n_tasks, n_rounds;       /* unit tasks; rounds of the greedy search (0 if it did not run)       */
    int32_t n_src_hosts, n_dst_hosts;
    int32_t dfs_finished, reserved;  /* 1 if the DFS ran and ended before the node budget (its result is optimal);
                                        0 if it hit the budget, was skipped (more than 4096 unit tasks,
                                        PAPER.md:179) or the algorithm runs no DFS                          */
    int64_t dfs_nodes;
    int64_t makespan;                /* Eq. 1 with T_i = slice bytes (R7)                         */
    int64_t busiest_host_bytes;      /* max over hosts of the bytes it sends or receives: no schedule of
                                        these senders can finish earlier                     */
} rs_schedule_info;

/* operations a plan can run */
enum { RS_OP_EXECUTE = 0, RS_OP_PACK = 1, RS_OP_UNPACK = 2,
       RS_OP_EXECUTE_SLABS = 3, /* execute cut into dim-0 slabs: the table reshard_execute_host runs (queries only) */
       RS_OP_SENDRECV = 4,      /* RS_STRATEGY_SENDRECV: one copy task per (unit task, receiver)                    */
       RS_OP_AG_SCATTER = 5,    /* RS_STRATEGY_ALLGATHER phase 1: part j of every slice -> receiver j               */
       RS_OP_AG_GATHER = 6,     /* RS_STRATEGY_ALLGATHER phase 2: receivers copy the other parts from their peers   */
       RS_OP_AGL_SCATTER = 7,   /* RS_STRATEGY_ALLGATHER_LOCAL phase 1: per receiver host, part j -> its j-th receiver */
       RS_OP_AGL_GATHER = 8     /* RS_STRATEGY_ALLGATHER_LOCAL phase 2: all-gather inside every receiver host        */ };

/* communication strategies for a unit task (S3.1), on chip */
enum {
    RS_STRATEGY_BROADCAST = 0,  /* slice read once, written to every receiver (= reshard_execute)    */
    RS_STRATEGY_SENDRECV = 1,   /* the sender sends the slice to each receiver one by one: the slice
                                   is re-read per receiver (k reads + k writes)                                    */
    RS_STRATEGY_ALLGATHER = 2,  /* PAPER.md:133 (global all-gather): the slice is split over its k receivers, one part
                                   sent to each, then the receivers all-gather: two dependent launches, 1 + (k-1)
                                   reads and 1 + (k-1) writes per slice byte                                       */
    RS_STRATEGY_ALLGATHER_LOCAL = 3 /* PAPER.md:131 (local all-gather): the same inside every receiver HOST
                                   (rs_plan_opts.dst_devices_per_host): the slice leaves the sender once per host  */
};
/* sides */
enum { RS_SRC = 0, RS_DST = 1 };

typedef struct rs_plan_info {
    int32_t ndim, elem_bytes;
    int32_t n_src, n_dst;            /* devices in Mesh_A, Mesh_B                                  */
    int32_t n_slices;                /* unit tasks (App. B.2)                                      */
    int32_t n_messages;              /* non-empty (sender, receiver) pairs                         */
    int64_t tensor_bytes;            /* size(D) * e                                                */
    int64_t src_shard_bytes;         /* bytes of ONE source shard buffer (all equal; padded, R5)   */
    int64_t dst_shard_bytes;         /* bytes of ONE destination shard                             */
    int64_t unique_read_bytes;       /* = tensor_bytes: every element read once      */
    int64_t write_bytes;             /* = tensor_bytes * r_B (r_B = destination replication)       */
    int64_t max_sender_bytes;        /* objective of Eq. 4 under the chosen senders                */
    int64_t arena_bytes;             /* message arena for pack/unpack = write_bytes (+alignment)   */
    int32_t lb_mode;                 /* RS_LB_GREEDY or RS_LB_NAIVE                                */
    int32_t device;                  /* CUDA device the tables live on, -1 if RS_HOST_ONLY         */
} rs_plan_info;

typedef struct rs_op_info {
    int32_t path;                    /* RS_PATH_LSU, RS_PATH_BULK, RS_PATH_BULK_SHIFT or RS_PATH_TMAP selected */
    int32_t vec_bytes;               /* widest access every offset/stride/run of the op allows     */
    int32_t n_tasks;                 /* copy tasks (execute/pack: one per slice; unpack: per
                                        (slice, receiver))                                         */
    int32_t n_dsts;                  /* (task, destination) entries                                */
    int32_t n_tiles;                 /* tiles one launch walks (units of GPU work; decoded, never stored)  */
    int32_t tile_bytes;              /* target bytes read per tile                                 */
    int32_t grid, block;             /* launch configuration                                       */
    int32_t smem_bytes;              /* dynamic shared memory per CTA                              */
    int64_t read_bytes, write_bytes; /* algorithmic bytes of one launch                            */
    int64_t min_run_bytes;           /* shortest contiguous run any tile copies                    */
    int32_t n_segs;                  /* segments: groups of tasks whose tiles are walked round-robin       */
    int32_t table_bytes;             /* bytes of this operation's tables in device memory: O(unit tasks),
                                        independent of the tensor size (the plan is the
                                        slice list)                                                        */
    int32_t pace_permille;           /* rs_copy_bulk rate matching: the launch offers this many permille of the
                                        DRAM peak (write-heavy operations); 0 = unpaced                    */
    int32_t reserved;
} rs_op_info;

/*
 * reshard_plan -- steps a1..a5 of the path (host): tile boxes, unit tasks, sender choice, flat
 * task/tile tables for execute, pack and unpack, message layout; uploads the tables to the
 * current CUDA device (one cudaMalloc + one cudaMemcpy) unless RS_HOST_ONLY.
 *   global_shape [HOST, ndim]   l_i >= 1, 1 <= ndim <= RS_MAX_NDIM
 *   elem_bytes                  1, 2, 4, 8 or 16; the payload is opaque bytes (R22)
 *   src/dst_mesh_shape [HOST]   m_a >= 1, 1 <= mesh_ndim <= RS_MAX_MESH_NDIM, product <= RS_MAX_DEVICES
 *   src/dst_spec [HOST]         NUL-terminated spec text, see above
 *   out_plan [HOST]             receives the plan; untouched on failure.  Caller frees it with
 *                               reshard_plan_destroy.
 */
RS_API rs_status reshard_plan(const int64_t *global_shape, int32_t ndim, int32_t elem_bytes,
                       const int32_t *src_mesh_shape, int32_t src_mesh_ndim, const char *src_spec,
                       const int32_t *dst_mesh_shape, int32_t dst_mesh_ndim, const char *dst_spec,
                       uint32_t flags, rs_plan **out_plan);

/* reshard_plan with options: opts->schedule != RS_SCHED_NONE runs S3.2 at host level; the chosen
 * host's least-loaded candidate device (lowest id on ties; RS_SCHED_NAIVE: its lowest-indexed device)
 * becomes the sender, and the task tables list the unit tasks in order of their start time S_i.
 * The data result is the same whatever the schedule (R10).  opts [HOST] may be NULL. */
RS_API rs_status reshard_plan_ex(const int64_t *global_shape, int32_t ndim, int32_t elem_bytes,
                          const int32_t *src_mesh_shape, int32_t src_mesh_ndim, const char *src_spec,
                          const int32_t *dst_mesh_shape, int32_t dst_mesh_ndim, const char *dst_spec,
                          const rs_plan_opts *opts, rs_plan **out_plan);
/* the schedule of a plan built with schedule != RS_SCHED_NONE (else RS_EINVAL): per unit task its
 * sender HOST, its start time S_i (bytes), and the global order.
 * sender_host, start, order [HOST, n_slices] may each be NULL. */
RS_API rs_status reshard_plan_schedule(const rs_plan *plan, rs_schedule_info *info, int32_t *sender_host,
                                int64_t *start, int32_t *order);

/* reshard_plan_group: ONE plan that runs the reshard_execute of several plans in a single launch -- every tensor
 * that crosses a stage boundary at once; for small tensors the launch, not HBM, is the cost.
 * The group's src_shards array is the concatenation of the members' source arrays in the order given, its
 * dst_shards array likewise (at most RS_MAX_DEVICES pointers on each side in total, else RS_EUNSUPPORTED).
 * The members may be destroyed afterwards.  A group supports reshard_execute, reshard_plan_info (counts and
 * byte totals), reshard_op_info / reshard_op_tables of RS_OP_EXECUTE, and reshard_plan_destroy; everything
 * else returns RS_EINVAL.  flags: RS_PATH_*, RS_HOST_ONLY.  plans [HOST array of n_plans plans, none a group]. */
RS_API rs_status reshard_plan_group(const rs_plan *const *plans, int32_t n_plans, uint32_t flags, rs_plan **out_plan);

RS_API void reshard_plan_destroy(rs_plan *plan);      /* NULL is allowed */

/* ---- queries (all host-side, no CUDA) ------------------------------------------------------ */
RS_API rs_status reshard_plan_info(const rs_plan *plan, rs_plan_info *out);
RS_API rs_status reshard_op_info(const rs_plan *plan, int32_t op, rs_op_info *out);
/* (padded) local shard shape c_i = ceil(l_i / k_i) of one side; out [HOST, ndim] */
RS_API rs_status reshard_plan_local_shape(const rs_plan *plan, int32_t side, int64_t *out);
/* box [lo, hi) of D that device `dev` of `side` holds (clipped to D, may be empty); lo, hi [HOST, ndim] */
RS_API rs_status reshard_plan_device_box(const rs_plan *plan, int32_t side, int32_t dev, int64_t *lo, int64_t *hi);
/* unit task i: box, chosen sender, candidate senders N_i, receivers M_i.
 * senders [HOST, n_src] / receivers [HOST, n_dst] may be NULL. */
RS_API rs_status reshard_plan_slice(const rs_plan *plan, int32_t i, int64_t *lo, int64_t *hi,
                             int32_t *sender, int32_t *n_senders, int32_t *senders,
                             int32_t *n_receivers, int32_t *receivers);
/* bytes each source device sends under the chosen senders; out [HOST, n_src] */
RS_API rs_status reshard_plan_sender_bytes(const rs_plan *plan, int64_t *out);
/* message m (ordered by (sender, receiver)): the concatenation, in ascending slice id, of every
 * slice with that sender needed by that receiver, each dense row-major (the wire model, north_star
 * item 3).  offset = byte offset inside the arena.  slice_ids [HOST, n_slices] may be NULL. */
RS_API rs_status reshard_plan_message(const rs_plan *plan, int32_t m, int32_t *sender, int32_t *receiver,
                               int64_t *offset, int64_t *bytes, int32_t *n_slice_ids, int32_t *slice_ids);

/* Raw copy of operation `op`'s flat tables (inspection and host-side tests; the layouts are the
 * structs RsTask / RsDst / RsSeg of paper_2211_05322_b200/csrc/tables.h: 224, 16 and 16 bytes).
 * tasks [HOST, n_tasks*224], dsts [HOST, n_dsts*16], segs [HOST, n_segs*16]; each may be NULL. */
RS_API rs_status reshard_op_tables(const rs_plan *plan, int32_t op, void *tasks, void *dsts, void *segs);
/* Tiles first_tile .. first_tile + n_tiles - 1 of operation `op`, decoded on the host by the same routine the
 * kernels run on the device (tables.h rs_tile_locate / rs_tile_decode), as 32-byte RsTile records
 * {u32 task, n_rows, col_bytes, flags; u64 a, b}.  tiles [HOST, n_tiles*32].  RS_EINVAL if the range leaves
 * [0, rs_op_info.n_tiles). */
RS_API rs_status reshard_op_tiles(const rs_plan *plan, int32_t op, int64_t first_tile, int64_t n_tiles, void *tiles);

/* ---- the data path (steps a6..a8): asynchronous, allocate nothing, never synchronise -------- */
/*
 * reshard_execute (PAPER.md:137 on-chip: read once, write to every receiver): for every unit task
 * copy the slice from the chosen sender's shard into each receiver's shard.
 *   src_shards [HOST array of n_src DEVICE pointers]  shard r = dense row-major local box of device r
 *   dst_shards [HOST array of n_dst DEVICE pointers]  written completely (every element exactly once)
 *   cuda_stream                                       cudaStream_t (NULL = legacy default stream)
 * Preconditions (undefined behaviour otherwise, not checked): replicas on the source side hold
 * identical bytes; no destination shard overlaps any other shard (Mesh_A and Mesh_B are
 * disjoint).  Pointers of source shards that no task reads may be NULL.
 * A plan built with rs_plan_opts.src_owner runs this rank's unit tasks only: source pointers of shards other
 * ranks hold may be NULL, destination pointers may be NULL for shards this rank never writes, and the others may
 * be peer memory (another GPU's shard mapped through CUDA IPC or peer access: the slice is moved by the kernel's
 * stores, "the sender's GPU issues the writes").
 * One kernel launch.  Returns RS_ECUDA if the launch fails, RS_EINVAL for a host-only plan.
 */
RS_API rs_status reshard_execute(const rs_plan *plan, const void *const *src_shards, void *const *dst_shards,
                          void *cuda_stream);
/*
 * reshard_execute_static: reshard_execute for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight
 * serving loops, harnesses that forbid it).  It needs no device allocation ANYWHERE: the plan may be built with
 * RS_HOST_ONLY (reshard_plan then makes no CUDA call at all; its grids are sized for a 148-SM part), and the kernels read
 * their task tables from a file-scope `static __device__` array of RS_STATIC_TABLE_BYTES = 256 KiB inside the library
 * (every GPU that loads the library holds it until exit) instead of the plan's own cudaMalloc block.  The call copies the
 * plan's execute tables into that array with cudaMemcpyAsync on `cuda_stream`, then launches the same kernels as
 * reshard_execute on it; it calls no cudaMalloc, cudaFree or allocating library routine, and returns without synchronising.
 *   - Limit: the execute tables (224 bytes per unit task + 16 per receiver + 16 per segment, each part rounded up to 256)
 *     must fit the array: about 1000 unit tasks.  Larger plans return RS_EUNSUPPORTED with a message that names both
 *     sizes; plans built with src_owner and plan groups return RS_EINVAL.
 *   - The array is SHARED by every call on the device and keeps the last call's tables.  Every byte a launch reads is
 *     rewritten by its own call first, so nothing has to be cleared; but calls that may overlap on the GPU (two
 *     streams, two host threads on different streams) RACE on it: issue them on one stream, or order them with events.
 *     Calls on one stream are ordered (these launches do not use programmatic dependent launch).
 *   - src_shards / dst_shards as for reshard_execute; the result is byte for byte that of reshard_execute.
 */
RS_API rs_status reshard_execute_static(const rs_plan *plan, const void *const *src_shards, void *const *dst_shards,
                                 void *cuda_stream);
/* reshard_execute_strategy: the same result as reshard_execute, reached with another of the paper's
 * strategies for a unit task.  The plan must have been built with RS_WITH_STRATEGIES
 * (else RS_EINVAL).  RS_STRATEGY_BROADCAST is reshard_execute; RS_STRATEGY_SENDRECV is one launch;
 * RS_STRATEGY_ALLGATHER is two launches on `cuda_stream`, the second reading destination shards. */
RS_API rs_status reshard_execute_strategy(const rs_plan *plan, int32_t strategy, const void *const *src_shards,
                                   void *const *dst_shards, void *cuda_stream);
/* reshard_pack: sender shards -> message arena [DEVICE, arena_bytes].  A slice needed by k receivers
 * is read once and written into k messages.  One kernel launch. */
RS_API rs_status reshard_pack(const rs_plan *plan, const void *const *src_shards, void *msg_arena, void *cuda_stream);
/* reshard_unpack: message arena -> receiver shards.  unpack(pack(x)) == execute(x) bit for bit. */
RS_API rs_status reshard_unpack(const rs_plan *plan, const void *msg_arena, void *const *dst_shards, void *cuda_stream);

/*
 * reshard_execute_host -- the same operation with HOST shard buffers (the end-to-end call).
 * Pipelined over slabs of tensor dim 0 (the chunk pipelining of PAPER.md:137 applied to the host
 * link): slab c of the source shards the plan reads is copied host->device into `workspace` on a
 * plan-owned upload stream, resharded by one kernel launch on `cuda_stream`, and its destination
 * byte ranges are copied device->host on a plan-owned download stream while slab c+1 uploads.
 * All work is ordered after prior work on `cuda_stream`, and `cuda_stream` waits for the last
 * download; returns without synchronising.  Calls on one plan from several host threads are serialised
 * while they enqueue (the plan owns the side streams, created on first use).
 *   src_shards_host [HOST array of n_src HOST pointers]  (pinned memory makes the copies async)
 *   dst_shards_host [HOST array of n_dst HOST pointers]
 *   workspace [DEVICE]  at least reshard_host_workspace_bytes(plan) bytes, 256-byte aligned (else RS_EINVAL)
 *   h2d_bytes, d2h_bytes [HOST, may be NULL]  receive the bytes copied in each direction
 */
RS_API rs_status reshard_execute_host(const rs_plan *plan, const void *const *src_shards_host,
                               void *const *dst_shards_host, void *workspace, void *cuda_stream,
                               int64_t *h2d_bytes, int64_t *d2h_bytes);
RS_API int64_t reshard_host_workspace_bytes(const rs_plan *plan);

/* ---- multi-process executor plumbing: CUDA IPC -------------------------------------------------
 * One process per GPU; every rank exports the destination shards it holds, the senders' ranks import them and
 * pass the mapped pointers to reshard_execute.  These three calls only wrap cudaIpcGetMemHandle /
 * cudaIpcOpenMemHandle / cudaIpcCloseMemHandle and deal with sub-allocated pointers (a caching allocator hands out
 * pieces of one cudaMalloc block: the handle names the block, the offset the piece). */
#define RS_IPC_HANDLE_BYTES 80
/* dev_ptr [DEVICE, from cudaMalloc in THIS process] -> handle_out [HOST, RS_IPC_HANDLE_BYTES], to be sent to peers */
RS_API rs_status reshard_ipc_export(const void *dev_ptr, void *handle_out);
/* handle [HOST, RS_IPC_HANDLE_BYTES, exported by ANOTHER process] -> *dev_ptr_out [DEVICE pointer valid in this
 * process].  Every exporting allocation is mapped once per process and kept until reshard_ipc_release_all. */
RS_API rs_status reshard_ipc_import(const void *handle, void **dev_ptr_out);
/* unmap everything reshard_ipc_import mapped (before the exporters free their memory) */
RS_API rs_status reshard_ipc_release_all(void);

/* ---- S4: pipeline schedules around the resharding tasks (host only, no CUDA) ------------------- */
#define RS_PIPE_MAX_STAGES 64
enum { RS_PIPE_1F1B = 0,        /* stage i warms up with #stages - i + 1 forwards              */
       RS_PIPE_EAGER_1F1B = 1   /* stage i warms up with 2 (#stages - i) + 1 forwards          */ };
enum { RS_PIPE_F = 0, RS_PIPE_B = 1, RS_PIPE_BA = 2 /* activation gradients */, RS_PIPE_BW = 3 /* weight gradients */ };

typedef struct rs_pipeline_opts {
    int32_t schedule;                /* RS_PIPE_1F1B or RS_PIPE_EAGER_1F1B                                   */
    int32_t n_stages;                /* 1..RS_PIPE_MAX_STAGES; stages are numbered 1..S in the paper, 0..S-1 in arrays */
    int32_t n_micro_batches;         /* >= 1; warm-up counts are capped at it (R28)                */
    int32_t overlap;                 /* 1: transfers run beside the sender's compute;
                                        0: the sender stage is busy until its transfer has finished           */
    int32_t bw_delay;                /* with bwd_act: ops by which the weight-gradient half is postponed (R32) */
    int32_t reserved;
    const int64_t *fwd, *bwd;        /* [HOST, n_stages] compute time of one forward / one whole backward, ticks */
    const int64_t *bwd_act;          /* [HOST, n_stages] or NULL: time of the activation-gradient half; not NULL
                                        splits every backward (backward weight delaying)    */
    int64_t comm_fwd, comm_bwd;      /* ticks one micro-batch's tensor needs across a stage boundary, e.g. the
                                        measured time of reshard_execute for that boundary's plan             */
} rs_pipeline_opts;

typedef struct rs_pipeline_result {
    int64_t makespan;                /* end of the last op of the iteration                                  */
    int32_t ops_per_stage;           /* 2 M, or 3 M with a split backward                                    */
    int32_t reserved;
    int32_t warmup[RS_PIPE_MAX_STAGES];            /* forwards before the first backward                     */
    int32_t peak_activations[RS_PIPE_MAX_STAGES];  /* most micro-batches alive at once        */
    int64_t busy[RS_PIPE_MAX_STAGES];              /* compute time of the stage                               */
} rs_pipeline_result;

/* Timeline of one iteration (R28-R32): every stage runs its op list strictly in order, an op starts
 * when the stage is free and its input has arrived; every boundary has one link per direction.  The four output
 * arrays [HOST, n_stages * ops_per_stage] (stage-major, in list order; query ops_per_stage with them NULL first)
 * receive op kind (RS_PIPE_*), micro-batch, start and end; each may be NULL. */
RS_API rs_status reshard_pipeline_simulate(const rs_pipeline_opts *opts, rs_pipeline_result *result, int32_t *op_kind,
                                    int32_t *op_micro_batch, int64_t *op_start, int64_t *op_end);
/* PAPER.md:217 "delay the least to cover all communications": the smallest bw_delay for which the compute a
 * stage (1-based) runs between an activation-gradient op and its weight-gradient op covers comm_bwd.
 * Returns -1 for bad arguments and when no delay up to 2 * n_micro_batches covers it. */
RS_API int32_t reshard_pipeline_least_delay(int32_t schedule, int32_t n_stages, int32_t stage, int32_t n_micro_batches,
                                     int64_t fwd, int64_t bwd, int64_t bwd_act, int64_t comm_bwd);

/* kernels launched by this library in the calling thread since it was loaded (bench bookkeeping) */
RS_API int64_t reshard_launch_count(void);

RS_API const char *reshard_strerror(rs_status s);
RS_API const char *reshard_last_error(void);          /* thread-local text of the last failure, "" if none */
RS_API const char *reshard_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RESHARD_H_ */

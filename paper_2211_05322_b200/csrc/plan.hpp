// plan.hpp -- host planner of a cross-mesh resharding task (steps a1..a5).  Internal header.
//
//   a1 spec -> tile boxes                      PAPER.md:78-86   (S2.2)
//   a2 cutpoints -> intervals -> slices        PAPER.md:488-492 (App. B.2)
//   a3 sender / receiver sets N_i, M_i
//   a4 load-balanced sender choice             PAPER.md:163 (naive), 167-171 Eq. 4 (greedy/LPT)
//   a5 flat task / tile tables, message layout north_star items (1), (3)
#pragma once
#include <stdint.h>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/reshard.h"
#include "tables.h"

namespace rs {

struct Layout {                          // one side of the task: (shape, mesh, spec)
    int ndim = 0;
    int64_t shape[RS_MAX_NDIM];          // l_i
    int mesh_ndim = 0;
    int64_t mesh[RS_MAX_MESH_NDIM];      // m_a
    int n_axes[RS_MAX_NDIM];             // 0 => R
    int axes[RS_MAX_NDIM][RS_MAX_MESH_NDIM];
    int64_t degree[RS_MAX_NDIM];         // k_i
    int64_t local[RS_MAX_NDIM];          // c_i = ceil(l_i / k_i): padded local extent (R5)
    int n_dev = 0;
    std::vector<int64_t> shard_index;    // [n_dev][ndim]: p_i of every device
    int64_t shard_elems() const { int64_t n = 1; for (int i = 0; i < ndim; i++) n *= local[i]; return n; }
};

struct Slice {                           // one unit task
    int64_t lo[RS_MAX_NDIM], hi[RS_MAX_NDIM];
    int64_t elems = 0;
    std::vector<int> senders;            // N_i, ascending device id
    std::vector<int> receivers;          // M_i, ascending device id
    int sender = -1;                     // n_i*
};

struct Message {                         // wire model: everything sender s ships to receiver r
    int sender, receiver;
    int64_t offset = 0, bytes = 0;       // inside the arena
    std::vector<int> slice_ids;          // ascending
    std::vector<int64_t> slice_off;      // byte offset of each slice inside the arena
};

struct OpTables {                        // one operation (execute / pack / unpack)
    std::vector<RsTask> tasks;
    std::vector<RsDst> dsts;
    std::vector<RsSeg> segs;             // tiles are never stored: decoded from (segs, tasks), tables.h
    rs_op_info info{};
    int stages = 0, lookahead = 0;       // TMA path: ring slots per warp, loads in flight
    uint32_t shift_stage = 0;            // rs_copy_bulk_shift: bytes per ring slot (rows padded), 0 if the path is not used
    int pace_permille = 0;               // rs_copy_bulk: offered load as permille of the DRAM peak (0: unpaced)
    int64_t mean_run_bytes = 0;          // bytes moved / rows moved (register path on unaligned layouts: which vector width)
    int64_t src_cap = 0, dst_cap = 0;    // bytes of every source / destination buffer of this operation (0: they differ, groups)
    RsTmapGeom tmap_src[RS_TMAP_BUFS] = {}, tmap_dst[RS_TMAP_BUFS] = {};   // RS_PATH_TMAP: geometry of the tensor map of every buffer
    uint32_t alt_stage = 0;              // TMA plans handed under-aligned pointers: shape of rs_copy_bulk_shift on the same tiles
    int alt_warps = 0, alt_stages = 0, alt_smem = 0;
    RsOpDev dev{};                       // device copies (null for a host-only plan)
};

struct HostCopy {                        // one contiguous host<->device copy of a shard byte range
    int dev;                             // device id on its side
    int64_t off, bytes;                  // inside the shard
};

struct HostSlab {                        // one stage of the reshard_execute_host pipeline: a slab of tensor dim 0
    uint32_t tile_begin = 0, tile_end = 0;       // tile range of op[RS_OP_SLABS] (its tasks are consecutive)
    std::vector<HostCopy> up, down;      // source ranges to upload before, destination ranges to download after
};

struct Schedule {                        // S3.2 at host level (schedule.cpp); algorithm 0 = not scheduled
    int algorithm = 0;
    int src_dph = 1, dst_dph = 1;        // devices per host (R8)
    int trials = 0;
    int64_t node_budget = 0;
    uint64_t seed = 0;
    int64_t makespan = 0;                // Eq. 1, in bytes (T_i = slice bytes, R7)
    int64_t busiest_host_bytes = 0;      // Eq. 4-style bound under the chosen senders
    int n_rounds = 0, winner = 0, dfs_finished = 1;
    int64_t dfs_nodes = 0;
    std::vector<int> sender_host, order; // per slice; global order
    std::vector<int64_t> start;          // S_i
};

enum { RS_OP_SLABS = 3, RS_N_OPS = 9 };  // internal 4th table: execute, cut into dim-0 slabs; 4..6: alternative strategies

struct Plan {
    Layout A, B;
    int elem_bytes = 0;
    uint32_t flags = 0;
    std::vector<Slice> slices;
    Schedule sched;
    std::vector<int> exec_order;         // slice ids in the order the tables list them (identity unless scheduled)
    std::vector<int64_t> sender_bytes;
    int64_t max_sender_bytes = 0;
    std::vector<Message> messages;
    int64_t arena_bytes = 0;
    int64_t r_B = 1;                     // destination replication factor
    OpTables op[RS_N_OPS];
    std::vector<HostSlab> slabs;         // reshard_execute_host pipeline (PAPER.md:137's chunked pipelining, over PCIe)
    // reshard_execute_host: plan-owned upload / download streams (cudaStream_t) and cudaEvent_t (2 per slab + 2),
    // created on first use; host_mu serialises the enqueue of concurrent calls
    mutable std::mutex host_mu;
    mutable void *streams[2] = {nullptr, nullptr};
    mutable std::vector<void *> events;
    std::vector<char> used_src;          // [n_src] 1 if some task reads that shard
    int device = -1;
    int sm_count = 148;
    double dram_peak_gbs = 7672.0;       // 2 x memory clock x bus width of the device (B200 default for host-only plans)
    int group_src = 0, group_dst = 0;    // > 0: this plan is a GROUP (reshard_plan_group): only its execute table exists
    int max_ctas = 0;                    // rs_plan_opts.max_ctas: cap on CTAs per launch (0: none)
    rs_tuning tune{};                    // rs_plan_opts.tuning (all zero: the library's launch shapes)
    // multi-process executor (rs_plan_opts.src_owner / rank): the tables list only the unit tasks whose chosen sender
    // this rank holds; the other ranks run the rest (unit tasks are independent)
    std::vector<int> src_owner;          // [n_src] rank holding source shard r; empty: single-process plan
    int rank = -1;
    std::vector<char> used_dst;          // [n_dst] 1 if some task of the execute table writes that shard
    void *dev_blob = nullptr;            // the ONE device allocation
};

void set_error(const std::string &msg);
const std::string &last_error();

rs_status make_layout(const int64_t *shape, int ndim, const int32_t *mesh, int mesh_ndim, const char *spec,
                      bool even_only, Layout *L);
void device_box(const Layout &L, int dev, int64_t *lo, int64_t *hi);
rs_status build_slices(Plan *P);                       // a2 + a3
void choose_senders(Plan *P);                          // a4
rs_status schedule_plan(Plan *P);                      // S3.2: senders + order at host level, schedule.cpp
rs_status build_messages(Plan *P);                     // message layout
rs_status build_tables(Plan *P);                       // a5 (host side), tables.cpp
rs_status build_group(Plan *G, const std::vector<const Plan *> &members);   // merged execute table, tables.cpp
rs_status pipeline_simulate(const rs_pipeline_opts &o, rs_pipeline_result *res, int32_t *op_kind, int32_t *op_micro,
                            int64_t *op_start, int64_t *op_end);                    // S4, pipeline.cpp
int pipeline_least_delay(int schedule, int S, int stage, int M, int64_t f, int64_t b, int64_t b_act, int64_t c_bwd);

}  // namespace rs

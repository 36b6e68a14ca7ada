// api.cu -- the C ABI of include/reshard.h: plan creation / upload / queries and the launch glue of
// execute, pack, unpack and the host-buffer entry point.
#include <cuda.h>                         // CUtensorMap and its enums only; the encoder is fetched through the runtime
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include "../../include/reshard.h"
#include "config.h"
#include "kernels.h"
#include "plan.hpp"

static_assert(sizeof(RsTask) == 224 && sizeof(RsDst) == 16 && sizeof(RsSeg) == 16 && sizeof(RsTile) == 32, "table layouts are part of reshard_op_tables / reshard_op_tiles");

struct rs_plan {
    rs::Plan p;
};

namespace {

rs_status cuda_fail(cudaError_t e, const char *what) {
    rs::set_error(std::string(what) + ": " + cudaGetErrorString(e));
    return RS_ECUDA;
}

size_t round256(size_t x) { return (x + 255) / 256 * 256; }

// SM count and DRAM peak of the current device: grids and pacing are sized from them, so they are read BEFORE the
// tables are built.  Queried once per device and process (the clock-rate attributes take milliseconds).
rs_status query_device(rs::Plan *P) {
    struct Info { int sms = 0; double peak = 0; };
    static std::mutex mu;
    static Info cache[64];
    cudaError_t e = cudaGetDevice(&P->device);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    std::lock_guard<std::mutex> lock(mu);
    Info local;
    Info &I = P->device >= 0 && P->device < 64 ? cache[P->device] : local;
    if (I.sms == 0) {
        e = cudaDeviceGetAttribute(&I.sms, cudaDevAttrMultiProcessorCount, P->device);
        if (e != cudaSuccess) { I.sms = 0; return cuda_fail(e, "cudaDeviceGetAttribute"); }
        int mem_khz = 0, bus_bits = 0;                         // DRAM peak = 2 x memory clock x bus width (B200: 7 672 GB/s)
        cudaDeviceGetAttribute(&mem_khz, cudaDevAttrMemoryClockRate, P->device);
        cudaDeviceGetAttribute(&bus_bits, cudaDevAttrGlobalMemoryBusWidth, P->device);
        if (mem_khz > 0 && bus_bits > 0) I.peak = 2.0 * mem_khz * 1e3 * bus_bits / 8 / 1e9;
    }
    P->sm_count = I.sms;
    if (I.peak > 0) P->dram_peak_gbs = I.peak;
    return RS_OK;
}

// One device allocation holding every operation's task / destination / segment tables: O(unit tasks) bytes
// (tiles are decoded by the kernels, tables.h), one cudaMalloc + one cudaMemcpy.
rs_status upload(rs::Plan *P) {
    size_t total = 0;
    for (rs::OpTables &o : P->op)
        total += round256(o.tasks.size() * sizeof(RsTask)) + round256(o.dsts.size() * sizeof(RsDst)) +
                 round256(o.segs.size() * sizeof(RsSeg));
    std::vector<char> host(total, 0);
    cudaError_t e = cudaMalloc(&P->dev_blob, std::max<size_t>(total, 256));
    if (e != cudaSuccess) { P->dev_blob = nullptr; return e == cudaErrorMemoryAllocation ? RS_ENOMEM : cuda_fail(e, "cudaMalloc"); }
    size_t off = 0;
    char *base = static_cast<char *>(P->dev_blob);
    for (rs::OpTables &o : P->op) {
        o.dev.tasks = reinterpret_cast<const RsTask *>(base + off);
        std::memcpy(host.data() + off, o.tasks.data(), o.tasks.size() * sizeof(RsTask));
        off += round256(o.tasks.size() * sizeof(RsTask));
        o.dev.dsts = reinterpret_cast<const RsDst *>(base + off);
        std::memcpy(host.data() + off, o.dsts.data(), o.dsts.size() * sizeof(RsDst));
        off += round256(o.dsts.size() * sizeof(RsDst));
        o.dev.segs = reinterpret_cast<const RsSeg *>(base + off);
        std::memcpy(host.data() + off, o.segs.data(), o.segs.size() * sizeof(RsSeg));
        off += round256(o.segs.size() * sizeof(RsSeg));
        o.dev.n_segs = (uint32_t)o.segs.size();
        o.dev.seg_tiles = o.segs.empty() ? 0 : o.segs[0].n_members * o.segs[0].tiles_each;
        for (const RsSeg &sg : o.segs) if (sg.n_members * sg.tiles_each != o.dev.seg_tiles) o.dev.seg_tiles = 0;
        o.dev.n_tasks = (uint32_t)o.tasks.size();
        o.dev.n_dsts = (uint32_t)o.dsts.size();
        o.dev.early_trigger = 0;
        o.dev.tile_base = 0;
        o.dev.n_tiles = (uint32_t)o.info.n_tiles;
    }
    e = cudaMemcpy(P->dev_blob, host.data(), total, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpy(tables)");
    static std::once_flag smem_once;                           // once per process: the four TMA kernels may use all of shared memory
    static cudaError_t smem_err = cudaSuccess;
    std::call_once(smem_once, [] { smem_err = rs::prepare_bulk(RS_SMEM_MAX); });
    if (smem_err != cudaSuccess) return cuda_fail(smem_err, "cudaFuncSetAttribute(rs_copy_bulk)");
    return RS_OK;
}

// reshard_execute_host: plan-owned upload / download streams and per-slab events, created on first use
rs_status host_streams(const rs::Plan &P) {
    if (P.streams[0]) return RS_OK;
    for (int i = 0; i < 2; i++) {
        cudaStream_t st;
        cudaError_t e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking);
        if (e != cudaSuccess) return cuda_fail(e, "cudaStreamCreate");
        P.streams[i] = st;
    }
    for (size_t i = 0; i < 2 * P.slabs.size() + 2; i++) {
        cudaEvent_t ev;
        cudaError_t e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
        if (e != cudaSuccess) return cuda_fail(e, "cudaEventCreate");
        P.events.push_back(ev);
    }
    return RS_OK;
}

}  // namespace

extern "C" {

rs_status reshard_plan(const int64_t *global_shape, int32_t ndim, int32_t elem_bytes,
                       const int32_t *src_mesh_shape, int32_t src_mesh_ndim, const char *src_spec,
                       const int32_t *dst_mesh_shape, int32_t dst_mesh_ndim, const char *dst_spec,
                       uint32_t flags, rs_plan **out_plan) {
    rs_plan_opts o;
    std::memset(&o, 0, sizeof(o));
    o.flags = flags;
    return reshard_plan_ex(global_shape, ndim, elem_bytes, src_mesh_shape, src_mesh_ndim, src_spec, dst_mesh_shape,
                           dst_mesh_ndim, dst_spec, &o, out_plan);
}

rs_status reshard_plan_ex(const int64_t *global_shape, int32_t ndim, int32_t elem_bytes,
                          const int32_t *src_mesh_shape, int32_t src_mesh_ndim, const char *src_spec,
                          const int32_t *dst_mesh_shape, int32_t dst_mesh_ndim, const char *dst_spec,
                          const rs_plan_opts *opts, rs_plan **out_plan) {
    rs::set_error("");
    rs_plan_opts defaults;
    std::memset(&defaults, 0, sizeof(defaults));
    if (!opts) opts = &defaults;
    const uint32_t flags = opts->flags;
    if (!out_plan) { rs::set_error("out_plan is null"); return RS_EINVAL; }
    if (elem_bytes != 1 && elem_bytes != 2 && elem_bytes != 4 && elem_bytes != 8 && elem_bytes != 16) {
        rs::set_error("elem_bytes must be 1, 2, 4, 8 or 16");
        return RS_EINVAL;
    }
    rs_plan *h = new (std::nothrow) rs_plan();
    if (!h) return RS_ENOMEM;
    rs::Plan *P = &h->p;
    P->elem_bytes = elem_bytes;
    P->flags = flags;
    P->sched.algorithm = opts->schedule;
    P->sched.src_dph = std::max(1, opts->src_devices_per_host);
    P->sched.dst_dph = std::max(1, opts->dst_devices_per_host);
    P->sched.trials = opts->trials;
    P->sched.node_budget = opts->node_budget;
    P->sched.seed = opts->seed;
    P->max_ctas = std::max(0, opts->max_ctas);
    if (opts->tuning) P->tune = *opts->tuning;
    rs_status st;
    try {
        st = (flags & RS_HOST_ONLY) ? RS_OK : query_device(P);
        if (st == RS_OK && opts->src_owner) {                  // multi-process executor: this rank's share of the unit tasks
            int64_t n_src = 1;
            for (int32_t a = 0; src_mesh_shape && a < src_mesh_ndim && a < RS_MAX_MESH_NDIM; a++) n_src *= std::max(1, src_mesh_shape[a]);
            if (n_src > RS_MAX_DEVICES) n_src = 0;             // make_layout reports the real error
            if (flags & RS_WITH_STRATEGIES) { rs::set_error("RS_WITH_STRATEGIES is not available with src_owner"); st = RS_EINVAL; }
            if (opts->rank < 0) { rs::set_error("rank < 0 with src_owner"); st = RS_EINVAL; }
            P->src_owner.assign(opts->src_owner, opts->src_owner + n_src);
            P->rank = opts->rank;
        }
        if (st == RS_OK) st = rs::make_layout(global_shape, ndim, src_mesh_shape, src_mesh_ndim, src_spec, (flags & RS_EVEN_ONLY) != 0, &P->A);
        if (st == RS_OK) st = rs::make_layout(global_shape, ndim, dst_mesh_shape, dst_mesh_ndim, dst_spec, (flags & RS_EVEN_ONLY) != 0, &P->B);
        if (st == RS_OK) st = rs::build_slices(P);
        if (st == RS_OK) {
            P->exec_order.resize(P->slices.size());
            for (size_t i = 0; i < P->slices.size(); i++) P->exec_order[i] = (int)i;
            if (opts->schedule == RS_SCHED_NONE) rs::choose_senders(P);
            else st = rs::schedule_plan(P);
        }
        if (st == RS_OK) st = rs::build_messages(P);
        if (st == RS_OK) st = rs::build_tables(P);
        if (st == RS_OK && !(flags & RS_HOST_ONLY)) st = upload(P);
    } catch (const std::bad_alloc &) {
        st = RS_ENOMEM;
    }
    if (st != RS_OK) { reshard_plan_destroy(h); return st; }
    *out_plan = h;
    return RS_OK;
}

rs_status reshard_plan_group(const rs_plan *const *plans, int32_t n_plans, uint32_t flags, rs_plan **out_plan) {
    rs::set_error("");
    if (!plans || !out_plan || n_plans < 1) { rs::set_error("null argument or empty group"); return RS_EINVAL; }
    std::vector<const rs::Plan *> members;
    for (int32_t i = 0; i < n_plans; i++) {
        if (!plans[i] || plans[i]->p.group_src || !plans[i]->p.src_owner.empty()) { rs::set_error("a member is null, is itself a group or was built with src_owner"); return RS_EINVAL; }
        members.push_back(&plans[i]->p);
    }
    rs_plan *h = new (std::nothrow) rs_plan();
    if (!h) return RS_ENOMEM;
    rs::Plan *G = &h->p;
    G->flags = flags;
    G->elem_bytes = members[0]->elem_bytes;
    G->tune = members[0]->tune;
    G->A.ndim = G->B.ndim = 0;
    rs_status st;
    try {
        st = (flags & RS_HOST_ONLY) ? RS_OK : query_device(G);
        if (st == RS_OK) st = rs::build_group(G, members);
        if (st == RS_OK && !(flags & RS_HOST_ONLY)) st = upload(G);
    } catch (const std::bad_alloc &) {
        st = RS_ENOMEM;
    }
    if (st != RS_OK) { reshard_plan_destroy(h); return st; }
    *out_plan = h;
    return RS_OK;
}

void reshard_plan_destroy(rs_plan *plan) {
    if (!plan) return;
    for (void *ev : plan->p.events) cudaEventDestroy(static_cast<cudaEvent_t>(ev));
    for (void *st : plan->p.streams) if (st) cudaStreamDestroy(static_cast<cudaStream_t>(st));
    if (plan->p.dev_blob) cudaFree(plan->p.dev_blob);
    delete plan;
}

rs_status reshard_plan_info(const rs_plan *plan, rs_plan_info *out) {
    if (!plan || !out) return RS_EINVAL;
    const rs::Plan &P = plan->p;
    std::memset(out, 0, sizeof(*out));
    out->ndim = P.A.ndim;
    out->elem_bytes = P.elem_bytes;
    out->n_src = P.A.n_dev;
    out->n_dst = P.B.n_dev;
    out->n_slices = (int32_t)P.slices.size();
    out->n_messages = (int32_t)P.messages.size();
    if (P.group_src) {                                        // a group: counts and byte totals only
        out->ndim = 0;
        out->n_slices = P.op[RS_OP_EXECUTE].info.n_tasks;
        out->n_messages = 0;
        out->tensor_bytes = out->unique_read_bytes = P.op[RS_OP_EXECUTE].info.read_bytes;
        out->write_bytes = P.op[RS_OP_EXECUTE].info.write_bytes;
        out->device = P.device;
        return RS_OK;
    }
    int64_t tb = P.elem_bytes;
    for (int d = 0; d < P.A.ndim; d++) tb *= P.A.shape[d];
    out->tensor_bytes = tb;
    out->src_shard_bytes = P.A.shard_elems() * P.elem_bytes;
    out->dst_shard_bytes = P.B.shard_elems() * P.elem_bytes;
    out->unique_read_bytes = tb;
    out->write_bytes = tb * P.r_B;
    out->max_sender_bytes = P.max_sender_bytes;
    out->arena_bytes = P.arena_bytes;
    out->lb_mode = (P.flags & RS_LB_NAIVE) ? RS_LB_NAIVE : RS_LB_GREEDY;
    out->device = P.device;
    return RS_OK;
}

rs_status reshard_op_info(const rs_plan *plan, int32_t op, rs_op_info *out) {
    if (!plan || !out || op < 0 || op >= rs::RS_N_OPS) return RS_EINVAL;
    *out = plan->p.op[op].info;
    return RS_OK;
}

rs_status reshard_op_tables(const rs_plan *plan, int32_t op, void *tasks, void *dsts, void *segs) {
    if (!plan || op < 0 || op >= rs::RS_N_OPS) return RS_EINVAL;
    const rs::OpTables &o = plan->p.op[op];
    if (tasks) std::memcpy(tasks, o.tasks.data(), o.tasks.size() * sizeof(RsTask));
    if (dsts) std::memcpy(dsts, o.dsts.data(), o.dsts.size() * sizeof(RsDst));
    if (segs) std::memcpy(segs, o.segs.data(), o.segs.size() * sizeof(RsSeg));
    return RS_OK;
}

rs_status reshard_op_tiles(const rs_plan *plan, int32_t op, int64_t first_tile, int64_t n_tiles, void *tiles) {
    if (!plan || !tiles || op < 0 || op >= rs::RS_N_OPS) return RS_EINVAL;
    const rs::OpTables &o = plan->p.op[op];
    if (first_tile < 0 || n_tiles < 0 || first_tile + n_tiles > o.info.n_tiles) { rs::set_error("tile range out of bounds"); return RS_EINVAL; }
    RsTile *out = static_cast<RsTile *>(tiles);
    for (int64_t i = 0; i < n_tiles; i++) {                   // the routine the kernels run (tables.h), on the host
        uint32_t task, u;
        rs_tile_locate(o.segs.data(), (uint32_t)o.segs.size(), (uint32_t)(first_tile + i), &task, &u);
        out[i] = rs_tile_decode(o.tasks[task], task, u);
    }
    return RS_OK;
}

rs_status reshard_plan_local_shape(const rs_plan *plan, int32_t side, int64_t *out) {
    if (plan && plan->p.group_src) { rs::set_error("not available for a plan group"); return RS_EINVAL; }
    if (!plan || !out || (side != RS_SRC && side != RS_DST)) return RS_EINVAL;
    const rs::Layout &L = side == RS_SRC ? plan->p.A : plan->p.B;
    for (int d = 0; d < L.ndim; d++) out[d] = L.local[d];
    return RS_OK;
}

rs_status reshard_plan_device_box(const rs_plan *plan, int32_t side, int32_t dev, int64_t *lo, int64_t *hi) {
    if (plan && plan->p.group_src) { rs::set_error("not available for a plan group"); return RS_EINVAL; }
    if (!plan || !lo || !hi || (side != RS_SRC && side != RS_DST)) return RS_EINVAL;
    const rs::Layout &L = side == RS_SRC ? plan->p.A : plan->p.B;
    if (dev < 0 || dev >= L.n_dev) return RS_EINVAL;
    rs::device_box(L, dev, lo, hi);
    return RS_OK;
}

rs_status reshard_plan_slice(const rs_plan *plan, int32_t i, int64_t *lo, int64_t *hi, int32_t *sender,
                             int32_t *n_senders, int32_t *senders, int32_t *n_receivers, int32_t *receivers) {
    if (!plan || i < 0 || (size_t)i >= plan->p.slices.size()) return RS_EINVAL;
    const rs::Slice &S = plan->p.slices[(size_t)i];
    for (int d = 0; d < plan->p.A.ndim; d++) {
        if (lo) lo[d] = S.lo[d];
        if (hi) hi[d] = S.hi[d];
    }
    if (sender) *sender = S.sender;
    if (n_senders) *n_senders = (int32_t)S.senders.size();
    if (senders) std::copy(S.senders.begin(), S.senders.end(), senders);
    if (n_receivers) *n_receivers = (int32_t)S.receivers.size();
    if (receivers) std::copy(S.receivers.begin(), S.receivers.end(), receivers);
    return RS_OK;
}

rs_status reshard_plan_schedule(const rs_plan *plan, rs_schedule_info *info, int32_t *sender_host, int64_t *start,
                                int32_t *order) {
    if (!plan) return RS_EINVAL;
    const rs::Plan &P = plan->p;
    const rs::Schedule &S = P.sched;
    if (S.algorithm == RS_SCHED_NONE) { rs::set_error("plan was built without a schedule"); return RS_EINVAL; }
    if (info) {
        std::memset(info, 0, sizeof(*info));
        info->algorithm = S.algorithm; info->winner = S.winner;
        info->n_tasks = (int32_t)P.slices.size(); info->n_rounds = S.n_rounds;
        info->n_src_hosts = (P.A.n_dev + S.src_dph - 1) / S.src_dph;
        info->n_dst_hosts = (P.B.n_dev + S.dst_dph - 1) / S.dst_dph;
        info->dfs_finished = S.dfs_finished; info->dfs_nodes = S.dfs_nodes;
        info->makespan = S.makespan; info->busiest_host_bytes = S.busiest_host_bytes;
    }
    if (sender_host) std::copy(S.sender_host.begin(), S.sender_host.end(), sender_host);
    if (start) std::copy(S.start.begin(), S.start.end(), start);
    if (order) std::copy(S.order.begin(), S.order.end(), order);
    return RS_OK;
}

rs_status reshard_plan_sender_bytes(const rs_plan *plan, int64_t *out) {
    if (plan && plan->p.group_src) { rs::set_error("not available for a plan group"); return RS_EINVAL; }
    if (!plan || !out) return RS_EINVAL;
    std::copy(plan->p.sender_bytes.begin(), plan->p.sender_bytes.end(), out);
    return RS_OK;
}

rs_status reshard_plan_message(const rs_plan *plan, int32_t m, int32_t *sender, int32_t *receiver,
                               int64_t *offset, int64_t *bytes, int32_t *n_slice_ids, int32_t *slice_ids) {
    if (!plan || m < 0 || (size_t)m >= plan->p.messages.size()) return RS_EINVAL;
    const rs::Message &M = plan->p.messages[(size_t)m];
    if (sender) *sender = M.sender;
    if (receiver) *receiver = M.receiver;
    if (offset) *offset = M.offset;
    if (bytes) *bytes = M.bytes;
    if (n_slice_ids) *n_slice_ids = (int32_t)M.slice_ids.size();
    if (slice_ids) std::copy(M.slice_ids.begin(), M.slice_ids.end(), slice_ids);
    return RS_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// the data path

namespace {

int ptr_align(const void *p) {
    uintptr_t x = reinterpret_cast<uintptr_t>(p);
    int a = 16;
    while (a > 1 && (x % (uintptr_t)a)) a /= 2;
    return a;
}

// RS_PATH_TMAP: one CUtensorMap per buffer that has a geometry, from the pointers of THIS call (plans are pointer
// agnostic).  cuTensorMapEncodeTiled is a host-side routine of the driver, reached through cudaGetDriverEntryPoint so
// that the library links against the runtime only.
typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                              const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

rs_status encode_tmaps(const rs::OpTables &op, const RsPtrTable &pt, unsigned char *out /* RS_TMAP_TABLE_BYTES */) {
    static encode_fn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess) fn = reinterpret_cast<encode_fn>(p);
    });
    if (!fn) { rs::set_error("cuTensorMapEncodeTiled is not available"); return RS_ECUDA; }
    static_assert(sizeof(CUtensorMap) == 128, "CUtensorMap size");
    std::memset(out, 0, RS_TMAP_TABLE_BYTES);
    for (int side = 0; side < 2; side++)
        for (int b = 0; b < RS_TMAP_BUFS; b++) {
            const RsTmapGeom &G = side == 0 ? op.tmap_src[b] : op.tmap_dst[b];
            void *base = side == 0 ? const_cast<char *>(pt.src[b]) : pt.dst[b];
            if (!G.valid || !base) continue;
            const int64_t cap = side == 0 ? op.src_cap : op.dst_cap;
            const cuuint64_t dims[2] = {(cuuint64_t)(G.pitch / RS_TMAP_ELEM), (cuuint64_t)((cap + G.pitch - 1) / G.pitch)};
            const cuuint64_t strides[1] = {(cuuint64_t)G.pitch};
            const cuuint32_t box[2] = {G.box_cols / RS_TMAP_ELEM, G.box_rows}, estr[2] = {1, 1};
            CUtensorMap *m = reinterpret_cast<CUtensorMap *>(out + (size_t)(side * RS_TMAP_BUFS + b) * 128);
            const CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) { rs::set_error("cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")"); return RS_ECUDA; }
        }
    return RS_OK;
}

// one launch of operation `opi` on the given buffers
rs_status run_op(const rs_plan *plan, int opi, const void *const *src, int n_src, void *const *dst, int n_dst,
                 const char *used_src, void *stream, uint32_t tile_begin = 0, uint32_t tile_end = 0,
                 const char *used_dst = nullptr, const RsOpDev *static_dev = nullptr /* reshard_execute_static: tables elsewhere */) {
    rs::set_error("");
    if (!plan || !src || !dst) { rs::set_error("null argument"); return RS_EINVAL; }
    const rs::Plan &P = plan->p;
    if (!P.dev_blob && !static_dev) { rs::set_error("plan was built with RS_HOST_ONLY"); return RS_EINVAL; }
    const rs::OpTables &op = P.op[opi];
    if (op.info.n_tiles == 0) return RS_OK;
    RsPtrTable pt;
    const bool small = n_src <= RS_PTRS_SMALL && n_dst <= RS_PTRS_SMALL;   // then the kernels get the 256-byte table
    for (int i = 0; i < RS_PTRS_SMALL; i++) { pt.src[i] = nullptr; pt.dst[i] = nullptr; }
    int align = op.info.vec_bytes;
    for (int i = 0; i < n_src; i++) {
        pt.src[i] = static_cast<const char *>(src[i]);
        if (used_src && !used_src[i]) continue;
        if (!src[i]) { rs::set_error("a source shard pointer the plan reads is null"); return RS_EINVAL; }
        align = std::min(align, ptr_align(src[i]));
    }
    for (int i = 0; i < n_dst; i++) {
        pt.dst[i] = static_cast<char *>(dst[i]);
        if (used_dst && !used_dst[i]) continue;                // a rank of the multi-process executor: shards it never writes
        if (!dst[i]) { rs::set_error("a destination pointer is null"); return RS_EINVAL; }
        align = std::min(align, ptr_align(dst[i]));
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    RsOpDev dev = static_dev ? *static_dev : op.dev;
    if (tile_end > tile_begin) { dev.tile_base = tile_begin; dev.n_tiles = tile_end - tile_begin; }   // one slab
    const int64_t n_tiles = dev.n_tiles;
    const bool bulk_family = op.info.path == RS_PATH_BULK || op.info.path == RS_PATH_BULK_SHIFT || op.info.path == RS_PATH_TMAP;
    const bool as_bulk = op.info.path == RS_PATH_BULK || op.info.path == RS_PATH_TMAP;   // aligned TMA plans
    const int warps = op.info.block / 32;
    const bool pdl = !P.tune.no_pdl && !static_dev;          // (the shared table array is rewritten between launches: full stream order)
    // shifted stores from registers; realigning the rows in the ring and storing them with cp.async.bulk (rs_tuning.shift_mode = 2) is 3-4 % faster for rows
    // >= 4 KiB on an idle chip (u4 6.31 against 6.10 TB/s) and 12-18 % slower on a power-limited one (5.3 against 5.97): more instructions per tile (config.h)
    const int shift_mode = P.tune.shift_mode == rs::RS_SHIFT_REG || P.tune.shift_mode == rs::RS_SHIFT_BULK ? P.tune.shift_mode : rs::RS_SHIFT_REG;
    if (as_bulk && align == 16) {
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(op.info.grid, (n_tiles + warps - 1) / warps));
        dev.early_trigger = grid >= P.sm_count;
        // rate matching: the launch as a whole offers pace_permille / 1000 of the DRAM peak
        const int permille = P.tune.pace_permille > 0 ? P.tune.pace_permille : P.tune.pace_permille < 0 ? 0 : op.pace_permille;
        const int burst = (P.tune.pace_burst > 0 ? std::min(P.tune.pace_burst, 255) : RS_PACE_BURST) | (P.tune.pace_adapt > 0 ? 0 : 0x100);
        const float pace = permille > 0 ? (float)((double)grid * warps / (P.dram_peak_gbs * permille / 1000.0)) : 0.f;
        if (op.info.path == RS_PATH_TMAP && small) {          // tensor maps of this call's pointers, then the same ring kernel
            alignas(64) unsigned char tm[RS_TMAP_TABLE_BYTES];
            rs_status ts = encode_tmaps(op, pt, tm);
            if (ts != RS_OK) return ts;
            e = rs::launch_tmap(dev, pt, tm, grid, op.info.block, op.info.smem_bytes, op.stages, op.lookahead,
                                (uint32_t)op.info.tile_bytes, pace, burst, pdl, st);
        } else
        e = rs::launch_bulk(dev, pt, small, grid, op.info.block, op.info.smem_bytes, op.stages, op.lookahead,
                            (uint32_t)op.info.tile_bytes, pace, burst, pdl, st);
    } else if (op.info.path == RS_PATH_BULK_SHIFT) {          // layout not 16-byte aligned: TMA loads, shifted stores
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(op.info.grid, (n_tiles + warps - 1) / warps));
        dev.early_trigger = grid >= P.sm_count;
        const int permille = P.tune.pace_permille > 0 ? P.tune.pace_permille : P.tune.pace_permille < 0 ? 0 : op.pace_permille;
        const float pace = permille > 0 ? (float)((double)grid * warps / (P.dram_peak_gbs * permille / 1000.0)) : 0.f;
        e = rs::launch_bulk_shift(dev, pt, small, grid, op.info.block, op.info.smem_bytes, op.stages, op.lookahead,
                                  op.shift_stage, shift_mode, pace, P.tune.pace_burst > 0 ? std::min(P.tune.pace_burst, 255) : RS_PACE_BURST, pdl, st);
    } else if (as_bulk && op.alt_stage) {                     // aligned plan, under-aligned pointers: same tiles, shifted stores
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(P.max_ctas > 0 ? std::min(P.sm_count, P.max_ctas) : P.sm_count,
                                                                     (n_tiles + op.alt_warps - 1) / op.alt_warps));
        dev.early_trigger = grid >= P.sm_count;
        e = rs::launch_bulk_shift(dev, pt, small, grid, op.alt_warps * 32, op.alt_smem, op.alt_stages, op.alt_stages - 1,
                                  op.alt_stage, shift_mode, 0.f, RS_PACE_BURST, pdl, st);
    } else {                                                  // register paths
        int64_t cap = bulk_family ? (int64_t)P.sm_count * RS_LSU_CTAS_DEFAULT : op.info.grid;
        if (P.max_ctas > 0) cap = std::min<int64_t>(cap, P.max_ctas);
        // 8 warps per CTA, every warp a worker (warp-major over the grid); an operation with fewer tiles than that still
        // gets one CTA on every SM while it has a tile for each: its dependents may then be launched at entry
        int64_t want = (n_tiles + 7) / 8;
        if (want < P.sm_count) want = std::min<int64_t>(n_tiles, P.sm_count);
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(want, cap));
        dev.early_trigger = grid >= P.sm_count;
        // measured (1 + 1 GiB-class operations): 8-byte aligned rows of 56-250 bytes 0.59 -> 1.78 and 1.44 -> 3.74 TB/s at 8-byte vectors;
        // 4-byte aligned: 28-byte rows 0.32 -> 0.78, but 100-byte rows 1.89 -> 1.08; 1-byte aligned: 2-3 byte rows 0.14 -> 0.57, 8-byte rows a loss
        const int64_t narrow_below = align >= 8 ? RS_NARROW_MAX_RUN : align == 4 ? 48 : 8;
        const bool narrow = P.tune.lsu_narrow > 0 || (P.tune.lsu_narrow == 0 && op.mean_run_bytes < narrow_below);
        if (align < 16 && narrow) e = rs::launch_narrow(dev, pt, small, align, grid, pdl, st);   // short rows: the layout's own vector width
        else if (align < 16) e = rs::launch_shift(dev, pt, small, grid, pdl, st);   // any alignment, still 16-byte accesses
        else {
            bool generic = false;
            for (const RsTask &T : op.tasks) generic = generic || T.kind == RS_TILING_GENERIC;
            e = rs::launch_lsu(dev, pt, small, generic, grid, pdl, st);
        }
    }
    if (e != cudaSuccess) return cuda_fail(e, "kernel launch");
    return RS_OK;
}

}  // namespace

extern "C" {

rs_status reshard_execute(const rs_plan *plan, const void *const *src_shards, void *const *dst_shards,
                          void *cuda_stream) {
    if (!plan) return RS_EINVAL;
    const rs::Plan &P = plan->p;
    return run_op(plan, RS_OP_EXECUTE, src_shards, P.A.n_dev, dst_shards, P.B.n_dev, P.used_src.data(), cuda_stream, 0, 0,
                  P.src_owner.empty() ? nullptr : P.used_dst.data());
}

rs_status reshard_execute_static(const rs_plan *plan, const void *const *src_shards, void *const *dst_shards,
                                 void *cuda_stream) {
    rs::set_error("");
    if (!plan || !src_shards || !dst_shards) { rs::set_error("null argument"); return RS_EINVAL; }
    const rs::Plan &P = plan->p;
    if (!P.src_owner.empty() || P.group_src) { rs::set_error("reshard_execute_static: not for plans built with src_owner or for plan groups"); return RS_EINVAL; }
    const rs::OpTables &o = P.op[RS_OP_EXECUTE];
    if (o.info.n_tiles == 0) return RS_OK;
    const size_t b_tasks = o.tasks.size() * sizeof(RsTask), b_dsts = o.dsts.size() * sizeof(RsDst), b_segs = o.segs.size() * sizeof(RsSeg);
    const size_t off_dsts = round256(b_tasks), off_segs = off_dsts + round256(b_dsts), total = off_segs + round256(b_segs);
    if (total > (size_t)RS_STATIC_TABLE_BYTES) {
        rs::set_error("reshard_execute_static: the execute tables of this plan take " + std::to_string(total) + " bytes (" +
                      std::to_string(o.tasks.size()) + " unit tasks), the static device array holds " + std::to_string(RS_STATIC_TABLE_BYTES) +
                      "; use reshard_execute");
        return RS_EUNSUPPORTED;
    }
    void *base_v = nullptr;                                    // device address of the file-scope array on the current device
    cudaError_t e = rs::static_tables(&base_v);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(static tables)");
    static std::once_flag smem_once;                           // a host-only plan never went through upload()
    static cudaError_t smem_err = cudaSuccess;
    std::call_once(smem_once, [] { smem_err = rs::prepare_bulk(RS_SMEM_MAX); });
    if (smem_err != cudaSuccess) return cuda_fail(smem_err, "cudaFuncSetAttribute(rs_copy_bulk)");
    char *base = static_cast<char *>(base_v);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // Three copies straight from the plan's host tables (pageable memory: staged before the call returns), in stream order
    // before the launch.  Every byte the kernels read is written here, so nothing of the previous call's contents is used
    // and nothing has to start at zero.
    e = cudaMemcpyAsync(base, o.tasks.data(), b_tasks, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && b_dsts) e = cudaMemcpyAsync(base + off_dsts, o.dsts.data(), b_dsts, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && b_segs) e = cudaMemcpyAsync(base + off_segs, o.segs.data(), b_segs, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync(static tables)");
    RsOpDev dev{};
    dev.tasks = reinterpret_cast<const RsTask *>(base);
    dev.dsts = reinterpret_cast<const RsDst *>(base + off_dsts);
    dev.segs = reinterpret_cast<const RsSeg *>(base + off_segs);
    dev.n_segs = (uint32_t)o.segs.size();
    dev.seg_tiles = o.segs.empty() ? 0 : o.segs[0].n_members * o.segs[0].tiles_each;
    for (const RsSeg &sg : o.segs) if (sg.n_members * sg.tiles_each != dev.seg_tiles) dev.seg_tiles = 0;
    dev.n_tasks = (uint32_t)o.tasks.size();
    dev.n_dsts = (uint32_t)o.dsts.size();
    dev.early_trigger = 0;
    dev.tile_base = 0;
    dev.n_tiles = (uint32_t)o.info.n_tiles;
    return run_op(plan, RS_OP_EXECUTE, src_shards, P.A.n_dev, dst_shards, P.B.n_dev, P.used_src.data(), cuda_stream, 0, 0, nullptr, &dev);
}

rs_status reshard_execute_strategy(const rs_plan *plan, int32_t strategy, const void *const *src_shards,
                                   void *const *dst_shards, void *cuda_stream) {
    if (!plan) return RS_EINVAL;
    const rs::Plan &P = plan->p;
    if (strategy == RS_STRATEGY_BROADCAST) return reshard_execute(plan, src_shards, dst_shards, cuda_stream);
    if (!P.src_owner.empty()) { rs::set_error("not available for a plan built with src_owner"); return RS_EINVAL; }
    if (!(P.flags & RS_WITH_STRATEGIES)) { rs::set_error("plan was built without RS_WITH_STRATEGIES"); return RS_EINVAL; }
    if (strategy == RS_STRATEGY_SENDRECV)
        return run_op(plan, RS_OP_SENDRECV, src_shards, P.A.n_dev, dst_shards, P.B.n_dev, P.used_src.data(), cuda_stream);
    if (strategy != RS_STRATEGY_ALLGATHER && strategy != RS_STRATEGY_ALLGATHER_LOCAL) { rs::set_error("unknown strategy"); return RS_EINVAL; }
    const int scatter = strategy == RS_STRATEGY_ALLGATHER ? RS_OP_AG_SCATTER : RS_OP_AGL_SCATTER;
    const int gather = strategy == RS_STRATEGY_ALLGATHER ? RS_OP_AG_GATHER : RS_OP_AGL_GATHER;
    rs_status st = run_op(plan, scatter, src_shards, P.A.n_dev, dst_shards, P.B.n_dev, P.used_src.data(), cuda_stream);
    if (st != RS_OK) return st;                               // phase 2 reads what phase 1 wrote: same stream, in order
    return run_op(plan, gather, dst_shards, P.B.n_dev, dst_shards, P.B.n_dev, nullptr, cuda_stream);
}

rs_status reshard_pack(const rs_plan *plan, const void *const *src_shards, void *msg_arena, void *cuda_stream) {
    if (plan && (plan->p.group_src || !plan->p.src_owner.empty())) { rs::set_error("not available for a plan group or a plan built with src_owner"); return RS_EINVAL; }
    if (!plan) return RS_EINVAL;
    void *dst[1] = {msg_arena};
    return run_op(plan, RS_OP_PACK, src_shards, plan->p.A.n_dev, dst, 1, plan->p.used_src.data(), cuda_stream);
}

rs_status reshard_unpack(const rs_plan *plan, const void *msg_arena, void *const *dst_shards, void *cuda_stream) {
    if (plan && (plan->p.group_src || !plan->p.src_owner.empty())) { rs::set_error("not available for a plan group or a plan built with src_owner"); return RS_EINVAL; }
    if (!plan) return RS_EINVAL;
    const void *src[1] = {msg_arena};
    return run_op(plan, RS_OP_UNPACK, src, 1, dst_shards, plan->p.B.n_dev, nullptr, cuda_stream);
}

int64_t reshard_host_workspace_bytes(const rs_plan *plan) {
    if (plan && (plan->p.group_src || !plan->p.src_owner.empty())) return -1;
    if (!plan) return -1;
    const rs::Plan &P = plan->p;
    int64_t n_used = 0;
    for (char u : P.used_src) n_used += u ? 1 : 0;
    return n_used * (int64_t)round256((size_t)(P.A.shard_elems() * P.elem_bytes)) +
           (int64_t)P.B.n_dev * (int64_t)round256((size_t)(P.B.shard_elems() * P.elem_bytes));
}

rs_status reshard_execute_host(const rs_plan *plan, const void *const *src_shards_host, void *const *dst_shards_host,
                               void *workspace, void *cuda_stream, int64_t *h2d_bytes, int64_t *d2h_bytes) {
    if (plan && (plan->p.group_src || !plan->p.src_owner.empty())) { rs::set_error("not available for a plan group or a plan built with src_owner"); return RS_EINVAL; }
    rs::set_error("");
    if (!plan || !src_shards_host || !dst_shards_host || !workspace) { rs::set_error("null argument"); return RS_EINVAL; }
    const rs::Plan &P = plan->p;
    if (!P.dev_blob) { rs::set_error("plan was built with RS_HOST_ONLY"); return RS_EINVAL; }
    if (reinterpret_cast<uintptr_t>(workspace) % 256) { rs::set_error("workspace must be 256-byte aligned"); return RS_EINVAL; }
    std::lock_guard<std::mutex> lock(P.host_mu);               // the side streams and events are the plan's
    { rs_status hs = host_streams(P); if (hs != RS_OK) return hs; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaStream_t up_st = static_cast<cudaStream_t>(P.streams[0]), down_st = static_cast<cudaStream_t>(P.streams[1]);
    const size_t sb = (size_t)(P.A.shard_elems() * P.elem_bytes), db = (size_t)(P.B.shard_elems() * P.elem_bytes);
    const void *src_dev[RS_MAX_DEVICES];
    void *dst_dev[RS_MAX_DEVICES];
    char *w = static_cast<char *>(workspace);
    // Replicas are identical by precondition, so only shards the chosen senders read get device space and
    // uploads: the bytes crossing the link are the lower bound size(D).
    for (int r = 0; r < P.A.n_dev; r++) {
        src_dev[r] = nullptr;
        if (!P.used_src[(size_t)r]) continue;
        if (!src_shards_host[r]) { rs::set_error("a source shard pointer the plan reads is null"); return RS_EINVAL; }
        src_dev[r] = w;
        w += round256(sb);
    }
    for (int q = 0; q < P.B.n_dev; q++) {
        if (!dst_shards_host[q]) { rs::set_error("a destination pointer is null"); return RS_EINVAL; }
        dst_dev[q] = w;
        w += round256(db);
    }
    // Pipeline over slabs of tensor dim 0 (PAPER.md:137's chunk pipelining, applied to the host link):
    //   upload stream:   H2D slab 0 | H2D slab 1 | ...
    //   caller's stream:            | kernel 0   | kernel 1 | ...
    //   download stream:                         | D2H 0    | D2H 1 | ...
    auto ev = [&](size_t i) { return static_cast<cudaEvent_t>(P.events[i]); };
    const size_t n = P.slabs.size();
    cudaError_t e = cudaEventRecord(ev(2 * n), st);            // everything is ordered after the caller's prior work
    if (e == cudaSuccess) e = cudaStreamWaitEvent(up_st, ev(2 * n), 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(down_st, ev(2 * n), 0);
    if (e != cudaSuccess) return cuda_fail(e, "stream fork");
    int64_t up = 0, down = 0;
    for (size_t c = 0; c < n; c++) {
        const rs::HostSlab &S = P.slabs[c];
        for (const rs::HostCopy &h : S.up) {
            e = cudaMemcpyAsync(const_cast<char *>(static_cast<const char *>(src_dev[h.dev])) + h.off,
                                static_cast<const char *>(src_shards_host[h.dev]) + h.off, (size_t)h.bytes,
                                cudaMemcpyHostToDevice, up_st);
            if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync(H2D)");
            up += h.bytes;
        }
        if ((e = cudaEventRecord(ev(2 * c), up_st)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
        if ((e = cudaStreamWaitEvent(st, ev(2 * c), 0)) != cudaSuccess) return cuda_fail(e, "cudaStreamWaitEvent");
        if (S.tile_end > S.tile_begin) {
            rs_status rc = run_op(plan, rs::RS_OP_SLABS, src_dev, P.A.n_dev, dst_dev, P.B.n_dev, P.used_src.data(),
                                  cuda_stream, S.tile_begin, S.tile_end);
            if (rc != RS_OK) return rc;
        }
        if ((e = cudaEventRecord(ev(2 * c + 1), st)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
        if ((e = cudaStreamWaitEvent(down_st, ev(2 * c + 1), 0)) != cudaSuccess) return cuda_fail(e, "cudaStreamWaitEvent");
        for (const rs::HostCopy &h : S.down) {
            e = cudaMemcpyAsync(static_cast<char *>(dst_shards_host[h.dev]) + h.off,
                                static_cast<char *>(dst_dev[h.dev]) + h.off, (size_t)h.bytes, cudaMemcpyDeviceToHost,
                                down_st);
            if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync(D2H)");
            down += h.bytes;
        }
    }
    e = cudaEventRecord(ev(2 * n + 1), down_st);               // join: the caller's stream sees the downloads
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev(2 * n + 1), 0);
    if (e != cudaSuccess) return cuda_fail(e, "stream join");
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return RS_OK;
}

// ---- CUDA IPC plumbing of the multi-process executor ------------------------------------------

namespace {
struct IpcWire {                                               // RS_IPC_HANDLE_BYTES on the wire
    cudaIpcMemHandle_t handle;                                 // 64 bytes: the exporting ALLOCATION
    int64_t offset;                                            // of the exported pointer inside it
    int64_t reserved;
};
static_assert(sizeof(IpcWire) == RS_IPC_HANDLE_BYTES, "rs ipc handle layout");
std::mutex g_ipc_mu;
std::vector<std::pair<cudaIpcMemHandle_t, void *>> g_ipc_open;  // one mapping per exporting allocation and process
}  // namespace

rs_status reshard_ipc_export(const void *dev_ptr, void *handle_out) {
    rs::set_error("");
    if (!dev_ptr || !handle_out) { rs::set_error("null argument"); return RS_EINVAL; }
    typedef int (*range_fn)(unsigned long long *, size_t *, unsigned long long);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &q);
    if (e != cudaSuccess || !fn) return cuda_fail(e, "cudaGetDriverEntryPoint(cuMemGetAddressRange)");
    unsigned long long base = 0;
    size_t size = 0;
    if (reinterpret_cast<range_fn>(fn)(&base, &size, (unsigned long long)reinterpret_cast<uintptr_t>(dev_ptr)) != 0) {
        rs::set_error("cuMemGetAddressRange failed: not a device allocation");
        return RS_ECUDA;
    }
    IpcWire w;
    std::memset(&w, 0, sizeof(w));
    e = cudaIpcGetMemHandle(&w.handle, reinterpret_cast<void *>(static_cast<uintptr_t>(base)));
    if (e != cudaSuccess) return cuda_fail(e, "cudaIpcGetMemHandle");
    w.offset = (int64_t)(reinterpret_cast<uintptr_t>(dev_ptr) - (uintptr_t)base);
    std::memcpy(handle_out, &w, sizeof(w));
    return RS_OK;
}

rs_status reshard_ipc_import(const void *handle, void **dev_ptr_out) {
    rs::set_error("");
    if (!handle || !dev_ptr_out) { rs::set_error("null argument"); return RS_EINVAL; }
    IpcWire w;
    std::memcpy(&w, handle, sizeof(w));
    std::lock_guard<std::mutex> lock(g_ipc_mu);
    for (auto &m : g_ipc_open)
        if (std::memcmp(&m.first, &w.handle, sizeof(w.handle)) == 0) { *dev_ptr_out = static_cast<char *>(m.second) + w.offset; return RS_OK; }
    void *base = nullptr;
    cudaError_t e = cudaIpcOpenMemHandle(&base, w.handle, cudaIpcMemLazyEnablePeerAccess);
    if (e != cudaSuccess) return cuda_fail(e, "cudaIpcOpenMemHandle");
    g_ipc_open.emplace_back(w.handle, base);
    *dev_ptr_out = static_cast<char *>(base) + w.offset;
    return RS_OK;
}

rs_status reshard_ipc_release_all(void) {
    std::lock_guard<std::mutex> lock(g_ipc_mu);
    cudaError_t first = cudaSuccess;
    for (auto &m : g_ipc_open) {
        cudaError_t e = cudaIpcCloseMemHandle(m.second);
        if (e != cudaSuccess && first == cudaSuccess) first = e;
    }
    g_ipc_open.clear();
    return first == cudaSuccess ? RS_OK : cuda_fail(first, "cudaIpcCloseMemHandle");
}

rs_status reshard_pipeline_simulate(const rs_pipeline_opts *opts, rs_pipeline_result *result, int32_t *op_kind,
                                    int32_t *op_micro_batch, int64_t *op_start, int64_t *op_end) {
    rs::set_error("");
    if (!opts) { rs::set_error("null argument"); return RS_EINVAL; }
    try {
        return rs::pipeline_simulate(*opts, result, op_kind, op_micro_batch, op_start, op_end);
    } catch (const std::bad_alloc &) {
        return RS_ENOMEM;
    }
}

int32_t reshard_pipeline_least_delay(int32_t schedule, int32_t n_stages, int32_t stage, int32_t n_micro_batches,
                                     int64_t fwd, int64_t bwd, int64_t bwd_act, int64_t comm_bwd) {
    if (n_stages < 1 || stage < 1 || stage > n_stages || n_micro_batches < 1) return -1;
    return rs::pipeline_least_delay(schedule, n_stages, stage, n_micro_batches, fwd, bwd, bwd_act, comm_bwd);
}

int64_t reshard_launch_count(void) { return rs::launch_count(); }

const char *reshard_strerror(rs_status s) {
    switch (s) {
        case RS_OK: return "ok";
        case RS_EINVAL: return "invalid argument";
        case RS_ESPEC: return "bad sharding spec";
        case RS_EDIVIS: return "tensor dim not divisible by its sharding degree";
        case RS_EUNSUPPORTED: return "unsupported size";
        case RS_ENOMEM: return "out of memory";
        case RS_ECUDA: return "CUDA error";
    }
    return "unknown status";
}

const char *reshard_last_error(void) { return rs::last_error().c_str(); }

const char *reshard_version(void) { return "reshard-b200 0.1 (sm_100a)"; }

}  // extern "C"

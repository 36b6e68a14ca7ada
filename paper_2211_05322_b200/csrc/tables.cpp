// tables.cpp -- step a5: unit tasks -> collapsed copy tasks -> flat tile tables for the three
// operations (execute / pack / unpack), plus the per-operation launch configuration.
// Paper analogue: "choose the better result as the schedule to launch broadcasts";
// north_star item (1): "emits a flat task table".  No CUDA here.
#include <algorithm>
#include <cstdlib>
#include <cstring>

#include "config.h"
#include "plan.hpp"

namespace rs {

namespace {

struct BoxDesc {                         // one box seen from both sides, per TENSOR dim, in bytes
    int ndim;
    int64_t ext[RS_MAX_NDIM];            // elements
    int64_t sstride[RS_MAX_NDIM];
    int64_t dstride[RS_MAX_NDIM];
};

// dense row-major byte strides of a local array
void dense_strides(const int64_t *shape, int ndim, int64_t e, int64_t *stride) {
    int64_t s = e;
    for (int d = ndim - 1; d >= 0; d--) { stride[d] = s; s *= shape[d]; }
}

int64_t box_offset(const int64_t *lo, const int64_t *origin, const int64_t *stride, int ndim) {
    int64_t off = 0;
    for (int d = 0; d < ndim; d++) off += (lo[d] - origin[d]) * stride[d];
    return off;
}

// Collapse a box: drop unit dims, merge dims that are contiguous on BOTH sides, turn the innermost
// dim into the byte run if it is dense on both sides.  Returns false if a row dim overflows 32 bits.
bool collapse(const BoxDesc &bx, int64_t e, RsTask *T) {
    int64_t ext[RS_MAX_NDIM + 1], ss[RS_MAX_NDIM + 1], ds[RS_MAX_NDIM + 1];
    int n = 0;
    for (int d = 0; d < bx.ndim; d++) {                       // outermost first
        if (bx.ext[d] == 1) continue;
        if (n > 0 && ss[n - 1] == bx.ext[d] * bx.sstride[d] && ds[n - 1] == bx.ext[d] * bx.dstride[d]) {
            ext[n - 1] *= bx.ext[d];                          // outer dim steps exactly over this one
            ss[n - 1] = bx.sstride[d];
            ds[n - 1] = bx.dstride[d];
        } else {
            ext[n] = bx.ext[d]; ss[n] = bx.sstride[d]; ds[n] = bx.dstride[d];
            n++;
        }
    }
    T->run_bytes = e;
    if (n > 0 && ss[n - 1] == e && ds[n - 1] == e) { T->run_bytes = ext[n - 1] * e; n--; }
    if (n > RS_ROW_DIMS) return false;
    T->nd = n;
    for (int i = 0; i <= RS_ROW_DIMS; i++) { T->ext[i] = 1; T->sstride[i] = 0; T->dstride[i] = 0; }
    for (int i = 0; i < n; i++) {                             // ext[0] = innermost row dim
        int src = n - 1 - i;
        if (ext[src] > 0xFFFFFFFFll) return false;
        T->ext[i] = (uint32_t)ext[src];
        T->sstride[i] = ss[src];
        T->dstride[i] = ds[src];
    }
    return true;
}

int64_t task_rows(const RsTask &T) {
    int64_t r = 1;
    for (int i = 0; i < T.nd; i++) r *= T.ext[i];
    return r;
}

int64_t pow2_align(int64_t x) {                               // largest power of two <= 16 dividing x
    if (x == 0) return 16;
    int64_t a = 1;
    while (a < 16 && x % (a * 2) == 0) a *= 2;
    return a;
}

int env_int(const char *name, int dflt) {
    const char *v = std::getenv(name);
    if (!v || !*v) return dflt;
    return std::atoi(v);
}

// Emit the tiles of one task.  tile_bytes is a multiple of 128.
void emit_tiles(const RsTask &T, uint32_t task_id, int64_t tile_bytes, std::vector<RsTile> *out) {
    const int64_t R = task_rows(T), B = T.run_bytes;
    auto row_offsets = [&](int64_t row, int64_t *so, int64_t *doff) {
        int64_t s = 0, d = 0;
        for (int i = 0; i < T.nd; i++) {
            int64_t c = row % T.ext[i];
            row /= T.ext[i];
            s += c * T.sstride[i];
            d += c * T.dstride[i];
        }
        *so = s; *doff = d;
    };
    if (B > tile_bytes) {                                     // long runs: split every row into column chunks
        int64_t n = (B + tile_bytes - 1) / tile_bytes;
        int64_t chunk = ((B + n - 1) / n + 127) / 128 * 128;
        for (int64_t r = 0; r < R; r++) {
            int64_t so, doff;
            row_offsets(r, &so, &doff);
            for (int64_t c = 0; c < B; c += chunk) {
                RsTile t{};
                t.task = task_id; t.n_rows = 1; t.col_bytes = (uint32_t)std::min(chunk, B - c);
                t.flags = RS_TILE_FAST;
                t.a = (uint64_t)(so + c); t.b = (uint64_t)(doff + c);
                out->push_back(t);
            }
        }
        return;
    }
    const int64_t rpt = std::max<int64_t>(1, tile_bytes / B);  // rows per tile
    const int64_t ext0 = T.nd > 0 ? T.ext[0] : 1;
    if (T.nd <= 1 || ext0 >= rpt) {                           // FAST tiles inside one span of row dim 0
        int64_t n = (ext0 + rpt - 1) / rpt, sz = (ext0 + n - 1) / n;
        for (int64_t span = 0; span < R / ext0; span++) {
            int64_t so, doff;
            row_offsets(span * ext0, &so, &doff);
            for (int64_t r0 = 0; r0 < ext0; r0 += sz) {
                RsTile t{};
                t.task = task_id; t.n_rows = (uint32_t)std::min(sz, ext0 - r0); t.col_bytes = (uint32_t)B;
                t.flags = RS_TILE_FAST;
                t.a = (uint64_t)(so + r0 * T.sstride[0]); t.b = (uint64_t)(doff + r0 * T.dstride[0]);
                out->push_back(t);
            }
        }
        return;
    }
    int64_t n = (R + rpt - 1) / rpt, sz = (R + n - 1) / n;     // GENERIC tiles: any run of linear rows
    for (int64_t r0 = 0; r0 < R; r0 += sz) {
        RsTile t{};
        t.task = task_id; t.n_rows = (uint32_t)std::min(sz, R - r0); t.col_bytes = (uint32_t)B;
        t.flags = 0;
        t.a = (uint64_t)r0; t.b = 0;
        out->push_back(t);
    }
}

// Which kernel an operation takes (rs_op_info.path).  AUTO: runs under 512 B and small aligned operations go to the
// register kernels (they start faster; small operations are launch-bound), 16-byte aligned layouts to the TMA
// kernel, everything else to TMA loads + shifted stores.
int pick_path(uint32_t forced, int64_t align, int64_t min_run, int64_t moved_bytes) {
    const bool bulk_ok = align == 16 && min_run >= 16;
    int path = forced == RS_PATH_LSU ? RS_PATH_LSU : forced == RS_PATH_BULK ? RS_PATH_BULK
             : forced == RS_PATH_BULK_SHIFT ? RS_PATH_BULK_SHIFT
             : min_run < RS_BULK_MIN_RUN ? RS_PATH_LSU
             : bulk_ok ? (moved_bytes <= RS_SMALL_OP_BYTES ? RS_PATH_LSU : RS_PATH_BULK)
             : RS_PATH_BULK_SHIFT;
    if (path == RS_PATH_BULK && !bulk_ok) path = RS_PATH_BULK_SHIFT;   // cp.async.bulk stores need 16-byte everything
    return path;
}

// Launch shape of the two TMA kernels, from measurement on B200.
struct BulkShape { int warps, stages, grid; int64_t tile_bytes; };

BulkShape bulk_shape(const Plan &P, bool shift, int64_t min_run, int64_t read_bytes, int64_t write_bytes) {
    // short runs = many bulk copies per tile: one warp issues them too slowly, so more, smaller pipelines
    // (Table 2 case 9, 512-byte runs: 3.6 TB/s with 2 warps, 5.7 with 4)
    const bool short_runs = min_run <= RS_BULK_SHORT_RUN;
    // a caller-imposed CTA cap (rs_plan_opts.max_ctas) is made up for with more warps per CTA:
    // 64 CTAs x 4 warps move 6.0 TB/s of a 1 : 1 layout, 64 x 2 only 3.9
    const bool capped = P.max_ctas > 0 && P.max_ctas * 4 < P.sm_count * 3;
    // shifted variant: rows of >= 1 KiB are stored row by row (cheap), shorter ones window by window (ALU-heavy)
    const bool shift_long = shift && min_run >= 1024;
    BulkShape sh;
    sh.warps = std::max(1, std::min(8, shift ? env_int("RS_SHIFT_WARPS", shift_long ? RS_SHIFT_WARPS_LONG : RS_SHIFT_WARPS)
                                             : env_int("RS_BULK_WARPS", short_runs || capped ? RS_BULK_WARPS_SHORT : RS_BULK_WARPS)));
    sh.stages = std::max(2, std::min(8, shift ? env_int("RS_SHIFT_STAGES", shift_long ? RS_SHIFT_STAGES_LONG : RS_SHIFT_STAGES)
                                              : env_int("RS_BULK_STAGES", RS_BULK_STAGES)));
    sh.tile_bytes = shift ? env_int("RS_SHIFT_TILE_BYTES", RS_SHIFT_TILE_BYTES)
                          : env_int("RS_BULK_TILE_BYTES", short_runs ? RS_BULK_TILE_BYTES_SHORT : RS_BULK_TILE_BYTES);
    sh.tile_bytes = std::max<int64_t>(128, sh.tile_bytes / 128 * 128);
    while ((int64_t)sh.warps * (sh.stages * sh.tile_bytes + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX && sh.tile_bytes > 1024) sh.tile_bytes -= 1024;
    // At most one CTA per SM -- and FEWER where the memory system prefers it (148 SMs):
    //  * write-heavy operations (a slice with k >= 2 receivers: 1 read + k writes): 148 writers hold 5.65 TB/s
    //    whatever the ring depth or tile size, 96 writers reach 6.1-6.2 TB/s (an SM sustains ~64 GB/s of this
    //    mix; beyond ~104 SMs the writers contend);
    //  * 1 : 1 operations with long runs (<= 3 bulk copies per tile): 132 CTAs are 1.5-3.7 % faster than 148;
    //  * short runs are issue-bound per SM: write-heavy ones do best from 136 CTAs (Table 2 case 9: 5.7 -> 6.2 TB/s),
    //    1 : 1 ones and the shifted variant from every SM;
    //  * operations under 256 MiB are latency-bound, not contention-bound: every SM.
    // Fractions of the SM count, so the rule survives a different part.
    const bool write_heavy = write_bytes >= 2 * read_bytes, big = read_bytes + write_bytes >= RS_BULK_CTAS_MIN_BYTES;
    int ctas = P.sm_count;
    if (big && !shift) {
        if (write_heavy) ctas = P.sm_count * (short_runs ? RS_BULK_CTAS_MCAST_SHORT_NUM : RS_BULK_CTAS_MCAST_NUM) / RS_BULK_CTAS_DEN;
        else if (min_run >= RS_BULK_LONG_RUN) ctas = P.sm_count * RS_BULK_CTAS_LONG_NUM / RS_BULK_CTAS_DEN;
    }
    sh.grid = std::max(1, std::min(P.sm_count, env_int(write_heavy ? "RS_BULK_CTAS_MCAST" : "RS_BULK_CTAS", std::max(1, ctas))));
    if (P.max_ctas > 0) sh.grid = std::min(sh.grid, P.max_ctas);
    return sh;
}

// Alignment class, path, tile size, grid of one operation; then its tile table.
rs_status finish_op(Plan *P, OpTables *op, int64_t read_bytes, int64_t write_bytes,
                    std::vector<uint32_t> *task_tile_begin = nullptr, bool dst_order = false) {
    int64_t align = 16, min_run = INT64_MAX, max_rows = 0;
    for (const RsTask &T : op->tasks) {
        align = std::min(align, pow2_align(T.run_bytes));
        align = std::min(align, pow2_align(T.src_off));
        for (int i = 0; i < T.nd; i++) {
            align = std::min(align, pow2_align(T.sstride[i]));
            align = std::min(align, pow2_align(T.dstride[i]));
        }
        for (int j = 0; j < T.k; j++) align = std::min(align, pow2_align(op->dsts[(size_t)T.dst_first + j].off));
        min_run = std::min(min_run, T.run_bytes);
        max_rows = std::max(max_rows, task_rows(T));
        if (task_rows(T) > 0x7FFFFFFFll) { set_error("more than 2^31-1 rows in one slice"); return RS_EUNSUPPORTED; }
    }
    rs_op_info &I = op->info;
    I.vec_bytes = (int32_t)align;
    I.n_tasks = (int32_t)op->tasks.size();
    I.n_dsts = (int32_t)op->dsts.size();
    I.read_bytes = read_bytes;
    I.write_bytes = write_bytes;

    const int path = pick_path(P->flags & RS_PATH_MASK, align, min_run, read_bytes + write_bytes);
    I.path = path;
    const bool bulk_family = path == RS_PATH_BULK || path == RS_PATH_BULK_SHIFT;

    int64_t tile_bytes;
    int workers;                                               // independent tile consumers in one launch
    int stages = 0;
    if (bulk_family) {
        const BulkShape sh = bulk_shape(*P, path == RS_PATH_BULK_SHIFT, min_run, read_bytes, write_bytes);
        tile_bytes = sh.tile_bytes;
        stages = sh.stages;
        I.block = sh.warps * 32;
        I.grid = sh.grid;
        workers = sh.grid * sh.warps;
    } else {
        tile_bytes = env_int("RS_LSU_TILE_BYTES", RS_LSU_TILE_BYTES);
        tile_bytes = std::max<int64_t>(128, tile_bytes / 128 * 128);
        I.block = RS_LSU_THREADS;
        I.grid = P->sm_count * std::max(1, std::min(RS_LSU_CTAS_PER_SM, env_int("RS_LSU_CTAS_PER_SM", RS_LSU_CTAS_DEFAULT)));
        if (P->max_ctas > 0) I.grid = std::min(I.grid, P->max_ctas);
        workers = I.grid * (RS_LSU_THREADS / 32);
    }
    // small problems: shrink tiles until every worker has a few (tail balance), floor 2 KiB
    while (tile_bytes > 2048 && read_bytes / tile_bytes < (int64_t)workers * 4) tile_bytes = tile_bytes / 2 / 128 * 128;
    tile_bytes = std::max<int64_t>(tile_bytes, 128);
    I.tile_bytes = (int32_t)tile_bytes;

    op->tiles.clear();
    for (size_t t = 0; t < op->tasks.size(); t++) {
        if (task_tile_begin) task_tile_begin->push_back((uint32_t)op->tiles.size());
        emit_tiles(op->tasks[t], (uint32_t)t, tile_bytes, &op->tiles);
    }
    if (task_tile_begin) task_tile_begin->push_back((uint32_t)op->tiles.size());
    // Tasks whose destination boxes interleave finely (a slice fills part of every destination row, another
    // slice the rest: config 2, sweep pairs P1 / P2 / P4) are walked in DESTINATION address order, so that the
    // pieces of one row are written close in time: +1-3 % on those layouts (P2 at 4 GiB 6.00 -> 6.18 TB/s).
    // Only for execute and unpack (they write shards); not for the slab table (its tile ranges are per task) and not for coarse
    // interleaves (config 4: 3 MiB runs).
    bool interleaved = false;
    for (const RsTask &T : op->tasks) interleaved = interleaved || (T.nd >= 1 && T.run_bytes <= RS_INTERLEAVE_MAX_RUN && T.dstride[0] > T.run_bytes);
    if (dst_order && env_int("RS_TILE_ORDER", 1) && !task_tile_begin && interleaved && op->tasks.size() > 1) {
        struct Key { int64_t buf, off; uint32_t idx; };
        std::vector<Key> keys(op->tiles.size());
        for (size_t i = 0; i < op->tiles.size(); i++) {
            const RsTile &t = op->tiles[i];
            const RsTask &T = op->tasks[t.task];
            int64_t doff = 0;
            if (t.flags & RS_TILE_FAST) doff = (int64_t)t.b;
            else {
                int64_t row = (int64_t)t.a;
                for (int d = 0; d < T.nd; d++) { int64_t c = row % T.ext[d]; row /= T.ext[d]; doff += c * T.dstride[d]; }
            }
            const RsDst &D = op->dsts[(size_t)T.dst_first];
            keys[i] = Key{D.buf, D.off + doff, (uint32_t)i};
        }
        std::stable_sort(keys.begin(), keys.end(), [](const Key &x, const Key &y) { return x.buf != y.buf ? x.buf < y.buf : x.off < y.off; });
        std::vector<RsTile> sorted(op->tiles.size());
        for (size_t i = 0; i < keys.size(); i++) sorted[i] = op->tiles[keys[i].idx];
        op->tiles.swap(sorted);
    }
    if (op->tiles.size() > 0x7FFFFFFFull) { set_error("tile table too large"); return RS_EUNSUPPORTED; }
    I.n_tiles = (int32_t)op->tiles.size();
    int64_t mr = INT64_MAX;
    for (const RsTile &t : op->tiles) mr = std::min<int64_t>(mr, t.col_bytes);
    I.min_run_bytes = op->tiles.empty() ? 0 : mr;
    op->shift_stage = 0;
    op->alt_stage = 0;
    bool lsu = !bulk_family;
    if (bulk_family) {
        const bool shift = path == RS_PATH_BULK_SHIFT;
        int warps = I.block / 32;
        int64_t stage = tile_bytes;
        if (shift) {                                           // a row of n bytes occupies (n + 77) & ~15 bytes of a ring slot
            stage = 0;
            for (const RsTile &t : op->tiles) stage = std::max<int64_t>(stage, (int64_t)t.n_rows * (((int64_t)t.col_bytes + 77) & ~15ll));
            while (stages > 2 && (int64_t)warps * (stages * stage + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX) stages--;
            while (warps > 1 && (int64_t)warps * (stages * stage + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX) warps--;
            I.block = warps * 32;
        }
        op->stages = stages;
        op->lookahead = std::max(1, std::min(stages - 1, shift ? env_int("RS_SHIFT_LOOKAHEAD", stages - 1) : env_int("RS_BULK_LOOKAHEAD", RS_BULK_LOOKAHEAD)));
        I.grid = (int32_t)std::max<int64_t>(1, std::min<int64_t>(I.grid, (I.n_tiles + warps - 1) / warps));
        I.smem_bytes = (int32_t)(warps * (stages * stage + RS_BULK_DESC_BYTES) + 1024);
        if (shift) op->shift_stage = (uint32_t)stage;
        if (!shift) {
            // An aligned plan may be handed under-aligned pointers at execute time: keep a launch shape of the
            // shifted TMA kernel for the SAME tile table (rows padded in the ring, so fewer warps or slots fit).
            int64_t pad = 0;
            for (const RsTile &t : op->tiles) pad = std::max<int64_t>(pad, (int64_t)t.n_rows * (((int64_t)t.col_bytes + 77) & ~15ll));
            const bool long_rows = min_run >= 1024;
            int aw = long_rows ? RS_SHIFT_WARPS_LONG : RS_SHIFT_WARPS, as = long_rows ? RS_SHIFT_STAGES_LONG : RS_SHIFT_STAGES;
            while (as > 2 && (int64_t)aw * (as * pad + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX) as--;
            while (aw > 1 && (int64_t)aw * (as * pad + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX) aw--;
            if ((int64_t)aw * (as * pad + RS_BULK_DESC_BYTES) + 1024 <= RS_SMEM_MAX && !op->tiles.empty()) {
                op->alt_stage = (uint32_t)pad; op->alt_warps = aw; op->alt_stages = as;
                op->alt_smem = (int)(aw * (as * pad + RS_BULK_DESC_BYTES) + 1024);
            }
        }
        if (shift && I.smem_bytes > RS_SMEM_MAX) {             // rows too sparse for the ring: the register kernels take it
            I.path = RS_PATH_LSU;
            I.block = RS_LSU_THREADS;
            I.grid = P->sm_count * RS_LSU_CTAS_DEFAULT;
            if (P->max_ctas > 0) I.grid = std::min(I.grid, P->max_ctas);
            op->shift_stage = 0;
            lsu = true;
        }
    }
    if (lsu) {
        const int warps = RS_LSU_THREADS / 32;
        I.grid = (int32_t)std::max<int64_t>(1, std::min<int64_t>(I.grid, (I.n_tiles + warps - 1) / warps));
        I.smem_bytes = 0;
    }
    return RS_OK;
}

// reshard_execute_host pipeline: cut tensor dim 0 into slabs.  Dim 0 is the outermost dim of every
// local layout, so a slab is ONE contiguous byte range in each source shard and each destination
// shard it touches: slab c can be uploaded, resharded and downloaded while slab c+1 is uploading.
// This is the paper's chunked pipelining (K chunks) applied to the host link.
rs_status build_slabs(Plan *P, const int64_t *sA, const int64_t *sB, int64_t tensor_bytes) {
    const Layout &A = P->A, &B = P->B;
    const int N = A.ndim;
    const int64_t e = P->elem_bytes, l0 = A.shape[0];
    OpTables &H = P->op[RS_OP_SLABS];
    H.tasks.clear(); H.dsts.clear(); H.tiles.clear();
    P->slabs.clear();
    int64_t C = std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(l0, RS_HOST_SLABS_MAX),
                                                       tensor_bytes / RS_HOST_SLAB_MIN_BYTES));
    std::vector<int64_t> bound((size_t)C + 1);
    for (int64_t c = 0; c <= C; c++) bound[(size_t)c] = c * l0 / C;
    std::vector<uint32_t> task_slab;
    for (int64_t c = 0; c < C; c++) {
        const int64_t b0 = bound[(size_t)c], b1 = bound[(size_t)c + 1];
        HostSlab S;
        std::vector<char> up_used((size_t)A.n_dev, 0);
        for (int i : P->exec_order) {
            const Slice &sl = P->slices[(size_t)i];
            int64_t lo[RS_MAX_NDIM], hi[RS_MAX_NDIM];
            for (int d = 0; d < N; d++) { lo[d] = sl.lo[d]; hi[d] = sl.hi[d]; }
            lo[0] = std::max(lo[0], b0); hi[0] = std::min(hi[0], b1);
            if (lo[0] >= hi[0]) continue;
            int64_t lo_s[RS_MAX_NDIM], hi_s[RS_MAX_NDIM];
            device_box(A, sl.sender, lo_s, hi_s);
            BoxDesc bx;
            bx.ndim = N;
            for (int d = 0; d < N; d++) { bx.ext[d] = hi[d] - lo[d]; bx.sstride[d] = sA[d]; bx.dstride[d] = sB[d]; }
            RsTask T{};
            if (!collapse(bx, e, &T)) { set_error("slice extent exceeds 32 bits"); return RS_EUNSUPPORTED; }
            T.src_buf = sl.sender; T.src_off = box_offset(lo, lo_s, sA, N);
            T.k = (int32_t)sl.receivers.size(); T.dst_first = (int32_t)H.dsts.size();
            for (int r : sl.receivers) {
                int64_t lo_r[RS_MAX_NDIM], hi_r[RS_MAX_NDIM];
                device_box(B, r, lo_r, hi_r);
                H.dsts.push_back(RsDst{box_offset(lo, lo_r, sB, N), r, 0});
            }
            H.tasks.push_back(T);
            task_slab.push_back((uint32_t)c);
            up_used[(size_t)sl.sender] = 1;
        }
        for (int r = 0; r < A.n_dev; r++) {                   // byte range of the slab inside every shard read
            if (!up_used[(size_t)r]) continue;
            int64_t lo_s[RS_MAX_NDIM], hi_s[RS_MAX_NDIM];
            device_box(A, r, lo_s, hi_s);
            int64_t a = std::max(b0, lo_s[0]), b = std::min(b1, hi_s[0]);
            if (a < b) S.up.push_back(HostCopy{r, (a - lo_s[0]) * sA[0], (b - a) * sA[0]});
        }
        for (int q = 0; q < B.n_dev; q++) {
            int64_t lo_r[RS_MAX_NDIM], hi_r[RS_MAX_NDIM];
            device_box(B, q, lo_r, hi_r);
            bool empty = false;                               // R5: a device past the end of some dim holds nothing
            for (int d = 1; d < N; d++) empty = empty || lo_r[d] >= hi_r[d];
            int64_t a = std::max(b0, lo_r[0]), b = std::min(b1, hi_r[0]);
            if (a < b && !empty) S.down.push_back(HostCopy{q, (a - lo_r[0]) * sB[0], (b - a) * sB[0]});
        }
        P->slabs.push_back(std::move(S));
    }
    std::vector<uint32_t> ttb;
    rs_status st = finish_op(P, &H, tensor_bytes, tensor_bytes * P->r_B, &ttb);
    if (st != RS_OK) return st;
    for (HostSlab &S : P->slabs) { S.tile_begin = 0xFFFFFFFFu; S.tile_end = 0; }
    for (size_t t = 0; t < task_slab.size(); t++) {
        HostSlab &S = P->slabs[task_slab[t]];
        S.tile_begin = std::min(S.tile_begin, ttb[t]);
        S.tile_end = std::max(S.tile_end, ttb[t + 1]);
    }
    return RS_OK;
}

}  // namespace

// A GROUP: the execute tables of several plans merged into one, so that all the cross-mesh resharding
// tasks of a stage boundary ("many cross-mesh resharding tasks for each tensor exchanged at the
// boundary of two pipeline stages") run in ONE launch.  Buffer ids are shifted so that the group's pointer
// arrays are the concatenation of the members' arrays.
rs_status build_group(Plan *G, const std::vector<const Plan *> &members) {
    OpTables &X = G->op[RS_OP_EXECUTE];
    for (OpTables &o : G->op) { o.tasks.clear(); o.dsts.clear(); o.tiles.clear(); o.info = rs_op_info{}; }
    int n_src = 0, n_dst = 0;
    int64_t rd = 0, wr = 0;
    G->used_src.clear();
    for (const Plan *M : members) {
        const OpTables &mx = M->op[RS_OP_EXECUTE];
        if (n_src + M->A.n_dev > RS_MAX_DEVICES || n_dst + M->B.n_dev > RS_MAX_DEVICES) { set_error("a group holds at most RS_MAX_DEVICES source and RS_MAX_DEVICES destination shards"); return RS_EUNSUPPORTED; }
        const int32_t d0 = (int32_t)X.dsts.size();
        for (RsTask T : mx.tasks) { T.src_buf += n_src; T.dst_first += d0; X.tasks.push_back(T); }
        for (RsDst D : mx.dsts) { D.buf += n_dst; X.dsts.push_back(D); }
        G->used_src.insert(G->used_src.end(), M->used_src.begin(), M->used_src.end());
        n_src += M->A.n_dev; n_dst += M->B.n_dev;
        rd += mx.info.read_bytes; wr += mx.info.write_bytes;
    }
    G->A.n_dev = n_src; G->B.n_dev = n_dst;
    G->group_src = n_src; G->group_dst = n_dst;
    return finish_op(G, &X, rd, wr, nullptr, true);
}

rs_status build_tables(Plan *P) {
    const Layout &A = P->A, &B = P->B;
    const int N = A.ndim;
    const int64_t e = P->elem_bytes;
    int64_t sA[RS_MAX_NDIM], sB[RS_MAX_NDIM];
    dense_strides(A.local, N, e, sA);
    dense_strides(B.local, N, e, sB);
    const int64_t tensor_bytes = [&] { int64_t n = e; for (int d = 0; d < N; d++) n *= A.shape[d]; return n; }();

    // which (message, position) holds slice i for receiver r
    std::vector<std::vector<int64_t>> arena_off(P->slices.size());
    for (size_t i = 0; i < P->slices.size(); i++) arena_off[i].assign(P->slices[i].receivers.size(), -1);
    for (const Message &M : P->messages)
        for (size_t j = 0; j < M.slice_ids.size(); j++) {
            const Slice &S = P->slices[(size_t)M.slice_ids[j]];
            size_t pos = (size_t)(std::find(S.receivers.begin(), S.receivers.end(), M.receiver) - S.receivers.begin());
            arena_off[(size_t)M.slice_ids[j]][pos] = M.slice_off[j];
        }

    OpTables &X = P->op[RS_OP_EXECUTE], &PK = P->op[RS_OP_PACK], &UP = P->op[RS_OP_UNPACK];
    for (OpTables *o : {&X, &PK, &UP}) { o->tasks.clear(); o->dsts.clear(); o->tiles.clear(); }

    for (int i : P->exec_order) {                              // slice-id order, or the schedule's (S3.2)
        const Slice &S = P->slices[(size_t)i];
        int64_t lo_s[RS_MAX_NDIM], hi_s[RS_MAX_NDIM], ext[RS_MAX_NDIM], dense[RS_MAX_NDIM];
        device_box(A, S.sender, lo_s, hi_s);
        for (int d = 0; d < N; d++) ext[d] = S.hi[d] - S.lo[d];
        dense_strides(ext, N, e, dense);
        const int64_t src_off = box_offset(S.lo, lo_s, sA, N);
        BoxDesc bx;
        bx.ndim = N;
        for (int d = 0; d < N; d++) { bx.ext[d] = ext[d]; bx.sstride[d] = sA[d]; }

        // execute: sender shard -> every receiver shard (read once, write k times)
        {
            RsTask T{};
            for (int d = 0; d < N; d++) bx.dstride[d] = sB[d];
            if (!collapse(bx, e, &T)) { set_error("slice extent exceeds 32 bits"); return RS_EUNSUPPORTED; }
            T.src_buf = S.sender; T.src_off = src_off;
            T.k = (int32_t)S.receivers.size(); T.dst_first = (int32_t)X.dsts.size();
            for (int r : S.receivers) {
                int64_t lo_r[RS_MAX_NDIM], hi_r[RS_MAX_NDIM];
                device_box(B, r, lo_r, hi_r);
                X.dsts.push_back(RsDst{box_offset(S.lo, lo_r, sB, N), r, 0});
            }
            X.tasks.push_back(T);
        }
        // pack: sender shard -> k dense copies in the arena
        {
            RsTask T{};
            for (int d = 0; d < N; d++) bx.dstride[d] = dense[d];
            if (!collapse(bx, e, &T)) { set_error("slice extent exceeds 32 bits"); return RS_EUNSUPPORTED; }
            T.src_buf = S.sender; T.src_off = src_off;
            T.k = (int32_t)S.receivers.size(); T.dst_first = (int32_t)PK.dsts.size();
            for (size_t j = 0; j < S.receivers.size(); j++) PK.dsts.push_back(RsDst{arena_off[(size_t)i][j], 0, 0});
            PK.tasks.push_back(T);
        }
        // unpack: one dense copy in the arena -> one receiver shard
        for (size_t j = 0; j < S.receivers.size(); j++) {
            RsTask T{};
            BoxDesc ux;
            ux.ndim = N;
            for (int d = 0; d < N; d++) { ux.ext[d] = ext[d]; ux.sstride[d] = dense[d]; ux.dstride[d] = sB[d]; }
            if (!collapse(ux, e, &T)) { set_error("slice extent exceeds 32 bits"); return RS_EUNSUPPORTED; }
            T.src_buf = 0; T.src_off = arena_off[(size_t)i][j];
            T.k = 1; T.dst_first = (int32_t)UP.dsts.size();
            int64_t lo_r[RS_MAX_NDIM], hi_r[RS_MAX_NDIM];
            device_box(B, S.receivers[j], lo_r, hi_r);
            UP.dsts.push_back(RsDst{box_offset(S.lo, lo_r, sB, N), S.receivers[j], 0});
            UP.tasks.push_back(T);
        }
    }
    // Alternative strategies for a unit task, as extra tables on request.  On chip
    // they differ from the broadcast table in BYTES: send/recv re-reads the slice once per receiver
    // (k reads + k writes instead of 1 + k); the all-gather strategy sends part j of the slice to
    // receiver j (1 read + 1 write in total), then every receiver copies the other k - 1 parts from
    // its peers' shards (k - 1 reads + k - 1 writes): again 2k, in two dependent launches.
    OpTables &SR = P->op[RS_OP_SENDRECV], &AS = P->op[RS_OP_AG_SCATTER], &AG = P->op[RS_OP_AG_GATHER];
    OpTables &LS = P->op[RS_OP_AGL_SCATTER], &LG = P->op[RS_OP_AGL_GATHER];
    for (OpTables *o : {&SR, &AS, &AG, &LS, &LG}) { o->tasks.clear(); o->dsts.clear(); o->tiles.clear(); o->info = rs_op_info{}; }
    if (P->flags & RS_WITH_STRATEGIES) {
        auto add = [&](OpTables &O, const int64_t *lo, const int64_t *hi, int src_buf, const int64_t *src_origin,
                       const int64_t *sstr, int dst_buf, const int64_t *dst_origin) -> bool {
            BoxDesc bx;
            bx.ndim = N;
            for (int d = 0; d < N; d++) { bx.ext[d] = hi[d] - lo[d]; bx.sstride[d] = sstr[d]; bx.dstride[d] = sB[d]; }
            RsTask T{};
            if (!collapse(bx, e, &T)) return false;
            T.src_buf = src_buf; T.src_off = box_offset(lo, src_origin, sstr, N);
            T.k = 1; T.dst_first = (int32_t)O.dsts.size();
            O.dsts.push_back(RsDst{box_offset(lo, dst_origin, sB, N), dst_buf, 0});
            O.tasks.push_back(T);
            return true;
        };
        for (int i : P->exec_order) {
            const Slice &S = P->slices[(size_t)i];
            const int k = (int)S.receivers.size();
            int64_t lo_s[RS_MAX_NDIM], hi_s[RS_MAX_NDIM];
            device_box(A, S.sender, lo_s, hi_s);
            std::vector<std::vector<int64_t>> org((size_t)k, std::vector<int64_t>(RS_MAX_NDIM));
            for (int j = 0; j < k; j++) { int64_t hi_r[RS_MAX_NDIM]; device_box(B, S.receivers[(size_t)j], org[(size_t)j].data(), hi_r); }
            for (int j = 0; j < k; j++)                           // send/recv: the whole slice, once per receiver
                if (!add(SR, S.lo, S.hi, S.sender, lo_s, sA, S.receivers[(size_t)j], org[(size_t)j].data())) { set_error("slice extent exceeds 32 bits"); return RS_EUNSUPPORTED; }
            // all-gather over a group G of receivers: part j of the slice goes to G[j], then everybody in G copies
            // the other parts from its peers.  Global: one group = all k receivers.  Local
            // (PAPER.md:131): one group per receiver HOST, so the slice leaves the sender once per host.
            auto allgather = [&](const std::vector<int> &G, OpTables &scatter, OpTables &gather) -> bool {
                const int g = (int)G.size();
                int cd = 0;                                    // cut the outermost dim that has >= g rows (else the longest)
                for (int d = 0; d < N; d++) if (S.hi[d] - S.lo[d] > S.hi[cd] - S.lo[cd]) cd = d;
                for (int d = N - 1; d >= 0; d--) if (S.hi[d] - S.lo[d] >= g) cd = d;
                const int64_t ext = S.hi[cd] - S.lo[cd], step = (ext + g - 1) / g;
                for (int j = 0; j < g; j++) {
                    int64_t lo[RS_MAX_NDIM], hi[RS_MAX_NDIM];
                    for (int d = 0; d < N; d++) { lo[d] = S.lo[d]; hi[d] = S.hi[d]; }
                    lo[cd] = std::min(S.lo[cd] + j * step, S.hi[cd]);
                    hi[cd] = std::min(S.lo[cd] + (j + 1) * step, S.hi[cd]);
                    if (lo[cd] >= hi[cd]) continue;
                    const int rj = G[(size_t)j];
                    if (!add(scatter, lo, hi, S.sender, lo_s, sA, S.receivers[(size_t)rj], org[(size_t)rj].data())) return false;
                    for (int q : G)                            // gather: part j from G[j]'s shard into every other member's
                        if (q != rj && !add(gather, lo, hi, S.receivers[(size_t)rj], org[(size_t)rj].data(), sB, S.receivers[(size_t)q], org[(size_t)q].data())) return false;
                }
                return true;
            };
            std::vector<int> all((size_t)k);
            for (int j = 0; j < k; j++) all[(size_t)j] = j;
            bool ok = allgather(all, AS, AG);
            for (int j = 0; j < k && ok;) {                    // receivers are ascending, so a host's receivers are adjacent
                std::vector<int> G;
                const int host = S.receivers[(size_t)j] / P->sched.dst_dph;
                while (j < k && S.receivers[(size_t)j] / P->sched.dst_dph == host) G.push_back(j++);
                ok = allgather(G, LS, LG);
            }
            if (!ok) { set_error("slice extent exceeds 32 bits"); return RS_EUNSUPPORTED; }
        }
    }
    rs_status st;
    if (P->flags & RS_WITH_STRATEGIES) {
        if ((st = finish_op(P, &SR, tensor_bytes * P->r_B, tensor_bytes * P->r_B)) != RS_OK) return st;
        if ((st = finish_op(P, &AS, tensor_bytes, tensor_bytes)) != RS_OK) return st;
        if ((st = finish_op(P, &AG, tensor_bytes * (P->r_B - 1), tensor_bytes * (P->r_B - 1))) != RS_OK) return st;
        int64_t ls = 0, lg = 0;                                // local variant: bytes depend on how receivers fall on hosts
        for (const RsTask &T : LS.tasks) ls += T.run_bytes * task_rows(T);
        for (const RsTask &T : LG.tasks) lg += T.run_bytes * task_rows(T);
        if ((st = finish_op(P, &LS, ls, ls)) != RS_OK) return st;
        if ((st = finish_op(P, &LG, lg, lg)) != RS_OK) return st;
    }
    if ((st = build_slabs(P, sA, sB, tensor_bytes)) != RS_OK) return st;
    if ((st = finish_op(P, &X, tensor_bytes, tensor_bytes * P->r_B, nullptr, true)) != RS_OK) return st;
    if ((st = finish_op(P, &PK, tensor_bytes, tensor_bytes * P->r_B)) != RS_OK) return st;
    if ((st = finish_op(P, &UP, tensor_bytes * P->r_B, tensor_bytes * P->r_B, nullptr, true)) != RS_OK) return st;
    return RS_OK;
}

}  // namespace rs

// tables.cpp -- step a5: unit tasks -> collapsed copy tasks -> flat task tables for the three
// operations (execute / pack / unpack), the shape of every task's tile grid (tiles themselves are
// never stored: tables.h), plus the per-operation launch configuration.  O(unit tasks) work and
// memory, whatever the tensor size (the plan is the slice list).
// Paper analogue: "choose the better result as the schedule to launch broadcasts";
// north_star item (1): "emits a flat task table".  No CUDA here, no environment variables: launch
// shapes are overridden only through rs_plan_opts.tuning.
#include <algorithm>
#include <cstring>
#include <map>

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

int pick(int override_value, int dflt) { return override_value > 0 ? override_value : dflt; }

// Shape of one task's tile grid (tables.h): nothing per tile is stored, the kernels decode tile u from
// these few numbers.  tile_bytes is a multiple of 128.
void set_tiling(RsTask *T, int64_t tile_bytes) {
    const int64_t R = task_rows(*T), B = T->run_bytes;
    T->n_rows = (uint32_t)R;
    T->tmap_ok = 0;
    T->chunk_bytes = (uint32_t)std::min<int64_t>(B, 0xFFFFFF80ll);
    T->n_chunks = 1; T->rows_per_tile = 1; T->tiles_per_span = 1;
    if (B > tile_bytes) {                                     // long runs: split every row into column chunks
        const int64_t n = (B + tile_bytes - 1) / tile_bytes;
        const int64_t chunk = ((B + n - 1) / n + 127) / 128 * 128;
        T->kind = RS_TILING_SPLIT;
        T->chunk_bytes = (uint32_t)chunk;
        T->n_chunks = (uint32_t)((B + chunk - 1) / chunk);
        T->n_tiles = (uint32_t)std::min<int64_t>(R * T->n_chunks, 0xFFFFFFFFll);
        return;
    }
    const int64_t rpt = std::max<int64_t>(1, tile_bytes / B);  // rows per tile
    const int64_t ext0 = T->nd > 0 ? T->ext[0] : 1;
    // (a span shorter than a tile still makes FAST tiles -- one per span -- when it holds >= RS_SPAN_TILE_MIN_BYTES: GENERIC tiles
    // pay a division per row or vector, which cost a feature map resharded from H to W, 64-byte rows in spans of 32, 2/3 of its rate)
    if (T->nd <= 1 || ext0 >= rpt || ext0 * B >= RS_SPAN_TILE_MIN_BYTES) {   // FAST tiles inside one span of row dim 0
        const int64_t n = (ext0 + rpt - 1) / rpt, sz = (ext0 + n - 1) / n;
        T->kind = RS_TILING_FAST;
        T->rows_per_tile = (uint32_t)sz;
        T->tiles_per_span = (uint32_t)((ext0 + sz - 1) / sz);
        T->n_tiles = (uint32_t)std::min<int64_t>(R / ext0 * T->tiles_per_span, 0xFFFFFFFFll);
        return;
    }
    const int64_t n = (R + rpt - 1) / rpt, sz = (R + n - 1) / n;   // GENERIC tiles: any run of linear rows
    T->kind = RS_TILING_GENERIC;
    T->rows_per_tile = (uint32_t)sz;
    T->n_tiles = (uint32_t)((R + sz - 1) / sz);
}

int64_t task_tiles_exact(const RsTask &T) {                   // n_tiles before the 32-bit clamp
    const int64_t R = task_rows(T);
    if (T.kind == RS_TILING_SPLIT) return R * T.n_chunks;
    if (T.kind == RS_TILING_FAST) return R / std::max<int64_t>(1, T.nd > 0 ? T.ext[0] : 1) * T.tiles_per_span;
    return (R + T.rows_per_tile - 1) / T.rows_per_tile;
}

int64_t task_min_col(const RsTask &T) {                       // shortest contiguous run any of its tiles copies
    if (T.kind != RS_TILING_SPLIT) return T.run_bytes;
    return std::min<int64_t>(T.chunk_bytes, T.run_bytes - (int64_t)(T.n_chunks - 1) * T.chunk_bytes);
}

int64_t task_shift_stage(const RsTask &T) {                   // ring-slot bytes its largest tile needs in rs_copy_bulk_shift
    const int64_t col = T.kind == RS_TILING_SPLIT ? T.chunk_bytes : T.run_bytes;
    const int64_t rows = T.kind == RS_TILING_SPLIT ? 1 : std::min<int64_t>(T.rows_per_tile, T.n_rows);
    return rows * ((col + 77) & ~15ll);                       // a row of n bytes occupies (n + 77) & ~15 bytes of a slot
}

// Which kernel an operation takes (rs_op_info.path).  AUTO: runs under 512 B and small aligned operations go to the
// register kernels (they start faster; small operations are launch-bound), 16-byte aligned layouts to the TMA
// kernel, everything else to TMA loads + shifted stores.
int pick_path(const Plan &P, int64_t align, int64_t min_run, int64_t max_run, int64_t moved_bytes, bool write_heavy, bool tmap_short, int n_src, int n_dst) {
    const uint32_t forced = P.flags & RS_PATH_MASK;
    // (write-heavy operations leave the register path earlier: k stores per load keep a thread busy, the ring's stores are
    // fire and forget -- 4 + 16 MiB: 6.4 us in registers, 4.8 us on the ring; 1 + 8 MiB: 3.1 against 4.5 us)
    const int64_t small_op = P.tune.small_op_bytes_mib < 0 ? -1 : P.tune.small_op_bytes_mib > 0 ? ((int64_t)P.tune.small_op_bytes_mib << 20)
                           : write_heavy ? RS_SMALL_OP_BYTES_MCAST : RS_SMALL_OP_BYTES;
    const bool bulk_ok = align == 16 && min_run >= 16;
    // Rows shorter than 512 bytes: a tensor-map copy moves a box of up to 256 of them with one instruction, whatever their length,
    // so a large operation made of short rows takes rs_copy_tmap (128-byte rows at 1 + 1 GiB: 6.15 TB/s against 5.53 in registers;
    // 1 + 4 GiB: 6.09 against 4.64) -- if (nearly) all of its tiles fit the tensor maps (finish_op checks and falls back).
    const bool short_tmap = tmap_short && bulk_ok && min_run >= RS_TMAP_SHORT_MIN_RUN && moved_bytes > small_op && !P.group_src &&
                            n_src <= RS_TMAP_BUFS && n_dst <= RS_TMAP_BUFS;
    int path = forced == RS_PATH_LSU ? RS_PATH_LSU : forced == RS_PATH_BULK ? RS_PATH_BULK
             : forced == RS_PATH_TMAP ? (bulk_ok ? RS_PATH_TMAP : RS_PATH_BULK_SHIFT)
             : forced == RS_PATH_BULK_SHIFT ? RS_PATH_BULK_SHIFT
             // (rows of 128-511 bytes that are NOT 16-byte aligned: TMA loads + shifted register stores beat the register shift
             //  kernel once the operation is large -- 130-byte rows 1.57 -> 2.05 TB/s, 257-byte rows 1.94 -> 2.92; 63-byte rows: a tie)
             : min_run < RS_BULK_MIN_RUN ? (short_tmap ? RS_PATH_TMAP : !bulk_ok && min_run >= RS_SHIFT_MIN_RUN && moved_bytes > small_op ? RS_PATH_BULK_SHIFT : RS_PATH_LSU)
             : bulk_ok ? (moved_bytes <= small_op ? RS_PATH_LSU : RS_PATH_BULK)
             : RS_PATH_BULK_SHIFT;
    // Mid-size operations made of short rows (config 2: 2 KiB destination runs, 128 + 128 MiB) are the one place
    // where tensor-map copies beat one bulk copy per row: +3-5 % at 64-256 MiB moved; from 512 MiB on they lose 1-2 %,
    // 512-byte rows with 4 warps are a tie (profiles/r02_tmap.md).  Not for groups (buffers of different sizes).
    if (!forced && path == RS_PATH_BULK && max_run <= 256 * RS_TMAP_ELEM && moved_bytes <= RS_TMAP_MAX_BYTES && !P.group_src &&
        n_src <= RS_TMAP_BUFS && n_dst <= RS_TMAP_BUFS)
        path = RS_PATH_TMAP;
    if (path == RS_PATH_BULK && !bulk_ok) path = RS_PATH_BULK_SHIFT;   // cp.async.bulk stores need 16-byte everything
    return path;
}

// Launch shape of the two TMA kernels, from measurement on B200.
struct BulkShape { int warps, stages, grid, pace_permille; int64_t tile_bytes; };

BulkShape bulk_shape(const Plan &P, bool shift, bool tmap, int64_t min_run, int64_t read_bytes, int64_t write_bytes, bool dst_dense, bool underfilled, bool tiny_tiles) {
    const rs_tuning &U = P.tune;
    // short runs = many bulk copies per tile: one warp issues them too slowly, so more, smaller pipelines
    // (Table 2 case 9, 512-byte runs: 3.6 TB/s with 2 warps, 5.7 with 4)
    // ... and so do tiles that would fill little of a 12 KiB slot (a run of 6160 bytes: one row per tile): a warp spends
    // ~220 instructions per tile at ~6 cycles each with nothing to overlap them, so 2 warps x half-empty tiles are
    // issue-bound (a4: 4.55 TB/s; 4 warps x 8 KiB slots: 6.33)
    const bool short_runs = min_run <= RS_BULK_SHORT_RUN || underfilled;
    // a caller-imposed CTA cap (rs_plan_opts.max_ctas) is made up for with more warps per CTA:
    // 64 CTAs x 4 warps move 6.0 TB/s of a 1 : 1 layout, 64 x 2 only 3.9
    const bool capped = P.max_ctas > 0 && P.max_ctas * 4 < P.sm_count * 3;
    // shifted variant: the ring shape by row length (all three classes ended on 8 warps x 2 slots; stores leave from registers unless rs_tuning.shift_mode = 2: api.cu)
    const bool shift_long = shift && min_run >= RS_SHIFT_LONG_RUN, shift_mid = shift && !shift_long && min_run >= RS_SHIFT_MID_RUN;
    // small write-heavy operations (4 MiB to 8 receivers) are over in 5-8 us: many short pipelines ramp up faster
    // ... and so do tiles of 1-4 KiB (a span of the innermost row dim that short: feature maps resharded across H / W): at ~1 340 cycles
    // per tile and warp, 2 KiB tiles need 8 warps per SM (fm_hw: 2.6 TB/s with 4 warps, 4.4 with 8 before source-order segments)
    const bool small_mcast = !shift && !capped && (tiny_tiles || (write_bytes >= 2 * read_bytes && read_bytes + write_bytes <= RS_SMALL_MCAST_BYTES));
    // paced write-heavy operations of medium size ramp faster on 4 warps x 8 KiB (16 + 128 MiB: 26.0 -> 25.3 us, 64 + 512 MiB +1.4 %; from ~1 GiB moved
    // on the two shapes are level)
    const bool mid_mcast = !shift && !capped && write_bytes >= 2 * read_bytes && read_bytes + write_bytes >= RS_PACE_MIN_BYTES && read_bytes + write_bytes <= RS_MID_MCAST_BYTES;
    // One CTA per SM.
    //  * Write-heavy operations (a slice with k >= 2 receivers: 1 read + k writes) are an OPEN loop: stores are fire and
    //    forget, every SM can push ~65 GB/s, 148 of them offer 9.6 TB/s and HBM collapses to 5.2-5.8 TB/s.  They run on
    //    every SM and are RATE MATCHED (kernels.cu pace_tile, config.h RS_PACE_PERMILLE): 6.2-6.3 TB/s.
    //  * 1 : 1 operations moving >= 384 MiB through per-row bulk copies: 4 warps x 12 KiB slots on 132 of 148 SMs, paced at
    //    860 permille (WIDE_11).  The loop of 2 unpaced warps per SM limits itself (bytes in flight / latency) and was the
    //    round's first shape: 6.3-6.5 TB/s on an idle chip, but 4.4-4.8 for rows of 3-6 KiB once the SM clock drops under
    //    power (latency in cycles is what it is; in ns it grows).  Twice the pipelines have the slack, and the pacing then
    //    sets the rate: idle +1 % per 10 permille up to 900 (6.39-6.56 TB/s at 880 on the twelve 1 : 1 layouts measured), the edge
    //    of the collapse at 900 idle, but at 870-880 on a hot chip of the pool's weakest box -- hence 860: 6.3-6.45 TB/s idle
    //    and hot (profiles/r02_pacing.md part 5).  On every SM the edge lies 10-20 permille lower, for every row length.
    const bool write_heavy = write_bytes >= 2 * read_bytes;
    const bool wide_11 = !shift && !tmap && !capped && !write_heavy && !small_mcast && read_bytes + write_bytes >= RS_WIDE_11_MIN_BYTES;
    //  * Smaller 1 : 1 operations keep the ramp of the lighter shapes; those made of runs >= 1 MiB and moving >= 128 MiB are paced on their two warps.
    const bool long_11 = !shift && !write_heavy && !wide_11 && min_run >= RS_PACE_11_MIN_RUN && read_bytes + write_bytes >= RS_PACE_11_MIN_BYTES;
    //  * Rows up to 512 bytes (24+ copies per 12 KiB) in large operations, 1 : 1 or write-heavy: 8 warps x 6 KiB.  At ~2 instructions
    //    per copy and ~6 cycles per instruction with one warp per scheduler, four warps keep up at the boost clock only (512-byte rows,
    //    1 + 1 GiB: 6.26 TB/s idle, 5.17 hot; on 8 warps 6.33 / 6.17; Table 2 case 9: 6.19 / 5.16 -> 6.19 / 5.55).
    const bool many_copies = !shift && !tmap && !capped && !small_mcast && min_run <= RS_BULK_VERY_SHORT_RUN &&
                             (wide_11 || (write_heavy && read_bytes + write_bytes > RS_MID_MCAST_BYTES));
    BulkShape sh;
    sh.warps = std::max(1, std::min(8, shift ? pick(U.shift_warps, shift_long ? RS_SHIFT_WARPS_LONG : shift_mid ? RS_SHIFT_WARPS_MID : RS_SHIFT_WARPS)
                                             : pick(U.bulk_warps, small_mcast || many_copies ? RS_BULK_WARPS_SMALL_MCAST : wide_11 || short_runs || capped || mid_mcast ? RS_BULK_WARPS_SHORT : RS_BULK_WARPS)));
    sh.stages = std::max(2, std::min(8, shift ? pick(U.shift_stages, shift_long ? RS_SHIFT_STAGES_LONG : shift_mid ? RS_SHIFT_STAGES_MID : RS_SHIFT_STAGES)
                                              : pick(U.bulk_stages, small_mcast ? RS_BULK_STAGES_SMALL_MCAST : RS_BULK_STAGES)));
    sh.tile_bytes = shift ? pick(U.shift_tile_bytes, RS_SHIFT_TILE_BYTES)
                          : pick(U.bulk_tile_bytes, small_mcast ? RS_BULK_TILE_BYTES_SMALL_MCAST : many_copies ? RS_BULK_TILE_BYTES_MANY : wide_11 ? RS_BULK_TILE_BYTES : short_runs || mid_mcast ? RS_BULK_TILE_BYTES_SHORT : RS_BULK_TILE_BYTES);
    sh.tile_bytes = std::max<int64_t>(128, sh.tile_bytes / 128 * 128);
    while ((int64_t)sh.warps * (sh.stages * sh.tile_bytes + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX && sh.tile_bytes > 1024) sh.tile_bytes -= 1024;
    int ctas = P.sm_count;
    // (large 1 : 1 operations through tensor maps too: 128-byte rows, 1 + 1 GiB, hot 5.75 TB/s on 148 CTAs, 6.17 on 132; idle 6.2 either way)
    if (wide_11 || (tmap && !capped && !write_heavy && read_bytes + write_bytes >= RS_WIDE_11_MIN_BYTES)) ctas = P.sm_count * RS_BULK_CTAS_LONG_NUM / RS_BULK_CTAS_DEN;
    sh.grid = std::max(1, std::min(P.sm_count, pick(write_heavy ? U.bulk_ctas_mcast : U.bulk_ctas, std::max(1, ctas))));
    if (P.max_ctas > 0) sh.grid = std::min(sh.grid, P.max_ctas);
    // (operations under 64 MiB are over before the pacing has anything to hold back: they keep the unpaced ramp)
    // short rows that are adjacent in every destination are stored with one bulk copy per tile and receiver (kernels.cu) and
    // take a higher rate than rows stored one by one (Table 2 case 9: 6.12 TB/s at 810, 6.26 at 830, 6.35-6.40 at 850 on two
    // boxes but 5.98 on a third, whose edge lies lower: 830)
    // The shifted kernel (unaligned layouts) offers too much as well -- 8 warps per SM, stores fire and forget: u4 5.65 -> 6.1 TB/s at 850 permille (6.31 with bulk stores), u1 5.86 -> 6.24,
    // their pack / unpack +6-15 %; write-heavy: 5.49 -> 6.08 and 4.79 -> 5.91 at 800, collapse from 830 on (profiles/r02_unaligned.md).  Rows >= 2 KiB only (1 KiB rows: issue-bound, 4.58 -> 4.47).
    sh.pace_permille = shift ? (min_run >= RS_PACE_SHIFT_MIN_RUN && read_bytes + write_bytes >= RS_PACE_SHIFT_MIN_BYTES ? (write_heavy ? RS_PACE_PERMILLE_SHIFT_MCAST : RS_PACE_PERMILLE_SHIFT) : 0)
                     : write_heavy && read_bytes + write_bytes >= RS_PACE_MIN_BYTES ? (short_runs ? (dst_dense ? RS_PACE_PERMILLE_SHORT_DENSE : RS_PACE_PERMILLE_SHORT) : RS_PACE_PERMILLE)
                     : wide_11 ? RS_PACE_PERMILLE_WIDE_11 : long_11 ? RS_PACE_PERMILLE_11
                     // 1 : 1 through tensor maps (rows of 64 B - 2 KiB; always the 4-warp shape): 128-byte rows 5.37 -> 6.15-6.33 TB/s at 850-870, collapse at 890
                     : !write_heavy && short_runs && !small_mcast && read_bytes + write_bytes >= RS_PACE_11_MIN_BYTES ? RS_PACE_PERMILLE_11_SHORT : 0;
    return sh;
}

// Slices that share destination rows (one slice fills part of every destination row, another slice the rest:
// config 2, sweep pairs P1 / P2 / P4) become ONE segment whose tiles are walked round-robin, i.e. in DESTINATION
// address order, so that the pieces of one row are written close in time: +1-3 % on those layouts (P2 at 4 GiB
// 6.00 -> 6.18 TB/s).  Members must have identical tile grids and destination buffers, and start in the same
// destination row.  Reorders op->tasks so that the members of a segment are consecutive (ascending destination
// offset); the order of the segments follows their first member.
void group_interleaved(OpTables *op, bool by_dst, bool by_src) {
    const size_t n = op->tasks.size();
    std::map<std::vector<int64_t>, std::vector<uint32_t>> buckets, src_buckets;
    std::vector<std::vector<int64_t>> key_of(n), src_key_of(n);
    auto grid_key = [](const RsTask &T) {
        return std::vector<int64_t>{T.k, T.nd, T.run_bytes, (int64_t)T.kind, T.chunk_bytes, T.n_chunks, T.rows_per_tile, T.tiles_per_span, T.n_tiles};
    };
    for (size_t i = 0; i < n; i++) {
        const RsTask &T = op->tasks[i];
        std::vector<int64_t> key;
        const bool cand = T.nd >= 1 && T.run_bytes <= RS_INTERLEAVE_MAX_RUN;   // (GENERIC tiles too: equal grids cover equal rows)
        if (by_dst && cand && T.dstride[0] > T.run_bytes) {
            const RsDst &D0 = op->dsts[(size_t)T.dst_first];
            key = grid_key(T);
            key.push_back(D0.off / T.dstride[0]);
            for (int d = 0; d < T.nd; d++) { key.push_back(T.ext[d]); key.push_back(T.dstride[d]); }
            for (int j = 0; j < T.k; j++) {                   // the same receivers, at the same distance from the first one
                const RsDst &D = op->dsts[(size_t)T.dst_first + j];
                key.push_back(D.buf); key.push_back(D.off - D0.off);
            }
        } else {
            key = {-1, (int64_t)i};                           // not a candidate: alone
        }
        buckets[key].push_back((uint32_t)i);
        key_of[i] = std::move(key);
        // Slices that share SOURCE rows (each reads part of every row of the sender's shard: a feature map resharded from a
        // split of H to a split of W reads 64 of every 128 bytes) are walked together as well, so that the pieces of a row are
        // read close in time -- only for tasks no destination group has taken.
        std::vector<int64_t> skey = {-2, (int64_t)i};
        if (by_src && cand && T.sstride[0] > T.run_bytes) {
            skey = grid_key(T);
            skey.push_back(-3); skey.push_back(T.src_buf); skey.push_back(T.src_off / T.sstride[0]);
            for (int d = 0; d < T.nd; d++) { skey.push_back(T.ext[d]); skey.push_back(T.sstride[d]); }
        }
        src_key_of[i] = std::move(skey);
    }
    for (size_t i = 0; i < n; i++)                             // tasks left alone by the destination rule: group by source
        if (buckets[key_of[i]].size() == 1) src_buckets[src_key_of[i]].push_back((uint32_t)i);
    for (size_t i = 0; i < n; i++) {
        if (buckets[key_of[i]].size() != 1) continue;
        const std::vector<uint32_t> &sb = src_buckets[src_key_of[i]];
        if (sb.size() > 1) { key_of[i] = src_key_of[i]; }
    }
    for (auto &kv : src_buckets)
        if (kv.second.size() > 1) {
            for (uint32_t m : kv.second) buckets.erase(std::vector<int64_t>{-1, (int64_t)m});
            buckets[kv.first] = kv.second;
        }
    std::vector<RsTask> ordered;
    ordered.reserve(n);
    std::vector<char> done(n, 0);
    op->segs.clear();
    for (size_t i = 0; i < n; i++) {
        if (done[i]) continue;
        std::vector<uint32_t> &members = buckets[key_of[i]];
        const bool src_group = key_of[i].size() > 9 && key_of[i][9] == -3;
        std::stable_sort(members.begin(), members.end(), [&](uint32_t a, uint32_t b) {
            if (src_group) return op->tasks[a].src_off < op->tasks[b].src_off;
            return op->dsts[(size_t)op->tasks[a].dst_first].off < op->dsts[(size_t)op->tasks[b].dst_first].off;
        });
        op->segs.push_back(RsSeg{0, (uint32_t)ordered.size(), (uint32_t)members.size(), op->tasks[i].n_tiles});
        for (uint32_t m : members) { ordered.push_back(op->tasks[m]); done[m] = 1; }
    }
    op->tasks.swap(ordered);
}

// Alignment class, path, tile size, grid of one operation; then the shape of every task's tile grid and the
// segments.  per_task: one segment per task, in task order (the slab table: its tile ranges are per task).
rs_status finish_op_impl(Plan *P, OpTables *op, int64_t read_bytes, int64_t write_bytes, bool per_task, bool dst_order, bool tmap_short, double *tmap_cover) {
    int64_t align = 16, min_run = INT64_MAX, max_run = 0;
    for (const RsTask &T : op->tasks) {
        align = std::min(align, pow2_align(T.run_bytes));
        align = std::min(align, pow2_align(T.src_off));
        for (int i = 0; i < T.nd; i++) {
            align = std::min(align, pow2_align(T.sstride[i]));
            align = std::min(align, pow2_align(T.dstride[i]));
        }
        for (int j = 0; j < T.k; j++) align = std::min(align, pow2_align(op->dsts[(size_t)T.dst_first + j].off));
        min_run = std::min(min_run, T.run_bytes);
        max_run = std::max(max_run, T.run_bytes);
        if (task_rows(T) > 0x7FFFFFFFll) { set_error("more than 2^31-1 rows in one slice"); return RS_EUNSUPPORTED; }
    }
    rs_op_info &I = op->info;
    I.vec_bytes = (int32_t)align;
    I.n_tasks = (int32_t)op->tasks.size();
    I.n_dsts = (int32_t)op->dsts.size();
    I.read_bytes = read_bytes;
    I.write_bytes = write_bytes;
    I.pace_permille = 0;
    op->pace_permille = 0;

    const int path = pick_path(*P, align, min_run, max_run, read_bytes + write_bytes, write_bytes >= 2 * read_bytes, tmap_short, P->A.n_dev, P->B.n_dev);
    I.path = path;
    const bool bulk_family = path == RS_PATH_BULK || path == RS_PATH_BULK_SHIFT || path == RS_PATH_TMAP;

    int64_t tile_bytes;
    int workers;                                               // independent tile consumers in one launch
    int stages = 0;
    if (bulk_family) {
        bool dst_dense = true;                                 // rows of every task adjacent in its destinations
        for (const RsTask &T : op->tasks) dst_dense = dst_dense && (T.nd == 0 || T.dstride[0] == T.run_bytes);
        // how full the default 12 KiB slots would be, averaged over the bytes moved
        const int64_t tb0 = std::max<int64_t>(128, pick(P->tune.bulk_tile_bytes, RS_BULK_TILE_BYTES) / 128 * 128);
        double filled = 0, total = 0;
        for (RsTask T : op->tasks) {
            set_tiling(&T, tb0);
            const double bytes = (double)task_rows(T) * (double)T.run_bytes, tiles = (double)task_tiles_exact(T);
            if (tiles > 0) { filled += bytes; total += tiles * (double)tb0; }
        }
        bool underfilled = total > 0 && filled < RS_BULK_MIN_FILL * total;
        const bool tiny_tiles = total > 0 && filled < RS_BULK_TINY_FILL * total;
        // 1 : 1 operations in the tensor-map window (rows <= 2 KiB, 128-320 MiB moved: config 2) also take the 4-warp shape and with it the
        // pacing of that shape: config 2 43.6 -> 41.8 us (torch copy_ 42.4), its unpack 43.1 -> 41.6, 64 + 64 MiB 22.2-22.4 -> 21.7-22.0;
        // unpaced the 4 warps lose (45.5 us)
        if (path == RS_PATH_TMAP && write_bytes < 2 * read_bytes && read_bytes + write_bytes >= RS_PACE_11_MIN_BYTES) underfilled = true;
        BulkShape sh = bulk_shape(*P, path == RS_PATH_BULK_SHIFT, path == RS_PATH_TMAP, min_run, read_bytes, write_bytes, dst_dense, underfilled, tiny_tiles);
        tile_bytes = sh.tile_bytes;
        stages = sh.stages;
        op->pace_permille = sh.pace_permille;
        I.pace_permille = P->tune.pace_permille > 0 ? P->tune.pace_permille : P->tune.pace_permille < 0 ? 0 : sh.pace_permille;
        I.block = sh.warps * 32;
        I.grid = sh.grid;
        workers = sh.grid * sh.warps;
    } else {
        tile_bytes = pick(P->tune.lsu_tile_bytes, RS_LSU_TILE_BYTES);
        tile_bytes = std::max<int64_t>(128, tile_bytes / 128 * 128);
        I.block = RS_LSU_THREADS;
        // small operations are ramp-bound: more warps per SM cover the start-up latency (c3: 11.2 -> 10.1 us with 4 CTAs
        // per SM); large ones are DRAM-bound and do best with 2 (more bytes in flight is slower on B200)
        const bool small_op = read_bytes + write_bytes <= RS_SMALL_OP_BYTES;
        I.grid = P->sm_count * std::max(1, std::min(RS_LSU_CTAS_PER_SM, pick(P->tune.lsu_ctas_per_sm, small_op ? RS_LSU_CTAS_SMALL : write_bytes >= 2 * read_bytes ? RS_LSU_CTAS_MCAST : RS_LSU_CTAS_DEFAULT)));
        if (P->max_ctas > 0) I.grid = std::min(I.grid, P->max_ctas);
        workers = I.grid * (RS_LSU_THREADS / 32);
    }
    // small problems: shrink tiles until every worker has a few (tail balance), floor 2 KiB
    while (tile_bytes > 2048 && read_bytes / tile_bytes < (int64_t)workers * pick(P->tune.tiles_per_worker, RS_TILES_PER_WORKER)) tile_bytes = tile_bytes / 2 / 128 * 128;
    tile_bytes = std::max<int64_t>(tile_bytes, 128);
    I.tile_bytes = (int32_t)tile_bytes;

    int64_t total_tiles = 0;
    for (RsTask &T : op->tasks) { set_tiling(&T, tile_bytes); total_tiles += task_tiles_exact(T); }
    if (total_tiles > 0x7FFFFFFFll) { set_error("more than 2^31-1 tiles in one operation"); return RS_EUNSUPPORTED; }
    // Destination-address order only for execute and unpack (they write shards), only where slices share
    // destination rows at a fine grain (not config 4: 3 MiB runs), and not under a schedule: there the tables list
    // the unit tasks in order of S_i and the tiles follow them.
    bool interleaved = false;
    for (const RsTask &T : op->tasks)
        interleaved = interleaved || (T.nd >= 1 && T.run_bytes <= RS_INTERLEAVE_MAX_RUN && ((dst_order && T.dstride[0] > T.run_bytes) || T.sstride[0] > T.run_bytes));
    if (!per_task && !P->tune.task_order && P->sched.algorithm == RS_SCHED_NONE && interleaved && op->tasks.size() > 1) {
        group_interleaved(op, dst_order, /*by_src=*/true);
    } else {
        op->segs.resize(op->tasks.size());
        for (size_t t = 0; t < op->tasks.size(); t++) op->segs[t] = RsSeg{0, (uint32_t)t, 1, op->tasks[t].n_tiles};
    }
    uint32_t begin = 0;
    for (RsSeg &s : op->segs) { s.tile_begin = begin; begin += s.n_members * s.tiles_each; }
    I.n_tiles = (int32_t)begin;
    I.n_segs = (int32_t)op->segs.size();
    I.table_bytes = (int32_t)(op->tasks.size() * sizeof(RsTask) + op->dsts.size() * sizeof(RsDst) + op->segs.size() * sizeof(RsSeg));
    int64_t mr = INT64_MAX, pad = 0;
    for (const RsTask &T : op->tasks) { mr = std::min(mr, task_min_col(T)); pad = std::max(pad, task_shift_stage(T)); }
    I.min_run_bytes = op->tasks.empty() ? 0 : mr;
    {
        double bytes = 0, rows = 0;
        for (const RsTask &T : op->tasks) { bytes += (double)task_rows(T) * (double)T.run_bytes; rows += (double)task_rows(T); }
        op->mean_run_bytes = rows > 0 ? (int64_t)(bytes / rows) : 0;
    }
    // RS_PATH_TMAP: every buffer is seen as ONE 2-D byte matrix [rows][pitch] with ONE box shape; a task whose full
    // tiles fit the matrices of its source and of all its destinations moves them with tensor-map copies, everything
    // else (ragged last tiles, long or odd rows, other pitches) with the per-row bulk copies of rs_copy_bulk.
    for (int b = 0; b < RS_TMAP_BUFS; b++) { op->tmap_src[b] = RsTmapGeom{}; op->tmap_dst[b] = RsTmapGeom{}; }
    for (RsTask &T : op->tasks) T.tmap_ok = 0;
    if (path == RS_PATH_TMAP && op->src_cap > 0 && op->dst_cap > 0) {
        auto fits = [](RsTmapGeom &G, int64_t pitch, uint32_t cols, uint32_t rows, int64_t origin) {
            if (pitch <= 0 || pitch % 16 || pitch / RS_TMAP_ELEM > 0xFFFFFFFFll || origin % pitch + cols > pitch) return false;
            if (!G.valid) { G = RsTmapGeom{pitch, cols, rows, 1, 0}; return true; }
            return G.pitch == pitch && G.box_cols == cols && G.box_rows == rows;
        };
        for (RsTask &T : op->tasks) {
            if (T.kind != RS_TILING_FAST || T.rows_per_tile < 2 || T.rows_per_tile > 256 || T.run_bytes > 256 * RS_TMAP_ELEM || T.run_bytes % 16 ||
                T.src_buf >= RS_TMAP_BUFS) continue;
            RsTmapGeom src_try = op->tmap_src[T.src_buf];
            if (!fits(src_try, T.sstride[0], (uint32_t)T.run_bytes, T.rows_per_tile, T.src_off)) continue;
            RsTmapGeom dst_try[RS_TMAP_BUFS];
            for (int b = 0; b < RS_TMAP_BUFS; b++) dst_try[b] = op->tmap_dst[b];
            bool ok = true;
            for (int j = 0; j < T.k && ok; j++) {
                const RsDst &D = op->dsts[(size_t)T.dst_first + j];
                ok = D.buf < RS_TMAP_BUFS && fits(dst_try[D.buf], T.dstride[0], (uint32_t)T.run_bytes, T.rows_per_tile, D.off);
            }
            if (!ok) continue;
            op->tmap_src[T.src_buf] = src_try;
            for (int b = 0; b < RS_TMAP_BUFS; b++) op->tmap_dst[b] = dst_try[b];
            T.tmap_ok = 1;
        }
    }
    if (tmap_cover) {                                          // share of the bytes that move as whole tensor-map boxes
        double whole = 0, all = 0;
        for (const RsTask &T : op->tasks) {
            const double bytes = (double)task_rows(T) * (double)T.run_bytes;
            all += bytes;
            if (T.tmap_ok && T.nd >= 1) whole += bytes / (double)T.ext[0] * (double)(T.ext[0] / T.rows_per_tile * T.rows_per_tile);
        }
        *tmap_cover = path == RS_PATH_TMAP && all > 0 ? whole / all : 0.0;
    }
    op->shift_stage = 0;
    op->alt_stage = 0;
    bool lsu = !bulk_family;
    if (bulk_family) {
        const bool shift = path == RS_PATH_BULK_SHIFT;
        int warps = I.block / 32;
        int64_t stage = tile_bytes;
        if (shift) {
            stage = pad;
            while (stages > 2 && (int64_t)warps * (stages * stage + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX) stages--;
            while (warps > 1 && (int64_t)warps * (stages * stage + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX) warps--;
            I.block = warps * 32;
        }
        op->stages = stages;
        op->lookahead = std::max(1, std::min(stages - 1, shift ? pick(P->tune.shift_lookahead, stages - 1) : pick(P->tune.bulk_lookahead, RS_BULK_LOOKAHEAD)));
        I.grid = (int32_t)std::max<int64_t>(1, std::min<int64_t>(I.grid, (I.n_tiles + warps - 1) / warps));
        // Never two ring CTAs on one SM: with programmatic dependent launch the CTAs of the NEXT launch are placed as SMs free up, and a
        // shape small enough to fit twice piles two of them on the SMs that finished first (a 107 KiB launch behind a 148 KiB one: 5.56
        // instead of 6.45 TB/s for the pair).  Asking for more than half of the SM's shared memory makes the hand-over one for one.
        // (Operations under 384 MiB keep their natural size: two of them share an SM on purpose -- the successor's prologue runs beside the
        // predecessor, config 3: 8.0 against 8.55 us -- and a pile-up lasts microseconds.)
        const int64_t min_smem = read_bytes + write_bytes >= RS_RING_MIN_SMEM_FROM ? pick(P->tune.ring_min_smem, RS_RING_MIN_SMEM) : 0;
        I.smem_bytes = (int32_t)std::max<int64_t>(warps * (stages * stage + RS_BULK_DESC_BYTES) + 1024, min_smem);
        if (shift) op->shift_stage = (uint32_t)stage;
        if (!shift) {
            // An aligned plan may be handed under-aligned pointers at execute time: keep a launch shape of the
            // shifted TMA kernel for the SAME tiles (rows padded in the ring, so fewer warps or slots fit).
            const bool long_rows = min_run >= RS_SHIFT_LONG_RUN;
            const bool mid_rows = !long_rows && min_run >= RS_SHIFT_MID_RUN;
            int aw = long_rows ? RS_SHIFT_WARPS_LONG : mid_rows ? RS_SHIFT_WARPS_MID : RS_SHIFT_WARPS;
            int as = long_rows ? RS_SHIFT_STAGES_LONG : mid_rows ? RS_SHIFT_STAGES_MID : RS_SHIFT_STAGES;
            while (as > 2 && (int64_t)aw * (as * pad + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX) as--;
            while (aw > 1 && (int64_t)aw * (as * pad + RS_BULK_DESC_BYTES) + 1024 > RS_SMEM_MAX) aw--;
            if ((int64_t)aw * (as * pad + RS_BULK_DESC_BYTES) + 1024 <= RS_SMEM_MAX && I.n_tiles > 0) {
                op->alt_stage = (uint32_t)pad; op->alt_warps = aw; op->alt_stages = as;
                op->alt_smem = (int)std::max<int64_t>(aw * (as * pad + RS_BULK_DESC_BYTES) + 1024, min_smem);
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
        // GENERIC tiles decode every vector's row (divisions): instruction-bound, so more warps per SM than the DRAM-bound
        // fast walk wants (spans of 128 bytes, 320 + 640 MiB: 2.8 TB/s with 1 CTA per SM, 4.2 with 2; 1 : 1: 3.3 with 2, 4.1 with 4)
        bool generic = false;
        for (const RsTask &T : op->tasks) generic = generic || T.kind == RS_TILING_GENERIC;
        if (generic && !P->tune.lsu_ctas_per_sm && I.path == RS_PATH_LSU) {
            I.grid = P->sm_count * (write_bytes >= 2 * read_bytes ? 2 : RS_LSU_CTAS_PER_SM);
            if (P->max_ctas > 0) I.grid = std::min(I.grid, P->max_ctas);
        }
        int64_t want = (I.n_tiles + warps - 1) / warps;
        if (want < P->sm_count) want = std::min<int64_t>(I.n_tiles, P->sm_count);   // few tiles: still one CTA on every SM (api.cu)
        I.grid = (int32_t)std::max<int64_t>(1, std::min<int64_t>(I.grid, want));
        I.smem_bytes = 0;
    }
    return RS_OK;
}

// AUTO may route an operation made of short rows through the tensor-map kernel; that only pays if nearly every tile moves as a
// whole box (a tile that does not falls back to one bulk copy per 128-byte row), so the choice is checked and undone otherwise.
rs_status finish_op(Plan *P, OpTables *op, int64_t read_bytes, int64_t write_bytes, bool per_task = false, bool dst_order = false) {
    double cover = 0;
    rs_status st = finish_op_impl(P, op, read_bytes, write_bytes, per_task, dst_order, /*tmap_short=*/!per_task, &cover);
    if (st != RS_OK) return st;
    int64_t min_run = INT64_MAX;
    for (const RsTask &T : op->tasks) min_run = std::min(min_run, T.run_bytes);
    // (1 : 1 operations whose tiles are tiny -- spans of 1-3 KiB -- are better off in registers, 16 warps per SM: fm_hw 5.7 against
    // 4.7 TB/s; write-heavy ones are not, the register path has no pacing: fm_hwm 4.7 against 6.0)
    const bool tiny_11 = write_bytes < 2 * read_bytes && op->info.n_tiles > 0 && read_bytes / op->info.n_tiles < RS_TMAP_SHORT_MIN_TILE;
    if (op->info.path == RS_PATH_TMAP && !(P->flags & RS_PATH_MASK) && min_run < RS_BULK_MIN_RUN && (cover < RS_TMAP_SHORT_MIN_COVER || tiny_11))
        st = finish_op_impl(P, op, read_bytes, write_bytes, per_task, dst_order, /*tmap_short=*/false, nullptr);
    return st;
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
    H.tasks.clear(); H.dsts.clear(); H.segs.clear();
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
    rs_status st = finish_op(P, &H, tensor_bytes, tensor_bytes * P->r_B, /*per_task=*/true);
    if (st != RS_OK) return st;
    for (HostSlab &S : P->slabs) { S.tile_begin = 0xFFFFFFFFu; S.tile_end = 0; }
    for (size_t t = 0; t < task_slab.size(); t++) {           // one segment per task, in task order
        HostSlab &S = P->slabs[task_slab[t]];
        S.tile_begin = std::min(S.tile_begin, H.segs[t].tile_begin);
        S.tile_end = std::max(S.tile_end, H.segs[t].tile_begin + H.segs[t].tiles_each);
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
    for (OpTables &o : G->op) { o.tasks.clear(); o.dsts.clear(); o.segs.clear(); o.info = rs_op_info{}; }
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
    return finish_op(G, &X, rd, wr, false, true);
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
    for (OpTables *o : {&X, &PK, &UP}) { o->tasks.clear(); o->dsts.clear(); o->segs.clear(); }

    const bool sharded = !P->src_owner.empty();               // multi-process executor: only this rank's unit tasks
    int64_t my_read = 0, my_write = 0;
    for (int i : P->exec_order) {                              // slice-id order, or the schedule's (S3.2)
        const Slice &S = P->slices[(size_t)i];
        if (sharded && P->src_owner[(size_t)S.sender] != P->rank) continue;
        my_read += S.elems * e;
        my_write += S.elems * e * (int64_t)S.receivers.size();
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
    for (OpTables *o : {&SR, &AS, &AG, &LS, &LG}) { o->tasks.clear(); o->dsts.clear(); o->segs.clear(); o->info = rs_op_info{}; }
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
    P->used_dst.assign((size_t)B.n_dev, 0);
    for (const RsDst &D : X.dsts) P->used_dst[(size_t)D.buf] = 1;
    if (sharded) {
        // A rank of the multi-process executor runs reshard_execute only: its share of the unit tasks, written to
        // local and peer-mapped destination shards.  pack / unpack / the host pipeline belong to single-process plans.
        PK.tasks.clear(); PK.dsts.clear(); UP.tasks.clear(); UP.dsts.clear();
        OpTables &H = P->op[RS_OP_SLABS];
        H.tasks.clear(); H.dsts.clear(); H.segs.clear(); H.info = rs_op_info{};
        P->slabs.clear();
        P->used_src.assign((size_t)A.n_dev, 0);
        for (const RsTask &T : X.tasks) P->used_src[(size_t)T.src_buf] = 1;
        if ((st = finish_op(P, &X, my_read, my_write, false, true)) != RS_OK) return st;
        if ((st = finish_op(P, &PK, 0, 0)) != RS_OK) return st;
        return finish_op(P, &UP, 0, 0);
    }
    if ((st = build_slabs(P, sA, sB, tensor_bytes)) != RS_OK) return st;
    const int64_t cap_a = A.shard_elems() * e, cap_b = B.shard_elems() * e;
    X.src_cap = cap_a; X.dst_cap = cap_b; PK.src_cap = cap_a; PK.dst_cap = P->arena_bytes; UP.src_cap = P->arena_bytes; UP.dst_cap = cap_b;
    if ((st = finish_op(P, &X, tensor_bytes, tensor_bytes * P->r_B, false, true)) != RS_OK) return st;
    if ((st = finish_op(P, &PK, tensor_bytes, tensor_bytes * P->r_B)) != RS_OK) return st;
    if ((st = finish_op(P, &UP, tensor_bytes * P->r_B, tensor_bytes * P->r_B, false, true)) != RS_OK) return st;
    return RS_OK;
}

}  // namespace rs

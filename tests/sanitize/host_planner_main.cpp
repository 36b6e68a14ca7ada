// host_planner_main.cpp -- TEST-ONLY driver: the host side of libreshard.so (planner, scheduler, table builder,
// procedural tile decode, pipeline simulator; no CUDA) compiled with -fsanitize=address,undefined and run over
// the BASELINE shapes, the unaligned / uneven workloads, Table 2 cases 4 and 6, the interface maxima, every
// schedule algorithm and path flag.  tests/test_sanitizers.py builds and runs it; any sanitizer report or
// out-of-bounds tile fails the test.  Every tile of every operation is decoded with the routine the kernels run
// (csrc/tables.h) and its byte ranges are checked against the buffer sizes.
#include <cstdio>
#include <cstring>

#include "../../paper_2211_05322_b200/csrc/plan.hpp"
using namespace rs;

static int64_t g_tiles = 0, g_plans = 0;

static bool check_op(const Plan &P, int opi, const char *what) {
    const OpTables &o = P.op[opi];
    const int64_t src_cap = opi == RS_OP_UNPACK ? P.arena_bytes : P.A.shard_elems() * P.elem_bytes;
    const int64_t dst_cap = opi == RS_OP_PACK ? P.arena_bytes : P.B.shard_elems() * P.elem_bytes;
    const int64_t gather_cap = P.B.shard_elems() * P.elem_bytes;          // all-gather phase 2 reads destination shards
    int64_t bytes = 0;
    const uint32_t step = o.info.n_tiles > 200000 ? 37 : 1;                // huge operations: every 37th tile + the last
    for (uint32_t t = 0; t < (uint32_t)o.info.n_tiles; t += (t + step < (uint32_t)o.info.n_tiles || t + 1 == (uint32_t)o.info.n_tiles) ? step : (uint32_t)o.info.n_tiles - 1 - t) {
        uint32_t task, u;
        rs_tile_locate(o.segs.data(), (uint32_t)o.segs.size(), t, &task, &u);
        if (task >= o.tasks.size() || u >= o.tasks[task].n_tiles) { std::printf("%s: tile %u -> task %u tile %u out of range\n", what, t, task, u); return false; }
        const RsTask &T = o.tasks[task];
        const RsTile tile = rs_tile_decode(T, task, u);
        const int64_t scap = (opi == RS_OP_AG_GATHER || opi == RS_OP_AGL_GATHER) ? gather_cap : src_cap;
        for (uint32_t r = 0; r < tile.n_rows; r += (tile.n_rows > 1 ? tile.n_rows - 1 : 1)) {   // first and last row
            int64_t so, doff;
            if (tile.flags & RS_TILE_FAST) { so = (int64_t)tile.a + (int64_t)r * T.sstride[0]; doff = (int64_t)tile.b + (int64_t)r * T.dstride[0]; }
            else { rs_row_offsets(T, 0, (uint32_t)tile.a + r, &so, &doff); }
            if (T.src_off + so < 0 || T.src_off + so + tile.col_bytes > scap) { std::printf("%s: tile %u reads outside its source\n", what, t); return false; }
            for (int j = 0; j < T.k; j++) {
                const RsDst &D = o.dsts[(size_t)T.dst_first + j];
                if (D.off + doff < 0 || D.off + doff + tile.col_bytes > dst_cap) { std::printf("%s: tile %u writes outside destination %d\n", what, t, j); return false; }
            }
        }
        bytes += (int64_t)tile.n_rows * tile.col_bytes;
        g_tiles++;
        if (step == 1 && t + 1 == (uint32_t)o.info.n_tiles) break;
    }
    if (step == 1 && bytes != o.info.read_bytes && opi <= RS_OP_SLABS) { std::printf("%s: tiles cover %lld of %lld bytes\n", what, (long long)bytes, (long long)o.info.read_bytes); return false; }
    return true;
}

static int run(std::vector<int64_t> shape, int e, std::vector<int32_t> sm, const char *ss, std::vector<int32_t> dm, const char *ds, uint32_t flags, int sched, int dph, int tile_bytes = 0) {
    Plan P; P.elem_bytes = e; P.flags = flags | RS_HOST_ONLY;
    P.sched.algorithm = sched; P.sched.src_dph = dph; P.sched.dst_dph = dph; P.sched.seed = 7; P.sched.node_budget = 20000;
    P.tune.bulk_tile_bytes = P.tune.lsu_tile_bytes = P.tune.shift_tile_bytes = tile_bytes;
    rs_status st = make_layout(shape.data(), (int)shape.size(), sm.data(), (int)sm.size(), ss, false, &P.A);
    if (st == RS_OK) st = make_layout(shape.data(), (int)shape.size(), dm.data(), (int)dm.size(), ds, false, &P.B);
    if (st == RS_OK) st = build_slices(&P);
    if (st != RS_OK) { std::printf("%s -> %s: status %d (%s)\n", ss, ds, st, last_error().c_str()); return 1; }
    P.exec_order.resize(P.slices.size());
    for (size_t i = 0; i < P.slices.size(); i++) P.exec_order[i] = (int)i;
    if (sched == 0) choose_senders(&P); else st = schedule_plan(&P);
    if (st == RS_OK) st = build_messages(&P);
    if (st == RS_OK) st = build_tables(&P);
    if (st != RS_OK) { std::printf("%s -> %s sched %d: status %d (%s)\n", ss, ds, sched, st, last_error().c_str()); return 1; }
    g_plans++;
    char what[256];
    for (int opi = 0; opi < RS_N_OPS; opi++) {
        std::snprintf(what, sizeof what, "%s -> %s sched %d flags %x op %d", ss, ds, sched, flags, opi);
        if (!check_op(P, opi, what)) return 1;
    }
    return 0;
}

int main() {
    int bad = 0;
    for (int sched = 0; sched <= 5; sched++) for (uint32_t fl : {0u, (uint32_t)RS_WITH_STRATEGIES, (uint32_t)RS_PATH_BULK_SHIFT, (uint32_t)RS_PATH_LSU}) {
        bad += run({8, 16}, 4, {1, 2}, "S0,R", {1, 2}, "R,S0", fl, sched, 1);                                   // BASELINE config 1
        bad += run({16, 1024, 4096}, 2, {2, 4}, "S0,R,S1", {2, 4}, "S0,S1,R", fl, sched, 4);                    // config 2
        bad += run({8, 320, 64, 64}, 2, {1, 4}, "S0,R,R,R", {2, 2}, "R,S0,S1,R", fl, sched, 2);                 // config 3
        bad += run({8, 320, 64, 64}, 2, {1, 4}, "S1,R,R,R", {2, 2}, "R,S0,R,R", fl, sched, 2);                  // config 3''
        bad += run({32, 2048, 12288}, 2, {2, 4}, "S0,S1,R", {4, 2}, "S1,R,S0", fl, sched, 4);                   // config 4
        bad += run({30, 2047, 12290}, 2, {2, 4}, "S0,S1,R", {4, 2}, "S1,R,S0", fl, sched, 1);                   // u4: nothing aligned
        bad += run({1024, 1024, 512}, 2, {2, 4}, "RS01R", {2, 4}, "S01RR", fl, sched, 4);                       // Table 2 case 4
        bad += run({1024, 1024, 512}, 2, {2, 4}, "S0RR", {3, 4}, "S0RR", fl, sched, 4);                         // Table 2 case 6 (uneven)
        bad += run({2, 3, 2, 2, 4, 2, 2, 6}, 2, {2, 2, 2, 2}, "S0,R,S1,R,S2,R,R,S3", {2, 2, 2, 2}, "R,S3,R,S2,R,S1,S0,R", fl, sched, 2);
        bad += run({256, 2}, 4, {1}, "R,R", {128}, "R,R", fl, sched, 3);
        bad += run({7, 5, 3}, 1, {2, 3}, "S1,R,S0", {3, 2}, "R,S0,S1", fl, sched, 1);
        bad += run({8, 6, 2, 16}, 4, {2, 2}, "S0,R,R,S1", {2, 2}, "R,S0,R,S1", fl, sched, 1, 128);              // GENERIC tiles
        bad += run({4, 6, 64}, 4, {2, 2}, "S0,S1,R", {2, 2}, "S1,S0,R", fl, sched, 1, 128);                     // SPLIT rows
    }
    for (const char *pair : {"S0,R,S1>S0,S1,R", "R,R,S0>S0,R,R", "S0,S1,R>S1,S0,R", "R,S0,S1>R,S1,S0", "S0,R,R>R,R,R", "R,R,R>S0,S1,R"}) {
        std::string a(pair, std::strchr(pair, '>') - pair), b(std::strchr(pair, '>') + 1);
        for (int64_t B : {8ll, 64ll, 256ll}) {                                                                  // config 5: 1 MiB .. 4 GiB
            const int64_t S = B == 8 ? 16 : 2048;
            bad += run({B, S, 4096}, 2, {2, 4}, a.c_str(), {2, 4}, b.c_str(), 0, 0, 1);
            bad += run({B, S, 4096}, 2, {1, 4}, a.c_str(), {2, 2}, b.c_str(), 0, 0, 1);
        }
    }
    int64_t f[4] = {3, 4, 5, 6}, b[4] = {6, 8, 10, 12}, ba[4] = {3, 4, 5, 6};
    for (int sc = 0; sc < 2; sc++) for (int ov = 0; ov < 2; ov++) for (int d = 0; d < 3; d++) {
        rs_pipeline_opts o; std::memset(&o, 0, sizeof(o));
        o.schedule = sc; o.n_stages = 4; o.n_micro_batches = 9; o.overlap = ov; o.bw_delay = d; o.fwd = f; o.bwd = b; o.bwd_act = d ? ba : nullptr; o.comm_fwd = 2; o.comm_bwd = 3;
        rs_pipeline_result r; std::vector<int32_t> k(4 * 27), m(4 * 27); std::vector<int64_t> s(4 * 27), e(4 * 27);
        if (pipeline_simulate(o, &r, k.data(), m.data(), s.data(), e.data()) != RS_OK || r.makespan <= 0) bad++;
    }
    std::printf("%lld plans, %lld tiles decoded and bounds-checked, %d failures\n", (long long)g_plans, (long long)g_tiles, bad);
    return bad ? 1 : 0;
}

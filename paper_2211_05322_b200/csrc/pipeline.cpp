// pipeline.cpp -- S4 of the paper on the host: 1F1B and eager-1F1B op orders and the timeline of one
// training iteration whose stage-boundary transfers are cross-mesh resharding tasks.
//
//   warm-up        1F1B: #stages - i + 1 forwards, eager-1F1B: 2 (#stages - i) + 1
//   dependency     compute(i, m) -> transfer i -> i+1 -> compute(i+1, m)
//   overlap        eager-1F1B puts other micro-batches' compute between dependent tasks
//   memory         at most #stages more live activations per stage
//   weight delay   backward = activation gradients (feed the transfer) + weight gradients
// Readings R28-R32.  Times are integer ticks; no CUDA here.
#include <algorithm>
#include <cstring>
#include <vector>

#include "../../include/reshard.h"
#include "plan.hpp"

namespace rs {

namespace {

struct Op { int32_t kind, micro; };      // kind: RS_PIPE_F / RS_PIPE_B / RS_PIPE_BA / RS_PIPE_BW

int warmup(int schedule, int S, int stage, int M) {
    const int w = schedule == RS_PIPE_EAGER_1F1B ? 2 * (S - stage) + 1 : S - stage + 1;
    return std::min(w, M);
}

// warm-up forwards, then one backward / one forward alternately, then the remaining backwards (R31);
// split: every B becomes BA and a BW `delay` ops later (R32)
std::vector<Op> stage_ops(int schedule, int S, int stage, int M, bool split, int delay) {
    std::vector<Op> ops;
    const int w = warmup(schedule, S, stage, M);
    for (int m = 0; m < w; m++) ops.push_back({RS_PIPE_F, m});
    for (int nf = w, nb = 0; nb < M; nb++) {
        ops.push_back({RS_PIPE_B, nb});
        if (nf < M) ops.push_back({RS_PIPE_F, nf++});
    }
    if (!split) return ops;
    std::vector<Op> out;
    std::vector<std::pair<int, int>> pending;              // (ops still to pass, micro-batch), FIFO
    for (const Op &o : ops) {
        for (auto &p : pending) p.first--;
        if (o.kind == RS_PIPE_B) { out.push_back({RS_PIPE_BA, o.micro}); pending.push_back({delay, o.micro}); }
        else out.push_back(o);
        while (!pending.empty() && pending.front().first <= 0) {
            out.push_back({RS_PIPE_BW, pending.front().second});
            pending.erase(pending.begin());
        }
    }
    for (auto &p : pending) out.push_back({RS_PIPE_BW, p.second});
    return out;
}

}  // namespace

rs_status pipeline_simulate(const rs_pipeline_opts &o, rs_pipeline_result *res, int32_t *op_kind, int32_t *op_micro,
                            int64_t *op_start, int64_t *op_end) {
    const int S = o.n_stages, M = o.n_micro_batches;
    if (S < 1 || S > RS_PIPE_MAX_STAGES || M < 1 || !o.fwd || !o.bwd) { set_error("pipeline: bad stage / micro-batch count or null times"); return RS_EINVAL; }
    if (o.schedule != RS_PIPE_1F1B && o.schedule != RS_PIPE_EAGER_1F1B) { set_error("pipeline: unknown schedule"); return RS_EINVAL; }
    if (o.comm_fwd < 0 || o.comm_bwd < 0 || o.bw_delay < 0) { set_error("pipeline: negative time or delay"); return RS_EINVAL; }
    const bool split = o.bwd_act != nullptr;
    for (int i = 0; i < S; i++)
        if (o.fwd[i] < 0 || o.bwd[i] < 0 || (split && (o.bwd_act[i] < 0 || o.bwd_act[i] > o.bwd[i]))) { set_error("pipeline: bad compute time"); return RS_EINVAL; }
    const int grad = split ? RS_PIPE_BA : RS_PIPE_B;
    std::vector<std::vector<Op>> ops((size_t)S);
    for (int i = 0; i < S; i++) ops[(size_t)i] = stage_ops(o.schedule, S, i + 1, M, split, o.bw_delay);
    const size_t per_stage = ops[0].size();                  // M forwards + M backwards (+ M weight-gradient ops)
    auto dur = [&](int i, int kind) -> int64_t {
        switch (kind) {
            case RS_PIPE_F: return o.fwd[i];
            case RS_PIPE_B: return o.bwd[i];
            case RS_PIPE_BA: return o.bwd_act[i];
            default: return o.bwd[i] - o.bwd_act[i];
        }
    };
    const int64_t NONE = -1;
    // end[kind][stage][micro], arrive[F or grad][stage][micro]
    std::vector<int64_t> end_f((size_t)S * M, NONE), end_g((size_t)S * M, NONE), arr_f((size_t)S * M, NONE), arr_g((size_t)S * M, NONE);
    std::vector<int64_t> free_at((size_t)S, 0), link_f((size_t)S, 0), link_b((size_t)S, 0), start((size_t)S * per_stage), end((size_t)S * per_stage);
    std::vector<size_t> pos((size_t)S, 0);
    size_t remaining = (size_t)S * per_stage;
    while (remaining) {
        bool progressed = false;
        for (int i = 0; i < S; i++) {
            while (pos[(size_t)i] < per_stage) {
                const Op op = ops[(size_t)i][pos[(size_t)i]];
                const size_t im = (size_t)i * M + (size_t)op.micro;
                int64_t ready;
                if (op.kind == RS_PIPE_F) ready = i == 0 ? 0 : arr_f[im];
                else if (op.kind == grad) ready = end_f[im] == NONE ? NONE : (i == S - 1 ? end_f[im] : arr_g[im]);
                else ready = end_g[im];                          // BW: after its BA
                if (ready == NONE) break;                        // strictly in list order (R29)
                const int64_t s = std::max(free_at[(size_t)i], ready), e = s + dur(i, op.kind);
                start[(size_t)i * per_stage + pos[(size_t)i]] = s;
                end[(size_t)i * per_stage + pos[(size_t)i]] = e;
                free_at[(size_t)i] = e;
                if (op.kind == RS_PIPE_F) end_f[im] = e;
                if (op.kind == grad) end_g[im] = e;
                if (op.kind == RS_PIPE_F && i < S - 1) {         // transfer i -> i+1 on that boundary's forward link (R30)
                    const int64_t ts = std::max(e, link_f[(size_t)i]);
                    link_f[(size_t)i] = ts + o.comm_fwd;
                    arr_f[im + (size_t)M] = ts + o.comm_fwd;
                    if (!o.overlap) free_at[(size_t)i] = ts + o.comm_fwd;
                } else if (op.kind == grad && i > 0) {
                    const int64_t ts = std::max(e, link_b[(size_t)i - 1]);
                    link_b[(size_t)i - 1] = ts + o.comm_bwd;
                    arr_g[im - (size_t)M] = ts + o.comm_bwd;
                    if (!o.overlap) free_at[(size_t)i] = ts + o.comm_bwd;
                }
                pos[(size_t)i]++;
                remaining--;
                progressed = true;
            }
        }
        if (!progressed) { set_error("pipeline: schedule deadlocks"); return RS_EINVAL; }
    }
    if (res) {
        std::memset(res, 0, sizeof(*res));
        res->ops_per_stage = (int32_t)per_stage;
        for (int i = 0; i < S; i++) {
            int live = 0, peak = 0;
            int64_t busy = 0;
            for (size_t k = 0; k < per_stage; k++) {
                const Op &op = ops[(size_t)i][k];
                if (op.kind == RS_PIPE_F) peak = std::max(peak, ++live);
                else if (op.kind == grad) live--;
                busy += dur(i, op.kind);
                res->makespan = std::max(res->makespan, end[(size_t)i * per_stage + k]);
            }
            res->peak_activations[i] = peak;
            res->busy[i] = busy;
            res->warmup[i] = warmup(o.schedule, S, i + 1, M);
        }
    }
    for (int i = 0; i < S; i++)
        for (size_t k = 0; k < per_stage; k++) {
            const size_t x = (size_t)i * per_stage + k;
            if (op_kind) op_kind[x] = ops[(size_t)i][k].kind;
            if (op_micro) op_micro[x] = ops[(size_t)i][k].micro;
            if (op_start) op_start[x] = start[x];
            if (op_end) op_end[x] = end[x];
        }
    return RS_OK;
}

// PAPER.md:217 cost model: the least delay whose intervening compute (the ops a stage runs between BA(m)
// and its BW(m), BW included) covers the backward transfer; -1 if none up to 2 M does
int pipeline_least_delay(int schedule, int S, int stage, int M, int64_t f, int64_t b, int64_t b_act, int64_t c_bwd) {
    for (int delay = 0; delay <= 2 * M; delay++) {
        const std::vector<Op> ops = stage_ops(schedule, S, stage, M, true, delay);
        size_t k = 0;
        while (k < ops.size() && ops[k].kind != RS_PIPE_BA) k++;
        if (k == ops.size()) return 0;
        int64_t covered = 0;
        for (size_t j = k + 1; j < ops.size(); j++) {
            covered += ops[j].kind == RS_PIPE_F ? f : ops[j].kind == RS_PIPE_BA ? b_act : b - b_act;
            if (ops[j].kind == RS_PIPE_BW && ops[j].micro == ops[k].micro) break;
        }
        if (covered >= c_bwd) return delay;
    }
    return -1;                                                 // no delay up to 2 M covers the transfer
}

}  // namespace rs

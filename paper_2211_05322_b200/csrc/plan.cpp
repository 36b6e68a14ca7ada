// plan.cpp -- host planner: spec -> boxes -> unit tasks -> senders -> messages (steps a1..a4).
// The table builder (a5) is in tables.cpp.  No CUDA here.
#include "plan.hpp"

#include <algorithm>
#include <cctype>
#include <functional>
#include <map>
#include <numeric>

namespace rs {

static thread_local std::string g_last_error;
void set_error(const std::string &msg) { g_last_error = msg; }
const std::string &last_error() { return g_last_error; }

// ------------------------------------------------------------------ a1: spec -> layout -> boxes

// X_0^{d_0} ... X_{N-1}^{d_{N-1}}, X in {S, R}.  Separators and TeX decoration are skipped.
static rs_status parse_spec(const char *text, int ndim, int mesh_ndim, Layout *L) {
    if (!text) return RS_EINVAL;
    bool used[RS_MAX_MESH_NDIM] = {false, false, false, false};
    int n = 0;
    const char *p = text;
    auto is_sep = [](char c) {
        return c == ',' || c == ' ' || c == '\t' || c == '(' || c == ')' || c == '[' || c == ']';
    };
    while (*p) {
        if (is_sep(*p)) { ++p; continue; }
        char c = (char)std::toupper((unsigned char)*p);
        if (c != 'R' && c != 'S') { set_error(std::string("spec: unexpected character in '") + text + "'"); return RS_ESPEC; }
        if (n >= ndim) { set_error(std::string("spec '") + text + "' has more entries than tensor dims"); return RS_ESPEC; }
        ++p;
        L->n_axes[n] = 0;
        if (c == 'S') {
            while (*p == '^' || *p == '{' || *p == '_' || *p == ' ') ++p;
            while (std::isdigit((unsigned char)*p)) {
                int a = *p - '0';
                if (a >= mesh_ndim) { set_error(std::string("spec '") + text + "': mesh axis out of range"); return RS_ESPEC; }
                if (used[a]) { set_error(std::string("spec '") + text + "': mesh axis used twice (R3)"); return RS_ESPEC; }
                used[a] = true;
                L->axes[n][L->n_axes[n]++] = a;
                ++p;
            }
            while (*p == '}') ++p;
            if (L->n_axes[n] == 0) { set_error(std::string("spec '") + text + "': S without a mesh axis"); return RS_ESPEC; }
        }
        ++n;
    }
    if (n != ndim) { set_error(std::string("spec '") + text + "' has fewer entries than tensor dims"); return RS_ESPEC; }
    return RS_OK;
}

rs_status make_layout(const int64_t *shape, int ndim, const int32_t *mesh, int mesh_ndim, const char *spec,
                      bool even_only, Layout *L) {
    if (!shape || !mesh || !spec) { set_error("null argument"); return RS_EINVAL; }
    if (ndim < 1 || ndim > RS_MAX_NDIM) { set_error("ndim out of range"); return RS_EINVAL; }
    if (mesh_ndim < 1 || mesh_ndim > RS_MAX_MESH_NDIM) { set_error("mesh_ndim out of range"); return RS_EINVAL; }
    L->ndim = ndim;
    L->mesh_ndim = mesh_ndim;
    int64_t n_dev = 1;
    for (int a = 0; a < mesh_ndim; a++) {
        if (mesh[a] < 1) { set_error("mesh extent < 1"); return RS_EINVAL; }
        L->mesh[a] = mesh[a];
        n_dev *= mesh[a];
        if (n_dev > RS_MAX_DEVICES) { set_error("more than RS_MAX_DEVICES devices in a mesh"); return RS_EUNSUPPORTED; }
    }
    L->n_dev = (int)n_dev;
    for (int i = 0; i < ndim; i++) {
        if (shape[i] < 1) { set_error("tensor extent < 1"); return RS_EINVAL; }
        L->shape[i] = shape[i];
    }
    rs_status st = parse_spec(spec, ndim, mesh_ndim, L);
    if (st != RS_OK) return st;
    for (int i = 0; i < ndim; i++) {
        int64_t k = 1;
        for (int j = 0; j < L->n_axes[i]; j++) k *= L->mesh[L->axes[i][j]];
        if (even_only && L->shape[i] % k) { set_error("tensor dim not divisible by its sharding degree (RS_EVEN_ONLY)"); return RS_EDIVIS; }
        L->degree[i] = k;
        L->local[i] = (L->shape[i] + k - 1) / k;              // R5: padded extent c_i = ceil(l_i / k_i)
    }
    // shard index p_i of every device: row-major coordinates, first listed axis most
    // significant (R2).
    L->shard_index.assign((size_t)L->n_dev * ndim, 0);
    for (int r = 0; r < L->n_dev; r++) {
        int64_t c[RS_MAX_MESH_NDIM];
        int64_t rem = r;
        for (int a = mesh_ndim - 1; a >= 0; a--) { c[a] = rem % L->mesh[a]; rem /= L->mesh[a]; }
        for (int i = 0; i < ndim; i++) {
            int64_t p = 0;
            for (int j = 0; j < L->n_axes[i]; j++) p = p * L->mesh[L->axes[i][j]] + c[L->axes[i][j]];
            L->shard_index[(size_t)r * ndim + i] = p;
        }
    }
    return RS_OK;
}

void device_box(const Layout &L, int dev, int64_t *lo, int64_t *hi) {
    for (int i = 0; i < L.ndim; i++) {
        int64_t p = L.shard_index[(size_t)dev * L.ndim + i];
        lo[i] = std::min(p * L.local[i], L.shape[i]);         // R5: clipped; empty when p c_i >= l_i
        hi[i] = std::min((p + 1) * L.local[i], L.shape[i]);
    }
}

// ------------------------------------------------------------------ a2 + a3: unit tasks (App. B.2)

rs_status build_slices(Plan *P) {
    const Layout &A = P->A, &B = P->B;
    const int N = A.ndim;
    // Cut(d) = {0, l_d} U {j l_d / k_A} U {j l_d / k_B}
    std::vector<std::vector<int64_t>> cut(N);
    int64_t n_slices = 1;
    for (int d = 0; d < N; d++) {
        std::vector<int64_t> &c = cut[d];
        for (int64_t j = 0; j <= A.degree[d]; j++) c.push_back(std::min(j * A.local[d], A.shape[d]));
        for (int64_t j = 0; j <= B.degree[d]; j++) c.push_back(std::min(j * B.local[d], A.shape[d]));
        std::sort(c.begin(), c.end());
        c.erase(std::unique(c.begin(), c.end()), c.end());
        n_slices *= (int64_t)c.size() - 1;                    // #slices = prod (#Cut(d) - 1)
        if (n_slices > (1 << 24)) { set_error("more than 2^24 unit tasks"); return RS_EUNSUPPORTED; }
    }
    P->slices.resize((size_t)n_slices);
    std::vector<int64_t> idx(N, 0);
    for (int64_t s = 0; s < n_slices; s++) {                  // row-major over I_0 x ... x I_{N-1}
        Slice &S = P->slices[(size_t)s];
        S.elems = 1;
        for (int d = 0; d < N; d++) {
            S.lo[d] = cut[d][(size_t)idx[d]];
            S.hi[d] = cut[d][(size_t)idx[d] + 1];
            S.elems *= S.hi[d] - S.lo[d];
        }
        // N_i / M_i: devices whose tile contains the slice.  A slice never straddles
        // a shard boundary of either side, so containment == "same shard index on every dim".
        for (int r = 0; r < A.n_dev; r++) {
            bool in = true;
            for (int d = 0; d < N && in; d++) in = A.shard_index[(size_t)r * N + d] == S.lo[d] / A.local[d];
            if (in) S.senders.push_back(r);
        }
        for (int r = 0; r < B.n_dev; r++) {
            bool in = true;
            for (int d = 0; d < N && in; d++) in = B.shard_index[(size_t)r * N + d] == S.lo[d] / B.local[d];
            if (in) S.receivers.push_back(r);
        }
        if (S.senders.empty() || S.receivers.empty()) { set_error("internal: slice without sender or receiver"); return RS_EINVAL; }
        for (int d = N - 1; d >= 0; d--) {                    // next multi-index
            if (++idx[d] < (int64_t)cut[d].size() - 1) break;
            idx[d] = 0;
        }
    }
    P->r_B = (int64_t)P->slices[0].receivers.size();          // every element has the same #holders
    return RS_OK;
}

// ------------------------------------------------------------------ a4: sender choice (Eq. 4)

// Exact minimum makespan of `w` (sorted descending) on m identical machines, branch and bound.
// Used to finish small replica groups (R9): LPT alone is only a 4/3-approximation when slice
// sizes differ.  This is the paper's DFS-with-pruning idea restricted to Eq. 4.
namespace {
struct ExactLB {
    const std::vector<int64_t> &w;
    int m;
    std::vector<int64_t> load;
    std::vector<int> cur, best_assign;
    int64_t best;
    int64_t nodes = 0;
    ExactLB(const std::vector<int64_t> &w_, int m_, int64_t ub, const std::vector<int> &ub_assign)
        : w(w_), m(m_), load((size_t)m_, 0), cur(w_.size(), 0), best_assign(ub_assign), best(ub) {}
    void dfs(size_t i, int64_t cur_max, int64_t lower) {
        if (best <= lower || nodes > 2000000) return;          // optimal already, or budget spent
        ++nodes;
        if (i == w.size()) {
            if (cur_max < best) { best = cur_max; best_assign = cur; }
            return;
        }
        for (int k = 0; k < m; k++) {
            bool dup = false;                                  // symmetry: skip machines with equal load
            for (int j = 0; j < k && !dup; j++) dup = load[(size_t)j] == load[(size_t)k];
            if (dup) continue;
            int64_t nl = load[(size_t)k] + w[i];
            if (std::max(cur_max, nl) >= best) continue;       // prune by the incumbent
            load[(size_t)k] = nl;
            cur[i] = k;
            dfs(i + 1, std::max(cur_max, nl), lower);
            load[(size_t)k] = nl - w[i];
        }
    }
};
}  // namespace

void choose_senders(Plan *P) {
    const int n_src = P->A.n_dev;
    const int64_t e = P->elem_bytes;
    P->sender_bytes.assign((size_t)n_src, 0);
    if (P->flags & RS_LB_NAIVE) {
        for (Slice &S : P->slices) {
            S.sender = S.senders.front();
            P->sender_bytes[(size_t)S.sender] += S.elems * e;
        }
    } else {
        // Replica groups: every slice lies in exactly one source tile and the replica sets of
        // different tiles are disjoint, so Eq. 4 splits into one identical-machines problem per
        // distinct candidate set.
        std::map<std::vector<int>, std::vector<int>> groups;
        for (size_t i = 0; i < P->slices.size(); i++) groups[P->slices[i].senders].push_back((int)i);
        for (auto &g : groups) {
            const std::vector<int> &cand = g.first;
            std::vector<int> &ids = g.second;
            // descending T_i (= bytes, R7); ties by slice id (R9)
            std::stable_sort(ids.begin(), ids.end(), [&](int a, int b) {
                return P->slices[(size_t)a].elems > P->slices[(size_t)b].elems;
            });
            const int m = (int)cand.size();
            std::vector<int64_t> load((size_t)m, 0), w(ids.size());
            std::vector<int> assign(ids.size(), 0);
            int64_t total = 0;
            for (size_t t = 0; t < ids.size(); t++) {
                w[t] = P->slices[(size_t)ids[t]].elems * e;
                total += w[t];
                int k = (int)(std::min_element(load.begin(), load.end()) - load.begin());   // lightest, lowest id
                assign[t] = k;
                load[(size_t)k] += w[t];
            }
            int64_t greedy_max = *std::max_element(load.begin(), load.end());
            int64_t lower = std::max(w.empty() ? 0 : w[0], (total + m - 1) / m);
            if (m > 1 && greedy_max > lower && ids.size() <= 16) {
                ExactLB ex(w, m, greedy_max, assign);
                ex.dfs(0, 0, lower);
                assign = ex.best_assign;
            }
            for (size_t t = 0; t < ids.size(); t++) {
                Slice &S = P->slices[(size_t)ids[t]];
                S.sender = cand[(size_t)assign[t]];
                P->sender_bytes[(size_t)S.sender] += w[t];
            }
        }
    }
    P->max_sender_bytes = *std::max_element(P->sender_bytes.begin(), P->sender_bytes.end());
    P->used_src.assign((size_t)n_src, 0);
    for (const Slice &S : P->slices) P->used_src[(size_t)S.sender] = 1;
}

// ------------------------------------------------------------------ message layout (wire model)

// Message (s, r) = concatenation in ascending slice id of every slice with sender s and r in M_i,
// each dense row-major; messages ordered by (s, r) and laid back to back in the arena, each
// starting at a 256-byte boundary so a message is a valid stand-alone wire buffer.
rs_status build_messages(Plan *P) {
    std::map<std::pair<int, int>, std::vector<int>> groups;
    for (size_t i = 0; i < P->slices.size(); i++)
        for (int r : P->slices[i].receivers) groups[{P->slices[i].sender, r}].push_back((int)i);
    P->messages.clear();
    int64_t off = 0;
    for (auto &g : groups) {
        Message M;
        M.sender = g.first.first;
        M.receiver = g.first.second;
        M.offset = off;
        M.slice_ids = g.second;
        for (int i : M.slice_ids) {
            M.slice_off.push_back(off);
            off += P->slices[(size_t)i].elems * P->elem_bytes;
        }
        M.bytes = off - M.offset;
        off = (off + 255) / 256 * 256;
        P->messages.push_back(std::move(M));
    }
    P->arena_bytes = off;
    return RS_OK;
}

}  // namespace rs

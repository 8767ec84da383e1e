// Host symbolic phase: canonical Y_bus, index maps, minimum-degree ordering on the bus graph, static block
// fill pattern, elimination levels and the static multiply-subtract program.  See sable_symbolic.hpp.
#include "sable_symbolic.hpp"

#include <algorithm>
#include <queue>
#include <set>
#include <tuple>

namespace sable {

namespace {
struct YEntry { int32_t c; double g, b; };

// union of two sorted vectors minus two excluded values
void merge_excluding(const std::vector<int32_t>& a, const std::vector<int32_t>& b, int32_t x0, int32_t x1,
                     std::vector<int32_t>& out) {
    out.clear();
    size_t i = 0, j = 0;
    while (i < a.size() || j < b.size()) {
        int32_t v;
        if (j >= b.size() || (i < a.size() && a[i] < b[j])) v = a[i++];
        else if (i >= a.size() || b[j] < a[i]) v = b[j++];
        else { v = a[i]; ++i; ++j; }
        if (v != x0 && v != x1) out.push_back(v);
    }
}
}  // namespace

int build_template(int32_t n_bus, const int32_t* row_ptr, const int32_t* col_idx, const double* y_re,
                   const double* y_im, const uint8_t* bus_type, int32_t slack, Template& T, std::string& err) {
    if (n_bus < 2 || !row_ptr || !col_idx || !y_re || !y_im || !bus_type) { err = "null pointer or n_bus < 2"; return 1; }
    if (slack < 0 || slack >= n_bus) { err = "slack index out of range"; return 1; }
    if (row_ptr[0] != 0) { err = "row_ptr[0] != 0"; return 2; }
    int n_slack = 0;
    for (int i = 0; i < n_bus; ++i) {
        if (row_ptr[i + 1] < row_ptr[i]) { err = "row_ptr not monotone"; return 2; }
        if (bus_type[i] > 2) { err = "bus_type must be 0 (PQ), 1 (PV) or 2 (slack)"; return 2; }
        if (bus_type[i] == 2) ++n_slack;
    }
    if (n_slack != 1 || bus_type[slack] != 2) { err = "exactly one slack bus required and it must equal `slack`"; return 2; }

    // ---- 1. canonical Y: sorted columns, duplicates summed, diagonal present, pattern symmetrised ------------
    std::vector<std::vector<YEntry>> rows(n_bus);
    for (int i = 0; i < n_bus; ++i)
        for (int k = row_ptr[i]; k < row_ptr[i + 1]; ++k) {
            int c = col_idx[k];
            if (c < 0 || c >= n_bus) { err = "column index out of range"; return 2; }
            rows[i].push_back({c, y_re[k], y_im[k]});
        }
    auto canon = [&](std::vector<YEntry>& r) {
        std::stable_sort(r.begin(), r.end(), [](const YEntry& a, const YEntry& b) { return a.c < b.c; });
        size_t w = 0;
        for (size_t k = 0; k < r.size(); ++k) {
            if (w > 0 && r[w - 1].c == r[k].c) { r[w - 1].g += r[k].g; r[w - 1].b += r[k].b; }
            else r[w++] = r[k];
        }
        r.resize(w);
    };
    for (int i = 0; i < n_bus; ++i) { rows[i].push_back({i, 0.0, 0.0}); canon(rows[i]); }
    {
        std::vector<std::vector<int32_t>> missing(n_bus);
        for (int i = 0; i < n_bus; ++i)
            for (const YEntry& e : rows[i]) {
                const auto& rj = rows[e.c];
                auto it = std::lower_bound(rj.begin(), rj.end(), i, [](const YEntry& a, int v) { return a.c < v; });
                if (it == rj.end() || it->c != i) missing[e.c].push_back(i);
            }
        for (int i = 0; i < n_bus; ++i)
            if (!missing[i].empty()) { for (int c : missing[i]) rows[i].push_back({c, 0.0, 0.0}); canon(rows[i]); }
    }
    T.nnz_y = 0;
    for (int i = 0; i < n_bus; ++i) T.nnz_y += (int64_t)rows[i].size();
    T.fptr.assign(n_bus + 1, 0); T.fcol.clear(); T.fg.clear(); T.fb.clear();
    for (int i = 0; i < n_bus; ++i) {
        for (const YEntry& e : rows[i]) { T.fcol.push_back(e.c); T.fg.push_back(e.g); T.fb.push_back(e.b); }
        T.fptr[i + 1] = (int32_t)T.fcol.size();
    }

    // ---- 2. every bus must reach the slack (otherwise J1 is structurally singular) ---------------------------
    {
        std::vector<char> seen(n_bus, 0);
        std::queue<int> q; q.push(slack); seen[slack] = 1; int cnt = 1;
        while (!q.empty()) { int v = q.front(); q.pop(); for (const YEntry& e : rows[v]) if (!seen[e.c]) { seen[e.c] = 1; ++cnt; q.push(e.c); } }
        if (cnt != n_bus) { err = "network is not connected to the slack bus"; return 2; }
    }

    // ---- 3. minimum degree on the non-slack bus graph, ties broken towards the shallowest elimination level ---
    const int N = n_bus - 1;
    std::vector<int32_t> loc(n_bus, -1), bus_of(N);           // provisional numbering: non-slack buses ascending
    { int p = 0; for (int i = 0; i < n_bus; ++i) if (i != slack) { loc[i] = p; bus_of[p] = i; ++p; } }
    std::vector<std::vector<int32_t>> adj(N);
    for (int p = 0; p < N; ++p)
        for (const YEntry& e : rows[bus_of[p]]) if (e.c != slack && e.c != bus_of[p]) adj[p].push_back(loc[e.c]);
    for (int p = 0; p < N; ++p) std::sort(adj[p].begin(), adj[p].end());
    std::vector<int32_t> lvl(N, 0), elim_pos(N, -1);
    std::vector<std::vector<int32_t>> upper(N);                // upper[v] = neighbours of v at its elimination (all eliminated later)
    {
        using Key = std::tuple<int32_t, int32_t, int32_t>;      // (degree, level-if-eliminated-now, id)
        std::set<Key> pq;
        for (int p = 0; p < N; ++p) pq.insert(Key((int32_t)adj[p].size(), 0, p));
        std::vector<int32_t> tmp;
        for (int step = 0; step < N; ++step) {
            Key kmin = *pq.begin(); pq.erase(pq.begin());
            int v = std::get<2>(kmin);
            elim_pos[v] = step;
            upper[v] = adj[v];
            for (int32_t u : upper[v]) {
                pq.erase(Key((int32_t)adj[u].size(), lvl[u], u));
                merge_excluding(adj[u], upper[v], u, v, tmp);
                adj[u].swap(tmp);
                lvl[u] = std::max(lvl[u], lvl[v] + 1);
                pq.insert(Key((int32_t)adj[u].size(), lvl[u], u));
            }
            std::vector<int32_t>().swap(adj[v]);
        }
    }

    // ---- 4. final order: by level, then by elimination step (any topological order of the elimination tree
    //         gives the same fill); positions, maps, levels --------------------------------------------------
    //         Within a level the order is free: nodes are placed next to the nodes that share their first later
    //         neighbour (levels are placed from the top down; key = position of the earliest-placed later neighbour), so
    //         that the leaves of one hub are contiguous -- the hub's Y row, its diagonal target's item list and the pairs
    //         those leaves own are then contiguous in memory and the lanes that walk them read neighbouring words.
    std::vector<int32_t> order(N);
    {
        int nlev = 0;
        for (int p = 0; p < N; ++p) nlev = std::max(nlev, lvl[p] + 1);
        std::vector<std::vector<int32_t>> by_level(nlev);
        for (int p = 0; p < N; ++p) by_level[lvl[p]].push_back(p);
        std::vector<int32_t> level_start(nlev + 1, 0), rank(N, 0);          // rank: position within the level
        for (int l = 0; l < nlev; ++l) level_start[l + 1] = level_start[l] + (int32_t)by_level[l].size();
        for (int l = nlev - 1; l >= 0; --l) {
            std::vector<int32_t>& v = by_level[l];
            std::vector<int64_t> key(N, 0);
            for (int32_t p : v) {
                int64_t k = (int64_t)N;                                    // nodes of the top level: elimination order
                for (int32_t u : upper[p]) k = std::min<int64_t>(k, (int64_t)level_start[lvl[u]] + rank[u]);
                key[p] = k;
            }
            std::stable_sort(v.begin(), v.end(), [&](int a, int b) { return key[a] != key[b] ? key[a] < key[b] : elim_pos[a] < elim_pos[b]; });
            for (size_t i = 0; i < v.size(); ++i) rank[v[i]] = (int32_t)i;
        }
        int q = 0;
        for (int l = 0; l < nlev; ++l) for (int32_t p : by_level[l]) order[q++] = p;
    }
    std::vector<int32_t> pos(N);
    for (int q = 0; q < N; ++q) pos[order[q]] = q;
    T.n_bus = n_bus; T.slack = slack; T.n_node = N;
    T.node_bus.resize(N); T.bus_node.assign(n_bus, N); T.node_pq.resize(N); T.node_level.resize(N);
    T.n_pq = T.n_pv = 0;
    for (int q = 0; q < N; ++q) {
        int bus = bus_of[order[q]];
        T.node_bus[q] = bus; T.bus_node[bus] = q;
        T.node_pq[q] = bus_type[bus] == 0 ? 1 : 0;
        (T.node_pq[q] ? T.n_pq : T.n_pv)++;
        T.node_level[q] = lvl[order[q]];
    }
    T.n_level = N ? T.node_level[N - 1] + 1 : 0;
    T.level_ptr.assign(T.n_level + 1, 0);
    for (int q = 0; q < N; ++q) T.level_ptr[T.node_level[q] + 1]++;
    for (int l = 0; l < T.n_level; ++l) T.level_ptr[l + 1] += T.level_ptr[l];

    // ---- 5. Y rows in node order ------------------------------------------------------------------------------
    T.yptr.assign(N + 1, 0); T.ycol.clear(); T.yg.clear(); T.yb.clear(); T.ydiag.assign(N, -1);
    for (int q = 0; q < N; ++q) {
        std::vector<YEntry> r = rows[T.node_bus[q]];
        for (YEntry& e : r) e.c = T.bus_node[e.c];
        std::sort(r.begin(), r.end(), [](const YEntry& a, const YEntry& b) { return a.c < b.c; });
        for (const YEntry& e : r) {
            if (e.c == q) T.ydiag[q] = (int32_t)T.ycol.size();
            T.ycol.push_back(e.c); T.yg.push_back(e.g); T.yb.push_back(e.b);
        }
        T.yptr[q + 1] = (int32_t)T.ycol.size();
    }
    auto yslot = [&](int m, int j) -> int32_t {
        auto b = T.ycol.begin() + T.yptr[m], e = T.ycol.begin() + T.yptr[m + 1];
        auto it = std::lower_bound(b, e, j);
        return (it != e && *it == j) ? (int32_t)(it - T.ycol.begin()) : -1;
    };

    // ---- 6. pairs ----------------------------------------------------------------------------------------------
    T.pair_ptr.assign(N + 1, 0); T.pair_row.clear(); T.pair_col.clear(); T.pair_yu.clear(); T.pair_yl.clear();
    T.n_pair_j = 0; T.max_pairs_node = 0;
    for (int q = 0; q < N; ++q) {
        std::vector<int32_t> up;
        for (int32_t u : upper[order[q]]) up.push_back(pos[u]);
        std::sort(up.begin(), up.end());
        for (int32_t j : up) {
            if (j <= q) { err = "internal: elimination order violated"; return 2; }
            T.pair_row.push_back(q); T.pair_col.push_back(j);
            int32_t su = yslot(q, j), sl = yslot(j, q);
            T.pair_yu.push_back(su); T.pair_yl.push_back(sl);
            if (su >= 0) T.n_pair_j++;
        }
        T.pair_ptr[q + 1] = (int32_t)T.pair_col.size();
        T.max_pairs_node = std::max<int32_t>(T.max_pairs_node, (int32_t)up.size());
    }
    const int32_t P = (int32_t)T.pair_col.size();
    auto pair_id = [&](int m, int j) -> int32_t {
        auto b = T.pair_col.begin() + T.pair_ptr[m], e = T.pair_col.begin() + T.pair_ptr[m + 1];
        auto it = std::lower_bound(b, e, j);
        return (it != e && *it == j) ? (int32_t)(it - T.pair_col.begin()) : -1;
    };

    // ---- 7. term lists (two passes: count, fill), terms of a target in ascending k ----------------------------
    T.term_ptr.assign(P + 1, 0); T.dterm_ptr.assign(N + 1, 0);
    for (int k = 0; k < N; ++k) {
        int32_t lo = T.pair_ptr[k], hi = T.pair_ptr[k + 1];
        for (int32_t a = lo; a < hi; ++a) {
            T.dterm_ptr[T.pair_col[a] + 1]++;
            for (int32_t b = a + 1; b < hi; ++b) {
                int32_t t = pair_id(T.pair_col[a], T.pair_col[b]);
                if (t < 0) { err = "internal: fill pattern not closed"; return 2; }
                T.term_ptr[t + 1]++;
            }
        }
    }
    for (int p = 0; p < P; ++p) T.term_ptr[p + 1] += T.term_ptr[p];
    for (int q = 0; q < N; ++q) T.dterm_ptr[q + 1] += T.dterm_ptr[q];
    T.term_a.assign(T.term_ptr[P], 0); T.term_b.assign(T.term_ptr[P], 0); T.dterm.assign(T.dterm_ptr[N], 0);
    {
        std::vector<int32_t> tfill(T.term_ptr.begin(), T.term_ptr.end() - 1), dfill(T.dterm_ptr.begin(), T.dterm_ptr.end() - 1);
        for (int k = 0; k < N; ++k) {
            int32_t lo = T.pair_ptr[k], hi = T.pair_ptr[k + 1];
            for (int32_t a = lo; a < hi; ++a) {
                T.dterm[dfill[T.pair_col[a]]++] = a;
                for (int32_t b = a + 1; b < hi; ++b) {
                    int32_t t = pair_id(T.pair_col[a], T.pair_col[b]);
                    T.term_a[tfill[t]] = a; T.term_b[tfill[t]] = b; tfill[t]++;
                }
            }
        }
    }

    // ---- 8. statistics on the unpadded scalar pattern -----------------------------------------------------------
    auto w = [&](int q) -> int64_t { return T.node_pq[q] ? 2 : 1; };
    T.nnz_j = T.nnz_lu = T.lu_flops = 0;
    for (int q = 0; q < N; ++q) { T.nnz_j += w(q) * w(q); T.nnz_lu += w(q) * w(q); }
    for (int p = 0; p < P; ++p) {
        int64_t blk = 2 * w(T.pair_row[p]) * w(T.pair_col[p]);
        T.nnz_lu += blk;
        if (T.pair_yu[p] >= 0) T.nnz_j += blk;
    }
    T.max_terms_pair = T.max_terms_diag = 0;
    for (int p = 0; p < P; ++p) {
        int32_t nt = T.term_ptr[p + 1] - T.term_ptr[p];
        T.max_terms_pair = std::max(T.max_terms_pair, nt);
        int64_t wm = w(T.pair_row[p]), wj = w(T.pair_col[p]);
        for (int32_t t = T.term_ptr[p]; t < T.term_ptr[p + 1]; ++t) T.lu_flops += 2 * 2 * wm * w(T.pair_row[T.term_a[t]]) * wj;
        T.lu_flops += 2 * wj * wm * wm;                         // L(j,m) = T_L D_m^-1
    }
    for (int q = 0; q < N; ++q) {
        int32_t nt = T.dterm_ptr[q + 1] - T.dterm_ptr[q];
        T.max_terms_diag = std::max(T.max_terms_diag, nt);
        for (int32_t t = T.dterm_ptr[q]; t < T.dterm_ptr[q + 1]; ++t) T.lu_flops += 2 * w(q) * w(T.pair_row[T.dterm[t]]) * w(q);
    }
    return 0;
}

}  // namespace sable

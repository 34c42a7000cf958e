// fv_mask.cu -- host-side builder of the paper's attention mask: the ordered Markov boundary of every
// vertex of the coupling graph (Sec. IV.A.1, Eq. 12-13, Eq. S1).
//
// boundary(i) = past vertices j < i adjacent to i, or joined to i by a path whose intermediate vertices
// are all in the future (> i).  Instead of one graph search per vertex this sweeps i = n-1 .. 0 once and
// keeps the connected components of the future subgraph {i+1 .. n-1} in a union-find; every component
// carries the sorted set of its not-yet-future neighbours.  Inserting vertex i joins i with every future
// component it touches (their sets are merged small into large, i itself is dropped from the result):
// the merged set IS boundary(i).  O((n + |E|) log^2 n) set operations plus the output.
#include <algorithm>
#include <set>
#include <string>
#include <utility>
#include <vector>

#include "fv_internal.h"

int fv_markov_rows(int32_t n, int64_t n_edges, const int32_t* edge_a, const int32_t* edge_b,
                   std::vector<std::vector<int32_t>>& rows, std::string& err) {
    rows.assign((size_t)n, {});
    // adjacency, CSR
    std::vector<int64_t> ptr((size_t)n + 1, 0);
    for (int64_t e = 0; e < n_edges; ++e) {
        const int32_t a = edge_a[e], b = edge_b[e];
        if (a < 0 || b < 0 || a >= n || b >= n || a == b) {
            err = "edge " + std::to_string(e) + " = (" + std::to_string(a) + ", " + std::to_string(b) + ") is out of range or a self loop";
            return -1;
        }
        ++ptr[a + 1];
        ++ptr[b + 1];
    }
    for (int32_t v = 0; v < n; ++v) ptr[v + 1] += ptr[v];
    std::vector<int32_t> adj((size_t)ptr[n]);
    {
        std::vector<int64_t> fill(ptr.begin(), ptr.end() - 1);
        for (int64_t e = 0; e < n_edges; ++e) {
            adj[fill[edge_a[e]]++] = edge_b[e];
            adj[fill[edge_b[e]]++] = edge_a[e];
        }
    }
    std::vector<int32_t> parent((size_t)n);
    std::vector<std::set<int32_t>> open((size_t)n);     // per component root: neighbours that are not future yet
    auto find = [&](int32_t v) {
        int32_t r = v;
        while (parent[r] != r) r = parent[r];
        while (parent[v] != r) {
            const int32_t nx = parent[v];
            parent[v] = r;
            v = nx;
        }
        return r;
    };
    for (int32_t i = n - 1; i >= 0; --i) {
        parent[i] = i;
        std::set<int32_t>& mine = open[i];
        for (int64_t e = ptr[i]; e < ptr[i + 1]; ++e)
            if (adj[e] < i) mine.insert(adj[e]);
        for (int64_t e = ptr[i]; e < ptr[i + 1]; ++e) {
            if (adj[e] < i) continue;
            const int32_t r = find(adj[e]);
            if (r == i) continue;
            std::set<int32_t>& other = open[r];
            if (other.size() > mine.size()) mine.swap(other);
            mine.insert(other.begin(), other.end());
            std::set<int32_t>().swap(other);
            parent[r] = i;
        }
        mine.erase(i);
        rows[i].assign(mine.begin(), mine.end());
    }
    return 0;
}

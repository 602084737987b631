// cg_rcm.cpp -- reverse Cuthill-McKee renumbering of a CSR pattern, on the host (set-up work of
// cg_reorder, include/cg.h).  Nothing of the CG arithmetic lives here: the routine only decides in
// which order the rows are numbered, so that the entries of p a warp gathers lie close together
// (the matrix comes from a FEM model, whose node numbering is whatever the mesh
// generator produced; config 3 of BASELINE.json mimics that with a random permutation).
//
// Cuthill & McKee 1969 as every textbook states it: breadth-first search from a node of small degree
// at the far end of the graph (found by repeated searches: George & Liu's pseudo-peripheral node),
// the unvisited neighbours of a node appended in order of increasing degree (ties: by index, which
// makes the result a pure function of the pattern), every connected component in turn, and the
// whole order reversed at the end.
#include <algorithm>
#include <cstdint>
#include <new>
#include <vector>

#include "../../include/cg.h"

namespace {

struct Graph {
    int64_t n;
    const int32_t* rp;
    const int32_t* ci;
    int degree(int v) const { return rp[v + 1] - rp[v]; }
};

// Breadth-first search from s over nodes whose mark is `fresh`; visited nodes get `stamp`.  Fills
// `order` (visit order) and returns the index in `order` where the last level starts.
size_t bfs_levels(const Graph& g, int s, std::vector<int>& mark, int fresh, int stamp, std::vector<int>& order) {
    order.clear();
    order.push_back(s);
    mark[s] = stamp;
    size_t level_begin = 0, level_end = 1, last_begin = 0;
    while (level_begin < level_end) {
        last_begin = level_begin;
        for (size_t q = level_begin; q < level_end; ++q) {
            const int v = order[q];
            for (int e = g.rp[v]; e < g.rp[v + 1]; ++e) {
                const int w = g.ci[e];
                if (w < 0 || w >= g.n || mark[w] != fresh) continue;
                mark[w] = stamp;
                order.push_back(w);
            }
        }
        level_begin = level_end;
        level_end = order.size();
    }
    return last_begin;
}

}  // namespace

extern "C" int cg_rcm_host(int64_t n, const int32_t* h_rowptr, const int32_t* h_colind, int32_t* h_perm) {
    if (n <= 0 || n >= (1LL << 31) - 64 || !h_rowptr || !h_perm) return CG_EINVAL;
    if (h_rowptr[0] != 0) return CG_EINVAL;
    for (int64_t i = 0; i < n; ++i)
        if (h_rowptr[i + 1] < h_rowptr[i]) return CG_EINVAL;
    if (h_rowptr[n] > 0 && !h_colind) return CG_EINVAL;
    try {
        const Graph g{n, h_rowptr, h_colind};
        // mark: 0 = not numbered yet; odd / even stamps of the trial searches are reset to 0 afterwards
        std::vector<int> mark((size_t)n, 0), trial, comp, nb;
        std::vector<int> by_degree((size_t)n);
        for (int64_t i = 0; i < n; ++i) by_degree[(size_t)i] = (int)i;
        std::stable_sort(by_degree.begin(), by_degree.end(), [&](int a, int b) { return g.degree(a) < g.degree(b); });
        std::vector<int> cm;
        cm.reserve((size_t)n);
        for (int64_t k = 0; k < n; ++k) {
            int s = by_degree[(size_t)k];
            if (mark[s] != 0) continue;
            // pseudo-peripheral start: search, move to a node of smallest degree in the last level, repeat
            // while the search gets deeper (at most a few rounds)
            size_t depth_prev = 0;
            for (int round = 0; round < 8; ++round) {
                const size_t last = bfs_levels(g, s, mark, 0, 1, trial);
                for (int v : trial) mark[v] = 0;
                // depth = number of levels is not kept by bfs_levels; the size of what precedes the last level
                // grows with it on a connected component, which is all the stopping rule needs
                int best = trial[last];
                for (size_t q = last; q < trial.size(); ++q)
                    if (g.degree(trial[q]) < g.degree(best) || (g.degree(trial[q]) == g.degree(best) && trial[q] < best)) best = trial[q];
                if (round > 0 && last <= depth_prev) break;
                depth_prev = last;
                if (best == s) break;
                s = best;
            }
            // Cuthill-McKee numbering of this component
            const size_t begin = cm.size();
            cm.push_back(s);
            mark[s] = 2;
            for (size_t q = begin; q < cm.size(); ++q) {
                const int v = cm[q];
                nb.clear();
                for (int e = g.rp[v]; e < g.rp[v + 1]; ++e) {
                    const int w = g.ci[e];
                    if (w < 0 || w >= n || mark[w] != 0) continue;
                    mark[w] = 2;
                    nb.push_back(w);
                }
                std::sort(nb.begin(), nb.end(), [&](int a, int b) {
                    const int da = g.degree(a), db = g.degree(b);
                    return da != db ? da < db : a < b;
                });
                cm.insert(cm.end(), nb.begin(), nb.end());
            }
        }
        if ((int64_t)cm.size() != n) return CG_EINVAL;
        for (int64_t i = 0; i < n; ++i) h_perm[i] = cm[(size_t)(n - 1 - i)];      // reversed: new number i <- old row
    } catch (const std::bad_alloc&) {
        return CG_ENOMEM;
    }
    return CG_OK;
}

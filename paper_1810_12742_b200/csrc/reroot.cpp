// f2, tree re-rooting (section 6 "Balance the dependency tree so that the depth of the tree is
// minimized"): host, setup time, O(N).  See include/hines.h (hines_reroot) for the interface and DESIGN.md readings
// R1-R3.  The compartment that minimises the depth is a centre of the tree: the middle of a longest path, found by two
// breadth-first searches (farthest compartment from anywhere, farthest from that one).  A tree has one centre (even
// diameter) or two neighbouring ones (odd): of two the larger index is taken (R2).  The renumbering walks the branches
// of the re-rooted tree breadth first (R3): a branch runs while compartments have exactly one child, its child
// branches are the children of its last compartment in ascending old index; new indices are handed out in the order
// of that walk, which is the order by (branch number, distance to the root) the paper asks for.
#include <algorithm>
#include <cstdint>
#include <new>
#include <string>
#include <vector>

#include "plan_internal.h"

namespace {

struct Scratch {
    std::vector<int32_t> cstart, clist, dist, from, queue, np_old, nstart, nlist, newidx;
};

// breadth-first search over the undirected tree (old parent + old children lists); returns the last compartment reached
// (one of the farthest); dist / from are filled for every compartment
int32_t bfs(int32_t n, const int32_t* parent, const Scratch& S, int32_t src, std::vector<int32_t>& dist, std::vector<int32_t>& from,
            std::vector<int32_t>& queue)
{
    std::fill(dist.begin(), dist.begin() + n, -1);
    int32_t head = 0, tail = 0;
    dist[src] = 0; from[src] = -1; queue[tail++] = src;
    while (head < tail) {
        const int32_t v = queue[head++];
        const int32_t p = parent[v];
        if (p >= 0 && dist[p] < 0) { dist[p] = dist[v] + 1; from[p] = v; queue[tail++] = p; }
        for (int32_t k = S.cstart[v]; k < S.cstart[v + 1]; ++k) {
            const int32_t w = S.clist[k];
            if (dist[w] < 0) { dist[w] = dist[v] + 1; from[w] = v; queue[tail++] = w; }
        }
    }
    return queue[tail - 1];
}

}  // namespace

extern "C" hines_status_t hines_reroot(const int32_t* parent, const int64_t* cell_offsets, int64_t ncells,
                                       int32_t* new_parent, int64_t* perm, int64_t* u_src, int32_t* root,
                                       int32_t* depth_before, int32_t* depth_after)
{
    using hines::set_error;
    if (!parent || !cell_offsets || !new_parent || !perm || !u_src) { set_error("hines_reroot: null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (ncells <= 0) { set_error("hines_reroot: ncells must be positive"); return HINES_ERR_INVALID_ARG; }
    if (cell_offsets[0] != 0) { set_error("cell_offsets[0] must be 0"); return HINES_ERR_BAD_TOPOLOGY; }
    try {
        Scratch S;
        for (int64_t c = 0; c < ncells; ++c) {
            const int64_t lo = cell_offsets[c], hi = cell_offsets[c + 1];
            if (hi <= lo || hi - lo >= ((int64_t)1 << 31)) {
                set_error("cell_offsets not strictly increasing at cell " + std::to_string(c));
                return HINES_ERR_BAD_TOPOLOGY;
            }
            const int32_t n = (int32_t)(hi - lo);
            const int32_t* p = parent + lo;
            if (p[0] != -1) { set_error("parent[first compartment of cell " + std::to_string(c) + "] must be -1"); return HINES_ERR_BAD_TOPOLOGY; }
            for (int32_t i = 1; i < n; ++i)
                if (p[i] < 0 || p[i] >= i) { set_error("parent out of range at compartment " + std::to_string(lo + i)); return HINES_ERR_BAD_TOPOLOGY; }
            for (auto* v : {&S.dist, &S.from, &S.queue, &S.np_old, &S.clist, &S.nlist, &S.newidx}) if ((int32_t)v->size() < n) v->resize(n);
            S.cstart.assign((size_t)n + 1, 0);
            S.nstart.assign((size_t)n + 1, 0);
            // children lists of the old tree (ascending by construction)
            for (int32_t i = 1; i < n; ++i) ++S.cstart[p[i] + 1];
            for (int32_t i = 0; i < n; ++i) S.cstart[i + 1] += S.cstart[i];
            {
                std::vector<int32_t>& fill = S.newidx;                  // borrowed as the fill cursor
                std::copy(S.cstart.begin(), S.cstart.begin() + n, fill.begin());
                for (int32_t i = 1; i < n; ++i) S.clist[fill[p[i]]++] = i;
            }
            // R1: the depth as given, and a centre of the tree
            bfs(n, p, S, 0, S.dist, S.from, S.queue);
            int32_t dep0 = 0;
            for (int32_t i = 0; i < n; ++i) dep0 = std::max(dep0, S.dist[i]);
            const int32_t a = S.queue[n - 1];                          // a farthest compartment from the old root
            const int32_t b = bfs(n, p, S, a, S.dist, S.from, S.queue); // a farthest one from a: a..b is a longest path
            const int32_t diam = S.dist[b];
            int32_t v = b;
            for (int32_t s = 0; s < diam / 2; ++s) v = S.from[v];       // diam / 2 steps from b towards a
            int32_t centre = v;
            if (diam & 1) centre = std::max(v, S.from[v]);              // two centres: R2, the larger index
            const int32_t dep1 = (diam + 1) / 2;
            // the re-rooted tree: new parents (old indices) and children lists, ascending old index
            bfs(n, p, S, centre, S.dist, S.from, S.queue);
            for (int32_t i = 0; i < n; ++i) { S.np_old[i] = S.from[i]; if (S.from[i] >= 0) ++S.nstart[S.from[i] + 1]; }
            for (int32_t i = 0; i < n; ++i) S.nstart[i + 1] += S.nstart[i];
            {
                std::vector<int32_t>& fill = S.newidx;
                std::copy(S.nstart.begin(), S.nstart.begin() + n, fill.begin());
                for (int32_t i = 0; i < n; ++i) if (S.np_old[i] >= 0) S.nlist[fill[S.np_old[i]]++] = i;
            }
            // R3: branches breadth first; new indices in the order of the walk
            int32_t head = 0, tail = 0, next = 0;
            S.queue[tail++] = centre;
            while (head < tail) {
                int32_t w = S.queue[head++];
                for (;;) {
                    S.newidx[w] = next++;
                    if (S.nstart[w + 1] - S.nstart[w] != 1) break;
                    w = S.nlist[S.nstart[w]];
                }
                for (int32_t k = S.nstart[w]; k < S.nstart[w + 1]; ++k) S.queue[tail++] = S.nlist[k];
            }
            for (int32_t i = 0; i < n; ++i) {
                const int32_t k = S.newidx[i], q = S.np_old[i];
                perm[lo + k] = lo + i;
                new_parent[lo + k] = q < 0 ? -1 : S.newidx[q];
                // the coupling of the edge (i, q) sits at its child end in the OLD tree
                u_src[lo + k] = lo + (q < 0 ? i : (p[i] == q ? i : q));
            }
            if (root) root[c] = centre;
            if (depth_before) depth_before[c] = dep0;
            if (depth_after) depth_after[c] = dep1;
        }
    } catch (const std::bad_alloc&) {
        set_error("hines_reroot: out of host memory");
        return HINES_ERR_ALLOC;
    }
    return HINES_OK;
}

/*
 * RE-ROOTING ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * The paper's first work-balancing strategy (section 6), written out as the plain definition and
 * independently of paper_1810_12742_b200/csrc/reroot.cpp (which finds the centre of the tree by two breadth-first
 * searches; this one tries EVERY compartment as the root and measures the depth of the tree it gives):
 *
 *   "Balance the dependency tree so that the depth of the tree is minimized."
 *   "we take each neuron and create a tree where each compartment is connected to its neighboring compartments ...
 *    we have to find a new root node that minimizes the depth of the tree and permute all unknowns such that they
 *    form a new Hines matrix based on the new root node.  In the example, this would be the compartment with index 7.
 *    ... To preserve the tridiagonal submatrices, we have to ensure that compartments in a dendrite branch get
 *    continuous indices.  This can be achieved by numbering all branches breadth first and then sorting all
 *    compartments by branch index and distance to the root."
 *
 * Readings:
 *   R1  depth = the largest distance, in compartments, from the root to any compartment (the eccentricity of the
 *       root in the undirected tree).
 *   R2  several compartments can give the same minimal depth (a tree has one or two centres): the one with the LARGER
 *       old index is taken.  The paper does not say; its example names index 7, and for the tree the survey infers for
 *       the missing Figure 1.1 (five branches of five compartments, widths 1-2-2) the minimisers are {6, 7}.
 *   R3  "numbering all branches breadth first": a branch of the re-rooted tree starts at the root and at every
 *       compartment whose (new) parent has two or more children, and runs while compartments have exactly one child;
 *       the branches are numbered in breadth-first order of the branch tree, the children of a branch in ascending
 *       order of the OLD index of their first compartment.  New index = rank by (branch number, distance to the root).
 *
 * Outputs per cell (all cell-local): root = old index of the new root; perm[new] = old; new_parent[new] (-1 for the
 * root, < new otherwise); usrc[new] = old index whose u[] holds the coupling of the edge (new, new_parent[new]) --
 * the child end of that edge in the OLD tree -- and perm[0] for the root (u of a root is never used).
 * The re-rooted system is d'[k] = d[perm[k]], b'[k] = b[perm[k]], u'[k] = u[usrc[k]]; its solution is x'[k] = x[perm[k]].
 *
 * Pins (tests/test_oracle_reroot.py): closed forms (a path: its middle; a star: the hub; depth = ceil(diameter / 2)),
 * the 1-2-2 example (weak pin, see R2), invariants (perm is a permutation, new_parent[k] < k, branches are runs of
 * consecutive indices), and the re-rooted system solved by Listing 2 gives the permuted solution of the original.
 */
#include <stdint.h>
#include <stdlib.h>

/* distance of every compartment from r in the undirected tree given by parent[]; returns the largest */
static int32_t depths_from(int32_t n, const int32_t* parent, const int32_t* cstart, const int32_t* clist, int32_t r,
                           int32_t* dist, int32_t* queue)
{
    for (int32_t i = 0; i < n; ++i) dist[i] = -1;
    int32_t head = 0, tail = 0, far = 0;
    dist[r] = 0; queue[tail++] = r;
    while (head < tail) {
        const int32_t v = queue[head++];
        if (dist[v] > far) far = dist[v];
        if (parent[v] >= 0 && dist[parent[v]] < 0) { dist[parent[v]] = dist[v] + 1; queue[tail++] = parent[v]; }
        for (int32_t k = cstart[v]; k < cstart[v + 1]; ++k)
            if (dist[clist[k]] < 0) { dist[clist[k]] = dist[v] + 1; queue[tail++] = clist[k]; }
    }
    return far;
}

/* One cell.  Returns the depth of the re-rooted tree, or -1 on allocation failure. */
int32_t oracle_reroot_cell(int32_t n, const int32_t* parent, int32_t* root_out, int32_t* depth_before,
                           int32_t* perm, int32_t* new_parent, int32_t* usrc)
{
    int32_t* cstart = (int32_t*)calloc((size_t)n + 2, sizeof(int32_t));
    int32_t* clist = (int32_t*)calloc((size_t)(n > 0 ? n : 1), sizeof(int32_t));
    int32_t* dist = (int32_t*)malloc(sizeof(int32_t) * (size_t)n);
    int32_t* queue = (int32_t*)malloc(sizeof(int32_t) * (size_t)n);
    int32_t* np_old = (int32_t*)malloc(sizeof(int32_t) * (size_t)n);     /* new parent, in old indices */
    int32_t* nchild = (int32_t*)calloc((size_t)n, sizeof(int32_t));
    int32_t* branch = (int32_t*)malloc(sizeof(int32_t) * (size_t)n);     /* branch number of every compartment */
    int32_t* newidx = (int32_t*)malloc(sizeof(int32_t) * (size_t)n);
    if (!cstart || !clist || !dist || !queue || !np_old || !nchild || !branch || !newidx) return -1;
    /* children lists of the old tree, ascending */
    for (int32_t i = 1; i < n; ++i) cstart[parent[i] + 2]++;
    for (int32_t i = 0; i < n; ++i) cstart[i + 2] += cstart[i + 1];
    for (int32_t i = 1; i < n; ++i) clist[cstart[parent[i] + 1]++] = i;
    /* cstart[v] .. cstart[v+1] now delimit v's children */

    /* R1, R2: every compartment as the root */
    int32_t best = -1, best_depth = 0;
    for (int32_t r = 0; r < n; ++r) {
        const int32_t dep = depths_from(n, parent, cstart, clist, r, dist, queue);
        if (r == 0) *depth_before = dep;
        if (best < 0 || dep < best_depth || (dep == best_depth && r > best)) { best = r; best_depth = dep; }
    }
    *root_out = best;
    depths_from(n, parent, cstart, clist, best, dist, queue);

    /* the re-rooted tree: the new parent of v is its neighbour one step closer to the root */
    for (int32_t v = 0; v < n; ++v) {
        np_old[v] = -1;
        if (v == best) continue;
        if (parent[v] >= 0 && dist[parent[v]] == dist[v] - 1) np_old[v] = parent[v];
        for (int32_t k = cstart[v]; k < cstart[v + 1]; ++k)
            if (dist[clist[k]] == dist[v] - 1) np_old[v] = clist[k];
        nchild[np_old[v]]++;
    }
    /* R3: branches, numbered breadth first over the branch tree.  A queue of branch heads; a branch is followed
     * down while its compartments have exactly one child; the heads of its child branches are the children of its
     * last compartment, taken in ascending old index. */
    int32_t nb = 0, head = 0, tail = 0;
    queue[tail++] = best;
    while (head < tail) {
        int32_t v = queue[head++];
        const int32_t bid = nb++;
        for (;;) {
            branch[v] = bid;
            if (nchild[v] != 1) break;
            int32_t next = -1;
            for (int32_t w = 0; w < n; ++w) if (np_old[w] == v) next = w;       /* plainly: scan for the only child */
            v = next;
        }
        for (int32_t w = 0; w < n; ++w) if (np_old[w] == v) queue[tail++] = w;   /* ascending old index */
    }
    /* new index = rank by (branch number, distance to the root): plain selection, O(n^2) */
    for (int32_t v = 0; v < n; ++v) {
        int32_t rank = 0;
        for (int32_t w = 0; w < n; ++w)
            if (branch[w] < branch[v] || (branch[w] == branch[v] && dist[w] < dist[v])) ++rank;
        newidx[v] = rank;
    }
    for (int32_t v = 0; v < n; ++v) {
        const int32_t k = newidx[v];
        perm[k] = v;
        new_parent[k] = np_old[v] < 0 ? -1 : newidx[np_old[v]];
        /* the edge (v, np_old[v]) of the old tree: its coupling sits at whichever end was the child there */
        usrc[k] = np_old[v] < 0 ? v : (parent[v] == np_old[v] ? v : np_old[v]);
    }
    free(cstart); free(clist); free(dist); free(queue); free(np_old); free(nchild); free(branch); free(newidx);
    return best_depth;
}

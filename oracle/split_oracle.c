/*
 * SPLIT ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * The paper's branch splitting pass (section 6), written out as plainly as possible and
 * independently of paper_1810_12742_b200/csrc/plan.cpp (which walks frontier lists; this one rescans all
 * branches on every level):
 *
 *   "Currently the branch splitting is performed on a per level basis.  On each level we compute the average
 *    length of all dendritic branches on this level and cut all branches that are longer than average.  Then
 *    we proceed to the next level and repeat the splitting until we reach the lowest level of the tree.  ...
 *    cutting a branch at a specific level causes all child branches to move one level down."
 *   "Instead of one long branch, we now model it as two shorter branches that are attached to each other."
 *
 *   "On each level, we compute the average length of all branches on this level in all dendritic trees."
 *
 *
 * Reading F1: the average is taken over ALL cells of the batch; with integer lengths
 * "longer than average" means len > c, c = ceil(mean); the cut leaves a head of exactly c compartments on the
 * level (so that no piece on a level is longer than c) and the rest becomes ONE piece on the next level, which
 * may be cut again there; the branch's children follow its last piece.  Where the paper cuts is not stated;
 * cutting at c is the choice that makes "all pieces of a level <= ceil(mean)" hold.
 *
 * Inputs are the canonical tables of tables_oracle.c (branch lengths, parent branches, per cell).
 * Pins (tests/test_oracle_split.py): a hand-worked example (tests/golden/split_example.json), closed forms
 * (equal lengths: nothing is cut; one long branch among unit ones), and invariants (pieces tile the branch,
 * every piece of level L <= ceil(mean of level L), a child's first piece sits one level below its parent's last).
 */
#include <stdint.h>
#include <stdlib.h>

/* Returns the number of pieces, or -1.  piece_* arrays need capacity for the total number of compartments at
 * most (a piece has at least one compartment).  piece_branch[k] is the GLOBAL branch index of piece k; pieces
 * are emitted level by level, inside a level in global branch order.  level_sum / level_cnt (capacity: max
 * pieces) receive the per-level statistics; *nlevels the number of levels of the split tree. */
int64_t oracle_level_mean_split(int64_t ncells, const int64_t* cell_branch_offsets, const int32_t* branch_len,
                                const int32_t* branch_parent_branch /* cell-local, -1 root */,
                                int64_t* piece_branch, int32_t* piece_len, int32_t* piece_level,
                                int64_t* level_sum, int64_t* level_cnt, int64_t* nlevels)
{
    const int64_t nb = cell_branch_offsets[ncells];
    int32_t* rem = (int32_t*)malloc((size_t)nb * sizeof(int32_t));     /* compartments of the branch not yet in a piece */
    int64_t* lvl = (int64_t*)malloc((size_t)nb * sizeof(int64_t));     /* level of its next piece; -1: parent not finished */
    int64_t* gpar = (int64_t*)malloc((size_t)nb * sizeof(int64_t));    /* global parent branch */
    if (!rem || !lvl || !gpar) return -1;
    for (int64_t c = 0; c < ncells; ++c)
        for (int64_t j = cell_branch_offsets[c]; j < cell_branch_offsets[c + 1]; ++j) {
            rem[j] = branch_len[j];
            gpar[j] = branch_parent_branch[j] < 0 ? -1 : cell_branch_offsets[c] + branch_parent_branch[j];
            lvl[j] = gpar[j] < 0 ? 0 : -1;
        }
    int64_t np = 0, L = 0;
    for (;; ++L) {
        int64_t sum = 0, cnt = 0;
        for (int64_t j = 0; j < nb; ++j) if (lvl[j] == L && rem[j] > 0) { sum += rem[j]; cnt++; }
        if (cnt == 0) break;
        const int64_t cut = (sum + cnt - 1) / cnt;                      /* ceil(mean) */
        level_sum[L] = sum; level_cnt[L] = cnt;
        for (int64_t j = 0; j < nb; ++j) {
            if (lvl[j] != L || rem[j] <= 0) continue;
            piece_branch[np] = j; piece_level[np] = (int32_t)L;
            if (rem[j] > cut) { piece_len[np] = (int32_t)cut; rem[j] -= (int32_t)cut; lvl[j] = L + 1; }
            else { piece_len[np] = rem[j]; rem[j] = 0; lvl[j] = -2; }   /* finished on level L */
            np++;
        }
        /* the children of a branch that finished on this level sit on the next one (a parent that finished on an
         * earlier level woke its children in that level's pass already) */
        for (int64_t j = 0; j < nb; ++j)
            if (lvl[j] == -1 && lvl[gpar[j]] == -2) lvl[j] = L + 1;
    }
    *nlevels = L;
    free(rem); free(lvl); free(gpar);
    return np;
}

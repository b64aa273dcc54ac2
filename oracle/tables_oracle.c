/*
 * TABLE ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Independent, serial re-derivation of the policy-free scheduler tables that
 * hines_plan_create must reproduce bit for bit: the branch dependency tree (PAPER.md:108,
 * "each node in this tree represents a submatrix"), its levels, the per-level
 * branch counts used for packing, the per-level lists sorted by size
 * and the one-parent-per-branch table.
 * Shares no code with paper_1810_12742_b200/.
 *
 * Readings:
 *   S4  compartment i starts a branch iff i is the root, or p[i] != i-1, or p[i] has >= 2
 *       children.  Branch ids are in order of start compartment.
 *   S5  level = depth from the root branch (root branch = level 0).
 *   S7  per-level order: length descending, ties by branch id ascending.
 *
 * All indices are cell-local (compartment index inside the cell, branch id inside the cell).
 * Pins (tests/test_oracle_tables.py): closed forms for configs 0, 1, 4, the
 * merge example p=[-1,0,1,2,3,4,5,4,7] -> starts [0,5,7], a pure-Python brute force on small
 * random trees.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* number of branches of the whole batch under rule S4; -1 on a malformed parent array */
int64_t oracle_tables_count(int64_t ncells, const int64_t* cell_offsets, const int32_t* parent)
{
    int64_t nb = 0;
    for (int64_t c = 0; c < ncells; ++c) {
        int64_t o = cell_offsets[c], n = cell_offsets[c + 1] - o;
        const int32_t* p = parent + o;
        if (n <= 0 || p[0] != -1) return -1;
        int32_t* nch = (int32_t*)calloc((size_t)n, sizeof(int32_t));
        for (int64_t i = 1; i < n; ++i) {
            if (p[i] < 0 || p[i] >= i) { free(nch); return -1; }
            nch[p[i]]++;
        }
        for (int64_t i = 0; i < n; ++i)
            if (i == 0 || p[i] != i - 1 || nch[p[i]] >= 2) nb++;
        free(nch);
    }
    return nb;
}

typedef struct { int32_t level, len, id; } sort_key_t;
static int cmp_key(const void* a, const void* b)
{
    const sort_key_t* x = (const sort_key_t*)a; const sort_key_t* y = (const sort_key_t*)b;
    if (x->level != y->level) return x->level < y->level ? -1 : 1;
    if (x->len != y->len) return x->len > y->len ? -1 : 1;      /* length descending (S7) */
    return x->id < y->id ? -1 : (x->id > y->id);
}

/*
 * Fill the tables.  Caller sizes (nb = oracle_tables_count):
 *   cell_branch_offsets int64[ncells+1]   branch_start/len/parent_comp/parent_branch/level int32[nb]
 *   cell_nlevels int32[ncells]            cell_level_offsets int64[ncells+1]
 *   level_count  int32[capacity >= sum nlevels]  (needed size returned through *n_level_count)
 *   level_list   int32[nb]                child_offsets int64[nb+1]   child_ids int32[nb-ncells]
 * Returns 0, or -1 if level_count capacity is too small (then *n_level_count has the need).
 */
int oracle_tables_build(int64_t ncells, const int64_t* cell_offsets, const int32_t* parent,
                        int64_t* cell_branch_offsets,
                        int32_t* branch_start, int32_t* branch_len, int32_t* branch_parent_comp,
                        int32_t* branch_parent_branch, int32_t* branch_level,
                        int32_t* cell_nlevels, int64_t* cell_level_offsets,
                        int32_t* level_count, int64_t level_count_capacity, int64_t* n_level_count,
                        int32_t* level_list, int64_t* child_offsets, int32_t* child_ids)
{
    int64_t nb = 0, nlc = 0, nchild_total = 0;
    int rc = 0;
    cell_branch_offsets[0] = 0; cell_level_offsets[0] = 0; child_offsets[0] = 0;
    for (int64_t c = 0; c < ncells; ++c) {
        int64_t o = cell_offsets[c], n = cell_offsets[c + 1] - o;
        const int32_t* p = parent + o;
        int32_t* nch = (int32_t*)calloc((size_t)n, sizeof(int32_t));
        int32_t* br_of = (int32_t*)malloc((size_t)n * sizeof(int32_t));   /* branch of compartment */
        for (int64_t i = 1; i < n; ++i) nch[p[i]]++;
        /* T1: branch starts and lengths (S4) */
        int64_t b0 = nb; int32_t k = -1;
        for (int64_t i = 0; i < n; ++i) {
            if (i == 0 || p[i] != i - 1 || nch[p[i]] >= 2) {
                ++k; branch_start[b0 + k] = (int32_t)i; branch_len[b0 + k] = 0;
            }
            br_of[i] = k; branch_len[b0 + k]++;
        }
        int32_t nbc = k + 1;
        if (nbc < 1) { free(nch); free(br_of); return -2; }   /* cannot happen: n >= 1 */
        /* T2-T4: parent compartment, parent branch, level (S5) */
        int32_t maxlev = 0;
        for (int32_t j = 0; j < nbc; ++j) {
            int32_t s = branch_start[b0 + j];
            if (s == 0) { branch_parent_comp[b0 + j] = -1; branch_parent_branch[b0 + j] = -1; branch_level[b0 + j] = 0; }
            else {
                int32_t pc = p[s], pb = br_of[pc];
                branch_parent_comp[b0 + j] = pc; branch_parent_branch[b0 + j] = pb;
                branch_level[b0 + j] = branch_level[b0 + pb] + 1;   /* pb < j because p[i] < i */
            }
            if (branch_level[b0 + j] > maxlev) maxlev = branch_level[b0 + j];
        }
        /* T5: per-level counts */
        int32_t nlev = maxlev + 1;
        cell_nlevels[c] = nlev;
        if (nlc + nlev > level_count_capacity) rc = -1;
        else {
            for (int32_t l = 0; l < nlev; ++l) level_count[nlc + l] = 0;
            for (int32_t j = 0; j < nbc; ++j) level_count[nlc + branch_level[b0 + j]]++;
        }
        nlc += nlev; cell_level_offsets[c + 1] = nlc;
        /* T6: per-level lists in S7 order */
        sort_key_t* keys = (sort_key_t*)malloc((size_t)nbc * sizeof(sort_key_t));
        for (int32_t j = 0; j < nbc; ++j) { keys[j].level = branch_level[b0 + j]; keys[j].len = branch_len[b0 + j]; keys[j].id = j; }
        qsort(keys, (size_t)nbc, sizeof(sort_key_t), cmp_key);
        for (int32_t j = 0; j < nbc; ++j) level_list[b0 + j] = keys[j].id;
        free(keys);
        /* T7: child lists (CSR over global branch index, ids cell-local ascending) */
        int32_t* cnt = (int32_t*)calloc((size_t)nbc, sizeof(int32_t));
        for (int32_t j = 1; j < nbc; ++j) cnt[branch_parent_branch[b0 + j]]++;
        for (int32_t j = 0; j < nbc; ++j) child_offsets[b0 + j + 1] = child_offsets[b0 + j] + cnt[j];
        memset(cnt, 0, (size_t)nbc * sizeof(int32_t));
        for (int32_t j = 1; j < nbc; ++j) {
            int32_t pb = branch_parent_branch[b0 + j];
            child_ids[child_offsets[b0 + pb] + cnt[pb]++] = j;
        }
        nchild_total += nbc - 1;
        free(cnt); free(nch); free(br_of);
        nb += nbc; cell_branch_offsets[c + 1] = nb;
    }
    (void)nchild_total;
    *n_level_count = nlc;
    return rc;
}

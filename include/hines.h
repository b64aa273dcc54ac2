/*
 * hines.h -- C ABI of the B200-native batched Hines solver (libhines_b200.so).
 *
 * The operation: every implicit-Euler time step of a compartmental neuron simulation solves, for
 * each cell, the symmetric strictly diagonally dominant system A x = b with
 *     A[i,i] = d[i],   A[i,p[i]] = A[p[i],i] = u[i]   (i >= 1),   p[i] < i,  p[root] = -1
 * (arXiv 1810.12742: PAPER.md:34-38 the discretisation, :44-50 the numbering and the statement of
 * the algorithm's inputs d, u, b, p, :78-100 Listing 2).  The solve is one backward elimination
 * from the leaves to the root and one forward substitution from the root to the leaves
 * (PAPER.md:50), for many independent cells at once.  The work distribution is
 * computed once at setup and reused every step.
 *
 * Conventions
 *   - "HOST" / "DEVICE" says where a pointer must live.  Device pointers must be 16-byte aligned.
 *   - Cells are concatenated; cell c owns compartments [cell_offsets[c], cell_offsets[c+1]).
 *     parent[] holds CELL-LOCAL indices (so identical morphologies have identical parent arrays).
 *   - The plan copies what it needs: parent / cell_offsets may be freed after hines_plan_create.
 *   - d, u, b are never written.  x may be exactly b (in place) or must not overlap d, u, b.
 *   - u[root] is never read in a way that can reach the result.
 *   - hines_solve only enqueues work on `stream` and never synchronises; it returns launch
 *     errors only.  One solve in flight per plan (the plan owns one workspace).
 *   - No C++ exception crosses this boundary.  Every function returns a status; details of the
 *     last failure on the calling thread are available from hines_last_error().
 *   - There is no CPU fallback: without a CUDA device the solve entry points return
 *     HINES_ERR_CUDA.  (hines_plan_create itself is host-only work and succeeds without a
 *     device, so the scheduler tables can be inspected anywhere; device tables are uploaded by
 *     the first solve or by hines_plan_upload.)
 */
#ifndef HINES_B200_H
#define HINES_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hines_plan hines_plan_t;          /* opaque, owned by the library            */
typedef struct CUstream_st* hines_stream_t;      /* == cudaStream_t; NULL = default stream  */

typedef enum {
    HINES_OK = 0,
    HINES_ERR_INVALID_ARG = 1,     /* null pointer, bad size, misaligned device pointer, bad option      */
    HINES_ERR_BAD_TOPOLOGY = 2,    /* parent / cell_offsets do not describe a forest of rooted trees      */
    HINES_ERR_ALLOC = 3,           /* host or device allocation failed                                    */
    HINES_ERR_CUDA = 4,            /* no device, or a CUDA call / kernel launch failed                    */
    HINES_ERR_UNSUPPORTED = 5      /* valid request this build cannot serve                               */
} hines_status_t;

typedef enum { HINES_F64 = 0, HINES_F32 = 1 } hines_dtype_t;

/* policy_flags */
enum {
    HINES_POLICY_DEFAULT      = 0,
    HINES_POLICY_FORCE_STREAM = 1,   /* every cell through the streaming (global-memory) path           */
    HINES_POLICY_NO_GROUPING  = 2,   /* one cell per shared-memory work item (paper: >= 1 cell per block) */
    HINES_POLICY_INPUT_ORDER  = 4,   /* launch work items in input order, not heaviest first, and group only cells that are
                                        neighbours in the input ("greedy": cells are taken in the order given) */
    HINES_POLICY_SERIAL_CLASSES = 16, /* launch the size classes one after the other on the caller's stream instead
                                        of concurrently on plan-owned side streams (forked from / joined to it)  */
    HINES_POLICY_POW2_CLUSTERS = 32, /* cluster sizes 2, 4, 8, 16 only (default: any size up to cluster_max, the one
                                        whose blocks fill their shared-memory slot best)                     */
    HINES_POLICY_NO_CLUSTER   = 8,   /* never cut a cell into parts: a cell either fits one block's shared memory
                                        or goes to the streaming path                                     */
    HINES_POLICY_NO_PCR       = 256, /* unbranched cables: the reduced chains go through the level sweeps like every other tree,
                                        not through parallel cyclic reduction                                          */
    HINES_POLICY_FACTORED     = 512, /* f3: the plan also serves hines_factor / hines_solve_rhs (with a fixed time
                                        step only the right-hand side changes between steps): parts are sized for four
                                        staged arrays (three factors + b) instead of three, and own N x 3 factor values  */
    HINES_POLICY_NO_QUADS     = 1024, /* every segment gets two lanes (default: four lanes for segments with >= 24 interior
                                        compartments: half the dependent steps in P1 / P3)                         */
    HINES_POLICY_NO_PDL       = 2048, /* split items: the three launches strictly one after the other (default: programmatic
                                        dependent launch, a phase starts while the one before it still runs)        */
    HINES_POLICY_NO_SPLIT     = 64,  /* no split items: a cell that fits no cluster goes to the streaming path  */
    HINES_POLICY_SPLIT_LEVEL_MEAN = 128, /* f1: cut branches by the paper's own rule first (level by
                                        level from the root, over all cells of the batch, a branch longer than
                                        c = ceil(mean length on the level) is cut into a head of c compartments and
                                        a rest that moves, with the branch's children, one level down); every piece is
                                        then still bounded by max_segment (set max_segment = 1023 for the paper's rule
                                        alone).  Tables HINES_TABLE_SPLIT_* hold the pieces with or without the flag  */
    HINES_POLICY_SPLIT_BLOCK_MEAN = 4096 /* f4 ("Some intermediate packing of the matrices in a block can be used to
                                        compute more local heuristics, like per block averages"): the same cutting rule, but
                                        the mean of a level is taken over the cells of ONE block (work item) -- the cells
                                        the packing, done on the uncut branches, has put together -- instead of the whole
                                        batch.  HINES_TABLE_SPLIT_PIECE_* then hold these pieces (cells of the streaming path:
                                        uncut), HINES_TABLE_SPLIT_LEVEL_STAT is empty.  Ignored with SPLIT_LEVEL_MEAN        */
};

typedef struct {
    int32_t struct_size;            /* = sizeof(hines_options_t); lets the struct grow                     */
    int32_t threads_per_block;      /* 0 = default (per size class: one lane per segment of the widest work item,
                                       64..384, within the register file); else multiple of 32, <= 384      */
    int32_t smem_bytes_per_block;   /* 0 = default (227 KiB: sm_100 opt-in maximum); upper bound for the
                                       shared memory one resident work item may use                       */
    int32_t policy_flags;           /* HINES_POLICY_*                                                      */
    int32_t stream_threads;         /* 0 = default (128): block size of the streaming-path kernels         */
    int32_t group_smem_bytes;       /* 0 = default (56 KiB): small cells are grouped into work items up to
                                       this much shared memory ("fit as many matrices into one
                                       block as possible")                                                 */
    int32_t max_segment;            /* 0 = default (40 for a cell in a block of its own, 64 for a cell spread over a
                                       cluster), 2..1023: target segment length.  A branch of len compartments
                                       is cut into max(1, floor(len / max_segment + 0.4)) chained segments of equal
                                       length, made odd when there are several (their starts then fall on
                                       distinct shared-memory banks), so a segment is at most 1.4 x max_segment + 2
                                       long ("we split branches that are too long")               */
    int32_t cluster_max;            /* 0 = default (8), 1..16: largest thread-block cluster a cell may be spread
                                       over (more than 8 needs the non-portable cluster size)                  */
    int32_t chunk_smem_bytes;       /* 0 = default (117 KiB, half an SM's shared memory: two blocks per SM overlap each
                                       other's phases; measured optimum of configs 2 and 3, +2 % over 227 KiB): the
                                       size above which a cell is cut into the parts of a cluster; the parts aim at
                                       1/2, 1/3 or 1/4 of an SM's shared memory, whichever they fill best, but never
                                       more than this                                                              */
    int32_t split_smem_bytes;       /* 0 = default (113 KiB): shared memory of one sub-tree part of a split item
                                       (a cell beyond the largest cluster, run as three dependent launches)     */
} hines_options_t;

typedef struct {
    int64_t n;                  /* unknowns of the whole batch                                             */
    int64_t ncells;
    int64_t nbranches;          /* under the canonical branch rule (reading S4)                  */
    int32_t max_levels;         /* deepest dependency tree in the batch                                    */
    int32_t dtype;              /* hines_dtype_t                                                           */
    int64_t n_resident_items;   /* shared-memory work items (cell groups)                                  */
    int64_t n_resident_cells;
    int64_t n_resident_unknowns;
    int64_t n_stream_cells;     /* cells too large for shared memory -> streaming path                     */
    int64_t n_stream_unknowns;
    int64_t n_stream_branches;
    int64_t padded_lane_steps;  /* sum over 32-lane tiles of (longest lane of the tile * 32) in the segment
                                   sweeps (resident path) and the branch sweeps (streaming path)           */
    int64_t useful_lane_steps;  /* the same without idle lanes: interior compartments of all segments +
                                   compartments of streamed branches; ratio = lane efficiency              */
    int64_t workspace_bytes;    /* device memory the plan owns (tables + streaming workspace)              */
    int64_t bytes_min;          /* n*4*w + 4*nbranches: d,u,b read, x written, one parent per branch
                                   (PAPER.md:138); the roofline numerator                                  */
    int64_t bytes_literal;      /* n*(4*w + 4): one parent per compartment (Listing 2 as printed)          */
    int32_t breadth_first;      /* 1 if every cell's branches are numbered level by level    */
    int32_t n_classes;          /* size classes in use = resident kernel launches per solve                */
    int64_t n_cluster_cells;    /* cells spread over a thread-block cluster (counted in n_resident_* too)  */
    int64_t n_cluster_unknowns;
    int64_t n_parts;            /* parts (= blocks' worth of shared memory) of all on-chip items           */
    int64_t n_split_cells;      /* cells run as split items: three dependent launches (counted in n_resident_* too) */
    int64_t n_split_unknowns;
    int64_t n_exports;          /* sub-tree roots that hand their value to another part (cluster + split items)    */
    int64_t n_blocks;           /* blocks the resident launches start per solve (split sub-tree parts count twice) */
} hines_plan_info_t;

/* Canonical, policy-free tables (bit-exact against the table oracle); all indices cell-local.
 * Branch ids are in order of start compartment (readings S4, S5, S7). */
typedef enum {
    HINES_TABLE_CELL_BRANCH_OFFSETS  = 0,   /* int64[ncells+1]                                              */
    HINES_TABLE_BRANCH_START         = 1,   /* int32[nbranches]  first compartment  */
    HINES_TABLE_BRANCH_LEN           = 2,   /* int32[nbranches]  compartments in the branch  */
    HINES_TABLE_BRANCH_PARENT_COMP   = 3,   /* int32[nbranches]  p[start], -1 for the root branch (:138)    */
    HINES_TABLE_BRANCH_PARENT_BRANCH = 4,   /* int32[nbranches]  -1 for the root branch                     */
    HINES_TABLE_BRANCH_LEVEL         = 5,   /* int32[nbranches]  depth from the root branch  */
    HINES_TABLE_CELL_NLEVELS         = 6,   /* int32[ncells]                                                */
    HINES_TABLE_CELL_LEVEL_OFFSETS   = 7,   /* int64[ncells+1]   into LEVEL_COUNT                           */
    HINES_TABLE_LEVEL_COUNT          = 8,   /* int32[sum nlevels] branches per (cell, level) */
    HINES_TABLE_LEVEL_LIST           = 9,   /* int32[nbranches]  per cell: ids by (level, length desc, id)  */
    HINES_TABLE_CHILD_OFFSETS        = 10,  /* int64[nbranches+1] CSR over global branch index              */
    HINES_TABLE_CHILD_IDS            = 11,  /* int32[nbranches-ncells] ascending                            */
    /* Policy tables (depend on options; validity-checked in tests and executed
     * lane by lane on the CPU by tests/plan_interpreter.py).  A PART is what one block stages into its shared
     * memory: whole branches, as runs of consecutive compartments.  A work item is one part (a run of whole
     * cells), or one cell cut into a top part (the root region) and parts that are unions of complete
     * sub-trees (cluster item: one part per block of a thread-block cluster; split item: three launches).
     * A part's reduced forest has one node per segment (the segment's last compartment, the "separator");
     * node ids are part-local. */
    HINES_TABLE_CELL_ITEM            = 32,  /* int32[ncells]  on-chip work item of the cell, -1 = streaming path       */
    HINES_TABLE_ITEM_CELL_OFFSETS    = 33,  /* int64[nitems+1] into ITEM_CELLS                                           */
    HINES_TABLE_ITEM_CELLS           = 37,  /* int64[] cells of each item, ascending (a group of small cells need not be
                                               neighbours in the input: large cells in between get items of their own)  */
    HINES_TABLE_ITEM_CLASS           = 34,  /* int32[nitems]  size class                                              */
    HINES_TABLE_ITEM_LAUNCH_ORDER    = 35,  /* int32[nitems]  items in launch order, per class heaviest first         */
    HINES_TABLE_ITEM_KIND            = 36,  /* int32[nitems]  0 = one part (a run of whole cells in one block), 1 = one cell cut
                                               into the parts of a thread-block cluster, 2 = split item (three launches)      */
    HINES_TABLE_ITEM_XCH             = 44,  /* int32[nitems]  first slot of the item in the global exchange buffers (split items)  */
    HINES_TABLE_ITEM_PART_OFFSETS    = 46,  /* int64[nitems+1] into the part tables; part 0 of a multi-part item is its top part    */
    HINES_TABLE_PART_HEADER          = 47,  /* int32[32*nparts] the 128-byte device record of each part:
                                               [0,1] meta_off (int64), [2] meta_len, [3] run_off, [4] nrun, [5] tx_elems, [6] L,
                                               [7] n, [8] nnode, [9] nlevnode, [10] nlev, [11] rounds, [12] kp_off, [13] exp_off,
                                               [14] gh_off, [15] seg_off, [16] nexp, [17] nghost, [18] nseg_lanes, [19] xch_base,
                                               [20] xs0, [21] item, [22] rank, [23] flags, [24] ntoplev, [25] lowlev                */
    HINES_TABLE_PART_META            = 48,  /* int32[] per part one blob (meta_off, meta_len), every section padded to 4 ints:
                                               lb[nlev+1]   first node of each local level (level = depth in the cell - smallest
                                                            depth in the part; level nodes are numbered level by level, the children
                                                            of a node consecutive, sorted by parent);
                                               kp[2*nnode]  per node {kids, pnode}: kids = first child | (children << 20), -1 for a
                                                            ghost child (a stand-in, in part 0, for the root of a sub-tree held by
                                                            another part: only its hand-off slot is used); pnode = the node the forward
                                                            sweep reads: the parent, itself for a root / ghost, for an exported sub-tree
                                                            root the ghost parent (ids >= nlevnode) that receives the parent's x; bit 30 set
                                                            for a top node (an ancestor of a ghost child: swept after the exchange);
                                               exps[4*nexp] per exported root {node, ghost child in part 0 (cluster) or exchange slot
                                                            (split), parent node in part 0, ghost parent};
                                               ghosts[4*nghost] {ghost child, exchange slot, its parent node, 0};
                                               seg[4*nseg_lanes] groups of 32 lanes.  Four-lane groups (kind 3; long segments): lane k + 8 j is
                                                            quarter j of segment k: {staged index of its first compartment, steps | j<<12 |
                                                            3<<24 | 1<<26, node, node of the separator above (j = 0 only)}; the middle nodes
                                                            q1, q2, q3 sit right above quarters 1, 2, 3.  Two-lane groups: lanes 0-15 the A
                                                            halves, lanes 16-31 their B partners (lane ^ 16).  A: {a = staged index of the first
                                                            compartment, word, node, node of the separator above (-1 = none)}; B: {a+mt+1,
                                                            word, node, -1}; word = mt | mb<<12 | kind<<24 | hasq<<26 | delay<<27 (kind 0
                                                            padding, 1 A, 2 B; mt/mb = compartments A / B eliminate, both top-down; the
                                                            middle node q = a+mt exists iff hasq; separator b = a+mt+mb+hasq)            */
    HINES_TABLE_PART_RUNS            = 49,  /* int32[4*nruns] {global first compartment, length, staged index of it, 0}: the runs of
                                               consecutive compartments a part stages (run_off, nrun in its header)            */
    HINES_TABLE_CLASS_PHASE          = 52,  /* int32[n_classes] 0 = ordinary; split items: 1 = sub-tree parts, backward sweep + export,
                                               2 = top parts, 3 = sub-tree parts again: backward sweep, import, forward sweep      */
    HINES_TABLE_CLASS_FIRST          = 53,  /* int64[n_classes] into CLASS_PARTS                                                */
    HINES_TABLE_CLASS_COUNT          = 54,  /* int64[n_classes] blocks of the class                                             */
    HINES_TABLE_CLASS_PARTS          = 55,  /* int32[] part ids in launch order, class by class (the blocks of a cluster item consecutive,
                                               rank 0 first)                                                                    */
    HINES_TABLE_SPLIT_PIECE_OFFSETS  = 60,  /* int64[nbranches+1] f1: pieces of every branch under the level-mean rule  */
    HINES_TABLE_SPLIT_PIECE_LEN      = 61,  /* int32[npieces] compartments of each piece, from the top of the branch             */
    HINES_TABLE_SPLIT_PIECE_LEVEL    = 62,  /* int32[npieces] level of the piece in the split dependency tree                    */
    HINES_TABLE_SPLIT_LEVEL_STAT     = 63,  /* int64[2*nsplit_levels] {sum of the piece lengths, pieces} on each level: cut = ceil(sum/count) */
    HINES_TABLE_STREAM_LEVEL_BEGIN   = 40,  /* int64[max_stream_levels+1] into STREAM_DESC                             */
    HINES_TABLE_STREAM_DESC          = 41,  /* int32[6*nstream_branches] {global start, len, global parent compartment
                                               (-1 root), workspace start, child_begin, nchild}                       */
    HINES_TABLE_STREAM_CHILD         = 42,  /* int32[2*nstream_children] {global start, workspace start} of each child */
    HINES_TABLE_CLASS_SMEM_BYTES     = 43,  /* int32[n_classes] dynamic shared memory per block of each class          */
    HINES_TABLE_CLASS_CLUSTER        = 50,  /* int32[n_classes] blocks per item = cluster size (1 = no cluster)        */
    HINES_TABLE_CLASS_THREADS        = 51   /* int32[n_classes] threads per block                                      */
} hines_table_id_t;

/*
 * Setup ("only once during the setup phase"): validates the topology, finds the
 * branches and the branch dependency tree, the per-level branch lists (:110, :128),
 * packs cells into work items (:128), sorts each level's branches by length and assigns them to
 * lanes (:130), and lays out the per-item tables.  HOST pointers; O(N) time and memory.
 *   parent        HOST int32[N], N = cell_offsets[ncells]; cell-local; parent[first of cell] = -1,
 *                 0 <= parent[i] < i otherwise.  Any such array is accepted; breadth-first branch
 *                 numbering is what makes branches long and is reported in info.
 *   cell_offsets  HOST int64[ncells+1]; [0] == 0, strictly increasing (no empty cell); N < 2^31.
 *   opt           NULL = defaults.
 * Errors: INVALID_ARG (null, ncells <= 0, bad dtype/options, N >= 2^31), BAD_TOPOLOGY (offsets
 * not increasing, parent out of range; hines_last_error names the first offending index), ALLOC.
 */
hines_status_t hines_plan_create(const int32_t* parent, const int64_t* cell_offsets, int64_t ncells,
                                 hines_dtype_t dtype, const hines_options_t* opt,
                                 hines_plan_t** out_plan);

/* Upload the plan's tables to the current CUDA device and allocate its workspace (done implicitly by
 * the first solve).  Synchronous.  Errors: CUDA (no device / API failure), ALLOC. */
hines_status_t hines_plan_upload(hines_plan_t* plan);

/*
 * The per-step call ("solved in every time step"): x = A^-1 b for every cell.
 *   d, u, b   DEVICE, N elements of the plan's dtype, natural (input) order, 16-byte aligned, read only.
 *   x         DEVICE, N elements; may be == b.
 * Steps run, all inside the library's kernels: load / permute-in,
 * backward elimination level by level, branch-end hand-off (:50),
 * root solve (:91), forward substitution (:97), store / permute-out (:173).
 */
hines_status_t hines_solve(hines_plan_t* plan, const void* d, const void* u, const void* b, void* x,
                           hines_stream_t stream);

/*
 * f3, factor once / solve many ("the matrix ... " changes only with the time step; with a fixed step only
 * the right-hand side changes between steps).  Needs a plan created with HINES_POLICY_FACTORED and no cell on the streaming path.
 *   hines_factor     everything that depends only on d and u (all reciprocals, the pivot recurrences): three factor
 *                    values per unknown, kept in plan-owned device memory (3*N*w bytes).  d, u DEVICE, read only.
 *   hines_solve_rhs  x = A^-1 b from those factors: per unknown one multiply-add on every dependent chain, no division.
 *                    b, x DEVICE; x may be exactly b.  Bytes moved per call: the factors (3w), b (w) read, x (w) written
 *                    = 5*N*w (+ one parent per branch), against 4*N*w for hines_solve: the entry trades bytes for the
 *                    dependent divide chain.
 * Both only enqueue on `stream`.  Errors: UNSUPPORTED (plan without the flag / streaming cells), INVALID_ARG
 * (null, misaligned, hines_solve_rhs before hines_factor, overlapping x), CUDA.
 */
hines_status_t hines_factor(hines_plan_t* plan, const void* d, const void* u, hines_stream_t stream);
hines_status_t hines_solve_rhs(hines_plan_t* plan, const void* b, void* x, hines_stream_t stream);

/*
 * Same solve with HOST buffers (pageable or pinned): copies d, u, b to plan-owned device buffers,
 * solves, copies x back and synchronises `stream`.  This is the end-to-end entry that bench.py times
 * as "e2e".  Bytes moved: 3*N*w host->device, N*w device->host.
 */
hines_status_t hines_solve_host(hines_plan_t* plan, const void* d, const void* u, const void* b, void* x,
                                hines_stream_t stream);

/*
 * Host buffers with the copies overlapped: the end-to-end entry bench.py times as "e2e".  hines_solve_host keeps the link
 * busy in one direction at a time; at 32 bytes per unknown the link is the step.  Cells are independent:
 * the pipeline cuts the batch into `nslices` slices of whole cells with about the same number of unknowns (0 = default
 * 8; fewer if there are fewer cells), builds one plan per slice, and runs copy-in, solve and copy-out of successive
 * slices on three streams, so that x of one slice goes back while d, u, b of the next ones come in (PCIe is full
 * duplex).  Result: bit-identical to hines_solve with the same options on each slice's cells.
 *   create   HOST parent / cell_offsets / options as for hines_plan_create; host-only work (no device needed)
 *   solve    HOST d, u, b (read), x (written; may be b), N elements each; pinned memory makes the copies asynchronous,
 *            pageable memory works (the runtime stages it).  Synchronous: x is complete on return.  The first call
 *            uploads the plans and allocates 4 device arrays of N elements (+ 32 per slice).
 *   slices   the slice boundaries: first_compartment[nslices + 1] (may be NULL to query the count)
 * Errors: as hines_plan_create / hines_solve; INVALID_ARG (null, nslices < 0 or > 1024).
 */
typedef struct hines_host_pipeline hines_host_pipeline_t;
hines_status_t hines_host_pipeline_create(const int32_t* parent, const int64_t* cell_offsets, int64_t ncells,
                                          hines_dtype_t dtype, const hines_options_t* opt, int32_t nslices,
                                          hines_host_pipeline_t** out);
hines_status_t hines_host_pipeline_solve(hines_host_pipeline_t* pipe, const void* d, const void* u, const void* b, void* x);
hines_status_t hines_host_pipeline_slices(const hines_host_pipeline_t* pipe, int32_t* nslices, int64_t* first_compartment,
                                          int64_t capacity);
hines_status_t hines_host_pipeline_destroy(hines_host_pipeline_t* pipe);

/*
 * The one entry point that allocates NOTHING, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Every other solve entry needs an uploaded plan, and the upload
 * allocates.  This one needs no plan: the topology comes as DEVICE arrays, and the kernel's scratch (the working
 * diagonal of the backward sweep, one value per unknown: what the streaming path keeps in the plan's workspace) is a
 * file-scope static __device__ array of HINES_STATIC_SCRATCH_BYTES inside the library, held by every GPU that loads the
 * library until the process exits.  It calls no cudaMalloc / cudaFree / allocating library routine and only enqueues on
 * `stream`.  The arithmetic is Listing 2 of the paper cell by cell, one thread per cell: a fallback,
 * several times slower than hines_solve -- not the path bench.py measures.
 *   parent        DEVICE int32[n], cell-local as for hines_plan_create (parent[first of cell] = -1, 0 <= parent[i] < i).
 *                 NOT validated (that would need a copy to the host): an entry outside [0, i) is treated as "no parent";
 *                 nothing is ever read or written outside [0, n).
 *   cell_offsets  DEVICE int64[ncells + 1], cell_offsets[0] = 0, increasing, cell_offsets[ncells] = n
 *   d, u, b       DEVICE, n elements of `dtype` (HINES_F64 / HINES_F32), natural order, read only
 *   x             DEVICE, n elements; may be exactly b, must not overlap it otherwise
 * Limit: n * sizeof(dtype) <= HINES_STATIC_SCRATCH_BYTES (1,048,576 unknowns in fp64, 2,097,152 in fp32); beyond it
 * UNSUPPORTED with a message naming the limit.  Other errors: INVALID_ARG (null, bad dtype, sizes, overlap), CUDA.
 * The scratch array is shared by every call on a device and keeps the last call's contents; nothing in it has to
 * start at zero (every cell's entries are written before they are read).  Two calls that overlap in time on the same
 * GPU (different streams, or two host threads) RACE on it: serialise them.  The first call on a device looks the
 * array's address up (cudaGetSymbolAddress): make that call outside stream capture.
 */
#define HINES_STATIC_SCRATCH_BYTES 8388608
hines_status_t hines_solve_static(const int32_t* parent, const int64_t* cell_offsets, int64_t ncells, int64_t n,
                                  const void* d, const void* u, const void* b, void* x, int32_t dtype,
                                  hines_stream_t stream);

hines_status_t hines_plan_destroy(hines_plan_t* plan);

/*
 * Multi-GPU: cells are independent, so a batch is spread over several devices by
 * giving every device a subset of the cells -- no exchange step, no collective.  This helper deals the cells to
 * nparts devices by longest-processing-time first on the per-cell cost (the cell's unknowns: the solve is linear in
 * them): cells by cost descending (ties by index), each to the device with the least cost so far (ties to
 * the lowest device).  The caller then builds one plan per device from that device's cells, in input order.
 *   cell_offsets  HOST int64[ncells+1] as for hines_plan_create
 *   cell_part     HOST int32[ncells]  out: device of every cell
 *   part_cost     HOST int64[nparts]  out: unknowns per device (may be NULL)
 * Errors: INVALID_ARG (null, ncells <= 0, nparts <= 0), BAD_TOPOLOGY (offsets not increasing).
 */
hines_status_t hines_partition_cells(const int64_t* cell_offsets, int64_t ncells, int32_t nparts,
                                     int32_t* cell_part, int64_t* part_cost);

/*
 * f2, tree re-rooting (section 6): "Balance the dependency tree so that the depth of the tree is
 * minimized ... find a new root node that minimizes the depth of the tree and permute all unknowns such that they form
 * a new Hines matrix based on the new root node ... numbering all branches breadth first and then sorting all
 * compartments by branch index and distance to the root."  Host, setup time, O(N); allocates host memory only.
 * Per cell: the compartment with the smallest largest distance to any other compartment becomes the root (of two such
 * compartments the one with the larger index, reading R2); the branches of the re-rooted tree are numbered
 * breadth first (children of a branch in ascending old index of their first compartment, R3) and the compartments
 * renumbered by (branch, distance to the root).  Cell sizes do not change: cell_offsets serves the new numbering too.
 *   parent, cell_offsets   HOST, as for hines_plan_create
 *   new_parent   HOST int32[N] out, cell-local, new numbering: feed it to hines_plan_create
 *   perm         HOST int64[N] out, GLOBAL: perm[new] = old compartment
 *   u_src        HOST int64[N] out, GLOBAL: old compartment whose u holds the coupling of `new` to new_parent[new]
 *                (edges on the path from the new root to the old one change direction; u_src[root] = perm[root])
 *   root, depth_before, depth_after   HOST int32[ncells] out, may be NULL: old cell-local index of the new root; the
 *                largest distance (compartments) from the root before and after
 * The re-rooted system is d'[k] = d[perm[k]], b'[k] = b[perm[k]], u'[k] = u[u_src[k]] -- a symmetric permutation of the
 * same matrix -- and its solution is x'[k] = x[perm[k]].  A caller that assembles its matrix in the new numbering pays
 * nothing per step; one that cannot uses hines_gather / hines_scatter below around the solve.
 * Errors: INVALID_ARG (null, ncells <= 0), BAD_TOPOLOGY (as hines_plan_create), ALLOC.
 */
hines_status_t hines_reroot(const int32_t* parent, const int64_t* cell_offsets, int64_t ncells,
                            int32_t* new_parent, int64_t* perm, int64_t* u_src, int32_t* root,
                            int32_t* depth_before, int32_t* depth_after);

/*
 * The permutation carried through load and store (f2): dst[k] = src[index[k]] (gather) and dst[index[k]] = src[k]
 * (scatter), k < n, elements of `dtype`; all pointers DEVICE, index int64, dst must not overlap src; only enqueue on
 * `stream`.  Bytes per element: 2w + 8.  Errors: INVALID_ARG (null, n < 0, bad dtype), CUDA.
 */
hines_status_t hines_gather(void* dst, const void* src, const int64_t* index, int64_t n, int32_t dtype, hines_stream_t stream);
hines_status_t hines_scatter(void* dst, const void* src, const int64_t* index, int64_t n, int32_t dtype, hines_stream_t stream);

/* Introspection: needed for the bit-exact table parity tests and for reporting. */
hines_status_t hines_plan_get_info(const hines_plan_t* plan, hines_plan_info_t* out);

/* Copies table `table_id` to host_dst if capacity_bytes suffices; always writes the size needed to
 * *needed_bytes (host_dst may be NULL to query).  Errors: INVALID_ARG (unknown id, null needed_bytes,
 * capacity too small). */
hines_status_t hines_plan_get_table(const hines_plan_t* plan, int32_t table_id, void* host_dst,
                                    int64_t capacity_bytes, int64_t* needed_bytes);

/* Device-side timing of the two paths, for the roofline report.  With timing enabled every
 * hines_solve records three CUDA events on its stream (before the shared-memory kernels, between the
 * two paths, after the streaming kernels).  hines_plan_get_timing waits for the last solve and returns
 * the milliseconds the resident (shared-memory) launches and the streaming launches took.
 * Errors: INVALID_ARG (null, timing not enabled, no solve yet), CUDA. */
hines_status_t hines_plan_enable_timing(hines_plan_t* plan, int32_t enable);
hines_status_t hines_plan_get_timing(hines_plan_t* plan, float* resident_ms, float* stream_ms);

/* Load-imbalance / phase hook (debug; SURVEY.md §8(d) "per-work-item cycle counts").  With phase clocks
 * enabled every block of the shared-memory kernel records, per solve, 8 x uint64: %globaltimer (ns) at
 * [0] block start, [1] inputs landed in shared memory, [2] segment interiors condensed, [3] backward
 * level sweep done, [4] forward sweep done (blocks of rank > 0: the wait for rank 0), [5] interiors expanded,
 * [6] x stored; [7] = (SM id << 32) | unknowns of the block.  Rows are in launch order (classes in order, inside a
 * class HINES_TABLE_ITEM_LAUNCH_ORDER, the blocks of a cluster item consecutive).
 * hines_plan_get_phase_clocks synchronises the device and copies the rows of the last solve
 * (host_dst may be NULL to query the size).  Errors: INVALID_ARG, CUDA, ALLOC. */
hines_status_t hines_plan_enable_phase_clocks(hines_plan_t* plan, int32_t enable);
hines_status_t hines_plan_get_phase_clocks(hines_plan_t* plan, uint64_t* host_dst, int64_t capacity_bytes,
                                           int64_t* needed_bytes);

/* Number of kernel launches one hines_solve enqueues with this plan (bench.py's gpu_launches). */
hines_status_t hines_plan_launches_per_solve(const hines_plan_t* plan, int32_t* out);

const char* hines_status_string(hines_status_t s);
const char* hines_last_error(void);      /* thread-local, never NULL */
const char* hines_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HINES_B200_H */

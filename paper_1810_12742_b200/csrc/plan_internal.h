// Internal layout of hines_plan (library-private; the public surface is include/hines.h).
#pragma once
#include <cstdint>
#include <functional>
#include <string>
#include <vector>

#include "hines.h"

namespace hines {

// One PART = what one block stages into its shared memory: whole branches, given as runs of consecutive
// compartments of the caller's natural-order arrays.  A work item is
//   single   one part holding a contiguous run of whole cells (cells are packed into a block
//            in the order given);
//   cluster  ONE cell too large for a block, cut into a top part (rank 0: the root region + some complete
//            sub-trees) and parts made of complete sub-trees, one part per block of a thread-block cluster;
//            a sub-tree's root hands (f U + parked, f B + parked) to rank 0 and reads its parent's x back through
//            distributed shared memory (PAPER.md:50 the hand-off at a branch point);
//   split    ONE cell too large for a cluster: the sub-tree parts run as ordinary blocks of a first launch
//            (backward sweep, hand-off exported to a global exchange buffer), the top part as a second
//            launch, and the sub-tree parts again as a third launch that repeats its backward sweep, imports
//            the parent's x and finishes ("one matrix per block" lifted by kernel boundaries).
// Device record of a part, one per launched block, in launch order (128 bytes).
struct PartHeader {
    int64_t meta_off;        // offset (int32 units, multiple of 4) of the part's metadata blob
    int32_t meta_len;        // int32 count (multiple of 4): brought into shared memory by one bulk copy
    int32_t run_off;         // index (int4 units) of the part's run table; the first kInlineRuns runs are also in the block record
    int32_t nrun;
    int32_t tx_elems;        // elements per array the bulk copies bring (runs widened to 16-byte words, clipped at N)
    int32_t L;               // elements per staged array (multiple of 16 / w)
    int32_t n;               // unknowns of the part
    int32_t nnode;           // node records: level nodes (real nodes + ghost children), then ghost parents
    int32_t nlevnode;        // nodes in the level lists = lb[nlev]
    int32_t nlev;            // local levels of the reduced forest (depth in the cell - smallest depth in the part);
                             // a part of unbranched cables (flags bit 0): the number of cables, lb[] = first node of each
    int32_t rounds;          // pointer-jumping rounds of the part's forward sweep
    int32_t kp_off, exp_off, gh_off, seg_off;   // offsets (ints, multiples of 4) inside the blob; lb[] sits at 0
    int32_t nexp;            // exports: sub-tree roots whose parent node lives in the item's part 0
    int32_t nghost;          // ghost children (part 0 only): stand-ins for the exported roots of the other parts
    int32_t nseg_lanes;      // segment lane descriptors (P1 / P3)
    int32_t xch_base;        // split items: first slot of the item in the plan's global exchange buffers
    int32_t xs0;             // cluster items: record slot that holds x in rank 0 after ITS forward sweep
    int32_t item, rank;
    int32_t flags;           // bit 0: every cell of the part is an unbranched cable of <= 32 nodes (PCR path)
    int32_t ntoplev;         // part 0 of a multi-part item: local levels that hold top nodes (ancestors of ghost children)
    int32_t lowlev;          // the smallest local level with a real node that is not a top node (nlev if there is none)
    int32_t maxwidth;        // widest local level (nodes)
    int32_t pad_[5];
};
static_assert(sizeof(PartHeader) == 128, "PartHeader is read as 8 x int4");

// What a block reads first: the part's header and its first runs side by side, at a fixed stride, so that one
// dependent global load stands between the block's start and its bulk copies.
enum { kInlineRuns = 24 };
struct BlockRecord {         // 512 bytes
    PartHeader h;
    int32_t runs[4 * kInlineRuns];
};
static_assert(sizeof(BlockRecord) == 512, "BlockRecord is read as 32 x int4");

enum { kPartFlagChains = 1, kPartFlagFactored = 2 };     // factored: a fourth staged array follows sb
enum { kItemSingle = 0, kItemCluster = 1, kItemSplit = 2 };
// launch phases of a size class: 0 = ordinary (single / cluster items); split items: 1 = sub-tree parts
// backward + export (A), 2 = top part (B), 3 = sub-tree parts again, import + forward (C)
enum { kPhaseAll = 0, kPhaseA = 1, kPhaseB = 2, kPhaseC = 3 };

// Streaming-path branch descriptor (24 bytes).
struct StreamDesc {
    int32_t gstart;       // global compartment index of the branch's first compartment
    int32_t len;
    int32_t gparent;      // global index of the parent compartment, -1 for a root branch
    int32_t ws;           // workspace index of the branch's first compartment
    int32_t child_begin;  // into stream_child
    int32_t nchild;
};

struct SplitPiece { int64_t j; int32_t len, level; };       // a piece of global branch j under a splitting pass (f1 / f4)

struct DeviceTables;      // solve.cu

void set_error(const std::string& msg);

}  // namespace hines

struct hines_plan {
    int64_t n = 0, ncells = 0, nbranches = 0;
    int32_t dtype = 0, width = 8;
    hines_options_t opt{};
    int32_t max_levels = 0;
    int32_t breadth_first = 1;
    int32_t quad_max_warps = 22;                       // ... where (blocks per SM) x (P1 warps with four lanes) stays within this
    int32_t quad_min = 24;                             // segments with at least this many interior nodes get four lanes (0: never)
    int32_t seg_single = 64, seg_cluster = 64;         // segment target (max_segment) of single-block / multi-part items

    std::vector<int64_t> cell_offsets;
    // canonical tables T1-T7
    std::vector<int64_t> cell_branch_offsets, cell_level_offsets, child_offsets;
    std::vector<int32_t> branch_start, branch_len, branch_parent_comp, branch_parent_branch,
        branch_level, cell_nlevels, level_count, level_list, child_ids;
    // f1: pieces of the level-mean splitting pass over the whole batch; with HINES_POLICY_SPLIT_BLOCK_MEAN (f4,
    // PAPER.md:189) replaced after packing by the pieces under every block's own level means
    std::vector<int64_t> split_piece_offsets;          // [nbranches+1] into split_piece_len
    std::vector<int32_t> split_piece_len, split_piece_level;
    std::vector<int64_t> split_level_stat;             // per level of the split tree: {sum of the piece lengths, pieces}
    std::vector<hines::SplitPiece> block_split;        // f4 (HINES_POLICY_SPLIT_BLOCK_MEAN): pieces under every block's own level means, item by item
    // policy tables
    std::vector<int32_t> cell_item, item_class, item_kind, item_launch_order, item_xch;
    std::vector<int64_t> item_cell_offsets, item_cells, item_unknowns, item_part_offsets;
    std::vector<hines::PartHeader> part_headers;       // indexed by part id (item order, parts of an item consecutive)
    std::vector<int32_t> part_meta;                    // device blob: per part [lb | kp | exports | ghosts | segment lanes]
    std::vector<int32_t> part_runs;                    // 4 ints per run, GLOBAL first compartment
    std::vector<int32_t> class_smem_bytes;             // per class: dynamic smem per block
    std::vector<int32_t> class_cluster;                // per class: blocks per item (cluster size), 1 = no cluster
    std::vector<int32_t> class_threads;                // per class: threads per block
    std::vector<int32_t> class_phase;                  // per class: kPhase*
    std::vector<int32_t> class_quads;                  // per class: some part has four-lane segment groups
    std::vector<int64_t> class_first, class_count;     // ranges in class_parts (blocks of the class, launch order)
    std::vector<int32_t> class_parts;                  // part ids in launch order, class by class
    int64_t n_xch = 0;                                 // exchange slots (split items)
    // streaming path
    std::vector<int64_t> stream_level_begin;           // [nstream_levels+1]
    std::vector<hines::StreamDesc> stream_desc;
    std::vector<int32_t> stream_child;                 // pairs {gstart, ws}
    int64_t n_stream_cells = 0, n_stream_unknowns = 0;
    int64_t n_resident_cells = 0, n_resident_unknowns = 0, n_cluster_cells = 0, n_cluster_unknowns = 0;
    int64_t n_split_cells = 0, n_split_unknowns = 0;
    int64_t padded_lane_steps = 0, useful_lane_steps = 0;
    int64_t n_exports = 0;

    hines::DeviceTables* dev = nullptr;                // null until uploaded
};

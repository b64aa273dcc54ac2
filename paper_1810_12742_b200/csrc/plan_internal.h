// Internal layout of hines_plan (library-private; the public surface is include/hines.h).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "hines.h"

namespace hines {

// One on-chip work item = a contiguous run of whole cells held in the shared memory of one block
// (nchunks == 1; cells are packed into a block in the order given), or ONE cell too
// large for that, spread over the shared memories of a thread-block cluster (nchunks == cluster
// size; chunk r lives in the block of cluster rank r, the level-synchronous part runs in rank 0).
struct ItemHeader {          // 56 bytes
    int64_t meta_off;        // offset (int32 units, multiple of 4) of the item's metadata blob:
                             //   [task blob (plan.cpp build_tasks) | pnode nnode | pad4]
    int32_t meta_len;        // int32 count (multiple of 4)
    int32_t grp_off;         // offsets inside the blob: group headers (36 ints each),
    int32_t ent_off;         //   entries (4 ints per node),
    int32_t pull_off;        //   pull list,
    int32_t pnode_off;       //   parent-node list
    int32_t ntier;           // tiers of the backward sweep (block barrier between tiers)
    int32_t nnode;           // nodes of the reduced tree
    int32_t first_chunk;     // index of the item's first chunk
    int32_t nchunks;
    int32_t n;               // unknowns of the item
    int32_t rounds;          // pointer-jumping rounds of the forward sweep over the reduced tree
    int32_t pad_;
};

// One chunk = the contiguous compartment range one block stages into its shared memory.
struct ChunkHeader {         // 32 bytes
    int64_t comp_begin;      // global index of the chunk's first compartment
    int64_t seg_off;         // offset (int32 units, multiple of 4) of the chunk's segment descriptors
    int32_t n;               // unknowns in the chunk
    int32_t nseg_lanes;      // segment descriptors (lanes of the condensation / expansion sweeps)
    int32_t item;
    int32_t rank;            // position inside the item = cluster rank
};

// Streaming-path branch descriptor (24 bytes).
struct StreamDesc {
    int32_t gstart;       // global compartment index of the branch's first compartment
    int32_t len;
    int32_t gparent;      // global index of the parent compartment, -1 for a root branch
    int32_t ws;           // workspace index of the branch's first compartment
    int32_t child_begin;  // into stream_child
    int32_t nchild;
};

struct DeviceTables;      // solve.cu

void set_error(const std::string& msg);

}  // namespace hines

struct hines_plan {
    int64_t n = 0, ncells = 0, nbranches = 0;
    int32_t dtype = 0, width = 8;
    hines_options_t opt{};
    int32_t max_levels = 0;
    int32_t breadth_first = 1;
    int32_t seg_single = 64, seg_cluster = 64;         // segment target (max_segment) of single-block / cluster items

    std::vector<int64_t> cell_offsets;
    // canonical tables T1-T7
    std::vector<int64_t> cell_branch_offsets, cell_level_offsets, child_offsets;
    std::vector<int32_t> branch_start, branch_len, branch_parent_comp, branch_parent_branch,
        branch_level, cell_nlevels, level_count, level_list, child_ids;
    // policy tables
    std::vector<int32_t> cell_item, item_class, item_launch_order, item_pnode,
        item_nnode, item_rounds, item_task_blob, chunk_seg;
    std::vector<int64_t> item_cell_range, item_node_offsets, item_task_offsets, item_chunk_offsets,
        chunk_comp_range, chunk_seg_offsets;
    std::vector<int32_t> class_smem_bytes;             // per class: dynamic smem per block
    std::vector<int32_t> class_cluster;                // per class: blocks per item (cluster size), 1 = no cluster
    std::vector<int32_t> class_threads;                // per class: threads per block
    std::vector<int64_t> class_first, class_count;     // ranges in item_launch_order
    std::vector<hines::ItemHeader> item_headers;       // indexed by item id
    std::vector<hines::ChunkHeader> chunk_headers;     // indexed by chunk id
    std::vector<int32_t> item_meta;                    // device blob
    // streaming path
    std::vector<int64_t> stream_level_begin;           // [nstream_levels+1]
    std::vector<hines::StreamDesc> stream_desc;
    std::vector<int32_t> stream_child;                 // pairs {gstart, ws}
    int64_t n_stream_cells = 0, n_stream_unknowns = 0;
    int64_t n_resident_cells = 0, n_resident_unknowns = 0, n_cluster_cells = 0, n_cluster_unknowns = 0;
    int64_t padded_lane_steps = 0, useful_lane_steps = 0;

    hines::DeviceTables* dev = nullptr;                // null until uploaded
};

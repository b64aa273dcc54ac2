// hines_plan_create: the setup-time scheduler (host only, O(N)).
//
// What it builds, with the passage of arXiv 1810.12742 each table comes from:
//   T1-T4  branches, their parent compartment / parent branch and level: the branch dependency
//          tree ("form a dependency tree. Each node in this tree represents a
//          submatrix"; :138 "it is sufficient to store only one parent compartment for each branch").
//   T5-T6  per-level branch counts and per-level lists sorted by size.
//   T7     child lists (the edges of the dependency tree, used by the streaming path's pull hand-off).
//   P1-P2  cells -> work items: greedy in input order while the item fits the block's shared memory
//          ("we assign matrices to a Cuda block as long as ... When a matrix doesn't fit
//          into a Cuda block any longer, we start a new Cuda block"); the fit test here is bytes of
//          shared memory instead of "branches per level <= threads", because a B200 block loops over
//          a level's lane list and is limited by its 227 KB of shared memory, not its thread count.
//          A cell too large for one block is cut into chunks held by the blocks of one thread-block
//          cluster (the paper requires one matrix per block; distributed shared memory
//          lifts that).  Cells that fit no cluster go to the streaming path.
//   P3     the reduced tree (one node per segment) and its backward sweep: sub-trees of at most 32 leaves,
//          one warp per group of sub-trees, lock-step over the height above the leaves (PAPER.md:110-112
//          with height in place of depth), a node in the lane of its first child so that the hand-off at
//          the branch point stays in registers or is a warp shuffle (build_tasks).
//   P4     segments.  Every branch is cut, from its end, into nseg = ceil(len / max_segment) segments
//          of Sj = ceil(len / nseg) compartments (the paper's branch splitting, with a
//          fixed bound instead of the level average).  The last compartment of a segment is its
//          separator; the compartments above it are its interior.  Interiors are eliminated
//          independently of the tree level (one lane per segment, all segments of the item at once),
//          which leaves the level-synchronous sweeps with one node per segment.  The segment lane list
//          is ordered so that the 16 (fp64) / 32 (fp32) lanes that access shared memory together start
//          at different bank residues and have similar lengths.
// Written policy: DESIGN.md "Scheduler policy".
#include <algorithm>
#include <cstring>
#include <new>
#include <numeric>
#include <string>

#include "plan_internal.h"

namespace hines {

static thread_local std::string g_last_error;
void set_error(const std::string& msg) { g_last_error = msg; }

static const int64_t kSmemPerSM = 233472;       // 228 KiB
static const int64_t kSmemMaxOptin = 232448;    // 227 KiB
static const int kClassK[] = {1, 2, 3, 4, 6, 8};
static const int kNumClassK = 6;
static const int kRegsPerThread = 80;           // the resident kernel is built for __launch_bounds__(384, 2): up to 85
static const int kMaxThreads = 384;
static const int kMaxClusterClass = 16;
static const int32_t kSegA = 1, kSegB = 2;          // segment lane kinds (descriptor word 1, bits 24-25)

static inline int64_t round_up(int64_t v, int64_t m) { return (v + m - 1) / m * m; }

static int64_t class_cap(int k, int64_t max_smem)
{
    int64_t cap = (kSmemPerSM / k - 1024) / 128 * 128;
    return std::min(cap, max_smem);
}

// One branch of the item while its lists are built.
struct Br {
    int32_t start, len, pc, level, parent;   // item-local positions; parent = index into the item's branch array
    int32_t nseg, sj;                        // segments, compartments per segment (the first may be shorter)
    int32_t e = -1, rest = -1;               // lane index (= id of the top node); id of the second node from the top
};

// Lists of one work item: cells [c0,c1) in nchunks chunks, policies P3 + P4.
struct ItemBuild {
    int64_t comp_begin = 0, n = 0;
    int32_t nlev = 0, ndesc = 0, nnode = 0, nchunks = 1;
    bool ok = true;                          // false: a field overflows its descriptor bits -> streaming path
    std::vector<int32_t> pnode;              // 1 per node: the node above it in the reduced tree; itself for a root / an unused id
    std::vector<int32_t> perm;               // node id used while the lists were built -> final node id (build_tasks)
    std::vector<int32_t> task_blob;          // device tables of the backward sweep (build_tasks), multiple of 4 ints
    int32_t ntier = 0, grp_off = 0, ent_off = 0, pull_off = 0, ngroups = 0;
    std::vector<int32_t> task_entry, task_group, task_pull, task_tier_begin;   // the same, for the table getters
    std::vector<unsigned char> task_nsh;
    int32_t rounds = 0;                      // pointer-jumping rounds of the forward sweep: 2^rounds >= nodes on the longest root path
    struct Chunk {
        int32_t begin = 0, n = 0;            // item-local compartment range
        std::vector<int32_t> seg;            // 4 per segment lane {a (chunk-local), m, node, tnode}; node = -1 padding
        int64_t smem_need = 0;
    };
    std::vector<Chunk> chunks;
    int64_t padded_steps = 0, useful_steps = 0;
    int64_t leader_extra = 0;                // bytes of the reduced arrays + item metadata (rank 0 only)
    int64_t smem_need = 0;                   // max over the chunks (rank 0 includes leader_extra)
    int64_t total_bytes = 0;                 // shared memory of the whole item, all chunks together
    int32_t max_lanes = 0;                   // widest segment lane list of a chunk
};

struct SegTmp { int32_t a, m, node, tnode, mt = -1; };   // mt: interior nodes lane A takes (-1: half)

// Segment lane list of one chunk.  R = 16 segments share a warp (A lanes 0-15, B lanes 16-31); the lanes of a
// half-warp access shared memory in one wavefront if, at every step, they sit on distinct residues mod R, and
// a warp runs as long as its longest lane.  Segments are sorted by length, longest first, and
// a group is cut from the head of the list: its step count is the longer half of the head segment.  A lane
// that is shorter than the group may START LATE: a delay of dl steps moves its residue by -dl in every step,
// at no cost.  For each of the next kLook candidates the split point (off the middle by up to two nodes) and
// the delays of both lanes are chosen so that the A lanes and the B lanes of the group keep distinct residues
// mod NB (fp64: NB = 16 banks of 8 bytes, A and B lanes are different wavefronts; fp32: NB = 32, all 32 lanes
// are one wavefront and share one set of residues);
// a candidate that cannot be placed stays in the list.  A group that ends up far from full is filled up with
// the longest remaining segments, conflicts and all.
// out: 4 ints per segment {a, m | mt << 12 | dA << 24 | dB << 28, node, tnode}, groups padded to R with node -1.
static void order_segments(const std::vector<SegTmp>& segs, int R, int NB, int32_t off, std::vector<int32_t>& out)
{
    std::vector<SegTmp> sorted(segs);
    std::stable_sort(sorted.begin(), sorted.end(), [](const SegTmp& x, const SegTmp& y) { return x.m > y.m; });
    const size_t n = sorted.size();
    std::vector<int32_t> next(n + 1);                       // singly linked list over the sorted order, n = end
    for (size_t k = 0; k <= n; ++k) next[k] = (int32_t)k + 1;
    int32_t head = n ? 0 : (int32_t)n;
    out.clear();
    std::vector<char> ua_(NB), ub_(NB);
    std::vector<char>& ua = ua_;
    std::vector<char>& ub = NB > R ? ua_ : ub_;            // one wavefront: one set
    size_t remaining = n;
    auto emit = [&](int32_t k, int mt, int dA, int dB) {
        const SegTmp& sg = sorted[k];
        const uint32_t word = (uint32_t)sg.m | ((uint32_t)mt << 12) | ((uint32_t)dA << 24) | ((uint32_t)dB << 28);
        out.insert(out.end(), {sg.a, (int32_t)word, sg.node, sg.tnode});
        --remaining;
    };
    const int kLook = 2 * R, kMinFill = R - 2, kMaxDelay = 15;
    static const int kDelta[5] = {0, 1, -1, 2, -2};
    while (remaining) {
        std::fill(ua_.begin(), ua_.end(), 0); std::fill(ub_.begin(), ub_.end(), 0);
        int taken = 0;
        const int nhalf = sorted[head].m / 2;              // steps of the group: mt = m/2 >= mb = m-1-mt of the head
        for (int pass = 0; pass < 2 && taken < R && remaining; ++pass) {
            if (pass > 0 && taken >= kMinFill) break;
            int32_t prev = -1, k = head;
            for (int looked = 0; k < (int32_t)n && taken < R && looked < kLook; ++looked) {
                const SegTmp& sg = sorted[k];
                int mt = sg.m / 2, dA = 0, dB = 0;
                bool ok = pass == 1 || sg.m == 0;
                for (int t = 0; t < 5 && !ok; ++t) {
                    const int cmt = sg.m / 2 + kDelta[t], cmb = sg.m - 1 - cmt;
                    if (cmt < 0 || cmb < 0 || cmt > nhalf || cmb > nhalf) continue;
                    int fa = -1, fb = -1;
                    for (int dl = 0; dl <= std::min(kMaxDelay, nhalf - cmt) && fa < 0; ++dl)
                        if (cmt == 0 || !ua[((sg.a + off - dl) % NB + NB) % NB]) fa = dl;
                    const int ra = NB > R && cmt > 0 && fa >= 0 ? ((sg.a + off - fa) % NB + NB) % NB : -1;
                    for (int dl = 0; dl <= std::min(kMaxDelay, nhalf - cmb) && fb < 0; ++dl) {
                        const int rb = ((sg.a + cmt + 1 + off - dl) % NB + NB) % NB;
                        if (cmb == 0 || (!ub[rb] && rb != ra)) fb = dl;
                    }
                    if (fa >= 0 && fb >= 0) { ok = true; mt = cmt; dA = cmt ? fa : 0; dB = cmb ? fb : 0; }
                }
                const int32_t nx = next[k];
                if (ok) {
                    const int mb = sg.m - 1 - mt;
                    if (mt > 0) ua[((sg.a + off - dA) % NB + NB) % NB] = 1;
                    if (mb > 0) ub[((sg.a + mt + 1 + off - dB) % NB + NB) % NB] = 1;
                    emit(k, mt, dA, dB); ++taken;
                    if (prev < 0) head = nx; else next[prev] = nx;       // unlink
                } else {
                    prev = k;
                }
                k = nx;
            }
        }
        if (remaining || (out.size() / 4) % R) while ((out.size() / 4) % R) out.insert(out.end(), {0, 0, -1, -1});
    }
}

// Backward sweep over the reduced tree (policy P3).  The tree is cut into sub-trees of at most 32 leaves;
// a sub-tree is swept by the lanes of ONE warp in lock-step over the node's height (PAPER.md:110-112 with
// height above the leaves in place of depth below the root): a node sits in the lane of its first child,
// so the first child's hand-off value is already in that lane's registers and the other children's values
// come by warp shuffle from their lanes -- no shared memory and no barrier on the dependent
// chain.  Sub-trees of a tier are packed into groups of at most 32 lanes (one warp each); what lies above
// the sub-trees forms the next tier, whose leaves pull the hand-off values of the tier below from shared
// memory after a block barrier.
//   group   36 ints: lane_begin[33] (into the item's entries), steps, offset of the per-step shuffle
//           counts (bytes), pad
//   entry   4 ints per node, by lane then step: node | step << 20, lanes of the other children in the
//           same group (bit mask, summed in ascending lane order), first of the pull list, count of the pull
//           list | (entries behind this one that continue its run with nothing to pull) << 16
//   pull    node ids whose hand-off slot the node adds (children swept in an earlier tier)
static void build_tasks(ItemBuild& out, const std::vector<int32_t>& depth)
{
    const int32_t nn = out.nnode;
    std::vector<std::vector<int32_t>> kids(nn);
    std::vector<int32_t> order(nn);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return depth[a] > depth[b]; });   // deepest first
    for (int32_t v = 0; v < nn; ++v) if (out.pnode[v] != v) kids[out.pnode[v]].push_back(v);                   // ascending id
    std::vector<int32_t> tier(nn, -1), leaves(nn), group_of(nn, -1), lane_of(nn, -1), step_of(nn, 0);
    struct Group { std::vector<int32_t> roots; int32_t lanes = 0, steps = 0; std::vector<std::vector<int32_t>> chain; };
    std::vector<Group> groups;
    std::vector<int32_t> tier_begin(1, 0);
    int32_t remaining = nn;
    for (int32_t t = 0; remaining > 0; ++t) {
        if (t >= 64) { out.ok = false; break; }
        // leaves of the remaining forest below every remaining node
        for (int32_t v : order) {
            if (tier[v] >= 0) continue;
            int32_t l = 0;
            for (int32_t c : kids[v]) if (tier[c] < 0) l += leaves[c];
            leaves[v] = l ? l : 1;
        }
        // sub-tree roots of this tier: at most 32 leaves, parent (if any) has more
        std::vector<int32_t> roots;
        for (int32_t v = 0; v < nn; ++v)
            if (tier[v] < 0 && leaves[v] <= 32 && (out.pnode[v] == v || leaves[out.pnode[v]] > 32)) roots.push_back(v);
        // pack into groups (first fit in id order), assign lanes and steps
        const size_t g0 = groups.size();
        for (int32_t r : roots) {
            size_t g = g0;
            while (g < groups.size() && groups[g].lanes + leaves[r] > 32) ++g;
            if (g == groups.size()) { groups.push_back(Group()); groups[g].chain.resize(32); }
            Group& G = groups[g];
            // iterative DFS: a node takes the lane of its first remaining child, a leaf the next free lane
            std::vector<std::pair<int32_t, int32_t>> stack(1, {r, 0});      // (node, phase)
            while (!stack.empty()) {
                auto [v, ph] = stack.back(); stack.pop_back();
                if (ph == 0) {
                    stack.push_back({v, 1});
                    for (auto it = kids[v].rbegin(); it != kids[v].rend(); ++it) if (tier[*it] < 0) stack.push_back({*it, 0});
                } else {
                    int32_t first = -1, h = 0;
                    for (int32_t c : kids[v]) if (tier[c] < 0) { if (first < 0) first = c; h = std::max(h, step_of[c] + 1); }
                    // in a sub-tree that is a plain chain (one leaf) every node continues its child's run: same
                    // step, no shuffle, no pull -- the lane walks the chain without waiting for the lock-step of
                    // the other lanes (in a branching sub-tree runs would make a step as long as its longest run)
                    if (leaves[r] == 1 && first >= 0) h = step_of[first];
                    lane_of[v] = first < 0 ? G.lanes++ : lane_of[first];
                    step_of[v] = h; group_of[v] = (int32_t)g;
                    G.chain[lane_of[v]].push_back(v);
                    G.steps = std::max(G.steps, h + 1);
                }
            }
            G.roots.push_back(r);
        }
        // commit the tier (after the DFS, which tests tier[] < 0 for "remaining")
        for (size_t g = g0; g < groups.size(); ++g)
            for (auto& ch : groups[g].chain) for (int32_t v : ch) { tier[v] = t; --remaining; }
        tier_begin.push_back((int32_t)groups.size());
        if (roots.empty()) { out.ok = false; break; }
    }
    if (!out.ok) { out.task_blob.assign(4, 0); return; }
    // tables
    out.ntier = (int32_t)tier_begin.size() - 1;
    out.ngroups = (int32_t)groups.size();
    out.task_tier_begin = tier_begin;
    out.task_entry.clear(); out.task_group.clear(); out.task_pull.clear(); out.task_nsh.clear();
    for (Group& G : groups) {
        std::vector<unsigned char> nsh(G.steps, 0);
        const size_t gh = out.task_group.size();
        out.task_group.resize(gh + 36, 0);
        for (int32_t l = 0; l < 32; ++l) {
            out.task_group[gh + l] = (int32_t)(out.task_entry.size() / 4);
            for (int32_t v : G.chain[l]) {
                if (step_of[v] >= 4096) out.ok = false;
                uint32_t mask = 0; int32_t first = -1;
                const int32_t pull0 = (int32_t)out.task_pull.size();
                for (int32_t c : kids[v]) {
                    if (tier[c] == tier[v]) { if (first < 0) first = c; else mask |= 1u << lane_of[c]; }
                    else out.task_pull.push_back(c);
                }
                int32_t pc = 0; for (uint32_t m = mask; m; m &= m - 1) ++pc;
                nsh[step_of[v]] = std::max<unsigned char>(nsh[step_of[v]], (unsigned char)pc);
                const int32_t npull = (int32_t)out.task_pull.size() - pull0;
                if (npull > 0xffff) out.ok = false;
                out.task_entry.insert(out.task_entry.end(), {v | (step_of[v] << 20), (int32_t)mask, pull0, npull});
            }
            // upper half of the last word: how many entries right behind this one continue its run with
            // nothing to pull (same step, only child = the node before): the kernel walks those in a tight loop
            const size_t e0 = (size_t)out.task_group[gh + l], e1 = out.task_entry.size() / 4;
            int32_t more = 0;
            for (size_t k = e1; k-- > e0;) {
                out.task_entry[4 * k + 3] |= std::min(more, 0xffff) << 16;
                const bool plain = (out.task_entry[4 * k + 3] & 0xffff) == 0 && k > e0 &&
                                   (out.task_entry[4 * k] >> 20) == (out.task_entry[4 * (k - 1)] >> 20);
                more = plain ? more + 1 : 0;
            }
        }
        out.task_group[gh + 32] = (int32_t)(out.task_entry.size() / 4);
        out.task_group[gh + 33] = G.steps;
        out.task_group[gh + 34] = (int32_t)out.task_nsh.size();      // byte offset, made absolute below
        out.task_nsh.insert(out.task_nsh.end(), nsh.begin(), nsh.end());
    }
    // Renumber the nodes in entry order (group, lane, position in the lane's chain): the records of a lane's
    // chain are then consecutive in shared memory, so the address of the lane's next record does not wait for
    // a descriptor.  From here on node id = entry index.
    out.perm.assign(nn, -1);
    for (size_t k = 0; k < out.task_entry.size() / 4; ++k) out.perm[out.task_entry[4 * k] & 0xfffff] = (int32_t)k;
    for (int32_t v = 0; v < nn; ++v) if (out.perm[v] < 0) { out.ok = false; out.task_blob.assign(4, 0); return; }
    for (size_t k = 0; k < out.task_entry.size() / 4; ++k)
        out.task_entry[4 * k] = (int32_t)k | (out.task_entry[4 * k] & ~0xfffff);
    for (int32_t& c : out.task_pull) c = out.perm[c];
    {
        std::vector<int32_t> np(nn);
        for (int32_t v = 0; v < nn; ++v) np[out.perm[v]] = out.perm[out.pnode[v]];
        out.pnode.swap(np);
    }
    // A lane whose chain ends in a root turns around there: x_root = c_root, then x = c - f x_parent down its own
    // chain, straight after the backward sweep (group word 35 = mask of such lanes).  Those nodes are final before
    // the pointer jumping starts and read themselves in it; the rounds follow from the distance of the other nodes
    // to their nearest final ancestor (2^rounds > distance; none left: no round at all, e.g. unbranched cables).
    {
        std::vector<char> fin(nn, 0);
        for (int32_t g = 0; g < out.ngroups; ++g) {
            int32_t* gh = &out.task_group[36 * (size_t)g];
            uint32_t mask = 0;
            for (int32_t l = 0; l < 32; ++l) {
                const int32_t b = gh[l], e = gh[l + 1];
                if (e > b && out.pnode[e - 1] == e - 1) { mask |= 1u << l; for (int32_t k = b; k < e; ++k) fin[k] = 1; }
            }
            gh[35] = (int32_t)mask;
        }
        std::vector<int32_t> byd(nn), dnew(nn), dist(nn, 0);
        for (int32_t v = 0; v < nn; ++v) dnew[out.perm[v]] = depth[v];
        std::iota(byd.begin(), byd.end(), 0);
        std::stable_sort(byd.begin(), byd.end(), [&](int32_t a, int32_t b) { return dnew[a] < dnew[b]; });   // parents first
        auto rounds_for = [&](bool turn) {
            int32_t maxdist = 0;
            for (int32_t v : byd) {
                const bool f = turn ? fin[v] != 0 : out.pnode[v] == v;
                dist[v] = f ? 0 : dist[out.pnode[v]] + 1;
                maxdist = std::max(maxdist, dist[v]);
            }
            int32_t r = 0;
            while ((1 << r) <= maxdist) ++r;
            return r;
        };
        // the turn-around lengthens the backward sweep by the root chains: taken only where it saves a round
        const int32_t r_plain = rounds_for(false), r_turn = rounds_for(true);
        if (r_turn < r_plain) {
            out.rounds = r_turn;
            for (int32_t v = 0; v < nn; ++v) if (fin[v]) out.pnode[v] = v;
        } else {
            out.rounds = r_plain;
            for (int32_t g = 0; g < out.ngroups; ++g) out.task_group[36 * (size_t)g + 35] = 0;
        }
    }
    // blob: [ntier, tier_begin (ntier+1), pad4 | groups | entries | pull, pad4 | shuffle counts, pad4]
    std::vector<int32_t>& B = out.task_blob;
    B.clear();
    B.push_back(out.ntier);
    B.insert(B.end(), tier_begin.begin(), tier_begin.end());
    B.resize(round_up((int64_t)B.size(), 4), 0);
    out.grp_off = (int32_t)B.size();
    B.insert(B.end(), out.task_group.begin(), out.task_group.end());
    out.ent_off = (int32_t)B.size();
    B.insert(B.end(), out.task_entry.begin(), out.task_entry.end());
    out.pull_off = (int32_t)B.size();
    B.insert(B.end(), out.task_pull.begin(), out.task_pull.end());
    B.resize(round_up((int64_t)B.size(), 4), 0);
    const int32_t nsh_off = (int32_t)B.size();
    B.resize(B.size() + round_up((int64_t)out.task_nsh.size(), 16) / 4, 0);
    if (!out.task_nsh.empty()) std::memcpy(&B[nsh_off], out.task_nsh.data(), out.task_nsh.size());
    for (int32_t g = 0; g < out.ngroups; ++g) B[out.grp_off + 36 * g + 34] += nsh_off * 4;     // byte offset inside the blob
}

static void build_item(const hines_plan& P, int64_t c0, int64_t c1, int32_t nchunks, ItemBuild& out)
{
    const int32_t smax = nchunks > 1 ? P.seg_cluster : P.seg_single;
    const int E = 16 / P.width;
    out = ItemBuild();
    out.nchunks = nchunks;
    out.comp_begin = P.cell_offsets[c0];
    out.n = P.cell_offsets[c1] - out.comp_begin;
    for (int64_t c = c0; c < c1; ++c) out.nlev = std::max(out.nlev, P.cell_nlevels[c]);
    const int64_t B0 = P.cell_branch_offsets[c0];
    const int32_t nb = (int32_t)(P.cell_branch_offsets[c1] - B0);
    std::vector<Br> br(nb);
    std::vector<std::vector<int32_t>> lv(out.nlev);
    for (int64_t c = c0; c < c1; ++c) {
        const int64_t b0 = P.cell_branch_offsets[c], b1 = P.cell_branch_offsets[c + 1];
        const int32_t shift = (int32_t)(P.cell_offsets[c] - out.comp_begin);
        for (int64_t j = b0; j < b1; ++j) {
            Br& e = br[j - B0];
            e.start = P.branch_start[j] + shift;
            e.len = P.branch_len[j];
            e.pc = P.branch_parent_comp[j] < 0 ? -1 : P.branch_parent_comp[j] + shift;
            e.level = P.branch_level[j];
            e.parent = P.branch_parent_branch[j] < 0 ? -1 : (int32_t)(b0 + P.branch_parent_branch[j] - B0);
            e.nseg = std::max<int32_t>(1, (int32_t)((5 * (int64_t)e.len + 2 * smax) / (5 * (int64_t)smax)));   // len/smax + 0.4, cut off
            e.sj = (e.len + e.nseg - 1) / e.nseg;
            if (e.nseg > 1 && e.sj % 2 == 0) ++e.sj;        // odd: the segments of one branch start on distinct banks
            e.nseg = (e.len + e.sj - 1) / e.sj;             // no empty segment
            if (e.nseg > 0xffff) out.ok = false;
            lv[e.level].push_back((int32_t)(j - B0));
        }
    }
    // ---- P3: nodes of the reduced tree ----------------------------------------------------------
    // Branches level by level, siblings contiguous, sibling groups by their longest member in segments,
    // descending, ties by (cell, branch id): the provisional node numbering from which
    // build_tasks derives the sweep (and the final numbering).
    std::vector<int32_t> lane_br;                       // branch of every lane, -1 = padding
    struct Group { int32_t first, count, maxseg, minord; };
    std::vector<Group> groups;
    for (int32_t l = 0; l < out.nlev; ++l) {
        auto& v = lv[l];
        auto key = [&](int32_t i) { return br[i].parent >= 0 ? (int64_t)br[i].parent : -(int64_t)i - 1; };
        std::sort(v.begin(), v.end(), [&](int32_t a, int32_t b) {
            if (key(a) != key(b)) return key(a) < key(b);
            if (br[a].nseg != br[b].nseg) return br[a].nseg > br[b].nseg;
            return a < b;
        });
        groups.clear();
        for (int32_t i = 0; i < (int32_t)v.size();) {
            int32_t j = i, mo = v[i];
            while (j < (int32_t)v.size() && key(v[j]) == key(v[i])) { mo = std::min(mo, v[j]); ++j; }
            groups.push_back({i, j - i, br[v[i]].nseg, mo});
            i = j;
        }
        std::sort(groups.begin(), groups.end(), [](const Group& a, const Group& b) {
            if (a.maxseg != b.maxseg) return a.maxseg > b.maxseg;
            return a.minord < b.minord;
        });
        for (const Group& g : groups)
            for (int32_t i = 0; i < g.count; ++i) {
                Br& e = br[v[g.first + i]];
                e.e = (int32_t)lane_br.size();
                lane_br.push_back(v[g.first + i]);
            }
    }
    out.ndesc = (int32_t)lane_br.size();
    int32_t next_id = out.ndesc;
    for (int32_t e = 0; e < out.ndesc; ++e) {
        if (lane_br[e] < 0) continue;
        Br& b = br[lane_br[e]];
        if (b.nseg > 1) { b.rest = next_id; next_id += b.nseg - 1; }
    }
    out.nnode = next_id;
    if (out.nnode >= (1 << 20)) out.ok = false;
    auto last_node = [&](const Br& b) { return b.nseg > 1 ? b.rest + b.nseg - 2 : b.e; };
    out.pnode.resize(out.nnode);
    std::iota(out.pnode.begin(), out.pnode.end(), 0);
    std::vector<int32_t> depth(out.nnode, 1);          // nodes on the path from the root, inclusive
    int32_t height = 1;
    for (int32_t e = 0; e < out.ndesc; ++e) {           // lanes are in level order: parents come first
        const Br& b = br[lane_br[e]];
        if (b.parent >= 0) { out.pnode[e] = last_node(br[b.parent]); depth[e] = depth[out.pnode[e]] + 1; }
        for (int32_t k = 1; k < b.nseg; ++k) {          // a root keeps itself as parent: its f is 0
            out.pnode[b.rest + k - 1] = k == 1 ? e : b.rest + k - 2;
            depth[b.rest + k - 1] = depth[e] + k;
        }
        height = std::max(height, depth[e] + b.nseg - 1);
    }
    (void)height;
    build_tasks(out, depth);                            // also sets out.rounds
    if (!out.ok) { out.perm.resize(out.nnode); std::iota(out.perm.begin(), out.perm.end(), 0); }
    // ---- P4: segments, in compartment order ------------------------------------------------------
    // Branch cut from its end into nseg segments of sj compartments (the paper's branch splitting,
    // PAPER.md:151, with a fixed bound); node ids from the top of the branch: e, rest, rest+1, ...
    std::vector<SegTmp> segs;                          // a item-local here
    segs.reserve(nb);
    for (int32_t i = 0; i < nb; ++i) {
        const Br& b = br[i];
        const int32_t end = b.start + b.len - 1;
        for (int32_t k = 0; k < b.nseg; ++k) {          // k-th segment from the top
            const int32_t q = b.nseg - 1 - k;           // counted from the branch's end
            const int32_t sb = end - q * b.sj;
            const int32_t sa = std::max(b.start, sb - b.sj + 1);
            const int32_t node = k == 0 ? b.e : b.rest + k - 1;
            const int32_t tnode = k > 0 ? (k == 1 ? b.e : b.rest + k - 2) : (b.parent >= 0 ? last_node(br[b.parent]) : -1);
            segs.push_back({sa, sb - sa, out.perm[node], tnode < 0 ? -1 : out.perm[tnode]});
            out.useful_steps += sb - sa;
        }
    }
    // ---- chunks: consecutive segments, balanced in shared-memory bytes -----------------------------
    const int64_t meta_item = (int64_t)out.task_blob.size() + round_up(out.nnode, 4);
    out.leader_extra = 6 * round_up(out.nnode, E) * P.width + 4 * meta_item;
    out.chunks.assign(nchunks, ItemBuild::Chunk());
    const int64_t per_comp = 3 * P.width, per_seg = 32;   // two lanes per segment
    const int64_t total = out.leader_extra + per_comp * out.n + per_seg * (int64_t)segs.size();
    out.total_bytes = total;
    size_t si = 0;
    int64_t acc = 0;
    std::vector<SegTmp> mine;
    for (int32_t r = 0; r < nchunks; ++r) {
        ItemBuild::Chunk& ch = out.chunks[r];
        const int64_t target = total * (r + 1) / nchunks;            // cumulative, so rounding does not pile up
        if (r == 0) acc = out.leader_extra;
        ch.begin = si < segs.size() ? segs[si].a : (int32_t)out.n;
        mine.clear();
        while (si < segs.size()) {
            const int64_t cost = per_comp * (segs[si].m + 1) + per_seg;
            const size_t left_chunks = (size_t)(nchunks - 1 - r);
            const bool must_take = mine.empty() && segs.size() - si > left_chunks;   // no empty chunk while segments remain
            const bool must_leave = segs.size() - si <= left_chunks;                   // keep one for every later chunk
            if (r == nchunks - 1 || must_take || (!must_leave && acc + cost / 2 <= target)) {
                mine.push_back(segs[si]); acc += cost; ++si;
            } else break;
        }
        ch.n = mine.empty() ? 0 : mine.back().a + mine.back().m + 1 - ch.begin;
        for (SegTmp& sg : mine) sg.a -= ch.begin;
        const int32_t off = (int32_t)((out.comp_begin + ch.begin) % E);
        // two lanes per segment: lane A eliminates the interior above the middle node q, lane B the interior
        // below it, both top-down (fill-in to t resp. q); A eliminates q last.  A warp holds
        // 16 segments: A lanes 0..15, their B partners 16..31 (partner = lane ^ 16).
        std::vector<int32_t> ord;
        order_segments(mine, 16, P.width == 8 ? 16 : 32, off, ord);
        while ((ord.size() / 4) % 16) ord.insert(ord.end(), {0, 0, -1, -1});
        const int32_t ngroups = (int32_t)(ord.size() / 64);
        ch.seg.assign((size_t)ngroups * 128, 0);
        for (int32_t gidx = 0; gidx < ngroups; ++gidx) {
            int32_t mx = 0;
            for (int32_t k = 0; k < 16; ++k) {
                const int32_t* sgp = &ord[(size_t)(gidx * 16 + k) * 4];
                int32_t* A = &ch.seg[(size_t)(gidx * 32 + k) * 4];
                int32_t* B = &ch.seg[(size_t)(gidx * 32 + 16 + k) * 4];
                const uint32_t ow = (uint32_t)sgp[1];
                const int32_t a = sgp[0], mm = (int32_t)(ow & 0xfff), node = sgp[2], tnode = sgp[3];
                if (node < 0) { A[2] = A[3] = B[2] = B[3] = -1; continue; }
                const int32_t hasq = mm > 0, mt = hasq ? std::min<int32_t>((ow >> 12) & 0xfff, mm - 1) : 0, mb = hasq ? mm - 1 - mt : 0;
                const int32_t dA = (int32_t)((ow >> 24) & 15), dB = (int32_t)(ow >> 28);
                const int32_t word = mt | (mb << 12) | (hasq << 26);
                A[0] = a; A[1] = word | (kSegA << 24) | (dA << 27); A[2] = node; A[3] = tnode;
                B[0] = a + mt + 1; B[1] = (int32_t)((uint32_t)word | ((uint32_t)kSegB << 24) | ((uint32_t)dB << 27)); B[2] = node; B[3] = -1;   // B starts below q = a + mt
                mx = std::max(mx, std::max(mt + dA, mb + dB));
            }
            out.padded_steps += 32 * (int64_t)(mx + 1);     // the loop steps of the warp + the step for q
        }
        const int32_t ns = (int32_t)(ch.seg.size() / 4);
        out.max_lanes = std::max(out.max_lanes, ns);
        const int64_t L = round_up(off + ch.n, E);
        ch.smem_need = 16 + (r == 0 ? out.leader_extra : 0) + 3 * L * P.width + 16 * (int64_t)ns;
        out.smem_need = std::max(out.smem_need, ch.smem_need);
    }
}

static hines_status_t canonical_tables(hines_plan& P, const int32_t* parent)
{
    const int64_t nc = P.ncells;
    P.cell_branch_offsets.assign(nc + 1, 0);
    P.cell_level_offsets.assign(nc + 1, 0);
    P.cell_nlevels.assign(nc, 0);
    std::vector<int32_t> nchild, branch_of, lens;
    std::vector<int32_t> order;
    P.max_levels = 0;
    P.breadth_first = 1;
    for (int64_t c = 0; c < nc; ++c) {
        const int64_t o = P.cell_offsets[c];
        const int32_t n = (int32_t)(P.cell_offsets[c + 1] - o);
        const int32_t* p = parent + o;
        if (p[0] != -1) {
            set_error("cell " + std::to_string(c) + ": parent of the first compartment is " +
                      std::to_string(p[0]) + ", expected -1 (global index " + std::to_string(o) + ")");
            return HINES_ERR_BAD_TOPOLOGY;
        }
        nchild.assign(n, 0);
        for (int32_t i = 1; i < n; ++i) {
            if (p[i] < 0 || p[i] >= i) {
                set_error("cell " + std::to_string(c) + ": parent[" + std::to_string(i) + "] = " +
                          std::to_string(p[i]) + " not in [0, " + std::to_string(i) + ") (global index " +
                          std::to_string(o + i) + ")");
                return HINES_ERR_BAD_TOPOLOGY;
            }
            nchild[p[i]]++;
        }
        // T1 (reading S4): a compartment continues its parent's branch only if it is the parent's
        // only child and is numbered right after it.
        branch_of.resize(n);
        const int64_t b0 = (int64_t)P.branch_start.size();
        for (int32_t i = 0; i < n; ++i) {
            const bool continues = i > 0 && p[i] == i - 1 && nchild[i - 1] == 1;
            if (!continues) { P.branch_start.push_back(i); P.branch_len.push_back(0); }
            branch_of[i] = (int32_t)(P.branch_start.size() - b0) - 1;
            P.branch_len.back()++;
        }
        const int32_t nbc = (int32_t)(P.branch_start.size() - b0);
        // T2-T4
        int32_t deepest = 0;
        for (int32_t j = 0; j < nbc; ++j) {
            const int32_t s = P.branch_start[b0 + j];
            int32_t pc = -1, pb = -1, lev = 0;
            if (s > 0) { pc = p[s]; pb = branch_of[pc]; lev = P.branch_level[b0 + pb] + 1; }
            P.branch_parent_comp.push_back(pc);
            P.branch_parent_branch.push_back(pb);
            if (j > 0 && lev < P.branch_level.back()) P.breadth_first = 0;
            P.branch_level.push_back(lev);
            deepest = std::max(deepest, lev);
        }
        // T5
        const int32_t nlev = deepest + 1;
        P.cell_nlevels[c] = nlev;
        P.max_levels = std::max(P.max_levels, nlev);
        const int64_t l0 = (int64_t)P.level_count.size();
        P.level_count.resize(l0 + nlev, 0);
        for (int32_t j = 0; j < nbc; ++j) P.level_count[l0 + P.branch_level[b0 + j]]++;
        P.cell_level_offsets[c + 1] = l0 + nlev;
        // T6 (reading S7): level ascending, length descending, id ascending
        order.resize(nbc);
        std::iota(order.begin(), order.end(), 0);
        const int32_t* lev = P.branch_level.data() + b0;
        const int32_t* len = P.branch_len.data() + b0;
        std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) {
            if (lev[a] != lev[b]) return lev[a] < lev[b];
            return len[a] > len[b];
        });
        P.level_list.insert(P.level_list.end(), order.begin(), order.end());
        P.cell_branch_offsets[c + 1] = b0 + nbc;
    }
    P.nbranches = (int64_t)P.branch_start.size();
    // T7
    P.child_offsets.assign(P.nbranches + 1, 0);
    P.child_ids.assign(P.nbranches - nc, 0);
    for (int64_t c = 0; c < nc; ++c) {
        const int64_t b0 = P.cell_branch_offsets[c], b1 = P.cell_branch_offsets[c + 1];
        for (int64_t j = b0 + 1; j < b1; ++j) P.child_offsets[b0 + P.branch_parent_branch[j] + 1]++;
    }
    for (int64_t j = 0; j < P.nbranches; ++j) P.child_offsets[j + 1] += P.child_offsets[j];
    {
        std::vector<int64_t> fill(P.child_offsets.begin(), P.child_offsets.end() - 1);
        for (int64_t c = 0; c < nc; ++c) {
            const int64_t b0 = P.cell_branch_offsets[c], b1 = P.cell_branch_offsets[c + 1];
            for (int64_t j = b0 + 1; j < b1; ++j)
                P.child_ids[fill[b0 + P.branch_parent_branch[j]]++] = (int32_t)(j - b0);
        }
    }
    return HINES_OK;
}

static void emit_item(hines_plan& P, int64_t c0, int64_t c1, const ItemBuild& ib)
{
    const int32_t item = (int32_t)P.item_class.size();
    for (int64_t c = c0; c < c1; ++c) P.cell_item[c] = item;
    P.item_cell_range.push_back(c0);
    P.item_cell_range.push_back(c1);
    P.item_class.push_back(0);                     // filled by assign_classes
    P.item_pnode.insert(P.item_pnode.end(), ib.pnode.begin(), ib.pnode.end());
    P.item_node_offsets.push_back((int64_t)P.item_pnode.size());
    P.item_rounds.push_back(ib.rounds);
    P.item_nnode.push_back(ib.nnode);
    P.item_task_blob.insert(P.item_task_blob.end(), ib.task_blob.begin(), ib.task_blob.end());
    P.item_task_offsets.push_back((int64_t)P.item_task_blob.size());
    // device blob of the item: [task blob | pnode | pad4]
    hines::ItemHeader h{};
    h.meta_off = (int64_t)P.item_meta.size();
    P.item_meta.insert(P.item_meta.end(), ib.task_blob.begin(), ib.task_blob.end());
    h.grp_off = ib.grp_off; h.ent_off = ib.ent_off; h.pull_off = ib.pull_off; h.ntier = ib.ntier;
    h.pnode_off = (int32_t)((int64_t)P.item_meta.size() - h.meta_off);
    P.item_meta.insert(P.item_meta.end(), ib.pnode.begin(), ib.pnode.end());
    P.item_meta.resize(round_up((int64_t)P.item_meta.size(), 4), 0);
    h.meta_len = (int32_t)((int64_t)P.item_meta.size() - h.meta_off);
    h.nnode = ib.nnode; h.rounds = ib.rounds;
    h.first_chunk = (int32_t)P.chunk_headers.size();
    h.nchunks = ib.nchunks;
    h.n = (int32_t)ib.n;
    P.item_headers.push_back(h);
    for (int32_t r = 0; r < ib.nchunks; ++r) {
        const ItemBuild::Chunk& ch = ib.chunks[r];
        hines::ChunkHeader k{};
        k.comp_begin = ib.comp_begin + ch.begin;
        k.n = ch.n;
        k.nseg_lanes = (int32_t)(ch.seg.size() / 4);
        k.item = item; k.rank = r;
        k.seg_off = (int64_t)P.item_meta.size();
        P.item_meta.insert(P.item_meta.end(), ch.seg.begin(), ch.seg.end());
        P.chunk_headers.push_back(k);
        P.chunk_comp_range.push_back(k.comp_begin);
        P.chunk_comp_range.push_back(k.comp_begin + k.n);
        P.chunk_seg.insert(P.chunk_seg.end(), ch.seg.begin(), ch.seg.end());
        P.chunk_seg_offsets.push_back((int64_t)P.chunk_seg.size() / 4);
    }
    P.item_chunk_offsets.push_back((int64_t)P.chunk_headers.size());
    P.padded_lane_steps += ib.padded_steps;
    P.useful_lane_steps += ib.useful_steps;
    if (ib.nchunks > 1) { P.n_cluster_cells += c1 - c0; P.n_cluster_unknowns += ib.n; }
    P.n_resident_cells += c1 - c0;
    P.n_resident_unknowns += ib.n;
}

struct ItemNeed { int64_t smem; int32_t lanes; int32_t nchunks; };

// P1 + P2: cells -> work items, greedy in input order.  A cell whose lists fit the
// group budget joins the open group while the group still fits; a cell that fits one block's budget
// gets its own item; a larger cell is spread over a cluster of 2, 4, 8 or 16 blocks ("long branches
// of large cells kept on their own blocks"); what fits nowhere goes to the streaming path.
static void pack_items(hines_plan& P, std::vector<ItemNeed>& need, std::vector<char>& is_stream)
{
    const int64_t nc = P.ncells;
    const int64_t max_smem = P.opt.smem_bytes_per_block;
    const int64_t group_cap = std::min<int64_t>(P.opt.group_smem_bytes, max_smem);
    const bool force_stream = P.opt.policy_flags & HINES_POLICY_FORCE_STREAM;
    const bool no_group = P.opt.policy_flags & HINES_POLICY_NO_GROUPING;
    const bool no_cluster = (P.opt.policy_flags & HINES_POLICY_NO_CLUSTER) || P.opt.cluster_max < 2;
    // a cell alone in a block may use up to single_cap; beyond that a cluster is preferred, because
    // blocks of at most chunk_smem_bytes leave room for a second resident block per SM
    const int64_t chunk_cap = std::min<int64_t>(P.opt.chunk_smem_bytes, max_smem);
    const int64_t single_cap = no_cluster ? max_smem : chunk_cap;
    const bool pow2_only = P.opt.policy_flags & HINES_POLICY_POW2_CLUSTERS;
    P.cell_item.assign(nc, -1);
    P.item_node_offsets.assign(1, 0);
    P.item_task_offsets.assign(1, 0);
    P.item_chunk_offsets.assign(1, 0);
    P.chunk_seg_offsets.assign(1, 0);
    is_stream.assign(nc, 0);
    ItemBuild cur, cand, alone;
    int64_t g0 = -1;                                   // first cell of the open group
    auto push = [&](int64_t a, int64_t b, const ItemBuild& ib) {
        emit_item(P, a, b, ib);
        need.push_back({ib.smem_need, ib.max_lanes, ib.nchunks});
    };
    auto flush = [&](int64_t c_end) { if (g0 >= 0) { push(g0, c_end, cur); g0 = -1; } };
    for (int64_t c = 0; c < nc; ++c) {
        const int64_t ncomp = P.cell_offsets[c + 1] - P.cell_offsets[c];
        bool placed = false, is_single = false;
        if (!force_stream) {
            const int64_t arrays = 16 + 3 * ncomp * P.width;             // lower bound of the need
            if (arrays <= single_cap) {
                build_item(P, c, c + 1, 1, alone);
                is_single = alone.ok && alone.smem_need <= single_cap;
            }
            if (!is_single && !no_cluster) {
                // cluster size: the one whose blocks fill their shared-memory slot best (slots = an SM's
                // shared memory divided by 1, 2, 3, 4, 6, 8); close calls go to the smaller cluster
                build_item(P, c, c + 1, 2, cand);
                if (cand.ok) {
                    const int64_t total = cand.total_bytes;
                    std::vector<std::pair<double, int32_t>> opts;                 // (-score, k)
                    for (int t = 1; t <= 3; ++t) {                                // slots of 1/2, 1/3, 1/4 of an SM
                        const int64_t slot = class_cap(kClassK[t], max_smem);
                        if (slot > chunk_cap) continue;
                        int32_t k = (int32_t)std::max<int64_t>(2, (total + slot - 2048 - 1) / (slot - 2048));
                        if (pow2_only) while (k & (k - 1)) ++k;
                        if (k > P.opt.cluster_max) continue;
                        opts.push_back({-((double)total / (double)(k * slot) - 0.01 * t), k});
                    }
                    if (opts.empty() && total / P.opt.cluster_max + 2048 <= max_smem) opts.push_back({0.0, P.opt.cluster_max});
                    std::sort(opts.begin(), opts.end());
                    for (size_t o = 0; o < opts.size() && o < 3 && !placed; ++o) {
                        const int32_t k = opts[o].second;
                        if (k != 2) build_item(P, c, c + 1, k, cand);
                        int64_t slot = 0;
                        for (int t = 0; t < kNumClassK; ++t) if (cand.smem_need <= class_cap(kClassK[t], chunk_cap)) slot = 1;
                        if (slot || (k == P.opt.cluster_max && cand.smem_need <= max_smem)) { flush(c); push(c, c + 1, cand); placed = true; }
                        else if (k == 2 && o + 1 < opts.size()) { /* rebuilt below for the next option */ }
                    }
                }
                if (!placed && arrays <= max_smem) {                      // last resort before streaming: one big block
                    build_item(P, c, c + 1, 1, alone);
                    is_single = alone.ok && alone.smem_need <= max_smem;
                }
            }
        }
        if (placed) continue;
        if (!is_single) { flush(c); is_stream[c] = 1; continue; }
        if (no_group || alone.smem_need > group_cap) { flush(c); push(c, c + 1, alone); continue; }
        if (g0 < 0) { g0 = c; std::swap(cur, alone); continue; }
        build_item(P, g0, c + 1, 1, cand);                                // greedy: does the next cell still fit?
        if (cand.ok && cand.smem_need <= group_cap) { std::swap(cur, cand); continue; }
        flush(c);
        g0 = c; std::swap(cur, alone);
    }
    flush(nc);
}

// Size classes.  By how many blocks of that size fit one SM (1, 2, 3, 4, 6, 8), separately for single-block
// items and for every cluster size.  Threads per block: enough lanes for the widest segment
// list of the class, within what the register file allows for that many resident blocks.
static void assign_classes(hines_plan& P, const std::vector<ItemNeed>& need)
{
    const int64_t nitems = (int64_t)need.size();
    const int64_t max_smem = P.opt.smem_bytes_per_block;
    const int nq = kNumClassK * (kMaxClusterClass + 2);   // single blocks, then per cluster size, each by blocks per SM
    std::vector<int> item_q(nitems, 0);
    std::vector<int64_t> need_max(nq, 0), count(nq, 0);
    std::vector<int32_t> lanes_max(nq, 0);
    for (int64_t i = 0; i < nitems; ++i) {
        int q = 0;
        for (int t = 0; t < kNumClassK; ++t) if (need[i].smem <= class_cap(kClassK[t], max_smem)) q = t;
        if (need[i].nchunks > 1) q += kNumClassK * need[i].nchunks;
        item_q[i] = q;
        need_max[q] = std::max(need_max[q], need[i].smem);
        lanes_max[q] = std::max(lanes_max[q], need[i].lanes);
        count[q]++;
    }
    // launch order of the classes: clusters first (largest first), then single blocks, biggest first
    std::vector<int> qs;
    for (int k = kMaxClusterClass; k >= 2; --k)
        for (int t = 0; t < kNumClassK; ++t) if (count[kNumClassK * k + t]) qs.push_back(kNumClassK * k + t);
    for (int q = 0; q < kNumClassK; ++q) if (count[q]) qs.push_back(q);
    std::vector<int> cls_of_q(nq, -1);
    for (int q : qs) {
        cls_of_q[q] = (int)P.class_smem_bytes.size();
        const int64_t smem = round_up(need_max[q], 128);
        P.class_smem_bytes.push_back((int32_t)smem);
        P.class_cluster.push_back(q >= kNumClassK ? q / kNumClassK : 1);
        const int64_t per_sm = std::max<int64_t>(1, kSmemPerSM / (smem + 1024));
        int64_t tmax = 65536 / (kRegsPerThread * per_sm) / 32 * 32;
        tmax = std::max<int64_t>(64, std::min<int64_t>(kMaxThreads, tmax));
        int64_t t = P.opt.threads_per_block ? P.opt.threads_per_block : round_up(std::max(lanes_max[q], 1), 32);
        t = std::max<int64_t>(P.opt.threads_per_block ? 32 : std::min<int64_t>(128, tmax), std::min(t, tmax));
        P.class_threads.push_back((int32_t)t);
    }
    for (int64_t i = 0; i < nitems; ++i) P.item_class[i] = cls_of_q[item_q[i]];
    const int ncls = (int)P.class_smem_bytes.size();
    P.class_first.assign(ncls, 0);
    P.class_count.assign(ncls, 0);
    P.item_launch_order.resize(nitems);
    std::iota(P.item_launch_order.begin(), P.item_launch_order.end(), 0);
    const bool input_order = P.opt.policy_flags & HINES_POLICY_INPUT_ORDER;
    std::stable_sort(P.item_launch_order.begin(), P.item_launch_order.end(), [&](int32_t a, int32_t b) {
        if (P.item_class[a] != P.item_class[b]) return P.item_class[a] < P.item_class[b];
        if (input_order) return false;
        return P.item_headers[a].n > P.item_headers[b].n;          // heaviest first
    });
    for (int64_t i = 0; i < nitems; ++i) P.class_count[P.item_class[P.item_launch_order[i]]]++;
    for (int q = 1; q < ncls; ++q) P.class_first[q] = P.class_first[q - 1] + P.class_count[q - 1];
}

static void build_stream(hines_plan& P, const std::vector<char>& is_stream)
{
    // workspace offsets of the streaming cells, in input order
    std::vector<int64_t> ws_off(P.ncells, -1);
    int64_t ws = 0; int32_t maxlev = 0;
    for (int64_t c = 0; c < P.ncells; ++c) {
        if (!is_stream[c]) continue;
        ws_off[c] = ws; ws += P.cell_offsets[c + 1] - P.cell_offsets[c];
        maxlev = std::max(maxlev, P.cell_nlevels[c]);
        P.n_stream_cells++;
    }
    P.n_stream_unknowns = ws;
    if (!P.n_stream_cells) { P.stream_level_begin.assign(1, 0); return; }
    struct SE { int64_t gbranch; int32_t len; };
    std::vector<std::vector<SE>> lv(maxlev);
    for (int64_t c = 0; c < P.ncells; ++c) {
        if (!is_stream[c]) continue;
        for (int64_t j = P.cell_branch_offsets[c]; j < P.cell_branch_offsets[c + 1]; ++j)
            lv[P.branch_level[j]].push_back({j, P.branch_len[j]});
    }
    // cell of a global branch id: walk cells alongside (branches are in cell order)
    std::vector<int32_t> cell_of_branch;   // only needed for stream branches; build lazily via search
    auto cell_of = [&](int64_t gb) {
        return (int64_t)(std::upper_bound(P.cell_branch_offsets.begin(), P.cell_branch_offsets.end(), gb) -
                         P.cell_branch_offsets.begin()) - 1;
    };
    P.stream_level_begin.assign(maxlev + 1, 0);
    for (int32_t l = 0; l < maxlev; ++l) {
        auto& v = lv[l];
        // whole-level order (reading S7 applied across the streaming cells): length descending, then id
        std::stable_sort(v.begin(), v.end(), [](const SE& a, const SE& b) { return a.len > b.len; });
        P.stream_level_begin[l] = (int64_t)P.stream_desc.size();
        for (size_t t = 0; t < v.size(); t += 32) P.padded_lane_steps += 32 * (int64_t)v[t].len;
        for (const SE& e : v) {
            const int64_t c = cell_of(e.gbranch);
            const int64_t o = P.cell_offsets[c], b0 = P.cell_branch_offsets[c];
            hines::StreamDesc s;
            s.gstart = (int32_t)(o + P.branch_start[e.gbranch]);
            s.len = e.len;
            s.gparent = P.branch_parent_comp[e.gbranch] < 0 ? -1 : (int32_t)(o + P.branch_parent_comp[e.gbranch]);
            s.ws = (int32_t)(ws_off[c] + P.branch_start[e.gbranch]);
            s.child_begin = (int32_t)(P.stream_child.size() / 2);
            s.nchild = (int32_t)(P.child_offsets[e.gbranch + 1] - P.child_offsets[e.gbranch]);
            for (int64_t k = P.child_offsets[e.gbranch]; k < P.child_offsets[e.gbranch + 1]; ++k) {
                const int64_t ch = b0 + P.child_ids[k];
                P.stream_child.push_back((int32_t)(o + P.branch_start[ch]));
                P.stream_child.push_back((int32_t)(ws_off[c] + P.branch_start[ch]));
            }
            P.stream_desc.push_back(s);
            P.useful_lane_steps += e.len;
        }
    }
    P.stream_level_begin[maxlev] = (int64_t)P.stream_desc.size();
}

}  // namespace hines

using namespace hines;

extern "C" {

hines_status_t hines_plan_create(const int32_t* parent, const int64_t* cell_offsets, int64_t ncells,
                                 hines_dtype_t dtype, const hines_options_t* opt, hines_plan_t** out_plan)
{
    if (out_plan) *out_plan = nullptr;
    if (!parent || !cell_offsets || !out_plan) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (ncells <= 0) { set_error("ncells must be positive"); return HINES_ERR_INVALID_ARG; }
    if (dtype != HINES_F64 && dtype != HINES_F32) { set_error("unknown dtype"); return HINES_ERR_INVALID_ARG; }
    hines_options_t o{};
    o.struct_size = (int32_t)sizeof(hines_options_t);
    if (opt) {
        if (opt->struct_size <= 0 || opt->struct_size > (int32_t)sizeof(hines_options_t)) {
            set_error("options: bad struct_size"); return HINES_ERR_INVALID_ARG;
        }
        std::memcpy(&o, opt, (size_t)opt->struct_size);
    }
    if (o.smem_bytes_per_block == 0) o.smem_bytes_per_block = (int32_t)kSmemMaxOptin;
    if (o.stream_threads == 0) o.stream_threads = 128;
    if (o.group_smem_bytes == 0) o.group_smem_bytes = 57344;
    const bool auto_segment = o.max_segment == 0;     // default: 40 in a block of its own, 64 in the blocks of a cluster
    if (auto_segment) o.max_segment = 64;
    if (o.cluster_max == 0) o.cluster_max = 16;
    if (o.chunk_smem_bytes == 0) o.chunk_smem_bytes = 113 * 1024;
    if (o.threads_per_block < 0 || o.threads_per_block > kMaxThreads || o.threads_per_block % 32 ||
        o.stream_threads < 32 || o.stream_threads > 1024 || o.stream_threads % 32 ||
        o.smem_bytes_per_block < 1024 || o.smem_bytes_per_block > kSmemMaxOptin || o.group_smem_bytes < 0 ||
        o.max_segment < 2 || o.max_segment > 1023 || (o.policy_flags & ~63) ||
        o.cluster_max < 1 || o.cluster_max > 16 || o.chunk_smem_bytes < 1024) {
        set_error("options: value out of range"); return HINES_ERR_INVALID_ARG;
    }
    if (cell_offsets[0] != 0) { set_error("cell_offsets[0] must be 0"); return HINES_ERR_BAD_TOPOLOGY; }
    for (int64_t c = 0; c < ncells; ++c)
        if (cell_offsets[c + 1] <= cell_offsets[c]) {
            set_error("cell_offsets not strictly increasing at cell " + std::to_string(c) + " (empty cells are rejected)");
            return HINES_ERR_BAD_TOPOLOGY;
        }
    if (cell_offsets[ncells] >= (int64_t)1 << 31) { set_error("N >= 2^31 is not supported"); return HINES_ERR_INVALID_ARG; }
    try {
        hines_plan* P = new hines_plan();
        P->n = cell_offsets[ncells]; P->ncells = ncells; P->dtype = dtype; P->width = dtype == HINES_F64 ? 8 : 4;
        P->opt = o;
        P->seg_cluster = o.max_segment;
        P->seg_single = auto_segment ? 40 : o.max_segment;
        P->cell_offsets.assign(cell_offsets, cell_offsets + ncells + 1);
        hines_status_t st = canonical_tables(*P, parent);
        if (st != HINES_OK) { delete P; return st; }
        std::vector<ItemNeed> item_need;
        std::vector<char> is_stream;
        pack_items(*P, item_need, is_stream);
        assign_classes(*P, item_need);
        build_stream(*P, is_stream);
        *out_plan = P;
        return HINES_OK;
    } catch (const std::bad_alloc&) {
        set_error("host allocation failed while building the plan"); return HINES_ERR_ALLOC;
    } catch (const std::exception& e) {
        set_error(std::string("internal error: ") + e.what()); return HINES_ERR_ALLOC;
    }
}

hines_status_t hines_plan_get_info(const hines_plan_t* P, hines_plan_info_t* out)
{
    if (!P || !out) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    std::memset(out, 0, sizeof(*out));
    out->n = P->n; out->ncells = P->ncells; out->nbranches = P->nbranches;
    out->max_levels = P->max_levels; out->dtype = P->dtype;
    out->n_resident_items = (int64_t)P->item_class.size();
    out->n_resident_cells = P->n_resident_cells; out->n_resident_unknowns = P->n_resident_unknowns;
    out->n_stream_cells = P->n_stream_cells; out->n_stream_unknowns = P->n_stream_unknowns;
    out->n_stream_branches = (int64_t)P->stream_desc.size();
    out->padded_lane_steps = P->padded_lane_steps; out->useful_lane_steps = P->useful_lane_steps;
    out->workspace_bytes = (int64_t)(P->item_meta.size() * 4 + P->item_headers.size() * sizeof(ItemHeader) +
                                     P->chunk_headers.size() * sizeof(ChunkHeader) +
                                     P->item_launch_order.size() * 4 + P->stream_desc.size() * sizeof(StreamDesc) +
                                     P->stream_child.size() * 4 + 2 * P->n_stream_unknowns * P->width);
    out->bytes_min = P->n * 4 * P->width + 4 * P->nbranches;
    out->bytes_literal = P->n * (4 * P->width + 4);
    out->breadth_first = P->breadth_first;
    out->n_classes = (int32_t)P->class_smem_bytes.size();
    out->n_cluster_cells = P->n_cluster_cells; out->n_cluster_unknowns = P->n_cluster_unknowns;
    out->n_chunks = (int64_t)P->chunk_headers.size();
    return HINES_OK;
}

hines_status_t hines_plan_get_table(const hines_plan_t* P, int32_t id, void* dst, int64_t cap, int64_t* needed)
{
    if (!P || !needed) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    const void* src = nullptr; int64_t bytes = 0;
#define TBL(ID, V) case ID: src = (V).data(); bytes = (int64_t)((V).size() * sizeof((V)[0])); break;
    switch (id) {
        TBL(HINES_TABLE_CELL_BRANCH_OFFSETS, P->cell_branch_offsets)
        TBL(HINES_TABLE_BRANCH_START, P->branch_start)
        TBL(HINES_TABLE_BRANCH_LEN, P->branch_len)
        TBL(HINES_TABLE_BRANCH_PARENT_COMP, P->branch_parent_comp)
        TBL(HINES_TABLE_BRANCH_PARENT_BRANCH, P->branch_parent_branch)
        TBL(HINES_TABLE_BRANCH_LEVEL, P->branch_level)
        TBL(HINES_TABLE_CELL_NLEVELS, P->cell_nlevels)
        TBL(HINES_TABLE_CELL_LEVEL_OFFSETS, P->cell_level_offsets)
        TBL(HINES_TABLE_LEVEL_COUNT, P->level_count)
        TBL(HINES_TABLE_LEVEL_LIST, P->level_list)
        TBL(HINES_TABLE_CHILD_OFFSETS, P->child_offsets)
        TBL(HINES_TABLE_CHILD_IDS, P->child_ids)
        TBL(HINES_TABLE_CELL_ITEM, P->cell_item)
        TBL(HINES_TABLE_ITEM_CELL_RANGE, P->item_cell_range)
        TBL(HINES_TABLE_ITEM_CLASS, P->item_class)
        TBL(HINES_TABLE_ITEM_LAUNCH_ORDER, P->item_launch_order)
        TBL(HINES_TABLE_ITEM_PNODE, P->item_pnode)
        TBL(HINES_TABLE_ITEM_NODE_OFFSETS, P->item_node_offsets)
        TBL(HINES_TABLE_ITEM_ROUNDS, P->item_rounds)
        TBL(HINES_TABLE_ITEM_TASK_OFFSETS, P->item_task_offsets)
        TBL(HINES_TABLE_ITEM_TASK_BLOB, P->item_task_blob)
        TBL(HINES_TABLE_ITEM_NNODE, P->item_nnode)
        TBL(HINES_TABLE_ITEM_CHUNK_OFFSETS, P->item_chunk_offsets)
        TBL(HINES_TABLE_CHUNK_COMP_RANGE, P->chunk_comp_range)
        TBL(HINES_TABLE_CHUNK_SEG_OFFSETS, P->chunk_seg_offsets)
        TBL(HINES_TABLE_CHUNK_SEG, P->chunk_seg)
        TBL(HINES_TABLE_CLASS_CLUSTER, P->class_cluster)
        TBL(HINES_TABLE_CLASS_THREADS, P->class_threads)
        TBL(HINES_TABLE_STREAM_LEVEL_BEGIN, P->stream_level_begin)
        TBL(HINES_TABLE_STREAM_DESC, P->stream_desc)
        TBL(HINES_TABLE_STREAM_CHILD, P->stream_child)
        TBL(HINES_TABLE_CLASS_SMEM_BYTES, P->class_smem_bytes)
        default: set_error("unknown table id " + std::to_string(id)); return HINES_ERR_INVALID_ARG;
    }
#undef TBL
    *needed = bytes;
    if (!dst) return HINES_OK;
    if (cap < bytes) { set_error("table buffer too small"); return HINES_ERR_INVALID_ARG; }
    if (bytes) std::memcpy(dst, src, (size_t)bytes);
    return HINES_OK;
}

hines_status_t hines_plan_launches_per_solve(const hines_plan_t* P, int32_t* out)
{
    if (!P || !out) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    *out = (int32_t)P->class_smem_bytes.size() + 2 * (int32_t)(P->stream_level_begin.size() - 1);
    return HINES_OK;
}

const char* hines_status_string(hines_status_t s)
{
    switch (s) {
        case HINES_OK: return "ok";
        case HINES_ERR_INVALID_ARG: return "invalid argument";
        case HINES_ERR_BAD_TOPOLOGY: return "bad topology";
        case HINES_ERR_ALLOC: return "allocation failed";
        case HINES_ERR_CUDA: return "CUDA error";
        case HINES_ERR_UNSUPPORTED: return "unsupported";
    }
    return "unknown status";
}

const char* hines_last_error(void) { return g_last_error.c_str(); }
const char* hines_version(void) { return "hines-b200 0.1 (sm_100a)"; }

}  // extern "C"

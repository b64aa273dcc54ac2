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
//          a level's node list and is limited by its 227 KB of shared memory, not its thread count.
//          A cell too large for one block is cut into PARTS made of whole branches: a top part (the
//          root region) and parts that are unions of complete sub-trees, balanced in bytes.  The parts
//          are held by the blocks of one thread-block cluster (the paper requires one matrix per block,
//          PAPER.md:114; distributed shared memory lifts that), or, beyond the largest cluster, run as
//          three dependent launches (sub-trees backward / top / sub-trees forward).  With breadth-first
//          branch numbering a complete sub-tree is ONE run of consecutive compartments per
//          level, so a part is a short list of runs, each moved by bulk copies.
//   P3     the reduced forest of a part (one node per segment), numbered level by level with the children
//          of a node consecutive: the backward sweep is the paper's level-synchronous sweep
//          over these nodes, a node pulling its children's hand-off values.
//   P4     segments.  Every branch is cut, from its end, into nseg = max(1, floor(len / max_segment + 0.4))
//          segments of ceil(len / nseg) compartments, one more if that is even and nseg > 1 (the paper's
//          branch splitting, with a fixed bound), or, with HINES_POLICY_SPLIT_LEVEL_MEAN,
//          first by the paper's own rule (per level, cut what is longer than the level's mean).
//          The last compartment of a segment is its separator; the compartments above it are its interior.
//          Interiors are eliminated independently of the tree level (two lanes per segment, all segments of
//          the part at once), which leaves the level-synchronous sweeps with one node per segment.  The
//          segment lane list is ordered so that the 16 (fp64) / 32 (fp32) lanes that access shared memory
//          together start at different bank residues and have similar lengths.
// Written policy: DESIGN.md "Scheduler policy".
#include <algorithm>
#include <cmath>
#include <cstring>
#include <memory>
#include <new>
#include <numeric>
#include <string>

#include "plan_internal.h"

namespace hines {

static thread_local std::string g_last_error;
void set_error(const std::string& msg) { g_last_error = msg; }

static const int64_t kSmemPerSM = 233472;       // 228 KiB
static const int64_t kSmemMaxOptin = 232448;    // 227 KiB
// size classes: shares of an SM's shared memory a block may take (num/den): the whole SM, 3/4 and 2/3 (such a block
// shares its SM with a block of another, smaller class launched beside it), then 2, 3, 4, 6, 8 blocks per SM
static const int kSlotNum[] = {1, 3, 2, 1, 1, 1, 1, 1};
static const int kSlotDen[] = {1, 4, 3, 2, 3, 4, 6, 8};
static const int kNumClassK = 8;
static const int kRegsPerThread = 80;           // fp64 instantiations of the resident kernel use 63-76 registers (allocated in eights)
static const int kRegsPerThreadF32 = 64;        // fp32 instantiations: 54-60
static const int kMaxThreads = 768;
static const int kMaxClusterClass = 16;
static const int32_t kSegA = 1, kSegB = 2;          // segment lane kinds (descriptor word 1, bits 24-25)

static inline int64_t round_up(int64_t v, int64_t m) { return (v + m - 1) / m * m; }

static int64_t class_cap(int t, int64_t max_smem)
{
    int64_t cap = (kSmemPerSM * kSlotNum[t] / kSlotDen[t] - 1024) / 128 * 128;
    return std::min(cap, max_smem);
}

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

// One branch of the item while its lists are built.
struct Br {
    int32_t start, len, pc, level, parent;   // item-local positions; parent = index into the item's branch array
    int32_t nseg = 1;                        // segments (pieces) of the branch
    int32_t piece0 = 0;                      // first of its piece lengths (top-down) in the item's piece list
    int32_t node0 = 0;                       // provisional id of its top node: nodes node0 .. node0+nseg-1, top-down
    int32_t part = 0;
    int32_t soff = 0;                        // staged (shared-memory) index of its first compartment
};

// Tables of one part (policies P3 + P4).
using hines::SplitPiece;

struct PartBuild {
    std::vector<int32_t> runs;               // 4 per run {item-local first compartment, length, staged index, 0}
    int32_t L = 0, n = 0, tx_elems = 0;
    int32_t nnode = 0, nlevnode = 0, nlev = 0, rounds = 0, nexp = 0, nghost = 0, nlanes = 0, flags = 0, ntoplev = 0, lowlev = 0, maxwidth = 0;
    std::vector<int32_t> lb, kp, exps, ghosts, seg;
    int64_t smem_need = 0;
};

// Lists of one work item: cells [c0,c1).
struct ItemBuild {
    int64_t comp_begin = 0, n = 0;
    int32_t kind = kItemSingle;
    bool ok = true;                          // false: does not fit the descriptor fields / the shared memory -> next option
    std::vector<PartBuild> parts;
    int32_t nxch = 0;                        // exchange slots (= exported sub-tree roots)
    int32_t nnode = 0;
    int64_t padded_steps = 0, useful_steps = 0;
    int64_t smem_need = 0;                   // max over the parts (split items: over the sub-tree parts)
    int64_t smem_top = 0;                    // split items: the top part
    int64_t total_bytes = 0;                 // estimate of the shared memory of the whole item, all parts together
    int32_t max_lanes = 0, max_lanes_top = 0;
    int32_t has_quads = 0;                   // some part has four-lane segment groups
    std::vector<SplitPiece> split;           // f4 (block means): the pieces of the item's branches under ITS level means
};

// Pieces of a branch under the fixed-bound rule (P4), top-down: nseg = max(1, floor(len/S + 0.4)) pieces of
// ceil(len/nseg) compartments (one more if that is even and nseg > 1), cut from the branch's END, so the
// first (top) piece takes what is left.
static void fixed_bound_pieces(int32_t len, int32_t smax, std::vector<int32_t>& out)
{
    int32_t nseg = std::max<int32_t>(1, (int32_t)((5 * (int64_t)len + 2 * smax) / (5 * (int64_t)smax)));   // len/smax + 0.4, cut off
    int32_t sj = (len + nseg - 1) / nseg;
    if (nseg > 1 && sj % 2 == 0) ++sj;       // odd: the segments of one branch start on distinct banks
    nseg = (len + sj - 1) / sj;              // no empty segment
    out.push_back(len - (nseg - 1) * sj);
    for (int32_t k = 1; k < nseg; ++k) out.push_back(sj);
}

struct NodeTmp { int32_t depth, pkey, gid, ghost; };
static void split_cells(const hines_plan& P, const std::vector<int64_t>& cells, std::vector<SplitPiece>& out, std::vector<int64_t>* stat);

// kind = single: the given cells (ascending, not necessarily adjacent) in one part.  kind = cluster: ONE cell in K parts, part 0 = top + sub-trees.
// kind = split: ONE cell, part 0 = top alone, the sub-trees packed into parts of at most `slot` bytes (K is
// then the result).
static void build_item(const hines_plan& P, const std::vector<int64_t>& cells, int32_t kind, int32_t K, int64_t slot, ItemBuild& out)
{
    const int32_t w = P.width, E = 16 / w;
    const int32_t smax = kind == kItemSingle ? P.seg_single : P.seg_cluster;
    const bool level_mean = (P.opt.policy_flags & HINES_POLICY_SPLIT_LEVEL_MEAN) != 0;
    const bool block_mean = !level_mean && (P.opt.policy_flags & HINES_POLICY_SPLIT_BLOCK_MEAN) != 0;
    const int32_t narr = (P.opt.policy_flags & HINES_POLICY_FACTORED) ? 4 : 3;     // staged arrays: d,u,b, or the three factors + b
    out = ItemBuild();
    out.kind = kind;
    out.comp_begin = P.cell_offsets[cells.front()];
    int32_t nb = 0;
    for (int64_t c : cells) { nb += (int32_t)(P.cell_branch_offsets[c + 1] - P.cell_branch_offsets[c]); out.n += P.cell_offsets[c + 1] - P.cell_offsets[c]; }
    std::vector<Br> br(nb);
    std::vector<int32_t> pieces;
    pieces.reserve(nb + nb / 4);
    // f4: the level means of THIS block's cells (the intermediate packing has chosen them); pieces by local branch
    std::vector<int32_t> bm_off, bm_len;
    if (block_mean) {
        split_cells(P, cells, out.split, nullptr);
        std::vector<int64_t> cb0;                                       // first global branch of each cell, and its local index
        std::vector<int32_t> cl0;
        int32_t acc = 0;
        for (int64_t c : cells) { cb0.push_back(P.cell_branch_offsets[c]); cl0.push_back(acc); acc += (int32_t)(P.cell_branch_offsets[c + 1] - P.cell_branch_offsets[c]); }
        auto local_of = [&](int64_t j) { const size_t k = (size_t)(std::upper_bound(cb0.begin(), cb0.end(), j) - cb0.begin()) - 1; return cl0[k] + (int32_t)(j - cb0[k]); };
        bm_off.assign((size_t)nb + 1, 0);
        for (const SplitPiece& sp : out.split) ++bm_off[(size_t)local_of(sp.j) + 1];
        for (int32_t k = 0; k < nb; ++k) bm_off[(size_t)k + 1] += bm_off[(size_t)k];
        bm_len.assign(out.split.size(), 0);
        std::vector<int32_t> fill(bm_off.begin(), bm_off.end() - 1);
        for (const SplitPiece& sp : out.split) bm_len[(size_t)fill[(size_t)local_of(sp.j)]++] = sp.len;      // top-down within a branch
    }
    int32_t nn = 0, lb0 = 0;
    for (int64_t c : cells) {
        const int64_t b0 = P.cell_branch_offsets[c], b1 = P.cell_branch_offsets[c + 1];
        const int64_t shift64 = P.cell_offsets[c] - out.comp_begin;
        const int32_t shift = (int32_t)shift64;
        for (int64_t j = b0; j < b1; ++j) {
            Br& e = br[lb0 + (j - b0)];
            e.start = P.branch_start[j] + shift;
            e.len = P.branch_len[j];
            e.pc = P.branch_parent_comp[j] < 0 ? -1 : P.branch_parent_comp[j] + shift;
            e.level = P.branch_level[j];
            e.parent = P.branch_parent_branch[j] < 0 ? -1 : lb0 + P.branch_parent_branch[j];
            e.piece0 = (int32_t)pieces.size();
            if (level_mean) {                           // the paper's pieces first, each then bounded
                for (int64_t q = P.split_piece_offsets[j]; q < P.split_piece_offsets[j + 1]; ++q)
                    fixed_bound_pieces(P.split_piece_len[q], smax, pieces);
            } else if (block_mean) {
                const int32_t lj = lb0 + (int32_t)(j - b0);
                for (int32_t q = bm_off[(size_t)lj]; q < bm_off[(size_t)lj + 1]; ++q) fixed_bound_pieces(bm_len[(size_t)q], smax, pieces);
            } else {
                fixed_bound_pieces(e.len, smax, pieces);
            }
            e.nseg = (int32_t)pieces.size() - e.piece0;
            if (e.nseg > 0xffff) out.ok = false;
            e.node0 = nn;
            nn += e.nseg;
        }
        lb0 += (int32_t)(b1 - b0);
    }
    out.nnode = nn;
    if (nn >= (1 << 20)) { out.ok = false; return; }
    // ---- nodes of the reduced forest: one per segment; (branch, k) -> node0 + k, top-down ------------------
    std::vector<int32_t> nparent(nn), ndepth(nn), nbr(nn);
    for (int32_t b = 0; b < nb; ++b) {                  // parents come first (parent_branch < branch)
        const Br& e = br[b];
        const int32_t pn = e.parent >= 0 ? br[e.parent].node0 + br[e.parent].nseg - 1 : -1;
        for (int32_t k = 0; k < e.nseg; ++k) {
            const int32_t g = e.node0 + k;
            nparent[g] = k == 0 ? pn : g - 1;
            ndepth[g] = nparent[g] < 0 ? 0 : ndepth[nparent[g]] + 1;
            nbr[g] = b;
        }
    }
    // ---- parts ----------------------------------------------------------------------------------------------
    const int64_t per_node = 6 * w + 32 + 8;            // record + two segment lanes + {kids, parent}
    std::vector<int64_t> bytes(nb), sub(nb);
    int64_t total = 0;
    for (int32_t b = 0; b < nb; ++b) { bytes[b] = narr * (int64_t)w * br[b].len + per_node * br[b].nseg; total += bytes[b]; }
    out.total_bytes = total + 1024;
    int32_t nparts = 1;
    if (kind != kItemSingle) {
        // Frontier of sub-trees: walking down from the root, a sub-tree heavier than Tsub gives its root branch
        // to the top and is replaced by its children's sub-trees.  Frontier roots in branch order (= breadth-first
        // order: neighbours share runs) are dealt to the parts in sequence, balanced in bytes.
        sub = bytes;
        for (int32_t b = nb - 1; b > 0; --b) if (br[b].parent >= 0) sub[br[b].parent] += sub[b];
        std::vector<int32_t> root_of(nb, -2), best_root, part_of_root(nb, 0), best_part;   // root_of: -2 = top, else its frontier root
        std::vector<int32_t> frontier;
        std::vector<int64_t> load;
        int64_t best_max = -1; int32_t best_nparts = 1;
        // cluster items: the finer the frontier, the better the parts balance but the heavier the top (all in part 0):
        // several thresholds are tried and the one with the lightest heaviest part is kept
        const int ntry = kind == kItemCluster ? 4 : 1;
        for (int t = 0; t < ntry; ++t) {
            static const int kNum[4] = {1, 1, 1, 2}, kDen[4] = {4, 3, 2, 3};
            const int64_t Tsub = kind == kItemCluster ? std::max<int64_t>(total * kNum[t] / (kDen[t] * (int64_t)K), 2048)
                                                      : std::max<int64_t>(slot * (K > 0 ? K : 80) / 100, 2048);   // split items: K = percent of the slot
            frontier.clear();
            int64_t top_bytes = 0;
            for (int32_t b = 0; b < nb; ++b) {
                if (br[b].parent < 0 || root_of[br[b].parent] == -2) {
                    if (sub[b] > Tsub) { root_of[b] = -2; top_bytes += bytes[b]; }
                    else { root_of[b] = b; frontier.push_back(b); }
                } else root_of[b] = root_of[br[b].parent];
            }
            int32_t np = 1;
            if (kind == kItemCluster) {
                np = K;
                load.assign(K, 0); load[0] = top_bytes;
                // from the last frontier root to the first: part 0, which also carries the top and sweeps it after the
                // exchange, gets the sub-trees rooted deepest (the fewest levels of its own to sweep before that)
                int64_t acc = top_bytes; int32_t r = 0;
                for (size_t q = frontier.size(); q-- > 0;) {
                    const int32_t f = frontier[q];
                    while (r < K - 1 && acc + sub[f] / 2 > total * (r + 1) / K) ++r;
                    part_of_root[f] = r; acc += sub[f]; load[r] += sub[f];
                }
            } else {
                int32_t r = 1; int64_t acc = 0;
                load.assign(1, top_bytes);
                for (int32_t f : frontier) {
                    if (acc > 0 && acc + sub[f] > slot) { ++r; acc = 0; }
                    part_of_root[f] = r; acc += sub[f];
                }
                np = frontier.empty() ? 1 : r + 1;
                if (np > 65535) { out.ok = false; return; }
            }
            const int64_t mx = *std::max_element(load.begin(), load.end());
            if (best_max < 0 || mx < best_max) { best_max = mx; best_root = root_of; best_part = part_of_root; best_nparts = np; }
        }
        nparts = best_nparts;
        root_of.swap(best_root); part_of_root.swap(best_part);
        for (int32_t b = 0; b < nb; ++b) br[b].part = root_of[b] == -2 ? 0 : part_of_root[root_of[b]];
    }
    out.parts.assign(nparts, PartBuild());
    // exported sub-tree roots (branches whose parent branch lies in another part, which must be part 0)
    std::vector<int32_t> g0_of_branch, p0_of_branch, x_of_branch, gp_of_branch;
    if (nparts > 1) {
        g0_of_branch.assign(nb, -1); p0_of_branch.assign(nb, -1); x_of_branch.assign(nb, -1); gp_of_branch.assign(nb, -1);
        for (int32_t b = 0; b < nb; ++b)
            if (br[b].parent >= 0 && br[br[b].parent].part != br[b].part && br[br[b].parent].part != 0) { out.ok = false; return; }
    }
    std::vector<int32_t> lmap(nn, -1);                  // provisional node id -> local id in the part being built
    std::vector<std::vector<int32_t>> part_br(nparts);
    for (int32_t b = 0; b < nb; ++b) part_br[br[b].part].push_back(b);
    std::vector<NodeTmp> nodes;
    std::vector<SegTmp> segs;
    std::vector<int32_t> ord, first, cnt, dist;
    for (int32_t p = 0; p < nparts; ++p) {
        PartBuild& pb = out.parts[p];
        const std::vector<int32_t>& mine = part_br[p];
        // ---- runs of consecutive compartments, staged one after the other; the staged index of a run has the
        //      parity of its global index, so that the 16-byte words of both sides coincide (bulk copies) ----
        int64_t cursor = 0;
        for (size_t i = 0; i < mine.size();) {
            size_t j = i; int32_t end = br[mine[i]].start;
            while (j < mine.size() && br[mine[j]].start == end) { end += br[mine[j]].len; ++j; }
            const int32_t start = br[mine[i]].start, len = end - start;
            const int64_t g = out.comp_begin + start;
            const int64_t so = round_up(cursor, E) + g % E;
            if (so + len >= ((int64_t)1 << 30)) { out.ok = false; return; }
            pb.runs.insert(pb.runs.end(), {start, len, (int32_t)so, 0});
            for (size_t k = i; k < j; ++k) br[mine[k]].soff = (int32_t)(so + br[mine[k]].start - start);
            cursor = so + len;
            const int64_t ga = g - g % E, ge = std::min<int64_t>(round_up(g + len, E), P.n / E * E);
            if (ge > ga) pb.tx_elems += (int32_t)(ge - ga);
            pb.n += len;
            i = j;
        }
        pb.L = (int32_t)round_up(cursor, E);
        // ---- P3: the part's reduced forest, level by level, children of a node consecutive --------------------
        nodes.clear();
        for (int32_t b : mine) for (int32_t k = 0; k < br[b].nseg; ++k) nodes.push_back({ndepth[br[b].node0 + k], -1, br[b].node0 + k, 0});
        if (p == 0 && nparts > 1)
            for (int32_t b = 0; b < nb; ++b)
                if (br[b].part != 0 && br[b].parent >= 0 && br[br[b].parent].part == 0) nodes.push_back({ndepth[br[b].node0], -1, br[b].node0, 1});
        std::stable_sort(nodes.begin(), nodes.end(), [](const NodeTmp& x, const NodeTmp& y) { return x.depth < y.depth; });
        pb.lb.assign(1, 0);
        int32_t next = 0;
        for (size_t i = 0; i < nodes.size();) {
            size_t j = i;
            while (j < nodes.size() && nodes[j].depth == nodes[i].depth) ++j;
            for (size_t k = i; k < j; ++k) {
                const int32_t pg = nparent[nodes[k].gid];
                nodes[k].pkey = pg >= 0 ? lmap[pg] : -1;                     // -1: root of the cell, or parent outside the part
            }
            std::sort(nodes.begin() + i, nodes.begin() + j, [](const NodeTmp& x, const NodeTmp& y) {
                return x.pkey != y.pkey ? x.pkey < y.pkey : x.gid < y.gid; });
            for (size_t k = i; k < j; ++k) {
                if (nodes[k].ghost) g0_of_branch[nbr[nodes[k].gid]] = next; else lmap[nodes[k].gid] = next;
                ++next;
            }
            pb.lb.push_back(next);
            i = j;
        }
        pb.nlev = (int32_t)pb.lb.size() - 1;
        pb.nlevnode = next;
        first.assign(next, 0); cnt.assign(next, 0);
        for (int32_t v = 0; v < next; ++v)
            if (nodes[v].pkey >= 0) { if (!cnt[nodes[v].pkey]) first[nodes[v].pkey] = v; ++cnt[nodes[v].pkey]; }
        // every cell of the part an unbranched cable of at most 32 nodes: the reduced systems are solved by
        // parallel cyclic reduction, one warp per cable; nodes are then numbered cable by cable (lb[] = first
        // node of each cable) instead of level by level
        bool chains = kind == kItemSingle && next > 0 && mine.size() == cells.size();
        if (chains) for (int32_t b : mine) if (br[b].nseg > 32 || br[b].parent >= 0) chains = false;
        if (chains && !(P.opt.policy_flags & (HINES_POLICY_NO_PCR | HINES_POLICY_FACTORED))) {
            pb.flags |= kPartFlagChains;
            pb.lb.assign(1, 0);
            int32_t id = 0;
            for (int32_t b : mine) {
                for (int32_t k = 0; k < br[b].nseg; ++k) lmap[br[b].node0 + k] = id++;
                pb.lb.push_back(id);
            }
            pb.nlev = (int32_t)mine.size();
            pb.kp.assign(4 * (size_t)next, 0);
            for (int32_t b : mine)
                for (int32_t k = 0; k < br[b].nseg; ++k) {
                    const int32_t v = lmap[br[b].node0 + k];
                    pb.kp[4 * v + 2] = k + 1 < br[b].nseg ? 1 : 0;
                    pb.kp[4 * v + 3] = k > 0 ? v - 1 : v;
                }
            pb.nnode = next; pb.rounds = 0; pb.ntoplev = 0; pb.lowlev = 0; pb.maxwidth = 0;
        } else {
        // per node {slot0, slot1, info, pnode}: slot0/slot1 = byte offsets (in the record array) of the hand-off
        // slots of its first two children, or of the all-zero record behind the last node; info = children |
        // top << 29, or -1 for a ghost child; pnode = the node the forward sweep reads
        const int32_t RSb = 6 * w, zero_slot = 0;             // the zero record sits at index nnode: patched below
        (void)zero_slot;
        pb.kp.assign(4 * (size_t)next, 0);
        dist.assign(next, 0);
        int32_t maxdist = 0;
        for (int32_t v = 0; v < next; ++v) {
            const NodeTmp& nt = nodes[v];
            int32_t pn = v;
            if (nt.ghost) {
                pb.kp[4 * v + 2] = -1;
                p0_of_branch[nbr[nt.gid]] = nt.pkey;
                x_of_branch[nbr[nt.gid]] = pb.nghost;
                pb.ghosts.insert(pb.ghosts.end(), {v, pb.nghost, nt.pkey, 0});
                ++pb.nghost;
            } else {
                if (cnt[v] > 4095) { out.ok = false; return; }
                pb.kp[4 * v] = cnt[v] > 0 ? first[v] : -1;             // node index for now, byte offset below
                pb.kp[4 * v + 1] = cnt[v] > 1 ? first[v] + 1 : -1;
                pb.kp[4 * v + 2] = cnt[v] | (cnt[v] > 2 ? 1 << 28 : 0);    // bit 28: more than two children (the sweep's rare loop)
                if (nt.pkey >= 0) pn = nt.pkey;
                else if (nparent[nt.gid] >= 0) {                               // exported sub-tree root: its parent is a ghost
                    const int32_t b = nbr[nt.gid];
                    pn = next + pb.nexp;
                    gp_of_branch[b] = pn;
                    if (g0_of_branch[b] < 0 || pn >= (1 << 20) || p == 0) { out.ok = false; return; }
                    if (kind == kItemCluster) {
                        // {node, ghost parent, ghost child in part 0, its parent there}; rank 0 sends the parent's x back
                        // to the block of this part, behind this entry (its last two ints are dead by then): the ghost
                        // child's entry names {rank << 20 | export}, turned into a shared-memory word by emit_item
                        pb.exps.insert(pb.exps.end(), {v, pn, g0_of_branch[b], p0_of_branch[b]});
                        out.parts[0].ghosts[4 * (size_t)x_of_branch[b] + 3] = (p << 20) | pb.nexp;
                    } else pb.exps.insert(pb.exps.end(), {v, pn, x_of_branch[b], 0});          // split item: exchange slot
                    ++pb.nexp;
                }
            }
            pb.kp[4 * v + 3] = pn;
            dist[v] = pn == v ? 0 : (pn >= next ? 1 : dist[pn] + 1);
            maxdist = std::max(maxdist, dist[v]);
        }
        pb.nnode = next + pb.nexp;
        for (int32_t e = 0; e < pb.nexp; ++e) pb.kp.insert(pb.kp.end(), {0, 0, 0, next + e});    // ghost parents read themselves
        for (int32_t v = 0; v < next; ++v)
            for (int q = 0; q < 2; ++q) pb.kp[4 * v + q] = (pb.kp[4 * v + q] < 0 ? pb.nnode : pb.kp[4 * v + q]) * RSb + 4 * w;
        while ((1 << pb.rounds) <= maxdist) ++pb.rounds;
        pb.maxwidth = 0;
        for (int32_t l = 0; l < pb.nlev; ++l) pb.maxwidth = std::max(pb.maxwidth, pb.lb[l + 1] - pb.lb[l]);
        // top nodes = the ancestors of ghost children (bit 29 of info): they wait for the other parts' hand-off values;
        // everything else in the part is swept before that.  ntoplev: levels [0, ntoplev) hold top nodes; lowlev: the
        // smallest level with a node that is not a top node.
        pb.ntoplev = 0; pb.lowlev = pb.nlev;
        if (pb.nghost) {
            std::vector<char> top(next, 0);
            for (int32_t v = next - 1; v >= 0; --v)
                if (nodes[v].pkey >= 0 && (nodes[v].ghost || top[v])) top[nodes[v].pkey] = 1;
            int32_t l = 0;
            for (int32_t v = 0; v < next; ++v) {
                while (v >= pb.lb[l + 1]) ++l;
                if (top[v]) { pb.kp[4 * v + 2] |= 1 << 29; pb.ntoplev = std::max(pb.ntoplev, l + 1); }
                else if (!nodes[v].ghost) pb.lowlev = std::min(pb.lowlev, l);
            }
        } else if (next > 0) pb.lowlev = 0;
        }
        if (p == 0) out.nxch = pb.nghost;
        // ---- P4: segments, in compartment order ---------------------------------------------------------------
        segs.clear();
        for (int32_t b : mine) {
            const Br& e = br[b];
            int32_t pos = e.soff;
            for (int32_t k = 0; k < e.nseg; ++k) {
                const int32_t plen = pieces[e.piece0 + k];
                const int32_t node = lmap[e.node0 + k];
                int32_t tnode;
                if (k > 0) tnode = lmap[e.node0 + k - 1];
                else if (e.parent < 0) tnode = -1;
                else if (br[e.parent].part == p) tnode = lmap[br[e.parent].node0 + br[e.parent].nseg - 1];
                else tnode = gp_of_branch[b];
                segs.push_back({pos, plen - 1, node, tnode});
                out.useful_steps += plen - 1;
                pos += plen;
            }
        }
        // two lanes per segment: lane A eliminates the interior above the middle node q, lane B the interior
        // below it, both top-down (fill-in to t resp. q); A eliminates q last.  A warp holds 16 segments:
        // A lanes 0..15, their B partners 16..31 (partner = lane ^ 16).
        // Long segments (interior >= quad_min) get FOUR lanes instead: the interior is cut at three middle nodes
        // q1 < q2 < q3 into quarters, lane j (= lane of the segment + 8 j) eliminates quarter j top-down with fill-in
        // to its top (t, q1, q2, q3); the first lane then eliminates q1, q2, q3 in turn.  Half the dependent steps
        // of the two-lane scheme for three more; a warp holds 8 such segments.
        std::vector<SegTmp> quads;
        if (P.quad_min > 0) {
            // ... but only where warps are to spare: four lanes double the warps a segment keeps busy, and the lone
            // warps of the level sweeps of the blocks beside it starve when the SM's schedulers fill up.  Estimate:
            // (blocks of this size per SM) x (warps of P1 with four lanes) <= quad_max_warps.
            size_t nlong = 0;
            for (const SegTmp& sg : segs) nlong += sg.m >= P.quad_min;
            const int64_t part_bytes = 16 + 512 + (int64_t)narr * w * pb.L + (int64_t)segs.size() * per_node;
            const int64_t per_sm = std::max<int64_t>(1, kSmemPerSM / (part_bytes + 2048));
            const int64_t warps4 = (int64_t)((nlong + 7) / 8 + (segs.size() - nlong + 15) / 16);
            if (per_sm * warps4 > P.quad_max_warps || warps4 > kMaxThreads / 32) nlong = 0;
            std::vector<SegTmp> rest;
            for (const SegTmp& sg : segs) (nlong && sg.m >= P.quad_min ? quads : rest).push_back(sg);
            segs.swap(rest);
            std::stable_sort(quads.begin(), quads.end(), [](const SegTmp& x, const SegTmp& y) { return x.m > y.m; });
        }
        order_segments(segs, 16, w == 8 ? 16 : 32, 0, ord);
        while ((ord.size() / 4) % 16) ord.insert(ord.end(), {0, 0, -1, -1});
        const int32_t ngroups2 = (int32_t)(ord.size() / 64), nquadg = (int32_t)((quads.size() + 7) / 8);
        if (nquadg) out.has_quads = 1;
        const int32_t ngroups = ngroups2 + nquadg;
        pb.seg.assign((size_t)ngroups * 128, 0);
        for (int32_t gq = 0; gq < nquadg; ++gq) {
            int32_t* G = &pb.seg[(size_t)(ngroups2 + gq) * 128];
            for (int32_t l = 0; l < 32; ++l) { G[4 * l + 2] = -1; G[4 * l + 3] = -1; }
            // The lanes of a shared-memory wavefront (fp64: lanes 0-15 = quarters 0, 1 and lanes 16-31 = quarters 2, 3;
            // fp32: all 32) should start on distinct bank residues: a quarter boundary may move by up to two nodes and a
            // lane may start up to 15 steps late (its residue moves with the delay), within the group's step count.
            // First fit, lane by lane; a lane that finds no free residue may push the owner of one of its candidate
            // residues to another free one (a later start of that lane), then take its place.
            const int NBq = w == 8 ? 16 : 32;
            int owner[2][32];                                              // residue -> lane (k + 8 j) that starts on it, per wavefront
            for (int h = 0; h < 2; ++h) for (int r = 0; r < 32; ++r) owner[h][r] = -1;
            const int32_t head_m = quads[(size_t)gq * 8].m;
            const int32_t cap = (head_m - 3 + 3) / 4 + 2;                  // steps of the group: the head's longest quarter + 2
            int32_t mqs[8][4], aqs[8][4], dqs[8][4];
            int32_t nk = 0;
            auto half_of = [&](int j) { return w == 8 ? j / 2 : 0; };
            auto residue = [&](int32_t a, int32_t dl) { return ((a - dl) % NBq + NBq) % NBq; };
            for (int32_t k = 0; k < 8 && (size_t)(gq * 8 + k) < quads.size(); ++k, ++nk) {
                const SegTmp& sg = quads[(size_t)gq * 8 + k];
                int32_t* mq = mqs[k]; int32_t* aq = aqs[k]; int32_t* dq = dqs[k];
                for (int32_t j = 0; j < 4; ++j) { mq[j] = (sg.m - 3) / 4 + (j < (sg.m - 3) % 4 ? 1 : 0); dq[j] = 0; }
                aq[0] = sg.a;
                for (int32_t j = 0; j < 4; ++j) {
                    if (j > 0) aq[j] = aq[j - 1] + mq[j - 1] + 1;
                    int* O = owner[half_of(j)];
                    static const int kShift[5] = {0, 1, -1, 2, -2};
                    bool done = false;
                    for (int pass = 0; pass < 2 && !done; ++pass)          // pass 1: with one displacement
                    for (int cost = 0; cost <= 17 && !done; ++cost)
                        for (int t = 0; t < 5 && !done; ++t) {
                            const int sh = j > 0 ? kShift[t] : 0, dl = cost - std::abs(sh);
                            if (dl < 0 || dl > 15 || (j == 0 && t > 0)) continue;
                            if (j > 0 && (mq[j - 1] + sh < 1 || mq[j] - sh < 1 || mq[j - 1] + sh + dq[j - 1] > cap)) continue;
                            if (mq[j] - sh + dl > cap) continue;
                            const int res = residue(aq[j] + sh, dl);
                            if (O[res] >= 0) {
                                if (pass == 0) continue;
                                // the owner moves to a free residue by starting later, if its steps allow
                                const int ok_ = O[res] & 7, oj = O[res] >> 3;
                                int32_t olen = mqs[ok_][oj];
                                if (ok_ == k && oj == j - 1) olen += sh;   // its length changes with this boundary
                                bool moved = false;
                                for (int32_t od = 0; od <= 15 && olen + od <= cap && !moved; ++od) {
                                    const int r2 = residue(aqs[ok_][oj], od);
                                    if (O[r2] >= 0 || r2 == res) continue;
                                    O[r2] = O[res]; dqs[ok_][oj] = od; moved = true;
                                }
                                if (!moved) continue;
                            }
                            O[res] = k + 8 * j; done = true;
                            if (j > 0) { mq[j - 1] += sh; aq[j] += sh; mq[j] -= sh; }
                            dq[j] = dl;
                        }
                }
            }
            int32_t mx = 0;
            for (int32_t k = 0; k < nk; ++k) {
                const SegTmp& sg = quads[(size_t)gq * 8 + k];
                for (int32_t j = 0; j < 4; ++j) {
                    int32_t* Lq = G + 4 * (k + 8 * j);
                    Lq[0] = aqs[k][j]; Lq[1] = (int32_t)((uint32_t)mqs[k][j] | ((uint32_t)j << 12) | (3u << 24) | (1u << 26) | ((uint32_t)dqs[k][j] << 27));
                    Lq[2] = sg.node; Lq[3] = j == 0 ? sg.tnode : -1;
                    mx = std::max(mx, mqs[k][j] + dqs[k][j]);
                }
            }
            out.padded_steps += 32 * (int64_t)(mx + 3);
        }
        for (int32_t gidx = 0; gidx < ngroups2; ++gidx) {
            int32_t mx = 0;
            for (int32_t k = 0; k < 16; ++k) {
                const int32_t* sgp = &ord[(size_t)(gidx * 16 + k) * 4];
                int32_t* A = &pb.seg[(size_t)(gidx * 32 + k) * 4];
                int32_t* B = &pb.seg[(size_t)(gidx * 32 + 16 + k) * 4];
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
        pb.nlanes = ngroups * 32;
        for (const SegTmp& sg : segs) if (sg.m >= 0xfff) out.ok = false;
        for (const SegTmp& sg : quads) if (sg.m >= 0xfff) out.ok = false;
        const int64_t meta = round_up(pb.nlev + 1, 4) + 4 * (int64_t)pb.nnode + 4 * (int64_t)pb.nexp +
                             4 * (int64_t)pb.nghost + 4 * (int64_t)pb.nlanes;
        pb.smem_need = 16 + 512 + 6 * round_up(pb.nnode + 1, E) * w + 4 * meta + narr * (int64_t)pb.L * w;
        if (kind == kItemSplit && p == 0) { out.smem_top = pb.smem_need; out.max_lanes_top = pb.nlanes; }
        else { out.smem_need = std::max(out.smem_need, pb.smem_need); out.max_lanes = std::max(out.max_lanes, pb.nlanes); }
        for (int32_t b : mine) for (int32_t k = 0; k < br[b].nseg; ++k) lmap[br[b].node0 + k] = -1;
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

// f1: the paper's branch splitting (reading F1).  Level by level from the root, over
// ALL cells given ("the average length of all dendritic branches on this level"): c = ceil(mean length of
// the pieces on the level); a piece longer than c is cut into a head of c compartments, which stays on the level,
// and the rest, which becomes its only child on the next level ("two shorter branches that are attached to each
// other") and takes the branch's children along ("causes all child branches to move one level down"); the rest
// may be cut again there.  Integer arithmetic throughout: c = (sum + count - 1) / count.
// The cells are the whole batch (f1, HINES_POLICY_SPLIT_LEVEL_MEAN) or the cells of one block (f4, "more
// local heuristics, like per block averages", HINES_POLICY_SPLIT_BLOCK_MEAN).
static void split_cells(const hines_plan& P, const std::vector<int64_t>& cells, std::vector<SplitPiece>& out, std::vector<int64_t>* stat)
{
    struct It { int64_t j, base; int32_t rem; };
    std::vector<It> cur, nxt;
    out.clear();
    for (int64_t c : cells) cur.push_back({P.cell_branch_offsets[c], P.cell_branch_offsets[c], P.branch_len[P.cell_branch_offsets[c]]});
    if (stat) stat->clear();
    for (int32_t level = 0; !cur.empty(); ++level) {
        int64_t sum = 0;
        for (const It& it : cur) sum += it.rem;
        const int64_t cnt = (int64_t)cur.size();
        const int64_t cut = (sum + cnt - 1) / cnt;
        if (stat) { stat->push_back(sum); stat->push_back(cnt); }
        nxt.clear();
        for (const It& it : cur) {
            if (it.rem > cut) {
                out.push_back({it.j, (int32_t)cut, level});
                nxt.push_back({it.j, it.base, (int32_t)(it.rem - cut)});
            } else {
                out.push_back({it.j, it.rem, level});
                for (int64_t k = P.child_offsets[it.j]; k < P.child_offsets[it.j + 1]; ++k) {
                    const int64_t ch = it.base + P.child_ids[k];
                    nxt.push_back({ch, it.base, P.branch_len[ch]});
                }
            }
        }
        cur.swap(nxt);
    }
}

// pieces (any order, the pieces of a branch top-down) -> the tables by branch
static void store_split_tables(hines_plan& P, const std::vector<SplitPiece>& out)
{
    const int64_t nbr = P.nbranches;
    P.split_piece_offsets.assign(nbr + 1, 0);
    for (const SplitPiece& p : out) P.split_piece_offsets[p.j + 1]++;
    for (int64_t j = 0; j < nbr; ++j) P.split_piece_offsets[j + 1] += P.split_piece_offsets[j];
    P.split_piece_len.assign(out.size(), 0);
    P.split_piece_level.assign(out.size(), 0);
    std::vector<int64_t> fill(P.split_piece_offsets.begin(), P.split_piece_offsets.end() - 1);
    for (const SplitPiece& p : out) { const int64_t q = fill[p.j]++; P.split_piece_len[q] = p.len; P.split_piece_level[q] = p.level; }
}

static void level_mean_split(hines_plan& P)
{
    std::vector<int64_t> all((size_t)P.ncells);
    std::iota(all.begin(), all.end(), (int64_t)0);
    std::vector<SplitPiece> out;
    split_cells(P, all, out, &P.split_level_stat);
    store_split_tables(P, out);
}

static void emit_item(hines_plan& P, const std::vector<int64_t>& cells, const ItemBuild& ib)
{
    const int32_t item = (int32_t)P.item_kind.size();
    for (int64_t c : cells) P.cell_item[c] = item;
    P.item_cells.insert(P.item_cells.end(), cells.begin(), cells.end());
    P.item_cell_offsets.push_back((int64_t)P.item_cells.size());
    P.item_unknowns.push_back(ib.n);
    P.block_split.insert(P.block_split.end(), ib.split.begin(), ib.split.end());
    P.item_class.push_back(0);                     // filled by assign_classes
    P.item_kind.push_back(ib.kind);
    P.item_xch.push_back((int32_t)P.n_xch);
    const int32_t xs0 = 2 * (ib.parts[0].rounds & 1) + 1;
    // where the blocks of a cluster item receive their parents' x: 4-byte word index, from the start of the block's
    // shared memory, of int 2 of the export's entry ([mbarriers 16 | block record | node records | lb | kp | exports ..])
    std::vector<int32_t> land0(ib.parts.size(), 0);
    const int64_t E = 16 / P.width;
    for (size_t r = 0; r < ib.parts.size(); ++r) {
        const PartBuild& pb = ib.parts[r];
        const int64_t NN = round_up((int64_t)pb.nnode + 1, E);
        const int64_t meta_word = (16 + (int64_t)sizeof(hines::BlockRecord) + 6 * P.width * NN) / 4;
        land0[r] = (int32_t)(meta_word + round_up((int64_t)pb.lb.size(), 4) + round_up((int64_t)pb.kp.size(), 4) + 2);
    }
    for (size_t r = 0; r < ib.parts.size(); ++r) {
        PartBuild pb_patched;
        if (r == 0 && ib.kind == kItemCluster) {
            pb_patched = ib.parts[0];
            for (int32_t g = 0; g < pb_patched.nghost; ++g) {
                const int32_t w = pb_patched.ghosts[4 * (size_t)g + 3], rr = w >> 20, e = w & 0xfffff;
                pb_patched.ghosts[4 * (size_t)g + 3] = (rr << 20) | (land0[rr] + 4 * e);
            }
        }
        const PartBuild& pb = (r == 0 && ib.kind == kItemCluster) ? pb_patched : ib.parts[r];
        hines::PartHeader h{};
        h.meta_off = (int64_t)P.part_meta.size();
        std::vector<int32_t>& M = P.part_meta;
        auto pad4 = [&]() { M.resize((size_t)round_up((int64_t)M.size(), 4), 0); };
        M.insert(M.end(), pb.lb.begin(), pb.lb.end()); pad4();
        h.kp_off = (int32_t)((int64_t)M.size() - h.meta_off);
        M.insert(M.end(), pb.kp.begin(), pb.kp.end()); pad4();
        h.exp_off = (int32_t)((int64_t)M.size() - h.meta_off);
        M.insert(M.end(), pb.exps.begin(), pb.exps.end());
        h.gh_off = (int32_t)((int64_t)M.size() - h.meta_off);
        M.insert(M.end(), pb.ghosts.begin(), pb.ghosts.end());
        h.seg_off = (int32_t)((int64_t)M.size() - h.meta_off);
        M.insert(M.end(), pb.seg.begin(), pb.seg.end());
        h.meta_len = (int32_t)((int64_t)M.size() - h.meta_off);
        h.run_off = (int32_t)(P.part_runs.size() / 4);
        h.nrun = (int32_t)(pb.runs.size() / 4);
        for (int32_t k = 0; k < h.nrun; ++k)
        {
            // {global first compartment, length, staged index, w}: w spares the loader and the store their index
            // arithmetic: bits 0-15 the elements the bulk copy brings (the run widened to 16-byte words, clipped at the
            // end of the arrays), bits 16-19 the elements in front of the first whole word of the run (stored by hand),
            // bits 20-23 the elements behind its last whole word, bit 24: elements beyond the arrays' last whole word
            // (loaded by hand)
            const int64_t g = ib.comp_begin + pb.runs[4 * k], len = pb.runs[4 * k + 1], E = 16 / P.width;
            const int64_t ga = g - g % E, ge = std::min<int64_t>(round_up(g + len, E), P.n / E * E);
            const int64_t cnt = std::max<int64_t>(0, ge - ga);
            const int64_t head = std::min<int64_t>(len, (E - g % E) % E), tail = std::max<int64_t>(head, (g + len) / E * E - g);
            const int32_t wd = (int32_t)(cnt | (head << 16) | ((len - tail) << 20) | ((int64_t)(g + len > ge) << 24));
            P.part_runs.insert(P.part_runs.end(), {(int32_t)g, (int32_t)len, pb.runs[4 * k + 2], wd});
        }
        h.tx_elems = pb.tx_elems; h.L = pb.L; h.n = pb.n;
        h.nnode = pb.nnode; h.nlevnode = pb.nlevnode; h.nlev = pb.nlev; h.rounds = pb.rounds;
        h.nexp = pb.nexp; h.nghost = pb.nghost; h.nseg_lanes = pb.nlanes;
        h.xch_base = (int32_t)P.n_xch; h.xs0 = xs0;
        h.item = item; h.rank = (int32_t)r; h.flags = pb.flags | ((P.opt.policy_flags & HINES_POLICY_FACTORED) ? kPartFlagFactored : 0); h.ntoplev = pb.ntoplev; h.lowlev = pb.lowlev; h.maxwidth = pb.maxwidth;
        P.part_headers.push_back(h);
        P.n_exports += pb.nexp;
    }
    P.item_part_offsets.push_back((int64_t)P.part_headers.size());
    if (ib.kind == kItemSplit) P.n_xch += ib.nxch;
    P.padded_lane_steps += ib.padded_steps;
    P.useful_lane_steps += ib.useful_steps;
    const int64_t ncell = (int64_t)cells.size();
    if (ib.kind == kItemCluster) { P.n_cluster_cells += ncell; P.n_cluster_unknowns += ib.n; }
    if (ib.kind == kItemSplit) { P.n_split_cells += ncell; P.n_split_unknowns += ib.n; }
    P.n_resident_cells += ncell;
    P.n_resident_unknowns += ib.n;
}

struct ItemNeed { int64_t smem; int32_t lanes; int32_t nparts; int32_t kind; int64_t smem_top; int32_t lanes_top; int32_t quads; };

// P1 + P2: cells -> work items, greedy in input order.  A cell whose lists fit the group budget
// joins the open group while the group still fits; a cell that fits one block's budget gets its own item; a
// larger cell is cut into the parts of a cluster of up to cluster_max blocks ("long branches of large cells kept
// on their own blocks"), beyond that into the parts of a split item (three launches); what fits nowhere goes to
// the streaming path.
static void pack_items(hines_plan& P, std::vector<ItemNeed>& need, std::vector<char>& is_stream)
{
    const int64_t nc = P.ncells;
    const int64_t max_smem = P.opt.smem_bytes_per_block;
    const int64_t group_cap = std::min<int64_t>(P.opt.group_smem_bytes, max_smem);
    const bool force_stream = P.opt.policy_flags & HINES_POLICY_FORCE_STREAM;
    const bool no_group = P.opt.policy_flags & HINES_POLICY_NO_GROUPING;
    const bool no_cluster = (P.opt.policy_flags & HINES_POLICY_NO_CLUSTER) || P.opt.cluster_max < 2;
    const bool no_split = (P.opt.policy_flags & HINES_POLICY_NO_SPLIT) != 0;
    // a cell alone in a block may use up to single_cap; beyond that a cluster is preferred, because
    // blocks of at most chunk_smem_bytes leave room for a second resident block per SM
    const int64_t chunk_cap = std::min<int64_t>(P.opt.chunk_smem_bytes, max_smem);
    const int64_t single_cap = no_cluster ? max_smem : chunk_cap;
    const bool pow2_only = P.opt.policy_flags & HINES_POLICY_POW2_CLUSTERS;
    const bool level_mean = (P.opt.policy_flags & HINES_POLICY_SPLIT_LEVEL_MEAN) != 0;
    const int32_t w = P.width;
    P.cell_item.assign(nc, -1);
    P.item_part_offsets.assign(1, 0);
    P.item_cell_offsets.assign(1, 0);
    is_stream.assign(nc, 0);
    ItemBuild cand, alone;
    auto push = [&](const std::vector<int64_t>& cells, const ItemBuild& ib) {
        emit_item(P, cells, ib);
        need.push_back({ib.smem_need, ib.max_lanes, (int32_t)ib.parts.size(), ib.kind, ib.smem_top, ib.max_lanes_top, ib.has_quads});
    };
    // additive estimate of a cell's shared-memory need as a single part (upper side): arrays + per node the
    // record, two segment lanes and the node descriptor; decides group membership without building the group
    std::vector<int32_t> tmp;
    auto estimate = [&](int64_t c) -> int64_t {
        int64_t nodes = 0;
        for (int64_t j = P.cell_branch_offsets[c]; j < P.cell_branch_offsets[c + 1]; ++j) {
            tmp.clear();
            if (level_mean) for (int64_t q = P.split_piece_offsets[j]; q < P.split_piece_offsets[j + 1]; ++q) fixed_bound_pieces(P.split_piece_len[q], P.seg_single, tmp);
            else fixed_bound_pieces(P.branch_len[j], P.seg_single, tmp);
            nodes += (int64_t)tmp.size();
        }
        return ((P.opt.policy_flags & HINES_POLICY_FACTORED) ? 4 : 3) * (int64_t)w * (P.cell_offsets[c + 1] - P.cell_offsets[c] + 2) + nodes * (6 * w + 32 + 16) + 4 * (P.cell_nlevels[c] + 1);
    };
    const int64_t group_fixed = 16 + 512 + 2048;    // mbarrier, block record, alignment slack, padding of the lane list to whole warps
    // The open group: small cells in input order ("greedy"); a large cell in between gets an item of its
    // own and does not close the group (a part is a list of runs: its cells need not be neighbours).
    std::vector<int64_t> group;
    int64_t gacc = 0;
    // a closed group is built once; should the build exceed the cap after all, it is halved
    std::function<void(const std::vector<int64_t>&)> flush_cells = [&](const std::vector<int64_t>& cells) {
        if (cells.empty()) return;
        ItemBuild ib;
        build_item(P, cells, kItemSingle, 1, 0, ib);
        if ((!ib.ok || ib.smem_need > group_cap) && cells.size() > 1) {
            const size_t mid = cells.size() / 2;
            flush_cells(std::vector<int64_t>(cells.begin(), cells.begin() + mid));
            flush_cells(std::vector<int64_t>(cells.begin() + mid, cells.end()));
            return;
        }
        if (!ib.ok || ib.smem_need > max_smem) { for (int64_t c : cells) is_stream[c] = 1; return; }
        push(cells, ib);
    };
    auto flush = [&]() { flush_cells(group); group.clear(); gacc = 0; };
    const bool adjacent_only = (P.opt.policy_flags & HINES_POLICY_INPUT_ORDER) != 0;
    std::vector<int64_t> one(1);
    for (int64_t c = 0; c < nc; ++c) {
        if (force_stream) { is_stream[c] = 1; continue; }
        const int64_t est = estimate(c);
        if (!no_group && est + group_fixed <= group_cap) {                  // a small cell: joins the open group, greedy in input order
            if (!group.empty() && (gacc + est + group_fixed > group_cap || group.size() >= 4096)) flush();
            group.push_back(c);
            gacc += est;
            continue;
        }
        if (adjacent_only) flush();
        one[0] = c;
        bool placed = false, is_single = false;
        if (est <= single_cap + 4096) {
            build_item(P, one, kItemSingle, 1, 0, alone);
            is_single = alone.ok && alone.smem_need <= single_cap;
        }
        if (!is_single && !no_cluster) {
            // cluster size: the one whose blocks fill their shared-memory slot best (slots = an SM's
            // shared memory divided by 2, 3, 4); close calls go to the smaller cluster
            const int64_t total = est + 1024;
            struct Opt { double score; int32_t k; int64_t slot; };
            std::vector<Opt> opts;
            for (int t = 3; t <= 5; ++t) {                                // slots of 1/2, 1/3, 1/4 of an SM
                const int64_t slot = class_cap(t, max_smem);
                if (slot > chunk_cap) continue;
                int32_t k = (int32_t)std::max<int64_t>(2, (total + slot - 4096 - 1) / (slot - 4096));
                if (pow2_only) while (k & (k - 1)) ++k;
                if (k > P.opt.cluster_max) continue;
                opts.push_back({-((double)total / (double)(k * slot) - 0.01 * t), k, slot});
            }
            if (opts.empty() && total / P.opt.cluster_max + 4096 <= max_smem) opts.push_back({0.0, P.opt.cluster_max, max_smem});
            std::sort(opts.begin(), opts.end(), [](const Opt& a, const Opt& b) { return a.score < b.score; });
            for (size_t o = 0; o < opts.size() && o < 3 && !placed; ++o) {
                // the sub-trees may not balance as well as the estimate assumes: one or two blocks more are tried too,
                // and an option counts only if every part fits the slot it was chosen for
                for (int32_t k = opts[o].k; k <= std::min<int32_t>(P.opt.cluster_max, opts[o].k + 2) && !placed; ++k) {
                    if (pow2_only && (k & (k - 1))) continue;
                    build_item(P, one, kItemCluster, k, 0, cand);
                    if (cand.ok && cand.smem_need <= opts[o].slot) { push(one, cand); placed = true; }
                }
            }
            if (!placed) {                                                // anything that fits a block
                for (int32_t k = opts.empty() ? P.opt.cluster_max : std::min<int32_t>(P.opt.cluster_max, opts[0].k + 3); k <= P.opt.cluster_max && !placed; k += std::max(1, k / 4)) {
                    if (pow2_only && (k & (k - 1))) continue;
                    build_item(P, one, kItemCluster, k, 0, cand);
                    if (cand.ok && cand.smem_need <= max_smem) { push(one, cand); placed = true; }
                }
            }
            if (!placed && est <= max_smem) {                             // one big block
                build_item(P, one, kItemSingle, 1, 0, alone);
                is_single = alone.ok && alone.smem_need <= max_smem;
            }
        }
        if (!placed && !is_single && !no_cluster && !no_split) {
            // beyond the largest cluster: sub-tree parts of at most a split_smem_bytes slot + the top part in one block
            // (should the top part not fit one block, larger sub-trees leave a smaller top: the slot is raised once)
            const int64_t sslots[3] = {std::min<int64_t>(P.opt.split_smem_bytes, max_smem), max_smem, max_smem};
            const int32_t pct[3] = {80, 80, 97};
            for (int t = 0; t < 3 && !placed; ++t) {
                build_item(P, one, kItemSplit, pct[t], sslots[t] - 6144, cand);
                if (cand.ok && cand.parts.size() > 1 && cand.smem_need <= sslots[t] && cand.smem_top <= max_smem) { push(one, cand); placed = true; }
            }
        }
        if (placed) continue;
        if (!is_single) { is_stream[c] = 1; continue; }
        push(one, alone);
    }
    flush();
}

// Size classes.  By how many blocks of that size fit one SM (1, 2, 3, 4, 6, 8), separately for single-block
// items, for every cluster size, and for the three launch phases of split items.  Threads per block: enough
// lanes for the widest segment list of the class, within what the register file allows for that many resident blocks.
static void assign_classes(hines_plan& P, const std::vector<ItemNeed>& need)
{
    const int64_t nitems = (int64_t)need.size();
    const int64_t max_smem = P.opt.smem_bytes_per_block;
    // queue index: [0, 6) single blocks; 6*k + t cluster of k; then split: sub-tree parts, top parts
    const int qSplitSub = kNumClassK * (kMaxClusterClass + 1), qSplitTop = qSplitSub + kNumClassK, nq = qSplitTop + kNumClassK;
    auto slot_of = [&](int64_t smem) { int q = 0; for (int t = 0; t < kNumClassK; ++t) if (smem <= class_cap(t, max_smem)) q = t; return q; };
    std::vector<int> item_q(nitems, 0);
    std::vector<int64_t> need_max(nq, 0), count(nq, 0);
    std::vector<int32_t> lanes_max(nq, 0), quads_any(nq, 0);
    for (int64_t i = 0; i < nitems; ++i) {
        int q = slot_of(need[i].smem);
        if (need[i].kind == kItemCluster) q += kNumClassK * need[i].nparts;
        if (need[i].kind == kItemSplit) {
            q += qSplitSub;
            const int qt = qSplitTop + slot_of(need[i].smem_top);
            need_max[qt] = std::max(need_max[qt], need[i].smem_top);
            lanes_max[qt] = std::max(lanes_max[qt], need[i].lanes_top);
            quads_any[qt] |= need[i].quads;
            count[qt]++;
        }
        item_q[i] = q;
        need_max[q] = std::max(need_max[q], need[i].smem);
        lanes_max[q] = std::max(lanes_max[q], need[i].lanes);
        quads_any[q] |= need[i].quads;
        count[q]++;
    }
    // launch order of the classes: clusters first (largest first), then single blocks, biggest first; the
    // classes of split items on a stream of their own: phase A, then B, then C
    struct Cls { int q, phase; };
    std::vector<Cls> qs;
    for (int k = kMaxClusterClass; k >= 2; --k)
        for (int t = 0; t < kNumClassK; ++t) if (count[kNumClassK * k + t]) qs.push_back({kNumClassK * k + t, kPhaseAll});
    for (int q = 0; q < kNumClassK; ++q) if (count[q]) qs.push_back({q, kPhaseAll});
    for (int q = qSplitSub; q < qSplitSub + kNumClassK; ++q) if (count[q]) qs.push_back({q, kPhaseA});
    for (int q = qSplitTop; q < qSplitTop + kNumClassK; ++q) if (count[q]) qs.push_back({q, kPhaseB});
    for (int q = qSplitSub; q < qSplitSub + kNumClassK; ++q) if (count[q]) qs.push_back({q, kPhaseC});
    std::vector<int> cls_of_q(nq, -1);
    for (const Cls& c : qs) {
        const int q = c.q;
        if (c.phase != kPhaseC) cls_of_q[q] = (int)P.class_smem_bytes.size();
        const int64_t smem = round_up(need_max[q], 128);
        P.class_smem_bytes.push_back((int32_t)smem);
        P.class_cluster.push_back(q >= kNumClassK && q < qSplitSub ? q / kNumClassK : 1);
        P.class_phase.push_back(c.phase);
        P.class_quads.push_back(quads_any[q]);
        const int64_t per_sm = std::max<int64_t>(1, kSmemPerSM / (smem + 1024));
        int64_t tmax = 65536 / ((P.width == 4 ? kRegsPerThreadF32 : kRegsPerThread) * per_sm) / 32 * 32;
        tmax = std::max<int64_t>(64, std::min<int64_t>(kMaxThreads, tmax));
        int64_t t = P.opt.threads_per_block ? P.opt.threads_per_block : round_up(std::max(lanes_max[q], 1), 32);
        t = std::max<int64_t>(P.opt.threads_per_block ? 32 : std::min<int64_t>(128, tmax), std::min(t, tmax));
        P.class_threads.push_back((int32_t)t);
    }
    for (int64_t i = 0; i < nitems; ++i) P.item_class[i] = cls_of_q[need[i].kind == kItemSplit ? qSplitTop + slot_of(need[i].smem_top) : item_q[i]];
    P.item_launch_order.resize(nitems);
    std::iota(P.item_launch_order.begin(), P.item_launch_order.end(), 0);
    const bool input_order = P.opt.policy_flags & HINES_POLICY_INPUT_ORDER;
    auto weight = [&](int32_t it) { return P.item_unknowns[it]; };
    std::stable_sort(P.item_launch_order.begin(), P.item_launch_order.end(), [&](int32_t a, int32_t b) {
        if (P.item_class[a] != P.item_class[b]) return P.item_class[a] < P.item_class[b];
        if (input_order) return false;
        return weight(a) > weight(b);                                  // heaviest first
    });
    // blocks of every class in launch order
    const int ncls = (int)P.class_smem_bytes.size();
    P.class_first.assign(ncls, 0);
    P.class_count.assign(ncls, 0);
    for (int k = 0; k < ncls; ++k) {
        const Cls& c = qs[k];
        P.class_first[k] = (int64_t)P.class_parts.size();
        for (int32_t it : P.item_launch_order) {
            const int64_t p0 = P.item_part_offsets[it], p1 = P.item_part_offsets[it + 1];
            if (c.phase == kPhaseAll) {
                if (need[it].kind == kItemSplit || item_q[it] != c.q) continue;
                for (int64_t p = p0; p < p1; ++p) P.class_parts.push_back((int32_t)p);
            } else if (need[it].kind == kItemSplit) {
                if (c.phase == kPhaseB) { if (qSplitTop + slot_of(need[it].smem_top) == c.q) P.class_parts.push_back((int32_t)p0); }
                else if (item_q[it] == c.q) for (int64_t p = p0 + 1; p < p1; ++p) P.class_parts.push_back((int32_t)p);
            }
        }
        P.class_count[k] = (int64_t)P.class_parts.size() - P.class_first[k];
    }
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
    if (o.cluster_max == 0) o.cluster_max = 8;
    if (o.chunk_smem_bytes == 0) o.chunk_smem_bytes = 117 * 1024;       // half an SM: two blocks per SM overlap each other's phases (measured optimum)
    if (o.split_smem_bytes == 0) o.split_smem_bytes = 113 * 1024;
    if (o.threads_per_block < 0 || o.threads_per_block > kMaxThreads || o.threads_per_block % 32 ||
        o.stream_threads < 32 || o.stream_threads > 1024 || o.stream_threads % 32 ||
        o.smem_bytes_per_block < 1024 || o.smem_bytes_per_block > kSmemMaxOptin || o.group_smem_bytes < 0 ||
        o.max_segment < 2 || o.max_segment > 1023 || (o.policy_flags & ~8191) ||
        o.cluster_max < 1 || o.cluster_max > 16 || o.chunk_smem_bytes < 1024 || o.split_smem_bytes < 8192) {
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
        std::unique_ptr<hines_plan> holder(new hines_plan());
        hines_plan* P = holder.get();
        P->n = cell_offsets[ncells]; P->ncells = ncells; P->dtype = dtype; P->width = dtype == HINES_F64 ? 8 : 4;
        P->opt = o;
        P->seg_cluster = o.max_segment;
        P->seg_single = auto_segment ? 40 : o.max_segment;
        P->quad_min = (o.policy_flags & HINES_POLICY_NO_QUADS) ? 0 : 24;
        P->quad_max_warps = 22;
        P->cell_offsets.assign(cell_offsets, cell_offsets + ncells + 1);
        hines_status_t st = canonical_tables(*P, parent);
        if (st != HINES_OK) return st;
        level_mean_split(*P);
        std::vector<ItemNeed> item_need;
        std::vector<char> is_stream;
        pack_items(*P, item_need, is_stream);
        if ((o.policy_flags & HINES_POLICY_SPLIT_BLOCK_MEAN) && !(o.policy_flags & HINES_POLICY_SPLIT_LEVEL_MEAN)) {
            // f4: the tables now describe what the blocks were built from; cells of the streaming path are not split
            for (int64_t c = 0; c < P->ncells; ++c)
                if (is_stream[c])
                    for (int64_t j = P->cell_branch_offsets[c]; j < P->cell_branch_offsets[c + 1]; ++j)
                        P->block_split.push_back({j, P->branch_len[j], P->branch_level[j]});
            store_split_tables(*P, P->block_split);
            P->split_level_stat.clear();
            std::vector<SplitPiece>().swap(P->block_split);
        }
        assign_classes(*P, item_need);
        build_stream(*P, is_stream);
        *out_plan = holder.release();
        return HINES_OK;
    } catch (const std::bad_alloc&) {
        set_error("host allocation failed while building the plan"); return HINES_ERR_ALLOC;
    } catch (const std::exception& e) {
        set_error(std::string("internal error: ") + e.what()); return HINES_ERR_ALLOC;
    }
}

hines_status_t hines_partition_cells(const int64_t* cell_offsets, int64_t ncells, int32_t nparts,
                                     int32_t* cell_part, int64_t* part_cost)
{
    if (!cell_offsets || !cell_part) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (ncells <= 0 || nparts <= 0) { set_error("ncells and nparts must be positive"); return HINES_ERR_INVALID_ARG; }
    for (int64_t c = 0; c < ncells; ++c)
        if (cell_offsets[c + 1] <= cell_offsets[c]) { set_error("cell_offsets not strictly increasing at cell " + std::to_string(c)); return HINES_ERR_BAD_TOPOLOGY; }
    try {
        std::vector<int64_t> order(ncells);
        std::iota(order.begin(), order.end(), 0);
        auto cost = [&](int64_t c) { return cell_offsets[c + 1] - cell_offsets[c]; };
        std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return cost(a) > cost(b); });
        // a heap of (cost so far, device): the lightest device first, ties to the lowest index
        std::vector<std::pair<int64_t, int32_t>> heap;
        for (int32_t p = 0; p < nparts; ++p) heap.push_back({0, p});
        auto cmp = [](const std::pair<int64_t, int32_t>& a, const std::pair<int64_t, int32_t>& b) { return a > b; };
        std::make_heap(heap.begin(), heap.end(), cmp);
        for (int64_t c : order) {
            std::pop_heap(heap.begin(), heap.end(), cmp);
            cell_part[c] = heap.back().second;
            heap.back().first += cost(c);
            std::push_heap(heap.begin(), heap.end(), cmp);
        }
        if (part_cost) for (const auto& h : heap) part_cost[h.second] = h.first;
        return HINES_OK;
    } catch (const std::exception&) {
        set_error("host allocation failed"); return HINES_ERR_ALLOC;
    }
}

hines_status_t hines_plan_get_info(const hines_plan_t* P, hines_plan_info_t* out)
{
    if (!P || !out) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    std::memset(out, 0, sizeof(*out));
    out->n = P->n; out->ncells = P->ncells; out->nbranches = P->nbranches;
    out->max_levels = P->max_levels; out->dtype = P->dtype;
    out->n_resident_items = (int64_t)P->item_kind.size();
    out->n_resident_cells = P->n_resident_cells; out->n_resident_unknowns = P->n_resident_unknowns;
    out->n_stream_cells = P->n_stream_cells; out->n_stream_unknowns = P->n_stream_unknowns;
    out->n_stream_branches = (int64_t)P->stream_desc.size();
    out->padded_lane_steps = P->padded_lane_steps; out->useful_lane_steps = P->useful_lane_steps;
    out->workspace_bytes = (int64_t)(P->part_meta.size() * 4 + P->part_runs.size() * 4 + P->class_parts.size() * sizeof(PartHeader) +
                                     3 * P->n_xch * P->width + P->class_parts.size() * (sizeof(BlockRecord) - sizeof(PartHeader)) + P->stream_desc.size() * sizeof(StreamDesc) +
                                     P->stream_child.size() * 4 + 2 * P->n_stream_unknowns * P->width);
    out->bytes_min = P->n * 4 * P->width + 4 * P->nbranches;
    out->bytes_literal = P->n * (4 * P->width + 4);
    out->breadth_first = P->breadth_first;
    out->n_classes = (int32_t)P->class_smem_bytes.size();
    out->n_cluster_cells = P->n_cluster_cells; out->n_cluster_unknowns = P->n_cluster_unknowns;
    out->n_parts = (int64_t)P->part_headers.size();
    out->n_split_cells = P->n_split_cells; out->n_split_unknowns = P->n_split_unknowns;
    out->n_exports = P->n_exports;
    out->n_blocks = (int64_t)P->class_parts.size();
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
        TBL(HINES_TABLE_ITEM_CELL_OFFSETS, P->item_cell_offsets)
        TBL(HINES_TABLE_ITEM_CELLS, P->item_cells)
        TBL(HINES_TABLE_ITEM_CLASS, P->item_class)
        TBL(HINES_TABLE_ITEM_LAUNCH_ORDER, P->item_launch_order)
        TBL(HINES_TABLE_ITEM_KIND, P->item_kind)
        TBL(HINES_TABLE_ITEM_XCH, P->item_xch)
        TBL(HINES_TABLE_ITEM_PART_OFFSETS, P->item_part_offsets)
        TBL(HINES_TABLE_PART_HEADER, P->part_headers)
        TBL(HINES_TABLE_PART_META, P->part_meta)
        TBL(HINES_TABLE_PART_RUNS, P->part_runs)
        TBL(HINES_TABLE_CLASS_PHASE, P->class_phase)
        TBL(HINES_TABLE_CLASS_FIRST, P->class_first)
        TBL(HINES_TABLE_CLASS_COUNT, P->class_count)
        TBL(HINES_TABLE_CLASS_PARTS, P->class_parts)
        TBL(HINES_TABLE_SPLIT_PIECE_OFFSETS, P->split_piece_offsets)
        TBL(HINES_TABLE_SPLIT_PIECE_LEN, P->split_piece_len)
        TBL(HINES_TABLE_SPLIT_PIECE_LEVEL, P->split_piece_level)
        TBL(HINES_TABLE_SPLIT_LEVEL_STAT, P->split_level_stat)
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
    int32_t k = 0;
    for (size_t q = 0; q < P->class_count.size(); ++q) if (P->class_count[q]) ++k;
    *out = k + 2 * (int32_t)(P->stream_level_begin.size() - 1);
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
const char* hines_version(void) { return "hines-b200 0.2 (sm_100a)"; }

}  // extern "C"

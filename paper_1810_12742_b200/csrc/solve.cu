// hines_solve: the per-step kernels (sm_100a) and their host launcher.
//
// Two paths, chosen per cell by the plan:
//   resident  whole cells / cell groups staged into shared memory by TMA bulk copies
//             (cp.async.bulk + mbarrier), level-synchronous sweeps with one lane per branch
//             (PAPER.md:110-114), block barrier per level, sibling hand-off by warp shuffle,
//             x written back by a bulk store.  d,u,b are read from and x written to the caller's
//             natural-order arrays directly: the paper's separate permute kernels
//             do not exist here.
//   stream    cells too large for one block's shared memory: one launch per level over all such
//             cells (global synchronisation = kernel boundary, which PAPER.md:114 avoids by
//             requiring one matrix per block), intermediates in a plan-owned global workspace.
//
// Arithmetic per compartment i with parent/previous compartment q (Listing 2 read
// with u[i], reading G1), written with the reciprocal r = 1/d'[i] (reading S12):
//   backward:  f = u[i] r;  c = b'[i] r;  d'[q] -= f u[i];  b'[q] -= f b'[i]
//   root:      x[0] = b'[0] r
//   forward:   x[i] = (b'[i] - u[i] x[q]) / d'[i] = c - f x[q]
// f overwrites d and c, then x, overwrite b in the on-chip copy; the caller's d,u,b are not written.
#include <cuda_runtime.h>
#include <cooperative_groups.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "plan_internal.h"

namespace hines {

struct BlockRec { ItemHeader it; ChunkHeader ch; };   // 80 bytes

struct DeviceTables {
    int device = -1;
    BlockRec* recs = nullptr;                                     // one per resident block, launch order
    int32_t* item_meta = nullptr;
    StreamDesc* stream_desc = nullptr;
    int32_t* stream_child = nullptr;
    void* ws_f = nullptr;           // streaming workspace: f (n_stream_unknowns elements)
    void* ws_c = nullptr;           // streaming workspace: c
    void* host_stage[4] = {nullptr, nullptr, nullptr, nullptr};   // hines_solve_host device buffers d,u,b,x
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};              // timing hook
    static const int kSide = 3;                                   // side streams: size classes run concurrently
    cudaStream_t side[kSide] = {nullptr, nullptr, nullptr};
    cudaEvent_t fork = nullptr, join[kSide] = {nullptr, nullptr, nullptr};
    cudaStream_t sstream = nullptr;                               // the streaming path runs beside the resident classes
    cudaEvent_t sjoin = nullptr;
    bool timing = false, timed_once = false;
    unsigned long long* prof = nullptr;                           // phase clocks: 8 x u64 per resident block, launch order
    bool prof_on = false;
    int64_t bytes = 0;
};

#define CUDA_TRY(expr)                                                                         \
    do {                                                                                       \
        cudaError_t e_ = (expr);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            set_error(std::string(#expr) + ": " + cudaGetErrorString(e_));                     \
            return e_ == cudaErrorMemoryAllocation ? HINES_ERR_ALLOC : HINES_ERR_CUDA;         \
        }                                                                                      \
    } while (0)


// ------------------------------------------------------------------------------------------------
// PTX helpers: mbarrier + 1-D TMA bulk copies (SASS: UBLKCP, SYNCS)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared bulk copy, completion counted in bytes on the mbarrier
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// shared -> global bulk copy (bulk async-group completion)
__device__ __forceinline__ void tma_store_1d(void* dst_gmem, const void* src_smem, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_store_commit_wait()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ unsigned smid()
{
    unsigned r;
    asm volatile("mov.u32 %0, %smid;" : "=r"(r));
    return r;
}

// fast reciprocal: hardware seed + Newton steps (no slow-path branch on the dependent chain; the
// pivots of a strictly diagonally dominant matrix are finite, non-zero and in the normal range)
template <typename T> __device__ __forceinline__ T rcp(T v);
template <> __device__ __forceinline__ double rcp<double>(double v)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(v));      // MUFU.RCP64H: ~20 bits
    double e = fma(-v, r, 1.0); r = fma(r, e, r);               // ~40 bits
    e = fma(-v, r, 1.0); r = fma(r, e, r);                      // full double
    return r;
}
template <> __device__ __forceinline__ float rcp<float>(float v)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    const float e = fmaf(-v, r, 1.0f);
    return fmaf(r, e, r);
}

template <typename T> __device__ __forceinline__ T fnma(T a, T b, T c);   // c - a*b
template <> __device__ __forceinline__ double fnma<double>(double a, double b, double c) { return fma(-a, b, c); }
template <> __device__ __forceinline__ float fnma<float>(float a, float b, float c) { return fmaf(-a, b, c); }
template <typename T> struct Vec2;
template <> struct Vec2<double> { typedef double2 type; };
template <> struct Vec2<float> { typedef float2 type; };
// shared-memory accesses by 32-bit shared address (no generic-to-shared conversion on the dependent chain)
template <typename T> __device__ __forceinline__ typename Vec2<T>::type lds2(uint32_t a);
template <> __device__ __forceinline__ double2 lds2<double>(uint32_t a)
{ double2 v; asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a) : "memory"); return v; }
template <> __device__ __forceinline__ float2 lds2<float>(uint32_t a)
{ float2 v; asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a) : "memory"); return v; }
template <typename T> __device__ __forceinline__ T lds1(uint32_t a);
template <> __device__ __forceinline__ double lds1<double>(uint32_t a)
{ double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory"); return v; }
template <> __device__ __forceinline__ float lds1<float>(uint32_t a)
{ float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a) : "memory"); return v; }
template <typename T> __device__ __forceinline__ void sts1(uint32_t a, T v);
template <> __device__ __forceinline__ void sts1<double>(uint32_t a, double v)
{ asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
template <> __device__ __forceinline__ void sts1<float>(uint32_t a, float v)
{ asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
template <typename T> __device__ __forceinline__ void sts2(uint32_t a, typename Vec2<T>::type v);
template <> __device__ __forceinline__ void sts2<double>(uint32_t a, double2 v)
{ asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.x), "d"(v.y) : "memory"); }
template <> __device__ __forceinline__ void sts2<float>(uint32_t a, float2 v)
{ asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(v.x), "f"(v.y) : "memory"); }
template <typename T> __device__ __forceinline__ T fmad(T a, T b, T c);   // c + a*b
template <> __device__ __forceinline__ double fmad<double>(double a, double b, double c) { return fma(a, b, c); }
template <> __device__ __forceinline__ float fmad<float>(float a, float b, float c) { return fmaf(a, b, c); }

// ------------------------------------------------------------------------------------------------
// Resident kernel: one block per chunk; an item is one block, or one cluster of blocks (CL).
//
// Shared memory of a block (bytes):
//   [0,16) mbarrier
//   rank 0 only:  nd[5 NN]  the reduced tree (one node per segment: its separator; per node the
//                 record {D -> f, B -> c -> x, U, pd, pb}), NN = nodes rounded up | item metadata
//                 (level_begin, branch desc, pnode)
//   sd[L] su[L] sb[L]  the chunk's d, u, b in natural order, L = chunk range widened to 16-byte
//                 boundaries; compartment j of the chunk sits at index j + off | segment descriptors
// Blocks of rank > 0 write their separators into rank 0's reduced arrays through distributed shared
// memory and read the separators' solution back from there.
//
// Phases:
//   P1 condense   every segment's interior a..b-1 is eliminated top-down, independently of the tree
//                 level (one lane per segment).  Node i keeps g = u[i+1]/D, h = e/D, c = B/D where e is
//                 the fill-in coupling to the separator t above the segment.  What is left of the
//                 separator b (pivot, right-hand side, coupling U to t) and the interior's contribution
//                 to t (sum h e, sum h B) go to the reduced arrays.
//   P2 reduced    the level-synchronous Hines sweeps of the paper on the reduced
//                 tree: one lane per branch, one step per segment, block barrier per level; at a branch
//                 point the siblings' hand-off values are summed by warp shuffles and the parent pulls
//                 the sum.
//   P3 expand     x[i] = c - g x[i+1] - h x[t] for every interior, again one lane per segment.
// Eliminating in this order is a symmetric permutation of the same LDL^T factorisation (the matrix is
// SPD and strictly diagonally dominant, so any order is stable without pivoting).
// ------------------------------------------------------------------------------------------------
template <typename T, bool CL>
__global__ void __launch_bounds__(384, 2)
hines_resident_kernel(const BlockRec* __restrict__ recs, const int32_t* __restrict__ meta_g,
                      const T* __restrict__ d, const T* __restrict__ u, const T* __restrict__ b, T* x,
                      int64_t n_total, unsigned long long* prof)
{
    extern __shared__ __align__(128) unsigned char smem[];
    namespace cg = cooperative_groups;
    // phase clocks (debug hook, prof == nullptr in normal runs): thread 0 stamps %globaltimer
    unsigned long long stamp[7];
#define HINES_STAMP(k) do { if (prof && threadIdx.x == 0) stamp[k] = globaltimer_ns(); } while (0)
    HINES_STAMP(0);
    constexpr int E = 16 / (int)sizeof(T);
    unsigned rank = 0, csize = 1;
    if (CL) { rank = cg::this_cluster().block_rank(); csize = cg::this_cluster().num_blocks(); }
    // one record per block, in launch order: the block's item and chunk headers side by side, so that
    // a single dependent global load stands between the block's start and its bulk copies
    const ItemHeader it = recs[blockIdx.x].it;
    const ChunkHeader ch = recs[blockIdx.x].ch;
    (void)csize;
    const int tid = threadIdx.x, lane = tid & 31, nthreads = blockDim.x;
    const int off = (int)(ch.comp_begin % E);
    const int64_t g0 = ch.comp_begin - off;                 // 16-byte aligned global element index
    const int L = (off + ch.n + E - 1) / E * E;             // landed elements
    // the last chunk may end beyond a 16-byte boundary of the arrays: copy that remainder by hand
    const int64_t avail = n_total - g0;
    const int Lb = (int)(avail >= L ? L : (avail / E * E)); // elements brought by the bulk copies
    const int NN = (it.nnode + E - 1) / E * E;

    uint64_t* bar = reinterpret_cast<uint64_t*>(smem);
    // rank 0's layout of the reduced arrays; the same offsets address rank 0's memory from any rank
    // node record: 6 values {D -> -f, B -> c, U, -, pd, pb}; the forward sweep reuses them as two
    // {g, c} buffers and two parent ids
    T* nd = reinterpret_cast<T*>(smem + 16);
    int32_t* imeta = reinterpret_cast<int32_t*>(nd + 6 * NN);
    unsigned char* chunk_base = rank == 0 ? reinterpret_cast<unsigned char*>(imeta + it.meta_len) : smem + 16;
    T* sd = reinterpret_cast<T*>(chunk_base);
    T* su = sd + L;
    T* sb = su + L;
    const int4* seg = reinterpret_cast<const int4*>(sb + L);

    if (tid == 0) mbar_init(bar, 1);
    __syncthreads();
    if (tid == 0) {
        const uint32_t bytes = (uint32_t)Lb * sizeof(T);
        const uint32_t mbytes = rank == 0 ? (uint32_t)it.meta_len * 4u : 0u;
        const uint32_t sbytes = (uint32_t)ch.nseg_lanes * 16u;
        mbar_expect_tx(bar, 3u * bytes + mbytes + sbytes);
        if (sbytes) tma_load_1d(const_cast<int4*>(seg), meta_g + ch.seg_off, sbytes, bar);
        if (bytes) {
            tma_load_1d(sd, d + g0, bytes, bar);
            tma_load_1d(sb, b + g0, bytes, bar);
            tma_load_1d(su, u + g0, bytes, bar);
        }
        if (mbytes) tma_load_1d(imeta, meta_g + it.meta_off, mbytes, bar);
    }
    // remainder of the very last chunk (fewer than E elements), plain loads
    for (int i = Lb + tid; i < L && g0 + i < n_total; i += nthreads) { sd[i] = d[g0 + i]; su[i] = u[g0 + i]; sb[i] = b[g0 + i]; }
    // reduced arrays as seen from this block
    T* ND = nd;
    if (CL) {
        cg::cluster_group cluster = cg::this_cluster();
        ND = cluster.map_shared_rank(nd, 0);
        cluster.sync();                                     // every block of the cluster is running
    }
    mbar_wait(bar, 0);
    __syncthreads();
    HINES_STAMP(1);
    const unsigned FULL = 0xffffffffu;

    // ---- P1: condense the interiors of all segments (no level dependency) ----
    // Two lanes per segment [a..b] (b = separator, t = separator above), split at a middle node q: lane A
    // eliminates a..q-1 top-down with fill-in coupling to t and arrives at q; lane B = A ^ 16 eliminates
    // q+1..b-1 top-down with fill-in coupling to q and arrives at b.  A then takes B's contribution to q,
    // eliminates q (couplings to t and to b) and writes the node record of b.  Both lanes run the same code.
    for (int base = (tid & ~31); base < ch.nseg_lanes; base += nthreads) {
        const int4 sg = seg[base + lane];
        const int kind = (sg.y >> 24) & 3, hasq = (sg.y >> 26) & 1;
        const int mt = sg.y & 0xfff, mb = (sg.y >> 12) & 0xfff;
        const bool isB = kind == 2;
        const int m = isB ? mb : (kind == 1 ? mt : 0);
        const int dl = (sg.y >> 27) & 15;                   // the lane starts dl steps late (bank residues, plan.cpp)
        const int mmax = __reduce_max_sync(FULL, m + dl);
        int i = sg.x + off;
        T D = T(1), B = T(0), ee = T(0), ddt = T(0), dbt = T(0), un = T(0), dn = T(0), bn = T(0);
        if (kind == 1 || (isB && hasq)) { D = sd[i]; B = sb[i]; if (isB || sg.w >= 0) ee = su[i]; }
        if (m > 0) { un = su[i + 1]; dn = sd[i + 1]; bn = sb[i + 1]; }
        {
            // The sweep proper, on 32-bit shared addresses: node i at pa (d), pa + LW (u), pa + 2 LW (b); the
            // loop is unrolled by two with the two register sets swapping roles (no register rotation).
            constexpr uint32_t W = (uint32_t)sizeof(T);
            const uint32_t LW = (uint32_t)L * W;
            uint32_t pa = smem_u32(sd + i), pu = pa + LW, pb = pa + 2u * LW;
            T un2 = un, dn2 = dn, bn2 = bn;                 // a lane's first step may fall on either half of the loop body
#define HINES_P1_STEP(UN, DN, BN, UN2, DN2, BN2)                                                     \
            if ((unsigned)sl < (unsigned)m) {                                                        \
                if (sl + 1 < m) { UN2 = lds1<T>(pu + 2u * W); DN2 = lds1<T>(pa + 2u * W); BN2 = lds1<T>(pb + 2u * W); } \
                const T r = rcp<T>(D);                                                               \
                const T g = UN * r, h = ee * r, c = B * r;                                           \
                sts1<T>(pa, g); sts1<T>(pu, h); sts1<T>(pb, c);                                      \
                ddt = fmad<T>(h, ee, ddt); dbt = fmad<T>(h, B, dbt);                                 \
                D = fnma<T>(g, UN, DN); B = fnma<T>(g, B, BN); ee = -h * UN;                         \
                pa += W; pu += W; pb += W;                                                           \
            }                                                                                        \
            ++sl;
            int sl = -dl;
            for (int s = 0; s < mmax; s += 2) {
                HINES_P1_STEP(un, dn, bn, un2, dn2, bn2)
                HINES_P1_STEP(un2, dn2, bn2, un, dn, bn)
            }
#undef HINES_P1_STEP
            i += m;
        }
        // B -> A: what is left of b (pD, pB), its coupling to q (pe), B's contribution parked for q (pdd, pdb)
        const T pD = __shfl_xor_sync(FULL, D, 16), pB = __shfl_xor_sync(FULL, B, 16), pe = __shfl_xor_sync(FULL, ee, 16);
        const T pdd = __shfl_xor_sync(FULL, ddt, 16), pdb = __shfl_xor_sync(FULL, dbt, 16);
        if (kind == 1) {
            T* q = ND + 6 * sg.z;
            if (hasq) {                                     // i is q now
                const T Dq = D - pdd, Bq = B - pdb;
                const T r = rcp<T>(Dq);
                const T gq = pe * r, hq = ee * r;
                sd[i] = gq; su[i] = hq; sb[i] = Bq * r;
                ddt = fmad<T>(hq, ee, ddt); dbt = fmad<T>(hq, Bq, dbt);
                q[0] = fnma<T>(gq, pe, pD); q[1] = fnma<T>(gq, Bq, pB); q[2] = -hq * pe; q[4] = ddt; q[5] = dbt;
            } else {                                        // a segment of one compartment: the separator as it is
                q[0] = D; q[1] = B; q[2] = ee; q[4] = T(0); q[5] = T(0);
            }
        }
    }
    if (CL) cg::this_cluster().sync(); else __syncthreads();
    HINES_STAMP(2);

    if (rank == 0) {
        typedef typename Vec2<T>::type V2;
        // ---- P2 backward on the reduced tree --------------------------------------
        // Sub-trees of at most 32 leaves, one warp per group of sub-trees, lock-step over the height above
        // the leaves.  A node sits in the lane of its first child: that child's hand-off value (f U + parked,
        // f B + parked) is already in the lane's registers, the other children's values come by warp shuffle
        // from their lanes, in ascending lane order.  No shared memory and no barrier on the dependent chain
        // inside a tier; between tiers a block barrier, and the leaves of the upper tier pull the hand-off
        // slots of the tier below.
        {
            const int4* ents = reinterpret_cast<const int4*>(imeta + it.ent_off);
            const int32_t* pull = imeta + it.pull_off;
            const int warp = tid >> 5, nwarps = nthreads >> 5;
            const uint32_t nd_sa = smem_u32(nd);
            for (int tier = 0; tier < it.ntier; ++tier) {
                const int gb = imeta[1 + tier], ge = imeta[2 + tier];
                for (int g = gb + warp; g < ge; g += nwarps) {
                    const int32_t* gh = imeta + it.grp_off + 36 * g;
                    int pos = gh[lane];
                    const int end = gh[lane + 1], nsteps = gh[33];
                    const unsigned char* nshb = reinterpret_cast<const unsigned char*>(imeta) + gh[34];
                    T outd = T(0), outb = T(0);
                    // Node ids are entry indices, so the records of the lane's chain are consecutive: the next
                    // record's address is known without its descriptor (one shared-memory hop, not two).
                    constexpr uint32_t RS = 6u * (uint32_t)sizeof(T), W = (uint32_t)sizeof(T);
                    int4 en = make_int4(0, 0, 0, 0);
                    uint32_t qa = nd_sa + (uint32_t)pos * RS;
                    V2 a0, a2; T U = T(0);
                    a0.x = T(1); a0.y = T(0); a2.x = T(0); a2.y = T(0);
                    int estep = 0x7fffffff;                         // step of the lane's next node
                    if (pos < end) {
                        en = ents[pos];
                        a0 = lds2<T>(qa); U = lds1<T>(qa + 2u * W); a2 = lds2<T>(qa + 4u * W);
                        estep = en.x >> 20;
                    }
                    int nsh = nshb[0];
#pragma unroll 1
                    for (int h = 0; h < nsteps; ++h) {
                        const int nsh_next = h + 1 < nsteps ? nshb[h + 1] : 0;
                        const bool act = estep == h;
                        T sd_ = outd, sb_ = outb;                       // the first child (own lane), or 0 at a leaf
                        if (nsh) {                                      // the other children, by shuffle
                            unsigned m = act ? (unsigned)en.y : 0u;
#pragma unroll 1
                            for (int t = 0; t < nsh; ++t) {
                                const int src = m ? __ffs(m) - 1 : lane;
                                const T vd = __shfl_sync(FULL, outd, src), vb = __shfl_sync(FULL, outb, src);
                                if (m) { sd_ += vd; sb_ += vb; m &= m - 1; }
                            }
                        }
                        // a run = a node and the single-child nodes above it, all on this step (no shuffle, no pull
                        // after the first): the lane walks it node by node
                        while (estep == h) {
                            const int npull = en.w & 0xffff;
                            int run = en.w >> 16;                       // plain nodes behind this one (same step, nothing to pull)
                            if (npull) {                                // children swept in an earlier tier
#pragma unroll 1
                                for (int k = 0; k < npull; ++k) {
                                    const V2 c2 = lds2<T>(nd_sa + (uint32_t)pull[en.z + k] * RS + 4u * W);
                                    sd_ += c2.x; sb_ += c2.y;
                                }
                            }
                            const T D = a0.x - sd_, B = a0.y - sb_;
                            ++pos;
                            const bool more = pos < end;
                            if (more) {                                 // next node: what its step needs first
                                en = ents[pos];
                                a0 = lds2<T>(qa + RS);
                                estep = en.x >> 20;
                            } else {
                                estep = 0x7fffffff;
                            }
                            const T r = rcp<T>(D);
                            const T f = U * r;
                            V2 o; o.x = -f; o.y = B * r;
                            sts2<T>(qa, o);
                            outd = fmad<T>(f, U, a2.x); outb = fmad<T>(f, B, a2.y);
                            if (more) {                                 // ... and what it needs after its reciprocal
                                qa += RS;
                                U = lds1<T>(qa + 2u * W); a2 = lds2<T>(qa + 4u * W);
                            } else {                                    // end of the lane's chain: leave the hand-off in the slot
                                V2 s2; s2.x = outd; s2.y = outb;
                                sts2<T>(qa + 4u * W, s2);
                            }
                            if (run) {
                                // The plain part of the run in a tight loop: records are consecutive, no descriptor is
                                // read, the next record is fetched while this one's reciprocal runs; two register
                                // sets swap roles.  On entry {a0, U, a2} hold the record at qa (= entry pos).
                                V2 b0, b2; T V;
                                b0 = a0; b2 = a2; V = U;
                                pos += run;
                                const bool ends = pos >= end;           // the run takes the lane's chain to its end
#define HINES_RUN_NODE(A0, UU, A2, B0, VV, B2)                                                               \
                                {                                                                            \
                                    const T D_ = A0.x - outd, B_ = A0.y - outb;                              \
                                    if (run > 1 || !ends) { B0 = lds2<T>(qa + RS); VV = lds1<T>(qa + RS + 2u * W); B2 = lds2<T>(qa + RS + 4u * W); } \
                                    const T r_ = rcp<T>(D_);                                                 \
                                    const T f_ = UU * r_;                                                    \
                                    V2 o_; o_.x = -f_; o_.y = B_ * r_;                                       \
                                    sts2<T>(qa, o_);                                                         \
                                    outd = fmad<T>(f_, UU, A2.x); outb = fmad<T>(f_, B_, A2.y);              \
                                    qa += RS;                                                                \
                                }
#pragma unroll 1
                                while (true) {
                                    HINES_RUN_NODE(a0, U, a2, b0, V, b2)
                                    if (--run == 0) { a0 = b0; U = V; a2 = b2; break; }
                                    HINES_RUN_NODE(b0, V, b2, a0, U, a2)
                                    if (--run == 0) break;
                                }
#undef HINES_RUN_NODE
                                if (ends) {
                                    V2 s2; s2.x = outd; s2.y = outb;
                                    sts2<T>(qa - RS + 4u * W, s2);
                                    estep = 0x7fffffff;
                                } else {
                                    en = ents[pos];
                                    estep = en.x >> 20;
                                }
                            }
                            sd_ = outd; sb_ = outb;                     // the next node of the run has this one as its only child
                        }
                        nsh = nsh_next;
                    }
                    // A chain that ended in a root turns around: x_root = c_root, then x = c - f x_parent down the
                    // lane's own chain (records consecutive, loads independent of the chain); these nodes are final
                    // before the pointer jumping ({g, c} := {0, x}).
                    if ((gh[35] >> lane) & 1) {
                        const int begin = gh[lane];
                        uint32_t qk = nd_sa + (uint32_t)(end - 1) * RS;
                        T xv = lds1<T>(qk + W);
                        int k = end - 2;
                        for (; k - 3 >= begin; k -= 4) {                // four records in flight under one chain
                            const V2 g0 = lds2<T>(qk - RS), g1 = lds2<T>(qk - 2u * RS), g2 = lds2<T>(qk - 3u * RS), g3 = lds2<T>(qk - 4u * RS);
                            V2 o; o.x = T(0);
                            xv = fmad<T>(g0.x, xv, g0.y); o.y = xv; sts2<T>(qk - RS, o);
                            xv = fmad<T>(g1.x, xv, g1.y); o.y = xv; sts2<T>(qk - 2u * RS, o);
                            xv = fmad<T>(g2.x, xv, g2.y); o.y = xv; sts2<T>(qk - 3u * RS, o);
                            xv = fmad<T>(g3.x, xv, g3.y); o.y = xv; sts2<T>(qk - 4u * RS, o);
                            qk -= 4u * RS;
                        }
                        for (; k >= begin; --k) {
                            qk -= RS;
                            const V2 gc = lds2<T>(qk);
                            xv = fmad<T>(gc.x, xv, gc.y);
                            V2 o; o.x = T(0); o.y = xv;
                            sts2<T>(qk, o);
                        }
                    }
                }
                __syncthreads();
            }
        }
    }
    HINES_STAMP(3);                 // outside the rank test: a stamp in both arms of it splits warp 0 for all of P2
    if (rank == 0) {
        const int32_t* pnode = imeta + it.pnode_off;
        typedef typename Vec2<T>::type V2;
        // ---- P2 forward by pointer jumping over the reduced tree --------------
        // x_v = c_v + g_v x_p(v), g = -f, g_root = 0.  One round replaces (g_v, c_v, p(v)) by
        // (g_v g_p, c_v + g_v c_p, p(p(v))): after `rounds` rounds (2^rounds >= nodes on the longest
        // root path) every g is 0 and c is x.  All nodes work in every round, with one barrier per
        // round instead of one per level.  Buffers: record slots {0,1} and {2,3}; parent ids in {4,5}.
        for (int r = 0; r < it.rounds; ++r) {
            const int sbuf = 2 * (r & 1), dbuf = 2 - sbuf;
            for (int v = tid; v < it.nnode; v += nthreads) {
                int* ip = reinterpret_cast<int*>(nd + 6 * v + 4);
                const int p = r == 0 ? pnode[v] : ip[(r - 1) & 1];
                const V2 a = *reinterpret_cast<const V2*>(nd + 6 * v + sbuf);
                const V2 ap = *reinterpret_cast<const V2*>(nd + 6 * p + sbuf);
                const int pp = r == 0 ? pnode[p] : reinterpret_cast<const int*>(nd + 6 * p + 4)[(r - 1) & 1];
                V2 o; o.x = a.x * ap.x; o.y = fmad<T>(a.x, ap.y, a.y);
                *reinterpret_cast<V2*>(nd + 6 * v + dbuf) = o;
                ip[r & 1] = pp;
            }
            __syncthreads();
        }
    }
    if (CL) cg::this_cluster().sync();
    HINES_STAMP(4);

    const int xs = 2 * (it.rounds & 1) + 1;               // record slot that holds x after the forward sweep
    // ---- P3: expand the interiors: A computes x[q] from x[b] and x[t]; then A walks up from q-1 to a
    //      (x[i] = c - g x[i+1] - h x[t]) and B walks up from b-1 to q+1 (x[i] = c - g x[i+1] - h x[q]), one FMA
    //      on the dependent chain per step ----
    for (int base = (tid & ~31); base < ch.nseg_lanes; base += nthreads) {
        const int4 sg = seg[base + lane];
        const int kind = (sg.y >> 24) & 3, hasq = (sg.y >> 26) & 1;
        const int mt = sg.y & 0xfff, mb = (sg.y >> 12) & 0xfff;
        const bool isB = kind == 2;
        const int m = isB ? mb : (kind == 1 ? mt : 0);
        const int dl = (sg.y >> 27) & 15;
        const int mmax = __reduce_max_sync(FULL, m + dl);
        const int p0 = sg.x + off;
        T xb = T(0), xt = T(0), xn = T(0);
        if (kind != 0) xb = ND[6 * sg.z + xs];
        if (kind == 1) {
            if (sg.w >= 0) xt = ND[6 * sg.w + xs];
            if (hasq) {
                const int iq = p0 + mt;
                xn = fnma<T>(sd[iq], xb, fnma<T>(su[iq], xt, sb[iq]));
                sb[iq] = xn; sb[iq + 1 + mb] = xb;
            } else {
                sb[p0] = xb;
            }
        }
        const T xq = __shfl_xor_sync(FULL, xn, 16);
        if (isB) { xn = xb; xt = xq; }
        T g1 = T(0), h1 = T(0), c1 = T(0);
        if (m > 0) { const int i = p0 + m - 1; g1 = sd[i]; h1 = su[i]; c1 = sb[i]; }
        for (int jj = mmax - 1; jj >= 0; --jj) {
            const int j = jj - dl;                          // the lane's own step: the same residue shift as in P1
            if ((unsigned)j < (unsigned)m) {
                T g2 = T(0), h2 = T(0), c2 = T(0);
                if (j > 0) { const int i2 = p0 + j - 1; g2 = sd[i2]; h2 = su[i2]; c2 = sb[i2]; }
                xn = fnma<T>(g1, xn, fnma<T>(h1, xt, c1));       // one FMA on the dependent chain
                sb[p0 + j] = xn;
                g1 = g2; h1 = h2; c1 = c2;
            }
        }
    }

    // ---- store x (natural order): bulk store of the 16-byte aligned interior, edges by hand ----
    const int head_end = min(ch.n, (E - off) % E);                     // chunk-local [0, head_end)
    const int tail_begin = max(head_end, (int)(((off + ch.n) / E) * E) - off);   // chunk-local [tail_begin, n)
    fence_proxy_async();
    __syncthreads();
    HINES_STAMP(5);
    if (tid == 0 && tail_begin > head_end) {
        tma_store_1d(x + ch.comp_begin + head_end, sb + off + head_end, (uint32_t)(tail_begin - head_end) * sizeof(T));
        tma_store_commit_wait();
    }
    for (int j = tid; j < head_end; j += nthreads) x[ch.comp_begin + j] = sb[off + j];
    for (int j = tail_begin + tid; j < ch.n; j += nthreads) x[ch.comp_begin + j] = sb[off + j];
    if (prof && tid == 0) {
        stamp[6] = globaltimer_ns();
        unsigned long long* o = prof + 8 * (size_t)blockIdx.x;
        for (int k = 0; k < 7; ++k) o[k] = stamp[k];
        o[7] = ((unsigned long long)smid() << 32) | (unsigned)ch.n;
    }
    if (CL) cg::this_cluster().sync();          // rank 0's shared memory stays alive while others read it
#undef HINES_STAMP
}

// ------------------------------------------------------------------------------------------------
// Streaming path: one launch per level, one thread per branch, lanes of a warp = 32 branches of
// similar length (sorted at setup).  f and c go to the plan's workspace.
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void hines_stream_backward(const StreamDesc* __restrict__ desc, int64_t begin, int64_t end,
                                      const int2* __restrict__ child, const T* __restrict__ d,
                                      const T* __restrict__ u, const T* __restrict__ b,
                                      T* __restrict__ wf, T* __restrict__ wc)
{
    const int64_t e = begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= end) return;
    const StreamDesc s = desc[e];
    const T* dp = d + s.gstart; const T* up = u + s.gstart; const T* bp = b + s.gstart;
    T* fp = wf + s.ws; T* cp = wc + s.ws;
    T D = dp[s.len - 1], B = bp[s.len - 1];
    // pull the children's contributions (ascending child id): d' -= f_c u_c, b' -= u_c c_c (= f_c b'_c)
    for (int k = 0; k < s.nchild; ++k) {
        const int2 ch = child[s.child_begin + k];
        const T uc = u[ch.x];
        D = fnma<T>(wf[ch.y], uc, D);
        B = fnma<T>(uc, wc[ch.y], B);
    }
    for (int k = s.len - 1; k >= 1; --k) {
        const T r = rcp<T>(D);
        const T uk = up[k];
        const T f = uk * r;
        fp[k] = f; cp[k] = B * r;
        D = fnma<T>(f, uk, dp[k - 1]);
        B = fnma<T>(f, B, bp[k - 1]);
    }
    const T r = rcp<T>(D);
    fp[0] = s.gparent >= 0 ? up[0] * r : T(0);
    cp[0] = B * r;
}

template <typename T>
__global__ void hines_stream_forward(const StreamDesc* __restrict__ desc, int64_t begin, int64_t end,
                                     const T* __restrict__ wf, const T* __restrict__ wc, T* x)
{
    const int64_t e = begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= end) return;
    const StreamDesc s = desc[e];
    const T* fp = wf + s.ws; const T* cp = wc + s.ws;
    T* xo = x + s.gstart;
    T xp = s.gparent >= 0 ? x[s.gparent] : T(0);
    for (int k = 0; k < s.len; ++k) { xp = fnma<T>(fp[k], xp, cp[k]); xo[k] = xp; }
}

// ------------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------------
template <typename V>
static hines_status_t upload_vec(const V& v, void** dst, int64_t& total)
{
    *dst = nullptr;
    const size_t bytes = v.size() * sizeof(v[0]);
    if (!bytes) return HINES_OK;
    CUDA_TRY(cudaMalloc(dst, bytes));
    CUDA_TRY(cudaMemcpy(*dst, v.data(), bytes, cudaMemcpyHostToDevice));
    total += (int64_t)bytes;
    return HINES_OK;
}

static void free_device(DeviceTables* D)
{
    if (!D) return;
    cudaFree(D->recs); cudaFree(D->item_meta); cudaFree(D->stream_desc);
    cudaFree(D->stream_child); cudaFree(D->ws_f); cudaFree(D->ws_c); cudaFree(D->prof);
    for (void* p : D->host_stage) cudaFree(p);
    for (cudaEvent_t e : D->ev) if (e) cudaEventDestroy(e);
    for (cudaStream_t t : D->side) if (t) cudaStreamDestroy(t);
    for (cudaEvent_t e : D->join) if (e) cudaEventDestroy(e);
    if (D->fork) cudaEventDestroy(D->fork);
    if (D->sstream) cudaStreamDestroy(D->sstream);
    if (D->sjoin) cudaEventDestroy(D->sjoin);
    delete D;
}

static hines_status_t upload(hines_plan* P)
{
    if (P->dev) return HINES_OK;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        set_error("no CUDA device: this library has no CPU fallback");
        return HINES_ERR_CUDA;
    }
    DeviceTables* D = new (std::nothrow) DeviceTables();
    if (!D) { set_error("host allocation failed"); return HINES_ERR_ALLOC; }
    hines_status_t st = HINES_OK;
    auto run = [&]() -> hines_status_t {
        CUDA_TRY(cudaGetDevice(&D->device));
        int max_optin = 0;
        CUDA_TRY(cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, D->device));
        for (int32_t s : P->class_smem_bytes)
            if (s > max_optin) {
                set_error("device offers " + std::to_string(max_optin) + " bytes of shared memory per block, plan needs " + std::to_string(s));
                return HINES_ERR_UNSUPPORTED;
            }
        {
            std::vector<BlockRec> recs;
            recs.reserve(P->chunk_headers.size());
            for (int32_t item : P->item_launch_order) {
                const ItemHeader& h = P->item_headers[item];
                for (int32_t r = 0; r < h.nchunks; ++r) recs.push_back(BlockRec{h, P->chunk_headers[h.first_chunk + r]});
            }
            if ((st = upload_vec(recs, (void**)&D->recs, D->bytes))) return st;
        }
        if ((st = upload_vec(P->item_meta, (void**)&D->item_meta, D->bytes))) return st;
        if ((st = upload_vec(P->stream_desc, (void**)&D->stream_desc, D->bytes))) return st;
        if ((st = upload_vec(P->stream_child, (void**)&D->stream_child, D->bytes))) return st;
        if (P->n_stream_unknowns) {
            const size_t wb = (size_t)P->n_stream_unknowns * P->width;
            CUDA_TRY(cudaMalloc(&D->ws_f, wb));
            CUDA_TRY(cudaMalloc(&D->ws_c, wb));
            D->bytes += 2 * (int64_t)wb;
        }
        int32_t max_smem[2] = {0, 0};
        bool nonportable = false;
        for (size_t q = 0; q < P->class_smem_bytes.size(); ++q) {
            const int cl = P->class_cluster[q] > 1;
            max_smem[cl] = std::max(max_smem[cl], P->class_smem_bytes[q]);
            nonportable |= P->class_cluster[q] > 8;
        }
        if (P->dtype == HINES_F64) {
            if (max_smem[0]) CUDA_TRY(cudaFuncSetAttribute(hines_resident_kernel<double, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem[0]));
            if (max_smem[1]) CUDA_TRY(cudaFuncSetAttribute(hines_resident_kernel<double, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem[1]));
            if (nonportable) CUDA_TRY(cudaFuncSetAttribute(hines_resident_kernel<double, true>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        } else {
            if (max_smem[0]) CUDA_TRY(cudaFuncSetAttribute(hines_resident_kernel<float, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem[0]));
            if (max_smem[1]) CUDA_TRY(cudaFuncSetAttribute(hines_resident_kernel<float, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem[1]));
            if (nonportable) CUDA_TRY(cudaFuncSetAttribute(hines_resident_kernel<float, true>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        }
        const bool has_stream_path = P->stream_level_begin.size() > 1;
        if (P->class_smem_bytes.size() + (has_stream_path ? 1 : 0) > 1 && !(P->opt.policy_flags & HINES_POLICY_SERIAL_CLASSES)) {
            CUDA_TRY(cudaEventCreateWithFlags(&D->fork, cudaEventDisableTiming));
            if (has_stream_path && !P->class_smem_bytes.empty()) {
                CUDA_TRY(cudaStreamCreateWithFlags(&D->sstream, cudaStreamNonBlocking));
                CUDA_TRY(cudaEventCreateWithFlags(&D->sjoin, cudaEventDisableTiming));
            }
            for (int k = 0; k < DeviceTables::kSide; ++k) {
                CUDA_TRY(cudaStreamCreateWithFlags(&D->side[k], cudaStreamNonBlocking));
                CUDA_TRY(cudaEventCreateWithFlags(&D->join[k], cudaEventDisableTiming));
            }
        }
        return HINES_OK;
    };
    st = run();
    if (st != HINES_OK) { free_device(D); return st; }
    P->dev = D;
    return HINES_OK;
}

template <typename T>
static hines_status_t launch_all(hines_plan* P, const T* d, const T* u, const T* b, T* x, cudaStream_t stream)
{
    DeviceTables* D = P->dev;
    if (D->timing) CUDA_TRY(cudaEventRecord(D->ev[0], stream));
    auto launch_streaming = [&](cudaStream_t ss) -> hines_status_t {
        const int nlev = (int)P->stream_level_begin.size() - 1;
        const int st = P->opt.stream_threads;
        T* wf = static_cast<T*>(D->ws_f); T* wc = static_cast<T*>(D->ws_c);
        for (int l = nlev - 1; l >= 0; --l) {
            const int64_t b0 = P->stream_level_begin[l], b1 = P->stream_level_begin[l + 1];
            hines_stream_backward<T><<<(unsigned)((b1 - b0 + st - 1) / st), st, 0, ss>>>(
                D->stream_desc, b0, b1, reinterpret_cast<const int2*>(D->stream_child), d, u, b, wf, wc);
        }
        for (int l = 0; l < nlev; ++l) {
            const int64_t b0 = P->stream_level_begin[l], b1 = P->stream_level_begin[l + 1];
            hines_stream_forward<T><<<(unsigned)((b1 - b0 + st - 1) / st), st, 0, ss>>>(
                D->stream_desc, b0, b1, wf, wc, x);
        }
        CUDA_TRY(cudaGetLastError());
        return HINES_OK;
    };
    // size classes are independent: the first runs on the caller's stream, the others on side streams
    // forked from it and joined back, so that their blocks share the SMs and fill each other's tails
    int64_t first_block = 0;
    const bool forked = D->fork != nullptr;
    bool used[DeviceTables::kSide] = {false, false, false};
    if (forked) CUDA_TRY(cudaEventRecord(D->fork, stream));
    if (D->sstream) {                                   // cells of the streaming path are independent of the rest
        CUDA_TRY(cudaStreamWaitEvent(D->sstream, D->fork, 0));
        if (hines_status_t sst = launch_streaming(D->sstream)) return sst;
        CUDA_TRY(cudaEventRecord(D->sjoin, D->sstream));
    }
    int nth = 0;
    for (size_t q = 0; q < P->class_smem_bytes.size(); ++q) {
        const int64_t cnt = P->class_count[q];
        if (!cnt) continue;
        const int cl = P->class_cluster[q];
        cudaStream_t ls = stream;
        if (forked && nth > 0) {
            const int k = (nth - 1) % DeviceTables::kSide;
            ls = D->side[k];
            if (!used[k]) { CUDA_TRY(cudaStreamWaitEvent(ls, D->fork, 0)); used[k] = true; }
        }
        ++nth;
        unsigned long long* prof = D->prof_on ? D->prof + 8 * first_block : nullptr;
        const BlockRec* recs = D->recs + first_block;
        if (cl == 1) {
            hines_resident_kernel<T, false><<<(unsigned)cnt, P->class_threads[q], P->class_smem_bytes[q], ls>>>(
                recs, D->item_meta, d, u, b, x, P->n, prof);
        } else {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)(cnt * cl));
            cfg.blockDim = dim3((unsigned)P->class_threads[q]);
            cfg.dynamicSmemBytes = (size_t)P->class_smem_bytes[q];
            cfg.stream = ls;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeClusterDimension;
            attr[0].val.clusterDim.x = (unsigned)cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
            cfg.attrs = attr; cfg.numAttrs = 1;
            CUDA_TRY(cudaLaunchKernelEx(&cfg, hines_resident_kernel<T, true>, recs, (const int32_t*)D->item_meta, d, u, b, x,
                                        (int64_t)P->n, prof));
        }
        first_block += cnt * cl;
    }
    for (int k = 0; k < DeviceTables::kSide; ++k)
        if (used[k]) { CUDA_TRY(cudaEventRecord(D->join[k], D->side[k])); CUDA_TRY(cudaStreamWaitEvent(stream, D->join[k], 0)); }
    if (D->timing) CUDA_TRY(cudaEventRecord(D->ev[1], stream));
    if (D->sstream) CUDA_TRY(cudaStreamWaitEvent(stream, D->sjoin, 0));
    else if (hines_status_t sst = launch_streaming(stream)) return sst;
    if (D->timing) { CUDA_TRY(cudaEventRecord(D->ev[2], stream)); D->timed_once = true; }
    CUDA_TRY(cudaGetLastError());
    return HINES_OK;
}

static hines_status_t check_ptrs(const hines_plan* P, const void* d, const void* u, const void* b, const void* x)
{
    if (!P || !d || !u || !b || !x) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    return HINES_OK;
}

}  // namespace hines

using namespace hines;

extern "C" {

hines_status_t hines_plan_upload(hines_plan_t* P)
{
    if (!P) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    return upload(P);
}

hines_status_t hines_solve(hines_plan_t* P, const void* d, const void* u, const void* b, void* x, hines_stream_t stream)
{
    hines_status_t st = check_ptrs(P, d, u, b, x);
    if (st != HINES_OK) return st;
    if (((uintptr_t)d | (uintptr_t)u | (uintptr_t)b | (uintptr_t)x) & 15) {
        set_error("device pointers must be 16-byte aligned"); return HINES_ERR_INVALID_ARG;
    }
    if (d == x || u == x) { set_error("x may alias b only"); return HINES_ERR_INVALID_ARG; }
    if ((st = upload(P)) != HINES_OK) return st;
    if (P->dtype == HINES_F64)
        return launch_all<double>(P, (const double*)d, (const double*)u, (const double*)b, (double*)x, (cudaStream_t)stream);
    return launch_all<float>(P, (const float*)d, (const float*)u, (const float*)b, (float*)x, (cudaStream_t)stream);
}

hines_status_t hines_solve_host(hines_plan_t* P, const void* d, const void* u, const void* b, void* x, hines_stream_t stream)
{
    hines_status_t st = check_ptrs(P, d, u, b, x);
    if (st != HINES_OK) return st;
    if ((st = upload(P)) != HINES_OK) return st;
    DeviceTables* D = P->dev;
    const size_t bytes = (size_t)P->n * P->width;
    for (int k = 0; k < 4; ++k)
        if (!D->host_stage[k]) { CUDA_TRY(cudaMalloc(&D->host_stage[k], bytes)); D->bytes += (int64_t)bytes; }
    cudaStream_t s = (cudaStream_t)stream;
    CUDA_TRY(cudaMemcpyAsync(D->host_stage[0], d, bytes, cudaMemcpyHostToDevice, s));
    CUDA_TRY(cudaMemcpyAsync(D->host_stage[1], u, bytes, cudaMemcpyHostToDevice, s));
    CUDA_TRY(cudaMemcpyAsync(D->host_stage[2], b, bytes, cudaMemcpyHostToDevice, s));
    st = hines_solve(P, D->host_stage[0], D->host_stage[1], D->host_stage[2], D->host_stage[3], stream);
    if (st != HINES_OK) return st;
    CUDA_TRY(cudaMemcpyAsync(x, D->host_stage[3], bytes, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    return HINES_OK;
}

hines_status_t hines_plan_enable_timing(hines_plan_t* P, int32_t enable)
{
    if (!P) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    hines_status_t st = upload(P);
    if (st != HINES_OK) return st;
    DeviceTables* D = P->dev;
    if (enable)
        for (auto& e : D->ev) if (!e) CUDA_TRY(cudaEventCreate(&e));
    D->timing = enable != 0;
    D->timed_once = false;
    return HINES_OK;
}

hines_status_t hines_plan_get_timing(hines_plan_t* P, float* resident_ms, float* stream_ms)
{
    if (!P || !resident_ms || !stream_ms) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (!P->dev || !P->dev->timing || !P->dev->timed_once) { set_error("timing not enabled or no solve yet"); return HINES_ERR_INVALID_ARG; }
    DeviceTables* D = P->dev;
    CUDA_TRY(cudaEventSynchronize(D->ev[2]));
    CUDA_TRY(cudaEventElapsedTime(resident_ms, D->ev[0], D->ev[1]));
    CUDA_TRY(cudaEventElapsedTime(stream_ms, D->ev[1], D->ev[2]));
    return HINES_OK;
}

hines_status_t hines_plan_enable_phase_clocks(hines_plan_t* P, int32_t enable)
{
    if (!P) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    hines_status_t st = upload(P);
    if (st != HINES_OK) return st;
    DeviceTables* D = P->dev;
    const size_t bytes = P->chunk_headers.size() * 8 * sizeof(unsigned long long);
    if (enable && !D->prof && bytes) {
        CUDA_TRY(cudaMalloc(&D->prof, bytes));
        CUDA_TRY(cudaMemset(D->prof, 0, bytes));
        D->bytes += (int64_t)bytes;
    }
    D->prof_on = enable != 0 && D->prof;
    return HINES_OK;
}

hines_status_t hines_plan_get_phase_clocks(hines_plan_t* P, uint64_t* host_dst, int64_t capacity_bytes, int64_t* needed_bytes)
{
    if (!P || !needed_bytes) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    const int64_t bytes = (int64_t)(P->chunk_headers.size() * 8 * sizeof(unsigned long long));
    *needed_bytes = bytes;
    if (!host_dst) return HINES_OK;
    if (!P->dev || !P->dev->prof) { set_error("phase clocks not enabled"); return HINES_ERR_INVALID_ARG; }
    if (capacity_bytes < bytes) { set_error("buffer too small"); return HINES_ERR_INVALID_ARG; }
    CUDA_TRY(cudaDeviceSynchronize());
    CUDA_TRY(cudaMemcpy(host_dst, P->dev->prof, (size_t)bytes, cudaMemcpyDeviceToHost));
    return HINES_OK;
}

hines_status_t hines_plan_destroy(hines_plan_t* P)
{
    if (!P) return HINES_OK;
    free_device(P->dev);
    delete P;
    return HINES_OK;
}

}  // extern "C"

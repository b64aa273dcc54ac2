// hines_solve: the per-step kernels (sm_100a) and their host launcher.
//
// Two paths, chosen per cell by the plan:
//   resident  whole cells / cell groups, or the parts of a large cell, staged into shared memory by TMA bulk
//             copies (cp.async.bulk + mbarrier) of their runs of consecutive compartments.  Segment interiors
//             are condensed before (P1) and expanded after (P3) the level-synchronous sweeps (P2) over the
//             reduced forest of the part: one node per segment, one thread per node, a block barrier per
//             level, the parent pulling its children's hand-off values.
//             Parts of one cell exchange two values per exported sub-tree root through distributed shared
//             memory (cluster items) or a global exchange buffer between launches (split items).  d,u,b are
//             read from and x written to the caller's natural-order arrays directly: the paper's separate
//             permute kernels do not exist here.
//   stream    cells that fit none of this: one launch per level over all such cells (global synchronisation
//             = kernel boundary, which PAPER.md:114 avoids by requiring one matrix per block), intermediates
//             in a plan-owned global workspace.
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

struct DeviceTables {
    int device = -1, num_sms = 148;
    BlockRecord* recs = nullptr;                                  // one per launched block, launch order (class by class)
    int32_t* meta = nullptr;
    int4* runs = nullptr;
    void* xch_h = nullptr;          // split items: exported hand-off values (2 per slot)
    void* xch_x = nullptr;          // split items: the parent's x of every exported sub-tree root
    void* fac[3] = {nullptr, nullptr, nullptr};   // f3: the factor arrays of hines_factor (N values each)
    bool factored = false;          // hines_factor has run
    StreamDesc* stream_desc = nullptr;
    int32_t* stream_child = nullptr;
    void* ws_f = nullptr;           // streaming workspace: f (n_stream_unknowns elements)
    void* ws_c = nullptr;           // streaming workspace: c
    void* host_stage[4] = {nullptr, nullptr, nullptr, nullptr};   // hines_solve_host device buffers d,u,b,x
    cudaStream_t copy_stream = nullptr;                           // hines_solve_host: D2H of x beside the H2D of the next slice
    cudaEvent_t slice_ev[2] = {nullptr, nullptr};
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};     // timing hook: resident start/end on the caller's stream, streaming start/end
    static const int kSide = 3;                                   // side streams: size classes run concurrently
    cudaStream_t side[kSide] = {nullptr, nullptr, nullptr};
    cudaEvent_t fork = nullptr, join[kSide] = {nullptr, nullptr, nullptr};
    cudaStream_t sstream = nullptr;                               // the streaming path runs beside the resident classes
    cudaEvent_t sjoin = nullptr;
    cudaStream_t pstream = nullptr;                               // the three phases of split items, in order, beside the rest
    cudaEvent_t pjoin = nullptr;
    bool timing = false, timed_once = false;
    unsigned long long* prof = nullptr;                           // phase clocks: 8 x u64 per launched block, launch order
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
__device__ __forceinline__ void tma_load_1d_sa(uint32_t dst_sa, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_sa), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
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
__device__ __forceinline__ int ldsi1(uint32_t a)
{ int v; asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ int4 ldsi4(uint32_t a)
{ int4 v; asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory"); return v; }
template <typename T> __device__ __forceinline__ void sts1(uint32_t a, T v);
template <> __device__ __forceinline__ void sts1<double>(uint32_t a, double v)
{ asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
template <> __device__ __forceinline__ void sts1<float>(uint32_t a, float v)
{ asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void stsi1(uint32_t a, int v) { asm volatile("st.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
template <typename T> __device__ __forceinline__ void sts2(uint32_t a, typename Vec2<T>::type v);
template <> __device__ __forceinline__ void sts2<double>(uint32_t a, double2 v)
{ asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.x), "d"(v.y) : "memory"); }
template <> __device__ __forceinline__ void sts2<float>(uint32_t a, float2 v)
{ asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(v.x), "f"(v.y) : "memory"); }
template <typename T> __device__ __forceinline__ T fmad(T a, T b, T c);   // c + a*b
template <> __device__ __forceinline__ double fmad<double>(double a, double b, double c) { return fma(a, b, c); }
template <> __device__ __forceinline__ float fmad<float>(float a, float b, float c) { return fmaf(a, b, c); }

// programmatic dependent launch (split items): the next launch of the stream may start while this one runs, and waits
// for this one's completion (and the visibility of its writes) only where it needs its results
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// split-phase cluster barrier (every thread of every block of the cluster arrives and waits, in turn)
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
// shared-memory address of the same variable in block `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
// store into another block's shared memory that counts its bytes on THAT block's mbarrier: data and signal in one
__device__ __forceinline__ void st_async_2(uint32_t raddr, double a, double b, uint32_t rbar)
{
    asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(raddr), "d"(a), "d"(b), "r"(rbar) : "memory");
}
__device__ __forceinline__ void st_async_2(uint32_t raddr, float a, float b, uint32_t rbar)
{
    asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];" ::"r"(raddr), "f"(a), "f"(b), "r"(rbar) : "memory");
}
__device__ __forceinline__ void st_async_1(uint32_t raddr, double a, uint32_t rbar)
{
    asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(raddr), "d"(a), "r"(rbar) : "memory");
}
__device__ __forceinline__ void st_async_1(uint32_t raddr, float a, uint32_t rbar)
{
    asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.f32 [%0], %1, [%2];" ::"r"(raddr), "f"(a), "r"(rbar) : "memory");
}
// wait for a phase of an mbarrier that blocks of the whole cluster complete
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAITC_LOOP:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAITC_DONE;\n"
        "bra WAITC_LOOP;\n"
        "WAITC_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}


// P2 backward over the levels lfrom .. lto of a part's reduced forest: deepest level first, one
// thread per node, a block barrier per level; a node pulls the hand-off values of its children.
// topsel selects the nodes of this sweep: 0 = nodes that do not wait for another part, 1 = top nodes (the
// ancestors of ghost children).  What the critical warp executes between two barriers is what a level costs
// (a lone warp issues dependent code at about 5 cycles per instruction), so the step is kept short: the plan
// stores, per node, the byte offsets of its first two children's hand-off slots (the all-zero record when there is
// none: no branch), more than two children are rare and take a loop; the record and descriptor of a thread's node
// on the NEXT level are fetched after this level's stores and land while the barrier is pending.
// Node record: {D -> g = -f, B -> c, -U, -, parked d -> hand-off d, parked b -> hand-off b}.
__device__ __forceinline__ void named_barrier(int nthreads_in)
{
    asm volatile("bar.sync 1, %0;" ::"r"(nthreads_in) : "memory");
}

// MODE 0: the whole step; 1 (factor): the pivot part only, the record keeps {g, r}; 2 (right-hand side): r comes from
// record slot 3, g stays as it is, no reciprocal.
template <typename T, int MODE>
__device__ __forceinline__ void node_step(uint32_t nd_sa, uint32_t qa, const int4 k, typename Vec2<T>::type a0, T Un,
                                          typename Vec2<T>::type a2)
{
    typedef typename Vec2<T>::type V2;
    constexpr uint32_t W = (uint32_t)sizeof(T), RS = 6u * W;
    const V2 h0 = lds2<T>(nd_sa + (uint32_t)k.x), h1 = lds2<T>(nd_sa + (uint32_t)k.y);
    T D = a0.x - h0.x, B = a0.y - h0.y;
    D -= h1.x; B -= h1.y;
    if (k.z & (1 << 28)) {                                  // more than two children (rare): the rest, consecutive records
        uint32_t ca = nd_sa + (uint32_t)k.y + RS;
#pragma unroll 1
        for (int nc = (k.z & 0xfff) - 2; nc > 0; --nc, ca += RS) { const V2 h = lds2<T>(ca); D -= h.x; B -= h.y; }
    }
    if (MODE == 2) {
        const T r = lds1<T>(qa + 3u * W);
        V2 o; o.x = a0.x; o.y = B * r;                      // g = -f is a factor; c = B r
        sts2<T>(qa, o);
        V2 s2; s2.x = T(0); s2.y = fnma<T>(a0.x, B, a2.y);
        sts2<T>(qa + 4u * W, s2);
    } else {
        const T r = rcp<T>(D);
        const T g = Un * r;                                 // -f
        V2 o; o.x = g; o.y = MODE == 1 ? r : B * r;
        sts2<T>(qa, o);
        V2 s2; s2.x = fmad<T>(g, Un, a2.x); s2.y = fnma<T>(g, B, a2.y);
        sts2<T>(qa + 4u * W, s2);
    }
}

// A level wider than the block (rare: a part with more nodes on one level than the block has threads): every thread loops
// over the level's nodes.  Out of line: code that hardly ever runs should not sit between the phases of the kernel
// (its instructions would take room in the instruction cache's lines).
template <typename T, int MODE>
__device__ __noinline__ void sweep_backward_wide(uint32_t nd_sa, uint32_t lb_sa, uint32_t kp_sa, int lfrom, int lto,
                                                 int topsel, int tid, int nthreads)
{
    typedef typename Vec2<T>::type V2;
    constexpr uint32_t W = (uint32_t)sizeof(T), RS = 6u * W;
#pragma unroll 1
    for (int l = lfrom; l >= lto; --l) {
        const int hi = ldsi1(lb_sa + 4u * (uint32_t)(l + 1));
        for (int v = ldsi1(lb_sa + 4u * (uint32_t)l) + tid; v < hi; v += nthreads) {
            const int4 k = ldsi4(kp_sa + 16u * (uint32_t)v);
            if (k.z >= 0 && ((k.z >> 29) & 1) == topsel) {
                const uint32_t qa = nd_sa + (uint32_t)v * RS;
                const V2 a0 = lds2<T>(qa), a2 = lds2<T>(qa + 4u * W);
                const T Un = lds1<T>(qa + 2u * W);
                node_step<T, MODE>(nd_sa, qa, k, a0, Un, a2);
            }
        }
        __syncthreads();
    }
}

template <typename T, int MODE>
__device__ __forceinline__ void sweep_backward(uint32_t nd_sa, uint32_t lb_sa, uint32_t kp_sa, int lfrom, int lto,
                                               int topsel, int maxwidth, int tid, int nthreads)
{
    typedef typename Vec2<T>::type V2;
    constexpr uint32_t W = (uint32_t)sizeof(T), RS = 6u * W;
    if (lfrom < lto) return;
    if (maxwidth <= nthreads) {
        // No level is wider than the block: at most one node per thread and level, and only the warps that can ever
        // hold a node take part (named barrier over those; the others wait at the block barrier behind the sweep).
        const int pthreads = (maxwidth + 31) & ~31;
        tid = nthreads - 1 - tid;                           // the LAST warps of the block sweep: P1 / P3 fill the first ones
        if (tid < pthreads) {
            // the thread's node on a level: index lb[l] + tid, if that is below lb[l + 1].  Whether the node takes part in
            // this sweep is read off its info word (bit 31: a ghost child, bit 29: a top node) when the step comes;
            // a thread without a node on the level carries the word of a ghost.
            const int want = topsel << 29;
            int lo = ldsi1(lb_sa + 4u * (uint32_t)lfrom), hi = ldsi1(lb_sa + 4u * (uint32_t)(lfrom + 1));
            int lo_n = lfrom > lto ? ldsi1(lb_sa + 4u * (uint32_t)(lfrom - 1)) : 0;
            uint32_t lbp = lb_sa + 4u * (uint32_t)(lfrom - 2);        // lb[l - 2] of the level in hand
            int v = lo + tid;
            int4 k = make_int4(0, 0, (int)0x80000000, 0);
            V2 a0, a2; T Un = T(0);
            a0.x = T(1); a0.y = T(0); a2.x = T(0); a2.y = T(0);
            uint32_t qa = nd_sa + (uint32_t)v * RS;
            if (v < hi) { k = ldsi4(kp_sa + 16u * (uint32_t)v); a0 = lds2<T>(qa); Un = lds1<T>(qa + 2u * W); a2 = lds2<T>(qa + 4u * W); }
#pragma unroll 1
            for (int n = lfrom - lto; n >= 0; --n, lbp -= 4u) {
                const int lo_nn = n > 1 ? ldsi1(lbp) : 0;             // two levels ahead: off the chain
                if (((k.z ^ want) & (int)0xA0000000) == 0) node_step<T, MODE>(nd_sa, qa, k, a0, Un, a2);
                hi = lo; lo = lo_n; lo_n = lo_nn;
                v = lo + tid;
                qa = nd_sa + (uint32_t)v * RS;
                k.z = (int)0x80000000;
                if (n > 0 && v < hi) {                      // this thread's node on the next level: lands while the barrier is pending
                    k = ldsi4(kp_sa + 16u * (uint32_t)v); a0 = lds2<T>(qa); Un = lds1<T>(qa + 2u * W); a2 = lds2<T>(qa + 4u * W);
                }
                named_barrier(pthreads);
            }
        }
        __syncthreads();
        return;
    }
    sweep_backward_wide<T, MODE>(nd_sa, lb_sa, kp_sa, lfrom, lto, topsel, tid, nthreads);
}

// Unbranched cables (the degenerate single-branch case): the reduced system of a cable is tridiagonal, one row per
// segment, and is solved inside ONE warp by parallel cyclic reduction: lane i holds row i = {a, b, c, d} (couplings
// to rows i-1 and i+1, pivot, right-hand side); a step with stride s eliminates the couplings to i-s and i+s
// (a' = -a ra[i-s], c' = -c rc[i+s], b' = b - a rc[i-s] - c ra[i+s], d' = d - a rd[i-s] - c rd[i+s], with
// ra = a/b, rc = c/b, rd = d/b of the source rows); after ceil(log2 m) steps x = d / b.  5 steps for the 25
// segments of a 1,000-compartment cable, instead of 25 dependent levels.  The matrix is strictly diagonally
// dominant and every step keeps it so.
template <typename T>
__device__ __forceinline__ void solve_cables_pcr(T* nd, const int32_t* cb, int ncables, int tid, int nthreads)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = tid & 31, nwarps = nthreads >> 5;
    for (int c = tid >> 5; c < ncables; c += nwarps) {
        const int n0 = cb[c], m = cb[c + 1] - n0;
        T a = T(0), bb = T(1), cc = T(0), dd = T(0), pd = T(0), pb = T(0);
        if (lane < m) {
            const T* q = nd + 6 * (n0 + lane);
            bb = q[0]; dd = q[1]; a = -q[2]; pd = q[4]; pb = q[5];      // record slot 2 holds -U
        }
        // the interior of segment i+1 left its contribution to its top = row i; row i+1's coupling is row i's c
        const T pdn = __shfl_down_sync(FULL, pd, 1), pbn = __shfl_down_sync(FULL, pb, 1), an = __shfl_down_sync(FULL, a, 1);
        if (lane + 1 < m) { bb -= pdn; dd -= pbn; cc = an; }
        if (lane == 0) a = T(0);
#pragma unroll 1
        for (int s = 1; s < m; s <<= 1) {
            const T r = rcp<T>(bb);
            const T ra = a * r, rc = cc * r, rd = dd * r;
            const T ra_u = __shfl_up_sync(FULL, ra, s), rc_u = __shfl_up_sync(FULL, rc, s), rd_u = __shfl_up_sync(FULL, rd, s);
            const T ra_d = __shfl_down_sync(FULL, ra, s), rc_d = __shfl_down_sync(FULL, rc, s), rd_d = __shfl_down_sync(FULL, rd, s);
            const bool up = lane >= s, dn = lane + s < 32;
            const T au = up ? a : T(0), cd = dn ? cc : T(0);
            bb = fnma<T>(au, rc_u, fnma<T>(cd, ra_d, bb));
            dd = fnma<T>(au, rd_u, fnma<T>(cd, rd_d, dd));
            a = -au * ra_u;
            cc = -cd * rc_d;
        }
        if (lane < m) nd[6 * (n0 + lane) + 1] = dd * rcp<T>(bb);
    }
}

// ------------------------------------------------------------------------------------------------
// Resident kernel: one block per part; an item is one block, one cluster of blocks (CL), or the
// blocks of three launches (split items, `phase`).
//
// Shared memory of a block (bytes):
//   [0,16) mbarrier | [16,528) the block's record (header + first runs) | nd[6 NN] node records of the part's reduced forest
//   {D -> -f, B -> c -> x, U, -, parked d -> hand-off d, parked b -> hand-off b}, NN = nodes rounded up |
//   metadata blob (level starts, {kids, parent} per node, exports, ghosts, segment lanes) |
//   sd[L] su[L] sb[L]  the part's runs of d, u, b, one after the other, each at an index with the parity
//   of its global index.
//
// Phases:
//   P1 condense   every segment's interior a..b-1 is eliminated top-down, independently of the tree
//                 level (two lanes per segment).  Node i keeps g = u[i+1]/D, h = e/D, c = B/D where e is
//                 the fill-in coupling to the separator t above the segment.  What is left of the
//                 separator b (pivot, right-hand side, coupling U to t) and the interior's contribution
//                 to t (sum h e, sum h B) go to the segment's node record.
//   P2 backward   the level-synchronous sweep of the paper over the reduced forest,
//                 deepest level first: one thread per node, a block barrier per level; a node pulls the
//                 hand-off values of its children (consecutive records), in ascending order:
//                 D -= sum hd; B -= sum hb; r = 1/D; f = U r; c = B r; hand-off = (f U + parked d, f B + parked b).
//                 A root has U = 0, so f = 0 and x = c.
//      exchange   the root of a sub-tree held by another block hands its value to a ghost child in the
//                 top part and later reads its parent's x into a ghost parent (cluster: distributed
//                 shared memory; split items: global exchange buffers between launches).
//   P2 forward    x_v = c_v - f_v x_parent by pointer jumping over the forest.
//   P3 expand     x[i] = c - g x[i+1] - h x[t] for every interior, the same two lanes per segment.
// Eliminating in this order is a symmetric permutation of the same LDL^T factorisation (the matrix is
// SPD and strictly diagonally dominant, so any order is stable without pivoting).
// ------------------------------------------------------------------------------------------------
// MODE (f3: with a fixed time step only the right-hand side changes):
//   kModeSolve   the whole solve from d, u, b;
//   kModeFactor  everything that touches only d and u: per interior g, h and r = 1/D, per separator g = -f, -U and r,
//                written to the plan's factor arrays f0, f1, f2 (natural order);
//   kModeRhs     the solve from those factors and b: no reciprocal, one FMA on every dependent chain.
enum { kModeSolve = 0, kModeFactor = 1, kModeRhs = 2 };

// QUAD: the class has four-lane segment groups (long segments); classes without them run the leaner instantiation.
template <typename T, bool CL, int MODE, bool QUAD>
__global__ void __launch_bounds__(768, 1)
hines_resident_kernel(const BlockRecord* __restrict__ recs, const int32_t* __restrict__ meta_g, const int4* __restrict__ runs_g,
                      const T* __restrict__ d, const T* __restrict__ u, const T* __restrict__ b, T* x,
                      T* f0, T* f1, T* f2,
                      int64_t n_total, T* xch_h, T* xch_x, int ctl, unsigned long long* prof)
{
    const int phase = ctl & 3;
    extern __shared__ __align__(128) unsigned char smem[];
    namespace cg = cooperative_groups;
    typedef typename Vec2<T>::type V2;
    // phase clocks (debug hook, prof == nullptr in normal runs): thread 0 stamps %globaltimer
    unsigned long long stamp[7];
    // A stamp behind a barrier must not be taken before the barrier has completed (BAR.SYNC.DEFER_BLOCKING lets independent
    // instructions behind it issue while the warp still waits): the timer read is made to depend on a shared-memory load.
#define HINES_STAMP(k) do { if (prof && threadIdx.x == 0) { if (ldsi1(smem_u32(smem) + 16 + 28) != (int)0x80000001) stamp[k] = globaltimer_ns(); } } while (0)
    if (prof && threadIdx.x == 0) stamp[0] = globaltimer_ns();
    constexpr int E = 16 / (int)sizeof(T);
    constexpr uint32_t W = (uint32_t)sizeof(T);
    const int tid = threadIdx.x, lane = tid & 31, nthreads = blockDim.x;
    unsigned rank = 0;
    if (CL) rank = cg::this_cluster().block_rank();
    // One 512-byte record per block, in launch order: the part's header and its first runs side by side, so that a
    // single dependent global load stands between the block's start and its bulk copies.
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem);
    const PartHeader& H = *reinterpret_cast<const PartHeader*>(smem + 16);
    const int4* myruns = reinterpret_cast<const int4*>(smem + 16 + sizeof(PartHeader));
    if (tid < 32) reinterpret_cast<int4*>(smem + 16)[tid] = reinterpret_cast<const int4*>(recs + blockIdx.x)[tid];
    if (tid < 4) {
        // the record of the block that will take this one's place on the SM (ctl >> 8 blocks later in the launch), into
        // L2: its one dependent global load then costs an L2 hit instead of a DRAM round trip
        const unsigned nb = blockIdx.x + (unsigned)(ctl >> 8);
        if (nb < gridDim.x) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(recs + nb) + 128 * tid));
    }
    if (tid == 0) { mbar_init(bar, 1); if (CL) mbar_init(bar + 1, 1); }
    __syncthreads();
    if (CL) cluster_arrive_relaxed();                       // barrier 0: this block runs and its exchange mbarrier is initialised
    if (!CL && (phase == kPhaseA || phase == kPhaseB)) pdl_launch_dependents();
    const int L = H.L, NN = (H.nnode + 1 + E - 1) / E * E;    // one all-zero record behind the last node
    T* nd = reinterpret_cast<T*>(smem + 16 + sizeof(BlockRecord));
    int32_t* meta = reinterpret_cast<int32_t*>(nd + 6 * NN);
    T* sd = reinterpret_cast<T*>(meta + H.meta_len);
    T* su = sd + L;
    T* sb = su + L;
    T* sr = sb + L;                                         // factored plans only (kPartFlagFactored): the fourth array
    const int4* seg = reinterpret_cast<const int4*>(meta + H.seg_off);
    constexpr int NARR = MODE == kModeSolve ? 3 : (MODE == kModeFactor ? 2 : 4);
    const int nseg_lanes = H.nseg_lanes, nrun = H.nrun;

    if (tid == 0) {
        // what the other blocks of the cluster will send: two values per ghost child (rank 0), one x per exported root
        if (CL) mbar_expect_tx(bar + 1, rank == 0 ? (uint32_t)H.nghost * 2u * W : (uint32_t)H.nexp * W);
        mbar_expect_tx(bar, (uint32_t)NARR * (uint32_t)H.tx_elems * W + (uint32_t)H.meta_len * 4u);
        tma_load_1d(meta, meta_g + H.meta_off, (uint32_t)H.meta_len * 4u, bar);
    }
    // No barrier between the expect-tx and the copies of the other warps: a copy that completes first takes the
    // barrier's tx-count below zero for a moment, which is allowed; the phase cannot complete before thread 0's
    // arrive.expect_tx, the only arrival the barrier waits for.
    {
        // a run [g, g+len) is brought as the 16-byte words that cover it (neighbouring compartments come along
        // and are ignored); words beyond the end of the arrays are not touched: that remainder by plain loads
        // (a bulk-copy instruction costs its warp ~70 cycles per active lane: one run per warp, its three arrays by
        // lanes 0-2, so that the copies of a part with many runs are issued by all warps side by side)
        // The lane's array is chosen once (solve: d, b, u; factor: d, u; right-hand side: f0, b, f1, f2); per run the plan
        // has the index arithmetic done (word 3 of the run: elements the copy brings, a flag for elements beyond the
        // arrays' last whole 16-byte word): the loop is a handful of instructions in front of each bulk copy.
        const int nwarps = nthreads >> 5, warp = tid >> 5;
        const T* src = nullptr; T* dst = nullptr;
        if (MODE == kModeSolve) { src = lane == 0 ? d : (lane == 1 ? b : (lane == 2 ? u : nullptr)); dst = lane == 0 ? sd : (lane == 1 ? sb : su); }
        if (MODE == kModeFactor) { src = lane == 0 ? d : (lane == 2 ? u : nullptr); dst = lane == 0 ? sd : su; }
        if (MODE == kModeRhs) { src = lane == 0 ? f0 : (lane == 1 ? b : (lane == 2 ? f1 : (lane == 3 ? f2 : nullptr))); dst = lane == 0 ? sd : (lane == 1 ? sb : (lane == 2 ? su : sr)); }
        if (src != nullptr) {
            const uint32_t dst_sa = smem_u32(dst);
#pragma unroll 1
            for (int r = warp; r < nrun; r += nwarps) {
                const int4 rd = r < kInlineRuns ? myruns[r] : runs_g[H.run_off + r];
                const int ga = rd.x & ~(E - 1);                        // N < 2^31 (hines_plan_create)
                const int sdst = rd.z - (rd.x - ga);
                const uint32_t cnt = (uint32_t)rd.w & 0xffffu;
                if (cnt) tma_load_1d_sa(dst_sa + (uint32_t)sdst * W, src + ga, cnt * W, bar);
                if (rd.w & (1 << 24))                                  // the elements beyond the arrays' last whole word
                    for (int i = ga + (int)cnt; i < rd.x + rd.y; ++i) dst[sdst + (i - ga)] = src[i];
            }
        }
    }
    if (tid < 2) nd[6 * H.nnode + 4 + tid] = T(0);          // the all-zero record: hand-off slot of a child that is not there
    // ONE warp polls the mbarrier, the others wait at the block barrier: a polling warp takes issue slots from the
    // working warps of the blocks beside it, a warp at a barrier does not
    if (tid < 32) mbar_wait(bar, 0);
    __syncthreads();
    HINES_STAMP(1);
    const unsigned FULL = 0xffffffffu;

    // ---- P1: condense the interiors of all segments (no level dependency) ----
    // Two lanes per segment [a..b] (b = separator, t = separator above), split at a middle node q: lane A
    // eliminates a..q-1 top-down with fill-in coupling to t and arrives at q; lane B = A ^ 16 eliminates
    // q+1..b-1 top-down with fill-in coupling to q and arrives at b.  A then takes B's contribution to q,
    // eliminates q (couplings to t and to b) and writes the node record of b.  Both lanes run the same code.
    if (MODE == kModeRhs) {
        // The right-hand side alone (f3): the factors g, h, r of every interior sit in sd, su, sr; the chain of a lane is
        // B' = b[i+1] - g B (one FMA); c = B r replaces b; the contribution sum h B to the top is accumulated.
        for (int base = (tid & ~31); base < nseg_lanes; base += nthreads) {
            const int4 sg = seg[base + lane];
            const int kind = (sg.y >> 24) & 3, hasq = (sg.y >> 26) & 1;
            const int mt = sg.y & 0xfff, mb = (sg.y >> 12) & 0xfff;
            const bool isB = kind == 2, quad = QUAD && __any_sync(FULL, kind == 3);
            const int jq = kind == 3 ? (sg.y >> 12) & 3 : 0;
            const int m = isB ? mb : (kind != 0 ? mt : 0);
            const int dl = (sg.y >> 27) & 15;
            const int mmax = __reduce_max_sync(FULL, m + dl);
            int i = sg.x;
            T B = T(0), dbt = T(0);
            if (kind == 1 || kind == 3 || (isB && hasq)) B = sb[i];
            T g1 = T(0), h1 = T(0), r1 = T(0), b1 = T(0);
            if (m > 0) { g1 = sd[i]; h1 = su[i]; r1 = sr[i]; b1 = sb[i + 1]; }
            {
                // the walk on shared addresses, two register sets, pointers moved once per double step (as in the solve path)
                const uint32_t LW = (uint32_t)L * W;
                uint32_t pg = smem_u32(sd + i) - (uint32_t)dl * W, ph = pg + LW, pc = pg + 2u * LW, pr = pg + 3u * LW;
                T g2 = g1, h2 = h1, r2 = r1, b2 = b1;       // a lane's first step may fall on either half of the loop body
                int sl = -dl;
#define HINES_P1R_STEP(G1, H1, R1, B1, G2, H2, R2, B2, OFF)                                              \
                if ((unsigned)sl < (unsigned)m) {                                                        \
                    if (sl + 1 < m) { G2 = lds1<T>(pg + (OFF + 1u) * W); H2 = lds1<T>(ph + (OFF + 1u) * W); R2 = lds1<T>(pr + (OFF + 1u) * W); B2 = lds1<T>(pc + (OFF + 2u) * W); } \
                    sts1<T>(pc + OFF * W, B * R1);                                                       \
                    dbt = fmad<T>(H1, B, dbt);                                                           \
                    B = fnma<T>(G1, B, B1);                                                              \
                }                                                                                        \
                ++sl;
#pragma unroll 1
                for (int s = 0; s < mmax; s += 2) {
                    HINES_P1R_STEP(g1, h1, r1, b1, g2, h2, r2, b2, 0u)
                    HINES_P1R_STEP(g2, h2, r2, b2, g1, h1, r1, b1, 1u)
                    pg += 2u * W; ph += 2u * W; pc += 2u * W; pr += 2u * W;
                }
#undef HINES_P1R_STEP
                i += m;
            }
            const bool lead = quad ? (kind == 3 && jq == 0) : (kind == 1);
            const int stride = quad ? 8 : 16, nq = quad ? 3 : 1;
            T Bc = B;
            int qi = i;
            for (int sq = 1; sq <= nq; ++sq) {              // the middle nodes, in turn (see the solve path)
                const int src = (lane + stride * sq) & 31;
                const T pB = __shfl_sync(FULL, B, src), pdb = __shfl_sync(FULL, dbt, src);
                const int pm = __shfl_sync(FULL, m, src);
                if (lead && hasq) {
                    const T Bq = Bc - pdb;
                    sb[qi] = Bq * sr[qi];
                    dbt = fmad<T>(su[qi], Bq, dbt);
                    Bc = fnma<T>(sd[qi], Bq, pB);
                    qi += pm + 1;
                }
            }
            if (lead) {                                     // qi is the separator: its factors g = -f, -U, r sit at its place
                T* q = nd + 6 * sg.z;
                q[0] = sd[qi]; q[1] = Bc; q[2] = su[qi]; q[3] = sr[qi]; q[4] = T(0); q[5] = hasq ? dbt : T(0);
            }
        }
    } else
    {
    for (int base = (tid & ~31); base < nseg_lanes; base += nthreads) {
        const int4 sg = seg[base + lane];
        const int kind = (sg.y >> 24) & 3, hasq = (sg.y >> 26) & 1;
        // kind 1 / 2: the A / B lane of a two-lane segment (partner = lane ^ 16); kind 3: lane j of a four-lane segment
        // (its lanes are 8 apart).  Every lane sweeps its piece top-down with fill-in to the node right above the piece.
        const int mt = sg.y & 0xfff, mb = (sg.y >> 12) & 0xfff;
        const bool isB = kind == 2, quad = QUAD && __any_sync(FULL, kind == 3);
        const int jq = kind == 3 ? (sg.y >> 12) & 3 : 0;
        const int m = isB ? mb : (kind != 0 ? mt : 0);
        const int dl = (sg.y >> 27) & 15;                   // the lane starts dl steps late (bank residues, plan.cpp)
        const int mmax = __reduce_max_sync(FULL, m + dl);
        int i = sg.x;
        T D = T(1), B = T(0), ee = T(0), ddt = T(0), dbt = T(0), un = T(0), dn = T(0), bn = T(0);
        if (kind == 1 || kind == 3 || (isB && hasq)) { D = sd[i]; if (MODE == kModeSolve) B = sb[i]; if (isB || jq > 0 || sg.w >= 0) ee = su[i]; }
        if (m > 0) { un = su[i + 1]; dn = sd[i + 1]; if (MODE == kModeSolve) bn = sb[i + 1]; }
        {
            // The sweep proper, on 32-bit shared addresses: node i at pa (d), pa + LW (u), pa + 2 LW (b); the
            // loop is unrolled by two with the two register sets swapping roles (no register rotation).
            const uint32_t LW = (uint32_t)L * W;
            // element i + sl of sd (sl = the warp's step - dl); the pointers move once per double step for every lane,
            // the half steps use constant offsets; nothing is dereferenced while sl is outside [0, m)
            uint32_t pa = smem_u32(sd + i) - (uint32_t)dl * W, pu = pa + LW, pb = pa + 2u * LW;
            T un2 = un, dn2 = dn, bn2 = bn;                 // a lane's first step may fall on either half of the loop body
#define HINES_P1_STEP(UN, DN, BN, UN2, DN2, BN2, OFF)                                                \
            if ((unsigned)sl < (unsigned)m) {                                                        \
                if (sl + 1 < m) { UN2 = lds1<T>(pu + (OFF + 2u) * W); DN2 = lds1<T>(pa + (OFF + 2u) * W); if (MODE == kModeSolve) BN2 = lds1<T>(pb + (OFF + 2u) * W); } \
                const T r = rcp<T>(D);                                                               \
                const T g = UN * r, h = ee * r, c = B * r;                                           \
                sts1<T>(pa + OFF * W, g); sts1<T>(pu + OFF * W, h); sts1<T>(pb + OFF * W, MODE == kModeFactor ? r : c); \
                ddt = fmad<T>(h, ee, ddt); dbt = fmad<T>(h, B, dbt);                                 \
                D = fnma<T>(g, UN, DN); B = fnma<T>(g, B, BN); ee = -h * UN;                         \
            }                                                                                        \
            ++sl;
            int sl = -dl;
#pragma unroll 1
            for (int s = 0; s < mmax; s += 2) {
                HINES_P1_STEP(un, dn, bn, un2, dn2, bn2, 0u)
                HINES_P1_STEP(un2, dn2, bn2, un, dn, bn, 1u)
                pa += 2u * W; pu += 2u * W; pb += 2u * W;
            }
#undef HINES_P1_STEP
            i += m;
        }
        // The middle nodes, in turn, by the segment's first lane: the lane of the piece below hands over what is left of
        // the node it arrived at (pD, pB), that node's coupling to the middle node (pe) and the piece's contribution
        // parked for the middle node (pdd, pdb).  One middle node for a two-lane segment, three for a four-lane one.
        if (!quad) {
            // B -> A: what is left of b (pD, pB), its coupling to q (pe), B's contribution parked for q (pdd, pdb)
            const T pD = __shfl_xor_sync(FULL, D, 16), pB = __shfl_xor_sync(FULL, B, 16), pe = __shfl_xor_sync(FULL, ee, 16);
            const T pdd = __shfl_xor_sync(FULL, ddt, 16), pdb = __shfl_xor_sync(FULL, dbt, 16);
            if (kind == 1) {
                T* q = nd + 6 * sg.z;
                if (hasq) {                                 // i is q now
                    const T Dq = D - pdd, Bq = B - pdb;
                    const T r = rcp<T>(Dq);
                    const T gq = pe * r, hq = ee * r;
                    sd[i] = gq; su[i] = hq; sb[i] = MODE == kModeFactor ? r : Bq * r;
                    ddt = fmad<T>(hq, ee, ddt); dbt = fmad<T>(hq, Bq, dbt);
                    q[0] = fnma<T>(gq, pe, pD); q[1] = fnma<T>(gq, Bq, pB); q[2] = hq * pe; q[4] = ddt; q[5] = dbt;     // slot 2 = -U
                    if (MODE == kModeFactor) q[3] = (T)(i + 1 + mb);                                                    // slot 3 = staged index of b
                } else {                                    // a segment of one compartment: the separator as it is
                    q[0] = D; q[1] = B; q[2] = -ee; q[4] = T(0); q[5] = T(0);
                    if (MODE == kModeFactor) q[3] = (T)i;
                }
            }
        } else {
            const bool lead = kind == 3 && jq == 0;
            T Dc = D, Bc = B, et = ee;
            int qi = i;
#pragma unroll
            for (int sq = 1; sq <= 3; ++sq) {
                const int src = (lane + 8 * sq) & 31;
                const T pD = __shfl_sync(FULL, D, src), pB = __shfl_sync(FULL, B, src), pe = __shfl_sync(FULL, ee, src);
                const T pdd = __shfl_sync(FULL, ddt, src), pdb = __shfl_sync(FULL, dbt, src);
                const int pm = __shfl_sync(FULL, m, src);
                if (lead) {                                 // qi is the middle node
                    const T Dq = Dc - pdd, Bq = Bc - pdb;
                    const T r = rcp<T>(Dq);
                    const T gq = pe * r, hq = et * r;
                    sd[qi] = gq; su[qi] = hq; sb[qi] = MODE == kModeFactor ? r : Bq * r;
                    ddt = fmad<T>(hq, et, ddt); dbt = fmad<T>(hq, Bq, dbt);
                    Dc = fnma<T>(gq, pe, pD); Bc = fnma<T>(gq, Bq, pB); et = -hq * pe;
                    qi += pm + 1;
                }
            }
            if (lead) {                                     // qi is the separator now; slot 2 = -U, slot 3 = its staged index
                T* q = nd + 6 * sg.z;
                q[0] = Dc; q[1] = Bc; q[2] = -et; q[4] = ddt; q[5] = dbt;
                if (MODE == kModeFactor) q[3] = (T)qi;
            }
        }
    }
    }
    __syncthreads();
    HINES_STAMP(2);

    const int4* ex = reinterpret_cast<const int4*>(meta + H.exp_off);
    const int4* gh = reinterpret_cast<const int4*>(meta + H.gh_off);
    const uint32_t nd_sa = smem_u32(nd), lb_sa = smem_u32(meta), kp_sa = smem_u32(meta + H.kp_off);
    const int nexp = H.nexp, nghost = H.nghost, nnode = H.nnode;
    int rounds = H.rounds;
    const bool cables = (H.flags & kPartFlagChains) != 0;
    if (cables) {
        // ---- unbranched cables: the reduced chains by parallel cyclic reduction, one warp per cable ----
        solve_cables_pcr<T>(nd, meta, H.nlev, tid, nthreads);
        __syncthreads();
    }
    // ---- P2 backward: what does not wait for another part, deepest level first ----
    if (!cables) sweep_backward<T, MODE>(nd_sa, lb_sa, kp_sa, H.nlev - 1, H.lowlev, 0, H.maxwidth, tid, nthreads);
    // ---- hand-off values of the sub-trees held by other blocks, into the ghost children; then
    //      the top nodes (the ancestors of the ghost children) ----
    if (CL) {
        if (rank == 0) { cluster_wait(); if (tid < 32) mbar_wait_cluster(bar + 1, 0); __syncthreads(); }      // every ghost child has its hand-off (one warp polls)
    } else if (phase == kPhaseB) {
        pdl_wait();                                         // phase A has completed: the hand-off values are there
#pragma unroll 1
        for (int e = tid; e < nghost; e += nthreads) {
            const int4 g = gh[e];
            *reinterpret_cast<V2*>(nd + 6 * g.x + 4) = reinterpret_cast<const V2*>(xch_h)[H.xch_base + g.y];
        }
        __syncthreads();
    }
    sweep_backward<T, MODE>(nd_sa, lb_sa, kp_sa, H.ntoplev - 1, 0, 1, H.maxwidth, tid, nthreads);
    HINES_STAMP(3);
    // ---- exchange: an exported root {node, ghost parent, ghost child in part 0 / exchange slot, -} hands its value
    //      up.  Cluster: a store into rank 0's shared memory that counts its bytes on rank 0's mbarrier (data and
    //      signal in one message, no cluster-wide barrier, no fence).  The ghost parent becomes the identity
    //      (g, c) = (1, 0) for the rounds below. ----
    const bool sub = MODE != kModeFactor && (CL ? rank != 0 : phase == kPhaseC);       // a part that waits for its parents' x
    if (CL) {
        if (rank != 0) {
            const uint32_t bar0 = mapa_u32(smem_u32(bar + 1), 0), nd0a = mapa_u32(nd_sa, 0);
            cluster_wait();                                 // barrier 0: rank 0 is running, its mbarrier initialised
#pragma unroll 1
            for (int e = tid; e < nexp; e += nthreads) {
                const int4 q = ex[e];
                const V2 hv = *reinterpret_cast<const V2*>(nd + 6 * q.x + 4);
                st_async_2(nd0a + (6u * (uint32_t)q.z + 4u) * W, hv.x, hv.y, bar0);
                nd[6 * q.y] = T(1); nd[6 * q.y + 1] = T(0);
            }
        }
    } else if (phase == kPhaseA) {
#pragma unroll 1
        for (int e = tid; e < nexp; e += nthreads) {
            const int4 q = ex[e];
            reinterpret_cast<V2*>(xch_h)[H.xch_base + q.z] = *reinterpret_cast<const V2*>(nd + 6 * q.x + 4);
        }
        if (MODE != kModeFactor && prof && tid == 0) {
            unsigned long long* o = prof + 8 * (size_t)blockIdx.x;
            for (int k = 0; k < 4; ++k) o[k] = stamp[k];
            o[4] = o[5] = o[6] = globaltimer_ns();
            o[7] = ((unsigned long long)smid() << 32) | (unsigned)H.n;
        }
        if (MODE != kModeFactor) return;
    } else if (phase == kPhaseC) {
#pragma unroll 1
        for (int e = tid; e < nexp; e += nthreads) { const int4 q = ex[e]; nd[6 * q.y] = T(1); nd[6 * q.y + 1] = T(0); }
    }
    // ---- P2 forward: first the top nodes, level by level (the other parts of the cell wait
    //      for their x), then everything by pointer jumping over the reduced forest.
    // x_v = c_v + g_v x_p(v), g = -f, g = 0 at a root and at a finished node.
    // One round replaces (g_v, c_v, p(v)) by (g_v g_p, c_v + g_v c_p, p(p(v))): after `rounds` rounds (2^rounds > the
    // longest path) every g is 0 and c is x.  All nodes work in every round, with one barrier per round instead of
    // one per level.  Buffers: record slots {0,1} and {2,3}; parent ids in {4,5}.
    // A part that waits for its parents' x does its rounds WHILE it waits: its ghost parents are fixed points with the
    // identity map, so after `rounds` rounds every node holds x_v = c_v + g_v x(its ghost parent); when x has arrived the
    // ghost parents become (0, x) and one more round finishes.
    if (MODE == kModeFactor) rounds = 0;
    const int4* kp = reinterpret_cast<const int4*>(meta + H.kp_off);
    if (sub) __syncthreads();                               // the ghost parents' identity records
    const int nrounds = rounds;
    if (sub) ++rounds;                                      // the round after x has arrived
    constexpr uint32_t RSB = 6u * W;                        // bytes per node record
    const bool one_node = nnode <= nthreads;
    const uint32_t my_qa = nd_sa + (uint32_t)tid * RSB;
    V2 my_gc; my_gc.x = T(0); my_gc.y = T(0);
    int my_p = 0;
    if (one_node && rounds > 0 && tid < nnode) { my_gc = lds2<T>(my_qa); my_p = ldsi1(kp_sa + 16u * (uint32_t)tid + 12u); }
#pragma unroll 1
    for (int r = 0; r < rounds; ++r) {
        if (sub && r == nrounds) {
            if (CL) { if (tid < 32) mbar_wait_cluster(bar + 1, 0); __syncthreads(); }     // rank 0 has sent every x this part waits for (behind the export's entry); one warp polls
            else pdl_wait();                                // phase B has completed: the parents' x is in the exchange buffer
            const int cur = 2 * (r & 1);
#pragma unroll 1
            for (int e = tid; e < nexp; e += nthreads) {
                const int4 q = ex[e];
                nd[6 * q.y + cur] = T(0);
                nd[6 * q.y + cur + 1] = CL ? *reinterpret_cast<const T*>(&ex[e].z) : xch_x[H.xch_base + q.z];
            }
            __syncthreads();
        }
        const int sbuf = 2 * (r & 1), dbuf = 2 - sbuf;
        if (one_node) {
            // one node per thread: its (g, c) and parent stay in registers over the rounds; a round is the parent's
            // (g, c) and parent from shared memory, two fp operations and the thread's own two stores
            if (tid < nnode) {
                const uint32_t pa = nd_sa + (uint32_t)my_p * RSB;
                const V2 ap = lds2<T>(pa + (uint32_t)sbuf * W);
                const int pp = r == 0 ? ldsi1(kp_sa + 16u * (uint32_t)my_p + 12u) : ldsi1(pa + 4u * W + 4u * (uint32_t)((r - 1) & 1));
                V2 o; o.x = my_gc.x * ap.x; o.y = fmad<T>(my_gc.x, ap.y, my_gc.y);
                sts2<T>(my_qa + (uint32_t)dbuf * W, o);
                stsi1(my_qa + 4u * W + 4u * (uint32_t)(r & 1), pp);
                my_gc = o; my_p = pp;
            }
            __syncthreads();
            continue;
        }
#pragma unroll 1
        for (int v = tid; v < nnode; v += nthreads) {
            int* ip = reinterpret_cast<int*>(nd + 6 * v + 4);
            const int p = r == 0 ? kp[v].w : ip[(r - 1) & 1];
            const V2 a = *reinterpret_cast<const V2*>(nd + 6 * v + sbuf);
            const V2 ap = *reinterpret_cast<const V2*>(nd + 6 * p + sbuf);
            const int pp = r == 0 ? kp[p].w : reinterpret_cast<const int*>(nd + 6 * p + 4)[(r - 1) & 1];
            V2 o; o.x = a.x * ap.x; o.y = fmad<T>(a.x, ap.y, a.y);
            *reinterpret_cast<V2*>(nd + 6 * v + dbuf) = o;
            ip[r & 1] = pp;
        }
        __syncthreads();
    }
    const int xs_now = 2 * (rounds & 1) + 1;              // record slot that holds x now
    if (CL) {
        if (rank == 0 && MODE != kModeFactor) {             // x of the top nodes goes to the roots that wait for it
            const uint32_t bar1 = smem_u32(bar + 1), base = smem_u32(smem);
#pragma unroll 1
            for (int e = tid; e < nghost; e += nthreads) {
                const int4 g = gh[e];                       // {ghost child, -, parent, rank << 20 | landing word in that block}
                const uint32_t r = (uint32_t)g.w >> 20, word = (uint32_t)g.w & 0xfffffu;
                st_async_1(mapa_u32(base + 4u * word, r), nd[6 * g.z + xs_now], mapa_u32(bar1, r));
            }
        }
    } else if (phase == kPhaseB && MODE != kModeFactor) {
#pragma unroll 1
        for (int e = tid; e < nghost; e += nthreads) {
            const int4 g = gh[e];
            xch_x[H.xch_base + g.y] = nd[6 * g.z + xs_now];
        }
    }
    const int xs = 2 * (rounds & 1) + 1;                  // record slot that holds x after the forward sweep
    HINES_STAMP(4);

    // ---- P3: expand the interiors: the segment's first lane computes x of the middle nodes from x[b] and x[t]; then
    //      every lane walks its piece upward, x[i] = c - g x[i+1] - h x[top of the piece]: one FMA on the dependent
    //      chain per step ----
    if (MODE == kModeFactor) {
        // the separators' factors go where their compartments are: g = -f, -U, r = 1 / pivot
        __syncthreads();
#pragma unroll 1
        for (int v = tid; v < H.nlevnode; v += nthreads) {
            const T* q = nd + 6 * v;
            if (reinterpret_cast<const int4*>(meta + H.kp_off)[v].z < 0) continue;       // a ghost child has no compartment here
            const int bpos = (int)q[3];                                                  // written by the segment's first lane in P1
            sd[bpos] = q[0]; su[bpos] = q[2]; sb[bpos] = q[1];
        }
    } else
    for (int base = (tid & ~31); base < nseg_lanes; base += nthreads) {
        const int4 sg = seg[base + lane];
        const int kind = (sg.y >> 24) & 3, hasq = (sg.y >> 26) & 1;
        const int mt = sg.y & 0xfff, mb = (sg.y >> 12) & 0xfff;
        const bool isB = kind == 2, quad = QUAD && __any_sync(FULL, kind == 3);
        const int jq = kind == 3 ? (sg.y >> 12) & 3 : (isB ? 1 : 0);          // which piece of its segment the lane holds
        const int m = isB ? mb : (kind != 0 ? mt : 0);
        const int dl = (sg.y >> 27) & 15;
        const int mmax = __reduce_max_sync(FULL, m + dl);
        const int p0 = sg.x;
        T xb = T(0), xt = T(0), xn = T(0);
        if (kind != 0) xb = nd[6 * sg.z + xs];
        if (!quad) {
            if (kind == 1) {
                if (sg.w >= 0) xt = nd[6 * sg.w + xs];
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
        } else {
            // the middle nodes, from the separator upward, by the segment's first lane: x[q] = c - g x[below] - h x[t]
            const bool lead = kind == 3 && jq == 0;
            const int m1 = __shfl_sync(FULL, m, (lane + 8) & 31), m2 = __shfl_sync(FULL, m, (lane + 16) & 31),
                      m3 = __shfl_sync(FULL, m, (lane + 24) & 31);
            T x1 = T(0), x2 = T(0), x3 = T(0);
            if (lead) {
                if (sg.w >= 0) xt = nd[6 * sg.w + xs];
                const int q1 = p0 + m, q2 = q1 + m1 + 1, q3 = q2 + m2 + 1;
                x3 = fnma<T>(sd[q3], xb, fnma<T>(su[q3], xt, sb[q3]));
                x2 = fnma<T>(sd[q2], x3, fnma<T>(su[q2], xt, sb[q2]));
                x1 = fnma<T>(sd[q1], x2, fnma<T>(su[q1], xt, sb[q1]));
                sb[q3] = x3; sb[q2] = x2; sb[q1] = x1; sb[q3 + m3 + 1] = xb;
            }
            // every lane: x of the node above its piece (the top) and of the node below it (where its walk starts)
            const int ll = (lane - 8 * jq) & 31;                               // the segment's first lane
            const T s1 = __shfl_sync(FULL, x1, ll), s2 = __shfl_sync(FULL, x2, ll), s3 = __shfl_sync(FULL, x3, ll);
            const T st = __shfl_sync(FULL, xt, ll);
            xt = jq == 0 ? st : (jq == 1 ? s1 : (jq == 2 ? s2 : s3));
            xn = jq == 0 ? s1 : (jq == 1 ? s2 : (jq == 2 ? s3 : xb));
        }
        // The walk, on 32-bit shared addresses like P1: the lane's step j (its piece's element p0 + j) runs from
        // m - 1 down to 0 while the warp's counter runs from mmax - 1 down to 0 (j = counter - dl: the same residue
        // shift as in P1).  Unrolled by two with two register sets that swap roles (no register rotation); the
        // pointers move once per double step, the half steps use constant offsets.  A step costs what the warp
        // issues for it (a lone warp: about 5 cycles per instruction), so the loop is kept to the loads of the next
        // element, two FMAs (one on the dependent chain) and the store.
        {
            const uint32_t LW = (uint32_t)L * W;
            int j = mmax - 1 - dl;
            // element p0 + j of sd; never dereferenced while j is outside [0, m)
            uint32_t pg = smem_u32(sd + p0) + (uint32_t)(j * (int)W), ph = pg + LW, pc = pg + 2u * LW;
            T g1 = T(0), h1 = T(0), c1 = T(0);
            if (m > 0) { const int i = p0 + m - 1; g1 = sd[i]; h1 = su[i]; c1 = sb[i]; }
            T g2 = g1, h2 = h1, c2 = c1;                    // a lane's first step may fall on either half of the loop body
#define HINES_P3_STEP(G1, H1, C1, G2, H2, C2, OFF)                                                                  \
            if ((unsigned)j < (unsigned)m) {                                                                        \
                if (j > 0) { G2 = lds1<T>(pg - (OFF + 1u) * W); H2 = lds1<T>(ph - (OFF + 1u) * W); C2 = lds1<T>(pc - (OFF + 1u) * W); } \
                xn = fnma<T>(G1, xn, fnma<T>(H1, xt, C1));                                                           \
                sts1<T>(pc - OFF * W, xn);                                                                           \
            }                                                                                                       \
            --j;
#pragma unroll 1
            for (int s2 = 0; s2 < mmax; s2 += 2) {
                HINES_P3_STEP(g1, h1, c1, g2, h2, c2, 0u)
                HINES_P3_STEP(g2, h2, c2, g1, h1, c1, 1u)
                pg -= 2u * W; ph -= 2u * W; pc -= 2u * W;
            }
#undef HINES_P3_STEP
        }
    }

    // ---- store x (natural order), run by run: bulk store of the 16-byte words inside the run, edges by hand ----
    fence_proxy_async();
    __syncthreads();
    HINES_STAMP(5);
#pragma unroll 1
    for (int r = tid >> 5; r < nrun; r += nthreads >> 5) {
        const int4 rd = r < kInlineRuns ? myruns[r] : runs_g[H.run_off + r];
        const int g = rd.x, len = rd.y, so = rd.z;                                       // N < 2^31 (hines_plan_create)
        const int head = (rd.w >> 16) & 15, tail = len - ((rd.w >> 20) & 15);            // run-local [0, head) and [tail, len): by hand
#pragma unroll
        for (int a = 0; a < (MODE == kModeFactor ? 3 : 1); ++a) {                        // x, or the three factor arrays
            T* dstg = MODE == kModeFactor ? (a == 0 ? f0 : (a == 1 ? f1 : f2)) : x;
            const T* srcs = MODE == kModeFactor ? (a == 0 ? sd : (a == 1 ? su : sb)) : sb;
            if (lane == 0 && tail > head) tma_store_1d(dstg + g + head, srcs + so + head, (uint32_t)(tail - head) * W);
            if (lane >= 1 && lane - 1 < head) dstg[g + lane - 1] = srcs[so + lane - 1];
            if (lane >= 8 && tail + lane - 8 < len) dstg[g + tail + lane - 8] = srcs[so + tail + lane - 8];
        }
    }
    tma_store_commit_wait();
    if (prof && tid == 0) {
        stamp[6] = globaltimer_ns();
        unsigned long long* o = prof + 8 * (size_t)blockIdx.x;
        for (int k = 0; k < 7; ++k) o[k] = stamp[k];
        o[7] = ((unsigned long long)smid() << 32) | (unsigned)H.n;
    }
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
    cudaFree(D->recs); cudaFree(D->meta); cudaFree(D->runs); cudaFree(D->xch_h); cudaFree(D->xch_x); for (void* f : D->fac) cudaFree(f);
    cudaFree(D->stream_desc); cudaFree(D->stream_child); cudaFree(D->ws_f); cudaFree(D->ws_c); cudaFree(D->prof);
    for (void* p : D->host_stage) cudaFree(p);
    for (cudaEvent_t e : D->ev) if (e) cudaEventDestroy(e);
    for (cudaStream_t t : D->side) if (t) cudaStreamDestroy(t);
    for (cudaEvent_t e : D->join) if (e) cudaEventDestroy(e);
    if (D->fork) cudaEventDestroy(D->fork);
    if (D->sstream) cudaStreamDestroy(D->sstream);
    if (D->sjoin) cudaEventDestroy(D->sjoin);
    if (D->pstream) cudaStreamDestroy(D->pstream);
    if (D->pjoin) cudaEventDestroy(D->pjoin);
    delete D;
}

// Per device and kernel instantiation, once per process: the opt-in maximum of dynamic shared memory and the
// non-portable cluster size.  (Set to the device maximum, never to a plan's own need: several plans may be live.)
template <typename T>
static hines_status_t prepare_kernels(int max_optin)
{
#define HINES_PREP(MODE, Q)                                                                                                          \
    CUDA_TRY(cudaFuncSetAttribute(hines_resident_kernel<T, false, MODE, Q>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_optin)); \
    CUDA_TRY(cudaFuncSetAttribute(hines_resident_kernel<T, true, MODE, Q>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_optin));  \
    CUDA_TRY(cudaFuncSetAttribute(hines_resident_kernel<T, true, MODE, Q>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    HINES_PREP(kModeSolve, false) HINES_PREP(kModeFactor, false) HINES_PREP(kModeRhs, false)
    HINES_PREP(kModeSolve, true) HINES_PREP(kModeFactor, true) HINES_PREP(kModeRhs, true)
#undef HINES_PREP
    return HINES_OK;
}

template <typename T>
static hines_status_t check_clusters(const hines_plan* P)
{
    for (size_t q = 0; q < P->class_smem_bytes.size(); ++q) {
        const int cl = P->class_cluster[q];
        if (cl <= 1 || !P->class_count[q]) continue;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)cl); cfg.blockDim = dim3((unsigned)P->class_threads[q]);
        cfg.dynamicSmemBytes = (size_t)P->class_smem_bytes[q];
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        int nclusters = 0;
        CUDA_TRY(cudaOccupancyMaxActiveClusters(&nclusters, hines_resident_kernel<T, true, kModeSolve, true>, &cfg));
        if (nclusters < 1) {
            set_error("this device cannot co-schedule a cluster of " + std::to_string(cl) + " blocks with " +
                      std::to_string(P->class_smem_bytes[q]) + " bytes of shared memory each: create the plan with a smaller cluster_max");
            return HINES_ERR_UNSUPPORTED;
        }
    }
    return HINES_OK;
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
        CUDA_TRY(cudaDeviceGetAttribute(&D->num_sms, cudaDevAttrMultiProcessorCount, D->device));
        int max_optin = 0;
        CUDA_TRY(cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, D->device));
        for (int32_t s : P->class_smem_bytes)
            if (s > max_optin) {
                set_error("device offers " + std::to_string(max_optin) + " bytes of shared memory per block, plan needs " + std::to_string(s));
                return HINES_ERR_UNSUPPORTED;
            }
        if ((st = P->dtype == HINES_F64 ? prepare_kernels<double>(max_optin) : prepare_kernels<float>(max_optin))) return st;
        if ((st = P->dtype == HINES_F64 ? check_clusters<double>(P) : check_clusters<float>(P))) return st;
        {
            std::vector<BlockRecord> recs(P->class_parts.size());
            for (size_t k = 0; k < recs.size(); ++k) {
                const PartHeader& h = P->part_headers[P->class_parts[k]];
                recs[k].h = h;
                std::memset(recs[k].runs, 0, sizeof(recs[k].runs));
                const int nr = std::min<int>(h.nrun, kInlineRuns);
                if (nr) std::memcpy(recs[k].runs, &P->part_runs[(size_t)h.run_off * 4], (size_t)nr * 16);
            }
            if ((st = upload_vec(recs, (void**)&D->recs, D->bytes))) return st;
        }
        if ((st = upload_vec(P->part_meta, (void**)&D->meta, D->bytes))) return st;
        if ((st = upload_vec(P->part_runs, (void**)&D->runs, D->bytes))) return st;
        if ((st = upload_vec(P->stream_desc, (void**)&D->stream_desc, D->bytes))) return st;
        if ((st = upload_vec(P->stream_child, (void**)&D->stream_child, D->bytes))) return st;
        if (P->n_xch) {
            CUDA_TRY(cudaMalloc(&D->xch_h, 2 * (size_t)P->n_xch * P->width));
            CUDA_TRY(cudaMalloc(&D->xch_x, (size_t)P->n_xch * P->width));
            D->bytes += 3 * P->n_xch * P->width;
        }
        if (P->n_stream_unknowns) {
            const size_t wb = (size_t)P->n_stream_unknowns * P->width;
            CUDA_TRY(cudaMalloc(&D->ws_f, wb));
            CUDA_TRY(cudaMalloc(&D->ws_c, wb));
            D->bytes += 2 * (int64_t)wb;
        }
        const bool has_stream_path = P->stream_level_begin.size() > 1;
        int n_ordinary = 0, n_split = 0;
        for (size_t q = 0; q < P->class_phase.size(); ++q) if (P->class_count[q]) (P->class_phase[q] == kPhaseAll ? n_ordinary : n_split)++;
        const int n_lines = n_ordinary + (n_split ? 1 : 0) + (has_stream_path ? 1 : 0);     // independent lines of work
        if (n_lines > 1 && !(P->opt.policy_flags & HINES_POLICY_SERIAL_CLASSES)) {
            CUDA_TRY(cudaEventCreateWithFlags(&D->fork, cudaEventDisableTiming));
            if (has_stream_path) {
                CUDA_TRY(cudaStreamCreateWithFlags(&D->sstream, cudaStreamNonBlocking));
                CUDA_TRY(cudaEventCreateWithFlags(&D->sjoin, cudaEventDisableTiming));
            }
            if (n_split) {
                CUDA_TRY(cudaStreamCreateWithFlags(&D->pstream, cudaStreamNonBlocking));
                CUDA_TRY(cudaEventCreateWithFlags(&D->pjoin, cudaEventDisableTiming));
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
static hines_status_t launch_all(hines_plan* P, const T* d, const T* u, const T* b, T* x, cudaStream_t stream, int mode = kModeSolve)
{
    DeviceTables* D = P->dev;
    T* f0 = static_cast<T*>(D->fac[0]); T* f1 = static_cast<T*>(D->fac[1]); T* f2 = static_cast<T*>(D->fac[2]);
    auto launch_streaming = [&](cudaStream_t ss) -> hines_status_t {
        const int nlev = (int)P->stream_level_begin.size() - 1;
        const int st = P->opt.stream_threads;
        T* wf = static_cast<T*>(D->ws_f); T* wc = static_cast<T*>(D->ws_c);
        if (D->timing) CUDA_TRY(cudaEventRecord(D->ev[2], ss));
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
        if (D->timing) CUDA_TRY(cudaEventRecord(D->ev[3], ss));
        CUDA_TRY(cudaGetLastError());
        return HINES_OK;
    };
    auto launch_class = [&](size_t q, cudaStream_t ls) -> hines_status_t {
        const int64_t cnt = P->class_count[q], first = P->class_first[q];
        const int cl = P->class_cluster[q];
        unsigned long long* prof = D->prof_on ? D->prof + 8 * first : nullptr;
        const BlockRecord* recs = D->recs + first;
        T* xh = static_cast<T*>(D->xch_h); T* xx = static_cast<T*>(D->xch_x);
        const int phase = (int)P->class_phase[q];
        if (mode == kModeFactor && phase == kPhaseC) return HINES_OK;       // the factors of a sub-tree part are complete after phase A
        typedef void (*kern_t)(const BlockRecord*, const int32_t*, const int4*, const T*, const T*, const T*, T*, T*, T*, T*,
                               int64_t, T*, T*, int, unsigned long long*);
        const bool quads = P->class_quads[q] != 0;
        kern_t kern;
#define HINES_PICK(CLV)                                                                                                        \
        kern = mode == kModeSolve ? (quads ? hines_resident_kernel<T, CLV, kModeSolve, true> : hines_resident_kernel<T, CLV, kModeSolve, false>)     \
             : mode == kModeFactor ? (quads ? hines_resident_kernel<T, CLV, kModeFactor, true> : hines_resident_kernel<T, CLV, kModeFactor, false>) \
                                   : (quads ? hines_resident_kernel<T, CLV, kModeRhs, true> : hines_resident_kernel<T, CLV, kModeRhs, false>);
        if (cl == 1) { HINES_PICK(false) } else { HINES_PICK(true) }
#undef HINES_PICK
        const int32_t* mg_ = D->meta; const int4* rg_ = D->runs; const int64_t n_ = P->n;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)cnt);
        cfg.blockDim = dim3((unsigned)P->class_threads[q]);
        cfg.dynamicSmemBytes = (size_t)P->class_smem_bytes[q];
        cfg.stream = ls;
        cudaLaunchAttribute attr[1];
        cfg.attrs = attr; cfg.numAttrs = 0;
        if (cl > 1) {
            attr[0].id = cudaLaunchAttributeClusterDimension;
            attr[0].val.clusterDim.x = (unsigned)cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
            cfg.numAttrs = 1;
        } else if ((phase == kPhaseB || phase == kPhaseC) && mode != kModeFactor && !(P->opt.policy_flags & HINES_POLICY_NO_PDL)) {
            // split items: phases B and C start while the phase before them still runs (load, P1, their own sweeps) and
            // wait for it only where they import its results
            attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[0].val.programmaticStreamSerializationAllowed = 1;
            cfg.numAttrs = 1;
        }
        // ctl = phase | (blocks resident on the device at a time << 8): how far ahead a block prefetches a record
        const int per_sm = std::max(1, (int)(233472 / (cfg.dynamicSmemBytes + 1024)));
        const int ctl = (cl > 1 ? 0 : phase) | ((D->num_sms * per_sm) << 8);
        CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, recs, mg_, rg_, d, u, b, x, f0, f1, f2, n_, xh, xx, ctl, prof));
        return HINES_OK;
    };
    // Size classes are independent: the first runs on the caller's stream, the others on side streams forked
    // from it and joined back, so that their blocks share the SMs and fill each other's tails.  The three phases
    // of split items run in order on a stream of their own, the streaming path on another.
    const bool forked = D->fork != nullptr;
    bool used[DeviceTables::kSide] = {false, false, false};
    if (forked) CUDA_TRY(cudaEventRecord(D->fork, stream));
    if (D->sstream) {                                   // cells of the streaming path are independent of the rest
        CUDA_TRY(cudaStreamWaitEvent(D->sstream, D->fork, 0));
        if (hines_status_t sst = launch_streaming(D->sstream)) return sst;
        CUDA_TRY(cudaEventRecord(D->sjoin, D->sstream));
    }
    if (D->pstream) {
        CUDA_TRY(cudaStreamWaitEvent(D->pstream, D->fork, 0));
        for (size_t q = 0; q < P->class_smem_bytes.size(); ++q)
            if (P->class_phase[q] != kPhaseAll && P->class_count[q]) if (hines_status_t s2 = launch_class(q, D->pstream)) return s2;
        CUDA_TRY(cudaEventRecord(D->pjoin, D->pstream));
    }
    if (D->timing) CUDA_TRY(cudaEventRecord(D->ev[0], stream));
    int nth = 0;
    for (size_t q = 0; q < P->class_smem_bytes.size(); ++q) {
        if (!P->class_count[q]) continue;
        if (P->class_phase[q] != kPhaseAll) {
            if (!D->pstream) if (hines_status_t s2 = launch_class(q, stream)) return s2;      // in order on the caller's stream
            continue;
        }
        cudaStream_t ls = stream;
        if (forked && nth > 0) {
            const int k = (nth - 1) % DeviceTables::kSide;
            ls = D->side[k];
            if (!used[k]) { CUDA_TRY(cudaStreamWaitEvent(ls, D->fork, 0)); used[k] = true; }
        }
        ++nth;
        if (hines_status_t s2 = launch_class(q, ls)) return s2;
    }
    for (int k = 0; k < DeviceTables::kSide; ++k)
        if (used[k]) { CUDA_TRY(cudaEventRecord(D->join[k], D->side[k])); CUDA_TRY(cudaStreamWaitEvent(stream, D->join[k], 0)); }
    if (D->pstream) CUDA_TRY(cudaStreamWaitEvent(stream, D->pjoin, 0));
    if (D->timing) CUDA_TRY(cudaEventRecord(D->ev[1], stream));
    if (D->sstream) CUDA_TRY(cudaStreamWaitEvent(stream, D->sjoin, 0));
    else if (P->stream_level_begin.size() > 1) { if (hines_status_t sst = launch_streaming(stream)) return sst; }
    if (D->timing) D->timed_once = true;
    CUDA_TRY(cudaGetLastError());
    return HINES_OK;
}

static hines_status_t check_ptrs(const hines_plan* P, const void* d, const void* u, const void* b, const void* x)
{
    if (!P || !d || !u || !b || !x) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    return HINES_OK;
}

static bool overlaps(const void* a, const void* b, size_t bytes)
{
    const uintptr_t p = (uintptr_t)a, q = (uintptr_t)b;
    return p < q + bytes && q < p + bytes;
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
    const size_t bytes = (size_t)P->n * P->width;
    if (overlaps(x, d, bytes) || overlaps(x, u, bytes) || (x != b && overlaps(x, b, bytes))) {
        set_error("x may be exactly b (in place) or must not overlap d, u, b"); return HINES_ERR_INVALID_ARG;
    }
    if ((st = upload(P)) != HINES_OK) return st;
    if (P->dtype == HINES_F64)
        return launch_all<double>(P, (const double*)d, (const double*)u, (const double*)b, (double*)x, (cudaStream_t)stream);
    return launch_all<float>(P, (const float*)d, (const float*)u, (const float*)b, (float*)x, (cudaStream_t)stream);
}

// f3: everything that depends only on d and u, once; then only the right-hand side per step.
hines_status_t hines_factor(hines_plan_t* P, const void* d, const void* u, hines_stream_t stream)
{
    if (!P || !d || !u) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (!(P->opt.policy_flags & HINES_POLICY_FACTORED)) { set_error("hines_factor needs a plan created with HINES_POLICY_FACTORED"); return HINES_ERR_UNSUPPORTED; }
    if (P->n_stream_cells) { set_error("hines_factor: cells on the streaming path are not supported"); return HINES_ERR_UNSUPPORTED; }
    if (((uintptr_t)d | (uintptr_t)u) & 15) { set_error("device pointers must be 16-byte aligned"); return HINES_ERR_INVALID_ARG; }
    hines_status_t st = upload(P);
    if (st != HINES_OK) return st;
    DeviceTables* D = P->dev;
    const size_t bytes = ((size_t)P->n * P->width + 15) / 16 * 16;
    for (void*& f : D->fac) if (!f) { CUDA_TRY(cudaMalloc(&f, bytes)); D->bytes += (int64_t)bytes; }
    if (P->dtype == HINES_F64) st = launch_all<double>(P, (const double*)d, (const double*)u, nullptr, nullptr, (cudaStream_t)stream, kModeFactor);
    else st = launch_all<float>(P, (const float*)d, (const float*)u, nullptr, nullptr, (cudaStream_t)stream, kModeFactor);
    if (st == HINES_OK) D->factored = true;
    return st;
}

hines_status_t hines_solve_rhs(hines_plan_t* P, const void* b, void* x, hines_stream_t stream)
{
    if (!P || !b || !x) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (!P->dev || !P->dev->factored) { set_error("hines_solve_rhs: call hines_factor first"); return HINES_ERR_INVALID_ARG; }
    if (((uintptr_t)b | (uintptr_t)x) & 15) { set_error("device pointers must be 16-byte aligned"); return HINES_ERR_INVALID_ARG; }
    const size_t bytes = (size_t)P->n * P->width;
    if (x != b && overlaps(x, b, bytes)) { set_error("x may be exactly b (in place) or must not overlap it"); return HINES_ERR_INVALID_ARG; }
    if (P->dtype == HINES_F64) return launch_all<double>(P, nullptr, nullptr, (const double*)b, (double*)x, (cudaStream_t)stream, kModeRhs);
    return launch_all<float>(P, nullptr, nullptr, (const float*)b, (float*)x, (cudaStream_t)stream, kModeRhs);
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
    *resident_ms = 0.f; *stream_ms = 0.f;
    CUDA_TRY(cudaEventSynchronize(D->ev[1]));
    CUDA_TRY(cudaEventElapsedTime(resident_ms, D->ev[0], D->ev[1]));
    if (P->stream_level_begin.size() > 1) {
        CUDA_TRY(cudaEventSynchronize(D->ev[3]));
        CUDA_TRY(cudaEventElapsedTime(stream_ms, D->ev[2], D->ev[3]));
    }
    return HINES_OK;
}

hines_status_t hines_plan_enable_phase_clocks(hines_plan_t* P, int32_t enable)
{
    if (!P) { set_error("null pointer argument"); return HINES_ERR_INVALID_ARG; }
    hines_status_t st = upload(P);
    if (st != HINES_OK) return st;
    DeviceTables* D = P->dev;
    const size_t bytes = P->class_parts.size() * 8 * sizeof(unsigned long long);
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
    const int64_t bytes = (int64_t)(P->class_parts.size() * 8 * sizeof(unsigned long long));
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

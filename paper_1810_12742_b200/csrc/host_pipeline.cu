// hines_host_pipeline_*: the end-to-end entry for HOST buffers with the copies overlapped (include/hines.h).
//
// hines_solve_host moves d, u, b to the device, solves, moves x back: the link is busy in one direction at a time, and
// at 32 bytes per unknown the link IS the step (config 3: 4.5 GB per step against 2 ms of solve).  The cells of a batch
// are independent, so the batch is cut into slices of whole cells with about the same number of unknowns,
// each with a plan of its own, and the slices are pipelined on three streams:
//     copy-in stream   H2D of d, u, b of slice s         (slices back to back)
//     solve stream     hines_solve of slice s            (after its copy-in)
//     copy-out stream  D2H of x of slice s               (after its solve) -- while slice s+1 .. are still coming in
// PCIe is full duplex: the step takes about the 24 bytes per unknown going in plus the last slice's way out, instead
// of 32.  Built on the public API only (hines_plan_create / hines_solve); no kernel of its own.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <new>
#include <string>
#include <vector>

#include "plan_internal.h"

struct hines_host_pipeline {
    int32_t dtype = 0, width = 8, device = -1;
    int64_t n = 0, ncells = 0;
    struct Slice {
        hines_plan_t* plan = nullptr;
        int64_t lo = 0, len = 0;          // compartments [lo, lo + len) of the batch
        int64_t off = 0;                  // element offset of the slice in the device buffers (32-element aligned)
        cudaEvent_t in = nullptr, out = nullptr;
    };
    std::vector<Slice> slices;
    void* dev[4] = {nullptr, nullptr, nullptr, nullptr};      // d, u, b, x
    cudaStream_t s_in = nullptr, s_solve = nullptr, s_out = nullptr;
};

namespace {

void destroy(hines_host_pipeline* P)
{
    if (!P) return;
    for (auto& s : P->slices) {
        if (s.plan) hines_plan_destroy(s.plan);
        if (s.in) cudaEventDestroy(s.in);
        if (s.out) cudaEventDestroy(s.out);
    }
    for (void*& p : P->dev) if (p) { cudaFree(p); p = nullptr; }
    for (cudaStream_t* s : {&P->s_in, &P->s_solve, &P->s_out}) if (*s) { cudaStreamDestroy(*s); *s = nullptr; }
    delete P;
}

#define PIPE_TRY(expr)                                                                               \
    do {                                                                                             \
        cudaError_t e_ = (expr);                                                                     \
        if (e_ != cudaSuccess) {                                                                     \
            hines::set_error(std::string("hines_host_pipeline: " #expr ": ") + cudaGetErrorString(e_)); \
            return e_ == cudaErrorMemoryAllocation ? HINES_ERR_ALLOC : HINES_ERR_CUDA;               \
        }                                                                                            \
    } while (0)

hines_status_t setup_device(hines_host_pipeline* P)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        hines::set_error("no CUDA device: this library has no CPU fallback");
        return HINES_ERR_CUDA;
    }
    // every resource is created once: a call that failed half way is picked up where it stopped by the next one, and the
    // pipeline counts as set up (device >= 0) only when everything is there
    int dev = -1;
    PIPE_TRY(cudaGetDevice(&dev));
    int64_t total = 0;
    for (auto& s : P->slices) { s.off = total; total += (s.len + 31) / 32 * 32; }
    for (void*& p : P->dev) if (!p) PIPE_TRY(cudaMalloc(&p, (size_t)total * P->width));
    for (cudaStream_t* st : {&P->s_in, &P->s_solve, &P->s_out}) if (!*st) PIPE_TRY(cudaStreamCreateWithFlags(st, cudaStreamNonBlocking));
    for (auto& s : P->slices) {
        if (!s.in) PIPE_TRY(cudaEventCreateWithFlags(&s.in, cudaEventDisableTiming));
        if (!s.out) PIPE_TRY(cudaEventCreateWithFlags(&s.out, cudaEventDisableTiming));
        if (hines_status_t st = hines_plan_upload(s.plan)) return st;
    }
    P->device = dev;
    return HINES_OK;
}

}  // namespace

extern "C" hines_status_t hines_host_pipeline_create(const int32_t* parent, const int64_t* cell_offsets, int64_t ncells,
                                                     hines_dtype_t dtype, const hines_options_t* opt, int32_t nslices,
                                                     hines_host_pipeline_t** out)
{
    using hines::set_error;
    if (!parent || !cell_offsets || !out) { set_error("hines_host_pipeline_create: null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (ncells <= 0 || nslices < 0 || nslices > 1024) { set_error("hines_host_pipeline_create: need ncells > 0 and 0 <= nslices <= 1024"); return HINES_ERR_INVALID_ARG; }
    *out = nullptr;
    hines_host_pipeline* P = nullptr;
    try {
        P = new hines_host_pipeline();
        P->dtype = dtype; P->width = dtype == HINES_F64 ? 8 : 4; P->ncells = ncells; P->n = cell_offsets[ncells];
        const int64_t want = std::min<int64_t>(nslices == 0 ? 8 : nslices, ncells);
        // slice k ends at the first cell boundary at or beyond k/want of the unknowns
        std::vector<int64_t> cut(1, 0);
        for (int64_t k = 1; k <= want; ++k) {
            const int64_t target = k == want ? P->n : P->n / want * k;
            const int64_t c = std::lower_bound(cell_offsets + cut.back(), cell_offsets + ncells, target) - cell_offsets;
            if (c > cut.back()) cut.push_back(std::min(c, ncells));
        }
        if (cut.back() != ncells) cut.back() = ncells;
        std::vector<int64_t> offs;
        for (size_t k = 0; k + 1 < cut.size(); ++k) {
            const int64_t c0 = cut[k], c1 = cut[k + 1];
            offs.resize((size_t)(c1 - c0 + 1));
            for (int64_t c = c0; c <= c1; ++c) offs[(size_t)(c - c0)] = cell_offsets[c] - cell_offsets[c0];
            hines_host_pipeline::Slice s;
            s.lo = cell_offsets[c0]; s.len = cell_offsets[c1] - cell_offsets[c0];
            // parent[] is cell-local: the slice's part of it serves as it is
            const hines_status_t st = hines_plan_create(parent + s.lo, offs.data(), c1 - c0, dtype, opt, &s.plan);
            if (st != HINES_OK) { destroy(P); return st; }
            P->slices.push_back(s);
        }
    } catch (const std::bad_alloc&) {
        destroy(P);
        set_error("hines_host_pipeline_create: out of host memory");
        return HINES_ERR_ALLOC;
    }
    *out = P;
    return HINES_OK;
}

extern "C" hines_status_t hines_host_pipeline_solve(hines_host_pipeline_t* P, const void* d, const void* u, const void* b, void* x)
{
    using hines::set_error;
    if (!P || !d || !u || !b || !x) { set_error("hines_host_pipeline_solve: null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (P->device < 0) { if (hines_status_t st = setup_device(P)) return st; }
    const int64_t w = P->width;
    const char* src[3] = {static_cast<const char*>(d), static_cast<const char*>(u), static_cast<const char*>(b)};
    for (auto& s : P->slices) {
        const size_t bytes = (size_t)(s.len * w);
        for (int a = 0; a < 3; ++a)
            PIPE_TRY(cudaMemcpyAsync(static_cast<char*>(P->dev[a]) + s.off * w, src[a] + s.lo * w, bytes, cudaMemcpyHostToDevice, P->s_in));
        PIPE_TRY(cudaEventRecord(s.in, P->s_in));
        PIPE_TRY(cudaStreamWaitEvent(P->s_solve, s.in, 0));
        const hines_status_t st = hines_solve(s.plan, static_cast<char*>(P->dev[0]) + s.off * w, static_cast<char*>(P->dev[1]) + s.off * w,
                                              static_cast<char*>(P->dev[2]) + s.off * w, static_cast<char*>(P->dev[3]) + s.off * w, P->s_solve);
        if (st != HINES_OK) return st;
        PIPE_TRY(cudaEventRecord(s.out, P->s_solve));
        PIPE_TRY(cudaStreamWaitEvent(P->s_out, s.out, 0));
        PIPE_TRY(cudaMemcpyAsync(static_cast<char*>(x) + s.lo * w, static_cast<char*>(P->dev[3]) + s.off * w, bytes, cudaMemcpyDeviceToHost, P->s_out));
    }
    PIPE_TRY(cudaStreamSynchronize(P->s_out));
    PIPE_TRY(cudaStreamSynchronize(P->s_in));
    return HINES_OK;
}

extern "C" hines_status_t hines_host_pipeline_slices(const hines_host_pipeline_t* P, int32_t* nslices, int64_t* first_compartment, int64_t capacity)
{
    if (!P || !nslices) { hines::set_error("hines_host_pipeline_slices: null pointer argument"); return HINES_ERR_INVALID_ARG; }
    *nslices = (int32_t)P->slices.size();
    if (first_compartment) {
        if (capacity < (int64_t)P->slices.size() + 1) { hines::set_error("hines_host_pipeline_slices: capacity too small"); return HINES_ERR_INVALID_ARG; }
        for (size_t k = 0; k < P->slices.size(); ++k) first_compartment[k] = P->slices[k].lo;
        first_compartment[P->slices.size()] = P->n;
    }
    return HINES_OK;
}

extern "C" hines_status_t hines_host_pipeline_destroy(hines_host_pipeline_t* P)
{
    destroy(P);
    return HINES_OK;
}

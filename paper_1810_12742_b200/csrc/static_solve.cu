// hines_solve_static: the one entry point of libhines_b200.so that allocates NOTHING (include/hines.h).
//
// For callers that cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid
// it.  Every other solve entry needs an uploaded plan (hines_plan_upload allocates the tables, the exchange buffers and
// the streaming workspace).  This one needs no plan: the caller passes the topology as DEVICE arrays next to d, u, b, x,
// and the kernel's scratch -- the working diagonal of the backward sweep, what the streaming path keeps in the
// plan-owned workspace (solve.cu, hines_stream_backward / hines_stream_forward: ws_f, ws_c) -- lives in a file-scope
// static __device__ array of HINES_STATIC_SCRATCH_BYTES.  Every GPU that loads the library holds that array until the
// process exits.
//
// The kernel is the whole-cell variant of the streaming kernels: one thread per cell walks Listing 2 of the paper
// (reading G1 of DESIGN.md: u[i] couples i to parent[i]) over the cell's compartments in natural order,
//     backward  i = last .. first+1:  f = u[i] / D[i];  D[p] -= f u[i];  B[p] -= f B[i]
//     forward   x[first] = B[first] / D[first];  x[i] = (B[i] - u[i] x[p]) / D[i]
// with D in the scratch array and B in x.  It is a fallback, not the fast path: a thread's accesses are not coalesced
// with its neighbours'; use hines_solve where a plan can be uploaded.
//
// The array's NAME is a host-side stand-in in host code, not a device address: its address on the current device comes
// from cudaGetSymbolAddress, looked up once per device, with that device current, by the first call on it.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>
#include <string>

#include "plan_internal.h"

namespace {

// Scratch of hines_solve_static: the working diagonal, one value per compartment.  Shared by every call; keeps the last
// call's contents.  Nothing in it has to start at zero: the kernel writes D[i] = d[i] for every compartment of a cell
// before it reads any of them.
static __device__ __align__(256) unsigned char g_static_scratch[HINES_STATIC_SCRATCH_BYTES];

enum { kMaxDevices = 64 };
std::mutex g_mu;
void* g_scratch_addr[kMaxDevices] = {};        // device address of g_static_scratch, per device ordinal

template <typename T>
__global__ void __launch_bounds__(128)
hines_cells_static_kernel(const int32_t* __restrict__ parent, const int64_t* __restrict__ cell_offsets, int64_t ncells,
                          int64_t n, const T* __restrict__ d, const T* __restrict__ u, const T* b, T* x, T* D)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncells) return;
    int64_t lo = cell_offsets[c], hi = cell_offsets[c + 1];
    if (lo < 0) lo = 0;
    if (hi > n) hi = n;                                  // never outside the arrays, whatever the offsets say
    if (hi <= lo) return;
    for (int64_t i = lo; i < hi; ++i) { D[i] = d[i]; x[i] = b[i]; }     // x may be b
    // a parent outside [0, i - lo) is treated as "no parent": no access outside the cell
    for (int64_t i = hi - 1; i > lo; --i) {
        const int64_t pl = parent[i];
        if (pl < 0 || pl >= i - lo) continue;
        const int64_t p = lo + pl;
        const T ui = u[i];
        const T f = ui / D[i];
        D[p] -= f * ui;
        x[p] -= f * x[i];
    }
    x[lo] = x[lo] / D[lo];
    for (int64_t i = lo + 1; i < hi; ++i) {
        const int64_t pl = parent[i];
        T Bi = x[i];
        if (pl >= 0 && pl < i - lo) Bi -= u[i] * x[lo + pl];
        x[i] = Bi / D[i];
    }
}

}  // namespace

extern "C" hines_status_t hines_solve_static(const int32_t* parent, const int64_t* cell_offsets, int64_t ncells, int64_t n,
                                             const void* d, const void* u, const void* b, void* x, int32_t dtype,
                                             hines_stream_t stream)
{
    using hines::set_error;
    if (!parent || !cell_offsets || !d || !u || !b || !x) { set_error("hines_solve_static: null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (dtype != HINES_F64 && dtype != HINES_F32) { set_error("hines_solve_static: dtype must be HINES_F64 or HINES_F32"); return HINES_ERR_INVALID_ARG; }
    if (ncells <= 0 || n <= 0 || ncells > n) { set_error("hines_solve_static: need 0 < ncells <= n"); return HINES_ERR_INVALID_ARG; }
    const int64_t w = dtype == HINES_F64 ? 8 : 4;
    if (n > (int64_t)HINES_STATIC_SCRATCH_BYTES / w) {
        set_error("hines_solve_static: n = " + std::to_string(n) + " exceeds the static scratch array (" +
                  std::to_string((int64_t)HINES_STATIC_SCRATCH_BYTES / w) + " unknowns of this dtype, HINES_STATIC_SCRATCH_BYTES = " +
                  std::to_string((int64_t)HINES_STATIC_SCRATCH_BYTES) + "); use hines_solve with an uploaded plan");
        return HINES_ERR_UNSUPPORTED;
    }
    if (x != b) {                                        // x may be exactly b, else the two must not overlap
        const uintptr_t xa = (uintptr_t)x, ba = (uintptr_t)b, bytes = (uintptr_t)(n * w);
        if (xa < ba + bytes && ba < xa + bytes) { set_error("hines_solve_static: x overlaps b without being equal to it"); return HINES_ERR_INVALID_ARG; }
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { set_error(std::string("hines_solve_static: cudaGetDevice: ") + cudaGetErrorString(e)); return HINES_ERR_CUDA; }
    if (dev < 0 || dev >= kMaxDevices) { set_error("hines_solve_static: device ordinal out of range"); return HINES_ERR_UNSUPPORTED; }
    void* scratch = nullptr;
    {
        // once per device, with that device current: the device address of the static array
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_scratch_addr[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_static_scratch);
            if (e != cudaSuccess || !p) {
                set_error(std::string("hines_solve_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
                return HINES_ERR_CUDA;
            }
            g_scratch_addr[dev] = p;
        }
        scratch = g_scratch_addr[dev];
    }
    const unsigned threads = 128, blocks = (unsigned)((ncells + threads - 1) / threads);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (dtype == HINES_F64)
        hines_cells_static_kernel<double><<<blocks, threads, 0, s>>>(parent, cell_offsets, ncells, n, static_cast<const double*>(d),
            static_cast<const double*>(u), static_cast<const double*>(b), static_cast<double*>(x), static_cast<double*>(scratch));
    else
        hines_cells_static_kernel<float><<<blocks, threads, 0, s>>>(parent, cell_offsets, ncells, n, static_cast<const float*>(d),
            static_cast<const float*>(u), static_cast<const float*>(b), static_cast<float*>(x), static_cast<float*>(scratch));
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string("hines_solve_static: launch: ") + cudaGetErrorString(e)); return HINES_ERR_CUDA; }
    return HINES_OK;
}

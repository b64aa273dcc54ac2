// hines_gather / hines_scatter (include/hines.h): the permutation of a re-rooted batch (f2, "permute all
// unknowns such that they form a new Hines matrix") carried through load and store on the device.  HBM-bound, one
// element per thread: the contiguous side is coalesced, the indexed side follows the permutation, which moves whole
// branches (runs of consecutive compartments), so most of its sectors are full too.
#include <cuda_runtime.h>

#include <cstdint>
#include <string>

#include "plan_internal.h"

namespace {

template <typename T, bool SCATTER>
__global__ void __launch_bounds__(256)
hines_permute_kernel(T* __restrict__ dst, const T* __restrict__ src, const int64_t* __restrict__ index, int64_t n)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += stride) {
        const int64_t j = index[k];
        if (SCATTER) dst[j] = src[k]; else dst[k] = src[j];
    }
}

template <bool SCATTER>
hines_status_t permute(void* dst, const void* src, const int64_t* index, int64_t n, int32_t dtype, hines_stream_t stream, const char* who)
{
    using hines::set_error;
    if (!dst || !src || !index) { set_error(std::string(who) + ": null pointer argument"); return HINES_ERR_INVALID_ARG; }
    if (n < 0) { set_error(std::string(who) + ": n < 0"); return HINES_ERR_INVALID_ARG; }
    if (dtype != HINES_F64 && dtype != HINES_F32) { set_error(std::string(who) + ": dtype must be HINES_F64 or HINES_F32"); return HINES_ERR_INVALID_ARG; }
    if (n == 0) return HINES_OK;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        set_error(std::string(who) + ": no CUDA device: this library has no CPU fallback");
        return HINES_ERR_CUDA;
    }
    const int64_t want = (n + 255) / 256;
    const unsigned blocks = (unsigned)(want < (int64_t)sms * 16 ? want : (int64_t)sms * 16);     // a multiple of the SM count when large
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (dtype == HINES_F64)
        hines_permute_kernel<double, SCATTER><<<blocks, 256, 0, s>>>(static_cast<double*>(dst), static_cast<const double*>(src), index, n);
    else
        hines_permute_kernel<float, SCATTER><<<blocks, 256, 0, s>>>(static_cast<float*>(dst), static_cast<const float*>(src), index, n);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string(who) + ": launch: " + cudaGetErrorString(e)); return HINES_ERR_CUDA; }
    return HINES_OK;
}

}  // namespace

extern "C" hines_status_t hines_gather(void* dst, const void* src, const int64_t* index, int64_t n, int32_t dtype, hines_stream_t stream)
{
    return permute<false>(dst, src, index, n, dtype, stream, "hines_gather");
}

extern "C" hines_status_t hines_scatter(void* dst, const void* src, const int64_t* index, int64_t n, int32_t dtype, hines_stream_t stream)
{
    return permute<true>(dst, src, index, n, dtype, stream, "hines_scatter");
}

// noalloc.cu -- sgp_rel_error_static (include/sgp.h): the relative reconstruction error of Eq.25 for callers
// that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The kernel is
// err_kernel of extra.cuh in its mode 0 (same grid, same reduction tree, same order of the partial sums) with the per-CTA
// partials and the arrival counter in a file-scope device array instead of the plan's workspace.  Nothing here calls
// cudaMalloc, cudaFree or a library routine that allocates.
//
// The array is shared by every call on a device and keeps the last call's contents: the partials are overwritten before
// they are read; the arrival counter, which must start at zero, is cleared on the stream in front of every launch
// (cudaMemsetAsync: no allocation), so a call that was cut short cannot poison the next one.  Two calls that overlap
// on the GPU (different streams, no ordering between them) race on it.
#include <cuda_runtime.h>
#include <string>
#include "../../include/sgp.h"
#include "sgp_dev.cuh"

namespace sgpk {

extern thread_local std::string g_last_cuda_error;      // api.cu

constexpr int kStaticMaxCtas = 1184;                     // 8 x 148: the grid cap of the plan's element-wise kernels (ew_grid)
constexpr int kStaticPartDoubles = 2 * kStaticMaxCtas;   // (sum e^2, sum t^2) per CTA
constexpr int kStaticScratchDoubles = kStaticPartDoubles + 32;   // + one 256-byte line for the arrival counter: 19 200 bytes

// In host code this name is a stand-in, not a device address: the host takes the address with cudaGetSymbolAddress
// (static_scratch_ptr below), device code may name the array directly.
static __device__ __align__(256) double sgp_static_scratch[kStaticScratchDoubles];

template <typename T>
__global__ void __launch_bounds__(256) rel_error_static_kernel(const T *f, const T *truth, size_t n, double *scratch, double *rho_out)
{
    __shared__ double red[2 * 32];
    double *part = scratch;
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch + kStaticPartDoubles);
    double acc[2] = {0.0, 0.0};
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double t = (double)truth[i], e = (double)f[i] - t;
        acc[0] += e * e; acc[1] += t * t;
    }
    block_reduce_sum<2>(acc, red);
    if (publish_partials<2>(acc, part, blockIdx.x, gridDim.x, ticket)) {      // re-arms the counter for the next call
        final_sum<2>(acc, part, gridDim.x, red);
        if (threadIdx.x == 0) *rho_out = sqrt(acc[0]) / sqrt(acc[1]);
    }
}

// device address of the array, looked up once per device with that device current
static int static_scratch_ptr(double **out)
{
    constexpr int kMaxDevices = 64;
    static double *ptrs[kMaxDevices];                    // written once per slot; a race between two threads writes the same value
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess && (dev < 0 || dev >= kMaxDevices)) { g_last_cuda_error = "sgp_rel_error_static: device index beyond 63"; return SGP_ERR_ARG; }
    if (e == cudaSuccess && !ptrs[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, sgp_static_scratch);
        if (e == cudaSuccess) ptrs[dev] = p;
    }
    if (e != cudaSuccess) {
        g_last_cuda_error = std::string("sgp_rel_error_static: ") + cudaGetErrorString(e);
        (void)cudaGetLastError();
        return SGP_ERR_CUDA;
    }
    *out = ptrs[dev];
    return SGP_OK;
}

}  // namespace sgpk

using namespace sgpk;

extern "C" {

size_t sgp_rel_error_static_max(void) { return (size_t)SGP_STATIC_MAX_ELEMS; }

int sgp_rel_error_static(const void *f, const void *truth, size_t n, int dtype, double *rho_out, void *stream)
{
    if (!f || !truth || !rho_out || n == 0) return SGP_ERR_ARG;
    if (dtype != SGP_F32 && dtype != SGP_F64) return SGP_ERR_ARG;
    if (n > (size_t)SGP_STATIC_MAX_ELEMS) {
        g_last_cuda_error = "sgp_rel_error_static: n exceeds SGP_STATIC_MAX_ELEMS (4096 x 4096 = 16777216 elements); "
                            "nothing was launched -- use a plan (sgp_plan_run with sgp_result.truth) for larger arrays";
        return SGP_ERR_ARG;
    }
    double *scratch = nullptr;
    int rc = static_scratch_ptr(&scratch);
    if (rc) return rc;
    size_t b = (n + 255) / 256;
    const int grid = (int)(b > (size_t)kStaticMaxCtas ? (size_t)kStaticMaxCtas : b);
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaMemsetAsync(scratch + kStaticPartDoubles, 0, 256, st);          // the counter's line starts at zero
    if (e != cudaSuccess) { g_last_cuda_error = std::string("sgp_rel_error_static: ") + cudaGetErrorString(e); (void)cudaGetLastError(); return SGP_ERR_CUDA; }
    if (dtype == SGP_F32) rel_error_static_kernel<float><<<grid, 256, 0, st>>>((const float *)f, (const float *)truth, n, scratch, rho_out);
    else                  rel_error_static_kernel<double><<<grid, 256, 0, st>>>((const double *)f, (const double *)truth, n, scratch, rho_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) { g_last_cuda_error = std::string("sgp_rel_error_static: ") + cudaGetErrorString(e); return SGP_ERR_CUDA; }
    return SGP_OK;
}

}  // extern "C"

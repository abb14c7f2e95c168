// plan.cuh -- host side of a plan: workspace, twiddle tables, kernel launch helpers and the two
// iteration drivers (SGP, RL).  One templated implementation per element type behind a small
// virtual interface used by the C ABI (api.cu).
#pragma once
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <string>
#include <vector>
#include <type_traits>
#include "dispatch.h"

namespace sgpk {

extern thread_local std::string g_last_cuda_error;

#define SGP_CUDA_TRY(call)                                                                 \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess) {                                                           \
            g_last_cuda_error = std::string(#call) + ": " + cudaGetErrorString(e_);        \
            return e_ == cudaErrorMemoryAllocation ? SGP_ERR_ALLOC : SGP_ERR_CUDA;         \
        }                                                                                  \
    } while (0)

struct PlanBase {
    int kind = 0, p = 1, ny = 0, nx = 0, dtype = 0;
    int nb = 1;                    // problems of a batched plan (sgp_plan_create_batched); 1 = an ordinary plan
    Geom G{};
    sgp_options opt{};
    bool psf_set = false;
    long nR = 0;
    size_t bytes_allocated = 0;
    long launches = 0;
    bool profiling = false;
    double prof_ms[SGP_PROF_SLOTS] = {0};
    long prof_count[SGP_PROF_SLOTS] = {0};
    virtual ~PlanBase() {}
    virtual int init() = 0;
    virtual int set_psf(const void *const *psf, cudaStream_t st) = 0;
    virtual int run(int algorithm, const void *const *g, const void *const *b_arr, const double *b_const,
                    const void *f0, void *f_out, const sgp_options *opt, sgp_result *res, cudaStream_t st) = 0;
    virtual int run_batched(int algorithm, const void *const *g, const void *const *b_arr, const double *b_const,
                            const void *const *f0, void *const *f_out, const sgp_options *opt, sgp_result *res, cudaStream_t st) = 0;
    virtual int apply(bool transpose, int j, const void *x, void *out, cudaStream_t st) = 0;
    virtual int get_mask(unsigned char *maskR_out, void *alpha_out, long *nR_out, cudaStream_t st) = 0;
    virtual int rfft2(const void *x, void *spec_out, cudaStream_t st) = 0;
    virtual int irfft2(const void *spec_in, void *x_out, cudaStream_t st) = 0;
};

int validate_options(const sgp_options *o);
int choose_tiles(int ny, int nx, int dtype, const sgp_options *opt, int *C, int *RB, int nb = 1);
size_t workspace_bytes(int kind, int p, int ny, int nx, int dtype);
PlanBase *make_plan_f32();
PlanBase *make_plan_f64();

}  // namespace sgpk

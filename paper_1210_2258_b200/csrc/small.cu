// small.cu -- instantiations of the one-cluster-per-problem SGP kernel (small.cuh) and their look-up
#include "small.cuh"

namespace sgpk {

template <typename T, int NY, int NX, int NC, bool TWO>
static small_kernel_t<T> pick2(bool masked, bool rl)
{
    if (rl) return masked ? small_sgp_kernel<T, NY, NX, NC, true, true, TWO> : small_sgp_kernel<T, NY, NX, NC, false, true, TWO>;
    return masked ? small_sgp_kernel<T, NY, NX, NC, true, false, TWO> : small_sgp_kernel<T, NY, NX, NC, false, false, TWO>;
}
template <typename T, int NY, int NX, int NC>
static small_kernel_t<T> pick(bool masked, bool rl, bool two, int *nc, int *threads, size_t *smem, int *er, int *ec)
{
    using K = SmallCfg<T, NY, NX, NC>;
    *nc = NC; *threads = K::NT; *smem = K::smem; *er = K::Er; *ec = K::Ec;
    return two ? pick2<T, NY, NX, NC, true>(masked, rl) : pick2<T, NY, NX, NC, false>(masked, rl);
}

template <> small_kernel_t<float> get_small<float>(int ny, int nx, bool masked, bool rl, bool two, int *nc, int *threads, size_t *smem, int *er, int *ec)
{
    if (ny == 128 && nx == 128) return pick<float, 128, 128, 8>(masked, rl, two, nc, threads, smem, er, ec);
    if (ny == 256 && nx == 256) return pick<float, 256, 256, 16>(masked, rl, two, nc, threads, smem, er, ec);
    return nullptr;
}
template <> small_kernel_t<double> get_small<double>(int ny, int nx, bool masked, bool rl, bool two, int *nc, int *threads, size_t *smem, int *er, int *ec)
{
    if (ny == 128 && nx == 128) return pick<double, 128, 128, 8>(masked, rl, two, nc, threads, smem, er, ec);
    if (ny == 256 && nx == 256) return pick<double, 256, 256, 16>(masked, rl, two, nc, threads, smem, er, ec);
    return nullptr;
}

}  // namespace sgpk

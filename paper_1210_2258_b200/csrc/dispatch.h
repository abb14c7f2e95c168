// dispatch.h -- look-up of the kernel instantiations by FFT length and mode (defined in inst_*.cu, one
// translation unit per element type and kernel family so that they compile in parallel).
#pragma once
#include "kernels.cuh"

namespace sgpk {

template <typename T> using row_kernel_t = void (*)(const RowParams<T>);
template <typename T> using col_kernel_t = void (*)(const ColParams<T>);

// L = nx/2 (row kernels) or ny (column kernel); nullptr if the length is not supported
template <typename T> row_kernel_t<T> get_row_fwd(int L, int mode, bool masked);
template <typename T> row_kernel_t<T> get_row_inv(int L, int mode, bool masked);
// tile_cols: the plan's tile width; the product modes have a variant compiled for the default width (col.cuh)
template <typename T> col_kernel_t<T> get_col(int L, int mode, bool multi, int tile_cols = 0);
// two-CTAs-per-SM form of the single-image product modes (col.cuh: col2_kernel); nullptr where it does not exist
template <typename T> col_kernel_t<T> get_col2(int L, int mode);

// supported grid sizes (ny and nx independently)
inline bool size_supported(int n)
{
    switch (n) {
    case 64: case 128: case 256: case 512: case 1024: case 2048: case 4096:                                  // 2^a
    case 80: case 160: case 200: case 320: case 400: case 640: case 800: case 1000: case 1280: case 1600:    // 2^a 5^b, multiples of 40
    case 2000: case 2560: case 3200: case 4000:
        return true;
    default: return false;
    }
}

}  // namespace sgpk

// included by the inst_col*.cu stubs with SGP_T, SGP_COL_PART (0 = powers of two + col2_kernel, 1 = 2^a 5^b lengths),
// SGP_COL_FN and SGP_COL2_FN (names of this translation unit's look-up functions) defined
#include "dispatch.h"
namespace sgpk {
// The product modes exist only in their image-loop form (MULTI = true; a single image is p = 1): ptxas allocates
// it without spills where the specialised single-image form spilled 116-170 bytes, and it is 2 us per pass faster at 2048^2.
template <int L> static col_kernel_t<SGP_T> pick_col(int mode, bool multi, int tile_cols)
{
    constexpr int CD = col_default_C<SGP_T>(L);
    const bool batch = tile_cols < 0;          // a negative tile width asks for the batched-plan variant (blockIdx.z = problem)
    if (batch) {
        (void)multi;
        if (-tile_cols == CD && mode == CM_CONJSUM) return col_kernel<SGP_T, L, CM_CONJSUM, true, CD, true>;
        if (-tile_cols == CD && mode == CM_MULT) return col_kernel<SGP_T, L, CM_MULT, true, CD, true>;
        if (mode == CM_CONJSUM) return col_kernel<SGP_T, L, CM_CONJSUM, true, 0, true>;
        if (mode == CM_MULT) return col_kernel<SGP_T, L, CM_MULT, true, 0, true>;
        return nullptr;
    }
    if (tile_cols == CD && mode == CM_CONJSUM) return col_kernel<SGP_T, L, CM_CONJSUM, true, CD>;
    if (tile_cols == CD && mode == CM_MULT) return col_kernel<SGP_T, L, CM_MULT, true, CD>;
    if (mode == CM_FWD) return col_kernel<SGP_T, L, CM_FWD, false>;
    if (mode == CM_INV) return col_kernel<SGP_T, L, CM_INV, false>;
    if (mode == CM_CONJSUM) return col_kernel<SGP_T, L, CM_CONJSUM, true>;
    return col_kernel<SGP_T, L, CM_MULT, true>;
}
col_kernel_t<SGP_T> SGP_COL_FN(int L, int mode, bool multi, int tile_cols)
{
    switch (L) {
#ifdef SGP_FAST_BUILD
#if SGP_COL_PART == 0
    case 256: return pick_col<256>(mode, multi, tile_cols);
    case 2048: return pick_col<2048>(mode, multi, tile_cols);
#endif
#elif SGP_COL_PART == 0
    case 64: return pick_col<64>(mode, multi, tile_cols);
    case 128: return pick_col<128>(mode, multi, tile_cols);
    case 256: return pick_col<256>(mode, multi, tile_cols);
    case 512: return pick_col<512>(mode, multi, tile_cols);
    case 1024: return pick_col<1024>(mode, multi, tile_cols);
    case 2048: return pick_col<2048>(mode, multi, tile_cols);
    case 4096: return pick_col<4096>(mode, multi, tile_cols);
#else
    case 80: return pick_col<80>(mode, multi, tile_cols);
    case 160: return pick_col<160>(mode, multi, tile_cols);
    case 200: return pick_col<200>(mode, multi, tile_cols);
    case 320: return pick_col<320>(mode, multi, tile_cols);
    case 400: return pick_col<400>(mode, multi, tile_cols);
    case 640: return pick_col<640>(mode, multi, tile_cols);
    case 800: return pick_col<800>(mode, multi, tile_cols);
    case 1000: return pick_col<1000>(mode, multi, tile_cols);
    case 1280: return pick_col<1280>(mode, multi, tile_cols);
    case 1600: return pick_col<1600>(mode, multi, tile_cols);
    case 2000: return pick_col<2000>(mode, multi, tile_cols);
    case 2560: return pick_col<2560>(mode, multi, tile_cols);
    case 3200: return pick_col<3200>(mode, multi, tile_cols);
    case 4000: return pick_col<4000>(mode, multi, tile_cols);
#endif
    default: return nullptr;
    }
}
#if SGP_COL_PART == 0
template <int L> static col_kernel_t<SGP_T> pick_col2(int mode)
{
    if constexpr (sizeof(SGP_T) == 4) {
        if (mode == CM_CONJSUM) return col2_kernel<SGP_T, L, CM_CONJSUM>;
        if (mode == CM_MULT) return col2_kernel<SGP_T, L, CM_MULT>;
    }
    return nullptr;
}
col_kernel_t<SGP_T> SGP_COL2_FN(int L, int mode)
{
    switch (L) {
#ifndef SGP_FAST_BUILD
    case 1024: return pick_col2<1024>(mode);
    case 4096: return pick_col2<4096>(mode);
#endif
    case 2048: return pick_col2<2048>(mode);
    default: return nullptr;
    }
}
#endif
}  // namespace sgpk

// included by inst_col_f32.cu / inst_col_f64.cu with SGP_T defined
#include "dispatch.h"
namespace sgpk {
// The product modes exist only in their image-loop form (MULTI = true; a single image is p = 1): ptxas allocates
// it without spills where the specialised single-image form spilled 116-170 bytes, and it is 2 us per pass faster at 2048^2.
template <int L> static col_kernel_t<SGP_T> pick_col(int mode, bool multi, int tile_cols)
{
    (void)multi;
    constexpr int CD = col_default_C<SGP_T>(L);
    if (tile_cols == CD && mode == CM_CONJSUM) return col_kernel<SGP_T, L, CM_CONJSUM, true, CD>;
    if (tile_cols == CD && mode == CM_MULT) return col_kernel<SGP_T, L, CM_MULT, true, CD>;
    if (mode == CM_FWD) return col_kernel<SGP_T, L, CM_FWD, false>;
    if (mode == CM_INV) return col_kernel<SGP_T, L, CM_INV, false>;
    if (mode == CM_CONJSUM) return col_kernel<SGP_T, L, CM_CONJSUM, true>;
    return col_kernel<SGP_T, L, CM_MULT, true>;
}
template <> col_kernel_t<SGP_T> get_col<SGP_T>(int L, int mode, bool multi, int tile_cols)
{
    switch (L) {
    case 64: return pick_col<64>(mode, multi, tile_cols);
    case 128: return pick_col<128>(mode, multi, tile_cols);
    case 256: return pick_col<256>(mode, multi, tile_cols);
    case 320: return pick_col<320>(mode, multi, tile_cols);
    case 512: return pick_col<512>(mode, multi, tile_cols);
    case 640: return pick_col<640>(mode, multi, tile_cols);
    case 1024: return pick_col<1024>(mode, multi, tile_cols);
    case 1280: return pick_col<1280>(mode, multi, tile_cols);
    case 2048: return pick_col<2048>(mode, multi, tile_cols);
    case 4096: return pick_col<4096>(mode, multi, tile_cols);
    default: return nullptr;
    }
}
template <int L> static col_kernel_t<SGP_T> pick_col2(int mode)
{
    if constexpr (sizeof(SGP_T) == 4) {
        if (mode == CM_CONJSUM) return col2_kernel<SGP_T, L, CM_CONJSUM>;
        if (mode == CM_MULT) return col2_kernel<SGP_T, L, CM_MULT>;
    }
    return nullptr;
}
template <> col_kernel_t<SGP_T> get_col2<SGP_T>(int L, int mode)
{
    switch (L) {
    case 1024: return pick_col2<1024>(mode);
    case 2048: return pick_col2<2048>(mode);
    case 4096: return pick_col2<4096>(mode);
    default: return nullptr;
    }
}
}  // namespace sgpk

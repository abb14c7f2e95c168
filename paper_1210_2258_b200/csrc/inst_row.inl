// included by the inst_row*.cu stubs with SGP_T, SGP_ROW_FWD (1 = forward, 0 = inverse), SGP_ROW_PART (which lengths) and
// SGP_ROW_FN (the name of the look-up function of this translation unit; inst_dispatch.cu puts the parts together) defined
#include "dispatch.h"
namespace sgpk {
#if SGP_ROW_FWD
template <int L, bool MK> static row_kernel_t<SGP_T> pick_rowf(int mode)
{
    switch (mode) {
    case RF_PLAIN: return row_fwd_kernel<SGP_T, L, RF_PLAIN, MK>;
    case RF_SETUP: return row_fwd_kernel<SGP_T, L, RF_SETUP, MK>;
    case RF_RATIO: return row_fwd_kernel<SGP_T, L, RF_RATIO, MK>;
    case RF_PROJECT: return row_fwd_kernel<SGP_T, L, RF_PROJECT, MK>;
    default: return nullptr;
    }
}
#define SGP_ROW_CASE(LEN) case LEN: return masked ? pick_rowf<LEN, true>(mode) : pick_rowf<LEN, false>(mode);
row_kernel_t<SGP_T> SGP_ROW_FN(int L, int mode, bool masked)
#else
template <int L, bool MK> static row_kernel_t<SGP_T> pick_rowi(int mode)
{
    switch (mode) {
    case RI_PLAIN: return row_inv_kernel<SGP_T, L, RI_PLAIN, MK>;
    case RI_GRAD: return row_inv_kernel<SGP_T, L, RI_GRAD, MK>;
    case RI_LS: return row_inv_kernel<SGP_T, L, RI_LS, MK>;
    case RI_QJ: return row_inv_kernel<SGP_T, L, RI_QJ, MK>;
    case RI_RLUPDATE: return row_inv_kernel<SGP_T, L, RI_RLUPDATE, MK>;
    case RI_LSF: return row_inv_kernel<SGP_T, L, RI_LSF, MK>;
    case RI_QJF: return row_inv_kernel<SGP_T, L, RI_QJF, MK>;
    case RI_RLUPF: return row_inv_kernel<SGP_T, L, RI_RLUPF, MK>;
    default: return nullptr;
    }
}
#define SGP_ROW_CASE(LEN) case LEN: return masked ? pick_rowi<LEN, true>(mode) : pick_rowi<LEN, false>(mode);
row_kernel_t<SGP_T> SGP_ROW_FN(int L, int mode, bool masked)
#endif
{
    switch (L) {
#ifdef SGP_FAST_BUILD      // developer builds (make FAST=1): 256^2 and 2048^2 only
#if SGP_ROW_PART == 0
        SGP_ROW_CASE(128) SGP_ROW_CASE(1024)
#endif
#else
#if SGP_ROW_PART == 0       // the lengths of a translation unit: 0 = powers of two, 1 and 2 = 2^a 5^b
        SGP_ROW_CASE(32) SGP_ROW_CASE(64) SGP_ROW_CASE(128) SGP_ROW_CASE(256) SGP_ROW_CASE(512) SGP_ROW_CASE(1024) SGP_ROW_CASE(2048)
#elif SGP_ROW_PART == 1
        SGP_ROW_CASE(40) SGP_ROW_CASE(80) SGP_ROW_CASE(100) SGP_ROW_CASE(160) SGP_ROW_CASE(200) SGP_ROW_CASE(320) SGP_ROW_CASE(400)
#else
        SGP_ROW_CASE(500) SGP_ROW_CASE(640) SGP_ROW_CASE(800) SGP_ROW_CASE(1000) SGP_ROW_CASE(1280) SGP_ROW_CASE(1600) SGP_ROW_CASE(2000)
#endif
#endif
    default: return nullptr;
    }
}
#undef SGP_ROW_CASE
}  // namespace sgpk

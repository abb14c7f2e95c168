// included by inst_row{f,i}_f32.cu / _f64.cu with SGP_T and SGP_ROW_FWD (1 = forward, 0 = inverse) defined
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
template <> row_kernel_t<SGP_T> get_row_fwd<SGP_T>(int L, int mode, bool masked)
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
    default: return nullptr;
    }
}
#define SGP_ROW_CASE(LEN) case LEN: return masked ? pick_rowi<LEN, true>(mode) : pick_rowi<LEN, false>(mode);
template <> row_kernel_t<SGP_T> get_row_inv<SGP_T>(int L, int mode, bool masked)
#endif
{
    switch (L) {
        SGP_ROW_CASE(32) SGP_ROW_CASE(64) SGP_ROW_CASE(128) SGP_ROW_CASE(160) SGP_ROW_CASE(256) SGP_ROW_CASE(320)
        SGP_ROW_CASE(512) SGP_ROW_CASE(640) SGP_ROW_CASE(1024) SGP_ROW_CASE(2048)
    default: return nullptr;
    }
}
#undef SGP_ROW_CASE
}  // namespace sgpk

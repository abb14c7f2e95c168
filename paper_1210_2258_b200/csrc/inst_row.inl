// included by inst_row_f32.cu / inst_row_f64.cu with SGP_T defined
#include "dispatch.h"
namespace sgpk {
#define SGP_ROW_CASE(LEN) case LEN: return row_fwd_kernel<SGP_T, LEN>;
template <> row_kernel_t<SGP_T> get_row_fwd<SGP_T>(int L)
{
    switch (L) {
        SGP_ROW_CASE(32) SGP_ROW_CASE(64) SGP_ROW_CASE(128) SGP_ROW_CASE(160) SGP_ROW_CASE(256) SGP_ROW_CASE(320)
        SGP_ROW_CASE(512) SGP_ROW_CASE(640) SGP_ROW_CASE(1024) SGP_ROW_CASE(2048)
    default: return nullptr;
    }
}
#undef SGP_ROW_CASE
#define SGP_ROW_CASE(LEN) case LEN: return row_inv_kernel<SGP_T, LEN>;
template <> row_kernel_t<SGP_T> get_row_inv<SGP_T>(int L)
{
    switch (L) {
        SGP_ROW_CASE(32) SGP_ROW_CASE(64) SGP_ROW_CASE(128) SGP_ROW_CASE(160) SGP_ROW_CASE(256) SGP_ROW_CASE(320)
        SGP_ROW_CASE(512) SGP_ROW_CASE(640) SGP_ROW_CASE(1024) SGP_ROW_CASE(2048)
    default: return nullptr;
    }
}
#undef SGP_ROW_CASE
}  // namespace sgpk

#define SGP_T float
#define SGP_ROW_FWD 0
#define SGP_ROW_PART 0
#define SGP_ROW_FN get_rowi_f32_p0
#include "inst_row.inl"

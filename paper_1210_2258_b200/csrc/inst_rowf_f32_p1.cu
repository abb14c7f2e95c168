#define SGP_T float
#define SGP_ROW_FWD 1
#define SGP_ROW_PART 1
#define SGP_ROW_FN get_rowf_f32_p1
#include "inst_row.inl"

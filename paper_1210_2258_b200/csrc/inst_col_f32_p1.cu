#define SGP_T float
#define SGP_COL_PART 1
#define SGP_COL_FN get_col_f32_p1
#define SGP_COL2_FN get_col2_f32
#include "inst_col.inl"

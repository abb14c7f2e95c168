#define SGP_T double
#define SGP_COL_PART 0
#define SGP_COL_FN get_col_f64_p0
#define SGP_COL2_FN get_col2_f64
#include "inst_col.inl"

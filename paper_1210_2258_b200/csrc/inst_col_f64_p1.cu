#define SGP_T double
#define SGP_COL_PART 1
#define SGP_COL_FN get_col_f64_p1
#define SGP_COL2_FN get_col2_f64
#include "inst_col.inl"

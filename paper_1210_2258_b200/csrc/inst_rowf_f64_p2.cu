#define SGP_T double
#define SGP_ROW_FWD 1
#define SGP_ROW_PART 2
#define SGP_ROW_FN get_rowf_f64_p2
#include "inst_row.inl"

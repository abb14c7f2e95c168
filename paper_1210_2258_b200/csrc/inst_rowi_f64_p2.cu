#define SGP_T double
#define SGP_ROW_FWD 0
#define SGP_ROW_PART 2
#define SGP_ROW_FN get_rowi_f64_p2
#include "inst_row.inl"

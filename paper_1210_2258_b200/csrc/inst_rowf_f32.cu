#define SGP_T float
#define SGP_ROW_FWD 1
#include "inst_row.inl"

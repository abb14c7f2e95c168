#define SGP_T float
#define SGP_ROW_FWD 0
#include "inst_row.inl"

#define SGP_T double
#define SGP_ROW_FWD 1
#include "inst_row.inl"

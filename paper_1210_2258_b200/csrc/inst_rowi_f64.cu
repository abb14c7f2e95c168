#define SGP_T double
#define SGP_ROW_FWD 0
#include "inst_row.inl"

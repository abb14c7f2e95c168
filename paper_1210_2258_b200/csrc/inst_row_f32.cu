#define SGP_T float
#include "inst_row.inl"

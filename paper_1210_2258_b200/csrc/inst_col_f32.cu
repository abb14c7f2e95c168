#define SGP_T float
#include "inst_col.inl"

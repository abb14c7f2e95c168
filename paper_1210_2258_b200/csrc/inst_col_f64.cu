#define SGP_T double
#include "inst_col.inl"

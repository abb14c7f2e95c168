#define SGP_T double
#include "inst_row.inl"

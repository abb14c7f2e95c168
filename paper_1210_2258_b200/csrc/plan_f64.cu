#define SGP_T double
#define SGP_MAKE make_plan_f64
#include "plan_impl.inl"
#include "plan_run.inl"

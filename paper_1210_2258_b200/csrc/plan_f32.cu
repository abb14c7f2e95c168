#define SGP_T float
#define SGP_MAKE make_plan_f32
#include "plan_impl.inl"
#include "plan_run.inl"

// kernels.cuh -- the hot-path kernels of the SGP / RL iteration:
// row_fwd.cuh / row_inv.cuh (row FFT passes with the fused elementwise stages), col.cuh (column pass with the
// transfer-function product), aux.cuh (backtracking, final update, set-up kernels).
#pragma once
#include "row_fwd.cuh"
#include "row_inv.cuh"
#include "col.cuh"
#include "aux.cuh"
#include "extra.cuh"

// inst_dispatch.cu -- puts the per-translation-unit kernel tables together (dispatch.h)
#include "dispatch.h"
namespace sgpk {
#define DECL_ROW(NM, T, TN) row_kernel_t<T> get_##NM##_##TN##_p0(int, int, bool); row_kernel_t<T> get_##NM##_##TN##_p1(int, int, bool); row_kernel_t<T> get_##NM##_##TN##_p2(int, int, bool);
DECL_ROW(rowf, float, f32) DECL_ROW(rowi, float, f32) DECL_ROW(rowf, double, f64) DECL_ROW(rowi, double, f64)
#define DECL_COL(T, TN) col_kernel_t<T> get_col_##TN##_p0(int, int, bool, int); col_kernel_t<T> get_col_##TN##_p1(int, int, bool, int); col_kernel_t<T> get_col2_##TN(int, int);
DECL_COL(float, f32) DECL_COL(double, f64)
#define TRY3(A, B, C_) do { if (auto k = A) return k; if (auto k = B) return k; return C_; } while (0)
template <> row_kernel_t<float> get_row_fwd<float>(int L, int m, bool mk) { TRY3(get_rowf_f32_p0(L, m, mk), get_rowf_f32_p1(L, m, mk), get_rowf_f32_p2(L, m, mk)); }
template <> row_kernel_t<float> get_row_inv<float>(int L, int m, bool mk) { TRY3(get_rowi_f32_p0(L, m, mk), get_rowi_f32_p1(L, m, mk), get_rowi_f32_p2(L, m, mk)); }
template <> row_kernel_t<double> get_row_fwd<double>(int L, int m, bool mk) { TRY3(get_rowf_f64_p0(L, m, mk), get_rowf_f64_p1(L, m, mk), get_rowf_f64_p2(L, m, mk)); }
template <> row_kernel_t<double> get_row_inv<double>(int L, int m, bool mk) { TRY3(get_rowi_f64_p0(L, m, mk), get_rowi_f64_p1(L, m, mk), get_rowi_f64_p2(L, m, mk)); }
template <> col_kernel_t<float> get_col<float>(int L, int m, bool mu, int tc) { if (auto k = get_col_f32_p0(L, m, mu, tc)) return k; return get_col_f32_p1(L, m, mu, tc); }
template <> col_kernel_t<double> get_col<double>(int L, int m, bool mu, int tc) { if (auto k = get_col_f64_p0(L, m, mu, tc)) return k; return get_col_f64_p1(L, m, mu, tc); }
template <> col_kernel_t<float> get_col2<float>(int L, int m) { return get_col2_f32(L, m); }
template <> col_kernel_t<double> get_col2<double>(int L, int m) { return get_col2_f64(L, m); }
}  // namespace sgpk

// instantiations of the Cshift / shifted-product kernels; see su3_tables.h
#include "su3_tables.h"
namespace su3tab {
shift_kernel_t shift_kernel(int prec, int op, int W, bool idx32) {
  return idx32 ? shift_pick<int>(prec, op, W) : shift_pick<long long>(prec, op, W);
}
shift_kernel_t cshift_async_kernel(int prec, int W, bool idx32) {
  if (prec == 8) return idx32 ? cshift_async_for_w<double, int>(W) : cshift_async_for_w<double, long long>(W);
  return idx32 ? cshift_async_for_w<float, int>(W) : cshift_async_for_w<float, long long>(W);
}
}  // namespace su3tab

// the pipeline with a shifted operand (su3_mul_shift, su3_cshift); see su3_tables.h
#include "su3_tables.h"
namespace su3tab {
stream_kernel_t shift_pipe_kernel(int prec, int op, int W) {
  return prec == 8 ? shift_pipe_any<double>(op, W) : shift_pipe_any<float>(op, W);
}
stream_kernel_t cshift_bulk_kernel(int prec, int W) { return prec == 8 ? cshift_bulk_for_w<double>(W) : cshift_bulk_for_w<float>(W); }
}  // namespace su3tab

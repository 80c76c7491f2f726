// fp64 instantiations of the streaming kernels (pipeline, direct, warp-staged); see su3_tables.h
#include "su3_tables.h"
namespace su3tab {
stream_kernel_t stream_f64(int family, int op, int W) { return stream_any<double>(family, op, W); }
}  // namespace su3tab

// fp32 instantiations of the menu programs of the pipeline (su3_kernels.cuh: menu_prog); see su3_tables.h
#include "su3_tables.h"
namespace su3tab {
stream_kernel_t menu_f32(int op, int W) { return menu_any<float>(op, W); }
}  // namespace su3tab

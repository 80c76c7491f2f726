// su3_tables.h -- kernel tables of libsu3stream.  The template instantiations are split over several translation
// units (su3_k_*.cu) that are compiled in parallel; su3_api.cu only sees the getters declared at the bottom.
#pragma once
#include "su3_kernels.cuh"

namespace su3tab {

typedef void (*stream_kernel_t)(const su3::StreamParams);
constexpr int NCW = 4;  // consumer warps per CTA of the pipeline kernel (tile <= 128 matrices)

template <typename R, int OP> stream_kernel_t pipe_for_w(int W) {
  switch (W) {
    case 1: return su3::su3_pipe_kernel<R, 1, OP, NCW>;
    case 2: return su3::su3_pipe_kernel<R, 2, OP, NCW>;
    case 4: return su3::su3_pipe_kernel<R, 4, OP, NCW>;
    case 8: return su3::su3_pipe_kernel<R, 8, OP, NCW>;
    case 16: return su3::su3_pipe_kernel<R, 16, OP, NCW>;
    case 32: return su3::su3_pipe_kernel<R, 32, OP, NCW>;
  }
  return nullptr;
}
template <typename R, int OP> stream_kernel_t direct_for_w(int W) {
  switch (W) {
    case 1: return su3::su3_direct_kernel<R, 1, OP>;
    case 2: return su3::su3_direct_kernel<R, 2, OP>;
    case 4: return su3::su3_direct_kernel<R, 4, OP>;
    case 8: return su3::su3_direct_kernel<R, 8, OP>;
    case 16: return su3::su3_direct_kernel<R, 16, OP>;
    case 32: return su3::su3_direct_kernel<R, 32, OP>;
  }
  return nullptr;
}
template <typename R, int OP> stream_kernel_t warp_for_w(int W) {
  switch (W) {
    case 1: return su3::su3_warp_kernel<R, 1, OP>;
    case 2: return su3::su3_warp_kernel<R, 2, OP>;
    case 4: return su3::su3_warp_kernel<R, 4, OP>;
    case 8: return su3::su3_warp_kernel<R, 8, OP>;
    case 16: return su3::su3_warp_kernel<R, 16, OP>;
    case 32: return su3::su3_warp_kernel<R, 32, OP>;
  }
  return nullptr;
}
template <typename R> stream_kernel_t pick_warp(int op, int W) {
  switch (op) {
    case su3::OP_MUL: return warp_for_w<R, su3::OP_MUL>(W);
    case su3::OP_MUL3: return warp_for_w<R, su3::OP_MUL3>(W);
    case su3::OP_MUL_ADD: return warp_for_w<R, su3::OP_MUL_ADD>(W);
    case su3::OP_ADD: return warp_for_w<R, su3::OP_ADD>(1);
  }
  return nullptr;
}
template <typename R> stream_kernel_t pick(int op, int W, bool direct) {
  switch (op) {
    case su3::OP_MUL: return direct ? direct_for_w<R, su3::OP_MUL>(W) : pipe_for_w<R, su3::OP_MUL>(W);
    case su3::OP_MUL3: return direct ? direct_for_w<R, su3::OP_MUL3>(W) : pipe_for_w<R, su3::OP_MUL3>(W);
    case su3::OP_MUL_ADD: return direct ? direct_for_w<R, su3::OP_MUL_ADD>(W) : pipe_for_w<R, su3::OP_MUL_ADD>(W);
    case su3::OP_ADD: return direct ? nullptr : pipe_for_w<R, su3::OP_ADD>(1);  // element-wise: layout-agnostic
  }
  return nullptr;
}

typedef void (*expr_kernel_t)(const su3::ExprParams);
template <typename R> expr_kernel_t expr_for_w(int W) {
  switch (W) {
    case 1: return su3::su3_expr_kernel<R, 1, NCW>;
    case 2: return su3::su3_expr_kernel<R, 2, NCW>;
    case 4: return su3::su3_expr_kernel<R, 4, NCW>;
    case 8: return su3::su3_expr_kernel<R, 8, NCW>;
    case 16: return su3::su3_expr_kernel<R, 16, NCW>;
    case 32: return su3::su3_expr_kernel<R, 32, NCW>;
  }
  return nullptr;
}

typedef void (*shift_kernel_t)(const su3::ShiftParams);
template <typename R, int OP, typename IT> shift_kernel_t shift_for_w(int W) {
  switch (W) {
    case 1: return su3::su3_shift_kernel<R, 1, OP, IT>;
    case 2: return su3::su3_shift_kernel<R, 2, OP, IT>;
    case 4: return su3::su3_shift_kernel<R, 4, OP, IT>;
    case 8: return su3::su3_shift_kernel<R, 8, OP, IT>;
    case 16: return su3::su3_shift_kernel<R, 16, OP, IT>;
    case 32: return su3::su3_shift_kernel<R, 32, OP, IT>;
  }
  return nullptr;
}
template <typename R, typename IT> shift_kernel_t cshift_async_for_w(int W) {
  switch (W) {
    case 1: return su3::su3_cshift_async_kernel<R, 1, IT>;
    case 2: return su3::su3_cshift_async_kernel<R, 2, IT>;
    case 4: return su3::su3_cshift_async_kernel<R, 4, IT>;
    case 8: return su3::su3_cshift_async_kernel<R, 8, IT>;
    case 16: return su3::su3_cshift_async_kernel<R, 16, IT>;
    case 32: return su3::su3_cshift_async_kernel<R, 32, IT>;
  }
  return nullptr;
}
template <typename IT> shift_kernel_t shift_pick(int prec, int op, int W) {
  if (prec == 8) return op == su3::SH_MUL ? shift_for_w<double, su3::SH_MUL, IT>(W) : shift_for_w<double, su3::SH_COPY, IT>(W);
  return op == su3::SH_MUL ? shift_for_w<float, su3::SH_MUL, IT>(W) : shift_for_w<float, su3::SH_COPY, IT>(W);
}

template <typename R> stream_kernel_t matvec_for_w(int W) {
  switch (W) {
    case 1: return su3::su3_matvec_kernel<R, 1, NCW>;
    case 2: return su3::su3_matvec_kernel<R, 2, NCW>;
    case 4: return su3::su3_matvec_kernel<R, 4, NCW>;
    case 8: return su3::su3_matvec_kernel<R, 8, NCW>;
    case 16: return su3::su3_matvec_kernel<R, 16, NCW>;
    case 32: return su3::su3_matvec_kernel<R, 32, NCW>;
  }
  return nullptr;
}


// ---------------------------------------------------------------- getters, one translation unit per precision
enum { FAM_PIPE = 0, FAM_DIRECT = 1, FAM_WARP = 2 };
template <typename R> stream_kernel_t stream_any(int family, int op, int W) {
  if (family == FAM_WARP) return pick_warp<R>(op, W);
  return pick<R>(op, W, family == FAM_DIRECT);
}
stream_kernel_t stream_f64(int family, int op, int W);
stream_kernel_t stream_f32(int family, int op, int W);
stream_kernel_t matvec_kernel(int prec, int W);
expr_kernel_t expr_kernel(int prec, int W);
shift_kernel_t shift_kernel(int prec, int op, int W, bool idx32);        // register version (SH_COPY / SH_MUL)
shift_kernel_t cshift_async_kernel(int prec, int W, bool idx32);
// layout conversion: launches the kernel for (prec, nc, W); returns false if W is not supported
bool launch_convert(int prec, int nc, int W, bool staged, const su3::ConvertParams &p, cudaStream_t s, const char **err);

}  // namespace su3tab

// su3_tables.h -- kernel tables of libsu3stream.  The template instantiations are split over several translation
// units (su3_k_*.cu) that are compiled in parallel; su3_api.cu only sees the getters declared at the bottom.
#pragma once
#include "su3_kernels.cuh"

namespace su3tab {

typedef void (*stream_kernel_t)(const su3::StreamParams);
constexpr int NCW = 4;  // consumer warps per CTA of the pipeline kernel (tile <= 128 matrices)

template <typename R, int OP, int SHIFT = 0> stream_kernel_t pipe_for_w(int W) {
  switch (W) {
    case 1: return su3::su3_pipe_kernel<R, 1, OP, NCW, SHIFT>;
    case 2: return su3::su3_pipe_kernel<R, 2, OP, NCW, SHIFT>;
    case 4: return su3::su3_pipe_kernel<R, 4, OP, NCW, SHIFT>;
    case 8: return su3::su3_pipe_kernel<R, 8, OP, NCW, SHIFT>;
    case 16: return su3::su3_pipe_kernel<R, 16, OP, NCW, SHIFT>;
    case 32: return su3::su3_pipe_kernel<R, 32, OP, NCW, SHIFT>;
  }
  return nullptr;
}
// the menu programs beyond su3_mul / mul3 / mul_add / add (su3_kernels.cuh: menu_prog): element-wise rows are layout-
// agnostic and exist for W = 1 only
template <typename R> stream_kernel_t menu_any(int op, int W) {
  switch (op) {
    case su3::OP_SUM_PROD: return pipe_for_w<R, su3::OP_SUM_PROD>(W);
    case su3::OP_MUL_MUL_ADD: return pipe_for_w<R, su3::OP_MUL_MUL_ADD>(W);
    case su3::OP_MUL_MUL_SUB: return pipe_for_w<R, su3::OP_MUL_MUL_SUB>(W);
    case su3::OP_MUL_SUB: return pipe_for_w<R, su3::OP_MUL_SUB>(W);
    case su3::OP_MUL4: return pipe_for_w<R, su3::OP_MUL4>(W);
    case su3::OP_MUL_R: return pipe_for_w<R, su3::OP_MUL_R>(W);
    case su3::OP_MULMUL_MUL: return pipe_for_w<R, su3::OP_MULMUL_MUL>(W);
    case su3::OP_ADD3: return su3::su3_pipe_kernel<R, 1, su3::OP_ADD3, NCW, 0>;
    case su3::OP_ADD4: return su3::su3_pipe_kernel<R, 1, su3::OP_ADD4, NCW, 0>;
    case su3::OP_SUB: return su3::su3_pipe_kernel<R, 1, su3::OP_SUB, NCW, 0>;
    case su3::OP_EMUL: return su3::su3_pipe_kernel<R, 1, su3::OP_EMUL, NCW, 0>;
    case su3::OP_SUM_EPROD: return su3::su3_pipe_kernel<R, 1, su3::OP_SUM_EPROD, NCW, 0>;
  }
  return nullptr;
}
inline bool menu_elementwise(int op) {
  return op == su3::OP_ADD || op == su3::OP_ADD3 || op == su3::OP_ADD4 || op == su3::OP_SUB || op == su3::OP_EMUL ||
         op == su3::OP_SUM_EPROD;
}
template <typename R> stream_kernel_t cshift_bulk_for_w(int W) {
  switch (W) {
    case 1: return su3::su3_cshift_bulk_kernel<R, 1>;
    case 2: return su3::su3_cshift_bulk_kernel<R, 2>;
    case 4: return su3::su3_cshift_bulk_kernel<R, 4>;
    case 8: return su3::su3_cshift_bulk_kernel<R, 8>;
    case 16: return su3::su3_cshift_bulk_kernel<R, 16>;
    case 32: return su3::su3_cshift_bulk_kernel<R, 32>;
  }
  return nullptr;
}
// the pipeline with a shifted last operand: z = x . y(+disp) (OP_MUL) and z = y(+disp) (OP_COPY, Cshift)
template <typename R> stream_kernel_t shift_pipe_any(int op, int W) {
  return op == su3::OP_MUL ? pipe_for_w<R, su3::OP_MUL, 1>(W) : pipe_for_w<R, su3::OP_COPY, 1>(W);
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
    case 1: return su3::su3_expr_kernel<R, 1>;
    case 2: return su3::su3_expr_kernel<R, 2>;
    case 4: return su3::su3_expr_kernel<R, 4>;
    case 8: return su3::su3_expr_kernel<R, 8>;
    case 16: return su3::su3_expr_kernel<R, 16>;
    case 32: return su3::su3_expr_kernel<R, 32>;
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
stream_kernel_t menu_f64(int op, int W);
stream_kernel_t menu_f32(int op, int W);
stream_kernel_t shift_pipe_kernel(int prec, int op, int W);
stream_kernel_t cshift_bulk_kernel(int prec, int W);
stream_kernel_t matvec_kernel(int prec, int W);
expr_kernel_t expr_kernel(int prec, int W);
shift_kernel_t shift_kernel(int prec, int op, int W, bool idx32);        // register version (SH_COPY / SH_MUL)
shift_kernel_t cshift_async_kernel(int prec, int W, bool idx32);
// layout conversion: launches the kernel for (prec, nc, W); returns false if W is not supported
bool launch_convert(int prec, int nc, int W, bool staged, const su3::ConvertParams &p, cudaStream_t s, const char **err);
// the TMA variant: complex numbers per tile, and the launch (p.pitch and p.run_recs must be set)
int convert_tma_tile(int prec);
bool launch_convert_tma(int prec, int nc, int W, const su3::ConvertParams &p, cudaStream_t s, const char **err);
// face of a slab: pack / unpack / field-to-field copy of planes (nc = 9 or 3)
void launch_face(int prec, int nc, bool idx32, unsigned grid, const su3::FaceParams &p, cudaStream_t s);

}  // namespace su3tab

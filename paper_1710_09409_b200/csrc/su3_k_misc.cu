// instantiations of the expression, matvec and layout-conversion kernels; see su3_tables.h
#include "su3_tables.h"
namespace su3tab {
expr_kernel_t expr_kernel(int prec, int W) { return prec == 8 ? expr_for_w<double>(W) : expr_for_w<float>(W); }
stream_kernel_t matvec_kernel(int prec, int W) { return prec == 8 ? matvec_for_w<double>(W) : matvec_for_w<float>(W); }

// TMA convert: N complex numbers per tile (18 KB), 128 threads, 8 blocks per SM by registers
template <typename C2, int NC, int N> bool convert_tma_w(int W, const su3::ConvertParams &p, cudaStream_t s, const char **err) {
  constexpr int NT = 128;
  const long long tr = N / (NC * W);
  const long long blocks = (p.nrec + tr - 1) / tr;
  if (blocks > 0x7fffffffLL) { *err = "lattice too large for one launch"; return false; }
  const size_t span = (size_t)W * p.pitch > (size_t)N ? (size_t)W * p.pitch : (size_t)N;
  const size_t smem = span * sizeof(C2) + 16;
  switch (W) {
#define SU3_TMA_CASE(WW) case WW: su3::su3_convert_tma_kernel<C2, WW, NC, N, NT><<<(unsigned)blocks, NT, smem, s>>>(p); return true;
    SU3_TMA_CASE(2) SU3_TMA_CASE(4) SU3_TMA_CASE(8) SU3_TMA_CASE(16) SU3_TMA_CASE(32)
#undef SU3_TMA_CASE
  }
  *err = "unsupported W";
  return false;
}
template <typename IT> void launch_face_it(int prec, int nc, unsigned grid, const su3::FaceParams &p, cudaStream_t s) {
  if (prec == 8 && nc == 9) su3::su3_face_kernel<double2, 9, IT><<<grid, 256, 0, s>>>(p);
  else if (prec == 8) su3::su3_face_kernel<double2, 3, IT><<<grid, 256, 0, s>>>(p);
  else if (nc == 9) su3::su3_face_kernel<float2, 9, IT><<<grid, 256, 0, s>>>(p);
  else su3::su3_face_kernel<float2, 3, IT><<<grid, 256, 0, s>>>(p);
}
void launch_face(int prec, int nc, bool idx32, unsigned grid, const su3::FaceParams &p, cudaStream_t s) {
  if (idx32) launch_face_it<int>(prec, nc, grid, p, s);
  else launch_face_it<long long>(prec, nc, grid, p, s);
}

int convert_tma_tile(int prec) { return prec == 8 ? 1152 : 2304; }
bool launch_convert_tma(int prec, int nc, int W, const su3::ConvertParams &p, cudaStream_t s, const char **err) {
  if (prec == 8) return nc == 9 ? convert_tma_w<double2, 9, 1152>(W, p, s, err) : convert_tma_w<double2, 3, 1152>(W, p, s, err);
  return nc == 9 ? convert_tma_w<float2, 9, 2304>(W, p, s, err) : convert_tma_w<float2, 3, 2304>(W, p, s, err);
}

bool launch_convert(int prec, int nc, int W, bool staged, const su3::ConvertParams &p, cudaStream_t s, const char **err) {
  if (staged) {
#define SU3_STAGED(WW, TRR)                                                                                  \
  case WW: {                                                                                                 \
    const long long blocks = (p.nrec + TRR - 1) / TRR;                                                       \
    if (blocks > 0x7fffffffLL) { *err = "lattice too large for one launch"; return false; }                  \
    const size_t smem = sizeof(float2) * TRR * nc * (WW + 1) + sizeof(long long) * TRR;                      \
    if (prec == 8) {                                                                                         \
      constexpr int TRD = TRR / 2 > 0 ? TRR / 2 : 1;                                                         \
      const long long blocksd = (p.nrec + TRD - 1) / TRD;                                                    \
      const size_t smemd = sizeof(double2) * TRD * nc * (WW + 1) + sizeof(long long) * TRD;                  \
      if (nc == 9) su3::su3_convert_staged_kernel<double2, WW, TRD, 9><<<(unsigned)blocksd, 256, smemd, s>>>(p); \
      else su3::su3_convert_staged_kernel<double2, WW, TRD, 3><<<(unsigned)blocksd, 256, smemd, s>>>(p);     \
    } else if (nc == 9) su3::su3_convert_staged_kernel<float2, WW, TRR, 9><<<(unsigned)blocks, 256, smem, s>>>(p);  \
    else su3::su3_convert_staged_kernel<float2, WW, TRR, 3><<<(unsigned)blocks, 256, smem, s>>>(p);          \
  } return true;
    switch (W) {
      SU3_STAGED(1, 256) SU3_STAGED(2, 128) SU3_STAGED(4, 64) SU3_STAGED(8, 32) SU3_STAGED(16, 16) SU3_STAGED(32, 8)  // 18 KB tiles
    }
#undef SU3_STAGED
    *err = "unsupported W";
    return false;
  }
  constexpr int TR = 64;
  const long long blocks = (p.nrec + TR - 1) / TR;
  if (blocks > 0x7fffffffLL) { *err = "lattice too large for one launch"; return false; }
  const unsigned grid = (unsigned)blocks;
#define SU3_CONVERT_CASE(WW)                                                                           \
  case WW:                                                                                             \
    if (prec == 8 && nc == 9) su3::su3_convert_kernel<double2, WW, TR, 9><<<grid, 256, 0, s>>>(p);     \
    else if (prec == 8) su3::su3_convert_kernel<double2, WW, TR, 3><<<grid, 256, 0, s>>>(p);           \
    else if (nc == 9) su3::su3_convert_kernel<float2, WW, TR, 9><<<grid, 256, 0, s>>>(p);              \
    else su3::su3_convert_kernel<float2, WW, TR, 3><<<grid, 256, 0, s>>>(p);                           \
    return true;
  switch (W) {
    SU3_CONVERT_CASE(1) SU3_CONVERT_CASE(2) SU3_CONVERT_CASE(4) SU3_CONVERT_CASE(8) SU3_CONVERT_CASE(16) SU3_CONVERT_CASE(32)
  }
#undef SU3_CONVERT_CASE
  *err = "unsupported W";
  return false;
}
}  // namespace su3tab

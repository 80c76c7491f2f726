// su3_api.cu -- the C ABI of libsu3stream (include/su3stream.h): descriptor validation,
// field handles, kernel selection and launch.  Host logic only; the arithmetic lives in
// su3_kernels.cuh.  No CPU fallback: without a CUDA device every arithmetic call fails
// with SU3_ERR_CUDA.
#include "../../include/su3stream.h"

#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <initializer_list>
#include <map>
#include <memory>
#include <utility>
#include <mutex>
#include <new>
#include <vector>

#include "su3_tables.h"

struct su3_field {
  su3_desc d;  // normalised
  void *ptr;
  size_t nbytes;
  int64_t volume;
  int64_t nmat;
  int ncomp;   // complex numbers per (site, mu): 9 = colour matrix, 3 = colour vector; 0 = real scalar field (1 real)
  int device;  // ordinal of the device that owns ptr, -1 if the runtime could not tell at wrap time
};

namespace {

using su3tab::NCW;
using su3tab::expr_kernel_t;
using su3tab::shift_kernel_t;
using su3tab::stream_kernel_t;

thread_local char g_err[512] = "";
std::atomic<int64_t> g_launches{0};
// launch knobs of the CALLING THREAD (su3_tune_set): no process-wide state, so threads never race on them
thread_local su3_tune g_tune = {0, 0, 0, 0, 0, 0, {0, 0}};

su3_status fail(su3_status st, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return st;
}

void default_simd(int W, int32_t simd[4]) {  // reading S4
  for (int d = 0; d < 4; d++) simd[d] = 1;
  for (int d = 3; W > 1; W >>= 1, d = (d + 3) & 3) simd[d] *= 2;
}

su3_status normalize(const su3_desc *in, su3_desc *out) {
  if (!in || !out) return fail(SU3_ERR_NULL, "descriptor pointer is NULL");
  su3_desc d = *in;
  for (int k = 0; k < 4; k++)
    if (d.L[k] <= 0) return fail(SU3_ERR_INVALID, "L[%d] = %d must be positive", k, d.L[k]);
  if (d.n_lorentz != 1 && d.n_lorentz != 4) return fail(SU3_ERR_INVALID, "n_lorentz = %d not in {1,4}", d.n_lorentz);
  if (d.prec != SU3_F32 && d.prec != SU3_F64) return fail(SU3_ERR_INVALID, "prec = %d not in {4,8}", d.prec);
  if (d.layout != SU3_SCALAR && d.layout != SU3_VECTOR) return fail(SU3_ERR_INVALID, "layout = %d not in {0,1}", d.layout);
  if (d.W < 1 || d.W > 32 || (d.W & (d.W - 1))) return fail(SU3_ERR_INVALID, "W = %d is not a power of two in 1..32", d.W);
  if (d.layout == SU3_SCALAR && d.W != 1) return fail(SU3_ERR_INVALID, "W = %d must be 1 for the scalar layout", d.W);
  bool any = false;
  for (int k = 0; k < 4; k++) any = any || d.simd[k] != 0;
  if (any) {
    long prod = 1;
    for (int k = 0; k < 4; k++) {
      if (d.simd[k] <= 0) return fail(SU3_ERR_INVALID, "simd[%d] = %d must be positive", k, d.simd[k]);
      prod *= d.simd[k];
    }
    if (prod != d.W) return fail(SU3_ERR_INVALID, "prod(simd) = %ld differs from W = %d", prod, d.W);
  } else {
    default_simd(d.W, d.simd);
  }
  for (int k = 0; k < 4; k++)
    if (d.L[k] % d.simd[k]) return fail(SU3_ERR_INVALID, "L[%d] = %d not divisible by simd[%d] = %d", k, d.L[k], k, d.simd[k]);
  *out = d;
  return SU3_OK;
}

int64_t volume_of(const su3_desc &d) { return (int64_t)d.L[0] * d.L[1] * d.L[2] * d.L[3]; }

bool same_lattice(const su3_desc &a, const su3_desc &b) {
  return !memcmp(a.L, b.L, sizeof a.L) && a.n_lorentz == b.n_lorentz && a.prec == b.prec;
}
bool same_desc(const su3_desc &a, const su3_desc &b) {
  return same_lattice(a, b) && a.layout == b.layout && a.W == b.W && !memcmp(a.simd, b.simd, sizeof a.simd);
}

// ---------------------------------------------------------------- device facts (cached per device ordinal)
constexpr int MAX_DEVICES = 64;
struct DevInfo {
  bool ok = false;
  int dev = -1, sms = 0, smem_optin = 0, mem_khz = 0, bus_bits = 0;
  long long l2 = 0;
  char name[256] = "";
  char err[256] = "";
};
// Facts of the device that is CURRENT on the calling thread, looked up per call (cudaGetDevice is a thread-local read)
// and cached per ordinal, so one process may drive several GPUs.  A failed query is not cached.
const DevInfo &devinfo() {
  static DevInfo table[MAX_DEVICES];
  static std::mutex mu;
  thread_local DevInfo bad;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess && (dev < 0 || dev >= MAX_DEVICES)) e = cudaErrorInvalidDevice;
  if (e == cudaSuccess) {
    std::lock_guard<std::mutex> lk(mu);
    DevInfo &di = table[dev];
    if (di.ok) return di;
    cudaDeviceProp pr;
    e = cudaGetDeviceProperties(&pr, dev);
    if (e == cudaSuccess) {
      di.dev = dev;
      di.sms = pr.multiProcessorCount;
      di.smem_optin = (int)pr.sharedMemPerBlockOptin;
      di.l2 = pr.l2CacheSize;
      snprintf(di.name, sizeof di.name, "%s", pr.name);
      int v = 0;
      if (cudaDeviceGetAttribute(&v, cudaDevAttrMemoryClockRate, dev) == cudaSuccess) di.mem_khz = v;
      if (cudaDeviceGetAttribute(&v, cudaDevAttrGlobalMemoryBusWidth, dev) == cudaSuccess) di.bus_bits = v;
      di.ok = true;
      return di;
    }
  }
  bad = DevInfo();
  snprintf(bad.err, sizeof bad.err, "no usable CUDA device: %s", cudaGetErrorString(e));
  (void)cudaGetLastError();
  return bad;
}

// ---------------------------------------------------------------- kernel tables
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is a per-DEVICE setting: once per (device, kernel), not per launch
cudaError_t allow_max_smem(const void *fn, int bytes) {
  static std::mutex mu;
  static std::vector<std::pair<int, const void *>> done;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lk(mu);
  for (const auto &d : done)
    if (d.first == dev && d.second == fn) return cudaSuccess;
  e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess) done.push_back({dev, fn});
  return e;
}

su3_status cuda_fail(const char *what, cudaError_t e) {
  return fail(SU3_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

// Every field of a call must live on the device that is current on the calling thread (the launch goes there).
su3_status on_current_device(std::initializer_list<const su3_field *> fs) {
  const DevInfo &di = devinfo();
  if (!di.ok) return fail(SU3_ERR_CUDA, "%s", di.err);
  for (const su3_field *f : fs)
    if (f && f->device >= 0 && f->device != di.dev)
      return fail(SU3_ERR_MISMATCH, "field memory is on device %d but device %d is current on this thread (cudaSetDevice first)",
                  f->device, di.dev);
  return SU3_OK;
}

// What launch_stream will launch for (op, prec, W, nmat, footprint) with the knobs `tn` on the device `di`: kernel
// family, geometry, ring depth and L2 policy.  Host arithmetic only, so that su3_launch_plan can report exactly the
// choice the arithmetic calls make.
struct StreamPlan {
  int family = 0;         // su3tab::FAM_PIPE / FAM_DIRECT / FAM_WARP
  unsigned grid = 0;
  int block = 0;
  size_t smem = 0;
  int tile_mats = 0, stages = 0, ctas = 0;
  int hint = 0;           // StreamParams::hint: 0 none, 1 evict_first, 2 pinned prefix (evict_last) + streamed rest
  int64_t pin_tiles = 0;
  size_t pin_bytes = 0;   // per operand
};

// shifted: the last operand is read at the shifted site (pipeline only).  one_shot: the operands were just written
// and no repeat of this call on the same pointers is expected (the chunk launches of su3_eval_host, whose data has
// just arrived from the host and is never re-read): the automatic pinned-prefix L2 policy, which pays only when the
// same call is repeated back to back (Listing 3's loop), is then not applied.  Shifted launches do not get it
// automatically either.  l2_hint = 3 still asks for it explicitly in every case.
su3_status plan_stream(int op, int prec, int W, int64_t nmat, size_t footprint_bytes, bool shifted, bool one_shot,
                       const su3_tune &tn, const DevInfo &di, StreamPlan *pl) {
  const int nin = su3::menu_prog(op).nin;
  const int nslot = (shifted && nin == 1) ? 2 : nin;
  const int cb = 2 * prec;
  const bool base_op = op <= su3::OP_ADD && !shifted;  // the direct and warp-staged kernels exist for su3_mul/mul3/mul_add(/add) only
  // auto path: the TMA pipeline everywhere, except L2-resident problems in a vector layout whose element
  // vectors fill whole sectors (W*c >= 32 B): there the per-lane loads are already sector-perfect and the
  // pipeline's fixed latency (barrier set-up, two smem hops) is what one measures
  // Up to 0.6 x L2 (everything stays resident from call to call) the direct kernel wins by 8-40 %; between 0.6 and 2 x L2
  // the pipeline with its pinned operand prefixes (below) is 6-18 % faster than the direct kernel, which has no L2 policy
  // (measured at 24^4 fp64 W=4: 7668 vs 7226 GB/s; 28^4 fp32 W=8: 7974 vs 7187).
  const bool direct = base_op && op != su3::OP_ADD &&  // OP_ADD has no direct kernel (su3_add's path = 2 is its own plain kernel)
                      (tn.path == 2 || (tn.path == 0 && W * cb >= 32 && footprint_bytes <= (size_t)di.l2 * 6 / 10));
  const bool warp = base_op && !direct && (tn.path == 3 || (tn.path == 0 && footprint_bytes <= (size_t)di.l2 / 2));
  pl->family = warp ? su3tab::FAM_WARP : (direct ? su3tab::FAM_DIRECT : su3tab::FAM_PIPE);
  if (warp) {
    pl->tile_mats = 32;
    const int64_t nwt = (nmat + 31) / 32;
    int wpb = 4;  // warps per block; fewer on small lattices so that every SM gets a block
    while (wpb > 1 && (nwt + wpb - 1) / wpb < 2 * (int64_t)di.sms) wpb >>= 1;
    pl->smem = (size_t)wpb * nin * 288 * cb;
    const int64_t blocks_needed = (nwt + wpb - 1) / wpb;
    const int64_t cap = (int64_t)di.sms * (tn.ctas_per_sm > 0 ? tn.ctas_per_sm : 8) * (4 / wpb);
    pl->grid = (unsigned)(blocks_needed < cap ? blocks_needed : cap);
    pl->block = wpb * 32;
    return SU3_OK;
  }
  if (direct) {
    int bs = 256;  // small lattices: smaller blocks so that every SM gets one
    while (bs > 32 && (nmat + bs - 1) / bs < 2 * (int64_t)di.sms) bs >>= 1;
    const int64_t blocks_needed = (nmat + bs - 1) / bs;
    const int64_t cap = (int64_t)di.sms * 8 * (tn.ctas_per_sm > 0 ? tn.ctas_per_sm : 1) * (256 / bs);
    pl->grid = (unsigned)(blocks_needed < cap ? blocks_needed : cap);
    pl->block = bs;
    return SU3_OK;
  }
  // defaults measured on B200: 9 KB operand slots (64 fp64 / 128 fp32 matrices),
  // a 3-deep ring, 2 persistent CTAs per SM
  // 2 persistent CTAs per SM; 3 for the copy through a shifted slot (Cshift of 72-byte records with odd run boundaries:
  // no arithmetic to hide behind, measured 0.81 -> 0.96 x copy)
  int ctas = tn.ctas_per_sm > 0 ? tn.ctas_per_sm : (shifted && nin == 1 ? 3 : 2);
  int tm = tn.tile_mats;
  if (tm == 0) {
    tm = 9216 / (9 * cb);
    // small lattices: shrink the tile until every persistent CTA has at least two tiles
    while (tm > 32 && (nmat + tm - 1) / tm < 2 * (int64_t)di.sms * ctas) tm >>= 1;
  }
  if (tm != 32 && tm != 64 && tm != 128) return fail(SU3_ERR_INVALID, "tile_mats = %d not in {32,64,128}", tm);
  const size_t stage_bytes = (size_t)nslot * tm * 9 * cb + (shifted ? 16 : 0);
  // 1 KB of every CTA's shared memory is reserved by the system; keep 256 B for the barriers
  size_t budget = ((size_t)di.smem_optin + 1024) / ctas - 1024;
  // auto CTAs/SM: a big tile may leave room for fewer resident CTAs than the default
  while (tn.ctas_per_sm == 0 && ctas > 1 && (budget - 256) / stage_bytes < 2) {
    ctas--;
    budget = ((size_t)di.smem_optin + 1024) / ctas - 1024;
  }
  const int64_t max_grid = (int64_t)di.sms * ctas;
  int stages = tn.stages;
  if (stages == 0) {
    // ring depth 3 at HBM-bound sizes (deeper rings open more DRAM pages at once and measured 1-3 % slower from 40^4
    // fp32 / 36^4 fp64 on); up to 3 x L2 a good part of the loads hits L2, latency rather than DRAM limits a 20-70 us
    // launch, and more bytes in flight pay: depth 4 measured +4..12 % at 20^4-28^4 fp64 and 24^4-36^4 fp32 (ncu at
    // 24^4 with depth 3, warm: DRAM 44 % busy, profiles/r02_knee.md)
    stages = footprint_bytes <= (size_t)di.l2 * 3 ? 4 : 3;
    while (stages > 2 && stages * stage_bytes + 256 > budget) stages--;
  }
  if (stages < 2 || stages > 16) return fail(SU3_ERR_INVALID, "stages = %d outside 2..16 (tile %d, %d CTAs/SM)", stages, tm, ctas);
  pl->smem = stages * stage_bytes + 3 * stages * sizeof(uint64_t);
  if (pl->smem > (size_t)di.smem_optin) return fail(SU3_ERR_INVALID, "pipeline needs %zu B of shared memory, device allows %d", pl->smem, di.smem_optin);
  pl->tile_mats = tm; pl->stages = stages; pl->ctas = ctas;
  // L2 policy (l2_hint): 0/1 none (evict_first measured neutral at every HBM-bound size), 2 evict_first
  // everywhere, 3 keep the first l2_pin_mb MB of every operand in L2 (evict_last) and stream the rest (evict_first)
  pl->hint = tn.l2_hint == 2 ? 1 : (tn.l2_hint == 3 ? 2 : 0);
  pl->pin_bytes = (size_t)tn.l2_pin_mb * 1000000;   // per operand
  if (tn.l2_hint == 0 && !one_shot && !shifted && footprint_bytes > (size_t)di.l2 * 6 / 10 && footprint_bytes <= (size_t)di.l2 * 2) {
    // auto, footprint between 0.6 and 2 x L2 ("straddling"): a plain LRU keeps NOTHING of a cyclic sweep that is a
    // little larger than the cache; keeping ~36 % of L2 worth of operand prefixes resident from one call to the next
    // (Listing 3 repeats z = x*y on the same fields) and streaming the rest measured +32 % at 24^4 fp64, +7 % at
    // 32^4 fp32; beyond 2 x L2 the same policy costs 2-4 %, so it is not applied there.  It helps only a call that is
    // repeated on the same pointers: not applied to one-shot chunk launches and to shifted launches (see above)
    pl->hint = 2;
    pl->pin_bytes = (size_t)di.l2 * 36 / 100 / nin;
  }
  if (pl->hint == 2) pl->pin_tiles = (int64_t)(pl->pin_bytes / ((size_t)tm * 9 * cb));
  else pl->pin_bytes = 0;
  const int64_t ntiles = (nmat + tm - 1) / tm;
  pl->grid = (unsigned)(ntiles < max_grid ? ntiles : max_grid);
  pl->block = (NCW + 1) * 32;
  return SU3_OK;
}

// Launch one ahead-of-time program (su3_kernels.cuh: menu_prog(op)) over `nmat` matrices starting at the given
// pointers; `sh` != NULL: the last operand is read at the shifted site (pipeline only).
su3_status launch_stream(int op, int prec, int W, void *z, const void *const *in, int64_t nmat,
                         size_t footprint_bytes, cudaStream_t stream, const su3::ShiftInfo *sh = nullptr, bool one_shot = false) {
  const DevInfo &di = devinfo();
  if (!di.ok) return fail(SU3_ERR_CUDA, "%s", di.err);
  if (nmat == 0) return SU3_OK;
  StreamPlan pl;
  if (su3_status st = plan_stream(op, prec, W, nmat, footprint_bytes, sh != nullptr, one_shot, g_tune, di, &pl)) return st;
  const int nin = su3::menu_prog(op).nin;
  stream_kernel_t k = nullptr;
  if (sh) k = su3tab::shift_pipe_kernel(prec, op, W);
  else if (op <= su3::OP_ADD) k = prec == SU3_F64 ? su3tab::stream_f64(pl.family, op, W) : su3tab::stream_f32(pl.family, op, W);
  else k = prec == SU3_F64 ? su3tab::menu_f64(op, W) : su3tab::menu_f32(op, W);
  if (!k) return fail(SU3_ERR_INVALID, "no kernel for op %d prec %d W %d", op, prec, W);

  su3::StreamParams p;
  memset(&p, 0, sizeof p);
  p.z = z; p.x = in[0]; p.y = nin > 1 ? in[1] : nullptr; p.u = nin > 2 ? in[2] : nullptr; p.v = nin > 3 ? in[3] : nullptr;
  p.nmat = nmat;
  if (sh) p.sh = *sh;
  p.tile_mats = pl.tile_mats; p.stages = pl.stages; p.hint = pl.hint; p.pin_tiles = pl.pin_tiles;
  if (pl.family != su3tab::FAM_DIRECT) {
    cudaError_t e = allow_max_smem((const void *)k, di.smem_optin);
    if (e != cudaSuccess) return cuda_fail("cudaFuncSetAttribute", e);
  }
  k<<<pl.grid, pl.block, pl.smem, stream>>>(p);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("kernel launch", e);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SU3_OK;
}

su3_status check_arith(const su3_field *z, const su3_field *x, const su3_field *y, const su3_field *u, bool has_u) {
  if (!z || !x || !y || (has_u && !u)) return fail(SU3_ERR_NULL, "field handle is NULL");
  if (z->ncomp != 9 || x->ncomp != 9 || y->ncomp != 9 || (has_u && u->ncomp != 9))
    return fail(SU3_ERR_MISMATCH, "this call takes colour-matrix fields, not colour-vector fields");
  if (!same_desc(z->d, x->d) || !same_desc(z->d, y->d) || (has_u && !same_desc(z->d, u->d)))
    return fail(SU3_ERR_MISMATCH, "operand descriptors differ (L, n_lorentz, prec, layout, W, simd must all agree)");
  return SU3_OK;
}

su3_status arith(int op, su3_field *z, const su3_field *x, const su3_field *y, const su3_field *u, void *stream) {
  su3_status st = check_arith(z, x, y, u, op != su3::OP_MUL);
  if (st != SU3_OK) return st;
  if ((st = on_current_device({z, x, y, u})) != SU3_OK) return st;
  const size_t fp = z->nbytes * (op == su3::OP_MUL ? 3 : 4);
  const void *in[4] = {x->ptr, y->ptr, u ? u->ptr : nullptr, nullptr};
  return launch_stream(op, z->d.prec, z->d.W, z->ptr, in, z->nmat, fp, (cudaStream_t)stream);
}

unsigned flat_grid(size_t n_items, size_t per_block, int blocks_per_sm) {
  const DevInfo &di = devinfo();
  size_t need = (n_items + per_block - 1) / per_block;
  size_t cap = (size_t)di.sms * blocks_per_sm;
  if (need < 1) need = 1;
  return (unsigned)(need < cap ? need : cap);
}

// ---------------------------------------------------------------- su3_expr: postfix -> register machine
struct ExprProgram {
  su3::ExprIns ins[16];
  int nins = 0, ntemp = 0, nmul = 0, naddsub = 0;
};

// Simulates the evaluation stack.  A stack entry is an operand slot (0..7), a temporary (8..15) or the
// accumulator (255); at most one entry lives in the accumulator: it is spilled to a temporary when a new
// result is produced while it is still needed.
su3_status compile_expr(const char *prog, int nops, ExprProgram *out) {
  if (!prog) return fail(SU3_ERR_NULL, "program is NULL");
  if (nops < 1 || nops > 8) return fail(SU3_ERR_INVALID, "n_operands = %d outside 1..8", nops);
  const size_t len = strlen(prog);
  if (len == 0 || len > 32) return fail(SU3_ERR_INVALID, "program has %zu tokens (1..32 allowed)", len);
  unsigned char stack[8];
  int sp = 0;
  bool used[8] = {false}, temp_busy[8] = {false};
  ExprProgram pr;
  for (size_t i = 0; i < len; i++) {
    const char t = prog[i];
    if (t >= '0' && t <= '7') {
      if (t - '0' >= nops) return fail(SU3_ERR_INVALID, "token %zu: operand %c but n_operands = %d", i, t, nops);
      if (sp == 8) return fail(SU3_ERR_INVALID, "token %zu: stack deeper than 8", i);
      used[t - '0'] = true;
      stack[sp++] = (unsigned char)(t - '0');
    } else if (t == '+' || t == '-' || t == '*') {
      if (sp < 2) return fail(SU3_ERR_INVALID, "token %zu: operator '%c' needs two values", i, t);
      if (pr.nins == 16) return fail(SU3_ERR_INVALID, "more than 16 operators");
      const unsigned char b = stack[--sp], a = stack[--sp];
      su3::ExprIns in;
      in.op = t == '*' ? su3::EX_MUL : (t == '+' ? su3::EX_ADD : su3::EX_SUB);
      in.a = a; in.b = b; in.spill = su3::EX_NONE;
      for (int k = 0; k < sp; k++)
        if (stack[k] == su3::EX_SRC_ACC) {  // an older result is still needed: park it in a temporary
          int tmp = 0;
          while (tmp < 8 && temp_busy[tmp]) tmp++;
          if (tmp == 8) return fail(SU3_ERR_INVALID, "expression needs more than 8 temporaries");
          temp_busy[tmp] = true;
          if (tmp + 1 > pr.ntemp) pr.ntemp = tmp + 1;
          in.spill = (unsigned char)(su3::EX_TEMP0 + tmp);
          stack[k] = in.spill;
        }
      if (a >= su3::EX_TEMP0 && a != su3::EX_SRC_ACC) temp_busy[a - su3::EX_TEMP0] = false;
      if (b >= su3::EX_TEMP0 && b != su3::EX_SRC_ACC) temp_busy[b - su3::EX_TEMP0] = false;
      (t == '*' ? pr.nmul : pr.naddsub)++;
      pr.ins[pr.nins++] = in;
      stack[sp++] = su3::EX_SRC_ACC;
    } else {
      return fail(SU3_ERR_INVALID, "token %zu: '%c' is not a digit 0..7 or one of + - *", i, t);
    }
  }
  if (sp != 1) return fail(SU3_ERR_INVALID, "program leaves %d values on the stack (must be 1)", sp);
  for (int k = 0; k < nops; k++)
    if (!used[k]) return fail(SU3_ERR_INVALID, "operand %d is never used", k);
  if (stack[0] != su3::EX_SRC_ACC) {  // the program is a bare operand: z = operand
    su3::ExprIns in;
    in.op = su3::EX_COPY; in.a = stack[0]; in.b = su3::EX_NONE; in.spill = su3::EX_NONE;
    pr.ins[pr.nins++] = in;
  }
  *out = pr;
  return SU3_OK;
}

// Does the compiled program equal row `op` of the ahead-of-time menu, up to a renaming of the operands and the order
// of the two sources of a commutative element-wise instruction?  map[k] = user operand held by menu slot k.
bool match_menu_from(const ExprProgram &pr, const su3::MenuProg &mp, int i, int map[4]) {
  if (i == pr.nins) return true;
  const su3::ExprIns u = pr.ins[i], m = mp.ins[i];
  if (u.op != m.op || u.spill != m.spill) return false;
  const int tries = (u.op == su3::EX_ADD || u.op == su3::EX_EMUL) ? 2 : 1;   // IEEE + and * are commutative bit for bit
  for (int t = 0; t < tries; t++) {
    const unsigned char ua = t ? u.b : u.a, ub = t ? u.a : u.b;
    int saved[4] = {map[0], map[1], map[2], map[3]};
    auto bind = [&](unsigned char us, unsigned char ms) {
      if (ms >= su3::EX_TEMP0) return us == ms;          // temporaries and the accumulator must agree literally
      if (us >= su3::EX_TEMP0) return false;
      if (map[ms] < 0) {
        for (int k = 0; k < 4; k++)
          if (map[k] == us) return false;                // injective: one slot per distinct field
        map[ms] = us;
        return true;
      }
      return map[ms] == us;
    };
    if (bind(ua, m.a) && (u.op == su3::EX_COPY || bind(ub, m.b)) && match_menu_from(pr, mp, i + 1, map)) return true;
    for (int k = 0; k < 4; k++) map[k] = saved[k];
  }
  return false;
}
int match_menu(const ExprProgram &pr, int nops, bool real, int map[4]) {
  for (int op = 0; op < su3::OP_COPY; op++) {
    const su3::MenuProg mp = su3::menu_prog(op);
    if (mp.nin != nops || mp.nins != pr.nins) continue;
    if (real && !su3tab::menu_elementwise(op)) continue;
    if (!real && (op == su3::OP_EMUL || op == su3::OP_SUM_EPROD)) continue;
    map[0] = map[1] = map[2] = map[3] = -1;
    if (match_menu_from(pr, mp, 0, map)) return op;
  }
  return -1;
}
const char *const kMenuPostfix[su3::OP_COUNT] = {"01*", "01*2*", "01*2+", "01+", "01+01*+", "01*23*+", "01*23*-", "01*2-",
                                                 "01+2+", "01+2+3+", "01-", "01*", "01+01*+", "01*2*3*", "012**", "01*23**", "0"};

// ---------------------------------------------------------------- Cshift / shifted product
// alt != NULL (su3_cshift_slab, op = SH_COPY only): the runs that leave the slab are read from the neighbouring slab
// `alt` by the bulk-copy kernel; returns SU3_ERR_INVALID + *fused = false when that kernel does not apply (the caller
// then shifts locally and copies the face).
su3_status launch_shift(int op, su3_field *z, const su3_field *x, const su3_field *y, int dim, int disp, void *stream,
                        const su3_field *alt = nullptr, bool *fused = nullptr) {
  if (!z || !y || (op == su3::SH_MUL && !x)) return fail(SU3_ERR_NULL, "field handle is NULL");
  if (!same_desc(z->d, y->d) || (x && !same_desc(z->d, x->d))) return fail(SU3_ERR_MISMATCH, "operand descriptors differ");
  if (z->ncomp != 9 || y->ncomp != 9 || (x && x->ncomp != 9)) return fail(SU3_ERR_MISMATCH, "colour-matrix fields expected");
  if (dim < 0 || dim > 3) return fail(SU3_ERR_INVALID, "dim = %d outside 0..3", dim);
  if (z->ptr == y->ptr) return fail(SU3_ERR_MISMATCH, "the output must not be the shifted operand's field");
  if (su3_status sd = on_current_device({z, x, y})) return sd;
  const DevInfo &di = devinfo();
  if (z->nmat == 0) return SU3_OK;
  const su3_desc &d = z->d;
  su3::ShiftParams p;
  memset(&p, 0, sizeof p);
  p.z = z->ptr; p.x = x ? x->ptr : nullptr; p.y = y->ptr; p.nmat = z->nmat; p.nl = d.n_lorentz;
  p.ostride = 1; p.lstride = 1;
  for (int k = 0; k < dim; k++) {
    p.ostride *= d.L[k] / d.simd[k];
    p.lstride *= d.simd[k];
  }
  p.Ld = d.L[dim]; p.simd_d = d.simd[dim]; p.rd = d.L[dim] / d.simd[dim];
  p.disp = ((disp % p.Ld) + p.Ld) % p.Ld;
  // 32-bit index arithmetic whenever every complex index (plus one tile of slack) fits 31 bits
  shift_kernel_t k = su3tab::shift_kernel(d.prec, op, d.W, (z->nmat + 64) * 9 < 0x7fffffffLL);
  if (!k) return fail(SU3_ERR_INVALID, "no shift kernel for W %d", d.W);
  const su3_tune tn = g_tune;
  // Default: the TMA pipeline with a shifted operand -- the sources of a tile are a few contiguous runs of records, moved
  // by bulk copies; across the sub-lattice boundary the consumer reads a rotated lane.  With 72-byte records (fp32,
  // scalar layout) all runs of a launch must agree in (source - destination) mod 16, true unless r[dim]*P is odd.
  const int64_t P = p.ostride * d.n_lorentz;
  const bool odd72 = d.prec == SU3_F32 && d.W == 1 && ((int64_t)p.rd * P) % 2 != 0;
  // Cshift: the pure TMA copy (su3_cshift_bulk_kernel: the ceiling kernel with its loads split into runs).  Bulk copies
  // need 16-byte alignment; with 72-byte records (fp32, scalar layout) that means every run boundary and every source
  // record is even: P even and an even record count.
  const int64_t nrec_all = z->nmat / d.W;
  const bool bulk72_ok = !(d.prec == SU3_F32 && d.W == 1) || (P % 2 == 0 && nrec_all % 2 == 0);
  const bool bulk_applies = op == su3::SH_COPY && (tn.path == 0 || tn.path == 1) && bulk72_ok && z->nmat < 0x7fffffffLL;
  if (alt) {
    const bool ok = bulk_applies && !(d.W > 1 && p.simd_d > 1) && p.disp != 0;   // lanes of one record would come from two slabs
    if (fused) *fused = ok;
    if (!ok) return SU3_ERR_INVALID;
  }
  if (bulk_applies) {
    stream_kernel_t kb = su3tab::cshift_bulk_kernel(d.prec, d.W);
    if (!kb) return fail(SU3_ERR_INVALID, "no shift kernel for W %d", d.W);
    const int cbb = 2 * d.prec, rbytes = 9 * d.W * cbb;
    // as su3_copy: 3 one-warp CTAs per SM with 18 KB tiles -- unless the shift crosses virtual nodes (W > 1 and the
    // dimension is split): the lane rotation is done by the CTA's one warp between load and store, so twice as many CTAs
    // with 9 KB tiles keep the TMA engine busy meanwhile (measured at 48^4 fp64 W=4, dims 2/3: 0.95 -> 0.995 x copy)
    const bool rotates = d.W > 1 && p.simd_d > 1;
    const int ctas = tn.ctas_per_sm > 0 ? tn.ctas_per_sm : (rotates ? 6 : 3);
    int tm = tn.tile_mats > 0 ? tn.tile_mats : (rotates ? 9216 : 18432) / (9 * cbb);
    if (tm < d.W) tm = d.W;
    tm = tm / d.W * d.W;
    while (tm > 2 * d.W && (z->nmat + tm - 1) / tm < 2 * (int64_t)di.sms * ctas && (tm / 2) % d.W == 0 && ((tm / 2 / d.W) * rbytes) % 16 == 0) tm >>= 1;
    if (((tm / d.W) * rbytes) % 16) tm += d.W;                           // fp32 scalar: an even number of 72-byte records per tile
    int stages = tn.stages > 0 ? tn.stages : 2;
    const size_t tile_bytes = (size_t)(tm / d.W) * rbytes;
    const size_t budget = ((size_t)di.smem_optin + 1024) / ctas - 1024;
    while (stages > 2 && (size_t)stages * tile_bytes + 256 > budget) stages--;
    const size_t smem_b = (size_t)stages * tile_bytes + stages * sizeof(uint64_t);
    if (smem_b > (size_t)di.smem_optin) return fail(SU3_ERR_INVALID, "su3_cshift pipeline needs %zu B of shared memory", smem_b);
    cudaError_t eb = allow_max_smem((const void *)kb, di.smem_optin);
    if (eb != cudaSuccess) return cuda_fail("cudaFuncSetAttribute", eb);
    su3::StreamParams sp;
    memset(&sp, 0, sizeof sp);
    sp.z = z->ptr; sp.x = y->ptr; sp.nmat = z->nmat; sp.tile_mats = tm; sp.stages = stages;
    sp.sh.P = P; sp.sh.rd = p.rd; sp.sh.dmod = p.disp % p.rd; sp.sh.qrot = p.disp / p.rd; sp.sh.simd_d = p.simd_d; sp.sh.lstride = p.lstride;
    if (alt) {
      sp.sh.alt = alt->ptr;
      sp.sh.alt_carry = disp > 0 ? 1 : 0;   // disp > 0: the wrapping (carry) runs belong to the next slab; disp < 0: the others to the previous one
    }
    const int64_t ntiles_b = (z->nmat + tm - 1) / tm, cap_b = (int64_t)di.sms * ctas;
    kb<<<(unsigned)(ntiles_b < cap_b ? ntiles_b : cap_b), 32, smem_b, (cudaStream_t)stream>>>(sp);
    eb = cudaGetLastError();
    if (eb != cudaSuccess) return cuda_fail("cshift kernel launch", eb);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return SU3_OK;
  }
  // The shifted product: the TMA pipeline with a shifted operand for fp64 (the producer warp issues the runs of a tile in
  // parallel, so even 5-6 runs per tile along the fastest dimension cost nothing: measured 0.92-1.00 x copy at 32^4-64^4
  // against 0.88-0.95 for the register kernel); fp32 stays on the register kernel (0.95-0.99 against 0.85-0.96: its
  // 4.6 KB operand slots make the pipeline's per-tile costs twice as visible).  path = 1 forces the pipeline, 2 the other.
  const bool pipe_pays = d.prec == SU3_F64;
  // Cshift of 72-byte records whose run boundaries are odd (no 16-byte alignment for the pure copy kernel above): the
  // pipeline with OP_COPY, whose consumers move the matrices out of the 8-byte-shifted slot (0.95-0.96 x copy against 0.88
  // for the cp.async gather kernel, which path = 3 still selects, and 0.82 for the register kernel, path = 2)
  const bool copy_pipe = op == su3::SH_COPY && !bulk_applies && (tn.path == 1 || tn.path == 0);
  if (((op == su3::SH_MUL && (tn.path == 1 || (tn.path == 0 && pipe_pays))) || copy_pipe) && !odd72 && z->nmat < 0x7fffffffLL) {  // record indices fit 31 bits (P <= records)
    su3::ShiftInfo sh = {};
    sh.P = P; sh.rd = p.rd; sh.dmod = p.disp % p.rd; sh.qrot = p.disp / p.rd; sh.simd_d = p.simd_d; sh.lstride = p.lstride;
    sh.phase = (d.prec == SU3_F32 && d.W == 1 && ((int64_t)sh.dmod * P) % 2) ? 8 : 0;
    const void *in[4] = {op == su3::SH_MUL ? x->ptr : y->ptr, op == su3::SH_MUL ? y->ptr : nullptr, nullptr, nullptr};
    return launch_stream(op == su3::SH_MUL ? su3::OP_MUL : su3::OP_COPY, d.prec, d.W, z->ptr, in, z->nmat,
                         z->nbytes * (op == su3::SH_MUL ? 3 : 2), (cudaStream_t)stream, &sh);
  }
  if (op == su3::SH_COPY && tn.path != 2) {  // cp.async gather + TMA store (path = 2 keeps the register version)
    const bool small = (z->nmat + 64) * 9 < 0x7fffffffLL;
    shift_kernel_t ka = su3tab::cshift_async_kernel(d.prec, d.W, small);
    if (!ka) return fail(SU3_ERR_INVALID, "no shift kernel for W %d", d.W);
    const size_t smem_a = 4 * 18432;
    cudaError_t ea = allow_max_smem((const void *)ka, di.smem_optin);
    if (ea != cudaSuccess) return cuda_fail("cudaFuncSetAttribute", ea);
    const int64_t nwt_a = (z->nmat + 31) / 32, need = (nwt_a + 3) / 4, cap_a = (int64_t)di.sms * (tn.ctas_per_sm > 0 ? tn.ctas_per_sm : (d.prec == SU3_F64 ? 6 : 3));  // 3 resident per SM; measured
    ka<<<(unsigned)(need < cap_a ? need : cap_a), 128, smem_a, (cudaStream_t)stream>>>(p);
    ea = cudaGetLastError();
    if (ea != cudaSuccess) return cuda_fail("cshift kernel launch", ea);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return SU3_OK;
  }
  const int64_t nwt = (z->nmat + 31) / 32;
  int wpb = 4;
  while (wpb > 1 && (nwt + wpb - 1) / wpb < 2 * (int64_t)di.sms) wpb >>= 1;
  const size_t smem = op == su3::SH_MUL ? (size_t)wpb * 2 * 288 * 2 * d.prec : 0;
  const int64_t blocks_needed = (nwt + wpb - 1) / wpb;
  // measured defaults: Cshift one tile per warp (no grid-stride loop); the shifted product 8 persistent blocks/SM
  const int64_t cap = tn.ctas_per_sm > 0 ? (int64_t)di.sms * tn.ctas_per_sm * (4 / wpb)
                                         : (op == su3::SH_COPY ? 0x7fffffffLL : (int64_t)di.sms * 8 * (4 / wpb));
  k<<<(unsigned)(blocks_needed < cap ? blocks_needed : cap), wpb * 32, smem, (cudaStream_t)stream>>>(p);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("shift kernel launch", e);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SU3_OK;
}

// ---------------------------------------------------------------- su3_mul_host / su3_eval_host resources
// One set of copy streams and events per (device, caller stream): two host threads that drive different streams never
// share anything and never serialise on each other; callers of the SAME stream are ordered by that stream anyway.
constexpr int MAX_HOST_CHUNKS = 64;
constexpr size_t MAX_HOST_PIPES = 64;
struct HostPipe {
  std::mutex mu;
  cudaStream_t h2d = nullptr, d2h = nullptr;
  std::vector<cudaEvent_t> ev;
  cudaError_t ensure(size_t nev) {
    cudaError_t e = cudaSuccess;
    if (!h2d && (e = cudaStreamCreateWithFlags(&h2d, cudaStreamNonBlocking)) != cudaSuccess) return e;
    if (!d2h && (e = cudaStreamCreateWithFlags(&d2h, cudaStreamNonBlocking)) != cudaSuccess) return e;
    while (ev.size() < nev) {
      cudaEvent_t v;
      if ((e = cudaEventCreateWithFlags(&v, cudaEventDisableTiming)) != cudaSuccess) return e;
      ev.push_back(v);
    }
    return e;
  }
  void destroy() {  // waits for the pipe's own copies, then frees its streams and events
    if (h2d) { cudaStreamSynchronize(h2d); cudaStreamDestroy(h2d); h2d = nullptr; }
    if (d2h) { cudaStreamSynchronize(d2h); cudaStreamDestroy(d2h); d2h = nullptr; }
    for (cudaEvent_t v : ev) cudaEventDestroy(v);
    ev.clear();
    (void)cudaGetLastError();
  }
};
std::mutex g_hp_mu;  // guards the map only, never held across CUDA calls of a pipeline
std::map<std::pair<int, cudaStream_t>, std::unique_ptr<HostPipe>> g_hp;

HostPipe *host_pipe(int dev, cudaStream_t user) {
  std::lock_guard<std::mutex> lk(g_hp_mu);
  auto key = std::make_pair(dev, user);
  auto it = g_hp.find(key);
  if (it != g_hp.end()) return it->second.get();
  if (g_hp.size() >= MAX_HOST_PIPES) return nullptr;
  HostPipe *hp = new (std::nothrow) HostPipe;
  if (hp) g_hp[key].reset(hp);
  return hp;
}

}  // namespace

extern "C" {

const char *su3_last_error(void) { return g_err; }
const char *su3_version(void) { return "su3stream 0.1 (sm_100a)"; }

su3_status su3_desc_normalize(const su3_desc *desc, su3_desc *out) { return normalize(desc, out); }

su3_status su3_field_bytes(const su3_desc *desc, size_t *nbytes) {
  if (!nbytes) return fail(SU3_ERR_NULL, "nbytes is NULL");
  su3_desc d;
  su3_status st = normalize(desc, &d);
  if (st != SU3_OK) return st;
  *nbytes = (size_t)volume_of(d) * d.n_lorentz * 18 * d.prec;
  return SU3_OK;
}

static su3_status wrap_kind(const su3_desc *desc, void *dev_ptr, size_t nbytes, su3_field **out, int ncomp) {
  if (!out) return fail(SU3_ERR_NULL, "out is NULL");
  su3_desc d;
  su3_status st = normalize(desc, &d);
  if (st != SU3_OK) return st;
  if (!dev_ptr) return fail(SU3_ERR_NULL, "device pointer is NULL");
  if ((uintptr_t)dev_ptr & 15) return fail(SU3_ERR_ALIGN, "device pointer %p is not 16-byte aligned", dev_ptr);
  const size_t need = (size_t)volume_of(d) * d.n_lorentz * (ncomp ? 2 * ncomp : 1) * d.prec;  // ncomp = 0: one REAL per (site, mu)
  if (nbytes < need) return fail(SU3_ERR_SIZE, "buffer of %zu bytes is smaller than the %zu the field needs", nbytes, need);
  su3_field *f = new (std::nothrow) su3_field;
  if (!f) return fail(SU3_ERR_SIZE, "out of host memory");
  f->d = d; f->ptr = dev_ptr; f->nbytes = need; f->volume = volume_of(d); f->nmat = f->volume * d.n_lorentz;
  f->ncomp = ncomp;
  f->device = -1;  // which device owns the memory (asked once, here; never dereferenced)
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, dev_ptr) == cudaSuccess && (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged))
    f->device = at.device;
  (void)cudaGetLastError();
  *out = f;
  return SU3_OK;
}

su3_status su3_field_wrap(const su3_desc *desc, void *dev_ptr, size_t nbytes, su3_field **out) {
  return wrap_kind(desc, dev_ptr, nbytes, out, 9);
}

su3_status su3_vec_wrap(const su3_desc *desc, void *dev_ptr, size_t nbytes, su3_field **out) {
  return wrap_kind(desc, dev_ptr, nbytes, out, 3);
}

su3_status su3_real_wrap(const su3_desc *desc, void *dev_ptr, size_t nbytes, su3_field **out) {
  return wrap_kind(desc, dev_ptr, nbytes, out, 0);
}

su3_status su3_real_bytes(const su3_desc *desc, size_t *nbytes) {
  if (!nbytes) return fail(SU3_ERR_NULL, "nbytes is NULL");
  su3_desc d;
  su3_status st = normalize(desc, &d);
  if (st != SU3_OK) return st;
  *nbytes = (size_t)volume_of(d) * d.n_lorentz * d.prec;
  return SU3_OK;
}

su3_status su3_fill(su3_field *z, double value, void *cuda_stream) {
  if (!z) return fail(SU3_ERR_NULL, "field handle is NULL");
  if (z->ncomp != 0) return fail(SU3_ERR_MISMATCH, "su3_fill takes a real scalar field");
  if (su3_status sd = on_current_device({z})) return sd;
  const DevInfo &di = devinfo();
  if (z->nmat == 0) return SU3_OK;
  const unsigned grid = flat_grid((size_t)z->nmat, 256, 8);
  if (z->d.prec == SU3_F64) su3::su3_real_fill_kernel<double><<<grid, 256, 0, (cudaStream_t)cuda_stream>>>((double *)z->ptr, z->nmat, value);
  else su3::su3_real_fill_kernel<float><<<grid, 256, 0, (cudaStream_t)cuda_stream>>>((float *)z->ptr, z->nmat, (float)value);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("su3_fill launch", e);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SU3_OK;
}

su3_status su3_vec_bytes(const su3_desc *desc, size_t *nbytes) {
  if (!nbytes) return fail(SU3_ERR_NULL, "nbytes is NULL");
  su3_desc d;
  su3_status st = normalize(desc, &d);
  if (st != SU3_OK) return st;
  *nbytes = (size_t)volume_of(d) * d.n_lorentz * 6 * d.prec;
  return SU3_OK;
}

su3_status su3_field_free(su3_field *f) {
  if (!f) return fail(SU3_ERR_NULL, "field handle is NULL");
  delete f;
  return SU3_OK;
}

su3_status su3_field_desc(const su3_field *f, su3_desc *out) {
  if (!f || !out) return fail(SU3_ERR_NULL, "NULL argument");
  *out = f->d;
  return SU3_OK;
}

su3_status su3_field_ptr(const su3_field *f, void **dev_ptr, size_t *nbytes) {
  if (!f || !dev_ptr || !nbytes) return fail(SU3_ERR_NULL, "NULL argument");
  *dev_ptr = f->ptr; *nbytes = f->nbytes;
  return SU3_OK;
}

su3_status su3_index(const su3_desc *desc, int64_t site, int mu, int i, int j, int reim, int64_t *off) {
  if (!off) return fail(SU3_ERR_NULL, "off is NULL");
  su3_desc d;
  su3_status st = normalize(desc, &d);
  if (st != SU3_OK) return st;
  if (site < 0 || site >= volume_of(d) || mu < 0 || mu >= d.n_lorentz || i < 0 || i > 2 || j < 0 || j > 2 || reim < 0 || reim > 1)
    return fail(SU3_ERR_INVALID, "index (site %lld, mu %d, i %d, j %d, reim %d) out of range", (long long)site, mu, i, j, reim);
  const int e = 3 * i + j;
  if (d.layout == SU3_SCALAR) {
    *off = ((site * d.n_lorentz + mu) * 9 + e) * 2 + reim;
    return SU3_OK;
  }
  int64_t o = 0, ostride = 1, l = 0, lstride = 1, s = site;
  for (int k = 0; k < 4; k++) {
    const int64_t xk = s % d.L[k];
    s /= d.L[k];
    const int64_t r = d.L[k] / d.simd[k];
    o += (xk % r) * ostride; ostride *= r;
    l += (xk / r) * lstride; lstride *= d.simd[k];
  }
  *off = (((o * d.n_lorentz + mu) * 9 + e) * d.W + l) * 2 + reim;
  return SU3_OK;
}

su3_status su3_mul(su3_field *z, const su3_field *x, const su3_field *y, void *s) {
  return arith(su3::OP_MUL, z, x, y, nullptr, s);
}
su3_status su3_mul3(su3_field *z, const su3_field *x, const su3_field *y, const su3_field *w, void *s) {
  return arith(su3::OP_MUL3, z, x, y, w, s);
}
su3_status su3_mul_add(su3_field *z, const su3_field *x, const su3_field *y, const su3_field *v, void *s) {
  return arith(su3::OP_MUL_ADD, z, x, y, v, s);
}

su3_status su3_expr_disasm(const char *program, int n_operands, char *buf, size_t buf_len) {
  if (!buf) return fail(SU3_ERR_NULL, "buf is NULL");
  ExprProgram pr;
  su3_status st = compile_expr(program, n_operands, &pr);
  if (st != SU3_OK) return st;
  static const char *names[] = {"mul", "add", "sub", "copy"};
  size_t used = 0;
  auto src = [](unsigned char v, char *out) {
    if (v == su3::EX_SRC_ACC) snprintf(out, 8, "acc");
    else if (v >= su3::EX_TEMP0) snprintf(out, 8, "t%d", v - su3::EX_TEMP0);
    else snprintf(out, 8, "o%d", v);
  };
  for (int i = 0; i < pr.nins; i++) {
    char a[8], b[8] = "-", line[64];
    src(pr.ins[i].a, a);
    if (pr.ins[i].op != su3::EX_COPY) src(pr.ins[i].b, b);
    int n = snprintf(line, sizeof line, "%s %s %s", names[pr.ins[i].op], a, b);
    if (pr.ins[i].spill != su3::EX_NONE) n += snprintf(line + n, sizeof line - n, " spill t%d", pr.ins[i].spill - su3::EX_TEMP0);
    n += snprintf(line + n, sizeof line - n, "\n");
    if (used + n + 1 > buf_len) return fail(SU3_ERR_SIZE, "listing needs more than %zu bytes", buf_len);
    memcpy(buf + used, line, n);
    used += n;
  }
  if (buf_len == 0) return fail(SU3_ERR_SIZE, "empty buffer");
  buf[used] = 0;
  return SU3_OK;
}

su3_status su3_expr_plan(const char *program, int n_operands, int real_fields, char *buf, size_t buf_len) {
  if (!buf || buf_len == 0) return fail(SU3_ERR_NULL, "buf is NULL or empty");
  ExprProgram pr;
  su3_status st = compile_expr(program, n_operands, &pr);
  if (st != SU3_OK) return st;
  if (real_fields)
    for (int i = 0; i < pr.nins; i++)
      if (pr.ins[i].op == su3::EX_MUL) pr.ins[i].op = su3::EX_EMUL;
  int map[4];
  const int op = match_menu(pr, n_operands, real_fields != 0, map);
  int n;
  if (op < 0) n = snprintf(buf, buf_len, "interpreter");
  else {
    n = snprintf(buf, buf_len, "menu %d %s", op, kMenuPostfix[op]);
    for (int k = 0; k < n_operands && n > 0 && (size_t)n < buf_len; k++) n += snprintf(buf + n, buf_len - n, " %d", map[k]);
  }
  if (n < 0 || (size_t)n >= buf_len) return fail(SU3_ERR_SIZE, "plan needs more than %zu bytes", buf_len);
  return SU3_OK;
}

su3_status su3_expr_cost(const char *program, int n_operands, int32_t *streams, int32_t *flops_per_matrix) {
  ExprProgram pr;
  su3_status st = compile_expr(program, n_operands, &pr);
  if (st != SU3_OK) return st;
  if (streams) *streams = n_operands + 1;
  if (flops_per_matrix) *flops_per_matrix = 198 * pr.nmul + 18 * pr.naddsub;
  return SU3_OK;
}

su3_status su3_expr(su3_field *z, const char *program, const su3_field *const *operands, int n_operands,
                    void *cuda_stream) {
  if (!z || !operands) return fail(SU3_ERR_NULL, "NULL argument");
  ExprProgram pr;
  su3_status st = compile_expr(program, n_operands, &pr);
  if (st != SU3_OK) return st;
  if (z->ncomp != 9 && z->ncomp != 0) return fail(SU3_ERR_MISMATCH, "su3_expr takes colour-matrix fields or real scalar fields");
  for (int k = 0; k < n_operands; k++) {
    if (!operands[k]) return fail(SU3_ERR_NULL, "operand %d is NULL", k);
    if (!same_desc(z->d, operands[k]->d) || operands[k]->ncomp != z->ncomp)
      return fail(SU3_ERR_MISMATCH, "operand %d: descriptor or field kind differs from z", k);
  }
  if (su3_status sd = on_current_device({z})) return sd;
  for (int k = 0; k < n_operands; k++)
    if (su3_status sd = on_current_device({operands[k]})) return sd;
  const DevInfo &di = devinfo();
  if (z->nmat == 0) return SU3_OK;
  const bool real = z->ncomp == 0;
  // Real scalar fields (the paper's Listing 2) are element-wise, so n reals = n / 18 records of 18 reals for the
  // matrix machinery below (W = 1; '*' becomes the element-wise EX_EMUL) plus a tail of n % 18 reals.
  const int64_t nrec = real ? z->nmat / 18 : z->nmat;
  const int W_eff = real ? 1 : z->d.W;
  if (real) {
    for (int i = 0; i < pr.nins; i++)
      if (pr.ins[i].op == su3::EX_MUL) pr.ins[i].op = su3::EX_EMUL;
    const int64_t ntail = z->nmat - nrec * 18;
    if (ntail) {
      su3::ExprParams pt;
      memset(&pt, 0, sizeof pt);
      const size_t off = (size_t)nrec * 18 * z->d.prec;
      pt.z = (char *)z->ptr + off;
      for (int i = 0; i < n_operands; i++) pt.ops[i] = (const char *)operands[i]->ptr + off;
      pt.nmat = ntail; pt.nops = n_operands; pt.nins = pr.nins; pt.ntemp = pr.ntemp;
      for (int i = 0; i < pr.nins; i++) pt.ins[i] = pr.ins[i];
      if (z->d.prec == SU3_F64) su3::su3_real_expr_kernel<double><<<1, 32, 0, (cudaStream_t)cuda_stream>>>(pt);
      else su3::su3_real_expr_kernel<float><<<1, 32, 0, (cudaStream_t)cuda_stream>>>(pt);
      cudaError_t er = cudaGetLastError();
      if (er != cudaSuccess) return cuda_fail("su3_expr (real tail) launch", er);
      g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    if (nrec == 0) return SU3_OK;
  }
  {
    // the ahead-of-time menu: programs that ARE one of the compiled-in kernels run on them (same FMA chains, same
    // order of operations as the interpreter, so the result is bit-identical either way)
    int map[4];
    const int op = g_tune.path == 3 ? -1 : match_menu(pr, n_operands, real, map);   // path = 3: always the interpreter
    if (op >= 0) {
      const void *in[4] = {nullptr, nullptr, nullptr, nullptr};
      for (int k = 0; k < n_operands; k++) in[k] = operands[map[k]]->ptr;
      return launch_stream(op, z->d.prec, su3tab::menu_elementwise(op) ? 1 : W_eff, z->ptr, in, nrec,
                           z->nbytes * (n_operands + 1), (cudaStream_t)cuda_stream);
    }
  }
  const su3_tune tn = g_tune;
  const int cb = 2 * z->d.prec;
  expr_kernel_t k = su3tab::expr_kernel(z->d.prec, W_eff);
  if (!k) return fail(SU3_ERR_INVALID, "no expression kernel for W %d", W_eff);
  // Every CTA (96 threads: three threads per matrix, su3_kernels.cuh) is a self-contained pipeline with a private ring of
  // `sw` stages of `mps` matrices per operand.  Interpreted programs are latency-bound per tile, so the launch maximises
  // resident CTAs per SM under the shared-memory budget (ring depth 3 if there is room for >= 4 CTAs anyway, else 2).
  // matrices per stage and operand: 32 (one per lane and row warp); fp32 programs with <= 3 operands take 64 (4608-byte
  // slots as in fp64)
  const int mps = tn.tile_mats > 0 ? tn.tile_mats : ((z->d.prec == SU3_F32 && n_operands <= 3) ? 64 : 32);
  const size_t slot = (size_t)mps * 9 * cb;
  const size_t stage_bytes = (size_t)n_operands * slot;
  int xchg = 0;  // a product whose RIGHT factor is the accumulator: one more slot to make it whole
  for (int i = 0; i < pr.nins; i++)
    if (pr.ins[i].op == su3::EX_MUL && pr.ins[i].b == su3::EX_SRC_ACC) xchg = 1;
  const size_t fixed = (size_t)(pr.ntemp + xchg + 2) * slot + 128;              // temporaries, exchange slot, two result slots, barriers
  const size_t sm_bytes = (size_t)di.smem_optin;                                // what one SM can give to its resident CTAs
  auto ctas_for = [&](int sw_) { return (int)((sm_bytes + 1024) / (sw_ * stage_bytes + fixed + 1024)); };  // 1 KB reserved per CTA
  // ring depth 2 and as many CTAs as fit: measured at 48^4, more resident warps beat a deeper ring for every program
  // (`01+01*+` fp64: 4 CTAs x 3 stages 0.79, 6 x 3 0.92, 8 x 2 0.99 x copy)
  int sw = tn.stages > 0 ? tn.stages : 2;
  int ctas = ctas_for(sw);
  const int reg_cap = z->d.prec == SU3_F64 ? 7 : 12;  // resident CTAs of 96 threads per SM that 88-90 (fp64) / 48-56 (fp32) registers per thread allow;
                                                      // asking for more would leave CTAs of the persistent grid waiting for a slot
  if (ctas > reg_cap) ctas = reg_cap;
  if (tn.ctas_per_sm > 0 && tn.ctas_per_sm < ctas) ctas = tn.ctas_per_sm;
  if (ctas < 1 || sw < 2) return fail(SU3_ERR_INVALID, "expression needs more shared memory than the device has (%d operands, %d temporaries)",
                                      n_operands, pr.ntemp);
  const size_t smem = (size_t)sw * stage_bytes + fixed;
  if (smem > (size_t)di.smem_optin) return fail(SU3_ERR_INVALID, "expression needs %zu B of shared memory, device allows %d", smem, di.smem_optin);
  cudaError_t e = allow_max_smem((const void *)k, di.smem_optin);
  if (e != cudaSuccess) return cuda_fail("cudaFuncSetAttribute", e);
  su3::ExprParams p;
  memset(&p, 0, sizeof p);
  p.z = z->ptr;
  for (int i = 0; i < n_operands; i++) p.ops[i] = operands[i]->ptr;
  p.nmat = nrec; p.tile_mats = mps; p.stages = sw; p.nops = n_operands; p.nins = pr.nins; p.ntemp = pr.ntemp; p.xchg = xchg;
  for (int i = 0; i < pr.nins; i++) {
    p.ins[i] = pr.ins[i];
    p.insx[i] = make_int4(pr.ins[i].op, pr.ins[i].a, pr.ins[i].b, pr.ins[i].spill);
  }
  const int64_t ntiles = (nrec + mps - 1) / mps, max_grid = (int64_t)di.sms * ctas;
  k<<<(unsigned)(ntiles < max_grid ? ntiles : max_grid), 96, smem, (cudaStream_t)cuda_stream>>>(p);
  e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("su3_expr launch", e);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SU3_OK;
}

su3_status su3_cshift(su3_field *z, const su3_field *x, int dim, int disp, void *cuda_stream) {
  return launch_shift(su3::SH_COPY, z, nullptr, x, dim, disp, cuda_stream);
}
su3_status su3_mul_shift(su3_field *z, const su3_field *x, const su3_field *y, int dim, int disp, void *cuda_stream) {
  return launch_shift(su3::SH_MUL, z, x, y, dim, disp, cuda_stream);
}

static su3_status launch_face_copy(const su3_field *geo, void *dst, bool dpacked, int dplane0, const void *src, bool spacked,
                                   int splane0, int dim, int nplanes, void *stream);

su3_status su3_cshift_slab(su3_field *z, const su3_field *x, const su3_field *x_nbr, int disp, void *cuda_stream) {
  if (!z || !x || !x_nbr) return fail(SU3_ERR_NULL, "field handle is NULL");
  if (!same_desc(z->d, x->d) || !same_desc(z->d, x_nbr->d)) return fail(SU3_ERR_MISMATCH, "operand descriptors differ");
  if (z->ncomp != 9 || x->ncomp != 9 || x_nbr->ncomp != 9) return fail(SU3_ERR_MISMATCH, "colour-matrix fields expected");
  if (z->ptr == x->ptr || z->ptr == x_nbr->ptr) return fail(SU3_ERR_MISMATCH, "the output must not be one of the shifted slabs");
  const int l3 = z->d.L[3];
  if (disp <= -l3 || disp >= l3) return fail(SU3_ERR_INVALID, "su3_cshift_slab: |disp| = %d must be below the slab's %d planes", disp < 0 ? -disp : disp, l3);
  if (disp == 0) return su3_copy(z, x, cuda_stream);
  bool fused = false;
  su3_status st = launch_shift(su3::SH_COPY, z, nullptr, x, 3, disp, cuda_stream, x_nbr, &fused);   // x_nbr may be peer memory: not device-checked
  if (fused || st != SU3_ERR_INVALID) return st;
  // two launches: the periodic shift of the slab, then the planes that wrapped, straight from the neighbouring slab
  if ((st = launch_shift(su3::SH_COPY, z, nullptr, x, 3, disp, cuda_stream)) != SU3_OK) return st;
  const int n = disp > 0 ? disp : -disp;
  return launch_face_copy(z, z->ptr, false, disp > 0 ? l3 - n : 0, x_nbr->ptr, false, disp > 0 ? 0 : l3 - n, 3, n, cuda_stream);
}

su3_status su3_vec_index(const su3_desc *desc, int64_t site, int mu, int i, int reim, int64_t *off) {
  if (!off) return fail(SU3_ERR_NULL, "off is NULL");
  su3_desc d;
  su3_status st = normalize(desc, &d);
  if (st != SU3_OK) return st;
  if (site < 0 || site >= volume_of(d) || mu < 0 || mu >= d.n_lorentz || i < 0 || i > 2 || reim < 0 || reim > 1)
    return fail(SU3_ERR_INVALID, "index (site %lld, mu %d, i %d, reim %d) out of range", (long long)site, mu, i, reim);
  if (d.layout == SU3_SCALAR) {
    *off = ((site * d.n_lorentz + mu) * 3 + i) * 2 + reim;
    return SU3_OK;
  }
  int64_t o = 0, ostride = 1, l = 0, lstride = 1, s = site;
  for (int k = 0; k < 4; k++) {
    const int64_t xk = s % d.L[k];
    s /= d.L[k];
    const int64_t r = d.L[k] / d.simd[k];
    o += (xk % r) * ostride; ostride *= r;
    l += (xk / r) * lstride; lstride *= d.simd[k];
  }
  *off = (((o * d.n_lorentz + mu) * 3 + i) * d.W + l) * 2 + reim;
  return SU3_OK;
}

su3_status su3_matvec(su3_field *y, const su3_field *U, const su3_field *psi, void *stream) {
  if (!y || !U || !psi) return fail(SU3_ERR_NULL, "field handle is NULL");
  if (U->ncomp != 9 || psi->ncomp != 3 || y->ncomp != 3)
    return fail(SU3_ERR_MISMATCH, "su3_matvec takes y, psi colour-vector fields and U a colour-matrix field");
  if (!same_desc(y->d, U->d) || !same_desc(y->d, psi->d)) return fail(SU3_ERR_MISMATCH, "operand descriptors differ");
  if (su3_status sd = on_current_device({y, U, psi})) return sd;
  const DevInfo &di = devinfo();
  if (y->nmat == 0) return SU3_OK;
  const su3_tune tn = g_tune;
  const int cb = 2 * y->d.prec;
  stream_kernel_t k = su3tab::matvec_kernel(y->d.prec, y->d.W);
  if (!k) return fail(SU3_ERR_INVALID, "no matvec kernel for W %d", y->d.W);
  // measured (48^4): ~110 KB in flight per SM is the sweet spot -> 2 CTAs/SM of 24.6 KB stages (fp64), 4 of 12.3 KB (fp32)
  const int ctas = tn.ctas_per_sm > 0 ? tn.ctas_per_sm : (y->d.prec == SU3_F64 ? 2 : 4);
  int tm = tn.tile_mats;
  if (tm == 0) {
    tm = 128;
    while (tm > 32 && (y->nmat + tm - 1) / tm < 2 * (int64_t)di.sms * ctas) tm >>= 1;
  }
  const size_t stage_bytes = (size_t)tm * 12 * cb;
  const size_t budget = ((size_t)di.smem_optin + 1024) / ctas - 1024;
  int stages = tn.stages > 0 ? tn.stages : 3;
  while (tn.stages == 0 && stages > 2 && stages * stage_bytes + 256 > budget) stages--;
  const size_t smem = stages * stage_bytes + 2 * stages * sizeof(uint64_t);
  if (smem + 256 > budget) return fail(SU3_ERR_INVALID, "su3_matvec pipeline needs %zu B of shared memory (tile %d, %d stages, %d CTAs/SM)", smem, tm, stages, ctas);
  cudaError_t e = allow_max_smem((const void *)k, di.smem_optin);
  if (e != cudaSuccess) return cuda_fail("cudaFuncSetAttribute", e);
  su3::StreamParams p;
  p.z = y->ptr; p.x = U->ptr; p.y = psi->ptr; p.u = nullptr; p.nmat = y->nmat; p.tile_mats = tm; p.stages = stages; p.hint = 0;
  const int64_t ntiles = (y->nmat + tm - 1) / tm, max_grid = (int64_t)di.sms * ctas;
  k<<<(unsigned)(ntiles < max_grid ? ntiles : max_grid), (NCW + 1) * 32, smem, (cudaStream_t)stream>>>(p);
  e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("su3_matvec launch", e);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SU3_OK;
}

su3_status su3_add(su3_field *z, const su3_field *x, const su3_field *y, void *stream) {
  su3_status st = check_arith(z, x, y, nullptr, false);
  if (st != SU3_OK) return st;
  if ((st = on_current_device({z, x, y})) != SU3_OK) return st;
  const DevInfo &di = devinfo();
  const int path = g_tune.path;
  if (path != 2) {  // element-wise, hence layout-agnostic: the W = 1 pipeline over 9-complex records
    const void *in[4] = {x->ptr, y->ptr, nullptr, nullptr};
    return launch_stream(su3::OP_ADD, z->d.prec, 1, z->ptr, in, z->nmat, 3 * z->nbytes, (cudaStream_t)stream);
  }
  const size_t n16 = z->nbytes / 16;
  const int nrem = (int)((z->nbytes % 16) / z->d.prec);
  const unsigned grid = flat_grid(n16, 512, 8);
  if (z->d.prec == SU3_F64)
    su3::su3_add_kernel<double><<<grid, 256, 0, (cudaStream_t)stream>>>((double *)z->ptr, (const double *)x->ptr, (const double *)y->ptr, n16, nrem);
  else
    su3::su3_add_kernel<float><<<grid, 256, 0, (cudaStream_t)stream>>>((float *)z->ptr, (const float *)x->ptr, (const float *)y->ptr, n16, nrem);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("su3_add launch", e);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SU3_OK;
}

static su3_status launch_copy(void *dst_ptr, const void *src_ptr, size_t nbytes, int prec, void *stream) {
  const DevInfo &di = devinfo();
  if (!di.ok) return fail(SU3_ERR_CUDA, "%s", di.err);
  if (nbytes == 0) return SU3_OK;
  const su3_tune tn = g_tune;
  if (tn.path != 2) {  // TMA bulk pipeline: global -> shared -> global, one issuing thread per CTA
    const int mat_bytes = 18 * prec;
    const int ctas = tn.ctas_per_sm > 0 ? tn.ctas_per_sm : 3;
    unsigned tile = tn.tile_mats > 0 ? (unsigned)tn.tile_mats * mat_bytes : 18432u;  // multiple of 16
    const size_t n16 = nbytes & ~(size_t)15;
    while (tile > 2304 && (n16 + tile - 1) / tile < (size_t)2 * di.sms * ctas) tile >>= 1;
    int stages = tn.stages > 0 ? tn.stages : 2;
    const size_t budget = ((size_t)di.smem_optin + 1024) / ctas - 1024;
    while (stages > 2 && (size_t)stages * tile + 256 > budget) stages--;
    const size_t smem = (size_t)stages * tile + stages * sizeof(uint64_t);
    if (smem > (size_t)di.smem_optin) return fail(SU3_ERR_INVALID, "su3_copy pipeline needs %zu B of shared memory", smem);
    cudaError_t e = allow_max_smem((const void *)su3::su3_bulk_copy_kernel, di.smem_optin);
    if (e != cudaSuccess) return cuda_fail("cudaFuncSetAttribute", e);
    su3::CopyParams p;
    p.dst = dst_ptr; p.src = src_ptr; p.nbytes = nbytes; p.tile_bytes = tile; p.stages = stages;
    p.hint = tn.l2_hint == 2;
    size_t ntiles = (n16 + tile - 1) / tile;
    if (ntiles < 1) ntiles = 1;
    const size_t cap = (size_t)di.sms * ctas;
    su3::su3_bulk_copy_kernel<<<(unsigned)(ntiles < cap ? ntiles : cap), 32, smem, (cudaStream_t)stream>>>(p);
  } else {
    const size_t n16 = nbytes / 16;
    const int tail8 = (nbytes % 16) ? 1 : 0;
    const unsigned grid = flat_grid(n16, 1024, 8);
    su3::su3_copy_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>((uint4 *)dst_ptr, (const uint4 *)src_ptr, n16, tail8);
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("su3_copy launch", e);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SU3_OK;
}

su3_status su3_copy(su3_field *dst, const su3_field *src, void *stream) {
  if (!dst || !src) return fail(SU3_ERR_NULL, "field handle is NULL");
  if (!same_desc(dst->d, src->d) || dst->ncomp != src->ncomp || dst->ncomp == 0)
    return fail(SU3_ERR_MISMATCH, "su3_copy needs identical descriptors and field kinds (matrix or vector)");
  if (su3_status sd = on_current_device({dst, src})) return sd;
  return launch_copy(dst->ptr, src->ptr, dst->nbytes, dst->d.prec, stream);
}

su3_status su3_convert(su3_field *dst, const su3_field *src, void *stream) {
  if (!dst || !src) return fail(SU3_ERR_NULL, "field handle is NULL");
  if (!same_lattice(dst->d, src->d)) return fail(SU3_ERR_MISMATCH, "su3_convert: L, n_lorentz and prec must agree");
  if (dst->d.layout == src->d.layout)
    return fail(SU3_ERR_MISMATCH, "su3_convert: exactly one of dst/src must be SU3_SCALAR and the other SU3_VECTOR");
  if (dst->ptr == src->ptr) return fail(SU3_ERR_MISMATCH, "su3_convert: dst and src must not alias");
  if (dst->ncomp != src->ncomp || dst->ncomp == 0) return fail(SU3_ERR_MISMATCH, "su3_convert: matrix and vector fields cannot be mixed; real scalar fields have no layout");
  const int nc = dst->ncomp;
  if (su3_status sd = on_current_device({dst, src})) return sd;
  if (dst->d.W == 1 && src->d.W == 1)  // the W = 1 vector layout is byte-identical to the scalar layout
    return launch_copy(dst->ptr, src->ptr, dst->nbytes, dst->d.prec, stream);
  const DevInfo &di = devinfo();
  if (!di.ok) return fail(SU3_ERR_CUDA, "%s", di.err);
  const su3_desc &v = (dst->d.layout == SU3_VECTOR) ? dst->d : src->d;
  su3::ConvertParams p;
  memset(&p, 0, sizeof p);
  p.dst = dst->ptr; p.src = src->ptr;
  p.nl = v.n_lorentz;
  p.nrec = dst->volume / v.W * v.n_lorentz;
  p.to_vector = dst->d.layout == SU3_VECTOR;
  long long stride = 1;
  for (int k = 0; k < 4; k++) {
    p.r[k] = v.L[k] / v.simd[k];
    p.sstride[k] = stride;
    stride *= v.L[k];
  }
  for (int l = 0; l < v.W; l++) {  // lane l = lexicographic index of ic over simd, d=0 fastest
    long long off = 0;
    int rem = l;
    for (int k = 0; k < 4; k++) {
      const int ic = rem % v.simd[k];
      rem /= v.simd[k];
      off += (long long)ic * p.r[k] * p.sstride[k];
    }
    p.lane_off[l] = off * v.n_lorentz * nc;
  }
  if (p.nrec == 0) return SU3_OK;
  const su3_tune tn_c = g_tune;
  // records whose scalar-side images are contiguous: up to the first dimension that is split over virtual nodes
  long long run_sites = 1;
  {
    int k = 0;
    for (; k < 4; k++) {
      run_sites *= p.r[k];
      if (v.simd[k] > 1) break;
    }
  }
  p.run_recs = run_sites * v.n_lorentz;
  const char *err = nullptr;
  // Default: the TMA kernel (bulk copies on both sides, transposition in shared memory).  With 8-byte complex numbers its
  // bulk copies are 16-byte aligned only if every run starts and ends on an even complex index; odd geometries (and
  // path = 2 / 3, kept for measurements) take the per-thread kernels: 3 = staged through shared memory, 2 = unstaged.
  bool tma = (tn_c.path == 0 || tn_c.path == 1) && dst->volume < 0x7fffffffLL;  // the kernel decodes sites in 32 bits
  if (tma && v.prec == SU3_F32) {
    tma = (p.run_recs * nc) % 2 == 0;
    for (int l = 0; l < v.W; l++) tma = tma && p.lane_off[l] % 2 == 0;
  }
  if (tma) {
    const int K = su3tab::convert_tma_tile(v.prec) / v.W;                  // complex numbers per lane row
    const int phase = v.prec == SU3_F32 ? 16 : 8;                          // complex numbers per 128-byte wavefront
    const int want = v.W < phase ? phase / v.W : 1;
    int pad = ((want - K) % phase + phase) % phase;
    if (v.prec == SU3_F32 && ((K + pad) & 1)) pad += 1;                    // rows must stay 16-byte aligned
    p.pitch = K + pad;
    if (!su3tab::launch_convert_tma(v.prec, nc, v.W, p, (cudaStream_t)stream, &err))
      return fail(SU3_ERR_SIZE, "su3_convert: %s", err ? err : "unsupported W");
  } else if (!su3tab::launch_convert(v.prec, nc, v.W, tn_c.path != 2 && (v.prec == SU3_F32 || (v.W >= 8 && !p.to_vector)), p, (cudaStream_t)stream, &err))
    return fail(SU3_ERR_SIZE, "su3_convert: %s", err ? err : "unsupported W");
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("su3_convert launch", e);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SU3_OK;
}

// ---------------------------------------------------------------- faces of a slab (multi-GPU Cshift)
static su3_status face_args(const su3_field *f, int dim, int plane0, int nplanes, size_t *bytes) {
  if (!f) return fail(SU3_ERR_NULL, "field handle is NULL");
  if (f->ncomp == 0) return fail(SU3_ERR_MISMATCH, "faces exist for colour-matrix and colour-vector fields only");
  if (dim < 0 || dim > 3) return fail(SU3_ERR_INVALID, "dim = %d outside 0..3", dim);
  if (nplanes < 0 || plane0 < 0 || (int64_t)plane0 + nplanes > f->d.L[dim])
    return fail(SU3_ERR_INVALID, "planes [%d, %d) outside 0..%d of dimension %d", plane0, plane0 + nplanes, f->d.L[dim], dim);
  *bytes = (size_t)(f->volume / f->d.L[dim]) * (size_t)nplanes * f->d.n_lorentz * f->ncomp * 2 * f->d.prec;
  return SU3_OK;
}

static void face_side(su3::FaceSide *g, const su3_field *f, bool packed, int plane0) {
  g->packed = packed ? 1 : 0;
  g->plane0 = plane0;
  g->W = f->d.W;
  g->nl = f->d.n_lorentz;
  for (int k = 0; k < 4; k++) {
    g->L[k] = f->d.L[k];
    g->simd[k] = f->d.simd[k];
  }
}

// geo = the field whose descriptor defines the face; dpacked / spacked say which side is the plane-order buffer
static su3_status launch_face_copy(const su3_field *geo, void *dst, bool dpacked, int dplane0, const void *src, bool spacked,
                                   int splane0, int dim, int nplanes, void *stream) {
  su3::FaceParams p;
  memset(&p, 0, sizeof p);
  p.dst = dst; p.src = src; p.dim = dim;
  face_side(&p.d, geo, dpacked, dplane0);
  face_side(&p.s, geo, spacked, splane0);
  long long n = 1;
  for (int k = 0; k < 4; k++) {
    p.F[k] = k == dim ? nplanes : geo->d.L[k];
    n *= p.F[k];
  }
  p.ncplx = n * geo->d.n_lorentz * geo->ncomp;
  if (p.ncplx == 0) return SU3_OK;
  // 32-bit indices when every complex index of the field (and a grid stride beyond the face) fits 31 bits
  const bool idx32 = (geo->nmat + 1) * geo->ncomp * geo->d.W < 0x3fffffffLL && p.ncplx < 0x3fffffffLL;
  su3tab::launch_face(geo->d.prec, geo->ncomp, idx32, flat_grid((size_t)p.ncplx, 1024, 8), p, (cudaStream_t)stream);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("su3_face launch", e);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SU3_OK;
}

// The packed buffer is a raw pointer, not a handle: ask the runtime where it lives (as su3_field_wrap does for fields).
// Plain device memory of ANOTHER device that the current one cannot reach as a peer would fault asynchronously inside
// the kernel; it is refused here instead.  Anything the runtime cannot classify (no device, unregistered host memory)
// and pinned / managed memory pass: their residency is the caller's business.
static su3_status face_buffer_reachable(const void *buf) {
  cudaPointerAttributes at;
  int cur = 0;
  if (cudaPointerGetAttributes(&at, buf) == cudaSuccess && at.type == cudaMemoryTypeDevice && cudaGetDevice(&cur) == cudaSuccess &&
      at.device != cur) {
    int can = 0;
    if (cudaDeviceCanAccessPeer(&can, cur, at.device) != cudaSuccess || !can) {
      (void)cudaGetLastError();
      return fail(SU3_ERR_MISMATCH, "the face buffer is memory of device %d, which device %d (current) cannot access as a peer", at.device, cur);
    }
  }
  (void)cudaGetLastError();
  return SU3_OK;
}

su3_status su3_face_bytes(const su3_field *f, int dim, int nplanes, size_t *nbytes) {
  if (!nbytes) return fail(SU3_ERR_NULL, "nbytes is NULL");
  return face_args(f, dim, 0, nplanes, nbytes);
}

su3_status su3_face_pack(void *buf_dev, size_t buf_bytes, const su3_field *x, int dim, int plane0, int nplanes, void *stream) {
  size_t need = 0;
  if (su3_status st = face_args(x, dim, plane0, nplanes, &need)) return st;
  if (!buf_dev) return fail(SU3_ERR_NULL, "buffer pointer is NULL");
  if ((uintptr_t)buf_dev % 16) return fail(SU3_ERR_ALIGN, "face buffer is not 16-byte aligned");
  if (buf_bytes < need) return fail(SU3_ERR_SIZE, "face buffer has %zu bytes, the face needs %zu", buf_bytes, need);
  if (su3_status sd = on_current_device({x})) return sd;
  if (su3_status sb = face_buffer_reachable(buf_dev)) return sb;
  return launch_face_copy(x, buf_dev, true, 0, x->ptr, false, plane0, dim, nplanes, stream);
}

su3_status su3_face_unpack(su3_field *z, const void *buf_dev, size_t buf_bytes, int dim, int plane0, int nplanes, void *stream) {
  size_t need = 0;
  if (su3_status st = face_args(z, dim, plane0, nplanes, &need)) return st;
  if (!buf_dev) return fail(SU3_ERR_NULL, "buffer pointer is NULL");
  if ((uintptr_t)buf_dev % 16) return fail(SU3_ERR_ALIGN, "face buffer is not 16-byte aligned");
  if (buf_bytes < need) return fail(SU3_ERR_SIZE, "face buffer has %zu bytes, the face needs %zu", buf_bytes, need);
  if (su3_status sd = on_current_device({z})) return sd;
  if (su3_status sb = face_buffer_reachable(buf_dev)) return sb;
  return launch_face_copy(z, z->ptr, false, plane0, buf_dev, true, 0, dim, nplanes, stream);
}

su3_status su3_face_copy(su3_field *z, int z_plane0, const su3_field *x, int x_plane0, int dim, int nplanes, void *stream) {
  size_t need = 0;
  if (su3_status st = face_args(z, dim, z_plane0, nplanes, &need)) return st;
  if (su3_status st = face_args(x, dim, x_plane0, nplanes, &need)) return st;
  if (!same_desc(z->d, x->d) || z->ncomp != x->ncomp) return fail(SU3_ERR_MISMATCH, "su3_face_copy needs identical descriptors and field kinds");
  if (z->ptr == x->ptr) return fail(SU3_ERR_MISMATCH, "su3_face_copy: z and x must be different fields");
  if (su3_status sd = on_current_device({z})) return sd;  // x may be peer memory: only the destination must be local
  return launch_face_copy(z, z->ptr, false, z_plane0, x->ptr, false, x_plane0, dim, nplanes, stream);
}

// ---------------------------------------------------------------- face move for callers that cannot allocate
// The packed staging buffer of the pack -> unpack route, owned by the library's device image instead of the caller
// (su3stream.h says who needs that and why).  File scope, so each device that loads this module holds its own 16 MiB
// copy until the process exits; uninitialised (.nv.global is NOBITS: the .so does not grow).
static __device__ __align__(256) unsigned char g_static_scratch[SU3_STATIC_SCRATCH_BYTES];

// Device address of g_static_scratch on the device that is current on the calling thread.  In host code the array's
// name is only the runtime's handle for the symbol -- not an address a kernel may be given -- so the address is asked
// for once per device ordinal, with that device current, and cached.  A failed look-up is not cached.
static su3_status static_scratch_ptr(void **out) {
  static void *table[MAX_DEVICES];  // zero-initialised: NULL = not looked up yet
  static std::mutex mu;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail("cudaGetDevice", e);
  if (dev < 0 || dev >= MAX_DEVICES) return fail(SU3_ERR_CUDA, "device ordinal %d outside 0..%d", dev, MAX_DEVICES - 1);
  std::lock_guard<std::mutex> lk(mu);
  if (!table[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess) return cuda_fail("cudaGetSymbolAddress(static face scratch)", e);
    if (!p || (uintptr_t)p % 256) return fail(SU3_ERR_CUDA, "static face scratch resolved to an unusable address %p", p);
    table[dev] = p;
  }
  *out = table[dev];
  return SU3_OK;
}

su3_status su3_face_move_static(su3_field *z, int z_plane0, const su3_field *x, int x_plane0, int dim, int nplanes,
                                void *stream) {
  size_t need = 0, need_x = 0;
  if (su3_status st = face_args(z, dim, z_plane0, nplanes, &need)) return st;
  if (su3_status st = face_args(x, dim, x_plane0, nplanes, &need_x)) return st;
  if (!same_lattice(z->d, x->d) || z->ncomp != x->ncomp)
    return fail(SU3_ERR_MISMATCH, "su3_face_move_static needs fields of one lattice, precision and kind (layouts may differ)");
  if (need > (size_t)SU3_STATIC_SCRATCH_BYTES)
    return fail(SU3_ERR_SIZE, "the face has %zu bytes, the library's static staging area holds %zu: move fewer planes per call, "
                "or use su3_face_pack / su3_face_unpack with a buffer of your own", need, (size_t)SU3_STATIC_SCRATCH_BYTES);
  if (su3_status sd = on_current_device({z, x})) return sd;
  void *area = nullptr;
  if (su3_status st = static_scratch_ptr(&area)) return st;  // first call on this device: the one-time address look-up
  // field -> area (plane order), then area -> field.  Stream order makes the second launch see the first one's bytes;
  // every byte it reads is one the first launch wrote, so what an earlier call left in the area never matters.
  if (su3_status st = launch_face_copy(x, area, true, 0, x->ptr, false, x_plane0, dim, nplanes, stream)) return st;
  return launch_face_copy(z, z->ptr, false, z_plane0, area, true, 0, dim, nplanes, stream);
}

su3_status su3_eval_host(int op, void *z_host, const void *x_host, const void *y_host, const void *u_host,
                         su3_field *zd, su3_field *xd, su3_field *yd, su3_field *ud, int chunks, void *cuda_stream) {
  if (op != SU3_OP_MUL && op != SU3_OP_MUL3 && op != SU3_OP_MUL_ADD) return fail(SU3_ERR_INVALID, "op = %d not in {0,1,2}", op);
  const bool has_u = op != SU3_OP_MUL;
  su3_status st = check_arith(zd, xd, yd, ud, has_u);
  if (st != SU3_OK) return st;
  if (!has_u && (u_host || ud)) return fail(SU3_ERR_INVALID, "SU3_OP_MUL takes no third operand");
  if ((st = on_current_device({zd, xd, yd, ud})) != SU3_OK) return st;
  const DevInfo &di = devinfo();
  cudaStream_t user = (cudaStream_t)cuda_stream;
  const int W = zd->d.W, prec = zd->d.prec;
  const int64_t nmat = zd->nmat;
  const size_t mat_bytes = (size_t)18 * prec;
  // chunk boundaries: multiples of 2*W matrices keep every chunk 16-byte aligned and lane-complete
  const int64_t gran = 2 * (int64_t)W;
  if (chunks > MAX_HOST_CHUNKS) return fail(SU3_ERR_INVALID, "chunks = %d exceeds %d", chunks, MAX_HOST_CHUNKS);
  if (chunks <= 0) chunks = 8;
  int64_t per = (nmat + chunks - 1) / chunks;
  per = (per + gran - 1) / gran * gran;
  if (per < gran) per = gran;
  const int64_t nchunks = nmat ? (nmat + per - 1) / per : 0;
  HostPipe *hp = host_pipe(di.dev, user);
  if (!hp) return fail(SU3_ERR_SIZE, "more than %zu distinct (device, stream) pairs hold host pipelines; call su3_host_release()", MAX_HOST_PIPES);
  HostPipe &g_hp = *hp;  // this (device, stream)'s resources
  std::lock_guard<std::mutex> lk(g_hp.mu);
  cudaError_t e = g_hp.ensure((size_t)(2 * nchunks + 2));
  if (e != cudaSuccess) return cuda_fail("su3_eval_host stream/event setup", e);
  cudaEvent_t ev_start = g_hp.ev[0], ev_done = g_hp.ev[1];
#define SU3_CK(call)                                         \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return cuda_fail(#call, e_);      \
  } while (0)
  SU3_CK(cudaEventRecord(ev_start, user));
  SU3_CK(cudaStreamWaitEvent(g_hp.h2d, ev_start, 0));
  SU3_CK(cudaStreamWaitEvent(g_hp.d2h, ev_start, 0));
  for (int64_t c = 0; c < nchunks; c++) {
    const int64_t m0 = c * per;
    const int64_t nm = (nmat - m0 < per) ? nmat - m0 : per;
    const size_t off = (size_t)m0 * mat_bytes, len = (size_t)nm * mat_bytes;
    cudaEvent_t ev_in = g_hp.ev[2 + 2 * c], ev_k = g_hp.ev[3 + 2 * c];
    if (x_host) SU3_CK(cudaMemcpyAsync((char *)xd->ptr + off, (const char *)x_host + off, len, cudaMemcpyHostToDevice, g_hp.h2d));
    if (y_host) SU3_CK(cudaMemcpyAsync((char *)yd->ptr + off, (const char *)y_host + off, len, cudaMemcpyHostToDevice, g_hp.h2d));
    if (u_host) SU3_CK(cudaMemcpyAsync((char *)ud->ptr + off, (const char *)u_host + off, len, cudaMemcpyHostToDevice, g_hp.h2d));
    SU3_CK(cudaEventRecord(ev_in, g_hp.h2d));
    SU3_CK(cudaStreamWaitEvent(user, ev_in, 0));
    const void *in[4] = {(const char *)xd->ptr + off, (const char *)yd->ptr + off, has_u ? (const char *)ud->ptr + off : nullptr, nullptr};
    st = launch_stream(op, prec, W, (char *)zd->ptr + off, in, nm, (has_u ? 4 : 3) * zd->nbytes, user, nullptr, /*one_shot=*/true);
    if (st != SU3_OK) return st;
    SU3_CK(cudaEventRecord(ev_k, user));
    SU3_CK(cudaStreamWaitEvent(g_hp.d2h, ev_k, 0));
    if (z_host) SU3_CK(cudaMemcpyAsync((char *)z_host + off, (const char *)zd->ptr + off, len, cudaMemcpyDeviceToHost, g_hp.d2h));
  }
  SU3_CK(cudaEventRecord(ev_done, g_hp.d2h));
  SU3_CK(cudaStreamWaitEvent(user, ev_done, 0));
#undef SU3_CK
  return SU3_OK;
}

su3_status su3_mul_host(void *z_host, const void *x_host, const void *y_host, su3_field *zd, su3_field *xd,
                        su3_field *yd, int chunks, void *cuda_stream) {
  if (!z_host || !x_host || !y_host) return fail(SU3_ERR_NULL, "host pointer is NULL");
  return su3_eval_host(SU3_OP_MUL, z_host, x_host, y_host, nullptr, zd, xd, yd, nullptr, chunks, cuda_stream);
}

su3_status su3_host_release(void) {
  std::map<std::pair<int, cudaStream_t>, std::unique_ptr<HostPipe>> old;
  {
    std::lock_guard<std::mutex> lk(g_hp_mu);
    old.swap(g_hp);
  }
  int cur = 0;
  const bool have = cudaGetDevice(&cur) == cudaSuccess;
  for (auto &kv : old) {
    std::lock_guard<std::mutex> lk(kv.second->mu);
    if (have) cudaSetDevice(kv.first.first);
    kv.second->destroy();
  }
  if (have) cudaSetDevice(cur);
  (void)cudaGetLastError();
  return SU3_OK;
}

su3_status su3_launch_plan(const su3_desc *desc, int op, char *buf, size_t buf_len) {
  if (!buf || buf_len == 0) return fail(SU3_ERR_NULL, "buf is NULL or empty");
  if (op != SU3_OP_MUL && op != SU3_OP_MUL3 && op != SU3_OP_MUL_ADD) return fail(SU3_ERR_INVALID, "op = %d not in {0,1,2}", op);
  su3_desc d;
  if (su3_status st = normalize(desc, &d)) return st;
  const DevInfo &di = devinfo();
  if (!di.ok) return fail(SU3_ERR_CUDA, "%s", di.err);
  const int64_t nmat = volume_of(d) * d.n_lorentz;
  const size_t field = (size_t)nmat * 18 * d.prec;
  const int kop = op == SU3_OP_MUL ? su3::OP_MUL : (op == SU3_OP_MUL3 ? su3::OP_MUL3 : su3::OP_MUL_ADD);
  StreamPlan pl;
  if (su3_status st = plan_stream(kop, d.prec, d.W, nmat, field * (op == SU3_OP_MUL ? 3 : 4), false, false, g_tune, di, &pl)) return st;
  const char *fam = pl.family == su3tab::FAM_WARP ? "warp" : (pl.family == su3tab::FAM_DIRECT ? "direct" : "pipe");
  const char *l2 = pl.hint == 2 ? "pin" : (pl.hint == 1 ? "evict_first" : "none");
  const int n = snprintf(buf, buf_len, "%s tile=%d depth=%d ctas=%d grid=%u block=%d smem=%zu l2=%s pin_bytes=%zu", fam, pl.tile_mats,
                         pl.stages, pl.ctas, pl.grid, pl.block, pl.smem, l2, pl.pin_bytes);
  if (n < 0 || (size_t)n >= buf_len) return fail(SU3_ERR_SIZE, "plan needs %d bytes, buf has %zu", n + 1, buf_len);
  return SU3_OK;
}

su3_status su3_tune_set(const su3_tune *t) {
  su3_tune v = {0, 0, 0, 0, 0, 0, {0, 0}};
  if (t) v = *t;
  if (v.tile_mats != 0 && v.tile_mats != 32 && v.tile_mats != 64 && v.tile_mats != 128)
    return fail(SU3_ERR_INVALID, "tile_mats = %d not in {0,32,64,128}", v.tile_mats);
  if (v.stages != 0 && (v.stages < 2 || v.stages > 16)) return fail(SU3_ERR_INVALID, "stages = %d outside 2..16", v.stages);
  if (v.ctas_per_sm < 0 || v.ctas_per_sm > 8) return fail(SU3_ERR_INVALID, "ctas_per_sm = %d outside 0..8", v.ctas_per_sm);
  if (v.l2_hint < 0 || v.l2_hint > 3) return fail(SU3_ERR_INVALID, "l2_hint = %d outside 0..3", v.l2_hint);
  if (v.l2_pin_mb < 0) return fail(SU3_ERR_INVALID, "l2_pin_mb = %d is negative", v.l2_pin_mb);
  if (v.path < 0 || v.path > 3) return fail(SU3_ERR_INVALID, "path = %d outside 0..3", v.path);
  g_tune = v;
  return SU3_OK;
}

su3_status su3_tune_get(su3_tune *out) {
  if (!out) return fail(SU3_ERR_NULL, "out is NULL");
  *out = g_tune;
  return SU3_OK;
}

int64_t su3_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

su3_status su3_device_name(char *buf, size_t buf_len, int32_t *ordinal) {
  if (!buf || buf_len == 0) return fail(SU3_ERR_NULL, "buf is NULL or empty");
  const DevInfo &di = devinfo();
  if (!di.ok) return fail(SU3_ERR_CUDA, "%s", di.err);
  snprintf(buf, buf_len, "%s", di.name);
  if (ordinal) *ordinal = di.dev;
  return SU3_OK;
}

su3_status su3_device_info(int32_t *sm_count, int64_t *l2_bytes, int32_t *mem_clock_khz, int32_t *bus_width_bits) {
  const DevInfo &di = devinfo();
  if (!di.ok) return fail(SU3_ERR_CUDA, "%s", di.err);
  if (sm_count) *sm_count = di.sms;
  if (l2_bytes) *l2_bytes = di.l2;
  if (mem_clock_khz) *mem_clock_khz = di.mem_khz;
  if (bus_width_bits) *bus_width_bits = di.bus_bits;
  return SU3_OK;
}

}  // extern "C"

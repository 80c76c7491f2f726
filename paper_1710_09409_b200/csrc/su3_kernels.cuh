// su3_kernels.cuh -- sm_100a device code of libsu3stream.
//
// Hot path of arXiv:1710.09409 section 4/5 (Listing 3):
// the lattice-wide, site-wise complex 3x3 product z = x*y and the fused one-pass
// expressions z = x*y*w, z = x*y + v, in the scalar (AoS) and the
// lane-interleaved vector layout, plus the layout permutation (extract/merge) and the
// streaming ceilings.  No code is shared with oracle/ (the CPU checker).
//
// Design: every field is a flat byte stream of records.  A record
// of the vector layout with W lanes is 9 element-vectors of W complex numbers; the
// scalar layout is the W = 1 case.  The arithmetic kernels are HBM-bound (0.46-1.4
// flop/byte), so the kernel is a persistent, warp-specialised streaming pipeline:
//
//   producer warp (1 elected lane)          consumer warps (1 thread = 1 matrix)
//   -------------------------------         ------------------------------------
//   wait  empty[s]                          wait  full[s]
//   cp.async.bulk  x,y(,u) tile -> smem     LDS   own matrix of x, y(, u)   (conflict-free)
//   (TMA 1-D bulk copy, mbarrier tx)        FMA   27 (54) complex multiply-adds in registers
//                                           STS   z into the x slot, fence.proxy.async
//                                           bar   consumers only
//                                           cp.async.bulk  smem -> z tile   (1 thread)
//                                           arrive empty[s-1] once its store has read smem
//
// A tile is a CONTIGUOUS byte range of every operand (T matrices = T*144 B fp64 / T*72 B
// fp32), so the 144/72-byte AoS records reach HBM as full-line bulk transactions whatever
// the layout; the layout only changes the shared-memory index of a thread's matrix.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace su3 {


// ---------------------------------------------------------------- complex helpers
template <typename R> struct Cplx;
template <> struct Cplx<float> { typedef float2 type; };
template <> struct Cplx<double> { typedef double2 type; };

__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float fma_rn(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double fma_rn(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }

// c = a.b, c_ij = sum_k a_ik b_kj (S7), k ascending, as a fixed chain of
// round-to-nearest FMAs.  Written with intrinsics so that every kernel that inlines it
// (scalar or vector layout, staged or direct path) produces bit-identical results.
template <typename C2>
__device__ __forceinline__ void mat33_mul(const C2 (&a)[9], const C2 (&b)[9], C2 (&c)[9]) {
#pragma unroll
  for (int i = 0; i < 3; i++) {
#pragma unroll
    for (int j = 0; j < 3; j++) {
      auto re = mul_rn(a[3 * i].x, b[j].x);
      auto im = mul_rn(a[3 * i].x, b[j].y);
      re = fma_rn(-a[3 * i].y, b[j].y, re);
      im = fma_rn(a[3 * i].y, b[j].x, im);
#pragma unroll
      for (int k = 1; k < 3; k++) {
        re = fma_rn(a[3 * i + k].x, b[3 * k + j].x, re);
        im = fma_rn(a[3 * i + k].x, b[3 * k + j].y, im);
        re = fma_rn(-a[3 * i + k].y, b[3 * k + j].y, re);
        im = fma_rn(a[3 * i + k].y, b[3 * k + j].x, im);
      }
      c[3 * i + j].x = re;
      c[3 * i + j].y = im;
    }
  }
}

// ---------------------------------------------------------------- PTX wrappers (sm_90+/sm_100a)
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
// TMA 1-D bulk copy global -> shared, completion on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar,
                                              uint64_t pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst_smem)),
      "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
      : "memory");
}
// TMA 1-D bulk copy shared -> global, bulk async-group completion.
__device__ __forceinline__ void bulk_s2g(void *dst_gmem, const void *src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_s2g_hint(void *dst_gmem, const void *src_smem, uint32_t bytes, uint64_t pol) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dst_gmem),
               "r"(smem_u32(src_smem)), "r"(bytes), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() {
  asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
template <int N> __device__ __forceinline__ void bulk_wait_all() {
  asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory");
}
// 8-byte asynchronous copy global -> shared (LDGSTS) and its completion as an arrival on an mbarrier
__device__ __forceinline__ void cp_async8(void *dst_smem, const void *src_gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_arrive_noinc(uint64_t *bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ---------------------------------------------------------------- the streaming pipeline (A1-A4, menu programs, shifts)
// Register-machine instructions shared by the ahead-of-time menu below and by the interpreter (su3_expr_kernel):
// sources 0..7 = operand slot of the stage, 8..15 = temporary, 255 = accumulator; the result goes to the accumulator;
// `spill` parks the accumulator in a temporary first.
enum { EX_MUL = 0, EX_ADD = 1, EX_SUB = 2, EX_COPY = 3, EX_EMUL = 4,  // EMUL: element-wise product of the reals (real scalar fields)
       EX_SRC_ACC = 255, EX_NONE = 255, EX_TEMP0 = 8 };
struct ExprIns {
  unsigned char op, a, b, spill;
};

// The ahead-of-time menu: small programs compiled INTO the pipeline kernel (template parameter OP), so that the whole
// tree is evaluated in registers by straight-line code (the expression is evaluated inside the one site loop;
// this is the ahead-of-time counterpart of the paper's Jitify back-end).  su3_expr matches a compiled program
// against these rows (up to a renaming of the operands and the order of the two sources of '+') and runs the
// interpreter only for programs that are not on the menu.  Rows 0-3 are su3_mul, su3_mul3, su3_mul_add, su3_add.
enum { OP_MUL = 0, OP_MUL3 = 1, OP_MUL_ADD = 2, OP_ADD = 3,
       OP_SUM_PROD = 4,     // a + b + a*b        "01+01*+"   (the paper's Listing 2 on matrices)
       OP_MUL_MUL_ADD = 5,  // a*b + c*d          "01*23*+"
       OP_MUL_MUL_SUB = 6,  // a*b - c*d          "01*23*-"
       OP_MUL_SUB = 7,      // a*b - c            "01*2-"
       OP_ADD3 = 8,         // a + b + c          "01+2+"
       OP_ADD4 = 9,         // a + b + c + d      "01+2+3+"
       OP_SUB = 10,         // a - b              "01-"
       OP_EMUL = 11,        // reals: a*b         "01*" on real scalar fields
       OP_SUM_EPROD = 12,   // reals: a + b + a*b "01+01*+" on real scalar fields (Listing 2 itself)
       OP_MUL4 = 13,        // a*b*c*d            "01*2*3*"   products of three and four matrices in every association:
       OP_MUL_R = 14,       // a*(b*c)            "012**"     the shapes of plaquette-like expressions
       OP_MULMUL_MUL = 15,  // (a*b)*(c*d)        "01*23**"
       OP_COPY = 16,        // z = a (only used with a shifted operand: Cshift)
       OP_COUNT = 17 };
struct MenuProg {
  int nin, nins, min_ctas;  // operands, instructions, resident CTAs per SM the registers must allow
  ExprIns ins[4];
};
__host__ __device__ constexpr MenuProg menu_prog(int op) {
  constexpr unsigned char A = EX_SRC_ACC, N = EX_NONE, T = EX_TEMP0;
  switch (op) {
    case OP_MUL: return {2, 1, 3, {{EX_MUL, 0, 1, N}}};
    case OP_MUL3: return {3, 2, 3, {{EX_MUL, 0, 1, N}, {EX_MUL, A, 2, N}}};
    case OP_MUL_ADD: return {3, 2, 3, {{EX_MUL, 0, 1, N}, {EX_ADD, A, 2, N}}};
    case OP_ADD: return {2, 1, 3, {{EX_ADD, 0, 1, N}}};
    case OP_SUM_PROD: return {2, 3, 2, {{EX_ADD, 0, 1, N}, {EX_MUL, 0, 1, T}, {EX_ADD, T, A, N}}};
    case OP_MUL_MUL_ADD: return {4, 3, 2, {{EX_MUL, 0, 1, N}, {EX_MUL, 2, 3, T}, {EX_ADD, T, A, N}}};
    case OP_MUL_MUL_SUB: return {4, 3, 2, {{EX_MUL, 0, 1, N}, {EX_MUL, 2, 3, T}, {EX_SUB, T, A, N}}};
    case OP_MUL_SUB: return {3, 2, 3, {{EX_MUL, 0, 1, N}, {EX_SUB, A, 2, N}}};
    case OP_ADD3: return {3, 2, 3, {{EX_ADD, 0, 1, N}, {EX_ADD, A, 2, N}}};
    case OP_ADD4: return {4, 3, 2, {{EX_ADD, 0, 1, N}, {EX_ADD, A, 2, N}, {EX_ADD, A, 3, N}}};
    case OP_SUB: return {2, 1, 3, {{EX_SUB, 0, 1, N}}};
    case OP_EMUL: return {2, 1, 3, {{EX_EMUL, 0, 1, N}}};
    case OP_SUM_EPROD: return {2, 3, 3, {{EX_ADD, 0, 1, N}, {EX_EMUL, 0, 1, T}, {EX_ADD, T, A, N}}};
    case OP_MUL4: return {4, 3, 2, {{EX_MUL, 0, 1, N}, {EX_MUL, A, 2, N}, {EX_MUL, A, 3, N}}};
    case OP_MUL_R: return {3, 2, 3, {{EX_MUL, 1, 2, N}, {EX_MUL, 0, A, N}}};
    case OP_MULMUL_MUL: return {4, 3, 2, {{EX_MUL, 0, 1, N}, {EX_MUL, 2, 3, T}, {EX_MUL, T, A, N}}};
    case OP_COPY: return {1, 1, 3, {{EX_COPY, 0, N, N}}};
  }
  return {0, 0, 1, {}};
}

// A shifted operand (f3): the LAST operand of the program is read at site s + disp*dim_hat.  In storage order a
// tile's sources are a few CONTIGUOUS runs of whole records: with oc = the outer coordinate of a record in the shifted
// dimension, records with oc + dmod < rd come from record + dmod*P, the others ("carry": they wrap around the
// sub-lattice) from record + (dmod - rd)*P, and oc advances every P = ostride*nl records.  The producer moves every
// run with one bulk copy; a consumer thread then reads its matrix from lane (ic + qrot + carry) mod simd_d instead of
// its own lane ic: across the sub-lattice boundary a shift is a lane rotation (the virtual-node map S3).
struct ShiftInfo {
  long long P;     // records per step of oc: prod_{k<dim} r[k] * n_lorentz
  int rd;          // r[dim] = L[dim] / simd[dim]
  int dmod, qrot;  // disp = qrot*rd + dmod, 0 <= disp < L[dim]
  int simd_d, lstride;  // simd[dim], prod_{k<dim} simd[k]
  int phase;       // fp32 scalar layout only: byte offset (0 or 8) of the shifted slot that makes source and destination
                   // of every run agree mod 16 (records are 72 B; bulk copies need 16-byte alignment)
  // su3_cshift_bulk_kernel on a slab of a multi-GPU lattice (su3_cshift_slab): the runs that leave the slab -- the
  // carry runs for disp > 0 (alt_carry = 1), the others for disp < 0 (alt_carry = 0) -- are read at the same record
  // offset from the NEIGHBOURING rank's slab `alt` (peer memory over NVLink, or local); NULL: periodic on the slab
  const void *alt;
  int alt_carry;
};

struct StreamParams {
  void *z;
  const void *x;
  const void *y;
  const void *u;   // third operand: w (OP_MUL3) or v (OP_MUL_ADD); unused for OP_MUL
  const void *v;   // fourth operand of the menu programs with four inputs
  long long nmat;  // matrices in the range handled by this launch (multiple of W)
  int tile_mats;   // matrices per tile: multiple of 32 (hence of W), <= NCW*32
  int stages;      // ring depth >= 2
  int hint;        // 0 none; 1: L2 evict_first on loads and stores; 2: loads of the first pin_tiles tiles evict_last
                   // (kept in L2 from one call to the next: Listing 3 repeats z = x*y on the same fields), rest evict_first
  long long pin_tiles;
  ShiftInfo sh;    // SHIFT kernels only
};

template <int OP> struct NumInputs { static const int value = menu_prog(OP).nin; };

__device__ __forceinline__ uint64_t policy_evict_last() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}

// straight-line evaluation of menu program OP for one matrix: src[k] points at element 0 of the thread's matrix in
// operand slot k (element e at src[k][e*W]); unrolled at compile time, so every source index is a constant
template <int OP, int I, int W, typename C2, int NIN>
__device__ __forceinline__ void menu_step(const C2 *const (&src)[NIN], C2 (&acc)[9], C2 (&t0)[9]) {
  constexpr MenuProg P = menu_prog(OP);
  if constexpr (I < P.nins) {
    constexpr ExprIns in = P.ins[I];
    static_assert(in.spill == EX_NONE || in.spill == EX_TEMP0, "menu programs use at most one temporary");
    if constexpr (in.spill != EX_NONE) {
#pragma unroll
      for (int e = 0; e < 9; e++) t0[e] = acc[e];
    }
    C2 a[9], b[9];
#pragma unroll
    for (int e = 0; e < 9; e++) {
      if constexpr (in.a == EX_SRC_ACC) a[e] = acc[e];
      else if constexpr (in.a == EX_TEMP0) a[e] = t0[e];
      else a[e] = src[in.a][e * W];
    }
    if constexpr (in.op != EX_COPY) {
#pragma unroll
      for (int e = 0; e < 9; e++) {
        if constexpr (in.b == EX_SRC_ACC) b[e] = acc[e];
        else if constexpr (in.b == EX_TEMP0) b[e] = t0[e];
        else b[e] = src[in.b][e * W];
      }
    }
    if constexpr (in.op == EX_MUL) {
      mat33_mul(a, b, acc);
    } else {
#pragma unroll
      for (int e = 0; e < 9; e++) {
        if constexpr (in.op == EX_ADD) {
          acc[e].x = add_rn(a[e].x, b[e].x);
          acc[e].y = add_rn(a[e].y, b[e].y);
        } else if constexpr (in.op == EX_SUB) {
          acc[e].x = add_rn(a[e].x, -b[e].x);
          acc[e].y = add_rn(a[e].y, -b[e].y);
        } else if constexpr (in.op == EX_EMUL) {
          acc[e].x = mul_rn(a[e].x, b[e].x);
          acc[e].y = mul_rn(a[e].y, b[e].y);
        } else {
          acc[e] = a[e];
        }
      }
    }
    menu_step<OP, I + 1, W>(src, acc, t0);
  }
}

// One thread's matrix: element e of lane l of record q sits at complex index (q*9 + e)*W + l
// of the slot.  Thread t owns (q = t / W, l = t % W).  Bank check: with
// 16-byte (fp64) or 8-byte (fp32) complex numbers every quarter-/half-warp request covers
// all 32 banks exactly once for every W in {1,2,4,8,16,32}.
// Stage layout: NSLOT operand slots of tile_mats*9 complex numbers (+16 bytes of slack for the phase of a shifted
// slot).  The result is written over slot 0 and leaves by a bulk store; for OP_COPY with SHIFT the shifted operand
// sits in slot 1 (a thread reads ANOTHER lane's matrix there, so it must not overwrite the slot it reads).
template <typename R, int W, int OP, int NCW, int SHIFT>
__global__ void __launch_bounds__((NCW + 1) * 32, menu_prog(OP).min_ctas) su3_pipe_kernel(const StreamParams p) {
  typedef typename Cplx<R>::type C2;
  constexpr int NIN = NumInputs<OP>::value;
  constexpr int NSLOT = (SHIFT && NIN == 1) ? 2 : NIN;
  constexpr int FIRST = NSLOT - NIN;  // slot of operand 0
  constexpr int CB = (int)sizeof(C2);
  // 72-byte records (fp32, scalar layout): a run of the shifted operand may start / end on an 8-byte boundary; those 8
  // bytes travel by cp.async (LDGSTS), whose completion is the SECOND arrival every phase of full[s] then waits for
  constexpr bool FIX8 = SHIFT && CB == 8 && W == 1;
  extern __shared__ __align__(128) unsigned char smem[];

  const int TM = p.tile_mats;
  const int S = p.stages;
  const uint32_t slot_bytes = (uint32_t)TM * 9u * CB;
  const uint32_t stage_bytes = NSLOT * slot_bytes + (SHIFT ? 16u : 0u);
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)S * stage_bytes);
  uint64_t *empty = full + S;
  int2 *tinfo = reinterpret_cast<int2 *>(empty + S);  // SHIFT: per stage (oc, record offset inside its P-block) of the tile's first record

  const int tid = threadIdx.x;
  const long long ntiles = (p.nmat + TM - 1) / TM;

  if (tid == 0) {
    for (int s = 0; s < S; s++) {
      mbar_init(&full[s], FIX8 ? 33 : 1);  // FIX8: + one cp.async arrival per producer lane
      mbar_init(&empty[s], 1);
    }
    fence_mbar_init();
    fence_proxy_async();
  }
  __syncthreads();

  if (tid >= NCW * 32) {
    // ------------------------------------------------ producer: one elected lane issues the TMA bulk loads; the runs of a
    // shifted operand are issued by the whole producer warp, lane k taking the k-th run of the tile (closed form: run
    // boundaries sit at blocks cyc + {0, rd - dmod} of every cycle of rd blocks) -- a shift along the fastest dimension
    // has 5-6 runs per tile.  With FIX8 a run may also need 8-byte head / tail copies (cp.async): every producer lane then
    // arrives on the stage's mbarrier once its own cp.async copies have landed (33 arrivals per phase).
    constexpr bool PAR = SHIFT;
    const int plane = tid - NCW * 32;
    if (plane == 0 || PAR) {
      const unsigned char *src[4] = {(const unsigned char *)p.x, (const unsigned char *)p.y,
                                     (const unsigned char *)p.u, (const unsigned char *)p.v};
      uint64_t pol = 0, pol_keep = 0;
      if (p.hint) pol = policy_evict_first();
      if (p.hint == 2) pol_keep = policy_evict_last();
      int s = 0;
      uint32_t ph = 0;
      for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        mbar_wait(&empty[s], ph ^ 1u);
        const long long m0 = tile * TM;
        const long long left = p.nmat - m0;
        const int nm = left < TM ? (int)left : TM;
        const uint32_t bytes = (uint32_t)nm * 9u * CB;
        const uint32_t b16 = bytes & ~15u;  // bulk copies move multiples of 16 bytes
        unsigned char *st = smem + (size_t)s * stage_bytes;
        const size_t goff = (size_t)m0 * 9u * CB;
        const uint64_t tpol = (p.hint == 2 && tile < p.pin_tiles) ? pol_keep : pol;
        constexpr int NPLAIN = SHIFT ? NIN - 1 : NIN;  // operands that are read at the site itself
        if (plane == 0 && bytes != b16) {  // fp32 with an odd matrix count: 8 trailing bytes per operand
#pragma unroll
          for (int o = 0; o < NPLAIN; o++)
            *reinterpret_cast<uint64_t *>(st + (FIRST + o) * slot_bytes + b16) =
                *reinterpret_cast<const uint64_t *>(src[o] + goff + b16);
        }
        uint32_t total = NPLAIN * b16;
        if (SHIFT) {
          // the shifted operand: runs of whole records [Ra, Rb) whose sources are contiguous.  Record indices fit 31 bits
          // (checked by the host), so the run arithmetic is 32-bit; only byte offsets are 64-bit.
          const unsigned char *gy = src[NIN - 1];
          unsigned char *sy = st + (NSLOT - 1) * slot_bytes + p.sh.phase;
          const int P = (int)p.sh.P, rd = p.sh.rd, dmod = p.sh.dmod;
          const int R0 = (int)(m0 / W), R1 = (int)((m0 + nm) / W);
          constexpr uint32_t rb = 9u * W * CB;  // bytes per record
          int blk = R0 / P;
          int oc = blk % rd;
          if (plane == 0) tinfo[s] = make_int2(oc, R0 - blk * P);
          uint32_t mine = 0;  // bytes of my bulk copies
          const int cyc0 = blk - oc;
          for (int m = (oc >= rd - dmod ? 1 : 0) + plane;; m += 32) {
            const long long ba = (long long)(cyc0 + (m >> 1) * rd + ((m & 1) ? rd - dmod : 0)) * P;
            if (ba >= R1) break;
            const long long bb = (long long)(cyc0 + ((m + 1) >> 1) * rd + (((m + 1) & 1) ? rd - dmod : 0)) * P;
            const int Ra = ba > R0 ? (int)ba : R0, Rb = bb < R1 ? (int)bb : R1;
            if (Rb <= Ra) continue;  // dmod = 0: the carry runs are empty
            const long long Rs = (long long)Ra + (long long)((m & 1) ? dmod - rd : dmod) * P;
            const size_t gs = (size_t)Rs * rb, ge = gs + (size_t)(Rb - Ra) * rb;
            unsigned char *d = sy + (size_t)(Ra - R0) * rb;
            size_t gs16 = gs, ge16 = ge;
            if (FIX8) {  // the first / last 8 bytes of a run that is not 16-byte aligned
              gs16 = (gs + 15) & ~(size_t)15;
              ge16 = ge & ~(size_t)15;
              if (gs16 != gs) cp_async8(d, gy + gs);
              if (ge16 != ge && ge16 >= gs16) cp_async8(d + (ge16 - gs), gy + ge16);
            }
            if (ge16 > gs16) {
              mine += (uint32_t)(ge16 - gs16);
              if (p.hint) bulk_g2s_hint(d + (gs16 - gs), gy + gs16, (uint32_t)(ge16 - gs16), &full[s], tpol);
              else bulk_g2s(d + (gs16 - gs), gy + gs16, (uint32_t)(ge16 - gs16), &full[s]);
            }
          }
          if (FIX8) {
            cp_async_arrive_noinc(&full[s]);  // arrives once this lane's cp.async copies have landed (at once if none)
            total += __reduce_add_sync(0xffffffffu, mine);
          } else {
            total += (uint32_t)(R1 - R0) * rb;
          }
        }
        if (plane == 0) {
#pragma unroll
          for (int o = 0; o < NPLAIN; o++) {
            if (p.hint)
              bulk_g2s_hint(st + (FIRST + o) * slot_bytes, src[o] + goff, b16, &full[s], tpol);
            else
              bulk_g2s(st + (FIRST + o) * slot_bytes, src[o] + goff, b16, &full[s]);
          }
          // expect-tx and the producer's arrival: the phase cannot complete before this arrival nor before every byte
          // counted in `total` has landed, whichever lane issues its copy and whenever (the transaction count may be
          // transiently negative until here)
          mbar_arrive_expect_tx(&full[s], total);
        }
        if (++s == S) {
          s = 0;
          ph ^= 1u;
        }
      }
    }
    return;
  }

  // -------------------------------------------------- consumers: one thread per matrix of the tile
  const int t = tid;
  const int base = (t / W) * 9 * W + (t % W);
  uint64_t pol = 0;
  if (p.hint && t == 0) pol = policy_evict_first();
  // SHIFT across virtual nodes: the lane that holds my neighbour, for records that do / do not wrap around the sub-lattice
  int lsrc_plain = t % W, lsrc_carry = t % W;
  if (SHIFT && W > 1 && p.sh.simd_d > 1) {
    const int ic = (lsrc_plain / p.sh.lstride) % p.sh.simd_d;
    lsrc_carry += ((ic + p.sh.qrot + 1) % p.sh.simd_d - ic) * p.sh.lstride;
    lsrc_plain += ((ic + p.sh.qrot) % p.sh.simd_d - ic) * p.sh.lstride;
  }
  int s = 0, prev_s = -1;
  uint32_t ph = 0;
  for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const long long m0 = tile * TM;
    const long long left = p.nmat - m0;
    const int nm = left < TM ? (int)left : TM;
    unsigned char *st = smem + (size_t)s * stage_bytes;
    mbar_wait(&full[s], ph);
    if (t < nm) {
      const C2 *src[NIN];
#pragma unroll
      for (int o = 0; o < NIN; o++) src[o] = reinterpret_cast<const C2 *>(st + (FIRST + o) * slot_bytes) + base;
      if (SHIFT) {
        int lsrc = t % W;
        if (W > 1 && p.sh.simd_d > 1) {  // which lane holds my neighbour: a step across the sub-lattice boundary rotates lanes
          const int2 ti = tinfo[s];
          const int r = ti.y + t / W, P = (int)p.sh.P, rd = p.sh.rd;
          // blocks of P records between the tile's first record and mine: 0 or 1 when a block is at least a tile long
          const int k = P >= TM / W ? (r >= P ? 1 : 0) : r / P;
          int oc = ti.x + k;
          if (oc >= rd) oc = k <= 1 ? oc - rd : oc % rd;
          lsrc = oc + p.sh.dmod >= rd ? lsrc_carry : lsrc_plain;
        }
        src[NIN - 1] = reinterpret_cast<const C2 *>(st + (NSLOT - 1) * slot_bytes + p.sh.phase) + (t / W) * 9 * W + lsrc;
      }
      C2 acc[9], t0[9];
      menu_step<OP, 0, W>(src, acc, t0);
      C2 *so = reinterpret_cast<C2 *>(st) + base;  // every read of this thread's own slots is done
#pragma unroll
      for (int e = 0; e < 9; e++) so[e * W] = acc[e];
    }
    fence_proxy_async();  // generic-proxy smem writes -> visible to the bulk (async-proxy) store
    named_bar_sync(1, NCW * 32);
    if (t == 0) {
      const uint32_t bytes = (uint32_t)nm * 9u * CB;
      const uint32_t b16 = bytes & ~15u;
      unsigned char *zdst = (unsigned char *)p.z + (size_t)m0 * 9u * CB;
      if (p.hint)
        bulk_s2g_hint(zdst, st, b16, pol);
      else
        bulk_s2g(zdst, st, b16);
      bulk_commit();
      if (bytes != b16) *reinterpret_cast<uint64_t *>(zdst + b16) = *reinterpret_cast<const uint64_t *>(st + b16);
      // the previous tile's store has finished READING its stage: hand that stage back
      bulk_wait_read<1>();
      if (prev_s >= 0) mbar_arrive(&empty[prev_s]);
    }
    prev_s = s;
    if (++s == S) {
      s = 0;
      ph ^= 1u;
    }
  }
  if (t == 0) bulk_wait_all<0>();  // smem must outlive the last store; writes complete before exit
}

// ---------------------------------------------------------------- Cshift as a pure TMA copy (f3)
// z[s] = y[s + disp*dim_hat] moves whole records, and in storage order a tile's sources are a few contiguous runs (see
// ShiftInfo).  So Cshift is the ceiling kernel su3_bulk_copy_kernel with its one load per tile split into runs: one warp
// per CTA moves tiles global -> shared -> global with bulk copies through a ring of `stages` buffers (the loads of a
// tile issued by all lanes, one run each; the store by lane 0), and no register ever holds data -- except for records that cross the sub-lattice boundary in a dimension that is split over
// virtual nodes (simd_d > 1): their lanes rotate (S3), which the warp does in place in shared memory before the store.
// p.x = the shifted field y, p.z = z; p.tile_mats = matrices per tile (a multiple of W).
template <typename R, int W>
__global__ void __launch_bounds__(32) su3_cshift_bulk_kernel(const StreamParams p) {
  typedef typename Cplx<R>::type C2;
  constexpr int CB = (int)sizeof(C2);
  constexpr uint32_t rb = 9u * W * CB;  // bytes per record
  extern __shared__ __align__(128) unsigned char smem[];
  const int S = p.stages, lane = threadIdx.x;
  const int TR = p.tile_mats / W;  // records per tile
  const uint32_t tile_bytes = (uint32_t)TR * rb;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)S * tile_bytes);
  const int P = (int)p.sh.P, rd = p.sh.rd, dmod = p.sh.dmod;
  const int nrec = (int)(p.nmat / W);
  const int ntiles = (nrec + TR - 1) / TR;
  const unsigned char *gy = (const unsigned char *)p.x;
  const unsigned char *galt = (const unsigned char *)p.sh.alt;
  unsigned char *gz = (unsigned char *)p.z;
  const int mine = ntiles > (int)blockIdx.x ? (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
  // runs of tile [R0, R1): fn(first record, one past the last, carry)
  auto for_runs = [&](int R0, int R1, auto &&fn) {
    int blk = R0 / P, oc = blk % rd, Ra = R0;
    while (Ra < R1) {
      const bool carry = oc + dmod >= rd;
      const int eb = blk - oc + (carry ? rd : rd - dmod);  // first block after this run
      const long long Rbl = (long long)eb * P;
      const int Rb = Rbl < R1 ? (int)Rbl : R1;
      fn(Ra, Rb, carry);
      Ra = Rb;
      blk = eb;
      oc = eb % rd;
    }
  };
  // The whole warp issues a tile's loads: run boundaries sit at blocks cyc + {0, rd - dmod} of every cycle of rd blocks,
  // so lane k finds the k-th run of the tile in closed form and issues its bulk copy -- a shift along the fastest
  // dimension has 5-6 runs per tile, and one lane walking them (two integer divisions per run) was what the kernel
  // waited for there.
  auto load = [&](int i) {  // all lanes
    const int s = i % S;
    const int R0 = ((int)blockIdx.x + i * (int)gridDim.x) * TR;
    const int R1 = R0 + TR < nrec ? R0 + TR : nrec;
    unsigned char *buf = smem + (size_t)s * tile_bytes;
    if (lane == 0) mbar_arrive_expect_tx(&full[s], (uint32_t)(R1 - R0) * rb);
    const int blk0 = R0 / P, oc0 = blk0 % rd, cyc0 = blk0 - oc0;
    const int m0 = oc0 >= rd - dmod ? 1 : 0;  // boundary m: block cyc0 + (m / 2) * rd + (m odd ? rd - dmod : 0); runs m odd carry
    for (int m = m0 + lane;; m += 32) {
      const long long ba = (long long)(cyc0 + (m >> 1) * rd + ((m & 1) ? rd - dmod : 0)) * P;
      if (ba >= R1) break;
      const long long bb = (long long)(cyc0 + ((m + 1) >> 1) * rd + (((m + 1) & 1) ? rd - dmod : 0)) * P;
      const int Ra = ba > R0 ? (int)ba : R0, Rb = bb < R1 ? (int)bb : R1;
      if (Rb <= Ra) continue;  // dmod = 0: the carry runs are empty
      const bool carry = m & 1;
      const long long Rs = (long long)Ra + (long long)(carry ? dmod - rd : dmod) * P;
      const unsigned char *base = (galt && (int)carry == p.sh.alt_carry) ? galt : gy;
      bulk_g2s(buf + (size_t)(Ra - R0) * rb, base + (size_t)Rs * rb, (uint32_t)(Rb - Ra) * rb, &full[s]);
    }
  };
  if (lane == 0) {
    for (int s = 0; s < S; s++) mbar_init(&full[s], 1);
    fence_mbar_init();
    fence_proxy_async();
  }
  __syncwarp();
  for (int i = 0; i < mine && i < S; i++) load(i);
  __syncwarp();
  for (int i = 0; i < mine; i++) {
    const int s = i % S;
    const int R0 = ((int)blockIdx.x + i * (int)gridDim.x) * TR;
    const int R1 = R0 + TR < nrec ? R0 + TR : nrec;
    unsigned char *buf = smem + (size_t)s * tile_bytes;
    mbar_wait(&full[s], (uint32_t)((i / S) & 1));
    if (W > 1 && p.sh.simd_d > 1) {
      // lane rotation of the records whose neighbour sits in another virtual node: new[e][l] = old[e][l'], with
      // ic' = (ic + qrot + carry) mod simd_d
      for_runs(R0, R1, [&](int Ra, int Rb, bool carry) {
        const int rot = (p.sh.qrot + (carry ? 1 : 0)) % p.sh.simd_d;
        if (rot == 0) return;
        // the run's complex numbers, flat: index j holds lane j % W of its element vector, and the source of j lies in the
        // same W-aligned group; chunks of 32*U numbers (whole groups) are read completely, then written back
        constexpr int U = 8;
        C2 *run = reinterpret_cast<C2 *>(buf + (size_t)(Ra - R0) * rb);
        const int cnt = (Rb - Ra) * 9 * W;
        const int l = lane % W, ic = (l / p.sh.lstride) % p.sh.simd_d;
        const int delta = ((ic + rot) % p.sh.simd_d - ic) * p.sh.lstride;   // source lane - own lane (32 % W == 0: same for all j of this thread)
        for (int c0 = 0; c0 < cnt; c0 += 32 * U) {
          C2 v[U];
#pragma unroll
          for (int u = 0; u < U; u++) {
            const int j = c0 + u * 32 + lane;
            if (j < cnt) v[u] = run[j + delta];
          }
          __syncwarp();
#pragma unroll
          for (int u = 0; u < U; u++) {
            const int j = c0 + u * 32 + lane;
            if (j < cnt) run[j] = v[u];
          }
          __syncwarp();
        }
      });
      fence_proxy_async();
    }
    __syncwarp();
    if (lane == 0) {
      bulk_s2g(gz + (size_t)R0 * rb, buf, (uint32_t)(R1 - R0) * rb);
      bulk_commit();
      // the store before this one has finished reading its buffer: refill that buffer
      if (i >= 1) bulk_wait_read<1>();
    }
    __syncwarp();
    if (i >= 1 && i - 1 + S < mine) load(i - 1 + S);
  }
  if (lane == 0) bulk_wait_all<0>();
}

// ---------------------------------------------------------------- direct path (path = 2)
// One thread per matrix, operands read straight from global memory with one complex number
// per load.  For W*sizeof(complex) >= 32 bytes every warp request is made of whole sectors
// (vector layout: each group of W threads reads one W*c-byte element vector).  For W = 1
// this is the paper's naive AoS kernel ("lack of memory coalescence"),
// kept as the measured counter-example.
template <typename R, int W, int OP>
__global__ void __launch_bounds__(256) su3_direct_kernel(const StreamParams p) {
  typedef typename Cplx<R>::type C2;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < p.nmat; t += stride) {
    const long long base = (t / W) * 9 * W + (t % W);
    const C2 *gx = reinterpret_cast<const C2 *>(p.x) + base;
    const C2 *gy = reinterpret_cast<const C2 *>(p.y) + base;
    C2 *gz = reinterpret_cast<C2 *>(p.z) + base;
    C2 a[9], b[9], c[9];
#pragma unroll
    for (int e = 0; e < 9; e++) a[e] = gx[e * W];
#pragma unroll
    for (int e = 0; e < 9; e++) b[e] = gy[e * W];
    if (OP == OP_MUL) {
      mat33_mul(a, b, c);
    } else if (OP == OP_MUL3) {
      const C2 *gu = reinterpret_cast<const C2 *>(p.u) + base;
      C2 w[9];
#pragma unroll
      for (int e = 0; e < 9; e++) w[e] = gu[e * W];
      mat33_mul(a, b, c);
      mat33_mul(c, w, a);
#pragma unroll
      for (int e = 0; e < 9; e++) c[e] = a[e];
    } else {
      const C2 *gu = reinterpret_cast<const C2 *>(p.u) + base;
      C2 w[9];
#pragma unroll
      for (int e = 0; e < 9; e++) w[e] = gu[e * W];
      mat33_mul(a, b, c);
#pragma unroll
      for (int e = 0; e < 9; e++) {
        c[e].x = add_rn(c[e].x, w[e].x);
        c[e].y = add_rn(c[e].y, w[e].y);
      }
    }
#pragma unroll
    for (int e = 0; e < 9; e++) gz[e * W] = c[e];
  }
}

// ---------------------------------------------------------------- general one-pass expression (f2)
// z = value of a small expression tree over matrix fields, evaluated per site in ONE pass (P:76-109,
// Listings 1-2: `eval(ss, expr)` inside the site loop; every extra operand adds one read stream, no
// intermediate ever goes to memory).  The host compiles the postfix program into at most 16 register-
// machine instructions (su3_api.cu): each takes its two sources from an operand slot of the stage, a
// thread-private temporary in shared memory, or the accumulator registers, and leaves its result in the
// accumulator.  The program is uniform over the grid, so the interpreter's branches never diverge.
// Same pipeline as su3_pipe_kernel (TMA bulk in, TMA bulk out), same mat33_mul, hence bit-identical
// to su3_mul / su3_mul3 / su3_mul_add on their three programs.
struct ExprParams {
  void *z;
  const void *ops[8];
  long long nmat;
  int tile_mats, stages, nops, nins, ntemp, hint;  // stages = ring depth of the CTA's private ring
  int xchg;                                          // 1: the program multiplies by a computed value on the RIGHT (one more slot)
  ExprIns ins[16];
  int4 insx[16];  // the same instructions, one int per field (op, a, b, spill): what the interpreter reads
};

// row `c` = row `a` of the left factor times the full right factor: the rows of mat33_mul, operation for operation
// (k ascending, the same FMA chain per element), so a row-split product is bit-identical to mat33_mul
template <typename C2>
__device__ __forceinline__ void mat33_mul_row(const C2 (&a)[3], const C2 (&b)[9], C2 (&c)[3]) {
#pragma unroll
  for (int j = 0; j < 3; j++) {
    auto re = mul_rn(a[0].x, b[j].x);
    auto im = mul_rn(a[0].x, b[j].y);
    re = fma_rn(-a[0].y, b[j].y, re);
    im = fma_rn(a[0].y, b[j].x, im);
#pragma unroll
    for (int k = 1; k < 3; k++) {
      re = fma_rn(a[k].x, b[3 * k + j].x, re);
      im = fma_rn(a[k].x, b[3 * k + j].y, im);
      re = fma_rn(-a[k].y, b[3 * k + j].y, re);
      im = fma_rn(a[k].y, b[3 * k + j].x, im);
    }
    c[j].x = re;
    c[j].y = im;
  }
}

// Pipeline granularity and work split.  An interpreted program is bound by the latency of its LDS -> FMA chain per
// tile, not by throughput, and the bytes a warp keeps in flight (its ring of stages) cost shared memory: with one thread
// per matrix a 4-operand program left room for 4-5 warps per SM, one per scheduler, issuing 0.3 instructions per clock
// (ncu, round 2) -- 0.69-0.80 x the copy ceiling.  So a CTA is ONE self-contained pipeline of 96 threads that evaluates a
// tile of MPS = 32 matrices (64 for fp32 programs with few operands) per stage with THREE threads per matrix: warp r
// computes row r of every intermediate.  A row of a product needs the same row of the left factor and the whole right
// factor; operands are whole in the stage, so only a product whose RIGHT factor is a computed value (the accumulator or
// a temporary) makes the three warps exchange rows through shared memory (two CTA barriers); element-wise
// instructions and spills are row-local.  Same smem per pipeline as before, three times the warps, a third of the
// registers per thread; tid 0 issues the CTA's bulk loads and stores (no producer warp), results leave through two
// alternating result slots so that a stage is re-armed the moment the CTA has finished reading it.
template <typename R, int W>
__global__ void __launch_bounds__(96) su3_expr_kernel(const ExprParams p) {
  typedef typename Cplx<R>::type C2;
  constexpr int CB = (int)sizeof(C2);
  extern __shared__ __align__(128) unsigned char smem[];
  const int MPS = p.tile_mats;
  const int SW = p.stages, NIN = p.nops;
  const uint32_t slot_bytes = (uint32_t)MPS * 9u * CB;
  const uint32_t stage_bytes = NIN * slot_bytes;
  unsigned char *temps = smem + (size_t)SW * stage_bytes;                       // [ntemp] slots
  unsigned char *xchg = temps + (size_t)p.ntemp * slot_bytes;                   // [xchg] slot: the accumulator, made whole
  unsigned char *outs = xchg + (size_t)p.xchg * slot_bytes;                     // [2] result slots: the bulk stores' sources
  uint64_t *full = reinterpret_cast<uint64_t *>(outs + 2 * (size_t)slot_bytes);
  const int tid = threadIdx.x, lane = tid & 31, row = tid >> 5;
  const long long ntiles = (p.nmat + MPS - 1) / MPS;
  const long long gw = blockIdx.x, GW = gridDim.x;
  const long long mine = ntiles > gw ? (ntiles - gw + GW - 1) / GW : 0;  // my tiles: gw, gw + GW, ...
  auto load = [&](int s, long long tile) {  // tid 0 only: tile `tile` into stage s
    const long long m0 = tile * MPS;
    const long long left = p.nmat - m0;
    const int nm = left < MPS ? (int)left : MPS;
    const uint32_t bytes = (uint32_t)nm * 9u * CB;
    const uint32_t b16 = bytes & ~15u;
    unsigned char *st = smem + (size_t)s * stage_bytes;
    const size_t goff = (size_t)m0 * 9u * CB;
    if (bytes != b16)
      for (int o = 0; o < NIN; o++)
        *reinterpret_cast<uint64_t *>(st + o * slot_bytes + b16) =
            *reinterpret_cast<const uint64_t *>((const unsigned char *)p.ops[o] + goff + b16);
    mbar_arrive_expect_tx(&full[s], NIN * b16);
    for (int o = 0; o < NIN; o++)
      bulk_g2s(st + o * slot_bytes, (const unsigned char *)p.ops[o] + goff, b16, &full[s]);
  };
  if (tid == 0) {
    for (int q = 0; q < SW; q++) mbar_init(&full[q], 1);
    fence_mbar_init();
    fence_proxy_async();
    for (long long j = 0; j < mine && j < SW; j++) load((int)j, gw + j * GW);
  }
  __syncthreads();
  int s = 0;          // stage of tile j = j % SW, kept as a counter (no division per tile)
  uint32_t ph = 0;    // its phase bit = (j / SW) & 1
  long long tile = gw;
  for (long long j = 0; j < mine; j++, tile += GW) {
    const long long m0 = tile * MPS;
    const long long left = p.nmat - m0;
    const int nm = left < MPS ? (int)left : MPS;
    unsigned char *st = smem + (size_t)s * stage_bytes;
    unsigned char *myout = outs + (size_t)(j & 1) * slot_bytes;
    mbar_wait(&full[s], ph);
    // every lane runs every iteration (the barriers below are CTA-wide); lanes past the ragged end compute on stale
    // shared memory inside the slot and their rows are never stored
#pragma unroll 1
    for (int t = lane; t < MPS; t += 32) {
      const int base = (t / W) * 9 * W + (t % W);   // element 0 of matrix t
      const int rbase = base + 3 * row * W;         // element (row, 0)
      // The dispatch is written so that NO copy of the accumulator is needed outside the one case that really needs it
      // (a product whose LEFT factor is the accumulator): with a generic "load a, load b, combine" body the compiler
      // copied the 12 accumulator registers at the top of every interpreted instruction (16 % of all executed
      // instructions, ncu), and unpacking the four bytes of an ExprIns cost six more: insx holds them as four ints.
      C2 acc[3];
#pragma unroll 1
      for (int i = 0; i < p.nins; i++) {
        const int4 in = p.insx[i];   // x = op, y = a, z = b, w = spill
        if (in.w != EX_NONE) {
          C2 *sp = reinterpret_cast<C2 *>(temps + (size_t)(in.w - EX_TEMP0) * slot_bytes) + rbase;
#pragma unroll
          for (int e = 0; e < 3; e++) sp[e * W] = acc[e];
        }
        const C2 *pa = reinterpret_cast<const C2 *>(in.y < EX_TEMP0 ? st + in.y * slot_bytes
                                                                   : temps + (size_t)(in.y - EX_TEMP0) * slot_bytes) + rbase;
        if (in.x == EX_MUL) {
          C2 b[9];
          if (in.z < EX_TEMP0) {
            const C2 *sb = reinterpret_cast<const C2 *>(st + in.z * slot_bytes) + base;
#pragma unroll
            for (int e = 0; e < 9; e++) b[e] = sb[e * W];
          } else {
            // the right factor is a computed value: its rows live in three different warps
            const C2 *whole;
            if (in.z == EX_SRC_ACC) {
              C2 *xs = reinterpret_cast<C2 *>(xchg) + rbase;
#pragma unroll
              for (int e = 0; e < 3; e++) xs[e * W] = acc[e];
              whole = reinterpret_cast<const C2 *>(xchg) + base;
            } else {
              whole = reinterpret_cast<const C2 *>(temps + (size_t)(in.z - EX_TEMP0) * slot_bytes) + base;
            }
            __syncthreads();  // all three rows written
#pragma unroll
            for (int e = 0; e < 9; e++) b[e] = whole[e * W];
            __syncthreads();  // all three warps have read: the slot may be written again
          }
          if (in.y == EX_SRC_ACC) {
            C2 r[3];
            mat33_mul_row(acc, b, r);
#pragma unroll
            for (int e = 0; e < 3; e++) acc[e] = r[e];
          } else {
            C2 a[3];
#pragma unroll
            for (int e = 0; e < 3; e++) a[e] = pa[e * W];
            mat33_mul_row(a, b, acc);
          }
        } else if (in.x == EX_COPY) {
#pragma unroll
          for (int e = 0; e < 3; e++) acc[e] = pa[e * W];
        } else {
          // element-wise: acc = a (op) b with a, b each an operand / temporary in shared memory or the accumulator itself
          const C2 *pb = reinterpret_cast<const C2 *>(in.z < EX_TEMP0 ? st + in.z * slot_bytes
                                                                     : temps + (size_t)(in.z - EX_TEMP0) * slot_bytes) + rbase;
          // four source combinations, each a straight-line body (no selects, no copies)
          auto ew = [&](const C2 (&av)[3], const C2 (&bv)[3]) {
#pragma unroll
            for (int e = 0; e < 3; e++) {
              if (in.x == EX_EMUL) {
                acc[e].x = mul_rn(av[e].x, bv[e].x);
                acc[e].y = mul_rn(av[e].y, bv[e].y);
              } else if (in.x == EX_ADD) {
                acc[e].x = add_rn(av[e].x, bv[e].x);
                acc[e].y = add_rn(av[e].y, bv[e].y);
              } else {
                acc[e].x = add_rn(av[e].x, -bv[e].x);
                acc[e].y = add_rn(av[e].y, -bv[e].y);
              }
            }
          };
          C2 a[3], bb[3];
          if (in.y != EX_SRC_ACC) {
#pragma unroll
            for (int e = 0; e < 3; e++) a[e] = pa[e * W];
          }
          if (in.z != EX_SRC_ACC) {
#pragma unroll
            for (int e = 0; e < 3; e++) bb[e] = pb[e * W];
          }
          if (in.y == EX_SRC_ACC) {
            if (in.z == EX_SRC_ACC) ew(acc, acc);
            else ew(acc, bb);
          } else {
            if (in.z == EX_SRC_ACC) ew(a, acc);
            else ew(a, bb);
          }
        }
      }
      C2 *so = reinterpret_cast<C2 *>(myout) + rbase;
#pragma unroll
      for (int e = 0; e < 3; e++) so[e * W] = acc[e];
    }
    fence_proxy_async();
    // store j-1 (issued a whole tile ago) has finished READING the other result slot, which tile j+1 writes
    if (tid == 0) bulk_wait_read<0>();
    __syncthreads();
    // every thread has read what it needs from stage s and written its rows of the result: re-arm the stage with my
    // tile j + SW at once -- the refill never waits for the store -- and send the result on its way
    if (tid == 0) {
      if (j + SW < mine) load(s, tile + (long long)SW * GW);
      const uint32_t bytes = (uint32_t)nm * 9u * CB;
      const uint32_t b16 = bytes & ~15u;
      unsigned char *zdst = (unsigned char *)p.z + (size_t)m0 * 9u * CB;
      bulk_s2g(zdst, myout, b16);
      bulk_commit();
      if (bytes != b16) *reinterpret_cast<uint64_t *>(zdst + b16) = *reinterpret_cast<const uint64_t *>(myout + b16);
    }
    if (++s == SW) {
      s = 0;
      ph ^= 1u;
    }
  }
  if (tid == 0) bulk_wait_all<0>();
}

// ---------------------------------------------------------------- real scalar fields (Listing 2 of the paper)
// `Lattice<double> v3 = v1+v2+v1*v2`: one real per (site, mu), element-wise, hence layout-agnostic.
// A real field of n reals is evaluated as n / 18 records of 18 reals by the matrix machinery (su3_pipe_kernel's OP_ADD
// for `a+b`, su3_expr_kernel with EX_EMUL for '*' otherwise: TMA in, TMA out); this plain kernel takes the n % 18 tail.
template <typename R>
__global__ void __launch_bounds__(32) su3_real_expr_kernel(const ExprParams p) {
  for (long long i = threadIdx.x; i < p.nmat; i += blockDim.x) {  // one block: this is the tail of < 18 reals
    R acc = 0, tmp[8];
#pragma unroll 1
    for (int k = 0; k < p.nins; k++) {
      const ExprIns in = p.ins[k];
      if (in.spill != EX_NONE) tmp[in.spill - EX_TEMP0] = acc;
      auto fetch = [&](unsigned char srcid) -> R {
        if (srcid == EX_SRC_ACC) return acc;
        if (srcid >= EX_TEMP0) return tmp[srcid - EX_TEMP0];
        return reinterpret_cast<const R *>(p.ops[srcid])[i];
      };
      const R a = fetch(in.a);
      const R b = in.op != EX_COPY ? fetch(in.b) : R(0);
      acc = (in.op == EX_MUL || in.op == EX_EMUL) ? mul_rn(a, b) : in.op == EX_ADD ? add_rn(a, b) : in.op == EX_SUB ? add_rn(a, -b) : a;
    }
    reinterpret_cast<R *>(p.z)[i] = acc;
  }
}

// field = value (Listing 2: `v1 = 1.0;`)
template <typename R> __global__ void __launch_bounds__(256) su3_real_fill_kernel(R *z, long long n, R value) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) z[i] = value;
}

// ---------------------------------------------------------------- y = U.psi on colour vectors (f4)
// Same pipeline as su3_pipe_kernel with two operand slots of different record size: U (9 complex per
// matrix) and psi (3 complex per vector; record of the vector layout = 3 element vectors of W lanes).
// p.x = U, p.y = psi, p.z = y.  y overwrites the psi slot and leaves by a bulk store.  66 flops and
// 144+48+48 B (fp64) per (site, mu).
template <typename R, int W, int NCW>
__global__ void __launch_bounds__((NCW + 1) * 32, 3) su3_matvec_kernel(const StreamParams p) {
  typedef typename Cplx<R>::type C2;
  constexpr int CB = (int)sizeof(C2);
  extern __shared__ __align__(128) unsigned char smem[];
  const int TM = p.tile_mats, S = p.stages;
  const uint32_t uslot = (uint32_t)TM * 9u * CB, vslot = (uint32_t)TM * 3u * CB;
  const uint32_t stage_bytes = uslot + vslot;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)S * stage_bytes);
  uint64_t *empty = full + S;
  const int tid = threadIdx.x;
  const long long ntiles = (p.nmat + TM - 1) / TM;
  if (tid == 0) {
    for (int s = 0; s < S; s++) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], 1);
    }
    fence_mbar_init();
    fence_proxy_async();
  }
  __syncthreads();
  if (tid >= NCW * 32) {
    if (tid == NCW * 32) {
      const unsigned char *gu = (const unsigned char *)p.x, *gv = (const unsigned char *)p.y;
      int s = 0;
      uint32_t ph = 0;
      for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        mbar_wait(&empty[s], ph ^ 1u);
        const long long m0 = tile * TM;
        const long long left = p.nmat - m0;
        const int nm = left < TM ? (int)left : TM;
        const uint32_t ub = (uint32_t)nm * 9u * CB, vb = (uint32_t)nm * 3u * CB;
        const uint32_t ub16 = ub & ~15u, vb16 = vb & ~15u;
        unsigned char *st = smem + (size_t)s * stage_bytes;
        if (ub != ub16)
          *reinterpret_cast<uint64_t *>(st + ub16) = *reinterpret_cast<const uint64_t *>(gu + (size_t)m0 * 9u * CB + ub16);
        if (vb != vb16)
          *reinterpret_cast<uint64_t *>(st + uslot + vb16) =
              *reinterpret_cast<const uint64_t *>(gv + (size_t)m0 * 3u * CB + vb16);
        mbar_arrive_expect_tx(&full[s], ub16 + vb16);
        bulk_g2s(st, gu + (size_t)m0 * 9u * CB, ub16, &full[s]);
        if (vb16) bulk_g2s(st + uslot, gv + (size_t)m0 * 3u * CB, vb16, &full[s]);
        if (++s == S) {
          s = 0;
          ph ^= 1u;
        }
      }
    }
    return;
  }
  const int t = tid;
  const int ubase = (t / W) * 9 * W + (t % W), vbase = (t / W) * 3 * W + (t % W);
  int s = 0, prev_s = -1;
  uint32_t ph = 0;
  for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const long long m0 = tile * TM;
    const long long left = p.nmat - m0;
    const int nm = left < TM ? (int)left : TM;
    unsigned char *st = smem + (size_t)s * stage_bytes;
    mbar_wait(&full[s], ph);
    if (t < nm) {
      const C2 *su = reinterpret_cast<const C2 *>(st) + ubase;
      C2 *sv = reinterpret_cast<C2 *>(st + uslot) + vbase;
      C2 a[9], b[3], c[3];
#pragma unroll
      for (int e = 0; e < 9; e++) a[e] = su[e * W];
#pragma unroll
      for (int j = 0; j < 3; j++) b[j] = sv[j * W];
#pragma unroll
      for (int i = 0; i < 3; i++) {  // y_i = sum_j U_ij psi_j, j ascending: the FMA chain of mat33_mul
        auto re = mul_rn(a[3 * i].x, b[0].x);
        auto im = mul_rn(a[3 * i].x, b[0].y);
        re = fma_rn(-a[3 * i].y, b[0].y, re);
        im = fma_rn(a[3 * i].y, b[0].x, im);
#pragma unroll
        for (int j = 1; j < 3; j++) {
          re = fma_rn(a[3 * i + j].x, b[j].x, re);
          im = fma_rn(a[3 * i + j].x, b[j].y, im);
          re = fma_rn(-a[3 * i + j].y, b[j].y, re);
          im = fma_rn(a[3 * i + j].y, b[j].x, im);
        }
        c[i].x = re;
        c[i].y = im;
      }
#pragma unroll
      for (int i = 0; i < 3; i++) sv[i * W] = c[i];
    }
    fence_proxy_async();
    named_bar_sync(1, NCW * 32);
    if (t == 0) {
      const uint32_t vb = (uint32_t)nm * 3u * CB, vb16 = vb & ~15u;
      unsigned char *ydst = (unsigned char *)p.z + (size_t)m0 * 3u * CB;
      if (vb16) bulk_s2g(ydst, st + uslot, vb16);
      bulk_commit();
      if (vb != vb16) *reinterpret_cast<uint64_t *>(ydst + vb16) = *reinterpret_cast<const uint64_t *>(st + uslot + vb16);
      bulk_wait_read<1>();
      if (prev_s >= 0) mbar_arrive(&empty[prev_s]);
    }
    prev_s = s;
    if (++s == S) {
      s = 0;
      ph ^= 1u;
    }
  }
  if (t == 0) bulk_wait_all<0>();
}

// ---------------------------------------------------------------- warp-staged path (path = 3)
// For L2-resident lattices the pipeline's fixed latency (mbarrier set-up, TMA in, TMA out) is what one
// measures.  Here every warp stages its own 32 matrices with coalesced per-lane loads of one complex
// number each (lane i of request j reads complex j*32+i of the warp's contiguous 32*9-complex range),
// multiplies out of shared memory exactly like the pipeline's consumers, and stores the same way.
// Only __syncwarp() is needed; any layout (W | 32) works through the same shared-memory index.
template <typename R, int W, int OP>
__global__ void __launch_bounds__(128) su3_warp_kernel(const StreamParams p) {
  typedef typename Cplx<R>::type C2;
  constexpr int NIN = NumInputs<OP>::value;
  extern __shared__ __align__(128) unsigned char smem[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5;
  C2 *sw = reinterpret_cast<C2 *>(smem) + (size_t)wib * NIN * 288;
  const long long nwt = (p.nmat + 31) / 32;
  const int base = (lane / W) * 9 * W + (lane % W);
  const C2 *src[3] = {reinterpret_cast<const C2 *>(p.x), reinterpret_cast<const C2 *>(p.y),
                      reinterpret_cast<const C2 *>(p.u)};
  C2 *gz = reinterpret_cast<C2 *>(p.z);
  for (long long wt = (long long)blockIdx.x * wpb + wib; wt < nwt; wt += (long long)gridDim.x * wpb) {
    const long long c0 = wt * 288;
    const long long left = p.nmat - wt * 32;
    const int nm = left < 32 ? (int)left : 32;
    const int nc = nm * 9;
    C2 r[NIN][9];
#pragma unroll
    for (int o = 0; o < NIN; o++)
#pragma unroll
      for (int j = 0; j < 9; j++)
        if (j * 32 + lane < nc) r[o][j] = src[o][c0 + j * 32 + lane];
#pragma unroll
    for (int o = 0; o < NIN; o++)
#pragma unroll
      for (int j = 0; j < 9; j++)
        if (j * 32 + lane < nc) sw[o * 288 + j * 32 + lane] = r[o][j];
    __syncwarp();
    if (lane < nm) {
      C2 a[9], b[9], c[9];
#pragma unroll
      for (int e = 0; e < 9; e++) a[e] = sw[base + e * W];
#pragma unroll
      for (int e = 0; e < 9; e++) b[e] = sw[288 + base + e * W];
      if (OP == OP_ADD) {
#pragma unroll
        for (int e = 0; e < 9; e++) {
          c[e].x = add_rn(a[e].x, b[e].x);
          c[e].y = add_rn(a[e].y, b[e].y);
        }
      } else {
        mat33_mul(a, b, c);
      }
      if (OP == OP_MUL3) {
#pragma unroll
        for (int e = 0; e < 9; e++) b[e] = sw[2 * 288 + base + e * W];
        mat33_mul(c, b, a);
#pragma unroll
        for (int e = 0; e < 9; e++) c[e] = a[e];
      } else if (OP == OP_MUL_ADD) {
#pragma unroll
        for (int e = 0; e < 9; e++) {
          C2 v = sw[2 * 288 + base + e * W];
          c[e].x = add_rn(c[e].x, v.x);
          c[e].y = add_rn(c[e].y, v.y);
        }
      }
#pragma unroll
      for (int e = 0; e < 9; e++) sw[base + e * W] = c[e];
    }
    __syncwarp();
#pragma unroll
    for (int j = 0; j < 9; j++)
      if (j * 32 + lane < nc) gz[c0 + j * 32 + lane] = sw[j * 32 + lane];
    __syncwarp();
  }
}

// ---------------------------------------------------------------- Cshift and the shifted product (f3)
// z[s] = y[s + disp*dim_hat] (SH_COPY, Grid's Cshift) and z[s] = x[s] . y[s + disp*dim_hat] (SH_MUL).
// Warp-staged like su3_warp_kernel, but the shifted operand is GATHERED: lane t works out, once per tile,
// where the neighbour of its own matrix lives -- in the vector layout a step across the sub-lattice
// boundary lands in another lane of outer site oc' (the virtual-node map S3), so the source is
// (record', lane') -- and every element load fetches that base from the owning lane with one shuffle.
// Neighbouring lanes read neighbouring addresses except at the wrap, so the loads stay coalesced.
enum { SH_COPY = 0, SH_MUL = 1 };
struct ShiftParams {
  void *z;
  const void *x;  // unshifted operand (SH_MUL only)
  const void *y;  // shifted operand
  long long nmat;
  long long ostride;  // prod_{k<dim} r[k]
  int nl, rd, Ld, lstride, simd_d, disp;  // r[dim], L[dim], prod_{k<dim} simd[k], simd[dim], 0 <= disp < L[dim]
};

// IT = index type: int when every complex index of the field fits 31 bits (all configs), else long long.
template <typename R, int W, int OP, typename IT>
__global__ void __launch_bounds__(128, OP == SH_COPY ? (sizeof(R) == 4 ? 12 : 8) : 3) su3_shift_kernel(const ShiftParams p) {
  typedef typename Cplx<R>::type C2;
  extern __shared__ __align__(128) unsigned char smem[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5;
  C2 *sw = reinterpret_cast<C2 *>(smem) + (size_t)wib * 2 * 288;
  const IT nwt = (IT)((p.nmat + 31) / 32);
  const IT ostride = (IT)p.ostride;
  const int base = (lane / W) * 9 * W + (lane % W);
  const C2 *gx = reinterpret_cast<const C2 *>(p.x);
  const C2 *gy = reinterpret_cast<const C2 *>(p.y);
  C2 *gz = reinterpret_cast<C2 *>(p.z);
  for (IT wt = (IT)blockIdx.x * wpb + wib; wt < nwt; wt += (IT)gridDim.x * wpb) {
    const IT c0 = wt * 288;
    const IT left = (IT)p.nmat - wt * 32;
    const int nm = left < 32 ? (int)left : 32;
    const int nc = nm * 9;
    // where does the neighbour of MY matrix (slot `lane` of this tile) live?
    IT srcbase = 0;
    if (lane < nm) {
      const IT g = wt * 32 + lane;
      const IT rec = g / W;
      const int l = (int)(g % W);
      const IT o = rec / p.nl;
      const int mu = (int)(rec - o * p.nl);
      const int oc = (int)((o / ostride) % p.rd);
      const int ic = (l / p.lstride) % p.simd_d;
      int xn = ic * p.rd + oc + p.disp;
      if (xn >= p.Ld) xn -= p.Ld;
      const int icn = xn / p.rd, ocn = xn - icn * p.rd;
      const IT on = o + (IT)(ocn - oc) * ostride;
      const int ln = l + (icn - ic) * p.lstride;
      srcbase = ((on * p.nl + mu) * 9) * W + ln;
    }
    C2 ry[9];
#pragma unroll
    for (int j = 0; j < 9; j++) {
      const int idx = j * 32 + lane;
      const int q = idx / (9 * W), rem = idx - q * 9 * W;
      const int e = rem / W, l = rem - e * W;
      const IT sb = __shfl_sync(0xffffffffu, srcbase, q * W + l);
      if (idx < nc) ry[j] = gy[sb + e * W];
    }
    if (OP == SH_COPY) {
#pragma unroll
      for (int j = 0; j < 9; j++)
        if (j * 32 + lane < nc) gz[c0 + j * 32 + lane] = ry[j];
    } else {
      C2 rx[9];
#pragma unroll
      for (int j = 0; j < 9; j++)
        if (j * 32 + lane < nc) rx[j] = gx[c0 + j * 32 + lane];
#pragma unroll
      for (int j = 0; j < 9; j++)
        if (j * 32 + lane < nc) {
          sw[j * 32 + lane] = rx[j];
          sw[288 + j * 32 + lane] = ry[j];
        }
      __syncwarp();
      if (lane < nm) {
        C2 a[9], b[9], c[9];
#pragma unroll
        for (int e = 0; e < 9; e++) a[e] = sw[base + e * W];
#pragma unroll
        for (int e = 0; e < 9; e++) b[e] = sw[288 + base + e * W];
        mat33_mul(a, b, c);
#pragma unroll
        for (int e = 0; e < 9; e++) sw[base + e * W] = c[e];
      }
      __syncwarp();
#pragma unroll
      for (int j = 0; j < 9; j++)
        if (j * 32 + lane < nc) gz[c0 + j * 32 + lane] = sw[j * 32 + lane];
      __syncwarp();
    }
  }
}

// Cshift without registers in the data path: every warp GATHERS its tile with per-lane cp.async (LDGSTS, 16 B
// for fp64 / 8 B for fp32 complex numbers, addresses as in su3_shift_kernel) into a private ring of NS stages
// and STORES each finished tile with one TMA bulk copy (the destination tile is contiguous).  The register
// version above is latency-bound (ncu: 55-67 % DRAM, throughput proportional to resident blocks); here the
// bytes in flight are bounded by shared memory instead: 12 warps x (NS-2) tiles per SM.
__device__ __forceinline__ void cp_async_c2(double2 *dst_smem, const double2 *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_c2(float2 *dst_smem, const float2 *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

template <typename R, int W, typename IT>
__global__ void __launch_bounds__(128, 3) su3_cshift_async_kernel(const ShiftParams p) {
  typedef typename Cplx<R>::type C2;
  constexpr int CB = (int)sizeof(C2);
  constexpr int NS = sizeof(R) == 8 ? 4 : 8;  // 18.4 KB ring per warp either way
  constexpr int D = NS - 2;                   // a tile is stored D iterations after its gather was issued
  extern __shared__ __align__(128) unsigned char smem[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5;
  C2 *ring = reinterpret_cast<C2 *>(smem) + (size_t)wib * NS * 288;
  const IT nwt = (IT)((p.nmat + 31) / 32);
  const IT ostride = (IT)p.ostride;
  const C2 *gy = reinterpret_cast<const C2 *>(p.y);
  unsigned char *gz = reinterpret_cast<unsigned char *>(p.z);
  const IT gw = (IT)blockIdx.x * wpb + wib, GW = (IT)gridDim.x * wpb;
  const IT mine = nwt > gw ? (nwt - gw + GW - 1) / GW : 0;
  for (IT j = 0; j < mine + D; j++) {
    if (j < mine) {
      // stage j % NS was last used by tile j - NS, whose bulk store must have finished reading it
      if (lane == 0) bulk_wait_read<1>();
      __syncwarp();
      const IT wt = gw + j * GW;
      const IT left = (IT)p.nmat - wt * 32;
      const int nm = left < 32 ? (int)left : 32;
      const int nc = nm * 9;
      IT srcbase = 0;
      if (lane < nm) {
        const IT g = wt * 32 + lane;
        const IT rec = g / W;
        const int l = (int)(g % W);
        const IT o = rec / p.nl;
        const int mu = (int)(rec - o * p.nl);
        const int oc = (int)((o / ostride) % p.rd);
        const int ic = (l / p.lstride) % p.simd_d;
        int xn = ic * p.rd + oc + p.disp;
        if (xn >= p.Ld) xn -= p.Ld;
        const int icn = xn / p.rd, ocn = xn - icn * p.rd;
        const IT on = o + (IT)(ocn - oc) * ostride;
        const int ln = l + (icn - ic) * p.lstride;
        srcbase = ((on * p.nl + mu) * 9) * W + ln;
      }
      C2 *st = ring + (size_t)(j % NS) * 288;
#pragma unroll
      for (int jj = 0; jj < 9; jj++) {
        const int idx = jj * 32 + lane;
        const int q = idx / (9 * W), rem = idx - q * 9 * W;
        const int e = rem / W, l = rem - e * W;
        const IT sb = __shfl_sync(0xffffffffu, srcbase, q * W + l);
        if (idx < nc) cp_async_c2(st + idx, gy + sb + e * W);
      }
    }
    cp_async_commit();  // one group per iteration, empty past the last tile, so that the count below is uniform
    if (j >= D) {
      const IT t = j - D;  // its gather is complete once at most D younger groups are pending
      cp_async_wait<D>();
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) {
        const IT wt = gw + t * GW;
        const IT left = (IT)p.nmat - wt * 32;
        const int nm = left < 32 ? (int)left : 32;
        const uint32_t bytes = (uint32_t)nm * 9u * CB, b16 = bytes & ~15u;
        const C2 *st = ring + (size_t)(t % NS) * 288;
        unsigned char *dst = gz + (size_t)wt * 288 * CB;
        if (b16) bulk_s2g(dst, st, b16);
        bulk_commit();
        if (bytes != b16)
          *reinterpret_cast<uint64_t *>(dst + b16) = *reinterpret_cast<const uint64_t *>((const unsigned char *)st + b16);
      }
    }
  }
  if (lane == 0) bulk_wait_all<0>();
}

// ---------------------------------------------------------------- streaming ceilings (A6) and z = x + y
// dst = src as a pure TMA pipeline: one thread per CTA moves tiles global -> shared -> global with
// 1-D bulk copies through a ring of `stages` slots; no register ever holds data.  The ceiling the
// arithmetic kernels are compared with uses the same memory machinery as they do.
struct CopyParams {
  void *dst;
  const void *src;
  unsigned long long nbytes;  // multiple of 8
  unsigned tile_bytes;        // multiple of 16
  int stages;
  int hint;
};

static __global__ void __launch_bounds__(32) su3_bulk_copy_kernel(const CopyParams p) {
  extern __shared__ __align__(128) unsigned char smem[];
  if (threadIdx.x != 0) return;
  const int S = p.stages;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)S * p.tile_bytes);
  for (int s = 0; s < S; s++) mbar_init(&full[s], 1);
  fence_mbar_init();
  fence_proxy_async();
  const unsigned long long n16 = p.nbytes & ~15ull;
  const unsigned long long ntiles = (n16 + p.tile_bytes - 1) / p.tile_bytes;
  const unsigned char *src = (const unsigned char *)p.src;
  unsigned char *dst = (unsigned char *)p.dst;
  uint64_t pol = 0;
  if (p.hint) pol = policy_evict_first();
  // my tiles: blockIdx.x, blockIdx.x + gridDim.x, ...
  const unsigned long long mine = ntiles > blockIdx.x ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  auto tile_off = [&](unsigned long long i) { return (blockIdx.x + i * gridDim.x) * (unsigned long long)p.tile_bytes; };
  auto tile_len = [&](unsigned long long off) {
    const unsigned long long left = n16 - off;
    return (uint32_t)(left < p.tile_bytes ? left : p.tile_bytes);
  };
  auto load = [&](unsigned long long i) {
    const int s = (int)(i % S);
    const unsigned long long off = tile_off(i);
    const uint32_t len = tile_len(off);
    mbar_arrive_expect_tx(&full[s], len);
    if (p.hint)
      bulk_g2s_hint(smem + (size_t)s * p.tile_bytes, src + off, len, &full[s], pol);
    else
      bulk_g2s(smem + (size_t)s * p.tile_bytes, src + off, len, &full[s]);
  };
  for (unsigned long long i = 0; i < mine && i < (unsigned long long)S; i++) load(i);
  for (unsigned long long i = 0; i < mine; i++) {
    const int s = (int)(i % S);
    mbar_wait(&full[s], (uint32_t)((i / S) & 1));
    const unsigned long long off = tile_off(i);
    if (p.hint)
      bulk_s2g_hint(dst + off, smem + (size_t)s * p.tile_bytes, tile_len(off), pol);
    else
      bulk_s2g(dst + off, smem + (size_t)s * p.tile_bytes, tile_len(off));
    bulk_commit();
    // the store before this one has finished reading its slot: refill that slot
    if (i >= 1) {
      bulk_wait_read<1>();
      if (i - 1 + S < mine) load(i - 1 + S);
    }
  }
  if (blockIdx.x == 0 && p.nbytes != n16)
    *reinterpret_cast<uint64_t *>(dst + n16) = *reinterpret_cast<const uint64_t *>(src + n16);
  bulk_wait_all<0>();
}

// dst = src over n16 16-byte words (+ an optional 8-byte tail), 4 independent 128-bit loads
// in flight per thread (path = 2: the plain LDG/STG copy, kept as the measured comparison).
static __global__ void __launch_bounds__(256) su3_copy_kernel(uint4 *__restrict__ dst, const uint4 *__restrict__ src,
                                                       size_t n16, int tail8) {
  const size_t bd = blockDim.x;
  const size_t stride = (size_t)gridDim.x * bd * 4;
  size_t i = (size_t)blockIdx.x * bd * 4 + threadIdx.x;
  for (; i + 3 * bd < n16; i += stride) {
    uint4 v0 = src[i], v1 = src[i + bd], v2 = src[i + 2 * bd], v3 = src[i + 3 * bd];
    dst[i] = v0;
    dst[i + bd] = v1;
    dst[i + 2 * bd] = v2;
    dst[i + 3 * bd] = v3;
  }
  for (; i < n16; i += bd) dst[i] = src[i];
  if (tail8 && blockIdx.x == 0 && threadIdx.x == 0)
    reinterpret_cast<uint2 *>(dst + n16)[0] = reinterpret_cast<const uint2 *>(src + n16)[0];
}

template <typename R> struct Vec16;
template <> struct Vec16<float> {
  typedef float4 type;
  static __device__ __forceinline__ float4 add(float4 a, float4 b) {
    return make_float4(__fadd_rn(a.x, b.x), __fadd_rn(a.y, b.y), __fadd_rn(a.z, b.z), __fadd_rn(a.w, b.w));
  }
};
template <> struct Vec16<double> {
  typedef double2 type;
  static __device__ __forceinline__ double2 add(double2 a, double2 b) {
    return make_double2(__dadd_rn(a.x, b.x), __dadd_rn(a.y, b.y));
  }
};

// z = x + y over n16 16-byte words (+ nrem trailing reals); layout-agnostic (element-wise).
template <typename R>
__global__ void __launch_bounds__(256) su3_add_kernel(R *z, const R *x, const R *y, size_t n16, int nrem) {
  typedef typename Vec16<R>::type V;
  V *z16 = reinterpret_cast<V *>(z);
  const V *x16 = reinterpret_cast<const V *>(x);
  const V *y16 = reinterpret_cast<const V *>(y);
  const size_t bd = blockDim.x;
  const size_t stride = (size_t)gridDim.x * bd * 2;
  size_t i = (size_t)blockIdx.x * bd * 2 + threadIdx.x;
  for (; i + bd < n16; i += stride) {
    V a0 = x16[i], a1 = x16[i + bd], b0 = y16[i], b1 = y16[i + bd];
    z16[i] = Vec16<R>::add(a0, b0);
    z16[i + bd] = Vec16<R>::add(a1, b1);
  }
  for (; i < n16; i += bd) z16[i] = Vec16<R>::add(x16[i], y16[i]);
  if (blockIdx.x == 0 && (int)threadIdx.x < nrem) {
    const size_t k = n16 * (16 / sizeof(R)) + threadIdx.x;
    z[k] = add_rn(x[k], y[k]);
  }
}

// ---------------------------------------------------------------- layout conversion (A5)
// vec[o][mu][e][l] = sca[site(o,l)][mu][e]  (extract/merge; virtual-node map S3).
// A block handles TR consecutive vector records (rec = o*nl + mu): the vector side is one
// contiguous, fully coalesced range; the scalar side is W streams of contiguous records.
struct ConvertParams {
  void *dst;
  const void *src;
  long long nrec;       // vector records = (volume / W) * nl
  int nl;
  int r[4];             // sub-lattice extents L[d] / simd[d]
  long long sstride[4]; // scalar-site stride of dimension d: 1, L0, L0*L1, L0*L1*L2
  long long lane_off[32]; // (site offset of lane l) * nl * NC, in complex numbers (NC = 9 matrix, 3 colour vector)
  int to_vector;        // 1: dst is the vector layout; 0: dst is the scalar layout
  long long run_recs;   // su3_convert_tma_kernel: consecutive vector records whose scalar-side images are contiguous
  int pitch;            // su3_convert_tma_kernel: shared-memory row pitch of one lane's run, in complex numbers
};

template <typename C2, int W, int TR, int NC>
__global__ void __launch_bounds__(256) su3_convert_kernel(const ConvertParams p) {
  __shared__ long long sbase[TR];  // scalar-side complex index of (rec, lane 0, e = 0)
  const long long rec0 = (long long)blockIdx.x * TR;
  const long long left = p.nrec - rec0;
  const int nr = left < TR ? (int)left : TR;
  if ((int)threadIdx.x < nr) {
    const long long rec = rec0 + threadIdx.x;
    long long o = rec / p.nl;
    const int mu = (int)(rec - o * p.nl);
    long long site = 0;
#pragma unroll
    for (int d = 0; d < 4; d++) {
      const long long q = o / p.r[d];
      site += (o - q * p.r[d]) * p.sstride[d];
      o = q;
    }
    sbase[threadIdx.x] = (site * p.nl + mu) * NC;
  }
  __syncthreads();
  const C2 *src = reinterpret_cast<const C2 *>(p.src);
  C2 *dst = reinterpret_cast<C2 *>(p.dst);
  const long long vbase = rec0 * NC * W;
  const int n = nr * NC * W;
  constexpr int U = 4;
  for (int i0 = threadIdx.x; i0 < n; i0 += 256 * U) {
    long long vi[U], si[U];
    C2 val[U];
#pragma unroll
    for (int u = 0; u < U; u++) {
      const int idx = i0 + u * 256;
      const int l = idx % W;
      const int q = idx / W;  // = rl*NC + e
      const int rl = q / NC;
      const int e = q - rl * NC;
      vi[u] = vbase + idx;
      si[u] = (idx < n) ? sbase[rl] + p.lane_off[l] + e : 0;
    }
#pragma unroll
    for (int u = 0; u < U; u++)
      if (i0 + u * 256 < n) val[u] = p.to_vector ? src[si[u]] : src[vi[u]];
#pragma unroll
    for (int u = 0; u < U; u++)
      if (i0 + u * 256 < n) {
        if (p.to_vector)
          dst[vi[u]] = val[u];
        else
          dst[si[u]] = val[u];
      }
  }
}

// Staged variant for 8-byte complex numbers (fp32): with direct per-element copies the scalar side is touched
// in 8-byte pieces scattered over W streams (ncu: 8 sectors/request, 19 % L2 hits, 5.4 TB/s).  Here a block
// moves TR vector records through shared memory: each side is read / written in ITS OWN natural order
// (vector side: one contiguous range; scalar side: for every lane a run of whole records), so every warp
// request is 256 contiguous bytes on both sides; the transposition happens in shared memory.
template <typename C2, int W, int TR, int NC>
__global__ void __launch_bounds__(256) su3_convert_staged_kernel(const ConvertParams p) {
  extern __shared__ __align__(128) unsigned char smem[];
  constexpr int TS = W + 1;  // padded row of one element vector: the transposed accesses (stride TS) stay conflict-free
  C2 *tile = reinterpret_cast<C2 *>(smem);                                   // [TR*NC][TS], the vector-layout image
  long long *sbase = reinterpret_cast<long long *>(smem + sizeof(C2) * TR * NC * TS);
  const long long rec0 = (long long)blockIdx.x * TR;
  const long long left = p.nrec - rec0;
  const int nr = left < TR ? (int)left : TR;
  if ((int)threadIdx.x < nr) {
    const long long rec = rec0 + threadIdx.x;
    long long o = rec / p.nl;
    const int mu = (int)(rec - o * p.nl);
    long long site = 0;
#pragma unroll
    for (int d = 0; d < 4; d++) {
      const long long q = o / p.r[d];
      site += (o - q * p.r[d]) * p.sstride[d];
      o = q;
    }
    sbase[threadIdx.x] = (site * p.nl + mu) * NC;
  }
  __syncthreads();
  const C2 *src = reinterpret_cast<const C2 *>(p.src);
  C2 *dst = reinterpret_cast<C2 *>(p.dst);
  const long long vbase = rec0 * NC * W;
  const int n = nr * NC * W, m = nr * NC;
  constexpr int U = 4;
  if (p.to_vector) {
    for (int i0 = threadIdx.x; i0 < n; i0 += 256 * U) {
      C2 val[U];
      int ti[U];
#pragma unroll
      for (int u = 0; u < U; u++) {
        const int idx = i0 + u * 256;  // scalar-natural order: lane slowest, then record, element fastest
        const int l = nr == TR ? idx / (TR * NC) : idx / m;
        const int k = idx - l * m, rl = k / NC, e = k - rl * NC;
        ti[u] = (rl * NC + e) * TS + l;
        if (idx < n) val[u] = src[sbase[rl] + p.lane_off[l] + e];
      }
#pragma unroll
      for (int u = 0; u < U; u++)
        if (i0 + u * 256 < n) tile[ti[u]] = val[u];
    }
    __syncthreads();
    if (W >= 2 && sizeof(C2) == 8) {  // vector side in 16-byte pieces: two lanes of one element vector
      float4 *d4 = reinterpret_cast<float4 *>(dst + vbase);
      for (int h = threadIdx.x; h < n / 2; h += 256) {
        const int idx = 2 * h;
        const float2 v0 = *reinterpret_cast<const float2 *>(&tile[(idx / W) * TS + idx % W]);
        const float2 v1 = *reinterpret_cast<const float2 *>(&tile[(idx / W) * TS + idx % W + 1]);
        d4[h] = make_float4(v0.x, v0.y, v1.x, v1.y);
      }
    } else {
      for (int idx = threadIdx.x; idx < n; idx += 256) dst[vbase + idx] = tile[(idx / W) * TS + idx % W];
    }
  } else {
    if (W >= 2 && sizeof(C2) == 8) {
      const float4 *s4 = reinterpret_cast<const float4 *>(src + vbase);
      for (int h0 = threadIdx.x; h0 < n / 2; h0 += 256 * U) {
        float4 val[U];
#pragma unroll
        for (int u = 0; u < U; u++)
          if (h0 + u * 256 < n / 2) val[u] = s4[h0 + u * 256];
#pragma unroll
        for (int u = 0; u < U; u++)
          if (h0 + u * 256 < n / 2) {
            const int idx = 2 * (h0 + u * 256);
            *reinterpret_cast<float2 *>(&tile[(idx / W) * TS + idx % W]) = make_float2(val[u].x, val[u].y);
            *reinterpret_cast<float2 *>(&tile[(idx / W) * TS + idx % W + 1]) = make_float2(val[u].z, val[u].w);
          }
      }
    } else {
      for (int i0 = threadIdx.x; i0 < n; i0 += 256 * U) {
        C2 val[U];
#pragma unroll
        for (int u = 0; u < U; u++)
          if (i0 + u * 256 < n) val[u] = src[vbase + i0 + u * 256];
#pragma unroll
        for (int u = 0; u < U; u++)
          if (i0 + u * 256 < n) tile[((i0 + u * 256) / W) * TS + (i0 + u * 256) % W] = val[u];
      }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < n; idx += 256) {
      const int l = nr == TR ? idx / (TR * NC) : idx / m;
      const int k = idx - l * m, rl = k / NC, e = k - rl * NC;
      dst[sbase[rl] + p.lane_off[l] + e] = tile[(rl * NC + e) * TS + l];
    }
  }
}


// TMA variant (default for every aligned geometry): NO per-thread global access at all.  For each lane l the
// scalar-side image of a tile of TR consecutive vector records is a handful of CONTIGUOUS runs (one, unless the tile
// crosses a row of the sub-lattice: runs break every p.run_recs records), so lane l's data moves between global
// memory and row l of a shared-memory tile with 1-D bulk copies issued by thread l; the vector side of the tile is
// one contiguous range and moves with a single bulk copy.  In between, the block transposes rows <-> element
// vectors through registers, in place ([lane][k] with a padded, conflict-free pitch <-> dense [k][lane]).
// Bulk copies need 16-byte alignment: with 8-byte complex numbers (fp32) the host only selects this kernel when every
// run starts and ends on an even complex index (true for every even lattice); otherwise the staged kernel above runs.
template <typename C2, int W, int NC, int N, int NT>
__global__ void __launch_bounds__(NT, 8) su3_convert_tma_kernel(const ConvertParams p) {
  constexpr int CB = (int)sizeof(C2);
  constexpr int TR = N / (NC * W);      // records per tile
  constexpr int PER = (N + NT - 1) / NT;
  static_assert(TR * NC * W == N && TR >= 1, "tile must hold whole records");
  extern __shared__ __align__(128) unsigned char smem[];
  C2 *tile = reinterpret_cast<C2 *>(smem);
  const int pitch = p.pitch;
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem + (size_t)CB * (W * pitch > N ? W * pitch : N));
  const int tid = threadIdx.x;
  const long long rec0 = (long long)blockIdx.x * TR;
  const long long left = p.nrec - rec0;
  const int nr = left < TR ? (int)left : TR;
  const int n = nr * NC * W;
  const unsigned char *src = reinterpret_cast<const unsigned char *>(p.src);
  unsigned char *dst = reinterpret_cast<unsigned char *>(p.dst);
  if (tid == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
    fence_proxy_async();
  }
  __syncthreads();
  // scalar-side complex index of (vector record rec, lane 0, element 0): the virtual-node map S3 for the outer site.
  // Record and site indices fit 31 bits (one launch has < 2^31 blocks of >= 1 record and the host checks the volume),
  // so the decomposition runs in 32-bit arithmetic; only the final complex index is 64-bit.
  auto sbase = [&](long long rec) {
    unsigned o = (unsigned)rec / (unsigned)p.nl;
    const unsigned mu = (unsigned)rec - o * (unsigned)p.nl;
    unsigned site = 0;
#pragma unroll
    for (int d = 0; d < 4; d++) {
      const unsigned q = o / (unsigned)p.r[d];
      site += (o - q * (unsigned)p.r[d]) * (unsigned)p.sstride[d];
      o = q;
    }
    return ((long long)site * p.nl + mu) * NC;
  };
  // lane l's runs of the tile: [a, b) in records, cut at multiples of run_recs
  auto for_runs = [&](auto &&fn) {
    long long a = rec0;
    const long long end = rec0 + nr;
    while (a < end) {
      long long b = (a / p.run_recs + 1) * p.run_recs;
      if (b > end) b = end;
      fn(a, b);
      a = b;
    }
  };
  if (p.to_vector) {
    if (tid < 32) {
      if (tid == 0) mbar_arrive_expect_tx(bar, (uint32_t)n * CB);
      __syncwarp();
      if (tid < W) {
        const long long loff = p.lane_off[tid];
        for_runs([&](long long a, long long b) {
          bulk_g2s(tile + (size_t)tid * pitch + (a - rec0) * NC, src + (size_t)(sbase(a) + loff) * CB,
                   (uint32_t)((b - a) * NC) * CB, bar);
        });
      }
    }
  } else if (tid == 0) {
    mbar_arrive_expect_tx(bar, (uint32_t)n * CB);
    bulk_g2s(tile, src + (size_t)rec0 * NC * W * CB, (uint32_t)n * CB, bar);
  }
  mbar_wait(bar, 0);
  // Slot idx = i*NT + tid of the block handles element (lane l, row index k).  Plain order (l fastest) is conflict-free on
  // both sides for 16-byte complex numbers and for W <= 8; with 8-byte complex numbers and W >= 16 a half-warp would hit
  // 16 rows whose bases are all even (rows are 16-byte aligned), i.e. 8 bank pairs: there lanes 0-7 of a 16-lane group
  // take row 2j and lanes 8-15 row 2j+1 in one half-warp, the other way round in the next (pitch = 2 mod 16).
  // Either way (l, k) is LINEAR in i -- l fixed per thread, k = k0 + i*DK -- so both passes are a pointer walk with a
  // constant stride: two instructions per element.  (Decoding idx per element cost ~50 instructions each and made the
  // fp32 kernel issue-bound at W >= 16: ncu, math-pipe throttle and 0.95 eligible warps per cycle.)
  const int K = nr * NC;
  int l, k0;
  constexpr bool SWZ = CB == 8 && W >= 16;
  constexpr int DK = SWZ ? 2 * (NT / 32) / (W / 16) : NT / W;  // rows advanced per i
  static_assert(NT % 32 == 0 && NT % W == 0 && (!SWZ || (NT / 32) % (W / 16) == 0), "slot order must be linear in i");
  if constexpr (SWZ) {
    constexpr int G = W / 16;  // 16-lane groups per record
    const int i5 = tid & 31, w = tid >> 5;
    l = 16 * (w % G) + (i5 & 15);
    k0 = 2 * (w / G) + (((i5 >> 4) + ((i5 & 15) >> 3)) & 1);
  } else {
    l = tid % W;
    k0 = tid / W;
  }
  const int row = l * pitch + k0, dense = k0 * W + l;     // element (l, k0) in the [lane][k] rows / in the dense [k][lane] tile
  const C2 *rp = tile + (p.to_vector ? row : dense);
  C2 *wp = tile + (p.to_vector ? dense : row);
  const int rs = p.to_vector ? DK : DK * W, ws = p.to_vector ? DK * W : DK;
  C2 v[PER];
  if (nr == TR) {
#pragma unroll
    for (int i = 0; i < PER; i++) v[i] = rp[i * rs];
    __syncthreads();
#pragma unroll
    for (int i = 0; i < PER; i++) wp[i * ws] = v[i];
  } else {  // the last, ragged block
#pragma unroll
    for (int i = 0; i < PER; i++)
      if (k0 + i * DK < K) v[i] = rp[i * rs];
    __syncthreads();
#pragma unroll
    for (int i = 0; i < PER; i++)
      if (k0 + i * DK < K) wp[i * ws] = v[i];
  }
  fence_proxy_async();
  __syncthreads();
  if (p.to_vector) {
    if (tid == 0) {
      bulk_s2g(dst + (size_t)rec0 * NC * W * CB, tile, (uint32_t)n * CB);
      bulk_commit();
      bulk_wait_read<0>();  // the tile may be handed to the next block once the store has READ it; the grid's completion covers the write
    }
  } else if (tid < W) {
    const long long loff = p.lane_off[tid];
    for_runs([&](long long a, long long b) {
      bulk_s2g(dst + (size_t)(sbase(a) + loff) * CB, tile + (size_t)tid * pitch + (a - rec0) * NC, (uint32_t)((b - a) * NC) * CB);
    });
    bulk_commit();
    bulk_wait_read<0>();
  }
}

// ---------------------------------------------------------------- faces of a slab (multi-GPU Cshift)
// A lattice split into x_dim slabs over ranks needs, for a shift along dim, the planes x_dim in [plane0, plane0+n) of a
// neighbouring rank's slab.  One kernel moves such a FACE between any two of: a field in its own layout (scalar or
// vector: the index function is S2/S3), and a packed buffer in plane order -- matrix b of the buffer is
// (site of the face in lexicographic order with x_dim - plane0 in place of x_dim, x0 fastest)*nl + mu, its NC complex
// numbers adjacent.  pack = field -> buffer (what is sent), unpack = buffer -> field (what was received), copy =
// field -> field (the source may be PEER memory mapped over NVLink: the exchange is then this one launch).
// One thread per complex number, consecutive threads = consecutive elements of one face matrix.
struct FaceSide {
  int packed;   // 1: packed buffer (plane order); 0: field
  int plane0;   // field: first plane of the face along dim
  int W, nl;
  int L[4], simd[4];
};
struct FaceParams {
  void *dst;
  const void *src;
  FaceSide d, s;
  int dim;
  int F[4];          // extents of the face: L with L[dim] replaced by the number of planes
  long long ncplx;   // complex numbers to move = prod(F) * nl * NC
};

template <int NC, typename IT>
__device__ __forceinline__ IT face_index(const FaceSide &g, int dim, const int (&c)[4], int mu, int e, IT packed_idx) {
  if (g.packed) return packed_idx;
  if (g.W == 1) {  // scalar layout: no virtual-node map
    IT site = 0, sstride = 1;
#pragma unroll
    for (int k = 0; k < 4; k++) {
      site += (c[k] + (k == dim ? g.plane0 : 0)) * sstride;
      sstride *= g.L[k];
    }
    return (site * g.nl + mu) * NC + e;
  }
  IT o = 0, ostride = 1;
  int l = 0, lstride = 1;
#pragma unroll
  for (int k = 0; k < 4; k++) {
    const int x = c[k] + (k == dim ? g.plane0 : 0);
    if (g.simd[k] > 1) {  // only split dimensions cost a division
      const int r = g.L[k] / g.simd[k];
      const int ic = x / r;
      o += (x - ic * r) * ostride;  ostride *= r;
      l += ic * lstride;  lstride *= g.simd[k];
    } else {
      o += x * ostride;  ostride *= g.L[k];
    }
  }
  return ((o * g.nl + mu) * NC + e) * g.W + l;
}

// One thread per complex number.  IT = int whenever every complex index of both sides fits 31 bits (the host checks):
// the kernel spends its time on integer divisions, not on memory (a 4-way unrolled version with more loads in flight
// was 2.6 x SLOWER), so 64-bit ones are avoided and unsplit dimensions skip theirs.
template <typename C2, int NC, typename IT>
__global__ void __launch_bounds__(256) su3_face_kernel(const FaceParams p) {
  const IT stride = (IT)gridDim.x * blockDim.x, n = (IT)p.ncplx;
  const int nlsh = p.d.nl == 4 ? 2 : 0;  // n_lorentz is 1 or 4
  for (IT i = (IT)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const int e = (int)(i % NC);
    IT b = i / NC;
    const int mu = (int)(b & (p.d.nl - 1));
    b >>= nlsh;
    int c[4];
#pragma unroll
    for (int k = 0; k < 3; k++) {
      const IT q = b / p.F[k];
      c[k] = (int)(b - q * p.F[k]);
      b = q;
    }
    c[3] = (int)b;
    const IT si = face_index<NC, IT>(p.s, p.dim, c, mu, e, i);
    const IT di = face_index<NC, IT>(p.d, p.dim, c, mu, e, i);
    reinterpret_cast<C2 *>(p.dst)[di] = reinterpret_cast<const C2 *>(p.src)[si];
  }
}

}  // namespace su3

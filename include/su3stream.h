/* su3stream.h -- C ABI of libsu3stream: lattice-wide, site-wise SU(3)xSU(3)
 * streaming products on NVIDIA B200 (sm_100a).
 *
 * What the calls compute follows arXiv:1710.09409 (P:N = PAPER.md line N):
 *   - a lattice field = one object per (outer) site, `Lattice<obj>`        P:76-89,  Listing 1
 *   - obj = complex 3x3 matrix (`Su3f`), the streaming test `z = x*y`      P:113-126, section 4, Listing 3
 *   - composite expressions evaluated in ONE pass over the sites           P:91-109, Listing 2
 *   - scalar ("naive", AoS) layout
 *   - vector layout: the lattice is split into N_sub virtual nodes, the
 *     split lives at the level of the basic complex type
 *   - extract / merge: lane l of each of the 9 element vectors <-> one
 *     scalar 3x3 matrix (this defines su3_convert)                         P:174-181, Listing 4
 *   - a same-run streaming ceiling next to every bandwidth number          P:199-201 (STREAM triad lines)
 * Where the paper is silent the readings S1..S19 of DESIGN.md apply.
 *
 * Conventions (all calls)
 *   - extern "C", plain pointers and sizes; no exceptions cross the ABI.
 *   - DEVICE memory is the caller's (e.g. a torch tensor): su3_field_wrap records
 *     the pointer and never allocates, frees or touches it.  A su3_field handle is
 *     host memory owned by the library until su3_field_free.
 *   - Every call returns su3_status.  On failure nothing is launched, outputs are
 *     untouched, and su3_last_error() (thread-local) describes the failure.
 *   - Arithmetic calls enqueue on `cuda_stream` (a cudaStream_t passed as void*;
 *     NULL = legacy default stream) and return without synchronising.
 *   - `z` may be the SAME field as any input.  Partially overlapping fields are
 *     undefined.
 *   - Handles are immutable after wrap; every call is thread-safe.  The only state besides handles is per
 *     thread (the last-error string and the launch knobs of su3_tune_set) or keyed by device ordinal (cached
 *     device facts and per-kernel attributes) or by (device, caller stream) (su3_eval_host's copy streams).
 *   - A call launches on the device that is CURRENT on the calling thread; su3_field_wrap records which device
 *     owns the memory (when the runtime can tell) and a call whose fields live elsewhere returns
 *     SU3_ERR_MISMATCH instead of launching.  One process may drive several GPUs.
 *   - There is no CPU fallback anywhere: without a CUDA device the arithmetic
 *     calls return SU3_ERR_CUDA.
 *
 * Data layout (reals are IEEE fp32 or fp64; a complex number is (re, im) adjacent)
 *   matrix element (i,j) is e = 3*i + j (row-major, S1); matrix index of (site, mu)
 *   is m = site*n_lorentz + mu (S6); site = x0 + L0*(x1 + L1*(x2 + L2*x3)) (S2).
 *   SU3_SCALAR : real offset = (m*9 + e)*2 + reim
 *   SU3_VECTOR : real offset = (((o*n_lorentz + mu)*9 + e)*W + l)*2 + reim, with
 *                r[d] = L[d]/simd[d], oc[d] = x[d] mod r[d], ic[d] = x[d] div r[d],
 *                o = lexicographic index of oc over r, l = lexicographic index of ic
 *                over simd, both d=0 fastest (the virtual-node map, S3).
 *   Default split of W over the dimensions (simd all 0, S4): factors of two handed
 *   out starting at d=3 and moving down, wrapping: 2->{1,1,1,2} 4->{1,1,2,2}
 *   8->{1,2,2,2} 16->{2,2,2,2} 32->{2,2,2,4}.
 */
#ifndef SU3STREAM_H
#define SU3STREAM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SU3_OK = 0,
  SU3_ERR_NULL = 1,     /* a required pointer argument is NULL                       */
  SU3_ERR_INVALID = 2,  /* bad enum, L[d]<=0, n_lorentz not in {1,4}, W not a power
                           of two in 1..32, W!=1 with SU3_SCALAR, prod(simd)!=W,
                           L[d] % simd[d] != 0                                      */
  SU3_ERR_MISMATCH = 3, /* operands disagree in L, n_lorentz, prec (and, for the
                           arithmetic calls, layout / W / simd)                     */
  SU3_ERR_ALIGN = 4,    /* device pointer not 16-byte aligned                        */
  SU3_ERR_SIZE = 5,     /* buffer smaller than su3_field_bytes                       */
  SU3_ERR_CUDA = 6      /* CUDA runtime error (string in su3_last_error)             */
} su3_status;

typedef enum { SU3_F32 = 4, SU3_F64 = 8 } su3_prec;          /* bytes per real */
typedef enum { SU3_SCALAR = 0, SU3_VECTOR = 1 } su3_layout;

/* Plain data, caller-owned, copied on use. */
typedef struct {
  int32_t L[4];      /* lattice extents                                              */
  int32_t n_lorentz; /* 1 (colour-matrix field) or 4 (gauge-field shape)             */
  int32_t prec;      /* su3_prec                                                     */
  int32_t layout;    /* su3_layout                                                   */
  int32_t W;         /* sites interleaved lane-wise; must be 1 for SU3_SCALAR        */
  int32_t simd[4];   /* virtual-node grid, product = W; all 0 => default split (S4)  */
} su3_desc;

typedef struct su3_field su3_field; /* opaque: validated descriptor + device pointer */

/* Launch knobs of the CALLING THREAD (0 = library default).  They never change results, only speed; bench.py and
 * the tests use them to pin the launch configuration that is being measured.  Meaning per kernel family:
 *   pipeline (su3_mul/mul3/mul_add/add, su3_matvec): tile_mats, stages = ring depth, ctas_per_sm, l2_hint, path
 *   su3_copy: tile = tile_mats x matrix bytes, stages, ctas_per_sm, l2_hint; path = 2 selects the plain LDG copy
 *   su3_expr: programs on the ahead-of-time menu run on the pipeline (knobs as above); path = 3 forces the interpreter,
 *             whose knobs are tile_mats = matrices per stage and operand (default 32; 64 for fp32 programs with <= 3
 *             operands), stages = ring depth per CTA (default 2) and ctas_per_sm (an upper limit on its 96-thread CTAs per SM)
 *   su3_cshift / su3_mul_shift: default = the pipeline with a shifted operand (knobs as above); path = 2 the register
 *             kernels, path = 3 the cp.async-gather Cshift; for those ctas_per_sm = blocks per SM of the grid
 *   su3_convert: default = TMA bulk copies on both sides;
 *                path = 3 the per-thread kernel staged through shared memory, path = 2 the unstaged kernel */
typedef struct {
  int32_t tile_mats;    /* matrices per pipeline tile: 32, 64 or 128 (su3_copy: x matrix bytes) */
  int32_t stages;       /* shared-memory ring depth, 2..16                             */
  int32_t ctas_per_sm;  /* persistent CTAs per SM, 1..8                                 */
  int32_t l2_hint;      /* 0 auto, 1 none, 2 evict_first loads+stores, 3 keep the first l2_pin_mb MB of every
                           operand in L2 across calls (evict_last), stream the rest (evict_first)     */
  int32_t path;         /* 0 auto (by footprint and layout), 1 TMA-bulk pipeline, 2 direct per-lane LDG, 3 warp-staged */
  int32_t l2_pin_mb;    /* see l2_hint = 3                                                */
  int32_t reserved[2];
} su3_tune;

/* Never NULL; thread-local; valid until the next failing call on this thread. */
const char *su3_last_error(void);

/* Library version string, e.g. "su3stream 0.1 (sm_100a)". */
const char *su3_version(void);

/* Bytes a field of this descriptor occupies: volume * n_lorentz * 18 * prec.
 * Validates the descriptor (SU3_ERR_INVALID).  Host-only, needs no GPU. */
su3_status su3_field_bytes(const su3_desc *desc, size_t *nbytes);

/* Normalise a descriptor: validates it and fills simd[] with the split in use. */
su3_status su3_desc_normalize(const su3_desc *desc, su3_desc *out);

/* Wrap caller-owned DEVICE memory.  dev_ptr must be 16-byte aligned (SU3_ERR_ALIGN)
 * and nbytes >= su3_field_bytes (SU3_ERR_SIZE).  Host-only bookkeeping. */
su3_status su3_field_wrap(const su3_desc *desc, void *dev_ptr, size_t nbytes, su3_field **out);
su3_status su3_field_free(su3_field *f); /* frees the handle only, never the device memory */
su3_status su3_field_desc(const su3_field *f, su3_desc *out); /* normalised descriptor     */
su3_status su3_field_ptr(const su3_field *f, void **dev_ptr, size_t *nbytes);

/* Host-side index map (for tests and for filling a field by hand): offset IN REALS of
 * (site, mu, row i, col j, reim) for this descriptor.  SU3_ERR_INVALID if out of range. */
su3_status su3_index(const su3_desc *desc, int64_t site, int mu, int i, int j, int reim, int64_t *off);

/* z = x*y, site by site: z_ij = sum_k x_ik y_kj (Listing 3).  All three fields
 * must have identical descriptors (SU3_ERR_MISMATCH).  A1 (scalar) / A2 (vector). */
su3_status su3_mul(su3_field *z, const su3_field *x, const su3_field *y, void *cuda_stream);

/* z = (x*y)*w in one pass, x*y kept in registers (composite expressions are
 * evaluated inside the one site loop; left-associative as C++ parses x*y*w).  A3. */
su3_status su3_mul3(su3_field *z, const su3_field *x, const su3_field *y, const su3_field *w, void *cuda_stream);

/* z = x*y + v in one pass (the `v1+v2+v1*v2` pattern of P:104-106 on matrices).  A4. */
su3_status su3_mul_add(su3_field *z, const su3_field *x, const su3_field *y, const su3_field *v, void *cuda_stream);

/* z = x + y, element-wise (P:104 `v3=v1+v2`).  Also the 2-read-1-write streaming
 * reference (the analogue of the paper's STREAM line). */
su3_status su3_add(su3_field *z, const su3_field *x, const su3_field *y, void *cuda_stream);

/* z = value of a small expression tree over matrix fields, evaluated site by site in ONE pass, intermediates
 * in registers / shared memory only (Listings 1-2: `eval(ss, expr)` inside the site loop, e.g.
 * `v3 = v1+v2+v1*v2`).  `program` is the tree in postfix order as a NUL-terminated string: a digit '0'..'7'
 * pushes operands[digit] at this site; '+', '-', '*' pop b, then a, and push a+b, a-b, a.b (3x3 complex
 * product).  Examples: "01*" = su3_mul, "01*2*" = su3_mul3, "01*2+" = su3_mul_add (bit-identical to them),
 * "01+01*+" = v1+v2+v1*v2.  At most 32 tokens, 16 operators, stack depth 8; every operand 0..n_operands-1
 * must be used; exactly one value must remain (SU3_ERR_INVALID otherwise).  All fields must have identical
 * descriptors and be of one kind -- all colour-matrix fields, or all real scalar fields (su3_real_wrap; '*' is then
 * the element-wise product) -- else SU3_ERR_MISMATCH; z may be the same field as any operand.  Every distinct
 * operand adds one read stream: bytes = (n_operands + 1) * field bytes. */
su3_status su3_expr(su3_field *z, const char *program, const su3_field *const *operands, int n_operands,
                    void *cuda_stream);

/* The register-machine listing the host compiler produces for `program` (what the interpreter kernel executes),
 * one instruction per line: "<op> <a> <b> [spill tK]" with op in {mul, add, sub, copy}, sources oK = operand K,
 * tK = temporary K, acc = accumulator; "spill tK" = the accumulator is parked in temporary K first.  Written
 * NUL-terminated into buf (SU3_ERR_SIZE if it does not fit).  Host-only; for debugging and for the tests. */
su3_status su3_expr_disasm(const char *program, int n_operands, char *buf, size_t buf_len);

/* Which kernel su3_expr would run for `program`: "menu <row> <row's postfix> <operand of slot 0> <slot 1> ..." when the
 * compiled program is one of the ahead-of-time rows of the pipeline kernel (up to a renaming of the operands and the
 * order of the sources of '+'), else "interpreter".  The rows, as postfix programs over distinct fields: 01* 01*2* 01*2+
 * 01+ 01+01*+ 01*23*+ 01*23*- 01*2- 01+2+ 01+2+3+ 01- 01*2*3* 012** 01*23** (and, for real scalar fields, 01+ 01* 01+01*+).
 * real_fields != 0: the operands are real scalar fields ('*' is element-wise).  Both routes give bit-identical
 * results; the menu rows run at the copy ceiling, the interpreter at 0.8-1.09 x of it for typical programs.  Host-only. */
su3_status su3_expr_plan(const char *program, int n_operands, int real_fields, char *buf, size_t buf_len);

/* Accounting of a program by reading S9: field streams (n_operands + 1) and flops per matrix (198 per '*',
 * 18 per '+' or '-').  Validates the program like su3_expr.  Host-only. */
su3_status su3_expr_cost(const char *program, int n_operands, int32_t *streams, int32_t *flops_per_matrix);

/* Circular shift, Grid's Cshift(x, dim, disp) (P:219 names it as the next obstacle after the site-local
 * product): z[s] = x[s + disp*dim_hat], periodic ON THE LOCAL LATTICE OF THE HANDLE (one rank's slab in a multi-GPU
 * job: see the su3_face_* calls below), for every site s and every mu; dim in 0..3, disp any integer.  A pure, bit-exact permutation of matrices in either layout (in the vector layout a step across
 * a sub-lattice boundary moves a matrix to another lane).  Identical descriptors (SU3_ERR_MISMATCH); z and
 * x must not be the same field (SU3_ERR_MISMATCH); dim outside 0..3 -> SU3_ERR_INVALID. */
su3_status su3_cshift(su3_field *z, const su3_field *x, int dim, int disp, void *cuda_stream);

/* z[s] = x[s] . y[s + disp*dim_hat] in one pass: the site-local product with a shifted second operand (the
 * building block of covariant shifts and plaquettes).  Same FMA chain as su3_mul: bit-identical to
 * su3_cshift followed by su3_mul.  z may be the same field as x but not as y. */
su3_status su3_mul_shift(su3_field *z, const su3_field *x, const su3_field *y, int dim, int disp, void *cuda_stream);

/* Colour-vector fields (f4; the operand of the Dslash-type stencils): 3 complex numbers per
 * (site, mu) instead of 9, same descriptor, same two layouts with 3 in place of 9:
 *   SU3_SCALAR : real offset = ((m*3) + i)*2 + reim        SU3_VECTOR : (((o*nl + mu)*3 + i)*W + l)*2 + reim
 * su3_vec_bytes = volume * n_lorentz * 6 * prec.  A handle made by su3_vec_wrap is a su3_field of vector kind:
 * su3_field_free / su3_field_desc / su3_field_ptr / su3_copy / su3_convert take it (both operands of the same
 * kind); the matrix-only calls return SU3_ERR_MISMATCH for it. */
su3_status su3_vec_bytes(const su3_desc *desc, size_t *nbytes);
su3_status su3_vec_wrap(const su3_desc *desc, void *dev_ptr, size_t nbytes, su3_field **out);
su3_status su3_vec_index(const su3_desc *desc, int64_t site, int mu, int i, int reim, int64_t *off);

/* y = U.psi, site by site: y_i = sum_j U_ij psi_j (66 flops, 144+48+48 B in fp64 per (site, mu)).  U a
 * colour-matrix field, psi and y colour-vector fields, identical descriptors.  y may be the same field as psi. */
su3_status su3_matvec(su3_field *y, const su3_field *U, const su3_field *psi, void *cuda_stream);

/* Real scalar fields, the operands of the paper's own example of the expression engine (Listing 2:
 * `Lattice<double> v1, v2, v3; v1 = 1.0; v2 = 2.0; v3 = v1+v2+v1*v2;`): one real per (site, mu),
 * su3_real_bytes = volume * n_lorentz * prec.  Element-wise operations only, so the layout of the descriptor
 * does not matter.  A handle made by su3_real_wrap goes to su3_fill, su3_expr (all operands and z of real kind:
 * '+', '-', '*' act element-wise) and su3_field_free/desc/ptr; every other call returns SU3_ERR_MISMATCH for it. */
su3_status su3_real_bytes(const su3_desc *desc, size_t *nbytes);
su3_status su3_real_wrap(const su3_desc *desc, void *dev_ptr, size_t nbytes, su3_field **out);
/* field = value at every (site, mu) (Listing 2: `v1 = 1.0;`).  Real scalar fields only. */
su3_status su3_fill(su3_field *z, double value, void *cuda_stream);

/* Layout conversion scalar <-> vector: a pure, bit-exact permutation of complex numbers,
 * vec[o][mu][e][l] = sca[site(o,l)][mu][e] (extract/merge).  Exactly one of
 * dst/src must be SU3_SCALAR and the other SU3_VECTOR; L, n_lorentz, prec must agree
 * (SU3_ERR_MISMATCH).  dst and src must not alias.  A5. */
su3_status su3_convert(su3_field *dst, const su3_field *src, void *cuda_stream);

/* dst = src, own 128-bit copy kernel: the same-run bandwidth ceiling.  Fields
 * must have identical descriptors.  A6. */
su3_status su3_copy(su3_field *dst, const su3_field *src, void *cuda_stream);

/* Faces of a slab: what a Cshift along `dim` needs from the neighbouring rank when the lattice is split into x_dim slabs
 * over GPUs (the first exchange step of this code base; P:219 names Cshift as the operation after the site-local
 * product, and Grid's Cshift sends exactly such faces).  su3_cshift / su3_mul_shift are periodic on the LOCAL lattice of
 * the handle; a multi-GPU shift = the local shift + these calls around one send/recv (paper_1710_09409_b200/halo.py).
 * The face of planes x_dim in [plane0, plane0 + nplanes) is moved between a field (either layout) and a PACKED device
 * buffer in plane order, the same for every layout so that ranks may exchange it blindly: matrix
 *   b = (x0 + L0*(x1 + L1*(x2 + L2*x3)) with (x_dim - plane0) in place of x_dim and nplanes in place of L[dim]) * n_lorentz + mu
 * sits at complex index b*9 (b*3 for colour-vector fields), row-major, (re, im) adjacent -- i.e. the packed face IS a
 * scalar-layout field of extents L with L[dim] = nplanes.  su3_face_bytes = its size.  Bit-exact permutations.
 *   su3_face_pack  : buffer <- planes of x          su3_face_unpack: planes of z <- buffer
 *   su3_face_copy  : planes [z_plane0, +n) of z <- planes [x_plane0, +n) of x, same descriptor; x may be memory of a PEER
 *                    device mapped into this process (NVLink P2P): the exchange is then this single launch.
 * plane range outside 0..L[dim] -> SU3_ERR_INVALID; buffer too small -> SU3_ERR_SIZE, misaligned -> SU3_ERR_ALIGN; a buffer
 * that is plain device memory of another GPU which the current one cannot reach as a peer -> SU3_ERR_MISMATCH (the runtime
 * is asked where the pointer lives; whether peer access has been ENABLED stays the caller's responsibility, as does the
 * residency of pinned or managed buffers). */
su3_status su3_face_bytes(const su3_field *f, int dim, int nplanes, size_t *nbytes);
su3_status su3_face_pack(void *buf_dev, size_t buf_bytes, const su3_field *x, int dim, int plane0, int nplanes, void *cuda_stream);
su3_status su3_face_unpack(su3_field *z, const void *buf_dev, size_t buf_bytes, int dim, int plane0, int nplanes, void *cuda_stream);
su3_status su3_face_copy(su3_field *z, int z_plane0, const su3_field *x, int x_plane0, int dim, int nplanes, void *cuda_stream);

/* Moving a face WITHOUT any device allocation by anybody.  su3_face_pack + su3_face_unpack need a packed buffer that
 * somebody has to allocate; some users of this library cannot do that at the point where they need a face moved:
 *   - a job whose framework has handed all of HBM to its own pool (a 64^4 run sized for the card, a torch process with
 *     a fixed memory fraction): a cudaMalloc from a plug-in library fails there, or succeeds and fragments the pool;
 *   - a communication thread that overlaps the face exchange with the bulk kernels of other streams: cudaMalloc and
 *     cudaFree serialise against work in flight on the whole device, which is exactly the stall it exists to hide;
 *   - an embedding (another language runtime, a sandboxed driver of this C ABI) that receives raw field pointers from
 *     its host and owns no allocator handle at all.
 * For them the library carries ONE fixed staging area of SU3_STATIC_SCRATCH_BYTES (16 MiB) inside its own device image
 * -- a file-scope device array, so every GPU that loads libsu3stream holds these 16 MiB from the moment the module is
 * loaded until the process exits, whether or not this call is ever used.
 *
 * su3_face_move_static: planes [z_plane0, +nplanes) of z along dim <- planes [x_plane0, +nplanes) of x, staged through
 * that area in the packed plane order described above: two launches of the face kernel (field -> area, area -> field)
 * on cuda_stream.  The result is bit-identical to su3_face_pack followed by su3_face_unpack through a buffer of the
 * caller's.  z and x must agree in L, n_lorentz, precision and kind (SU3_ERR_MISMATCH) but, unlike su3_face_copy, NOT
 * in layout: the packed order is the same for every layout, so a face may go from a vector-layout slab into a
 * scalar-layout one.  z may be x itself (planes are copied inside one field; overlapping source and destination plane
 * ranges are fine, the first launch has read everything before the second writes).  Both fields must live on the
 * current device.  The caller passes only its input and output fields.
 *   Limit   : a face of more than SU3_STATIC_SCRATCH_BYTES (su3_face_bytes tells) is refused with SU3_ERR_SIZE and
 *             nothing is launched -- one x3 plane of a 48^4 fp64 colour-matrix field (15.9 MB) fits, one of 64^4
 *             (37.7 MB) does not; move larger faces in several calls, or use su3_face_pack with your own buffer.
 *   Set-up  : the first call on each device looks up the device address of the area (cudaGetSymbolAddress with that
 *             device current; a failure is returned as SU3_ERR_CUDA).  That look-up may make the runtime load the
 *             module, so make this first call -- any valid call, nplanes = 0 included -- during initialisation, before
 *             any stream capture is begun in the process.  Later calls only launch kernels.
 *   No alloc: no cudaMalloc, cudaFree, stream/event creation or other allocating routine is called, ever.
 *   Sharing : all calls on one device use the same area and it keeps whatever the last call left in it.  Nothing in it
 *             has to start at zero: every byte the second launch reads was written by the first launch of the same
 *             call, so there is nothing to clear.  Calls that can overlap on the GPU -- on different streams, from
 *             different threads or from different handles of the library in one process -- race on the area and may
 *             deliver each other's faces: keep all calls of a device on one stream, or order them with events. */
#define SU3_STATIC_SCRATCH_BYTES (16u << 20)
su3_status su3_face_move_static(su3_field *z, int z_plane0, const su3_field *x, int x_plane0, int dim, int nplanes,
                                void *cuda_stream);

/* Cshift along x3 on one slab of an x3-split lattice with the neighbouring slab mapped into this process (peer memory
 * over NVLink, or simply another field on the same device): z[s] = X[s + disp*e3], X = the slab x continued by x_nbr --
 * the NEXT rank's slab for disp > 0, the PREVIOUS rank's for disp < 0; 0 < |disp| < L[3] of the slab (disp = 0 copies x;
 * SU3_ERR_INVALID beyond).  Identical descriptors, colour-matrix fields.  Exchange and shift are ONE kernel whenever no
 * record mixes lanes of the two slabs (scalar layout, or simd[3] = 1): the TMA copy kernel of su3_cshift reads the runs
 * that leave the slab from x_nbr at the same record offset.  Otherwise (x3 split over virtual nodes) two launches: the
 * periodic shift of x, then su3_face_copy of the |disp| wrapped planes from x_nbr.  Bit-exact either way.  z and x
 * must live on the current device; x_nbr is only read. */
su3_status su3_cshift_slab(su3_field *z, const su3_field *x, const su3_field *x_nbr, int disp, void *cuda_stream);

/* End-to-end z = x*y with HOST buffers: x_host, y_host (inputs) and z_host (output) are host
 * arrays of su3_field_bytes bytes in the layout of the (identical) descriptors of the three
 * DEVICE staging fields zd, xd, yd.  Enqueues, on cuda_stream, chunked host->device copies
 * of x and y, the product kernel per chunk, and the device->host copy of z, overlapped on
 * internal copy streams, then makes cuda_stream wait for all of it.  Does not synchronise
 * the host; pinned host memory is needed for the copies to be asynchronous.  `chunks` <= 0
 * picks a default; more than 64 chunks -> SU3_ERR_INVALID.  The internal copy streams and events are
 * kept per (device, cuda_stream): threads driving different streams do not serialise on each other. */
su3_status su3_mul_host(void *z_host, const void *x_host, const void *y_host,
                        su3_field *zd, su3_field *xd, su3_field *yd, int chunks, void *cuda_stream);

/* The same chunked, copy/compute-overlapped pipeline for the three ahead-of-time expressions, with operands that
 * may already be resident: op = SU3_OP_MUL (z = x*y), SU3_OP_MUL3 (z = x*y*u), SU3_OP_MUL_ADD (z = x*y + u).  A NULL
 * x_host / y_host / u_host means "that operand is already in its device field" (no copy); a NULL z_host leaves the
 * result in zd only.  u_host and ud must be NULL for SU3_OP_MUL.  Otherwise as su3_mul_host. */
typedef enum { SU3_OP_MUL = 0, SU3_OP_MUL3 = 1, SU3_OP_MUL_ADD = 2 } su3_op;
su3_status su3_eval_host(int op, void *z_host, const void *x_host, const void *y_host, const void *u_host,
                         su3_field *zd, su3_field *xd, su3_field *yd, su3_field *ud, int chunks, void *cuda_stream);

/* Which launch su3_mul / su3_mul3 / su3_mul_add (op = su3_op) would make on fields of this descriptor, with the calling
 * thread's knobs (su3_tune_set) on the current device -- the library picks kernel family, tile, ring depth and L2 policy
 * from the footprint (3 or 4 fields) against the L2 size, and this call reports that choice without launching anything:
 *   "<family> tile=<matrices> depth=<ring depth> ctas=<per SM> grid=<blocks> block=<threads> smem=<bytes> l2=<policy> pin_bytes=<n>"
 * family: "direct" (per-lane loads, L2-resident vector layouts), "warp" (warp-staged, L2-resident), "pipe" (the TMA
 * pipeline); l2: "none", "evict_first", or "pin" = the first pin_bytes of every operand are kept in L2 from call to call
 * (evict_last) and the rest is streamed -- chosen automatically between 0.6 and 2 x L2 for repeated calls on the same
 * fields (the loop of Listing 3), never for the chunk launches of su3_eval_host nor for shifted operands.
 * Written NUL-terminated into buf (SU3_ERR_SIZE if it does not fit).  Host arithmetic only, but it needs the current
 * device's facts: SU3_ERR_CUDA without a device.  For bench.py's sweep rows and for the tests. */
su3_status su3_launch_plan(const su3_desc *desc, int op, char *buf, size_t buf_len);

/* Destroys the copy streams and events that su3_mul_host / su3_eval_host created (after waiting for their own
 * copies).  Optional teardown; must not run concurrently with those two calls.  At most 64 distinct
 * (device, stream) pairs may hold such resources at a time (SU3_ERR_SIZE beyond that). */
su3_status su3_host_release(void);

/* Launch knobs of the calling thread (see su3_tune; thread-local, so concurrent threads never race on them).
 * su3_tune_set(NULL) restores the defaults. */
su3_status su3_tune_set(const su3_tune *t);
su3_status su3_tune_get(su3_tune *out);

/* Number of kernels this library has launched in this process (monotonic). */
int64_t su3_launch_count(void);

/* Device facts the harness prints next to its numbers: SM count, L2 bytes, memory clock
 * (kHz), bus width (bits), of the current CUDA device.  SU3_ERR_CUDA without a device. */
su3_status su3_device_info(int32_t *sm_count, int64_t *l2_bytes, int32_t *mem_clock_khz, int32_t *bus_width_bits);

/* Name (NUL-terminated, truncated to buf_len) and ordinal of the current CUDA device. */
su3_status su3_device_name(char *buf, size_t buf_len, int32_t *ordinal);

#ifdef __cplusplus
}
#endif
#endif /* SU3STREAM_H */

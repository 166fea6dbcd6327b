/* ==============================================================================================
 * lqx -- site-parallel evaluation of QDP++-style lattice field expressions on one B200 (sm_100a).
 *
 * C-ABI boundary of the hot path of arXiv 1105.2279 (F. Winter, "Accelerating QDP++ using GPUs").
 * The paper's method evaluates an expression over lattice-wide objects by running the whole
 * expression once per site, with no temporaries (PAPER.md:61-63 sec.3, :115 sec.5.4), including
 * the nearest-neighbour `shift` operator that reads its operand through a periodic site table
 * (sec.5.2).  This library is that evaluation for a fixed catalogue of
 * expressions (BASELINE.json north_star / configs; SURVEY.md sec.8(a),(b)): every call below is
 * ONE fused CUDA kernel pass (plus a tiny deterministic second stage for reductions).
 *
 * Conventions (all calls)
 *   * return 0 (LQX_OK) on success, a negative lqx_status otherwise; nothing is printed, nothing
 *     aborts, no exception crosses the boundary.  lqx_last_error(ctx) holds a detail string.
 *   * `host` pointers are caller-owned host memory, touched only during the call.
 *     `dev`  pointers are device memory on the context's device.
 *   * External ("QDP++ order", reading A7) layout of a host field:
 *     site-major array of structs, sites lexicographic with x0 fastest,
 *     site(x) = x0 + L0*(x1 + L1*(x2 + L2*x3)); inside a site, outer->inner:
 *     [spin][colour row][colour column][re,im]; real index of a colour matrix element
 *     ((s*3+i)*3+j)*2+c, fermion ((s*4+a)*3+i)*2+c, colour vector (s*3+i)*2+c, complex s*2+c.
 *   * Internal device layout: blocked site-fastest structure of arrays.  Sites are grouped in
 *     blocks of 32 consecutive lexicographic sites; inside a block the 2*kind reals of a site
 *     object (QDP order) are cut into 128-bit chunks of W = 16/prec reals, and chunk q of the 32
 *     sites is contiguous (a trailing half chunk of 2 reals exists for fp32 when 2*kind % 4 == 2).
 *     Element (site s, real r), q = r / W, lies at
 *         (s/32)*32*2*kind + q*32*W + (s%32)*w_q + (r - q*W),   w_q = W (full chunk) or 2 (half).
 *     lqx_field_offset() evaluates this; a field occupies lqx_padded_volume()*2*kind reals.
 *   * shift(f, LQX_FORWARD, mu)(x) = f(x + mu^), shift(f, LQX_BACKWARD, mu)(x) = f(x - mu^)
 *     (fixed by Listing 1 line 25 against Eq. 2), periodic in every
 *     direction.
 *   * Evaluation calls are asynchronous on the context's stream.  pop, the reductions and the
 *     *_host calls synchronise that stream.  A context is used from one host thread at a time.
 *   * All operands of a call must belong to the same context and have the same precision
 *     (QDP++ fixes the precision per build): otherwise LQX_ETYPE / LQX_EGEOM.
 *   * Site-local forms may alias destination and operands; anything that reads an operand
 *     through a shift must be out of place (LQX_EALIAS).
 *   * Real scalars arrive as double and are rounded once to the field precision (reading A10).
 * ============================================================================================== */
#ifndef LQX_H
#define LQX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lqx_ctx lqx_ctx;     /* opaque; owned by the library, destroyed by lqx_finalize   */
typedef struct lqx_field lqx_field; /* opaque handle; storage owned by the library or borrowed   */

typedef enum { LQX_F32 = 4, LQX_F64 = 8 } lqx_prec; /* bytes per real */
/* complex numbers per site: LatticeComplex, LatticeColorVector, LatticeColorMatrix, LatticeFermion
 * (PAPER.md:69 sec.4, :138-145 Listing 1; BASELINE.json configs[1],[4]) */
typedef enum { LQX_COMPLEX = 1, LQX_COLORVEC = 3, LQX_COLORMAT = 9, LQX_FERMION = 12 } lqx_kind;
typedef enum { LQX_BACKWARD = -1, LQX_FORWARD = +1 } lqx_dir;

typedef enum {
    LQX_OK = 0,
    LQX_EINVAL = -1,  /* null pointer, mu outside 0..3, dir not +-1, nsteps < 0, bad enum        */
    LQX_ETYPE = -2,   /* operand kind / precision does not fit the expression                   */
    LQX_EGEOM = -3,   /* extent < 1, V >= 2^31, operands from different contexts                */
    LQX_EALIAS = -4,  /* destination aliases an operand that is read through a shift            */
    LQX_ECUDA = -5,   /* a CUDA call failed; lqx_last_error has cudaGetErrorString              */
    LQX_ENOMEM = -6   /* host or device allocation failed                                       */
} lqx_status;

/* ---------------------------------------------------------------------------------------------
 * Geometry (the paper's "layout" + site tables)
 * ------------------------------------------------------------------------------------------- */
/* Create a context for an L0 x L1 x L2 x L3 periodic lattice on CUDA device `device`.
 * `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream); the library
 * never creates or destroys it.  Host pointer in (dims), handle out. */
int lqx_init(const int dims[4], int device, void* cuda_stream, lqx_ctx** out);
/* Frees every field handle still alive, library-owned device memory and scratch
 * (the paper's theDeviceStorage::freeAll). */
int lqx_finalize(lqx_ctx* ctx);
/* Switch the stream later calls are enqueued on; synchronises the old stream first (the context's scratch
 * buffers are ordered by its stream). */
int lqx_set_stream(lqx_ctx* ctx, void* cuda_stream);
int64_t lqx_volume(const lqx_ctx* ctx);       /* V = L0*L1*L2*L3, or negative status            */
int64_t lqx_padded_volume(const lqx_ctx* ctx); /* V rounded up to whole 32-site blocks          */
/* Element offset of (site, QDP-order real index) inside a field of this kind/precision in the
 * internal layout, or a negative status. */
int64_t lqx_field_offset(const lqx_ctx* ctx, lqx_kind kind, lqx_prec prec, int64_t site, int real_index);
/* Bytes of device memory a field of this kind/precision occupies in the internal layout. */
int64_t lqx_field_bytes(const lqx_ctx* ctx, lqx_kind kind, lqx_prec prec);
/* Periodic neighbour table computed ON THE DEVICE by the same index arithmetic the kernels use:
 * host_out[s] = site index of x(s) + dir*mu^ .  host_out: V int32, host memory.  Synchronises. */
int lqx_neighbor_table(lqx_ctx* ctx, lqx_dir dir, int mu, int32_t* host_out);

/* ---------------------------------------------------------------------------------------------
 * Device field store (pushToDevice / popFromDevice / freeDeviceMem,
 * PAPER.md:195-202 sec.6)
 * ------------------------------------------------------------------------------------------- */
int lqx_field_alloc(lqx_ctx* ctx, lqx_kind kind, lqx_prec prec, lqx_field** out);
/* Borrow caller-owned device memory (e.g. a torch tensor) of at least lqx_field_bytes() bytes,
 * 256-byte aligned; it is interpreted in the internal layout and never freed by the library. */
int lqx_field_attach(lqx_ctx* ctx, lqx_kind kind, lqx_prec prec, void* dev_ptr, size_t bytes,
                     lqx_field** out);
int lqx_field_free(lqx_field* f);
void* lqx_field_data(const lqx_field* f); /* device pointer of plane 0 (NULL on bad handle)     */
int lqx_field_kind(const lqx_field* f);
int lqx_field_prec(const lqx_field* f);
/* host QDP order -> device blocked SoA.  host: V*2*kind reals of the field precision.  Bit-exact. */
int lqx_field_push(lqx_field* f, const void* host_qdp_order);
/* device blocked SoA -> host QDP order.  Synchronises.  Bit-exact.  Does not free (reading A4). */
int lqx_field_pop(const lqx_field* f, void* host_qdp_order);
/* Same converters between two DEVICE buffers (dev_qdp_order: V*2*kind reals, AoS, 16-byte aligned -- LQX_EINVAL
 * otherwise: the converter moves 128-bit words). Asynchronous. */
int lqx_field_import_dev(lqx_field* f, const void* dev_qdp_order);
int lqx_field_export_dev(const lqx_field* f, void* dev_qdp_order);

/* ---------------------------------------------------------------------------------------------
 * Expression catalogue.  Destination first.
 * ------------------------------------------------------------------------------------------- */
/* E0 of Listing 1: r = a.  Any kind. */
int lqx_copy(lqx_field* r, const lqx_field* a);
/* r = shift(a, dir, mu): r(x) = a(x + dir*mu^).  Any kind.  Bit-exact.  r must not alias a. */
int lqx_shift(lqx_field* r, const lqx_field* a, lqx_dir dir, int mu);
/* form (i)  R = A*B + C*adj(D), colour matrices (BASELINE.json configs[4]) */
int lqx_mm_plus_madj(lqx_field* r, const lqx_field* a, const lqx_field* b, const lqx_field* c,
                     const lqx_field* d);
/* form (ii) c = trace(A*B): colour matrices -> LatticeComplex */
int lqx_trace_mm(lqx_field* c, const lqx_field* a, const lqx_field* b);
/* form (iii) R = alpha*A - shift(B, dir, mu), colour matrices (configs[4]: alpha=2.5, BACKWARD, 2) */
int lqx_ax_minus_shift(lqx_field* r, double alpha, const lqx_field* a, const lqx_field* b,
                       lqx_dir dir, int mu);
/* form (iv) w = M*v: colour matrix times colour vector, or times fermion (per spin component) */
int lqx_mat_vec(lqx_field* w, const lqx_field* m, const lqx_field* v);
/* The paper's hot expression E1/E2 (Listing 1 lines 25/27; Eq. 2 :215) fused
 * over mu (BASELINE.json configs[1]):
 *   chi(x) = sum_mu U_mu(x) psi(x+mu^) + adj(U_mu(x-mu^)) psi(x-mu^).
 * psi, chi: fermion or colour vector; u[4]: colour matrices.  chi must not alias psi. */
int lqx_hop(lqx_field* chi, const lqx_field* const u[4], const lqx_field* psi);
/* The same with norm2(chi) fused into the pass; *norm2_out (host double) after a sync. */
int lqx_hop_norm2(lqx_field* chi, const lqx_field* const u[4], const lqx_field* psi,
                  double* norm2_out);
/* E3 (reading A3): r = s0 + kappa*h.  Any kind. */
int lqx_axpy(lqx_field* r, const lqx_field* s0, double kappa, const lqx_field* h);
/* r = s*a (real scalar scaling) and E4 r = a / nrm as a true division (A22). */
int lqx_scale(lqx_field* r, double s, const lqx_field* a);
int lqx_divide(lqx_field* r, const lqx_field* a, double nrm);

/* The paper's complete routine (Listing 1 jacobiSmear; Eq. 1-2 :208-218; readings
 * A2, A3):  s_0 = chi;  iter x { psi = chi;  h = sum_{mu != no_smear_dir} u[mu]*shift(psi,FORWARD,mu)
 * + shift(adj(u[mu])*psi,BACKWARD,mu);  chi = s_0 + kappa*h };  chi /= norm  -- the power series
 * sum_{n<=iter} kappa^n H^n chi / norm.  One fused kernel per iteration (E0-E3; E4 in the last).
 * chi (fermion or colour vector) is input and output; tmp[2] are caller-provided scratch fields of
 * chi's kind and precision, all distinct.  no_smear_dir outside 0..3 smears in all four directions.
 * Asynchronous.  LQX_EINVAL for iter < 0 or norm == 0. */
int lqx_jacobi_smear(lqx_field* chi, const lqx_field* const u[4], double kappa, int iter,
                     int no_smear_dir, double norm, lqx_field* const tmp[2]);

/* ---------------------------------------------------------------------------------------------
 * Run-time expression fusion -- the paper's own mechanism:
 * the expression arrives as a flattened POD tree in postfix order ("a linear
 * container"), the library generates ONE fused kernel for it, compiles it with NVRTC for sm_100a
 * on first use and keeps it loaded until lqx_finalize, so that every expression is compiled once
 * per process.  Scalars are kernel arguments: expressions that differ only in their
 * scalars share a kernel.
 *   LEAF  a = index into leaves[]           pushes that field
 *   ADJ                                     adj(top)                    colour matrix
 *   MUL                                     left * right                matrix*matrix, matrix*vector, matrix*fermion
 *   ADD / SUB                               left + right, left - right  same kind
 *   SCALE s = real scalar                   s * top                     any kind
 *   SHIFT a = LQX_FORWARD/LQX_BACKWARD, b = mu   shift(top, a, b): the operand evaluated at x + a*mu^
 *   TRACE                                   trace(top): colour matrix -> LatticeComplex (configs[4] form ii)
 * (shifts nest: shift(adj(u)*psi, BACKWARD, mu) is the Listing's form).
 * dst = expr (accumulate == 0) or dst += expr (accumulate != 0, E2 of the Listing).  dst may alias
 * a leaf that is not read through a shift; otherwise LQX_EALIAS.  At most 16 leaves and 16 scalars.
 * Errors: LQX_EINVAL malformed sequence, LQX_ETYPE kind mismatch, LQX_ECUDA compilation / load
 * failure (lqx_last_error holds the NVRTC log).  Asynchronous on the context's stream.
 * ------------------------------------------------------------------------------------------- */
typedef enum { LQX_X_LEAF = 0, LQX_X_ADJ = 1, LQX_X_MUL = 2, LQX_X_ADD = 3, LQX_X_SUB = 4, LQX_X_SCALE = 5,
               LQX_X_SHIFT = 6, LQX_X_TRACE = 7 } lqx_xop;
typedef enum { LQX_R_NORM2 = 1, LQX_R_SUM = 2 } lqx_xreduce;
typedef struct {
    int32_t op; /* lqx_xop */
    int32_t a, b;
    double s;
} lqx_xnode;
int lqx_expr_eval(lqx_field* dst, int accumulate, const lqx_xnode* nodes, int nnodes,
                  const lqx_field* const* leaves, int nleaves);
/* Global reduction of an expression without materialising it (configs[4]: "each with norm2/sum/trace
 * reduction"): what = LQX_R_NORM2 -> out[0] = sum_x sum_components |expr|^2; LQX_R_SUM -> out[0..2*kind) =
 * sum_x expr(x) as one site object in QDP order (sum of trace(expr) is the global trace, reading A12).
 * fp64 accumulation, fixed summation tree; *out_count (may be NULL) = doubles written.  Synchronises.
 * The context and precision are those of leaves[0]. */
int lqx_expr_reduce(int what, const lqx_xnode* nodes, int nnodes, const lqx_field* const* leaves,
                    int nleaves, double* out, int* out_count);
/* The CUDA source the library generates for an expression (for inspection and tests; needs no GPU:
 * ctx may be NULL): written NUL-terminated into buf; returns its full length or a negative status.
 * accumulate: 0 '=', 1 '+=', 2 / 3 the norm2 / sum kernel lqx_expr_reduce uses (dst_kind = the expression's). */
int lqx_expr_source(lqx_ctx* ctx, lqx_kind dst_kind, lqx_prec prec, int accumulate, const lqx_xnode* nodes,
                    int nnodes, const lqx_kind* leaf_kinds, int nleaves, char* buf, size_t buflen);
/* Number of distinct expression kernels this context has compiled so far. */
int lqx_expr_cache_size(const lqx_ctx* ctx);

/* ---------------------------------------------------------------------------------------------
 * Global reductions.  fp64 accumulation for both precisions, fixed summation
 * tree (deterministic run to run).  Results to host double; these calls synchronise.
 * ------------------------------------------------------------------------------------------- */
int lqx_sum(const lqx_field* f, double* out);   /* out: 2*kind doubles, one site object, QDP order */
int lqx_norm2(const lqx_field* f, double* out); /* sum_x sum_components |c|^2                      */
int lqx_trace(const lqx_field* m, double out[2]); /* sum_x tr M(x) (reading A12)                   */
/* norm2 for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): the same sum as lqx_norm2 (Listing 1, norm2() of the Jacobi routine), with the
 * reduction scratch -- one fp64 partial per CTA of 2048 sites and the last-block ticket -- in a file-scope __device__
 * array of LQX_NOALLOC_SCRATCH_BYTES instead of the context's cudaMalloc'ed, grow-on-demand buffer.  The call makes
 * no cudaMalloc / cudaFree and calls no allocating routine; every GPU that loads the library holds the array until
 * the process exits.
 *   f        field of any kind and precision (device memory, blocked layout, owned by the caller)
 *   out_dev  one double in DEVICE memory (or pinned mapped host memory), 8-byte aligned, owned by the caller;
 *            written by the kernel.  The call is asynchronous on the context's stream and does not synchronise.
 * Errors: LQX_EINVAL for null / misaligned pointers and for a lattice of more than LQX_NOALLOC_MAX_SITES sites (the
 * array then has too few partial slots; nothing is launched; lqx_last_error says so); LQX_ECUDA if the array's device
 * address cannot be obtained (cudaGetSymbolAddress, asked once per device on the first call there) or a launch fails.
 * All calls share the one array per device and it keeps the last call's contents: the ticket is cleared on the stream
 * before every launch, the partials are overwritten before they are read; calls that OVERLAP on the GPU (two streams
 * or two contexts on one device) race on it -- serialise them.  The summation tree depends on the volume only (same
 * result on every GPU); it is not lqx_norm2's tree, so the two agree to rounding, not bit for bit. */
#define LQX_NOALLOC_MAX_SITES (1 << 24)
#define LQX_NOALLOC_SCRATCH_BYTES (8192 * 8 + 256)
int lqx_norm2_noalloc(const lqx_field* f, double* out_dev);
/* P = sum_x sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu^) adj(U_mu(x+nu^)) adj(U_nu(x))];
 * *plaq_sum = P, *plaq_avg = P/(18 V) (reading A11).  Either pointer may be NULL. */
int lqx_plaquette(const lqx_field* const u[4], double* plaq_sum, double* plaq_avg);

/* ---------------------------------------------------------------------------------------------
 * Staple sum and smearing (BASELINE.json configs[0],[2],[3])
 *   S_mu(x)  = sum_{nu != mu} [ U_nu(x) U_mu(x+nu^) adj(U_nu(x+mu^))
 *                             + adj(U_nu(x-nu^)) U_mu(x-nu^) U_nu(x-nu^+mu^) ]
 *   U'_mu(x) = (1-alpha) U_mu(x) + (alpha/6) S_mu(x)          (no projection, reading A9)
 * ------------------------------------------------------------------------------------------- */
/* out = S_mu for one direction (test/diagnostic entry). */
int lqx_staple_sum(lqx_field* out, const lqx_field* const u[4], int mu);
/* One smearing step, all four directions, out of place.  If plaq_in_or_null != NULL the plaquette
 * sum of the INPUT field is accumulated in the same pass and stored there (host double; the call
 * then synchronises). */
int lqx_smear_step(lqx_field* const uout[4], const lqx_field* const uin[4], double alpha,
                   double* plaq_in_or_null);
/* nsteps iterated steps (configs[3]): result ends in u; tmp is ping-pong scratch.
 * plaq_avg_after_each (host, nsteps doubles, may be NULL) = plaquette average of the field after
 * every step.  One synchronisation at the end. */
int lqx_smear_iterate(lqx_field* const u[4], lqx_field* const tmp[4], double alpha, int nsteps,
                      double* plaq_avg_after_each);
/* End-to-end form with HOST buffers (bench `e2e`): host_u_in[4] / host_u_out[4] are host colour
 * matrix fields in QDP order of precision `prec` (host_u_out[mu] may be host_u_in[mu]); pushes,
 * iterates, pops; the host buffers are not touched after the call returns.  Work fields stay cached
 * in the context until lqx_finalize.  A single step (nsteps == 1) is streamed: the lattice is cut
 * into slabs of time slices whose upload, update and download overlap on three streams (page-locked
 * host buffers are needed for the copies to overlap; pageable ones work, serially); the result is
 * bit-identical to the serial path.  Option "host_slabs": -1 automatic, 0 serial, n at most n slabs. */
int lqx_smear_iterate_host(lqx_ctx* ctx, lqx_prec prec, const void* const host_u_in[4],
                           void* const host_u_out[4], double alpha, int nsteps,
                           double* plaq_avg_after_each);

/* ---------------------------------------------------------------------------------------------
 * NEXT-4 (sec.9 "parallelisation to multiple GPUs per host"): building blocks of a
 * decomposition along t.  A rank's context is a t-slab with one halo slice on either side (local extent
 * L3/ranks + 2); paper_1105_2279_b200/tsplit.py drives the halo exchange (torch.distributed or peer copies) and
 * overlaps it with the interior launch.  Nothing here communicates.
 *   lqx_smear_step_range : the smear step of the time slices [t0, t1) only (asynchronous).  The caller guarantees
 *       that the input slices t0-1 .. t1 hold what the step should read.  Bit-identical to lqx_smear_step on those sites.
 *   lqx_plaquette_range  : sum over the sites of [t0, t1) of the six plaquettes (synchronises, host double).
 *   lqx_field_slice      : byte offset and size of time slice t inside a field's device storage.  A slice is one
 *       contiguous range (sites are lexicographic with t slowest and blocks of 32 sites are contiguous) iff
 *       L0*L1*L2 is a multiple of 32; otherwise LQX_EGEOM.
 * ------------------------------------------------------------------------------------------- */
int lqx_smear_step_range(lqx_field* const uout[4], const lqx_field* const uin[4], double alpha, int t0, int t1);
int lqx_plaquette_range(const lqx_field* const u[4], int t0, int t1, double* plaq_sum);
int lqx_field_slice(const lqx_field* f, int t, int64_t* offset_bytes, int64_t* nbytes);

/* ---------------------------------------------------------------------------------------------
 * Harness support: device micro-benchmarks that give the roofline denominators.
 * ------------------------------------------------------------------------------------------- */
/* kind: 0 = fp32 FMA, 1 = packed fp32x2 FMA, 2 = fp64 FMA (one dependent chain per accumulator, constant multiplicands);
 * 3 = fp32, 4 = fp64: a stream of 3x3 complex products on register operands -- the instruction mix of the lattice
 * kernels (fp32: FFMA2 with broadcast and swapped operands), three distinct register operands per instruction.
 * Returns achieved FMA lane-ops/s (one fused multiply-add on one real = 1 lane-op = 2 flop) in *lane_ops_per_s. */
int lqx_bench_fma_peak(lqx_ctx* ctx, int kind, double* lane_ops_per_s);
/* Plain device copy of `bytes` bytes (read + write counted): achieved bytes/s. */
int lqx_bench_copy_peak(lqx_ctx* ctx, size_t bytes, double* bytes_per_s);
/* Per-kernel-class device timing for the harness.  lqx_set_option(ctx, "time_kernels", 1) makes
 * the library bracket every launch of the classes below with CUDA events on the context's stream;
 * lqx_kernel_time synchronises the stream, returns the summed duration and launch count of one
 * class since the last read, and clears it. */
enum { LQX_K_SMEAR = 0, LQX_K_PLAQUETTE = 1, LQX_K_HOP = 2, LQX_K_CATALOGUE = 3, LQX_K_REDUCE = 4,
       LQX_NUM_KERNEL_CLASSES = 5 };
int lqx_kernel_time(lqx_ctx* ctx, int kernel_class, double* total_ms, int* count);
/* Number of kernels this context has launched since init (for bench.py's gpu_launches). */
int64_t lqx_launch_count(const lqx_ctx* ctx);
/* What the last lqx_smear_step / lqx_smear_iterate launch of this context ran: the variant in effect after options,
 * tuned choice and fall-backs, the FMA lane-operations it executes per site (48 products x 108 + 144 for the literal
 * evaluation), and the kernel's name (truncated to name_len - 1 characters).  Any out pointer may be NULL. */
int lqx_smear_info(const lqx_ctx* ctx, int* variant, int* lane_ops_per_site, char* kernel_name, int name_len);

/* ---------------------------------------------------------------------------------------------
 * Auto-tuning of the launch geometry -- the paper's to-do (sec.5.4 "auto-tuning ... geometry
 * parameters ... stored for later inclusion"; sec.9), its sweeps PAPER.md:242-262 (Figs. 1-2).
 * lqx_autotune times, on the context's lattice and stream (it synchronises), every geometry the library can select for
 * one kernel class and precision and keeps the fastest in the context; later calls use it unless an explicit
 * lqx_set_option overrides it.  kernel_class: LQX_K_SMEAR (param = smear_variant, tile), LQX_K_PLAQUETTE
 * (param = plaq_variant), LQX_K_HOP (param[0] > 0: CTA size of lqx_hop; param[0] < 0: N_threads = -param[0] and
 * N_site = param[1] of one lqx_jacobi_smear iteration).  rows (caller-owned, may be NULL) receives up to max_rows
 * table rows: ms = median of `reps` launches, chosen = 1 for the kept geometry; *nrows = rows measured.
 * It allocates and frees its own scratch fields (eight link fields, or four links and four fermions).
 * lqx_tuned reads back what is kept (0 / -1 = nothing): smear {variant, tile}, plaquette {variant},
 * hop {hop_block, jacobi_block, jacobi_sites}. */
typedef struct {
    int kernel_class;
    int prec;
    int param[2];
    double ms;
    int chosen;
} lqx_tune_row;
int lqx_autotune(lqx_ctx* ctx, int kernel_class, lqx_prec prec, int reps, lqx_tune_row* rows, int max_rows, int* nrows);
int lqx_tuned(const lqx_ctx* ctx, int kernel_class, lqx_prec prec, int out[4]);
/* Options: "smear_variant" 0 = default (fp32 on lattices whose rows are 40 or 48 sites: 10; otherwise 9; 3 where the row tiles do
 * not fit the lattice), 3 = rolled literal kernel, 1 = first-cut literal kernel,
 * 2 = shared-corner kernel (36 products, lower staples exchanged through shared memory), 4 = four
 * threads per site, 6 = operands staged in shared memory with cp.async (fp32), 7 = the CTA tile's own links in
 * shared memory and the halo through L1, 8 = plane-ordered 42-product evaluation on whole-x-row tiles, persistent
 * double-buffered CTAs (fp32; with "tile" 6: one tile per CTA, two CTAs per SM, 7: the same with the halo operands
 * prefetched into L1), 9 = the literal evaluation of 3 on whole-x-row tiles whose own links sit in shared
 * memory (both precisions; same summation order as 3, bit-identical), 10 = the per-link evaluation of 9 with the common
 * factor of the two upper staples of a plane kept in tensor memory between the two links (fp32, rows of a multiple of 8 up
 * to 48 sites: 42 products and 64 operand fetches per site; falls back to 9); variants fall back to 3 where their tiles do
 * not fit the lattice.
 * "tile" -1 = automatic, 0 = linear 128-site blocks, 1..6 = CTA tile shape (8x4x4x2, 8x4x2x2,
 * 4x4x4x2, 16x4x2x2, 16x2x2x2, 32x2x2x2) of the nearest-neighbour kernels, used if it divides the
 * lattice.  "jacobi_block" (32, 64, 128, 256) and "jacobi_sites" (1, 2, 4): the paper's launch
 * geometry parameters N_threads and N_site for lqx_jacobi_smear; 0 = tuned default.
 * "hop_block" (32, 64, 128, 256): CTA size of lqx_hop on
 * linear blocks; 0 = tuned or default (128).  "host_slabs": see lqx_smear_iterate_host.
 * "plaq_variant" 0 = automatic (fp32: the site's four links held in registers, 16 matrix loads per site;
 * fp64: rolled plane loops, 21 loads at half the registers -- each the faster one measured), 1 = rolled, 2 = held.
 * "bulk_fill" 1 = the row-tile kernel (9) fills its tile by TMA bulk copies (cp.async.bulk + mbarrier) where the tile's rows
 * are whole 32-site blocks, 0 (default) = by per-thread cp.async; bit-identical results, the bulk form measured 2 % slower.
 * "time_kernels" 0/1 (see above).  All variants agree within rounding; DESIGN.md sec.6. */
int lqx_set_option(lqx_ctx* ctx, const char* key, int value);

const char* lqx_strerror(int code);
const char* lqx_last_error(const lqx_ctx* ctx);
const char* lqx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LQX_H */

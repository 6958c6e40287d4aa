/* coarse_op.h — C ABI of libcoarseop: the coarse-grid Dirac operator apply on one B200.
 *
 * The operation (BASELINE.json north_star; the paper names it "the coarse stencil operator",
 * PAPER.md:L99 §3.1, stored as "nine 48^2 matrices per super-site: eight for the hopping terms
 * and one for the [local] term", §3.1):
 *
 *   dagger = 0:  out(x) = X(x).in(x) + sum_{mu=0..3} [ Y_{+mu}(x).in(x+mu^) + Y_{-mu}(x).in(x-mu^) ]
 *   dagger = 1:  out(x) = X(x)^H.in(x) + sum_mu [ Y_{+mu}(x-mu^)^H.in(x-mu^) + Y_{-mu}(x+mu^)^H.in(x+mu^) ]
 *                (the true adjoint for arbitrary links; needed by the CGNE setup solver,
 *                 PAPER.md:L123 Table 1)
 *
 * on a periodic 4-D lattice, X and Y dense Nc x Nc complex matrices, Nc = 2 N_vec after the
 * chiral doubling of PAPER.md:L41/L87, applied to nrhs vectors at once (block variant;
 * multi-RHS is the paper's future work).  Links are stored either as complex64
 * or in the paper's "16-bit fixed point format": int16 (re,im) pairs with one
 * fp32 scale per matrix, scale = max|component|/32767 (BASELINE.json config 4).
 *
 * Everything runs in hand-written sm_100a kernels.  There is no CPU fallback: every entry point
 * that needs the GPU returns COARSE_ECUDA when no usable device is present.
 *
 * LAYOUTS (all device pointers unless a name ends in _host; all 16-byte aligned)
 *   site index      s(x) = x0 + L0*(x1 + L1*(x2 + L2*x3)), dims = {L0,L1,L2,L3}; neighbours wrap
 *                   periodically (extent 2: both hops come from the same site and both are added;
 *                   extent 1: both come from the site itself).
 *   links           links[s][m][i][j], m = 0:X, 1+mu:Y_{+mu}, 5+mu:Y_{-mu}; row-major,
 *                   out_i = sum_j M_ij in_j.
 *                   COARSE_LINK_C64: float[2] = (re,im) per entry.
 *                   COARSE_LINK_I16: int16_t[2] = (re,im) per entry, entry = scales[s][m]*(re + i im).
 *   scales          float scales[s][m] (COARSE_LINK_I16 only).
 *   vectors         v[s][a][r], float[2] = (re,im), a in [0,Nc) colour-spin (a = chi*N_vec + k),
 *                   r in [0,nrhs) innermost.
 *
 * OWNERSHIP  Link, scale, in and out buffers are the caller's.  coarse_op_set_links borrows the link and
 *   scale pointers, which must stay valid and unchanged until destroy or the next set_links.  The handle
 *   owns its metadata and two kinds of device scratch: two vector-sized staging buffers plus two copy
 *   streams (only if coarse_op_apply_host is used), and, on lattices with fewer sites than SMs, a few-MB
 *   workspace for the split dagger apply.  Because of that scratch a handle may have work in flight on
 *   ONE stream at a time (two concurrent split applies would share the workspace and its counters); use one handle per stream for concurrent solves on the same links (handles
 *   are cheap and may share link buffers).  A handle belongs to the device that was current in
 *   coarse_op_create; calls made with another device current return COARSE_EINVAL.
 *
 * ERRORS  int-returning calls return COARSE_OK (0) or a negative code; coarse_op_create returns
 *   NULL.  coarse_op_last_error() gives a thread-local message.  No exception crosses the ABI.
 *   Asynchronous device faults surface at the caller's next synchronisation.
 *
 * STREAMS  `stream` is a cudaStream_t passed as void* (0 = legacy default stream).  coarse_op_apply
 *   enqueues and returns; it never synchronises and never allocates.  Results are bit-identical
 *   from run to run (no floating-point atomics).
 */
#ifndef COARSE_OP_H
#define COARSE_OP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct coarse_op coarse_op_t; /* opaque */

enum { COARSE_LINK_C64 = 0, COARSE_LINK_I16 = 1 };

enum {
    COARSE_OK = 0,
    COARSE_EINVAL = -1,       /* bad argument (NULL, misaligned, overlapping in/out, nrhs < 1, ...) */
    COARSE_EUNSUPPORTED = -2, /* valid but not compiled in (see coarse_op_set_option)              */
    COARSE_ENOTREADY = -3,    /* apply before set_links                                            */
    COARSE_ECUDA = -4,        /* CUDA runtime error, or no sm_100 device                           */
    COARSE_ENOMEM = -5
};

/* Kernel families, each compiled for Nc in {32,48,64,96,128,192}; every family computes the same operation and the
 * tests run parity on each.  AUTO: 1 RHS -> STREAM; 2-4 RHS -> STREAM (its multi-RHS kernel), except int16 links
 * (Nc = 48: only at 4 RHS; 2-3 RHS only on lattices with at least two tensor work items per SM) and complex64 links with exactly 4 RHS in dagger = 0 (Nc >= 48) -> TENSOR; 5 RHS and more -> TENSOR; BLOCK only on request (or when no tensor map can be made for the links);
 * Nc outside the compiled set -> SIMPLE. */
enum {
    COARSE_PATH_AUTO = 0,
    COARSE_PATH_SIMPLE = 1,  /* one thread per output element, any even Nc, any nrhs                           */
    COARSE_PATH_STREAM = 2,  /* persistent TMA-bulk -> smem ring -> CUDA-core consumers, nrhs <= 4              */
    COARSE_PATH_TENSOR = 3,  /* block apply on the tcgen05 tensor cores, any nrhs (column tiles of 8 / 16, one launch
                                per 16): complex64 links as 3xTF32, int16 links on the integer tensor cores (int8
                                planes, exact), see COARSE_OPT_TENSOR_I8                                         */
    COARSE_PATH_BLOCK = 4    /* block apply on the CUDA cores (same TMA ring), nrhs <= 16: the comparison arm    */
};

enum {
    COARSE_OPT_PATH = 0,     /* one of COARSE_PATH_*                                              */
    COARSE_OPT_GRID = 1,     /* persistent grid size for STREAM/TENSOR; 0 = one CTA per SM        */
    COARSE_OPT_STAGES = 2,   /* cap on the STREAM shared-memory ring depth; 0 = library default   */
    COARSE_OPT_FINE = 3,     /* STREAM dagger=0 small-lattice row-block split: 0 auto, 1 never, 2 always */
    COARSE_OPT_KEEP_LINKS = 4, /* L2 policy of the link stream: 0 auto (keep if links <= L2/2), 1 evict_first, 2 keep */
    COARSE_OPT_PDL = 5,      /* programmatic dependent launch of the 1-RHS STREAM kernels: in a chain of applies on one
                                stream the next kernel's CTAs start on SMs the previous one has left and prefetch
                                their link stages before waiting for its output (the latency-limited small-lattice
                                regime of PAPER.md:L99).  0 (default) auto: when the links fit L2, for every apply but
                                the first after coarse_op_set_links (work that produced the links may still be in
                                flight in front of that one); 1 always: the LINK and scale arrays must then not be
                                written by work still in flight on the stream (they are read before the kernel orders
                                itself against its predecessor); 2 never.  Results are bit-identical either way. */
    COARSE_OPT_SPLIT_DAGGER = 6, /* dagger = 1, 1-4 RHS on STREAM, lattices so small that every site can have a cluster of
                                4 (2) CTAs to itself at once (sites x cluster size <= SMs): split each site's
                                contraction over its row chunks.  The kernel is launched as thread-block clusters
                                of 4 (2) CTAs, one site per cluster at a time; the partial vectors meet in the
                                shared memory of the cluster's first CTA behind one cluster barrier (one launch,
                                deterministic): 0 auto, 1 never, 2 always, 3 always with the global-memory scheme
                                instead (partial vectors in a workspace coarse_op_set_links allocates on such
                                lattices, the CTA that counts a site's last chunk in adds them in chunk order; also
                                the fallback where clusters cannot be launched) */
    COARSE_OPT_WARP_ITEMS = 7, /* 1-RHS plain apply: the STREAM variant in which small teams of consumer warps own
                                whole work items and every stage of theirs (csrc/stream2_kernel.cuh) instead of all
                                eight warps sharing every stage: 0 auto (int16 links with Nc >= 48, and Nc = 32, on lattices with at
                                least 4 items per team of the chip), 1 never, 2 always, 12 / 14 always with 2 / 4 warps per
                                team (2 = 14).  With it COARSE_OPT_STAGES is the ring's slot count. */
    COARSE_OPT_TENSOR_I8 = 8  /* TENSOR path on int16 links: 0 auto / 2: the integer tensor-core kernel (csrc/tensor_i8_kernel.cuh:
                                link entries as two int8 planes, exact, vectors in 23-bit fixed point per site), 1: the
                                3xTF32 kernel.  Site-range launches of coarse_op_apply_host always use the latter;
                                coarse_op_apply_hvec and coarse_op_apply_static (integer kernel only) ignore the option. */
};

/* Create an operator descriptor for a periodic lattice dims[0..3] (each >= 1), Nc even and
 * >= 2, link_precision one of COARSE_LINK_*.  Returns NULL on error (see coarse_op_last_error). */
coarse_op_t* coarse_op_create(const int dims[4], int Nc, int link_precision);

/* V*9*Nc*Nc*8 bytes (C64) or V*9*Nc*Nc*4 bytes (I16); 0 for NULL. */
size_t coarse_op_link_bytes(const coarse_op_t* op);
/* V*9*4 bytes for I16, 0 for C64. */
size_t coarse_op_scale_bytes(const coarse_op_t* op);
/* V*Nc*nrhs*8 bytes. */
size_t coarse_op_vector_bytes(const coarse_op_t* op, int nrhs);

/* Borrow the device link array (layout above) and, for I16, the device scale array.
 * scales_dev must be NULL for C64 and non-NULL for I16. */
int coarse_op_set_links(coarse_op_t* op, const void* links_dev, const float* scales_dev);

/* Select a kernel family / tuning knob (COARSE_OPT_*).  COARSE_EUNSUPPORTED if the requested
 * family cannot run this operator's (Nc, precision); the nrhs-dependent check happens in apply. */
int coarse_op_set_option(coarse_op_t* op, int option, int value);

/* out = A.in (dagger = 0) or A^H.in (dagger = 1) for nrhs >= 1 right-hand sides.
 * in_dev and out_dev are device vectors [V][Nc][nrhs] complex64 and must not overlap. */
int coarse_op_apply(coarse_op_t* op, const void* in_dev, void* out_dev, int nrhs, int dagger,
                    void* stream);

/* Parts apply: the building block of the even/odd ("Schur-preconditioned", PAPER.md:L127/L135
 * Table 1) and block-preconditioned coarse operators.  With the site parity
 * pi(x) = (x0+x1+x2+x3) mod 2, for every site x of `parity` (COARSE_PARITY_*):
 *
 *     out(x) = alpha * Loc(x) + beta * Hop(x)
 *     Loc(x) = X(x).u(x) (COARSE_LOCAL_X) | u(x) (COARSE_LOCAL_IDENTITY) | 0 (COARSE_LOCAL_NONE)
 *     Hop(x) = sum_mu [ Y_{+mu}(x).w(x+mu^) + Y_{-mu}(x).w(x-mu^) ]
 *
 * and for dagger = 1 the same split of the adjoint (X(x)^H.u(x) and the adjoint hop of
 * coarse_op_apply).  Sites of the other parity are NOT written.  u_dev may be NULL for
 * COARSE_LOCAL_NONE.  Aliasing: w_dev must never overlap out_dev (the stencil reads neighbours).  With
 * COARSE_LOCAL_IDENTITY u_dev may be the SAME pointer as out_dev (in place: every output element reads
 * only its own u element first); a partial overlap, or any overlap with COARSE_LOCAL_X (X.u reads all of
 * u(x) while other work items write out(x)), returns COARSE_EINVAL.
 * COARSE_PARITY_EVEN/ODD need every extent even (COARSE_EINVAL otherwise).
 * Examples (hat = an operator whose links are Yhat_m = X^{-1} Y_m):
 *     t_o   = Dhat_oe v_e           : apply_parts(hat, NULL, v, t, .., COARSE_PARITY_ODD, COARSE_LOCAL_NONE, 0, 1)
 *     out_e = v_e - Dhat_eo t_o     : apply_parts(hat, v, t, out, .., COARSE_PARITY_EVEN, COARSE_LOCAL_IDENTITY, 1, -1)
 *     out_e = X_e v_e - D_eo t_o    : apply_parts(op, v, t, out, .., COARSE_PARITY_EVEN, COARSE_LOCAL_X, 1, -1)
 * nrhs = 1 runs on the STREAM kernels (8 or 9 link matrices streamed per site of the parity), several right-hand
 * sides on the TENSOR kernels (SIMPLE outside the compiled Nc). */
enum { COARSE_PARITY_EVEN = 0, COARSE_PARITY_ODD = 1, COARSE_PARITY_ALL = 2 };
enum { COARSE_LOCAL_NONE = 0, COARSE_LOCAL_X = 1, COARSE_LOCAL_IDENTITY = 2 };
int coarse_op_apply_parts(coarse_op_t* op, const void* u_dev, const void* w_dev, void* out_dev, int nrhs,
                          int dagger, int parity, int local, float alpha, float beta, void* stream);

/* The plain apply on HALF-PRECISION input vectors ("half precision" = 16-bit fixed
 * point with a per-site fp32 norm): in(x)_jr = in_norms[x][r] * (q_re + i q_im), in_q_dev =
 * int16_t[V][Nc][nrhs][2], in_norms_dev = float[V][nrhs].  The output is complex64 (coarse_op_apply_hout adds the
 * half-precision result).  Nc % 4 == 0.
 * nrhs = 1 runs on the STREAM kernels (the norm is folded into the vector operand like the int16
 * link scale; int16 links on large lattices: the warp-team kernel, as for complex64 vectors).  Several right-hand sides on int16 links - the paper's storage for both operands (L97, L99) - run on
 * the integer tensor cores (COARSE_PATH_TENSOR; one launch per 16 columns): the two bytes of an int16 link entry and
 * of an int16 vector component are the int8 operands, int32 accumulation is exact, and the only rounding is the fp32
 * recombination by link scale x vector norm in the epilogue.  Complex64 links with several right-hand sides: SIMPLE. */
int coarse_op_apply_hvec(coarse_op_t* op, const void* in_q_dev, const float* in_norms_dev, void* out_dev, int nrhs,
                         int dagger, void* stream);

/* The apply with a HALF-PRECISION RESULT: out_c64_dev receives the complex64 result as coarse_op_apply
 * would write it, and (out_q_dev, out_norms_dev) the same vector as 16-bit fixed point with a per-(site, rhs) fp32 norm,
 * exactly what coarse_op_quantize_vec_i16 makes of out_c64_dev (norm = max|component| / 32767, q = clamp(rint(component /
 * norm))).  in_norms_dev = NULL: in_dev is a complex64 vector; else the half-precision input of coarse_op_apply_hvec.
 * For 1 RHS on the STREAM kernels it is ONE launch: a CTA owns whole sites (all row blocks of a site in a row), keeps
 * the site's rows in shared memory and ends each site with a CTA-local epilogue (norm, 16-bit vector); int16 links on
 * large lattices: the warp-team kernel, where a team of warps holds a whole site (dagger 1; dagger 0 for Nc <= 64).  Other
 * nrhs / shapes: the apply followed by the vector quantiser.  The three vector buffers must not overlap. */
int coarse_op_apply_hout(coarse_op_t* op, const void* in_dev, const float* in_norms_dev, void* out_c64_dev, void* out_q_dev,
                         float* out_norms_dev, int nrhs, int dagger, void* stream);

/* The plain apply for callers that cannot call cudaMalloc (code under CUDA stream capture, tight serving loops,
 * harnesses that forbid allocation): out = D in (dagger 0) or D^dagger in (1) for INT16 links and any
 * nrhs >= 1, on the integer tensor-core kernel of COARSE_PATH_TENSOR - the same kernels, launches and
 * results as coarse_op_apply with that path - but with the kernel's scratch memory (the power-of-two scales of the
 * fixed-point vector operand, one (g, 1/g) pair per site and column) in a file-scope __device__ array of the library
 * instead of the buffer coarse_op_set_links allocates.  This call reaches no cudaMalloc / cudaFree and no allocating
 * library routine; the handle itself must have been created and given its links beforehand.
 * Limit: at most COARSE_STATIC_MAX_SITES lattice sites (the array is COARSE_STATIC_MAX_SITES * 128 bytes = 1 MiB,
 * held by every GPU that loads the library until the process exits); more sites, complex64 links or an Nc outside
 * the compiled set return COARSE_EUNSUPPORTED with a message.  in_dev / out_dev: device, complex64 [V][Nc][nrhs],
 * 16-byte aligned, not overlapping; the handle's device must be current.
 * The array is shared by ALL calls and handles of the process on that GPU and keeps the last call's contents:
 * nothing in it needs to start at zero (each call rewrites every entry it reads), calls on one stream are ordered,
 * but calls that overlap on the GPU (other streams without an ordering event) RACE on it. */
#define COARSE_STATIC_MAX_SITES 8192
int coarse_op_apply_static(coarse_op_t* op, const void* in_dev, void* out_dev, int nrhs, int dagger, void* stream);

/* Vector quantiser: for each (site, rhs) norm = max|component|/32767 (fp32 division) and
 * q = clamp(rint(component/norm), -32767, 32767); an all-zero vector gets norm 0 and q = 0.
 * v_c64_dev: float[n_sites][Nc][nrhs][2]; q_dev: int16_t same shape; norms_dev: float[n_sites][nrhs]. */
int coarse_op_quantize_vec_i16(const void* v_c64_dev, int64_t n_sites, int Nc, int nrhs, void* q_dev,
                               float* norms_dev, void* stream);

/* Same operation on HOST vectors: copies in_host to a device staging buffer owned by the handle
 * (allocated on first use, grown when nrhs grows), applies, copies the result to out_host and
 * synchronises the stream before returning.  Pinned host memory gives full PCIe rate.
 * On the STREAM (1-4 RHS) and TENSOR kernels, with dims[3] >= 8 and vectors of at least 4 MiB, the call is
 * pipelined: the lattice is cut into 4 ranges of x3-slices (8 when the vectors are 32 MiB or more), each launched as
 * soon as the slices it reads are on the device, its result copied back while the next range computes (H2D, kernels
 * and D2H on three streams, two of them owned by the handle); the result is bit-identical to coarse_op_apply's (int16
 * links on the TENSOR path, i.e. several right-hand sides: to its result with COARSE_OPT_PATH = COARSE_PATH_TENSOR and
 * COARSE_OPT_TENSOR_I8 = 1, see there). */
int coarse_op_apply_host(coarse_op_t* op, const void* in_host, void* out_host, int nrhs, int dagger,
                         void* stream);

/* Kernel launches the most recent coarse_op_apply / coarse_op_apply_host on this handle enqueued. */
int coarse_op_last_launches(const coarse_op_t* op);
/* Family (COARSE_PATH_*) the most recent apply actually ran; 0 before the first apply. */
int coarse_op_last_path(const coarse_op_t* op);

/* The paper's reduced-precision link storage (BASELINE.json config 4), on the device:
 * for each of n_matrices Nc x Nc complex64 matrices, scale = max|component|/32767 (fp32 division)
 * and q = clamp(rint(component/scale), -32767, 32767) (fp32, round-half-to-even); an all-zero
 * matrix gets scale 0 and q = 0.  links_c64_dev: float[n][Nc][Nc][2]; q_dev: int16[n][Nc][Nc][2];
 * scales_dev: float[n]. */
int coarse_op_quantize_i16(const void* links_c64_dev, int64_t n_matrices, int Nc, void* q_dev,
                           float* scales_dev, void* stream);

/* Block-preconditioned links ("coarsening the block-preconditioned operator"; the operator
 * the paper's "Schur-preconditioned" levels iterate on, Table 1 L127/L135), built on the device from this
 * handle's links (either precision; int16 is dequantised exactly):
 *
 *     out[s][m] = X(s)^-1 . Y_m(s)  for m = 1..8,     out[s][0] = identity (COARSE_HAT_SLOT0_IDENTITY)
 *                                                              or X(s)^-1 (COARSE_HAT_SLOT0_XINV)
 *
 * out_links_c64_dev: complex64 [V][9][Nc][Nc] in the canonical link layout (V*9*Nc*Nc*8 bytes, caller
 * owned, must not overlap the handle's links); hand it to a second COARSE_LINK_C64 handle, or quantise it
 * with coarse_op_quantize_i16 for a COARSE_LINK_I16 one.  With X^-1 in slot 0, "apply X^-1" is
 * coarse_op_apply_parts(.., COARSE_LOCAL_X, alpha = 1, beta = 0) on that handle.
 * work_dev: coarse_op_hat_work_bytes(op) bytes of scratch (16-byte aligned).  info_dev: NULL or int[1], set
 * to the number of sites whose X has a zero pivot (those sites' outputs are non-finite).
 * All arithmetic is fp64 (Gauss-Jordan with partial pivoting + eight Nc^3 products per site), rounded to
 * complex64 once.  Any even Nc.  One launch; enqueues and returns. */
enum { COARSE_HAT_SLOT0_IDENTITY = 0, COARSE_HAT_SLOT0_XINV = 1 };
size_t coarse_op_hat_work_bytes(const coarse_op_t* op);
int coarse_op_build_hat_links(coarse_op_t* op, void* out_links_c64_dev, int slot0, void* work_dev, int* info_dev,
                              void* stream);

/* CA-GCR(s), the paper's smoother ("CA-GCR(8)", Table 1 L116/L122/L130; its coarsest-level solver is a
 * "Chebyshev-basis CA-GCR(16)", L134), on this operator, 1 RHS.  Each of `cycles` cycles minimises the residual
 * over x + K_s(A, r0), r0 = b - A x, the communication-avoiding way: the whole basis first - the Chebyshev basis
 * p_k = T_k((A - c)/d) r0 with t_k = A p_k kept beside it (s chained coarse_op_apply + s - 1 fused recurrence
 * steps) - then ONE fused pass of block inner products (fp64, the single reduction per cycle), the s x s normal
 * equations (fp64 Cholesky on the device) and one fused update x += sum_k alpha_k p_k, r = r0 - sum_k alpha_k t_k.
 * The basis spans the same Krylov space as the power basis A^k r0 - the minimiser is the same - but stays well
 * conditioned at every s <= 16.
 *   interval       coarse_op_cagcr / coarse_op_cagcr_schur estimate [c - d, c + d] on the device, in the first
 *                  cycle, from the moments of r0 (c = Re <r0, A r0>/<r0, r0>, d = twice the spread of A as r0 sees
 *                  it): no caller-supplied bounds, no host round trip.  coarse_op_cagcr_cheb takes real bounds
 *                  [lambda_min, lambda_max] that roughly enclose the spectrum (both 0: estimate as above).
 *   b_dev, x_dev   complex64 [V][Nc]; x_is_zero != 0: x is cleared first and b is used as r0 directly.
 *   work_dev       coarse_op_cagcr_work_bytes(op, s) bytes of caller-owned scratch (16-byte aligned): 2s + 2 vectors.
 *   info_dev       NULL, or double[3 * cycles]: per cycle ||r0||^2, the predicted ||r||^2 after the
 *                  cycle, and the number of basis vectors the factorisation kept (s unless the Gram
 *                  matrix lost positive definiteness).
 * 1 <= s <= 16.  Enqueues 2s + 2 kernels per cycle for A (s applies, s - 1 recurrence steps, Gram, solve, update)
 * plus 2 for the interval estimate (1 when the bounds are given); never synchronises.
 * coarse_op_cagcr_schur (and schur_parity = 0 | 1 of coarse_op_cagcr_cheb): the same smoother on the
 * left-preconditioned even/odd Schur operator Shat_p v = v - Dhat_pq Dhat_qp v of a handle whose links are
 * block-preconditioned (Yhat = X^-1 Y; Table 1 L127/L135: the levels the paper smooths with
 * CA-GCR(8) are Schur-preconditioned).  b and x are full-lattice vectors whose entries on the other parity must
 * be zero (x is kept so); every operator application is two parity-restricted launches (coarse_op_apply_parts).
 * schur_parity = -1: the operator is A. */
size_t coarse_op_cagcr_work_bytes(const coarse_op_t* op, int s);
size_t coarse_op_cagcr_cheb_work_bytes(const coarse_op_t* op, int s);   /* the same number */
int coarse_op_cagcr(coarse_op_t* op, const void* b_dev, void* x_dev, int s, int cycles, int x_is_zero,
                    void* work_dev, double* info_dev, void* stream);
int coarse_op_cagcr_schur(coarse_op_t* op_hat, const void* b_dev, void* x_dev, int s, int cycles, int x_is_zero,
                          int parity, void* work_dev, double* info_dev, void* stream);
int coarse_op_cagcr_cheb(coarse_op_t* op, const void* b_dev, void* x_dev, int s, int cycles, int x_is_zero,
                         float lambda_min, float lambda_max, int schur_parity, void* work_dev, double* info_dev,
                         void* stream);

/* Diagnostic: stream floor(bytes / stage_bytes) * stage_bytes bytes of device memory through the STREAM
 * kernels' TMA ring (one CTA per SM, `stages` slots of `stage_bytes`, evict_first bulk copies) with an
 * idle consumer.  Timed by the caller with CUDA events it gives the pure-read ceiling of this GPU for
 * the access pattern of the apply; bench.py reports it beside the roofline. */
int coarse_op_probe_read(const void* src_dev, size_t bytes, int stage_bytes, int stages, void* stream);

void coarse_op_destroy(coarse_op_t* op); /* NULL is a no-op */

const char* coarse_op_last_error(void); /* thread-local, never NULL */

#ifdef __cplusplus
}
#endif
#endif /* COARSE_OP_H */

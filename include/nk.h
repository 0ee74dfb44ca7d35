/* nk.h -- C-ABI of libnk: matrix-free, sum-factorised spectral/hp elemental
 * operators on batches ("blocks") of like elements, fp64, one NVIDIA B200.
 *
 * Citations: P:<n> = line n of the paper text (arxiv/paper_2606_20917,
 * "NektarIR"); A<n> = reading n in DESIGN.md section 3.
 *
 * A *block* is a set of elements with one shape, one polynomial
 * order P, one quadrature order Q and one "deformed" flag.  Here a block is the
 * triple (nk_basis, nk_geom, nelem) plus caller-owned field pointers.
 *
 * Conventions
 *   - nm = P+1 modes per direction (A1); Q quadrature points per direction;
 *     Nq = Q^3 points per element, point index n = i + Q*(j + Q*k), direction-1
 *     index fastest (A11); Nm modes per element in the nest order of Eq. 17
 *     (A3): p outermost, r innermost.
 *   - fields are fp64, element-major: coefficients [nelem][Nm], point values
 *     [nelem][Nq].  All field pointers are DEVICE pointers owned by the caller
 *     unless the name of the call says "_host".  in/out must not alias.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls
 *     enqueue work and return without synchronising (except *_host calls and
 *     nk_geom_upload with host input, which synchronise `stream`).
 *   - handles (nk_basis, nk_geom) are created and destroyed by the library;
 *     every other buffer stays the caller's.
 *   - errors are return codes; nk_last_error() gives a thread-local message.
 *     Nothing throws across the boundary.  There is no CPU fallback: without a
 *     CUDA device every compute call returns NK_ERR_CUDA.
 */
#ifndef NK_H
#define NK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    NK_OK = 0,
    NK_ERR_INVALID_ARG = 1,
    NK_ERR_UNSUPPORTED = 2,    /* (shape,P,Q) outside the instantiation table */
    NK_ERR_SHAPE_MISMATCH = 3, /* basis / geom / nelem do not belong together */
    NK_ERR_ALLOC = 4,
    NK_ERR_CUDA = 5
} nk_status;

typedef enum { NK_HEX = 0, NK_TET = 1, NK_PRISM = 2 } nk_shape;

/* tables readable through nk_basis_get_table (for tests) */
typedef enum {
    NK_TAB_NODES = 0,   /* z^(dir)[Q]                                              */
    NK_TAB_WEIGHTS = 1, /* w^(dir)[Q], collapse Jacobian folded in (A16)           */
    NK_TAB_DERIV = 2,   /* D^(dir)[Q][Q], D[i][r] = h_r'(z_i) (Eq. 22; A5)  */
    NK_TAB_KRON = 4,    /* hexes only; dir 0: M = B^T w B, 1: K = (DB)^T w (DB), 2: C = B^T w (DB), each [nm][nm], row =
                           test mode: the 1-D matrices of the coefficient-space form of the affine operators       */
    NK_TAB_PSI = 3      /* dir 0: psi^a_p(z1_i) as [Q][nm];
                           dir 1: hex/prism psi^a_q(z2_j) as [Q][nm];
                                  tet psi^b_{pq}(z2_j) as [Q][nm(nm+1)/2], column (p,q) = sum_{a<p}(nm-a)+q;
                           dir 2: hex psi^a_r(z3_k) as [Q][nm];
                                  tet/prism psi^b_{sr}(z3_k) as [Q][nm(nm+1)/2], column (s,r) (A7)  */
} nk_table;

typedef struct nk_basis nk_basis; /* opaque: shape, P, Q, host tables (+ device copies, made lazily) */
typedef struct nk_geom nk_geom;   /* opaque: nelem, deformed flag, repacked device streams          */

/* ---- basis / quadrature precompute (host only; needs no GPU) ----------------------------------
 * Modified C0 basis (A7, A8) with Gauss-Lobatto-Legendre points on hexes, GLL x Gauss-Radau-Jacobi(1,0)
 * x GRJ(2,0) on tets, GLL x GLL x GRJ(1,0) on prisms (A9).  Prebuilt kernels: Q == P+2 with
 * hex P in 1..10, tet and prism P in 1..8.  Any other (P, Q) with 1 <= P <= 10, P+1 <= Q <= 12 is accepted too, on every
 * shape, and its kernels are specialised at run time on first use ("run-time specialisation" below); anything else
 * returns NK_ERR_UNSUPPORTED.                                                                              */
nk_status nk_basis_create(nk_shape shape, int P, int Q, nk_basis** out);
nk_status nk_basis_destroy(nk_basis* b);
int nk_basis_num_modes(const nk_basis* b);  /* Nm; -1 if b is NULL */
int nk_basis_num_points(const nk_basis* b); /* Nq = Q^3           */
int nk_basis_interleave(const nk_basis* b, int deformed); /* E: elements per thread block = width of the
                                               internal element-interleaved layout (A12) of affine (0) or
                                               deformed (1) blocks */
/* copies table `which` of direction dir (0,1,2) into host_out; cap = capacity in doubles.
 * NK_ERR_INVALID_ARG if cap is too small.  *count (may be NULL) receives the number of doubles.    */
nk_status nk_basis_get_table(const nk_basis* b, int which, int dir, double* host_out, size_t cap, size_t* count);
/* standard-element coordinates xi of the Nq quadrature points, xi_out[n][3] (cap in doubles >= 3*Nq):
 * the collapsed nodes eta mapped by the inverse of Eq. 13 (A2).  For building geometry inputs. */
nk_status nk_basis_get_points(const nk_basis* b, double* xi_out, size_t cap);
/* storage rank of mode (p,q,r) (Eq. 18; A3); -1 if (p,q,r) is not a mode of the expansion   */
int nk_basis_mode_index(const nk_basis* b, int p, int q, int r);

/* ---- geometry (A13, A14) -------------------------------------------------
 * dxi_dx: [nelem][npt][3][3], entry [j][i] = d xi_j / d x_i, xi = STANDARD-element coordinates (the
 *         collapsed eta of Eq. 13 are internal); detJ: [nelem][npt] > 0.
 * npt = 1 if !deformed (affine: constant factors per element), Nq if deformed (point index n as above).
 * on_device: 0 = the two pointers are host memory, 1 = device memory.  The caller keeps its arrays;
 * the library builds its own element-interleaved streams:
 *   metric stream  G = w|J| (dxi/dx)(dxi/dx)^T (6, symmetric) + w|J| (1)   -- Laplacian / Helmholtz / mass / iprod
 *   factor stream  dxi/dx (9) + w|J| (1)                                    -- physderiv / iprod_deriv
 * with the collapsed-coordinate chain of Eq. 23 (A17) and the quadrature weights folded in when
 * deformed.  nelem == 0 is valid (every apply is then a no-op).                                      */
nk_status nk_geom_upload(const nk_basis* b, int64_t nelem, int deformed, const double* dxi_dx,
                         const double* detJ, int on_device, void* stream, nk_geom** out);
/* The same, building only the streams asked for (a Helmholtz-only caller saves 10 of 17 doubles per point):
 * NK_GEOM_METRIC serves nk_iprod, nk_mass_apply, nk_laplacian_apply and every nk_helmholtz_* call,
 * NK_GEOM_FACTORS serves nk_physderiv and nk_iprod_deriv.  An operator whose stream is missing returns
 * NK_ERR_INVALID_ARG.  nk_geom_upload builds both.                                                    */
enum { NK_GEOM_METRIC = 1, NK_GEOM_FACTORS = 2 };
nk_status nk_geom_upload_streams(const nk_basis* b, int64_t nelem, int deformed, const double* dxi_dx,
                                 const double* detJ, int on_device, unsigned streams, void* stream, nk_geom** out);
nk_status nk_geom_destroy(nk_geom* g);
int64_t nk_geom_num_elements(const nk_geom* g);

/* ---- elemental operators --------------------------------------------------------------------- */
/* BwdTrans, u = B uhat (Eq. 14-17): coeffs [nelem][Nm] -> phys [nelem][Nq].             */
nk_status nk_bwdtrans(const nk_basis* b, int64_t nelem, const double* coeffs, double* phys, void* stream);
/* IProductWRTBase, uhat = B^T W u (Eq. 19-21): phys [nelem][Nq] -> coeffs [nelem][Nm].  */
nk_status nk_iprod(const nk_basis* b, const nk_geom* g, const double* phys, double* coeffs, void* stream);
/* PhysDeriv (Eq. 22, 23, 9): phys -> d_i = du/dx_i, each [nelem][Nq].
 * A NULL d_i skips that component.                                                                 */
nk_status nk_physderiv(const nk_basis* b, const nk_geom* g, const double* phys, double* d0, double* d1,
                       double* d2, void* stream);
/* IProductWRTDerivBase (Eq. 7): coeffs_m = sum_n W_n sum_i (d phi_m/d x_i)(xi_n) g_i[n].
 * A NULL g_i counts as zero.                                                                       */
nk_status nk_iprod_deriv(const nk_basis* b, const nk_geom* g, const double* g0, const double* g1,
                         const double* g2, double* coeffs, void* stream);
/* M uhat = B^T W B uhat (Eq. 7).                                                      */
nk_status nk_mass_apply(const nk_basis* b, const nk_geom* g, const double* in, double* out, void* stream);
/* L uhat = sum_i (D_xi B)^T W (D_xi B) uhat (Eq. 7).                                         */
nk_status nk_laplacian_apply(const nk_basis* b, const nk_geom* g, const double* in, double* out, void* stream);
/* out = (L + lambda M) in (Eq. 5-6; A6), one fused kernel: point data never leaves the SM. */
nk_status nk_helmholtz_apply(const nk_basis* b, const nk_geom* g, double lambda, const double* in,
                             double* out, void* stream);

/* Multi-field block (the `Fields` attribute of a block): the Helmholtz operator applied to nfields
 * (1..8) coefficient fields that share one geometry, e.g. the d velocity components of the velocity-correction
 * scheme, in ONE launch: out[f] = (L + lambda M) in[f].  in / out are HOST arrays of nfields DEVICE
 * pointers, each field [nelem][Nm]; no in[f] may equal any out[h], outputs must be distinct.  The geometry
 * stream is read from HBM once per group and shared by the fields through L2.                             */
nk_status nk_helmholtz_apply_fields(const nk_basis* b, const nk_geom* g, double lambda, int nfields,
                                    const double* const* in, double* const* out, void* stream);

/* several blocks (possibly of different shape / order) in one call, e.g. a hybrid prism + tet mesh   */
typedef struct {
    const nk_basis* basis;
    const nk_geom* geom;
    const double* in; /* device [nelem][Nm] */
    double* out;      /* device [nelem][Nm] */
} nk_block;
/* Block 0 is launched on `stream`, the others on internal side streams forked from and joined to `stream` by events:
 * the kernels of different blocks may overlap (the tail of one with the head of the next), and everything is ordered
 * after earlier and before later work on `stream`.  Blocks must not share output buffers.                     */
nk_status nk_helmholtz_apply_blocks(int nblocks, const nk_block* blocks, double lambda, void* stream);

/* End-to-end variant with HOST field buffers: copies host_in to an internal device buffer, applies the
 * Helmholtz operator and copies the result back into host_out; synchronises `stream` before returning.
 * The work is cut into up to 16 chunks of element groups (at least 2 MB each) and pipelined over two internal copy
 * streams, so that the host-to-device copy of one chunk, the kernel of the previous one and the device-to-host copy
 * of the one before overlap (PCIe is full duplex).  Pinned host memory is needed for the overlap; pageable memory
 * works but serialises.  The staging buffers and the pipeline's streams and events belong to the nk_geom handle
 * (allocated on first use, freed by nk_geom_destroy): calls on ONE geometry are serialised by a lock inside the
 * handle, so the call is thread-safe but not concurrent per geometry; use one nk_geom per concurrent caller.
 * On any error everything that was enqueued is drained before the call returns.                              */
nk_status nk_helmholtz_apply_host(const nk_basis* b, const nk_geom* g, double lambda, const double* host_in,
                                  double* host_out, void* stream);

/* ---- assembly and solver ---------------------------------------------------
 * The paper leaves global assembly out and names the consumer of the elemental operators: "operator evaluations
 * are required within the solver as part of a conjugate gradient or GMRES iteration".  A C0 expansion shares
 * its vertex / edge / face modes between neighbouring elements: (Q u)[e][m] = sign[e][m] * u[l2g[e][m]] gathers a
 * global vector into element-major local coefficients, Q^T adds local contributions into the global vector, and
 * the assembled Helmholtz operator is A = Q^T diag(L^e + lambda M^e) Q (Eq. 6).  The map is the caller's
 * (mesh connectivity is not part of this library).
 * l2g: HOST [nelem][nm_local] global dof of every local mode, 0 <= l2g < nglobal; sign: HOST [nelem][nm_local] of +1 / -1
 * (orientation of shared edge / face modes) or NULL for all +1.  Needs a CUDA device (the map lives on the device). */
typedef struct nk_gs nk_gs;
nk_status nk_gs_create(int64_t nelem, int nm_local, int64_t nglobal, const int64_t* l2g, const signed char* sign, nk_gs** out);
nk_status nk_gs_destroy(nk_gs* gs);
int64_t nk_gs_num_global(const nk_gs* gs);
/* Constrained (Dirichlet) dofs: HOST list of n global dofs (n = 0 removes the constraints).  nk_assembled_helmholtz_apply
 * and nk_cg_solve then work with A_c = P A P + (I - P), P = projector on the free dofs: identity rows and columns at the
 * constrained dofs, so A_c is symmetric positive definite also for lambda = 0 (Poisson) once the boundary is held, and
 * the solution equals the right-hand side at the constrained dofs (0 for homogeneous conditions; for inhomogeneous ones
 * the caller moves A_fc x_c to the right-hand side).  nk_gs_gather / nk_gs_scatter_add themselves ignore the constraints. */
nk_status nk_gs_set_constrained(nk_gs* gs, int64_t n, const int64_t* dofs);
/* local = Q global: device [nglobal] -> device [nelem][nm_local]                                                  */
nk_status nk_gs_gather(const nk_gs* gs, const double* global, double* local, void* stream);
/* global = Q^T local (overwrites global).  Deterministic: one thread per global dof sums its local copies in the
 * order of their local index (transposed map built by nk_gs_create); no atomics.                                  */
nk_status nk_gs_scatter_add(const nk_gs* gs, const double* local, double* global, void* stream);
/* out = Q^T (L + lambda M) Q in on device vectors [nglobal]: gather, ONE fused elemental kernel, scatter.          */
nk_status nk_assembled_helmholtz_apply(const nk_basis* b, const nk_geom* g, const nk_gs* gs, double lambda, const double* in,
                                       double* out, void* stream);
/* The same operation for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): this call allocates NOTHING -- no cudaMalloc / cudaFree, no allocating library routine.  Its two
 * local work vectors ([nelem][nm_local] doubles each) live in a file-scope __device__ array of the library,
 * 2 x NK_STATIC_MAX_LOCAL_DOFS doubles = 16 MiB, which every GPU that loads libnk holds until the process exits.
 *   - nelem * nm_local > NK_STATIC_MAX_LOCAL_DOFS: NK_ERR_UNSUPPORTED (nothing is launched); nk_static_max_local_dofs()
 *     returns the limit of the loaded library.
 *   - a block whose elemental operator would still build device tables (affine block on the reference-matrix form
 *     whose matrices are not resident yet, or a run-time-specialised kernel): NK_ERR_UNSUPPORTED; call
 *     nk_helmholtz_apply once on the block at set-up, or select form 1.  Deformed blocks and affine hexes of order
 *     >= 2 never need that.
 *   - EVERY call on a device shares the one array: calls whose GPU work overlaps (different streams, or two host
 *     threads on one device) race on it -- keep them on one stream or order them with events.  The array keeps the last
 *     call's contents; no entry is read before the same call has written it, so nothing needs clearing.
 * Results are bit-identical to nk_assembled_helmholtz_apply (same kernels, same order of sums).                    */
#define NK_STATIC_MAX_LOCAL_DOFS 1048576
int64_t nk_static_max_local_dofs(void);
nk_status nk_assembled_helmholtz_apply_static(const nk_basis* b, const nk_geom* g, const nk_gs* gs, double lambda, const double* in,
                                              double* out, void* stream);
/* Conjugate gradients on A x = rhs, A as above or its constrained form A_c (symmetric positive definite for lambda > 0,
 * or for lambda = 0 with enough constrained dofs).
 * precond: NK_PRECOND_NONE, or NK_PRECOND_JACOBI = diag(A)^-1 with diag(A) = Q^T diag(H^e); the elemental diagonals are
 * obtained by applying the elemental operator to the Nm unit vectors (Nm launches, once per (geometry, lambda), cached in
 * the nk_gs handle).  The modified basis is badly conditioned without it (16^3 deformed hexes at P4, lambda = 1, to
 * 1e-8: 11384 iterations without, 705 with; profiles/r2_notes.md).
 * x: initial guess on entry, solution on return (device [nglobal]); stops when ||r|| <= rtol ||rhs|| or after maxit
 * iterations; *iters and *relres (may be NULL) receive the iteration count and the last ||r|| / ||rhs||.  All vector
 * work runs on `stream`; the call synchronises it once per iteration to read the residual norm (8 bytes) and before
 * returning.  Sums are reproducible run to run (fixed reduction grid).  Calls on one nk_gs are serialised by a lock
 * in the handle (it owns the work vectors).                                                                        */
enum { NK_PRECOND_NONE = 0, NK_PRECOND_JACOBI = 1 };
nk_status nk_cg_solve(const nk_basis* b, const nk_geom* g, const nk_gs* gs, double lambda, const double* rhs, double* x,
                      int precond, double rtol, int maxit, int* iters, double* relres, void* stream);

/* ---- the same system on a mesh split over ranks (the one exchange step) --------------
 * Elements are independent and the paper's runs give every rank a segment of elements; the ASSEMBLED
 * system couples the segments through the dofs on the cuts.  Each rank (one process per GPU) holds its elements, an
 * nk_gs over its OWN numbering of the dofs its elements touch, and an nk_part that lists which of those dofs other ranks
 * hold too:
 *   shared_dof[i]   rank-local dof (0 <= . < nk_gs_num_global), each at most once;
 *   shared_slot[i]  its position in the interface vector of n_interface entries -- the same numbering on every rank;
 *   shared_mult[i]  number of ranks that hold it (>= 2).
 * Vectors are CONSISTENT: a shared dof carries the same value on every rank that holds it (rhs and the initial x on
 * entry; x on return).  Then
 *   nk_part_assembled_helmholtz_apply:  out = A in, A the operator of the WHOLE mesh: the rank's own Q^T (L + lambda M) Q,
 *       then out[shared] summed over the ranks (pack into the interface vector, all-reduce, unpack);
 *   nk_part_exchange_sum:               that sum alone, in place (e.g. to assemble a right-hand side);
 *   nk_part_cg_solve:                   nk_cg_solve on the whole mesh: dot products weigh a shared dof by 1 / multiplicity
 *       and are all-reduced (one all-reduce of 1 and one of 2 doubles per iteration, one interface all-reduce per
 *       operator application); NK_PRECOND_JACOBI uses the diagonal of the whole mesh's operator.
 * Constrained dofs (nk_gs_set_constrained) must be constrained on every rank that holds them; they are not exchanged.
 * The all-reduce is the caller's: `allreduce(user, device_buf, n, stream)` sums n doubles at the DEVICE pointer in place
 * over all ranks and returns 0; its work must be ordered after everything enqueued on `stream` before the call and
 * before everything enqueued after it (run it on that stream).  The Python binding passes torch.distributed (NCCL over
 * NVLink).  Every rank must make the same sequence of calls (they are collective); a rank without elements takes part
 * with an nk_gs of zero elements.  Iteration counts and residuals are identical on all ranks.                      */
typedef int (*nk_allreduce_fn)(void* user, double* device_buf, int64_t n, void* stream);
typedef struct nk_part nk_part;
nk_status nk_part_create(nk_gs* gs, int64_t n_shared, const int64_t* shared_dof, const int64_t* shared_slot, const int32_t* shared_mult,
                         int64_t n_interface, nk_allreduce_fn allreduce, void* user, nk_part** out);
nk_status nk_part_destroy(nk_part* p);
nk_status nk_part_exchange_sum(nk_part* p, double* vec, void* stream);
nk_status nk_part_assembled_helmholtz_apply(const nk_basis* b, const nk_geom* g, nk_part* p, double lambda, const double* in,
                                            double* out, void* stream);
nk_status nk_part_cg_solve(const nk_basis* b, const nk_geom* g, nk_part* p, double lambda, const double* rhs, double* x, int precond,
                           double rtol, int maxit, int* iters, double* relres, void* stream);

/* ---- form of the affine simplex operators ------------------------------------------------------
 * With constant dxi/dx and |J| the operators of Eq. 6-7 are (L + lambda M)_e = sum_{c<6} G^e_c K_c +
 * lambda |J_e| K_6 with seven Nm x Nm matrices of the STANDARD element (the quadrature sums of Eq. 7 with the chain of
 * Eq. 23 applied to the basis, taken over the points first) and the element's metric G^e = |J| (dxi/dx)(dxi/dx)^T:
 * a dense GEMM with a fixed right-hand matrix, run on the FP64 tensor cores (DMMA) for tets up to P = 5 where it
 * needs fewer flops than the sum-factorised chain.  nk_mass_apply, nk_laplacian_apply and every
 * nk_helmholtz_* call on an AFFINE simplex block take
 *   form 0 (default)  the reference-matrix kernel where it is the faster one (tets of every order, prisms up to P = 3,
 *                     trilinear hexes), else the sum-factorised / Kronecker kernel,
 *   form 1            the sum-factorised kernel (Eq. 17 / 21 / 23 step by step, as on deformed blocks),
 *   form 2            the reference-matrix kernel on EVERY affine block (prisms and hexes of any order too): where no kernel
 *                     is prebuilt for the block's number of modes, the kernel source is specialised for it at run time
 *                     (NVRTC, next paragraph); NK_ERR_UNSUPPORTED at apply time if that is not possible.
 * Process-wide; the initial value is the environment variable NK_SIMPLEX_FORM (0 if unset).                     */
nk_status nk_set_affine_simplex_form(int form);
int nk_get_affine_simplex_form(void);
/* matrix c = 0..6 of the standard element, [Nm][Nm] row-major, symmetric (host memory, cap in doubles >= Nm^2):
 * c = 0 (1,1), 1 (1,2)+(2,1), 2 (1,3)+(3,1), 3 (2,2), 4 (2,3)+(3,2), 5 (3,3): sum_q w_q d_a phi_m d_b phi_n in
 * standard-element coordinates; c = 6: sum_q w_q phi_m phi_n.  Built on first use (host only; needs no GPU).   */
nk_status nk_basis_get_reference_matrix(const nk_basis* b, int c, double* host_out, size_t cap);

/* ---- run-time specialisation (the paper's JIT: "< 1 second" P:350) ----------------
 * Kernels are prebuilt for Q = P+2 (hex P1..P10, tet / prism P1..P8).  What falls outside is compiled by NVRTC on first
 * use from the kernel sources embedded in libnk.so, loaded through the driver API and cached per device; libnvrtc and
 * libcuda are dlopen'ed (no link-time dependency), and a failure surfaces as NK_ERR_UNSUPPORTED at apply time.
 *  - Reference-matrix kernels (one number, the modes per element): csrc/nk_dense.cuh for a mode count outside the
 *    prebuilt table (tets P1..P8, trilinear hexes); cached per (device, modes, operator).
 *  - Sum-factorised kernels: nk_basis_create accepts ANY (shape, P, Q) with 1 <= P <= 10 and P+1 <= Q <= 12 (tets and
 *    prisms of order 10 keep one copy of their psi^b tables instead of two so that they fit the 32 KB kernel-parameter
 *    space): nk_kernel<shape, P, deformed, operator, Q> is instantiated per first use with the launch rules of the prebuilt table (they depend on Q); cached
 *    per (device, shape, P, Q, deformed, operator).  Every operator of this header works on such a basis.
 * nk_jit_compile_check: compile the reference-matrix Helmholtz kernel for `nmodes` without loading it (needs NO GPU):
 * NVRTC's wall time in ms and the cubin size.  nk_jit_compile_check_kernel: the same for one sum-factorised
 * instantiation (op: 0 bwdtrans, 1 iprod, 2 physderiv, 3 iprod_deriv, 4 mass, 5 laplacian, 6 helmholtz, 7 helmholtz on
 * fields).  nk_jit_stats: kernels specialised for launching so far in this process and their compile time. */
nk_status nk_jit_compile_check(int nmodes, double* compile_ms, size_t* cubin_bytes);
nk_status nk_jit_compile_check_kernel(nk_shape shape, int P, int Q, int deformed, int op, double* compile_ms, size_t* cubin_bytes);
nk_status nk_jit_stats(int64_t* kernels, double* compile_ms);

/* ---- diagnostics ----------------------------------------------------------------------------- */
/* Register-only DFMA chains on every SM for `iters` x 1024 FMAs per thread (8 independent chains); *tflops receives the
 * sustained fp64 rate (2 flop per FMA).  This is the measured FP64 roofline denominator.            */
nk_status nk_probe_fp64_peak(int iters, double* tflops, double* ms);
/* The same on the FP64 tensor-core path: mma.sync m8n8k4 f64 (SASS DMMA.8x8x4), 8 independent accumulator chains per
 * warp, `iters` x 128 DMMA per warp.  On B200 both probes read 37.05 TFLOP/s: DMMA and DFMA share one pipe with one
 * peak; what DMMA saves is issue slots and operand traffic (8 FMA per lane and instruction).                        */
nk_status nk_probe_fp64_dmma_peak(int iters, double* tflops, double* ms);
/* number of kernels this library has launched from the calling process so far                      */
int64_t nk_launch_count(void);
const char* nk_last_error(void);
const char* nk_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NK_H */

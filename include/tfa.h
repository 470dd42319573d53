/* include/tfa.h — C ABI of libtfa: two-fluid finite-volume assembly on one B200 (sm_100a).
 *
 * What it computes: one Newton-step assembly of the implicit ideal two-fluid (ion + electron +
 * full Maxwell with hyperbolic divergence cleaning) finite-volume method of arXiv 1809.02532 on
 * an unstructured 2-D mesh of triangles and convex quadrilaterals (mixed freely; the paper's own meshes are
 * Cartesian quadrilaterals, L433, L559) with 18 FP64 unknowns per cell: the pseudo-steady residual
 * R~ (Eq. 13) and its block Jacobian dR~/dP (Eq. 14; computed numerically,
 * L130, by the perturbation loop of Algorithm 1) in 18x18 BSR form, ready for an
 * external Krylov solver.  "L<n>" cites a line of the paper text; "S<n>" a reading in DESIGN.md.
 *
 * Conventions
 *   NEQ = 18.  Variable (column) order: 0..2 B, 3..5 E, 6 Psi, 7 Phi, 8 rho_i, 9 rho_e,
 *   10..12 u_i, 13..15 u_e, 16 T_i, 17 T_e  (update variables "RhoiViTi", L181).  Equation (row)
 *   order is the same with rho -> mass, u -> momentum, T -> total energy (Eq. 3-6).
 *   Normalisation: mu0 = 1, eps0 = 1/c^2, k_B = 1, m_i = 1, m_e = 1/mass_ratio, q_i = +1, q_e = -1.
 *   States are array-of-structs [n_cells][18] FP64.  All cell ids are POST-reorder ids.
 *
 * Pointers: every `const double* state...`, `double* rhs`, `double* bsr_vals`, `grad`, `phi` of
 * the device entry points is a DEVICE pointer owned by the caller (e.g. a torch tensor's
 * data_ptr()); the library neither frees nor retains them.  Mesh inputs of tfa_mesh_create are
 * HOST pointers and are copied.  `tfa_mesh_get` writes to HOST memory.  Entry points ending in
 * `_host` take HOST pointers and do the copies themselves.
 *
 * Streams: `stream` is a cudaStream_t passed as void* (NULL = default stream).  Device entry
 * points are asynchronous on it and never synchronise; `_host` entry points and the mesh
 * builders synchronise the stream before returning.
 *
 * Errors: every int-returning function gives 0 on success or a negative TFA_E* code; no C++
 * exception crosses the ABI; tfa_last_error() returns a thread-local message for the last
 * failure.  Non-physical face states (rho <= 0 or T <= 0) are counted on the device and
 * reported lazily by tfa_check().
 */
#ifndef TFA_H
#define TFA_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define TFA_NEQ 18
#define TFA_BLOCK (TFA_NEQ * TFA_NEQ)
/* entries of an off-diagonal block in the packed Jacobian: its structural non-zeros, 8x8 + 5x5 + 5x5 */
#define TFA_PACKED_BLOCK 114

enum { TFA_OK = 0, TFA_EINVAL = -1, TFA_EMESH = -2, TFA_ENOMEM = -3, TFA_ECUDA = -4, TFA_ENONPHYS = -5, TFA_ESINGULAR = -6 };

/* Physical constants of the model (the paper's "dco" of EulerMFMHDTerm, L177). */
typedef struct tfa_physics {
  double gamma_gas;     /* specific-heat ratio of both fluids (L555); default 5/3 */
  double mass_ratio;    /* m_i/m_e (L555); default 25 */
  double c;             /* speed of light in normalised units (L431); default 20 */
  double gamma_psi;     /* B-cleaning speed factor: flux term gamma^2 Psi (Eq. 2; S1); default 1 */
  double chi_phi;       /* E-cleaning speed factor: flux term (chi c)^2 Phi (Eq. 2); default 1 */
  double rusanov_alpha; /* scale of the Rusanov dissipation |A_n| (Eq. 9; S3); default 1 */
} tfa_physics;

/* Constants of the numerical methods (the "dco"s of the flux, limiter and Jacobian, L195). */
typedef struct tfa_numerics {
  double fd_delta;              /* relative perturbation of the numerical Jacobian (L130; S7); 1e-6 */
  double fd_ref[TFA_NEQ];       /* eps_k = fd_delta * max(|P_k|, fd_ref[k]); 1, except rho_e: 1/mass_ratio */
  double venkat_K;              /* Venkatakrishnan K, eps^2 = (K sqrt(Omega))^3 (L208; S13); 1 */
  double lsq_weight_power;      /* least-squares weight w = |d|^-p (L74; S12); 2 */
  double ausm_Kp, ausm_Ku, ausm_sigma, ausm_beta;  /* AUSM+-up constants (L95-99; S4): 1/4, 3/4, 1, 1/8 */
  double ausm_Minf[2];          /* cut-off Mach number per species (S4); 0.1 */
  int32_t term_mask;            /* bit0 convective flux, bit1 source, bit2 BDF2 time term; 7 */
  int32_t pad_;
} tfa_numerics;

typedef struct tfa_mesh tfa_mesh;
typedef struct tfa_ctx tfa_ctx;

/* items for tfa_mesh_get / tfa_mesh_device_ptr */
enum {
  TFA_FACE_CELLS = 0,      /* int32 [n_faces][2]: (L, R) with L < R, R = -1 on the boundary (S10) */
  TFA_CELL_FACES = 1,      /* int32 [n_cells][F]: face of local edge k = (node k -> node k+1); F = max_faces of
                              tfa_mesh_info (3 or 4); -1 in the fourth slot of a triangle of a mixed mesh */
  TFA_STENCIL_PTR = 2,     /* int32 [n_cells+1]: CSR of the face-vertex neighbour stencil (L74) */
  TFA_STENCIL_IDX = 3,     /* int32 [n_stencil]: ascending, unique, without the cell itself */
  TFA_BSR_ROWPTR = 4,      /* int32 [n_cells+1] */
  TFA_BSR_COL = 5,         /* int32 [nnzb]: self + face neighbours, ascending (cuSPARSE bsr layout) */
  TFA_PERM = 6,            /* int32 [n_cells]: new cell id -> cell id in the arrays given to mesh_create */
  TFA_VOLUME = 7,          /* f64 [n_cells]: cell area Omega_i */
  TFA_FACE_NORMAL_LEN = 8, /* f64 [n_faces][3]: unit normal (L -> R) and length Sigma_f */
  TFA_CENTROID = 9,        /* f64 [n_cells][2] (in the cell's own, unwrapped frame) */
  TFA_FACE_NODES = 10,     /* int32 [n_faces][2]: (lo, hi) node ids; faces are sorted by this key */
  TFA_CELL_NBR = 11,       /* int32 [n_cells][F]: neighbour across local edge k, -1 on the boundary / no such edge */
  TFA_BFACES = 12,         /* int32 [n_bfaces]: the boundary faces (R = -1) in ascending face id; faces are numbered by
                              their node pair, so this list and the tags attached to it survive tfa_mesh_reorder */
  TFA_BC_TAGS = 13         /* int32 [n_bfaces]: TFA_BC_* of each boundary face */
};

/* Rule for the far side P_R of a boundary face (the paper's separate boundary loop, L260; readings S9, S24).
 * Periodic boundaries are not a tag: periodic images are identified topologically in cell_nodes (S9). */
enum {
  TFA_BC_TRANSMISSIVE = 0, /* P_R := P_L; the perturbations of the Jacobian move both arguments (default) */
  TFA_BC_GHOST = 1,        /* P_R := the caller's ghost state of that face (tfa_set_ghost_states), held fixed while
                              P_L is perturbed: Dirichlet / far-field data, or whatever a host loop over the boundary
                              faces (L260) wrote there before the call */
  TFA_BC_WALL = 2          /* P_R := mirror image of P_L: perfectly conducting slip wall, B.n = 0, E_t = 0, u_s.n = 0
                              at the face (B and u_s flip their normal component, E its tangential ones, Phi flips,
                              Psi, rho_s, T_s are kept; S24); moves with P_L */
};

/* ---- step a1: connectivity, geometry, stencil, BSR pattern (L74, L230, L276-319 Listing 1) ----
 * node_xy [n_nodes][2] f64, cell_nodes [n_cells][3] int32 counter-clockwise, cell_xy
 * [n_cells][3][2] f64 per-cell corner coordinates (needed for periodic meshes, where node ids are
 * identified topologically; NULL = gather from node_xy).  HOST pointers, copied.  All derived
 * arrays are built by CUDA kernels on `stream` and owned by the mesh.
 * TFA_EMESH: clockwise/degenerate cell, node pair shared by > 2 cells, a cell that neighbours
 * itself or reaches one neighbour through two faces (periodic direction narrower than 3 cells). */
int tfa_mesh_create(tfa_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                    const int32_t* cell_nodes, const double* cell_xy, void* stream);
/* Mixed mesh of triangles and convex quadrilaterals: the corners of cell i are
 * cell_nodes[cell_ptr[i] .. cell_ptr[i+1]) (3 or 4 of them, counter-clockwise), cell_xy [cell_ptr[n_cells]][2] in the
 * same layout (or NULL).  HOST pointers, copied.  A quadrilateral has 5 BSR blocks in its row.  TFA_EMESH also for a
 * non-convex quadrilateral; TFA_EINVAL for a cell with another number of corners.
 * Limit of both builders: the cells around the corners of one cell (with repetitions) may not exceed 192. */
int tfa_mesh_create_poly(tfa_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                         const int32_t* cell_ptr, const int32_t* cell_nodes, const double* cell_xy, void* stream);
/* max_faces: 3 for a pure triangle mesh, else 4; n_bfaces: number of boundary faces. */
int tfa_mesh_info(const tfa_mesh* m, int32_t* max_faces, int64_t* n_bfaces);
/* Boundary rule of every boundary face: tags [n_bfaces] (HOST pointer, copied) in the order of TFA_BFACES. */
int tfa_mesh_set_bc(tfa_mesh* m, const int32_t* tags, void* stream);
/* Renumber the cells for locality and rebuild every derived array under the same rules.
 * kind 0: none; 1: reverse Cuthill-McKee on the face-neighbour graph, computed on the device
 * (S11: start = unvisited cell of minimum (degree, id); neighbours appended by (degree, id));
 * 2: user_perm[new] = old (HOST pointer, must be a bijection); 3: Z-order (Morton) curve through the cell centroids
 * (16 bits per axis over the centroids' bounding box, ties by cell id), computed on the device: consecutive cells form
 * compact patches, which the gather-bound gradient kernel likes better than RCM's level sets.  The
 * centroids are the cells' own (unwrapped) ones, so on a periodic mesh the curve does not wrap either.
 * Permutations compose into PERM. */
int tfa_mesh_reorder(tfa_mesh* m, int kind, const int32_t* user_perm, void* stream);
int tfa_mesh_sizes(const tfa_mesh* m, int64_t* n_cells, int64_t* n_faces, int64_t* nnzb,
                   int64_t* n_stencil);
/* Copy one item to host memory; `bytes` must equal the item's size.  Blocking: it synchronises the device (the
 * two derived items TFA_VOLUME and TFA_FACE_NORMAL_LEN run a small kernel on the default stream first). */
int tfa_mesh_get(const tfa_mesh* m, int which, void* host_dst, int64_t bytes);
/* Device pointer of an int32 pattern item (TFA_BSR_ROWPTR, TFA_BSR_COL, TFA_PERM, ...) for the
 * solver hand-over (zero copy, as Listing 3); valid until destroy/reorder. */
const void* tfa_mesh_device_ptr(const tfa_mesh* m, int which);
void tfa_mesh_destroy(tfa_mesh* m);

/* ---- constants and workspace ---- */
void tfa_default_physics(tfa_physics* p);
void tfa_default_numerics(tfa_numerics* n, const tfa_physics* p);
int  tfa_ctx_create(tfa_ctx** out);
int  tfa_set_physics(tfa_ctx* ctx, const tfa_physics* p);
int  tfa_set_numerics(tfa_ctx* ctx, const tfa_numerics* n);
/* Ghost states of the TFA_BC_GHOST faces: ghost [n_bfaces][18] FP64, DEVICE pointer in the order of TFA_BFACES,
 * owned by the caller and read (not copied) by every later assembly of this context until replaced; rows of
 * faces with another tag are ignored.  NULL forgets it.  An assembly on a mesh with TFA_BC_GHOST faces and no
 * (or a wrongly sized) ghost array returns TFA_EINVAL. */
int  tfa_set_ghost_states(tfa_ctx* ctx, const double* ghost, int64_t n_bfaces);
/* A context holds the workspace of one assembly at a time: use it from one thread and one stream at a time. */
void tfa_ctx_destroy(tfa_ctx* ctx);

/* ---- step a2 (test hook): least-squares gradient (L74) and Venkatakrishnan limiter (L208) ----
 * grad [n_cells][18][2], phi [n_cells][18]: DEVICE pointers. */
int tfa_gradients(tfa_ctx* ctx, const tfa_mesh* m, const double* state, double* grad, double* phi,
                  void* stream);

/* ---- steps a2..a7: residual + BSR Jacobian (Alg. 1; Eq. 8-14) ----
 * rhs [n_cells][18] = -R~(P);  bsr_vals [nnzb][18][18] row-major blocks of dR~/dP in the
 * mesh's BSR pattern (64-bit offsets inside).  Every entry of both is overwritten (no memset
 * needed, unlike Listing 4); bsr_vals may be NULL for a residual-only evaluation.
 * state_n / state_nm1 are P^n and P^{n-1} of the BDF2 term (Eq. 13).  Deterministic: two calls
 * on the same inputs give bit-identical outputs (no atomics on the data path). */
int tfa_assemble(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n,
                 const double* state_nm1, double dt, double* rhs, double* bsr_vals, void* stream);
/* Same with HOST buffers: copies the three states in, assembles, copies rhs and bsr_vals out,
 * synchronises.  Pinned host memory makes the copies asynchronous DMA; pageable memory works. */
int tfa_assemble_host(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n,
                      const double* state_nm1, double dt, double* rhs, double* bsr_vals, void* stream);
/* The two kernels of tfa_assemble as separate calls, for callers that put something between them (the face-state
 * halo exchange of a sharded assembly, below): tfa_assemble_gradient runs step a2 and leaves the reconstructed
 * face states in the context; tfa_face_states returns that buffer ([n_cells][F][18] FP64, DEVICE pointer owned by
 * the context, valid until the context meets another mesh); tfa_assemble_faces runs steps a3..a7 on it. */
int tfa_assemble_gradient(tfa_ctx* ctx, const tfa_mesh* m, const double* state, void* stream);
int tfa_assemble_faces(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n,
                       const double* state_nm1, double dt, double* rhs, double* bsr_vals, void* stream);
double* tfa_face_states(tfa_ctx* ctx);
/* tfa_assemble_faces writing the packed Jacobian (tfa_assemble_packed, below).  On a shard's mesh: diag_vals
 * [n_owned][18][18] indexed by the owned cell (local id - first_owned_local), offd_vals [nnzb_owned - n_owned][114]:
 * the owned rows' off-diagonal blocks in pattern order -- the same values, bit for bit, as the corresponding pieces
 * of the single-GPU packed arrays (half the Jacobian memory per rank). */
int tfa_assemble_faces_packed(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n,
                              const double* state_nm1, double dt, double* rhs, double* diag_vals, double* offd_vals,
                              void* stream);
/* Step a2 without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): face_states [n_cells][F][18] (DEVICE pointer, caller-owned) = the
 * reconstructed face states tfa_assemble_gradient leaves in the context, bit for bit, from state [n_cells][18]
 * (DEVICE pointer).  The least-squares coefficients, the only scratch of the step, live in a static device array of
 * the library -- 32 MiB on every GPU that loads it, held until the process exits -- that holds
 * TFA_STATIC_MAX_STENCIL stencil entries (STENCIL_PTR[n_cells]: about 170 000 triangles or 260 000 Cartesian
 * quadrilaterals); a mesh with more returns TFA_EINVAL.  The call allocates and frees nothing, on the device or
 * through a library, and does not synchronise; the first call on a device looks the array's address up (make it
 * before a capture starts).  The array is shared by all calls, contexts and streams: every call rewrites the part
 * it reads (nothing needs clearing), so calls in stream order are independent of each other, but two calls that
 * OVERLAP on the GPU (different streams or threads) race on it.  Reads the context's numerics only (weight power,
 * Venkatakrishnan K) and leaves the context's own workspace alone. */
#define TFA_STATIC_MAX_STENCIL 2097152
int tfa_face_states_static(const tfa_ctx* ctx, const tfa_mesh* m, const double* state, double* face_states,
                           void* stream);
/* Synchronise and report: 0, or TFA_ENONPHYS if any assembly since the last check met a face
 * state with rho <= 0 or T <= 0 (S16), or TFA_ECUDA for a sticky CUDA error. */
int tfa_check(tfa_ctx* ctx, void* stream);

/* ---- measurement probes (roofline denominators measured in the same run) ----
 * tfa_probe_dfma: `grid` CTAs x 256 threads each run `iters` x 8 independent FP64 FMAs per
 * thread (2 flops each) -> flops = grid*256*iters*8*2.  tfa_probe_copy: dst[i] = src[i] for n
 * doubles with 16-byte vector accesses -> bytes = 16*n.  Both asynchronous on `stream`. */
int tfa_probe_dfma(int grid, int iters, double* sink, void* stream);
int tfa_probe_copy(const double* src, double* dst, int64_t n, void* stream);
/* The square root and the reciprocal the AUSM flux kernel uses (single-precision hardware seed refined by
 * Newton steps in FP64), applied to x[0..n): sqrt_out[i], rcp_out[i].  DEVICE pointers.
 * Lets the tests bound their error against the correctly rounded results. */
int tfa_probe_math(const double* x, double* sqrt_out, double* rcp_out, int64_t n, void* stream);

/* ---- next step of the method: the linear solve of Eq. 14 (L123) on the assembled BSR system,
 * restarted GMRES with a block-Jacobi preconditioner as in the paper's runs (L28, L392).  All vector and
 * matrix arguments are DEVICE pointers owned by the caller; x, y, b have 18 * n_cells entries. ---- */
/* y = A x for A = bsr_vals in the mesh's BSR pattern. */
int tfa_bsr_spmv(const tfa_mesh* m, const double* bsr_vals, const double* x, double* y, void* stream);
/* dinv [n_cells][18][18] = inverses of the diagonal blocks (Gauss-Jordan with partial pivoting, five blocks per
 * warp; the pivot is the largest remaining entry of the column up to 2^-15 relative, ties to the smallest row).  A
 * singular block (pivot 0, subnormal or not finite) gets a zero inverse and is reported by tfa_check as
 * TFA_ESINGULAR.  bsr_vals and dinv must be 16-byte aligned (the blocks move by TMA bulk copies), else TFA_EINVAL. */
int tfa_block_jacobi(tfa_ctx* ctx, const tfa_mesh* m, const double* bsr_vals, double* dinv, void* stream);
/* Solve A x = b by right-preconditioned GMRES(restart): A M^-1 u = b, x = x0 + M^-1 u, M^-1 = dinv (block
 * diagonal; NULL = no preconditioner).  x holds the initial guess on entry and the solution on return.
 * Orthogonalisation: classical Gram-Schmidt, repeated once when it cancelled more than a factor 10; the small Hessenberg problem is solved on the host
 * with Givens rotations (each iteration synchronises the stream).  Stops when the true residual norm
 * ||b - A x|| <= rtol * ||b|| (checked at every restart; the recurrence's estimate ends a cycle) or after
 * max_iters iterations.  info[0] = iterations done, info[1] = ||b - A x|| / ||b|| on return.
 * The Krylov basis ((restart + 2) vectors) lives in the context's workspace.
 * TFA_ESINGULAR: a residual norm or Krylov vector is not finite, or the Hessenberg column vanished (singular
 * operator); x then holds the last completed cycle's iterate. */
int tfa_gmres(tfa_ctx* ctx, const tfa_mesh* m, const double* bsr_vals, const double* dinv, const double* b,
              double* x, int restart, int max_iters, double rtol, double* info, void* stream);

/* ---- one implicit time step (Eq. 12-14): Newton sub-iterations on the BDF2 pseudo-steady residual ----
 * Repeats  assemble R~(P), dR~/dP  ->  block-Jacobi  ->  GMRES: (dR~/dP) dP = -R~  ->  P += dP   until ||dP||_2 <=
 * newton_tol * (1 + ||P||_2) (the paper's stopping rule ||dP|| < eps, L128, made relative) or max_newton iterations,
 * entirely on the device apart from the scalar tests.  state: P^k, on entry the initial guess (usually P^n), on
 * return P^{n+1}; state_n, state_nm1: P^n, P^{n-1} (must not alias state).  Work arrays, DEVICE pointers owned by the
 * caller: rhs and dP [n_cells][18], bsr_vals [nnzb][18][18], dinv [n_cells][18][18].  matrix_free != 0 solves with
 * the matrix-free operator (tfa_gmres_jfnk; the assembled Jacobian then only feeds the preconditioner).
 * matrix_free == 2 is the fastest assembled variant: packed Jacobian (tfa_assemble_packed; bsr_vals is then only
 * storage and holds the packed form on return: diagonal blocks first, off-diagonal blocks behind them) and the
 * mixed-precision solve tfa_gmres_packed_f32, whose FP32 copies live in the context; not on a shard's mesh.
 * info[0] = Newton iterations done, info[1] = ||dP||_2 / (1 + ||P||_2) of the last one, info[2] = GMRES iterations
 * in total, info[3] = relative residual of the last linear solve.  Errors of the steps it calls are passed on. */
int tfa_implicit_step(tfa_ctx* ctx, const tfa_mesh* m, double* state, const double* state_n, const double* state_nm1,
                      double dt, double* rhs, double* bsr_vals, double* dinv, double* dP, int max_newton,
                      double newton_tol, int restart, int max_iters, double rtol, int matrix_free, double* info,
                      void* stream);

/* ---- packed Jacobian (second option) ----
 * The flux Jacobian of a face is block diagonal -- fields 8x8, ions 5x5, electrons 5x5 (only the source couples the
 * groups, on the diagonal block) -- so 210 of the 324 entries of every off-diagonal BSR block are structural zeros:
 * 5040 of the 10368 bytes per cell the BSR assembly writes.  The packed form stores the same matrix in two arrays:
 *   diag_vals [n_cells][18][18]        the diagonal blocks, full, indexed by the cell;
 *   offd_vals [nnzb - n_cells][114]    the off-diagonal blocks in BSR order with the diagonal ones taken out (row i:
 *                                      slots BSR_ROWPTR[i] - i ..., columns = the row's BSR_COL entries other than
 *                                      i); per block: the 8x8 field sub-block (rows / columns 0..7), then the ion
 *                                      5x5 (rows / columns 8, 10, 11, 12, 16), then the electron 5x5 (9, 13, 14, 15,
 *                                      17), each row-major.
 * tfa_assemble_packed = tfa_assemble writing that form (same arithmetic, same rhs, bit-identical entries; 5328
 * instead of 10368 bytes of Jacobian per triangle); tfa_packed_to_bsr expands it into the mesh's BSR value array;
 * tfa_packed_spmv, tfa_block_jacobi_packed and tfa_gmres_packed are the linear-solve entry points on it (single
 * mesh only; a shard assembles the packed form with tfa_assemble_faces_packed, tfa_assemble_packed refuses its mesh).  All pointers DEVICE pointers; the packed arrays, x and dinv must be 16-byte aligned
 * (the blocks move by TMA bulk copies and 16-byte loads; TFA_EINVAL otherwise). */
int tfa_assemble_packed(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n,
                        const double* state_nm1, double dt, double* rhs, double* diag_vals, double* offd_vals,
                        void* stream);
int tfa_packed_to_bsr(const tfa_mesh* m, const double* diag_vals, const double* offd_vals, double* bsr_vals,
                      void* stream);
int tfa_packed_spmv(const tfa_mesh* m, const double* diag_vals, const double* offd_vals, const double* x, double* y,
                    void* stream);
int tfa_block_jacobi_packed(tfa_ctx* ctx, const tfa_mesh* m, const double* diag_vals, double* dinv, void* stream);
/* Mixed-precision solve on the packed Jacobian: the Krylov cycles of GMRES(restart) run on an FP32 copy of the matrix
 * (and, when dinv32 is given, of the block-Jacobi inverses; NULL = no preconditioner) and keep their basis vectors
 * in FP32 (each is rounded once, when it is normalised; the projections, the work vector, the sums and the Hessenberg
 * problem are FP64); the residual b - A x at every restart, and the one reported in info[1], is computed with the FP64
 * matrix, and a cycle ends once it has reduced its own residual by 1e-5 (iterative refinement with GMRES as the
 * inner solver: the FP32 copy perturbs the operator by 6e-8 relative, which a restart corrects).  Same stopping
 * rule, same error codes as tfa_gmres_packed (matrix entries beyond the FP32 range become infinite in the copy and
 * end the solve with TFA_ESINGULAR).  The copies are the caller's: tfa_packed_to_f32 fills
 * diag32 [n_cells][18][18] and offd32 [nnzb - n_cells][TFA_PACKED_BLOCK_F32] (114 entries + 2 of padding: blocks
 * 464 bytes apart), tfa_to_f32 converts any array (the inverses dinv -> dinv32).  DEVICE pointers, 16-byte aligned. */
#define TFA_PACKED_BLOCK_F32 116
int tfa_to_f32(const double* src, float* dst, int64_t n, void* stream);
int tfa_packed_to_f32(const tfa_mesh* m, const double* diag_vals, const double* offd_vals, float* diag32, float* offd32,
                      void* stream);
int tfa_gmres_packed_f32(tfa_ctx* ctx, const tfa_mesh* m, const double* diag_vals, const double* offd_vals,
                         const float* diag32, const float* offd32, const float* dinv32, const double* b, double* x,
                         int restart, int max_iters, double rtol, double* info, void* stream);
int tfa_gmres_packed(tfa_ctx* ctx, const tfa_mesh* m, const double* diag_vals, const double* offd_vals,
                     const double* dinv, const double* b, double* x, int restart, int max_iters, double rtol,
                     double* info, void* stream);

/* ---- matrix-free operator (the paper's future work, L130): out = (dR~/dP) v by a forward
 * difference of the residual-only assembly, (R~(P + eps v) - R~(P)) / eps — the full dependence, gradient and
 * limiter included (the assembled Jacobian freezes them, S8): NOT the same linearisation as bsr_vals; where the
 * limiter is active its min/max make the residual non-smooth and the difference quotient noisy.
 * eps <= 0: eps = 1e-7 (1 + rms(P)) / rms(v).
 * DEVICE pointers; synchronises the stream when eps is chosen automatically. */
int tfa_jvp(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n, const double* state_nm1,
            double dt, const double* v, double* out, double eps, void* stream);
/* tfa_gmres with that operator in place of the assembled matrix (no 10 KB/cell Jacobian to write or read); dinv
 * (optional) is a block-Jacobi preconditioner from an assembled, possibly lagged, Jacobian. */
int tfa_gmres_jfnk(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n,
                   const double* state_nm1, double dt, const double* dinv, const double* b, double* x, int restart,
                   int max_iters, double rtol, double* info, void* stream);

/* ---- sharding over several GPUs (device memory is the limit the paper names, L26) ----
 * Rank r of n owns the cells [r nc / n, (r+1) nc / n) of the global mesh's current order (reorder it first), their
 * rows of rhs and of the BSR matrix, and keeps ghost copies of the cells its reconstruction stencils reach.  Local
 * cell ids are ascending in global id: ghosts below the owned range, the owned range [first_owned_local,
 * first_owned_local + n_owned), ghosts above; an owned row comes out bit-identical to the single-GPU assembly.
 * One assembly = two neighbour-only exchanges, no reduction (the caller moves the packed buffers, e.g. with NCCL
 * send/recv; api.py does):
 *     exchange TFA_HALO_STATE on the state arrays          (18 doubles per ghost cell)
 *     tfa_assemble_gradient(ctx, tfa_shard_mesh(s), state)
 *     exchange TFA_HALO_FACE on tfa_face_states(ctx)       (F x 18 doubles per ghost cell next to an owned cell)
 *     tfa_assemble_faces(ctx, tfa_shard_mesh(s), ..., rhs, vals)
 * rhs has n_local rows (ghost rows are scratch); vals has nnzb_owned blocks: the owned rows of the local mesh's
 * pattern, i.e. blocks [block_offset, block_offset + nnzb_owned) of it (rowptr / col: the local mesh's
 * TFA_BSR_ROWPTR entries first_owned_local .. minus block_offset, TFA_BSR_COL from block_offset on; columns are
 * LOCAL cell ids).  Boundary rules are taken over from the global mesh at creation; do not call tfa_mesh_set_bc
 * on the shard's mesh.  Ghost states: row b of the context's array belongs to the LOCAL boundary face b, whose
 * global boundary-face index (or -1 for a cut face) tfa_shard_bface_global gives.
 *
 * tfa_partition_* is the host-only half (no CUDA call): the same lists from HOST copies of the global mesh's
 * TFA_CELL_NBR, TFA_STENCIL_PTR, TFA_STENCIL_IDX.  Lists hold LOCAL cell ids in ascending global id, so that the
 * sender's TFA_PART_SEND_* list for a peer and that peer's TFA_PART_RECV_* list for the sender name the same
 * cells in the same order. */
typedef struct tfa_partition tfa_partition;
typedef struct tfa_shard tfa_shard;
enum { TFA_PART_LOCAL_TO_GLOBAL = 0, TFA_PART_SEND_STATE = 1, TFA_PART_RECV_STATE = 2, TFA_PART_SEND_FACE = 3,
       TFA_PART_RECV_FACE = 4 };
enum { TFA_HALO_STATE = 0, TFA_HALO_FACE = 1 };
int  tfa_partition_create(tfa_partition** out, int64_t n_cells, int max_faces, const int32_t* cell_nbr,
                          const int32_t* stencil_ptr, const int32_t* stencil_idx, int n_ranks, int rank);
void tfa_partition_destroy(tfa_partition* p);
int  tfa_partition_sizes(const tfa_partition* p, int64_t* n_local, int64_t* n_owned, int64_t* first_owned_local,
                         int64_t* first_owned_global);
/* number of entries of a list (peer ignored for TFA_PART_LOCAL_TO_GLOBAL), -1 on a bad argument */
int64_t tfa_partition_count(const tfa_partition* p, int which, int peer);
int  tfa_partition_get(const tfa_partition* p, int which, int peer, int32_t* host_dst, int64_t count);
/* Build rank `rank`'s shard from the global mesh (which every rank builds for itself and may destroy afterwards). */
int  tfa_shard_create(tfa_shard** out, const tfa_mesh* global_mesh, int n_ranks, int rank, void* stream);
void tfa_shard_destroy(tfa_shard* s);
const tfa_mesh* tfa_shard_mesh(const tfa_shard* s);             /* owned by the shard */
const tfa_partition* tfa_shard_partition(const tfa_shard* s);   /* owned by the shard */
int  tfa_shard_info(const tfa_shard* s, int64_t* nnzb_owned, int64_t* block_offset);
int  tfa_shard_bface_global(const tfa_shard* s, int32_t* host_dst, int64_t count /* = local n_bfaces */);
/* buf[r] = row (send list of `peer`)[r] of src;  row (recv list of `peer`)[r] of dst = buf[r].  Rows are 18 doubles
 * (TFA_HALO_STATE) or F x 18 doubles (TFA_HALO_FACE).  DEVICE pointers, asynchronous on `stream`. */
int  tfa_shard_pack(const tfa_shard* s, int kind, int peer, const double* src, double* buf, void* stream);
int  tfa_shard_unpack(const tfa_shard* s, int kind, int peer, const double* buf, double* dst, void* stream);

/* Per-kernel timing with CUDA events recorded on the launching stream (bench.py's roofline).
 * tfa_timing_enable(ctx, 1): every later tfa_assemble records events before, between and after
 * its two kernels and accumulates their durations at the next tfa_timing_read, which
 * synchronises on the last event, writes the accumulated milliseconds since the previous read
 * to ms[0] (gradient + limiter kernel) and ms[1] (assembly kernel), the number of assemblies
 * to *n_calls, and resets the accumulators.  At most 64 assemblies may be outstanding (the residual evaluations
 * inside tfa_jvp / tfa_gmres_jfnk are not timed and do not count). */
int tfa_timing_enable(tfa_ctx* ctx, int on);
int tfa_timing_read(tfa_ctx* ctx, double* ms /*[2]*/, int* n_calls);

/* Number of kernels the last tfa_assemble launched (for bench.py's gpu_launches). */
int tfa_launches_per_assemble(const tfa_ctx* ctx);
const char* tfa_last_error(void);
const char* tfa_version(void);

#ifdef __cplusplus
}
#endif
#endif

/* oracle/tfo.h — CPU ORACLE of the two-fluid FV residual + BSR-Jacobian assembly.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_1809_02532_b200/, include/,
 * csrc/) includes, links or calls this.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load liboracle_tfo.so.
 *
 * Plain, slow, step-by-step C++ restatement of the method of arXiv 1809.02532
 * (PAPER.md; line numbers "L<n>" cite /root/reference/PAPER.md) in FP64, following the
 * readings S1..S23 listed in DESIGN.md.  No blocking, fusion or reordering beyond what
 * Algorithm 1 (L221-256) states.  All pointers are HOST pointers.
 *
 * Cells are triangles or convex quadrilaterals, mixed freely (the paper's meshes are Cartesian
 * quadrilaterals, L433, L559); boundary faces follow one of three rules (L260; S9, S24).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   connectivity  : Euler counts, tests/golden/ hand-worked 2x2 meshes (triangles, quadrilaterals),
 *                   brute-force O(n^2) adjacency, independent serial RCM
 *   geometry      : Green's-theorem area and centroid, both diagonal splits of a quadrilateral, closed normals
 *   gradient      : exact for linear fields; on Cartesian quads equal to the weighted central differences;
 *                   limiter closed forms: phi = 1 (constant field), 0.75 point, K = 0 and finite K on a linear
 *                   field (eps^2 = (K sqrt(Omega))^3)
 *   Maxwell flux  : consistency L85, exact upwind vs numpy eig of A_n, eigenvalues, antisymmetry
 *   AUSM+-up      : consistency L85, antisymmetry, supersonic upwinding, rotation covariance; magnitudes of the
 *                   pressure-diffusion term M_p (fluid at rest, closed form) and of the velocity-diffusion term
 *                   p_u (symmetric streams, closed form)
 *   source        : momentum/energy bookkeeping  sum_s S_mom = rho_c E + J x B, sum S_en = J.E
 *   residual      : free-stream preservation, periodic telescoping, rotation covariance
 *   Jacobian      : brute-force central differences of the oracle's own frozen residual (triangles, quadrilaterals,
 *                   mixed, with all three boundary rules); Maxwell sub-block linear; time term vs dU/dP by FD
 *   boundary      : wall mirror state is an involution with B.n = E_t = u.n = 0 at the face and no mass, energy,
 *                   Psi or tangential flux through it; a ghost-state face fed the neighbour's face state is an
 *                   interior face (cut-mesh test)
 *   against the paper (tests/test_exact_wave.py, test_oracle_quads.py): the exact circularly polarised wave of
 *                   Eq. 15-18 makes the spatial residual converge at second order (split triangles, and the
 *                   paper's 2N x N quadrilaterals); Newton on a BDF2 step of it contracts and lands on the exact
 *                   solution; Harris-sheet total force balance and Ampere's law (GEM set-up)
 * Unpinned (no independent value available):
 *   |A_n| vs ref. [4] of the paper (S3), AUSM+-up constants / a_1/2 choice vs COOLFluiD (S4),
 *   LS weight exponent (S12: any weight is exact on linear fields).  (The wall rule, S24, is this library's own
 *   definition -- the paper defines no wall -- and is pinned by the properties that define it.)
 */
#ifndef TFO_H
#define TFO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define TFO_NEQ 18

typedef struct tfo_physics {
  double gamma_gas;     /* specific-heat ratio (L555) */
  double mass_ratio;    /* m_i/m_e (L555) ; m_i = 1 */
  double c;             /* speed of light, normalised (L431) */
  double gamma_psi;     /* B-divergence cleaning speed factor (L50 "gamma^2 Psi"), reading S1 */
  double chi_phi;       /* E-divergence cleaning speed factor (L50 "(chi c)^2 Phi") */
  double rusanov_alpha; /* scaling of the Rusanov dissipation (L89 "scaled dissipation"), S3 */
} tfo_physics;

typedef struct tfo_numerics {
  double fd_delta;          /* relative finite-difference step (S7) */
  double fd_ref[TFO_NEQ];   /* reference magnitudes for the step (S7) */
  double venkat_K;          /* Venkatakrishnan K (S13) */
  double lsq_weight_power;  /* w = |d|^-p (S12) */
  double ausm_Kp, ausm_Ku, ausm_sigma, ausm_beta;   /* AUSM+-up constants (S4) */
  double ausm_Minf[2];      /* cut-off Mach number per species (S4) */
  int32_t term_mask;        /* bit0 convective flux, bit1 source, bit2 BDF2 time term */
  int32_t pad_;
} tfo_numerics;

typedef struct tfo_mesh tfo_mesh;

enum { TFO_FACE_CELLS = 0, TFO_CELL_FACES = 1 /* [nc][max_faces], -1 padded */, TFO_STENCIL_PTR = 2,
       TFO_STENCIL_IDX = 3, TFO_BSR_ROWPTR = 4, TFO_BSR_COL = 5, TFO_PERM = 6, TFO_VOLUME = 7,
       TFO_FACE_NORMAL_LEN = 8, TFO_CENTROID = 9, TFO_FACE_NODES = 10,
       TFO_BFACES = 12 /* int32 [n_bfaces]: boundary faces, ascending face id */, TFO_BC_TAGS = 13 };

/* cells are triangles or convex quadrilaterals (the paper's meshes are Cartesian quads, L433, L559) */
#define TFO_MAXV 4
/* rule for the far side of a boundary face (the paper's separate boundary loop, L260; readings S9, S24) */
enum { TFO_BC_TRANSMISSIVE = 0 /* P_R := P_L */, TFO_BC_GHOST = 1 /* P_R := given ghost state, held fixed */,
       TFO_BC_WALL = 2 /* P_R := mirror image of P_L: perfectly conducting slip wall */ };

/* connectivity + geometry (L74, L230) */
int  tfo_mesh_create(tfo_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                     const int32_t* cell_nodes, const double* cell_xy);
/* mixed triangle / quadrilateral mesh: corners of cell i are cell_nodes[cell_ptr[i] .. cell_ptr[i+1]),
 * counter-clockwise; cell_xy [cell_ptr[n_cells]][2] in the same layout (or NULL) */
int  tfo_mesh_create_poly(tfo_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                          const int32_t* cell_ptr, const int32_t* cell_nodes, const double* cell_xy);
int  tfo_mesh_reorder(tfo_mesh* m, int kind /*0 none, 1 RCM, 2 user*/, const int32_t* user_perm);
int  tfo_mesh_info(const tfo_mesh* m, int32_t* max_faces, int64_t* n_bfaces);
/* tags [n_bfaces] (order of TFO_BFACES); ghost [n_bfaces][18] (copied; may be NULL without TFO_BC_GHOST faces) */
int  tfo_mesh_set_bc(tfo_mesh* m, const int32_t* tags, const double* ghost);
int  tfo_mesh_sizes(const tfo_mesh* m, int64_t* n_cells, int64_t* n_faces, int64_t* nnzb,
                    int64_t* n_stencil);
int  tfo_mesh_get(const tfo_mesh* m, int which, void* dst, int64_t bytes);
void tfo_mesh_destroy(tfo_mesh* m);

void tfo_default_physics(tfo_physics* p);
void tfo_default_numerics(tfo_numerics* n, const tfo_physics* p);

/* step a2: LS gradient (L74) + Venkatakrishnan limiter (L208). grad[nc][18][2], phi[nc][18] */
int tfo_gradients(const tfo_mesh* m, const tfo_numerics* nu, const double* state, double* grad,
                  double* phi);

/* steps a3..a7 (Alg. 1; Eq. 8-13).  rows==NULL: all rows, rhs[nc][18], scale[nc][18]
 * (sum of |terms| per entry, may be NULL), vals[nnzb][18][18] (may be NULL -> residual only).
 * rows!=NULL: compact output for the listed rows: rhs[n_rows][18], scale[n_rows][18],
 * vals[n_rows][max_faces+1][18][18] (the row's blocks in BSR column order, zero padded). */
int tfo_assemble(const tfo_mesh* m, const tfo_physics* ph, const tfo_numerics* nu,
                 const double* state, const double* state_n, const double* state_nm1, double dt,
                 double* rhs, double* scale, double* vals, int64_t n_rows, const int32_t* rows);

/* residual with caller-supplied (frozen) gradient and limiter — used by the brute-force pin */
int tfo_residual_frozen(const tfo_mesh* m, const tfo_physics* ph, const tfo_numerics* nu,
                        const double* state, const double* grad, const double* phi,
                        const double* state_n, const double* state_nm1, double dt, double* rhs);

/* point functions, exported for the pins */
void tfo_flux_maxwell(const tfo_physics* ph, const double* UL, const double* UR, double nx,
                      double ny, double* H8);
void tfo_flux_ausm(const tfo_physics* ph, const tfo_numerics* nu, int species, const double* PL5,
                   const double* PR5, double nx, double ny, double* H5);
void tfo_flux_face(const tfo_physics* ph, const tfo_numerics* nu, const double* PL18,
                   const double* PR18, double nx, double ny, double* H18);
void tfo_phys_flux(const tfo_physics* ph, const double* P18, double nx, double ny, double* F18);
void tfo_wall_ghost(const double* P18, double nx, double ny, double* G18);   /* S24 */
void tfo_source(const tfo_physics* ph, const double* P18, double* S18);
void tfo_cons(const tfo_physics* ph, const double* P18, double* U18);
void tfo_dcons_dprim(const tfo_physics* ph, const double* P18, double* dUdP /*[18][18]*/);
/* AUSM+-up split functions: out = {M4+(M), M4-(M), P5+(M), P5-(M)} */
void tfo_ausm_split(double M, double alpha, double beta, double* out4);
int  tfo_num_threads(void);
void tfo_set_num_threads(int n);   /* size of the OpenMP team of later calls (bench.py's one-thread timing) */
const char* tfo_last_error(void);

#ifdef __cplusplus
}
#endif
#endif

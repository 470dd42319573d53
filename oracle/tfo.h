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
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   connectivity  : Euler counts, tests/golden/ hand-worked 2x2 mesh, brute-force O(n^2) adjacency
 *   gradient      : exact for linear fields; limiter closed forms (phi=1 const field, 0.75 point)
 *   Maxwell flux  : consistency L85, exact upwind vs numpy eig of A_n, eigenvalues, antisymmetry
 *   AUSM+-up      : consistency L85, antisymmetry, supersonic upwinding, rotation covariance
 *   source        : momentum/energy bookkeeping  sum_s S_mom = rho_c E + J x B, sum S_en = J.E
 *   residual      : free-stream preservation, periodic telescoping, rotation covariance
 *   Jacobian      : brute-force central differences of the oracle's own frozen residual;
 *                   Maxwell sub-block against the closed-form matrix; time term vs dU/dP by FD
 *   against the paper (tests/test_exact_wave.py): the exact circularly polarised wave of Eq. 15-18 makes the
 *                   spatial residual converge at second order; Newton on a BDF2 step of it contracts and lands
 *                   on the exact solution; Harris-sheet total force balance and Ampere's law (GEM set-up)
 * Unpinned (no independent value available):
 *   |A_n| vs ref. [4] of the paper (S3), AUSM+-up constants / a_1/2 choice vs COOLFluiD (S4),
 *   LS weight exponent (S12), Venkatakrishnan eps^2=(K h)^3 (S13).
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

enum { TFO_FACE_CELLS = 0, TFO_CELL_FACES = 1, TFO_STENCIL_PTR = 2, TFO_STENCIL_IDX = 3,
       TFO_BSR_ROWPTR = 4, TFO_BSR_COL = 5, TFO_PERM = 6, TFO_VOLUME = 7,
       TFO_FACE_NORMAL_LEN = 8, TFO_CENTROID = 9, TFO_FACE_NODES = 10 };

/* connectivity + geometry (L74, L230) */
int  tfo_mesh_create(tfo_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                     const int32_t* cell_nodes, const double* cell_xy);
int  tfo_mesh_reorder(tfo_mesh* m, int kind /*0 none, 1 RCM, 2 user*/, const int32_t* user_perm);
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
 * vals[n_rows][4][18][18] (the row's blocks in BSR column order, zero padded). */
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
void tfo_source(const tfo_physics* ph, const double* P18, double* S18);
void tfo_cons(const tfo_physics* ph, const double* P18, double* U18);
void tfo_dcons_dprim(const tfo_physics* ph, const double* P18, double* dUdP /*[18][18]*/);
/* AUSM+-up split functions: out = {M4+(M), M4-(M), P5+(M), P5-(M)} */
void tfo_ausm_split(double M, double alpha, double beta, double* out4);
int  tfo_num_threads(void);
const char* tfo_last_error(void);

#ifdef __cplusplus
}
#endif
#endif

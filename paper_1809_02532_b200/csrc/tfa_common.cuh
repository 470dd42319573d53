// tfa_common.cuh — internal types shared by the translation units of libtfa (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "../../include/tfa.h"

#define NEQ TFA_NEQ
#define BLK TFA_BLOCK

namespace tfa {

int set_error(int code, const std::string& msg);
uint64_t next_mesh_uid();

#define TFA_CUDA(expr)                                                                          \
  do {                                                                                          \
    cudaError_t e__ = (expr);                                                                   \
    if (e__ != cudaSuccess)                                                                     \
      return tfa::set_error(e__ == cudaErrorMemoryAllocation ? TFA_ENOMEM : TFA_ECUDA,          \
                            std::string(#expr) + ": " + cudaGetErrorString(e__));               \
  } while (0)

#define TFA_TRY(expr)          \
  do {                         \
    int rc__ = (expr);         \
    if (rc__ != 0) return rc__; \
  } while (0)

inline unsigned cdiv(int64_t a, int64_t b) { return (unsigned)((a + b - 1) / b); }

// Index limits of one assembly, for the bounds-checking build (-DTFA_DEBUG_BOUNDS: `TFA_NVCC_EXTRA=-DTFA_DEBUG_BOUNDS
// python -m paper_1809_02532_b200.build --force`).  compute-sanitizer is closed on the GPU pool this was developed on
// (profiles/r2_sanitizers.md); this build checks every gathered row index and every block index the per-step kernels
// form against the sizes of the arrays they address and counts violations in flags[2], which tfa_check reports.
struct Limits {
  int64_t n_cells, n_face_rows, n_blocks, n_mirror_blocks, n_ghost, n_stencil;
};
#ifdef TFA_DEBUG_BOUNDS
#define TFA_BOUND(flags, cond)                 \
  do {                                         \
    if (!(cond)) atomicAdd((flags) + 2, 1);    \
  } while (0)
#else
#define TFA_BOUND(flags, cond) \
  do {                         \
  } while (0)
#endif

// Per-cell geometry record, 8 F doubles (F = faces per cell slot of the mesh: 3 -> 192 B, 4 -> 256 B; DESIGN.md
// "Data layout"):
//   for local face k = 0..F-1 at [8k .. 8k+7]:
//     0 nx, 1 ny   unit normal pointing OUT of this cell: the face's normal, computed from its L
//                  cell's corners (S10), with the sign flipped when this cell is the face's R cell
//     2 len        face length Sigma_f
//     3 dxo, 4 dyo face midpoint minus OWN centroid (own corner coordinates)
//     5 dxn, 6 dyn face midpoint minus NEIGHBOUR centroid (neighbour's corner coordinates);
//                  on a boundary face the own-side values again
//     7 extra      k=0: volume Omega_i;  k=1: sqrt(Omega_i);  else unused (0)
//   The fourth slot of a triangle in a mixed mesh is a face of zero length (normal (1,0), zero offsets): it runs
//   through the same code as a transmissive boundary face and contributes exactly nothing.
constexpr int cgeo_stride(int F) { return 8 * F; }
// block map of cell i: [0] = BSR block index of (i,i), [1+k] = of (nbr_k, i), the block cell i writes INTO ITS
// NEIGHBOUR'S ROW; -1 if none.  Stride 4 ints for F = 3, 8 ints for F = 4 (16-byte aligned rows).
constexpr int blk_stride(int F) { return F == 3 ? 4 : 8; }
// Packed neighbour of local face k (nbrf): interior 4 * neighbour + (the face's local index in the neighbour);
// boundary -1 - (4 * boundary-face index + TFA_BC_* tag); a triangle's fourth slot -1 (= transmissive, zero length).

template <class T>
struct DevBuf {
  T* p = nullptr;
  int64_t n = 0;
  DevBuf() = default;
  DevBuf(const DevBuf&) = delete;
  DevBuf& operator=(const DevBuf&) = delete;
  ~DevBuf() { release(); }
  void release() {
    if (p) cudaFree(p);
    p = nullptr;
    n = 0;
  }
  cudaError_t alloc(int64_t count) {
    release();
    if (count <= 0) count = 1;
    cudaError_t e = cudaMalloc((void**)&p, (size_t)count * sizeof(T));
    if (e == cudaSuccess) n = count;
    return e;
  }
  void swap(DevBuf& o) {
    T* tp = p; p = o.p; o.p = tp;
    int64_t tn = n; n = o.n; o.n = tn;
  }
};

}  // namespace tfa

struct tfa_mesh {
  int64_t nn = 0, nc = 0, nf = 0, nnzb = 0, nst = 0, nb = 0;
  int F = 3;                 // face slots per cell: 3 (triangles only) or 4 (some quadrilaterals)
  bool has_ghost = false;    // some boundary face carries TFA_BC_GHOST
  bool shard_local = false;  // the local mesh of a tfa_shard: its tables are the shard's (no set_bc, no packed output)
  uint64_t uid = 0;          // process-wide monotonic stamp, new at every (re)build; ctx workspaces key on it
  tfa::DevBuf<double> node_xy;     // [nn][2]
  tfa::DevBuf<int32_t> cell_nodes; // [nc][F], -1 in the fourth slot of a triangle
  tfa::DevBuf<double> cell_xy;     // [nc][F][2]
  tfa::DevBuf<int32_t> perm;       // [nc] new -> original
  // derived
  tfa::DevBuf<int32_t> face_nodes, face_cells;  // [nf][2]
  tfa::DevBuf<int32_t> cell_faces, cell_nbr;    // [nc][F]
  tfa::DevBuf<int32_t> nbrf;                    // [nc][F] packed neighbour (see above)
  tfa::DevBuf<int32_t> st_ptr, st_idx;          // CSR stencil
  tfa::DevBuf<double> st_d;                     // [nst][2] centroid displacement (S9)
  tfa::DevBuf<int32_t> bsr_rowptr, bsr_col;
  tfa::DevBuf<int32_t> blkmap;                  // [nc][blk_stride(F)]
  tfa::DevBuf<int32_t> pblkmap;                 // the same for the packed Jacobian: [0] = the cell, [1+k] = slot of (nbr_k, i)
                                                // in the off-diagonal array (tfa.h TFA_PACKED_BLOCK)
  tfa::DevBuf<double> cen;                      // [nc][2]
  tfa::DevBuf<double> cgeo;                     // [nc][8 F]
  tfa::DevBuf<double> ggeo;                     // [nc][2 F + 2]: what the gradient kernel needs of it, packed for 16-byte
                                                // loads: (dxo, dyo) of each face, then sqrt(Omega), 0
  tfa::DevBuf<int32_t> bfaces, bface_of, bc_tag;  // [nb], [nf], [nb]
};

struct tfa_ctx {
  tfa_physics ph;
  tfa_numerics nu;
  // workspace, keyed on (mesh uid, lsq_weight_power).  A context serves one stream at a time and is not thread-safe.
  uint64_t ws_uid = 0;
  double ws_power = -1.0;
  tfa::DevBuf<double> lsq_coef;   // [nst][2]
  tfa::DevBuf<double> fown;       // [nc][F][18] own-side face states P_i + phi grad P_i . (x_f - x_i)  (L232)
  const double* ghost = nullptr;  // caller-owned device array [ghost_n][18] (tfa_set_ghost_states)
  int64_t ghost_n = 0;
  tfa::DevBuf<int32_t> flags;     // [4] device counters: 0 = non-physical states
  // Krylov workspace of tfa_gmres: (restart + 2) vectors of 18 nc doubles, and reduction scratch
  tfa::DevBuf<double> krylov, red;
  // matrix-free operator: perturbed state and its residual; the base residual
  tfa::DevBuf<double> jfnk, jfnk0;
  // FP32 copies of the packed Jacobian and of the block-Jacobi inverses (tfa_implicit_step, mode 2)
  tfa::DevBuf<float> mixed;
  // device staging buffers of tfa_assemble_host
  tfa::DevBuf<double> stage_state[3], stage_rhs, stage_vals;
  int launches = 0;
  int asm_resident_ctas[4] = {0, 0, 0, 0};   // persistent grid of k_assemble<F = 3, 4> x <BSR, packed> on this context's device
  // optional per-kernel timing (tfa_timing_enable): a ring of event triples
  static constexpr int kMaxTimed = 64;
  bool timing = false;
  int timed = 0;
  cudaEvent_t ev[kMaxTimed][3] = {};
  ~tfa_ctx() {
    for (auto& t : ev)
      for (auto& e : t)
        if (e) cudaEventDestroy(e);
  }
};

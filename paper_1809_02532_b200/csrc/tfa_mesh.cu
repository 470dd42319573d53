// tfa_mesh.cu — step a1: mesh connectivity, geometry, stencil, BSR pattern, boundary-face list and cell
// reordering, built on the device (PAPER.md L74 stencil, L230 cell->faces loop, L260 boundary faces, L276-319
// Listing 1 pattern).
//
// Everything derived from (cell_nodes, cell_xy) is produced by the kernels below under the
// canonical rules of DESIGN.md (readings S9-S11), so that the result is bit-exact and independent
// of thread scheduling: faces are numbered by sorted (lo node, hi node) key, L is the smaller cell
// id, stencil and BSR columns are ascending.  Sorting and prefix sums use CUB device primitives
// (library steps); the rest is hand-written.
//
// Cells are triangles or convex quadrilaterals.  Every per-cell table has F slots per cell,
// F = 3 for a pure triangle mesh and 4 as soon as one cell is a quadrilateral; a triangle of a mixed mesh has
// node -1 in its fourth slot.  These are once-per-mesh kernels: F is a run-time argument here (the per-step
// kernels are compiled for F = 3 and F = 4).
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include <atomic>
#include <vector>

#include "tfa_common.cuh"

namespace tfa {

thread_local std::string g_last_error;
int set_error(int code, const std::string& msg) {
  g_last_error = msg;
  return code;
}
// Every (re)built mesh gets a stamp no other mesh of the process ever had: a context's per-mesh workspace keys
// on it, so a new mesh allocated at the address of a destroyed one is never mistaken for it.
uint64_t next_mesh_uid() {
  static std::atomic<uint64_t> counter{0};
  return ++counter;
}

namespace {

enum MeshErr : int {
  ERR_CW = 1,          // non-positive area / not convex
  ERR_REPEAT = 2,      // a cell repeats a node id
  ERR_RANGE = 4,       // node id out of range
  ERR_NONMANIFOLD = 8, // node pair shared by > 2 cells
  ERR_SELFNBR = 16,    // a cell is its own neighbour
  ERR_DUPNBR = 32,     // two faces of a cell lead to the same neighbour
  ERR_STENCIL = 64,    // stencil candidate list overflow
  ERR_PERM = 128       // permutation is not a bijection
};

constexpr int TPB = 256;
constexpr int MAXCAND = 192;   // sum of the node degrees of a cell's corners (Delaunay: ~18, max seen 30; quads: 16)
constexpr int MAXF = 4;

__device__ __forceinline__ int cell_nv(const int32_t* __restrict__ cell_nodes, int F, int64_t i) {
  return (F == 4 && cell_nodes[4 * i + 3] >= 0) ? 4 : 3;
}

// ---- geometry of each cell from its own corner coordinates ----
__global__ void k_cell_geom(int64_t nc, int64_t nn, int F, const int32_t* __restrict__ cell_nodes,
                            const double* __restrict__ cell_xy, double* __restrict__ cen,
                            double* __restrict__ vol, double* __restrict__ olen, double* __restrict__ onrm,
                            double* __restrict__ ooff, int32_t* err) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  const int nv = cell_nv(cell_nodes, F, i);
  const double* X = cell_xy + 2 * F * i;
  double x[MAXF], y[MAXF];
  for (int k = 0; k < MAXF; ++k) {
    x[k] = k < nv ? X[2 * k] : 0.0;
    y[k] = k < nv ? X[2 * k + 1] : 0.0;
  }
  double cx, cy, area;
  if (nv == 3) {
    cx = (x[0] + x[1] + x[2]) / 3.0;
    cy = (y[0] + y[1] + y[2]) / 3.0;
    area = 0.5 * ((x[1] - x[0]) * (y[2] - y[0]) - (y[1] - y[0]) * (x[2] - x[0]));
    if (!(area > 0.0)) { atomicOr(err, ERR_CW); atomicMin(err + 1, (int32_t)i); }
  } else {
    // quadrilateral: the two triangles on the diagonal (0, 2), offsets from corner 0; the area centroid is the
    // area-weighted mean of the triangles' centroids
    const double ax = x[1] - x[0], ay = y[1] - y[0], bx = x[2] - x[0], by = y[2] - y[0];
    const double gx = x[3] - x[0], gy = y[3] - y[0];
    const double t1 = ax * by - ay * bx, t2 = bx * gy - by * gx;   // twice the two areas
    area = 0.5 * (t1 + t2);
    cx = x[0] + (t1 * (ax + bx) + t2 * (bx + gx)) / (3.0 * (t1 + t2));
    cy = y[0] + (t1 * (ay + by) + t2 * (by + gy)) / (3.0 * (t1 + t2));
    bool convex = area > 0.0;
    for (int k = 0; k < 4; ++k) {   // every corner turns left
      const int k1 = (k + 1) & 3, k2 = (k + 2) & 3;
      convex &= (x[k1] - x[k]) * (y[k2] - y[k1]) - (y[k1] - y[k]) * (x[k2] - x[k1]) > 0.0;
    }
    if (!convex) { atomicOr(err, ERR_CW); atomicMin(err + 1, (int32_t)i); }
  }
  cen[2 * i] = cx;
  cen[2 * i + 1] = cy;
  vol[i] = area;
  for (int k = 0; k < F; ++k) {
    if (k < nv) {
      const int k1 = k + 1 == nv ? 0 : k + 1;
      const double dx = x[k1] - x[k], dy = y[k1] - y[k];
      const double len = sqrt(dx * dx + dy * dy);
      olen[F * i + k] = len;
      onrm[2 * (F * i + k)] = dy / len;
      onrm[2 * (F * i + k) + 1] = -dx / len;
      ooff[2 * (F * i + k)] = 0.5 * (x[k] + x[k1]) - cx;
      ooff[2 * (F * i + k) + 1] = 0.5 * (y[k] + y[k1]) - cy;
    } else {   // the missing fourth edge of a triangle: a face of zero length
      olen[F * i + k] = 0.0;
      onrm[2 * (F * i + k)] = 1.0;
      onrm[2 * (F * i + k) + 1] = 0.0;
      ooff[2 * (F * i + k)] = 0.0;
      ooff[2 * (F * i + k) + 1] = 0.0;
    }
  }
  bool repeat = false, range = false;
  for (int a = 0; a < nv; ++a) {
    const int32_t va = cell_nodes[F * i + a];
    range |= va < 0 || va >= nn;
    for (int b = a + 1; b < nv; ++b) repeat |= va == cell_nodes[F * i + b];
  }
  if (repeat) { atomicOr(err, ERR_REPEAT); atomicMin(err + 1, (int32_t)i); }
  if (range) atomicOr(err, ERR_RANGE);
}

__global__ void k_gather_xy(int64_t nslots, int64_t nn, const int32_t* __restrict__ cell_nodes,
                            const double* __restrict__ node_xy, double* __restrict__ cell_xy, int32_t* err) {
  int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (q >= nslots) return;
  int32_t v = cell_nodes[q];
  if (v < 0) {   // empty fourth slot of a triangle (a negative id in a real slot is caught by k_cell_geom)
    cell_xy[2 * q] = cell_xy[2 * q + 1] = 0.0;
    return;
  }
  if (v >= nn) { atomicOr(err, ERR_RANGE); v = 0; }
  cell_xy[2 * q] = node_xy[2 * (int64_t)v];
  cell_xy[2 * q + 1] = node_xy[2 * (int64_t)v + 1];
}

// ---- faces: unique (lo, hi) node pairs, numbered in sorted key order (S10) ----
// slot e = F * cell + k; the empty slot of a triangle gets the key nn * nn, above every real key
__global__ void k_edge_keys(int64_t nc, int64_t nn, int F, const int32_t* __restrict__ cell_nodes,
                            uint64_t* __restrict__ keys, int32_t* __restrict__ vals) {
  int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (e >= F * nc) return;
  const int64_t c = e / F;
  const int k = (int)(e - c * F);
  const int nv = cell_nv(cell_nodes, F, c);
  vals[e] = (int32_t)e;
  if (k >= nv) { keys[e] = (uint64_t)nn * (uint64_t)nn; return; }
  const int32_t a = cell_nodes[F * c + k], b = cell_nodes[F * c + (k + 1 == nv ? 0 : k + 1)];
  const uint64_t lo = (uint64_t)min(a, b), hi = (uint64_t)max(a, b);
  keys[e] = lo * (uint64_t)nn + hi;
}

__global__ void k_face_heads(int64_t ne, uint64_t sentinel, const uint64_t* __restrict__ keys,
                             int32_t* __restrict__ head, int32_t* err) {
  int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (e >= ne) return;
  const bool real = keys[e] != sentinel;
  head[e] = (real && (e == 0 || keys[e] != keys[e - 1])) ? 1 : 0;
  if (real && e >= 2 && keys[e] == keys[e - 2]) atomicOr(err, ERR_NONMANIFOLD);
}

__global__ void k_faces(int64_t ne, int64_t nn, int F, uint64_t sentinel, const uint64_t* __restrict__ keys,
                        const int32_t* __restrict__ vals, const int32_t* __restrict__ fid,
                        int32_t* __restrict__ face_nodes, int32_t* __restrict__ face_cells,
                        int32_t* __restrict__ cell_faces, int32_t* err) {
  int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (e >= ne) return;
  const uint64_t key = keys[e];
  const int32_t v = vals[e];
  if (key == sentinel) { cell_faces[v] = -1; return; }
  const int32_t f = fid[e] - 1;
  const int32_t c = v / F;
  cell_faces[v] = f;
  const bool is_head = (e == 0 || keys[e - 1] != key);
  if (is_head) {
    face_nodes[2 * (int64_t)f] = (int32_t)(key / (uint64_t)nn);
    face_nodes[2 * (int64_t)f + 1] = (int32_t)(key % (uint64_t)nn);
    face_cells[2 * (int64_t)f] = c;   // stable sort of ascending values: the smaller cell id comes first
    if (!(e + 1 < ne && keys[e + 1] == key)) face_cells[2 * (int64_t)f + 1] = -1;
  } else {
    face_cells[2 * (int64_t)f + 1] = c;
    if (vals[e - 1] / F == c) atomicOr(err, ERR_SELFNBR);
  }
}

__global__ void k_cell_nbr(int64_t nc, int F, const int32_t* __restrict__ cell_faces,
                           const int32_t* __restrict__ face_cells, int32_t* __restrict__ cell_nbr,
                           int32_t* __restrict__ rowcnt, int32_t* err) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  int32_t nb[MAXF];
  int cnt = 1;
  for (int k = 0; k < F; ++k) {
    const int64_t f = cell_faces[F * i + k];
    nb[k] = -1;
    if (f >= 0) {
      const int32_t L = face_cells[2 * f], R = face_cells[2 * f + 1];
      nb[k] = (L == (int32_t)i) ? R : L;
    }
    cell_nbr[F * i + k] = nb[k];
    cnt += nb[k] >= 0;
  }
  bool dup = false;
  for (int a = 0; a < F; ++a)
    for (int b = a + 1; b < F; ++b) dup |= nb[a] >= 0 && nb[a] == nb[b];
  if (dup) atomicOr(err, ERR_DUPNBR);
  rowcnt[i] = cnt;
}

// BSR columns: self + face neighbours, ascending (Listing 1's allNonZero = nbEqs x blocks per row)
__global__ void k_bsr_cols(int64_t nc, int F, const int32_t* __restrict__ cell_nbr,
                           const int32_t* __restrict__ rowptr, int32_t* __restrict__ col) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  int32_t c[MAXF + 1];
  c[0] = (int32_t)i;
  for (int k = 0; k < F; ++k) c[1 + k] = cell_nbr[F * i + k];
  const int32_t base = rowptr[i];
  for (int a = 0; a <= F; ++a) {
    if (c[a] < 0) continue;
    int rank = 0;
    for (int b = 0; b <= F; ++b) rank += (c[b] >= 0 && c[b] < c[a]);
    col[base + rank] = c[a];
  }
}

// ---- vertex-neighbour stencil (L74) ----
// (node, cell) pairs; the empty slot of a triangle gets the key nn, above every real node id
__global__ void k_node_pairs(int64_t nslots, int64_t nn, int F, const int32_t* __restrict__ cell_nodes,
                             uint32_t* __restrict__ keys, int32_t* __restrict__ vals, int32_t* __restrict__ node_cnt) {
  int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (e >= nslots) return;
  const int32_t v = cell_nodes[e];
  vals[e] = (int32_t)(e / F);
  if (v < 0) { keys[e] = (uint32_t)nn; return; }
  keys[e] = (uint32_t)v;
  atomicAdd(node_cnt + v, 1);   // integer count: the result does not depend on the order
}

// candidates = union of the cell lists of the cell's corners, sorted, unique, without self
__device__ int stencil_candidates(int64_t i, int F, const int32_t* __restrict__ cell_nodes,
                                  const int32_t* __restrict__ node_ptr, const int32_t* __restrict__ node_cells,
                                  int32_t* cand, bool* overflow) {
  int n = 0;
  const int nv = cell_nv(cell_nodes, F, i);
  for (int k = 0; k < nv; ++k) {
    int32_t v = cell_nodes[F * i + k];
    for (int32_t q = node_ptr[v]; q < node_ptr[v + 1]; ++q) {
      int32_t j = node_cells[q];
      if (j == (int32_t)i) continue;
      if (n >= MAXCAND) { *overflow = true; return n; }
      int p = n++;   // insertion sort keeps the list ascending
      while (p > 0 && cand[p - 1] > j) { cand[p] = cand[p - 1]; --p; }
      cand[p] = j;
    }
  }
  int u = 0;
  for (int p = 0; p < n; ++p)
    if (p == 0 || cand[p] != cand[p - 1]) cand[u++] = cand[p];
  return u;
}

__global__ void k_stencil_count(int64_t nc, int F, const int32_t* __restrict__ cell_nodes,
                                const int32_t* __restrict__ node_ptr, const int32_t* __restrict__ node_cells,
                                int32_t* __restrict__ cnt, int32_t* err) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  int32_t cand[MAXCAND];
  bool ovf = false;
  cnt[i] = stencil_candidates(i, F, cell_nodes, node_ptr, node_cells, cand, &ovf);
  if (ovf) atomicOr(err, ERR_STENCIL);
}

__global__ void k_stencil_fill(int64_t nc, int F, const int32_t* __restrict__ cell_nodes,
                               const int32_t* __restrict__ node_ptr, const int32_t* __restrict__ node_cells,
                               const int32_t* __restrict__ st_ptr, const double* __restrict__ cell_xy,
                               const double* __restrict__ cen, int32_t* __restrict__ st_idx,
                               double* __restrict__ st_d) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  int32_t cand[MAXCAND];
  bool ovf = false;
  const int n = stencil_candidates(i, F, cell_nodes, node_ptr, node_cells, cand, &ovf);
  const int32_t base = st_ptr[i];
  const int nvi = cell_nv(cell_nodes, F, i);
  for (int p = 0; p < n; ++p) {
    const int64_t j = cand[p];
    const int nvj = cell_nv(cell_nodes, F, j);
    // displacement through the smallest shared node id (S9, S22): periodic-safe, no min-image
    int32_t v = INT32_MAX;
    int ai = 0, bj = 0;
    for (int a = 0; a < nvi; ++a)
      for (int b = 0; b < nvj; ++b) {
        const int32_t na = cell_nodes[F * i + a], nj = cell_nodes[F * j + b];
        if (na == nj && nj < v) { v = nj; ai = a; bj = b; }
      }
    double dx = (cen[2 * j] - cell_xy[2 * (F * j + bj)]) - (cen[2 * i] - cell_xy[2 * (F * i + ai)]);
    double dy = (cen[2 * j + 1] - cell_xy[2 * (F * j + bj) + 1]) - (cen[2 * i + 1] - cell_xy[2 * (F * i + ai) + 1]);
    st_idx[base + p] = (int32_t)j;
    st_d[2 * (int64_t)(base + p)] = dx;
    st_d[2 * (int64_t)(base + p) + 1] = dy;
  }
}

// ---- where cell i writes: its diagonal block (i,i) and, for each local face k with neighbour j,
// the block (j,i) of the NEIGHBOUR's row ("mirror" block); -1 where there is none ----
__global__ void k_blkmap(int64_t nc, int F, int BS, const int32_t* __restrict__ cell_nbr,
                         const int32_t* __restrict__ rowptr, int32_t* __restrict__ blkmap) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  const int32_t me = (int32_t)i;
  int32_t n[MAXF];
  int rank = 0;
  for (int k = 0; k < F; ++k) {
    n[k] = cell_nbr[F * i + k];
    rank += (n[k] >= 0 && n[k] < me);
  }
  for (int q = 0; q < BS; ++q) blkmap[BS * i + q] = -1;
  blkmap[BS * i] = rowptr[i] + rank;
  for (int k = 0; k < F; ++k) {
    const int64_t j = n[k];
    if (j < 0) continue;
    int r = (int32_t)j < me;   // the neighbour's own diagonal column
    for (int q = 0; q < F; ++q) {
      const int32_t c = cell_nbr[F * j + q];
      r += (c >= 0 && c < me);
    }
    blkmap[BS * i + 1 + k] = rowptr[j] + r;
  }
}

// ---- the block map of the packed Jacobian (tfa.h TFA_PACKED_BLOCK): diagonal blocks are an array of their own
// indexed by the cell; the off-diagonal blocks keep their BSR order with the diagonal ones taken out, so block b of
// row j sits in slot b - j - (b lies after row j's diagonal block) ----
__global__ void k_pblkmap(int64_t nc, int F, int BS, const int32_t* __restrict__ cell_nbr,
                          const int32_t* __restrict__ blkmap, int32_t* __restrict__ pblkmap) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  for (int q = 0; q < BS; ++q) pblkmap[BS * i + q] = -1;
  pblkmap[BS * i] = (int32_t)i;
  for (int k = 0; k < F; ++k) {
    const int32_t mb = blkmap[BS * i + 1 + k];
    if (mb < 0) continue;
    const int64_t j = cell_nbr[F * i + k];
    pblkmap[BS * i + 1 + k] = mb - (int32_t)j - (mb > blkmap[BS * j] ? 1 : 0);
  }
}

// ---- packed neighbour of each local face (tfa_common.cuh): interior 4 * neighbour + the face's local index there;
// boundary -1 - (4 * boundary-face index + tag); a triangle's fourth slot -1 ----
__global__ void k_nbr_face(int64_t nc, int F, const int32_t* __restrict__ cell_nbr,
                           const int32_t* __restrict__ cell_faces, const int32_t* __restrict__ bface_of,
                           const int32_t* __restrict__ bc_tag, int32_t* __restrict__ nbrf) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  for (int k = 0; k < F; ++k) {
    const int64_t j = cell_nbr[F * i + k];
    const int32_t f = cell_faces[F * i + k];
    int32_t packed = -1;
    if (j >= 0) {
      int kj = 0;
      for (int q = 0; q < F; ++q)
        if (cell_faces[F * j + q] == f) kj = q;
      packed = (int32_t)(4 * j + kj);
    } else if (f >= 0) {
      const int32_t b = bface_of[f];
      packed = -1 - (4 * b + bc_tag[b]);
    }
    nbrf[F * i + k] = packed;
  }
}

// ---- per-cell geometry record, face normals pointing out of the cell (tfa_common.cuh) ----
__global__ void k_cgeo(int64_t nc, int F, const int32_t* __restrict__ cell_nbr, const int32_t* __restrict__ cell_faces,
                       const double* __restrict__ vol, const double* __restrict__ olen,
                       const double* __restrict__ onrm, const double* __restrict__ ooff,
                       double* __restrict__ cgeo, double* __restrict__ ggeo) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  double* g = cgeo + 8 * F * i;
  for (int k = 0; k < F; ++k) {
    const int64_t j = cell_nbr[F * i + k];
    const int32_t f = cell_faces[F * i + k];
    int kj = 0;
    if (j >= 0)
      for (int q = 0; q < F; ++q)
        if (cell_faces[F * j + q] == f) kj = q;
    const bool own_is_L = (j < 0) || (i < j);
    const int64_t eL = own_is_L ? F * i + k : F * j + kj;
    // the face's normal is its L cell's (S10); seen from the R cell it is exactly minus that
    g[8 * k + 0] = own_is_L ? onrm[2 * eL] : -onrm[2 * eL];
    g[8 * k + 1] = own_is_L ? onrm[2 * eL + 1] : -onrm[2 * eL + 1];
    g[8 * k + 2] = olen[eL];
    g[8 * k + 3] = ooff[2 * (F * i + k)];
    g[8 * k + 4] = ooff[2 * (F * i + k) + 1];
    // boundary face: the own-side values again
    g[8 * k + 5] = j >= 0 ? ooff[2 * (F * j + kj)] : ooff[2 * (F * i + k)];
    g[8 * k + 6] = j >= 0 ? ooff[2 * (F * j + kj) + 1] : ooff[2 * (F * i + k) + 1];
    g[8 * k + 7] = 0.0;
  }
  g[7] = vol[i];
  g[15] = sqrt(vol[i]);
  double* gg = ggeo + (2 * F + 2) * i;
  for (int k = 0; k < F; ++k) {
    gg[2 * k] = g[8 * k + 3];
    gg[2 * k + 1] = g[8 * k + 4];
  }
  gg[2 * F] = g[15];
  gg[2 * F + 1] = 0.0;
}

// ---- boundary faces in ascending face id (L260) ----
__global__ void k_bface_flag(int64_t nf, const int32_t* __restrict__ face_cells, int32_t* __restrict__ flag) {
  int64_t f = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (f < nf) flag[f] = face_cells[2 * f + 1] < 0;
}
__global__ void k_bface_list(int64_t nf, const int32_t* __restrict__ flag, const int32_t* __restrict__ scan,
                             int32_t* __restrict__ bface_of, int32_t* __restrict__ bfaces) {
  int64_t f = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (f >= nf) return;
  const int32_t b = flag[f] ? scan[f] : -1;   // scan = exclusive prefix sum of the flags
  bface_of[f] = b;
  if (b >= 0) bfaces[b] = (int32_t)f;
}

// ---- reverse Cuthill-McKee, one CTA, level-synchronous, deterministic (S11) ----
// Equivalent to the serial queue algorithm: a cell's parent is the earliest-ordered frontier
// cell adjacent to it; children of one parent are appended sorted by (degree, id).
constexpr int RCM_T = 1024;
__global__ void __launch_bounds__(RCM_T) k_rcm(int32_t nc, int F, const int32_t* __restrict__ nbr,
                                              int32_t* __restrict__ order, int32_t* __restrict__ pos,
                                              int32_t* __restrict__ parent) {
  __shared__ int32_t s_scan[RCM_T];
  __shared__ unsigned long long s_best;
  __shared__ int32_t s_lb, s_le, s_total;
  const int t = threadIdx.x;
  auto degree = [&](int32_t c) {
    int d = 0;
    for (int k = 0; k < F; ++k) d += nbr[F * c + k] >= 0;
    return d;
  };
  for (int32_t c = t; c < nc; c += RCM_T) { pos[c] = -1; parent[c] = INT32_MAX; }
  if (t == 0) { s_lb = 0; s_le = 0; }
  __syncthreads();
  while (true) {
    int32_t placed = s_le;
    if (placed >= nc) break;
    // start of a new component: unvisited cell with minimum (degree, id)
    if (t == 0) s_best = ~0ull;
    __syncthreads();
    unsigned long long best = ~0ull;
    for (int32_t c = t; c < nc; c += RCM_T)
      if (pos[c] < 0) {
        unsigned long long key = ((unsigned long long)degree(c) << 32) | (unsigned)c;
        best = key < best ? key : best;
      }
    atomicMin(&s_best, best);
    __syncthreads();
    if (t == 0) {
      int32_t c = (int32_t)(s_best & 0xffffffffu);
      order[placed] = c;
      pos[c] = placed;
      s_lb = placed;
      s_le = placed + 1;
    }
    __syncthreads();
    // breadth-first levels
    while (true) {
      const int32_t lb = s_lb, le = s_le;
      if (lb == le) break;
      // 1. every unvisited neighbour of the frontier records its earliest parent
      for (int32_t p = lb + t; p < le; p += RCM_T) {
        const int32_t v = order[p];
        for (int k = 0; k < F; ++k) {
          const int32_t w = nbr[F * v + k];
          if (w >= 0 && pos[w] < 0) atomicMin(parent + w, p);
        }
      }
      __syncthreads();
      // 2. children per frontier cell, exclusive scan over the frontier in chunks of RCM_T
      int32_t running = 0;
      for (int32_t p0 = lb; p0 < le; p0 += RCM_T) {
        const int32_t p = p0 + t;
        int32_t ch[MAXF];
        int n = 0;
        if (p < le) {
          const int32_t v = order[p];
          for (int k = 0; k < F; ++k) {
            const int32_t w = nbr[F * v + k];
            if (w >= 0 && pos[w] < 0 && parent[w] == p) ch[n++] = w;
          }
        }
        s_scan[t] = n;
        __syncthreads();
        for (int off = 1; off < RCM_T; off <<= 1) {   // Hillis-Steele inclusive scan
          int32_t x = t >= off ? s_scan[t - off] : 0;
          __syncthreads();
          s_scan[t] += x;
          __syncthreads();
        }
        const int32_t excl = s_scan[t] - n;
        if (t == RCM_T - 1) s_total = s_scan[t];
        // sort the <= F children by (degree, id) and append
        for (int a = 1; a < n; ++a) {
          int32_t w = ch[a];
          int dw = degree(w);
          int b = a;
          while (b > 0 && (degree(ch[b - 1]) > dw || (degree(ch[b - 1]) == dw && ch[b - 1] > w))) {
            ch[b] = ch[b - 1];
            --b;
          }
          ch[b] = w;
        }
        for (int a = 0; a < n; ++a) order[le + running + excl + a] = ch[a];
        __syncthreads();
        running += s_total;
        __syncthreads();
      }
      // 3. publish positions of the new level (after all parent tests of this level are done)
      for (int32_t q = le + t; q < le + running; q += RCM_T) pos[order[q]] = q;
      __syncthreads();
      if (t == 0) { s_lb = le; s_le = le + running; }
      __syncthreads();
    }
  }
}

// ---- Z-order (Morton) curve through the cell centroids: an ordering whose consecutive cells form compact patches,
// so that the cells of one CTA share most of their stencils (tfa_mesh_reorder kind 3) ----
__device__ __forceinline__ unsigned long long ordered_bits(double x) {   // monotone map double -> uint64
  const unsigned long long u = (unsigned long long)__double_as_longlong(x);
  return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}
__device__ __forceinline__ double from_ordered_bits(unsigned long long u) {
  return __longlong_as_double((long long)((u >> 63) ? (u & 0x7fffffffffffffffull) : ~u));
}
__global__ void k_bbox(int64_t nc, const double* __restrict__ cen, unsigned long long* __restrict__ box) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  atomicMin(box + 0, ordered_bits(cen[2 * i]));
  atomicMax(box + 1, ordered_bits(cen[2 * i]));
  atomicMin(box + 2, ordered_bits(cen[2 * i + 1]));
  atomicMax(box + 3, ordered_bits(cen[2 * i + 1]));
}
__device__ __forceinline__ unsigned spread16(unsigned v) {   // abcd -> 0a0b0c0d
  v = (v | (v << 8)) & 0x00ff00ffu;
  v = (v | (v << 4)) & 0x0f0f0f0fu;
  v = (v | (v << 2)) & 0x33333333u;
  v = (v | (v << 1)) & 0x55555555u;
  return v;
}
__global__ void k_morton_keys(int64_t nc, const double* __restrict__ cen, const unsigned long long* __restrict__ box,
                              uint64_t* __restrict__ keys, int32_t* __restrict__ vals) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  const double x0 = from_ordered_bits(box[0]), x1 = from_ordered_bits(box[1]);
  const double y0 = from_ordered_bits(box[2]), y1 = from_ordered_bits(box[3]);
  const double sx = x1 > x0 ? 65535.0 / (x1 - x0) : 0.0, sy = y1 > y0 ? 65535.0 / (y1 - y0) : 0.0;
  const unsigned qx = (unsigned)min(65535.0, max(0.0, (cen[2 * i] - x0) * sx));
  const unsigned qy = (unsigned)min(65535.0, max(0.0, (cen[2 * i + 1] - y0) * sy));
  // ties (cells in one quantisation box) are broken by the cell id: the order is unique
  keys[i] = ((uint64_t)(spread16(qx) | (spread16(qy) << 1)) << 32) | (uint64_t)(uint32_t)i;
  vals[i] = (int32_t)i;
}

__global__ void k_reverse(int32_t n, const int32_t* __restrict__ in, int32_t* __restrict__ out) {
  int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = in[n - 1 - i];
}

__global__ void k_check_perm(int64_t nc, const int32_t* __restrict__ p, int32_t* __restrict__ hit, int32_t* err) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  int32_t v = p[i];
  if (v < 0 || v >= nc) { atomicOr(err, ERR_PERM); return; }
  if (atomicAdd(hit + v, 1) != 0) atomicOr(err, ERR_PERM);
}

__global__ void k_permute_cells(int64_t nc, int F, const int32_t* __restrict__ p, const int32_t* __restrict__ cn_in,
                                const double* __restrict__ cx_in, const int32_t* __restrict__ perm_in,
                                int32_t* __restrict__ cn, double* __restrict__ cx, int32_t* __restrict__ perm) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  const int64_t o = p[i];
  for (int k = 0; k < F; ++k) cn[F * i + k] = cn_in[F * o + k];
  for (int k = 0; k < 2 * F; ++k) cx[2 * F * i + k] = cx_in[2 * F * o + k];
  perm[i] = perm_in[o];
}

__global__ void k_iota(int64_t n, int32_t* p) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) p[i] = (int32_t)i;
}

__global__ void k_face_geom_out(int64_t nf, int F, const int32_t* __restrict__ face_cells,
                                const int32_t* __restrict__ cell_faces, const double* __restrict__ cgeo,
                                double* __restrict__ out) {
  int64_t f = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (f >= nf) return;
  const int64_t L = face_cells[2 * f];
  int k = 0;
  for (int q = 0; q < F; ++q)
    if (cell_faces[F * L + q] == (int32_t)f) k = q;
  out[3 * f] = cgeo[8 * F * L + 8 * k];
  out[3 * f + 1] = cgeo[8 * F * L + 8 * k + 1];
  out[3 * f + 2] = cgeo[8 * F * L + 8 * k + 2];
}

__global__ void k_volume_out(int64_t nc, int F, const double* __restrict__ cgeo, double* __restrict__ out) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < nc) out[i] = cgeo[8 * F * i + 7];
}

std::string describe(int bits, int cell) {
  std::string s;
  if (bits & ERR_CW)
    s += "cell " + std::to_string(cell) + " is not counter-clockwise (area <= 0) or not a convex quadrilateral; ";
  if (bits & ERR_REPEAT) s += "a cell repeats a node id (periodic direction too narrow); ";
  if (bits & ERR_RANGE) s += "node id out of range; ";
  if (bits & ERR_NONMANIFOLD) s += "a node pair is shared by more than 2 cells; ";
  if (bits & ERR_SELFNBR) s += "a cell is its own neighbour (periodic direction too narrow); ";
  if (bits & ERR_DUPNBR) s += "two faces of a cell lead to the same neighbour (periodic direction too narrow); ";
  if (bits & ERR_STENCIL) s += "vertex stencil exceeds the internal candidate limit (192 cells around a cell's corners); ";
  if (bits & ERR_PERM) s += "permutation is not a bijection; ";
  return s;
}

int check_err(DevBuf<int32_t>& err, cudaStream_t st) {
  int32_t h[2];
  TFA_CUDA(cudaMemcpyAsync(h, err.p, sizeof(h), cudaMemcpyDeviceToHost, st));
  TFA_CUDA(cudaStreamSynchronize(st));
  if (h[0]) return set_error(TFA_EMESH, describe(h[0], h[1]));
  return 0;
}

// out[0..n] : out[i] = sum_{q<i} in[q]; out[n] = total
int exclusive_scan_with_total(const DevBuf<int32_t>& in, int64_t n, DevBuf<int32_t>& out, int64_t* total,
                              cudaStream_t st) {
  size_t tmp_bytes = 0;
  cub::DeviceScan::InclusiveSum(nullptr, tmp_bytes, in.p, out.p + 1, (int)n, st);
  DevBuf<char> tmp;
  TFA_CUDA(tmp.alloc((int64_t)tmp_bytes));
  TFA_CUDA(cudaMemsetAsync(out.p, 0, sizeof(int32_t), st));
  TFA_CUDA(cub::DeviceScan::InclusiveSum(tmp.p, tmp_bytes, in.p, out.p + 1, (int)n, st));
  int32_t h = 0;
  TFA_CUDA(cudaMemcpyAsync(&h, out.p + n, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  TFA_CUDA(cudaStreamSynchronize(st));
  *total = (int64_t)h;
  return 0;
}

int bits_for(uint64_t max_value) {
  int b = 1;
  while (b < 64 && (max_value >> b)) ++b;
  return b;
}

}  // namespace

// (re)write the packed neighbour table from the current boundary tags
int refresh_nbrf(tfa_mesh& m, cudaStream_t st) {
  if (m.nc == 0) return 0;
  k_nbr_face<<<cdiv(m.nc, TPB), TPB, 0, st>>>(m.nc, m.F, m.cell_nbr.p, m.cell_faces.p, m.bface_of.p, m.bc_tag.p,
                                             m.nbrf.p);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

// Build every derived array of the mesh from (cell_nodes, cell_xy).
int build_mesh(tfa_mesh& m, cudaStream_t st) {
  const int F = m.F, BS = blk_stride(F);
  const int64_t nc = m.nc, nn = m.nn, ne = (int64_t)F * nc;
  if (ne >= (int64_t)INT32_MAX) return set_error(TFA_EINVAL, "mesh too large for 32-bit face-edge ids");
  DevBuf<int32_t> err;
  TFA_CUDA(err.alloc(2));
  {
    int32_t h[2] = {0, INT32_MAX};
    TFA_CUDA(cudaMemcpyAsync(err.p, h, sizeof(h), cudaMemcpyHostToDevice, st));
  }
  DevBuf<double> vol, olen, onrm, ooff;
  TFA_CUDA(m.cen.alloc(2 * nc));
  TFA_CUDA(vol.alloc(nc));
  TFA_CUDA(olen.alloc(ne));
  TFA_CUDA(onrm.alloc(2 * ne));
  TFA_CUDA(ooff.alloc(2 * ne));
  if (nc == 0) {
    m.nf = m.nnzb = m.nst = m.nb = 0;
    m.has_ghost = false;
    TFA_CUDA(m.st_ptr.alloc(1));
    TFA_CUDA(m.bsr_rowptr.alloc(1));
    TFA_CUDA(cudaMemsetAsync(m.st_ptr.p, 0, 4, st));
    TFA_CUDA(cudaMemsetAsync(m.bsr_rowptr.p, 0, 4, st));
    TFA_CUDA(m.face_nodes.alloc(0)); TFA_CUDA(m.face_cells.alloc(0)); TFA_CUDA(m.cell_faces.alloc(0));
    TFA_CUDA(m.cell_nbr.alloc(0)); TFA_CUDA(m.nbrf.alloc(0)); TFA_CUDA(m.st_idx.alloc(0)); TFA_CUDA(m.st_d.alloc(0));
    TFA_CUDA(m.bsr_col.alloc(0)); TFA_CUDA(m.cgeo.alloc(0)); TFA_CUDA(m.blkmap.alloc(0)); TFA_CUDA(m.pblkmap.alloc(0));
    TFA_CUDA(m.ggeo.alloc(0));
    TFA_CUDA(m.bfaces.alloc(0)); TFA_CUDA(m.bface_of.alloc(0)); TFA_CUDA(m.bc_tag.alloc(0));
    m.uid = next_mesh_uid();
    return 0;
  }
  k_cell_geom<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, nn, F, m.cell_nodes.p, m.cell_xy.p, m.cen.p, vol.p, olen.p, onrm.p,
                                            ooff.p, err.p);
  TFA_TRY(check_err(err, st));

  // faces
  DevBuf<uint64_t> keys, keys_s;
  DevBuf<int32_t> vals, vals_s, head, fid;
  TFA_CUDA(keys.alloc(ne)); TFA_CUDA(keys_s.alloc(ne));
  TFA_CUDA(vals.alloc(ne)); TFA_CUDA(vals_s.alloc(ne));
  TFA_CUDA(head.alloc(ne)); TFA_CUDA(fid.alloc(ne));
  const uint64_t sentinel = (uint64_t)nn * (uint64_t)nn;
  k_edge_keys<<<cdiv(ne, TPB), TPB, 0, st>>>(nc, nn, F, m.cell_nodes.p, keys.p, vals.p);
  {
    const int end_bit = bits_for(sentinel);
    size_t tmp_bytes = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys.p, keys_s.p, vals.p, vals_s.p, (int)ne, 0, end_bit, st);
    DevBuf<char> tmp;
    TFA_CUDA(tmp.alloc((int64_t)tmp_bytes));
    TFA_CUDA(cub::DeviceRadixSort::SortPairs(tmp.p, tmp_bytes, keys.p, keys_s.p, vals.p, vals_s.p, (int)ne, 0,
                                             end_bit, st));
    TFA_CUDA(cudaStreamSynchronize(st));
  }
  k_face_heads<<<cdiv(ne, TPB), TPB, 0, st>>>(ne, sentinel, keys_s.p, head.p, err.p);
  {
    size_t tmp_bytes = 0;
    cub::DeviceScan::InclusiveSum(nullptr, tmp_bytes, head.p, fid.p, (int)ne, st);
    DevBuf<char> tmp;
    TFA_CUDA(tmp.alloc((int64_t)tmp_bytes));
    TFA_CUDA(cub::DeviceScan::InclusiveSum(tmp.p, tmp_bytes, head.p, fid.p, (int)ne, st));
    int32_t nf = 0;
    TFA_CUDA(cudaMemcpyAsync(&nf, fid.p + ne - 1, 4, cudaMemcpyDeviceToHost, st));
    TFA_CUDA(cudaStreamSynchronize(st));
    m.nf = nf;
  }
  TFA_TRY(check_err(err, st));
  TFA_CUDA(m.face_nodes.alloc(2 * m.nf));
  TFA_CUDA(m.face_cells.alloc(2 * m.nf));
  TFA_CUDA(m.cell_faces.alloc(ne));
  TFA_CUDA(m.cell_nbr.alloc(ne));
  k_faces<<<cdiv(ne, TPB), TPB, 0, st>>>(ne, nn, F, sentinel, keys_s.p, vals_s.p, fid.p, m.face_nodes.p,
                                        m.face_cells.p, m.cell_faces.p, err.p);
  DevBuf<int32_t> cnt;
  TFA_CUDA(cnt.alloc(nc));
  k_cell_nbr<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, F, m.cell_faces.p, m.face_cells.p, m.cell_nbr.p, cnt.p, err.p);
  TFA_TRY(check_err(err, st));

  // BSR pattern
  TFA_CUDA(m.bsr_rowptr.alloc(nc + 1));
  TFA_TRY(exclusive_scan_with_total(cnt, nc, m.bsr_rowptr, &m.nnzb, st));
  TFA_CUDA(m.bsr_col.alloc(m.nnzb));
  k_bsr_cols<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, F, m.cell_nbr.p, m.bsr_rowptr.p, m.bsr_col.p);
  TFA_CUDA(m.blkmap.alloc(BS * nc));
  k_blkmap<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, F, BS, m.cell_nbr.p, m.bsr_rowptr.p, m.blkmap.p);
  TFA_CUDA(m.pblkmap.alloc(BS * nc));
  k_pblkmap<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, F, BS, m.cell_nbr.p, m.blkmap.p, m.pblkmap.p);

  // vertex-neighbour stencil
  {
    DevBuf<uint32_t> nk, nk_s;
    DevBuf<int32_t> node_cnt, node_ptr;
    TFA_CUDA(nk.alloc(ne)); TFA_CUDA(nk_s.alloc(ne));
    TFA_CUDA(node_cnt.alloc(nn)); TFA_CUDA(node_ptr.alloc(nn + 1));
    TFA_CUDA(cudaMemsetAsync(node_cnt.p, 0, (size_t)nn * 4, st));
    k_node_pairs<<<cdiv(ne, TPB), TPB, 0, st>>>(ne, nn, F, m.cell_nodes.p, nk.p, vals.p, node_cnt.p);
    const int end_bit = bits_for((uint64_t)nn);
    size_t tmp_bytes = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, nk.p, nk_s.p, vals.p, vals_s.p, (int)ne, 0, end_bit, st);
    DevBuf<char> tmp;
    TFA_CUDA(tmp.alloc((int64_t)tmp_bytes));
    TFA_CUDA(cub::DeviceRadixSort::SortPairs(tmp.p, tmp_bytes, nk.p, nk_s.p, vals.p, vals_s.p, (int)ne, 0, end_bit,
                                             st));
    int64_t tot = 0;
    TFA_TRY(exclusive_scan_with_total(node_cnt, nn, node_ptr, &tot, st));
    k_stencil_count<<<cdiv(nc, 128), 128, 0, st>>>(nc, F, m.cell_nodes.p, node_ptr.p, vals_s.p, cnt.p, err.p);
    TFA_TRY(check_err(err, st));
    TFA_CUDA(m.st_ptr.alloc(nc + 1));
    TFA_TRY(exclusive_scan_with_total(cnt, nc, m.st_ptr, &m.nst, st));
    TFA_CUDA(m.st_idx.alloc(m.nst));
    TFA_CUDA(m.st_d.alloc(2 * m.nst));
    k_stencil_fill<<<cdiv(nc, 128), 128, 0, st>>>(nc, F, m.cell_nodes.p, node_ptr.p, vals_s.p, m.st_ptr.p, m.cell_xy.p,
                                                 m.cen.p, m.st_idx.p, m.st_d.p);
    TFA_CUDA(cudaStreamSynchronize(st));
  }
  TFA_CUDA(m.cgeo.alloc(8 * F * nc));
  TFA_CUDA(m.ggeo.alloc((2 * F + 2) * nc));
  k_cgeo<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, F, m.cell_nbr.p, m.cell_faces.p, vol.p, olen.p, onrm.p, ooff.p, m.cgeo.p,
                                       m.ggeo.p);

  // boundary faces in ascending face id; faces are numbered by their node pair, so the list -- and the tags the
  // caller attached to it -- do not change when the cells are renumbered
  {
    DevBuf<int32_t> flag, scan;
    TFA_CUDA(flag.alloc(m.nf)); TFA_CUDA(scan.alloc(m.nf + 1));
    k_bface_flag<<<cdiv(m.nf, TPB), TPB, 0, st>>>(m.nf, m.face_cells.p, flag.p);
    int64_t nb = 0;
    TFA_TRY(exclusive_scan_with_total(flag, m.nf, scan, &nb, st));
    TFA_CUDA(m.bface_of.alloc(m.nf));
    DevBuf<int32_t> bf;
    TFA_CUDA(bf.alloc(nb));
    k_bface_list<<<cdiv(m.nf, TPB), TPB, 0, st>>>(m.nf, flag.p, scan.p, m.bface_of.p, bf.p);
    TFA_CUDA(cudaStreamSynchronize(st));
    m.bfaces.swap(bf);
    if (m.nb != nb || !m.bc_tag.p) {   // a new mesh: every boundary face transmissive
      TFA_CUDA(m.bc_tag.alloc(nb));
      TFA_CUDA(cudaMemsetAsync(m.bc_tag.p, 0, (size_t)std::max<int64_t>(nb, 1) * 4, st));
      m.has_ghost = false;
    }
    m.nb = nb;
  }
  TFA_CUDA(m.nbrf.alloc(ne));
  TFA_TRY(refresh_nbrf(m, st));
  TFA_CUDA(cudaStreamSynchronize(st));
  m.uid = next_mesh_uid();
  return 0;
}

}  // namespace tfa

using namespace tfa;

namespace tfa {
// shared by the builders (and by tfa_shard_create): cells given as padded rows of F slots (host arrays)
int create_mesh_from_padded(tfa_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells, int F,
                       const int32_t* cell_nodes, const double* cell_xy, cudaStream_t st) {
  tfa_mesh* m = new (std::nothrow) tfa_mesh;
  if (!m) return set_error(TFA_ENOMEM, "host allocation failed");
  m->nn = n_nodes;
  m->nc = n_cells;
  m->F = F;
  auto body = [&]() -> int {
    TFA_CUDA(m->node_xy.alloc(2 * n_nodes));
    TFA_CUDA(m->cell_nodes.alloc(F * n_cells));
    TFA_CUDA(m->cell_xy.alloc(2 * F * n_cells));
    TFA_CUDA(m->perm.alloc(n_cells));
    if (node_xy && n_nodes)
      TFA_CUDA(cudaMemcpyAsync(m->node_xy.p, node_xy, (size_t)n_nodes * 16, cudaMemcpyHostToDevice, st));
    if (n_cells) {
      TFA_CUDA(cudaMemcpyAsync(m->cell_nodes.p, cell_nodes, (size_t)n_cells * F * 4, cudaMemcpyHostToDevice, st));
      if (cell_xy) {
        TFA_CUDA(cudaMemcpyAsync(m->cell_xy.p, cell_xy, (size_t)n_cells * F * 16, cudaMemcpyHostToDevice, st));
      } else {
        DevBuf<int32_t> err;
        TFA_CUDA(err.alloc(2));
        TFA_CUDA(cudaMemsetAsync(err.p, 0, 8, st));
        k_gather_xy<<<cdiv(F * n_cells, TPB), TPB, 0, st>>>(F * n_cells, n_nodes, m->cell_nodes.p, m->node_xy.p,
                                                           m->cell_xy.p, err.p);
        TFA_TRY(check_err(err, st));
      }
      k_iota<<<cdiv(n_cells, TPB), TPB, 0, st>>>(n_cells, m->perm.p);
    }
    TFA_CUDA(cudaStreamSynchronize(st));   // the host arrays may be temporaries of the caller
    return build_mesh(*m, st);
  };
  int rc = body();
  if (rc) { delete m; return rc; }
  *out = m;
  return 0;
}
}  // namespace tfa

extern "C" {

const char* tfa_last_error(void) { return tfa::g_last_error.c_str(); }
const char* tfa_version(void) { return "tfa 0.2 (sm_100a)"; }

int tfa_mesh_create(tfa_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                    const int32_t* cell_nodes, const double* cell_xy, void* stream) {
  if (!out || n_nodes < 0 || n_cells < 0 || (n_cells > 0 && !cell_nodes) || (!node_xy && !cell_xy && n_cells > 0))
    return set_error(TFA_EINVAL, "tfa_mesh_create: bad argument");
  return create_mesh_from_padded(out, n_nodes, node_xy, n_cells, 3, cell_nodes, cell_xy, (cudaStream_t)stream);
}

int tfa_mesh_create_poly(tfa_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                         const int32_t* cell_ptr, const int32_t* cell_nodes, const double* cell_xy, void* stream) {
  if (!out || n_nodes < 0 || n_cells < 0 || !cell_ptr || (n_cells > 0 && !cell_nodes) ||
      (!node_xy && !cell_xy && n_cells > 0))
    return set_error(TFA_EINVAL, "tfa_mesh_create_poly: bad argument");
  if (cell_ptr[0] != 0) return set_error(TFA_EINVAL, "tfa_mesh_create_poly: cell_ptr must start at 0");
  int F = 3;
  for (int64_t i = 0; i < n_cells; ++i) {
    const int nv = cell_ptr[i + 1] - cell_ptr[i];
    if (nv != 3 && nv != 4)
      return set_error(TFA_EINVAL, "tfa_mesh_create_poly: cell " + std::to_string(i) + " must have 3 or 4 corners");
    if (nv == 4) F = 4;
  }
  // argument marshalling: the CSR rows become rows of F slots (node -1 in the fourth slot of a triangle)
  std::vector<int32_t> cn((size_t)F * n_cells, -1);
  std::vector<double> cx;
  if (cell_xy) cx.assign((size_t)2 * F * n_cells, 0.0);
  for (int64_t i = 0; i < n_cells; ++i)
    for (int32_t q = cell_ptr[i]; q < cell_ptr[i + 1]; ++q) {
      const size_t slot = (size_t)F * i + (q - cell_ptr[i]);
      cn[slot] = cell_nodes[q];
      if (cell_xy) { cx[2 * slot] = cell_xy[2 * (size_t)q]; cx[2 * slot + 1] = cell_xy[2 * (size_t)q + 1]; }
    }
  return create_mesh_from_padded(out, n_nodes, node_xy, n_cells, F, cn.data(), cell_xy ? cx.data() : nullptr,
                            (cudaStream_t)stream);
}

int tfa_mesh_info(const tfa_mesh* m, int32_t* max_faces, int64_t* n_bfaces) {
  if (!m) return set_error(TFA_EINVAL, "null mesh");
  if (max_faces) *max_faces = m->F;
  if (n_bfaces) *n_bfaces = m->nb;
  return 0;
}

int tfa_mesh_set_bc(tfa_mesh* m, const int32_t* tags, void* stream) {
  if (!m || (m->nb > 0 && !tags)) return set_error(TFA_EINVAL, "null argument");
  if (m->shard_local) return set_error(TFA_EINVAL, "tfa_mesh_set_bc: set the rules on the global mesh before sharding");
  bool ghost = false;
  for (int64_t b = 0; b < m->nb; ++b) {
    if (tags[b] < TFA_BC_TRANSMISSIVE || tags[b] > TFA_BC_WALL) return set_error(TFA_EINVAL, "unknown boundary tag");
    ghost |= tags[b] == TFA_BC_GHOST;
  }
  cudaStream_t st = (cudaStream_t)stream;
  if (m->nb) TFA_CUDA(cudaMemcpyAsync(m->bc_tag.p, tags, (size_t)m->nb * 4, cudaMemcpyHostToDevice, st));
  m->has_ghost = ghost;
  TFA_TRY(refresh_nbrf(*m, st));
  TFA_CUDA(cudaStreamSynchronize(st));
  return 0;
}

int tfa_mesh_reorder(tfa_mesh* m, int kind, const int32_t* user_perm, void* stream) {
  if (!m) return set_error(TFA_EINVAL, "null mesh");
  if (kind == 0 || m->nc == 0) return 0;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t nc = m->nc;
  const int F = m->F;
  DevBuf<int32_t> p;
  TFA_CUDA(p.alloc(nc));
  if (kind == 1) {
    DevBuf<int32_t> order, pos, parent;
    TFA_CUDA(order.alloc(nc)); TFA_CUDA(pos.alloc(nc)); TFA_CUDA(parent.alloc(nc));
    k_rcm<<<1, RCM_T, 0, st>>>((int32_t)nc, F, m->cell_nbr.p, order.p, pos.p, parent.p);
    k_reverse<<<cdiv(nc, TPB), TPB, 0, st>>>((int32_t)nc, order.p, p.p);
    TFA_CUDA(cudaGetLastError());
    TFA_CUDA(cudaStreamSynchronize(st));
  } else if (kind == 3) {
    DevBuf<unsigned long long> box;
    DevBuf<uint64_t> keys, keys_s;
    DevBuf<int32_t> ids;
    TFA_CUDA(box.alloc(4)); TFA_CUDA(keys.alloc(nc)); TFA_CUDA(keys_s.alloc(nc)); TFA_CUDA(ids.alloc(nc));
    const unsigned long long init[4] = {~0ull, 0ull, ~0ull, 0ull};
    TFA_CUDA(cudaMemcpyAsync(box.p, init, sizeof(init), cudaMemcpyHostToDevice, st));
    k_bbox<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, m->cen.p, box.p);
    k_morton_keys<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, m->cen.p, box.p, keys.p, ids.p);
    size_t tmp_bytes = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys.p, keys_s.p, ids.p, p.p, (int)nc, 0, 64, st);
    DevBuf<char> tmp;
    TFA_CUDA(tmp.alloc((int64_t)tmp_bytes));
    TFA_CUDA(cub::DeviceRadixSort::SortPairs(tmp.p, tmp_bytes, keys.p, keys_s.p, ids.p, p.p, (int)nc, 0, 64, st));
    TFA_CUDA(cudaStreamSynchronize(st));
  } else if (kind == 2) {
    if (!user_perm) return set_error(TFA_EINVAL, "user permutation missing");
    TFA_CUDA(cudaMemcpyAsync(p.p, user_perm, (size_t)nc * 4, cudaMemcpyHostToDevice, st));
    DevBuf<int32_t> hit, err;
    TFA_CUDA(hit.alloc(nc)); TFA_CUDA(err.alloc(2));
    TFA_CUDA(cudaMemsetAsync(hit.p, 0, (size_t)nc * 4, st));
    TFA_CUDA(cudaMemsetAsync(err.p, 0, 8, st));
    k_check_perm<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, p.p, hit.p, err.p);
    int rc = check_err(err, st);
    if (rc) return set_error(TFA_EINVAL, tfa::g_last_error);
  } else {
    return set_error(TFA_EINVAL, "unknown reorder kind");
  }
  DevBuf<int32_t> cn, pm;
  DevBuf<double> cx;
  TFA_CUDA(cn.alloc(F * nc)); TFA_CUDA(pm.alloc(nc)); TFA_CUDA(cx.alloc(2 * F * nc));
  k_permute_cells<<<cdiv(nc, TPB), TPB, 0, st>>>(nc, F, p.p, m->cell_nodes.p, m->cell_xy.p, m->perm.p, cn.p, cx.p,
                                                pm.p);
  TFA_CUDA(cudaStreamSynchronize(st));
  m->cell_nodes.swap(cn);
  m->cell_xy.swap(cx);
  m->perm.swap(pm);
  return build_mesh(*m, st);
}

int tfa_mesh_sizes(const tfa_mesh* m, int64_t* n_cells, int64_t* n_faces, int64_t* nnzb, int64_t* n_stencil) {
  if (!m) return set_error(TFA_EINVAL, "null mesh");
  if (n_cells) *n_cells = m->nc;
  if (n_faces) *n_faces = m->nf;
  if (nnzb) *nnzb = m->nnzb;
  if (n_stencil) *n_stencil = m->nst;
  return 0;
}

static const void* item_ptr(const tfa_mesh* m, int which, int64_t* bytes) {
  switch (which) {
    case TFA_FACE_CELLS: *bytes = m->nf * 8; return m->face_cells.p;
    case TFA_FACE_NODES: *bytes = m->nf * 8; return m->face_nodes.p;
    case TFA_CELL_FACES: *bytes = m->nc * m->F * 4; return m->cell_faces.p;
    case TFA_CELL_NBR: *bytes = m->nc * m->F * 4; return m->cell_nbr.p;
    case TFA_STENCIL_PTR: *bytes = (m->nc + 1) * 4; return m->st_ptr.p;
    case TFA_STENCIL_IDX: *bytes = m->nst * 4; return m->st_idx.p;
    case TFA_BSR_ROWPTR: *bytes = (m->nc + 1) * 4; return m->bsr_rowptr.p;
    case TFA_BSR_COL: *bytes = m->nnzb * 4; return m->bsr_col.p;
    case TFA_PERM: *bytes = m->nc * 4; return m->perm.p;
    case TFA_CENTROID: *bytes = m->nc * 16; return m->cen.p;
    case TFA_BFACES: *bytes = m->nb * 4; return m->bfaces.p;
    case TFA_BC_TAGS: *bytes = m->nb * 4; return m->bc_tag.p;
    default: return nullptr;
  }
}

int tfa_mesh_get(const tfa_mesh* m, int which, void* host_dst, int64_t bytes) {
  if (!m || !host_dst) return set_error(TFA_EINVAL, "null argument");
  int64_t need = 0;
  if (which == TFA_VOLUME || which == TFA_FACE_NORMAL_LEN) {
    const int64_t n = which == TFA_VOLUME ? m->nc : 3 * m->nf;
    if (bytes != n * 8) return set_error(TFA_EINVAL, "tfa_mesh_get: size mismatch, need " + std::to_string(n * 8));
    if (n == 0) return 0;
    DevBuf<double> tmp;
    TFA_CUDA(tmp.alloc(n));
    if (which == TFA_VOLUME) k_volume_out<<<cdiv(m->nc, TPB), TPB>>>(m->nc, m->F, m->cgeo.p, tmp.p);
    else k_face_geom_out<<<cdiv(m->nf, TPB), TPB>>>(m->nf, m->F, m->face_cells.p, m->cell_faces.p, m->cgeo.p, tmp.p);
    TFA_CUDA(cudaMemcpy(host_dst, tmp.p, (size_t)n * 8, cudaMemcpyDeviceToHost));
    return 0;
  }
  const void* src = item_ptr(m, which, &need);
  if (!src && need == 0 && (which == TFA_BFACES || which == TFA_BC_TAGS) && bytes == 0) return 0;
  if (!src) return set_error(TFA_EINVAL, "tfa_mesh_get: unknown item");
  if (bytes != need) return set_error(TFA_EINVAL, "tfa_mesh_get: size mismatch, need " + std::to_string(need));
  if (need) TFA_CUDA(cudaMemcpy(host_dst, src, (size_t)need, cudaMemcpyDeviceToHost));
  return 0;
}

const void* tfa_mesh_device_ptr(const tfa_mesh* m, int which) {
  if (!m) return nullptr;
  int64_t b = 0;
  return item_ptr(m, which, &b);
}

void tfa_mesh_destroy(tfa_mesh* m) { delete m; }

}  // extern "C"

// oracle/tfo.cpp — CPU ORACLE (TEST INFRASTRUCTURE ONLY; see tfo.h for the rules and the pins).
//
// Step-by-step restatement of the assembly of arXiv 1809.02532 in the paper's order and
// notation.  "L<n>" = line of /root/reference/PAPER.md; "S<n>" = reading listed in DESIGN.md.
// Shares no code with paper_1809_02532_b200/csrc.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif
#ifdef TFO_COUNT_OPS
// measurement build (oracle/count_ops.py): every `double` below is the op-counting scalar of opcount.h
#include "opcount.h"
#define double tfo_count::real
#endif
#include "tfo.h"

namespace {

constexpr int NEQ = TFO_NEQ;
thread_local std::string g_err;

int fail(int code, const std::string& msg) {
  g_err = msg;
  return code;
}

// Variable order (S: "Conventions"): 0..2 B, 3..5 E, 6 Psi, 7 Phi, 8 rho_i, 9 rho_e,
// 10..12 u_i, 13..15 u_e, 16 T_i, 17 T_e.  Equation rows in the same order with
// rho->mass, u->momentum, T->total energy.
inline int i_rho(int s) { return 8 + s; }
inline int i_u(int s) { return 10 + 3 * s; }
inline int i_T(int s) { return 16 + s; }

// Normalisation: mu0 = 1, eps0 = 1/c^2, k_B = 1, m_i = 1, m_e = 1/mass_ratio,
// q_i = +1, q_e = -1.  R_s = k_B/m_s, q_s/m_s = charge-to-mass ratio.
inline double R_s(const tfo_physics& ph, int s) { return s == 0 ? 1.0 : ph.mass_ratio; }
inline double qm_s(const tfo_physics& ph, int s) { return s == 0 ? 1.0 : -ph.mass_ratio; }

}  // namespace

struct tfo_mesh {
  int64_t nn = 0, nc = 0, nf = 0;
  int maxf = 3;                      // largest number of faces of a cell (3 triangles only, 4 with quadrilaterals)
  std::vector<double> node_xy;       // [nn][2]
  std::vector<int32_t> cptr;         // [nc+1]: corners (= local faces) of cell i are cptr[i] .. cptr[i+1]-1
  std::vector<int32_t> cell_nodes;   // [cptr[nc]], counter-clockwise
  std::vector<double> cell_xy;       // [cptr[nc]][2]
  std::vector<int32_t> face_nodes;   // [nf][2] (lo, hi)
  std::vector<int32_t> face_cells;   // [nf][2] (L, R or -1)
  std::vector<int32_t> cell_faces;   // [cptr[nc]]: face of local edge k = (corner k -> corner k+1)
  std::vector<int32_t> st_ptr, st_idx;
  std::vector<double> st_d;          // [nst][2] displacement centroid_j - centroid_i (S9)
  std::vector<int32_t> bsr_rowptr, bsr_col;
  std::vector<int32_t> perm;         // new -> old
  // geometry, per cell from its own corners
  std::vector<double> cen;           // [nc][2]
  std::vector<double> vol;           // [nc]
  std::vector<double> fmid_off;      // [cptr[nc]][2]  midpoint of local edge k minus centroid
  std::vector<double> fnrm;          // [cptr[nc]][2]  outward unit normal of local edge k
  std::vector<double> flen;          // [cptr[nc]]
  // boundary conditions (L260: a separate loop over the boundary faces; S9, S24)
  std::vector<int32_t> bfaces;       // boundary faces (R = -1) in ascending face id
  std::vector<int32_t> bface_of;     // [nf] index into bfaces, -1 for interior faces
  std::vector<int32_t> bc_tag;       // [nb] TFO_BC_*
  std::vector<double> ghost;         // [nb][18] ghost states of the TFO_BC_GHOST faces (empty = none given)
  int nv(int64_t i) const { return cptr[i + 1] - cptr[i]; }
};

namespace {

// ------------------------------------------------------------------------------------------
// step 1-2: connectivity and geometry
// ------------------------------------------------------------------------------------------
int build(tfo_mesh& m) {
  const int64_t nc = m.nc;
  const int64_t ncorn = nc ? m.cptr[nc] : 0;
  m.maxf = 3;
  // geometry per cell
  m.cen.assign(2 * nc, 0.0);
  m.vol.assign(nc, 0.0);
  m.fmid_off.assign(2 * ncorn, 0.0);
  m.fnrm.assign(2 * ncorn, 0.0);
  m.flen.assign(ncorn, 0.0);
  for (int64_t i = 0; i < nc; ++i) {
    const int nv = m.nv(i);
    const int64_t c0 = m.cptr[i];
    if (nv < 3 || nv > TFO_MAXV) return fail(-2, "cell " + std::to_string(i) + " must have 3 or 4 corners");
    m.maxf = std::max(m.maxf, nv);
    const double* X = &m.cell_xy[2 * c0];
    double cx, cy, area;
    if (nv == 3) {
      cx = (X[0] + X[2] + X[4]) / 3.0;
      cy = (X[1] + X[3] + X[5]) / 3.0;
      area = 0.5 * ((X[2] - X[0]) * (X[5] - X[1]) - (X[3] - X[1]) * (X[4] - X[0]));
      if (!(area > 0.0)) return fail(-2, "cell " + std::to_string(i) + " is not counter-clockwise");
    } else {
      // polygon: shoelace area and area centroid, taken relative to corner 0 (no cancellation against the
      // cell's position in the domain); every corner must turn left (convex, counter-clockwise)
      double a2 = 0.0, sx = 0.0, sy = 0.0;
      for (int k = 1; k + 1 < nv; ++k) {
        const double ax = X[2 * k] - X[0], ay = X[2 * k + 1] - X[1];
        const double bx = X[2 * k + 2] - X[0], by = X[2 * k + 3] - X[1];
        const double cr = ax * by - ay * bx;   // twice the area of the triangle (corner 0, k, k+1)
        a2 += cr;
        sx += cr * (ax + bx);                  // times three times that triangle's centroid offset
        sy += cr * (ay + by);
      }
      area = 0.5 * a2;
      for (int k = 0; k < nv; ++k) {
        const int k1 = (k + 1) % nv, k2 = (k + 2) % nv;
        const double ux = X[2 * k1] - X[2 * k], uy = X[2 * k1 + 1] - X[2 * k + 1];
        const double vx = X[2 * k2] - X[2 * k1], vy = X[2 * k2 + 1] - X[2 * k1 + 1];
        if (!(ux * vy - uy * vx > 0.0))
          return fail(-2, "cell " + std::to_string(i) + " is not a convex counter-clockwise polygon");
      }
      if (!(area > 0.0)) return fail(-2, "cell " + std::to_string(i) + " is not counter-clockwise");
      cx = X[0] + sx / (3.0 * a2);
      cy = X[1] + sy / (3.0 * a2);
    }
    m.cen[2 * i] = cx;
    m.cen[2 * i + 1] = cy;
    m.vol[i] = area;
    for (int k = 0; k < nv; ++k) {
      int k1 = (k + 1) % nv;
      double ax = X[2 * k], ay = X[2 * k + 1], bx = X[2 * k1], by = X[2 * k1 + 1];
      double dx = bx - ax, dy = by - ay;
      double len = std::sqrt(dx * dx + dy * dy);
      m.flen[c0 + k] = len;
      m.fnrm[2 * (c0 + k)] = dy / len;        // outward for a CCW cell: (dy, -dx)/len
      m.fnrm[2 * (c0 + k) + 1] = -dx / len;
      m.fmid_off[2 * (c0 + k)] = 0.5 * (ax + bx) - cx;
      m.fmid_off[2 * (c0 + k) + 1] = 0.5 * (ay + by) - cy;
    }
    const int32_t* cn = &m.cell_nodes[c0];
    for (int a = 0; a < nv; ++a)
      for (int b = a + 1; b < nv; ++b)
        if (cn[a] == cn[b])
          return fail(-2, "cell " + std::to_string(i) + " repeats a node (periodic direction too narrow)");
    for (int k = 0; k < nv; ++k)
      if (cn[k] < 0 || cn[k] >= m.nn) return fail(-2, "node id out of range");
  }
  // faces = unique node pairs, sorted by (lo, hi) (S10)
  struct Edge { int64_t key; int32_t cell, k; };
  std::vector<Edge> edges(ncorn);
  for (int64_t i = 0; i < nc; ++i)
    for (int k = 0; k < m.nv(i); ++k) {
      int32_t a = m.cell_nodes[m.cptr[i] + k], b = m.cell_nodes[m.cptr[i] + (k + 1) % m.nv(i)];
      int64_t lo = std::min(a, b), hi = std::max(a, b);
      edges[m.cptr[i] + k] = {lo * (int64_t)m.nn + hi, (int32_t)i, k};
    }
  std::sort(edges.begin(), edges.end(), [](const Edge& x, const Edge& y) {
    return x.key != y.key ? x.key < y.key : (x.cell != y.cell ? x.cell < y.cell : x.k < y.k);
  });
  m.face_nodes.clear();
  m.face_cells.clear();
  m.cell_faces.assign(ncorn, -1);
  for (size_t e = 0; e < edges.size();) {
    size_t e2 = e;
    while (e2 < edges.size() && edges[e2].key == edges[e].key) ++e2;
    if (e2 - e > 2) return fail(-2, "non-manifold edge: a node pair is shared by more than 2 cells");
    int32_t f = (int32_t)(m.face_cells.size() / 2);
    m.face_nodes.push_back((int32_t)(edges[e].key / m.nn));
    m.face_nodes.push_back((int32_t)(edges[e].key % m.nn));
    m.face_cells.push_back(edges[e].cell);                       // L = smaller cell id
    m.face_cells.push_back(e2 - e == 2 ? edges[e + 1].cell : -1);
    if (e2 - e == 2 && edges[e].cell == edges[e + 1].cell)
      return fail(-2, "a cell is its own neighbour (periodic direction too narrow)");
    for (size_t q = e; q < e2; ++q) m.cell_faces[m.cptr[edges[q].cell] + edges[q].k] = f;
    e = e2;
  }
  m.nf = (int64_t)m.face_cells.size() / 2;
  // vertex-neighbour stencil (L74: "all face-vertex cell neighbors"), ascending, unique, no self
  std::vector<std::vector<int32_t>> node_cells(m.nn);
  for (int64_t i = 0; i < nc; ++i)
    for (int k = 0; k < m.nv(i); ++k) node_cells[m.cell_nodes[m.cptr[i] + k]].push_back((int32_t)i);
  m.st_ptr.assign(nc + 1, 0);
  m.st_idx.clear();
  m.st_d.clear();
  for (int64_t i = 0; i < nc; ++i) {
    std::vector<int32_t> s;
    for (int k = 0; k < m.nv(i); ++k)
      for (int32_t j : node_cells[m.cell_nodes[m.cptr[i] + k]])
        if (j != i) s.push_back(j);
    std::sort(s.begin(), s.end());
    s.erase(std::unique(s.begin(), s.end()), s.end());
    for (int32_t j : s) {
      // displacement through the smallest shared node id (S9, S22)
      int32_t v = INT32_MAX;
      for (int a = 0; a < m.nv(i); ++a)
        for (int b = 0; b < m.nv(j); ++b)
          if (m.cell_nodes[m.cptr[i] + a] == m.cell_nodes[m.cptr[j] + b]) v = std::min(v, m.cell_nodes[m.cptr[i] + a]);
      int ai = 0, bj = 0;
      for (int a = 0; a < m.nv(i); ++a)
        if (m.cell_nodes[m.cptr[i] + a] == v) ai = a;
      for (int a = 0; a < m.nv(j); ++a)
        if (m.cell_nodes[m.cptr[j] + a] == v) bj = a;
      double dx = (m.cen[2 * j] - m.cell_xy[2 * (m.cptr[j] + bj)]) - (m.cen[2 * i] - m.cell_xy[2 * (m.cptr[i] + ai)]);
      double dy = (m.cen[2 * j + 1] - m.cell_xy[2 * (m.cptr[j] + bj) + 1]) -
                  (m.cen[2 * i + 1] - m.cell_xy[2 * (m.cptr[i] + ai) + 1]);
      m.st_idx.push_back(j);
      m.st_d.push_back(dx);
      m.st_d.push_back(dy);
    }
    m.st_ptr[i + 1] = (int32_t)m.st_idx.size();
  }
  // BSR pattern: self + face neighbours, ascending (L321: "blocks ... linking two different cells")
  m.bsr_rowptr.assign(nc + 1, 0);
  m.bsr_col.clear();
  for (int64_t i = 0; i < nc; ++i) {
    std::vector<int32_t> cols{(int32_t)i};
    for (int k = 0; k < m.nv(i); ++k) {
      int32_t f = m.cell_faces[m.cptr[i] + k];
      int32_t j = m.face_cells[2 * f] == i ? m.face_cells[2 * f + 1] : m.face_cells[2 * f];
      if (j >= 0) cols.push_back(j);
    }
    std::sort(cols.begin(), cols.end());
    if (std::adjacent_find(cols.begin(), cols.end()) != cols.end())
      return fail(-2, "two faces of a cell lead to the same neighbour (periodic direction too narrow)");
    for (int32_t j : cols) m.bsr_col.push_back(j);
    m.bsr_rowptr[i + 1] = (int32_t)m.bsr_col.size();
  }
  // boundary faces in ascending face id.  Faces are numbered by their node pair, so neither this list nor the
  // tags attached to it change when the cells are reordered.
  m.bfaces.clear();
  m.bface_of.assign(m.nf, -1);
  for (int64_t f = 0; f < m.nf; ++f)
    if (m.face_cells[2 * f + 1] < 0) {
      m.bface_of[f] = (int32_t)m.bfaces.size();
      m.bfaces.push_back((int32_t)f);
    }
  if (m.bc_tag.size() != m.bfaces.size()) {
    m.bc_tag.assign(m.bfaces.size(), TFO_BC_TRANSMISSIVE);
    m.ghost.clear();
  }
  return 0;
}

// S11: reverse Cuthill-McKee on the face-neighbour graph
std::vector<int32_t> rcm_order(const tfo_mesh& m) {
  const int64_t nc = m.nc;
  std::vector<int32_t> deg(nc);
  for (int64_t i = 0; i < nc; ++i) deg[i] = m.bsr_rowptr[i + 1] - m.bsr_rowptr[i] - 1;
  std::vector<char> seen(nc, 0);
  std::vector<int32_t> order;
  order.reserve(nc);
  int64_t scan_from = 0;
  (void)scan_from;
  while ((int64_t)order.size() < nc) {
    int32_t start = -1;
    for (int64_t i = 0; i < nc; ++i)
      if (!seen[i] && (start < 0 || deg[i] < deg[start])) start = (int32_t)i;
    size_t head = order.size();
    order.push_back(start);
    seen[start] = 1;
    while (head < order.size()) {
      int32_t v = order[head++];
      std::vector<int32_t> nb;
      for (int32_t q = m.bsr_rowptr[v]; q < m.bsr_rowptr[v + 1]; ++q) {
        int32_t w = m.bsr_col[q];
        if (w != v && !seen[w]) nb.push_back(w);
      }
      std::sort(nb.begin(), nb.end(), [&](int32_t a, int32_t b) {
        return deg[a] != deg[b] ? deg[a] < deg[b] : a < b;
      });
      for (int32_t w : nb) {
        seen[w] = 1;
        order.push_back(w);
      }
    }
  }
  std::reverse(order.begin(), order.end());
  return order;   // new -> old
}

// ------------------------------------------------------------------------------------------
// physics, point-wise
// ------------------------------------------------------------------------------------------
// Eq. 2/3 (L50, L56) contracted with n=(nx,ny,0) (S2): H(U) = F.n for the 8 Maxwell rows.
void maxwell_physical_flux(const tfo_physics& ph, const double* U, double nx, double ny, double* H) {
  const double c2 = ph.c * ph.c;
  const double gp2 = ph.gamma_psi * ph.gamma_psi;
  const double xc2 = (ph.chi_phi * ph.c) * (ph.chi_phi * ph.c);
  const double Bx = U[0], By = U[1], Bz = U[2], Ex = U[3], Ey = U[4], Ez = U[5], Psi = U[6], Phi = U[7];
  // n x V = (ny Vz, -nx Vz, nx Vy - ny Vx)
  H[0] = ny * Ez + gp2 * Psi * nx;
  H[1] = -nx * Ez + gp2 * Psi * ny;
  H[2] = nx * Ey - ny * Ex;
  H[3] = -c2 * (ny * Bz) + xc2 * Phi * nx;
  H[4] = -c2 * (-nx * Bz) + xc2 * Phi * ny;
  H[5] = -c2 * (nx * By - ny * Bx);
  H[6] = c2 * (Bx * nx + By * ny);
  H[7] = Ex * nx + Ey * ny;
}

// Eq. 9 (L91) with |A_n| = alpha R|Lambda|R^-1 in closed form (S3)
void maxwell_flux(const tfo_physics& ph, const double* UL, const double* UR, double nx, double ny,
                  double* H) {
  double HL[8], HR[8], D[8], dU[8];
  maxwell_physical_flux(ph, UL, nx, ny, HL);
  maxwell_physical_flux(ph, UR, nx, ny, HR);
  for (int r = 0; r < 8; ++r) dU[r] = UR[r] - UL[r];
  const double c = ph.c;
  const double dBn = dU[0] * nx + dU[1] * ny;   // n_z = 0
  const double dEn = dU[3] * nx + dU[4] * ny;
  const double nvec[3] = {nx, ny, 0.0};
  for (int d = 0; d < 3; ++d) {
    D[d] = c * (dU[d] - dBn * nvec[d]) + ph.gamma_psi * c * dBn * nvec[d];
    D[3 + d] = c * (dU[3 + d] - dEn * nvec[d]) + ph.chi_phi * c * dEn * nvec[d];
  }
  D[6] = ph.gamma_psi * c * dU[6];
  D[7] = ph.chi_phi * c * dU[7];
  for (int r = 0; r < 8; ++r) H[r] = 0.5 * (HL[r] + HR[r]) - 0.5 * ph.rusanov_alpha * D[r];
}

// AUSM+-up split functions (Liou 2006, ref. [30] of the paper; S4)
inline double M1p(double M) { return 0.5 * (M + std::fabs(M)); }
inline double M1m(double M) { return 0.5 * (M - std::fabs(M)); }
inline double M2p(double M) { return 0.25 * (M + 1.0) * (M + 1.0); }
inline double M2m(double M) { return -0.25 * (M - 1.0) * (M - 1.0); }
inline double M4p(double M, double beta) {
  return std::fabs(M) >= 1.0 ? M1p(M) : M2p(M) * (1.0 - 16.0 * beta * M2m(M));
}
inline double M4m(double M, double beta) {
  return std::fabs(M) >= 1.0 ? M1m(M) : M2m(M) * (1.0 + 16.0 * beta * M2p(M));
}
inline double P5p(double M, double alpha) {
  return std::fabs(M) >= 1.0 ? M1p(M) / M : M2p(M) * ((2.0 - M) - 16.0 * alpha * M * M2m(M));
}
inline double P5m(double M, double alpha) {
  return std::fabs(M) >= 1.0 ? M1m(M) / M : M2m(M) * ((-2.0 - M) + 16.0 * alpha * M * M2p(M));
}

// Eq. 10 (L97): H_s = M a (rho, rho u, rho H) + p (0, n, 0); P = (rho, u, v, w, T)
void ausm_flux(const tfo_physics& ph, const tfo_numerics& nu, int s, const double* L, const double* R,
               double nx, double ny, double* H) {
  const double g = ph.gamma_gas, Rs = R_s(ph, s);
  const double cp = g * Rs / (g - 1.0);
  const double rhoL = L[0], rhoR = R[0], TL = L[4], TR = R[4];
  const double pL = rhoL * Rs * TL, pR = rhoR * Rs * TR;
  const double aL = std::sqrt(g * Rs * TL), aR = std::sqrt(g * Rs * TR);
  const double unL = L[1] * nx + L[2] * ny, unR = R[1] * nx + R[2] * ny;
  const double HtL = cp * TL + 0.5 * (L[1] * L[1] + L[2] * L[2] + L[3] * L[3]);
  const double HtR = cp * TR + 0.5 * (R[1] * R[1] + R[2] * R[2] + R[3] * R[3]);
  const double a12 = 0.5 * (aL + aR);
  const double ML = unL / a12, MR = unR / a12;
  const double Mbar2 = (unL * unL + unR * unR) / (2.0 * a12 * a12);
  const double Minf = nu.ausm_Minf[s];
  const double Mo = std::sqrt(std::min(1.0, std::max(Mbar2, Minf * Minf)));
  const double fa = Mo * (2.0 - Mo);
  const double alpha = (3.0 / 16.0) * (-4.0 + 5.0 * fa * fa);
  const double rho12 = 0.5 * (rhoL + rhoR);
  const double Mp = -(nu.ausm_Kp / fa) * std::max(1.0 - nu.ausm_sigma * Mbar2, 0.0) * (pR - pL) /
                    (rho12 * a12 * a12);
  const double M12 = M4p(ML, nu.ausm_beta) + M4m(MR, nu.ausm_beta) + Mp;
  const double mdot = a12 * M12 * (M12 > 0.0 ? rhoL : rhoR);
  const double Pp = P5p(ML, alpha), Pm = P5m(MR, alpha);
  const double pu = -nu.ausm_Ku * Pp * Pm * (rhoL + rhoR) * (fa * a12) * (unR - unL);
  const double p12 = Pp * pL + Pm * pR + pu;
  const double* U = mdot > 0.0 ? L : R;
  const double Ht = mdot > 0.0 ? HtL : HtR;
  H[0] = mdot;
  H[1] = mdot * U[1] + p12 * nx;
  H[2] = mdot * U[2] + p12 * ny;
  H[3] = mdot * U[3];
  H[4] = mdot * Ht;
}

void gather_species(const double* P, int s, double* Q) {
  Q[0] = P[i_rho(s)];
  Q[1] = P[i_u(s)];
  Q[2] = P[i_u(s) + 1];
  Q[3] = P[i_u(s) + 2];
  Q[4] = P[i_T(s)];
}
void scatter_species(const double* H5, int s, double* H) {
  H[i_rho(s)] = H5[0];
  H[i_u(s)] = H5[1];
  H[i_u(s) + 1] = H5[2];
  H[i_u(s) + 2] = H5[3];
  H[i_T(s)] = H5[4];
}

// FLUXSCHEME of Alg. 1 (L233): all 18 rows of the numerical flux at a face
void face_flux(const tfo_physics& ph, const tfo_numerics& nu, const double* PL, const double* PR,
               double nx, double ny, double* H) {
  maxwell_flux(ph, PL, PR, nx, ny, H);
  for (int s = 0; s < 2; ++s) {
    double L[5], R[5], H5[5];
    gather_species(PL, s, L);
    gather_species(PR, s, R);
    ausm_flux(ph, nu, s, L, R, nx, ny, H5);
    scatter_species(H5, s, H);
  }
}

// Eq. 4 (L60) and Eq. 6 (L65-68) with charge density rho_s q_s/m_s (S5), eps0 = 1/c^2
void source(const tfo_physics& ph, const double* P, double* S) {
  for (int r = 0; r < NEQ; ++r) S[r] = 0.0;
  const double c2 = ph.c * ph.c;
  const double* B = P;
  const double* E = P + 3;
  double J[3] = {0, 0, 0}, rhoc = 0.0;
  for (int s = 0; s < 2; ++s) {
    const double qn = qm_s(ph, s) * P[i_rho(s)];   // q_s n_s
    const double* u = P + i_u(s);
    rhoc += qn;
    for (int d = 0; d < 3; ++d) J[d] += qn * u[d];
    const double uxB[3] = {u[1] * B[2] - u[2] * B[1], u[2] * B[0] - u[0] * B[2], u[0] * B[1] - u[1] * B[0]};
    for (int d = 0; d < 3; ++d) S[i_u(s) + d] = qn * (E[d] + uxB[d]);
    S[i_T(s)] = qn * (u[0] * E[0] + u[1] * E[1] + u[2] * E[2]);
  }
  for (int d = 0; d < 3; ++d) S[3 + d] = -c2 * J[d];   // -J/eps0
  S[7] = c2 * rhoc;                                     // rho_c/eps0
}

// U(P) (L50: U=P for the field; L63 Eq. 5: eps = c_v T + u^2/2)
void cons(const tfo_physics& ph, const double* P, double* U) {
  for (int r = 0; r < 8; ++r) U[r] = P[r];
  for (int s = 0; s < 2; ++s) {
    const double cv = R_s(ph, s) / (ph.gamma_gas - 1.0);
    const double rho = P[i_rho(s)];
    const double* u = P + i_u(s);
    U[i_rho(s)] = rho;
    for (int d = 0; d < 3; ++d) U[i_u(s) + d] = rho * u[d];
    U[i_T(s)] = rho * (cv * P[i_T(s)] + 0.5 * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]));
  }
}

// analytic dU/dP (S15)
void dcons_dprim(const tfo_physics& ph, const double* P, double* D) {
  for (int q = 0; q < NEQ * NEQ; ++q) D[q] = 0.0;
  for (int r = 0; r < 8; ++r) D[r * NEQ + r] = 1.0;
  for (int s = 0; s < 2; ++s) {
    const double cv = R_s(ph, s) / (ph.gamma_gas - 1.0);
    const int ir = i_rho(s), iu = i_u(s), iT = i_T(s);
    const double rho = P[ir], T = P[iT];
    const double* u = P + iu;
    D[ir * NEQ + ir] = 1.0;
    for (int d = 0; d < 3; ++d) {
      D[(iu + d) * NEQ + ir] = u[d];
      D[(iu + d) * NEQ + iu + d] = rho;
      D[iT * NEQ + iu + d] = rho * u[d];
    }
    D[iT * NEQ + ir] = cv * T + 0.5 * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
    D[iT * NEQ + iT] = rho * cv;
  }
}

// ------------------------------------------------------------------------------------------
// step a2: gradient + limiter for one cell
// ------------------------------------------------------------------------------------------
void grad_cell(const tfo_mesh& m, const tfo_numerics& nu, const double* P, int64_t i, double* g /*[18][2]*/,
               double* phi /*[18]*/) {
  const int32_t b = m.st_ptr[i], e = m.st_ptr[i + 1];
  for (int v = 0; v < NEQ; ++v) {
    const double Pi = P[NEQ * i + v];
    double a11 = 0, a12 = 0, a22 = 0, b1 = 0, b2 = 0;
    double umax = Pi, umin = Pi;
    for (int32_t q = b; q < e; ++q) {
      const int32_t j = m.st_idx[q];
      const double dx = m.st_d[2 * q], dy = m.st_d[2 * q + 1];
      const double w = std::pow(dx * dx + dy * dy, -0.5 * nu.lsq_weight_power);
      const double dP = P[NEQ * (int64_t)j + v] - Pi;
      a11 += w * dx * dx;
      a12 += w * dx * dy;
      a22 += w * dy * dy;
      b1 += w * dx * dP;
      b2 += w * dy * dP;
      umax = std::max(umax, P[NEQ * (int64_t)j + v]);
      umin = std::min(umin, P[NEQ * (int64_t)j + v]);
    }
    const double det = a11 * a22 - a12 * a12;
    const double tr = a11 + a22;
    double gx = 0.0, gy = 0.0;
    if (det > 1e-12 * tr * tr) {
      gx = (a22 * b1 - a12 * b2) / det;
      gy = (a11 * b2 - a12 * b1) / det;
    }
    g[2 * v] = gx;
    g[2 * v + 1] = gy;
    // Venkatakrishnan (L208, S13)
    const double h = std::sqrt(m.vol[i]);
    const double Kh = nu.venkat_K * h;
    const double eps2 = Kh * Kh * Kh;
    double ph_i = 1.0;
    for (int k = 0; k < m.nv(i); ++k) {
      const double d2 = gx * m.fmid_off[2 * (m.cptr[i] + k)] + gy * m.fmid_off[2 * (m.cptr[i] + k) + 1];
      double pf = 1.0;
      if (d2 != 0.0) {
        const double d1 = d2 > 0.0 ? umax - Pi : umin - Pi;
        pf = (d1 * d1 + eps2 + 2.0 * d1 * d2) / (d1 * d1 + 2.0 * d2 * d2 + d1 * d2 + eps2);
      }
      ph_i = std::min(ph_i, pf);
    }
    phi[v] = std::min(1.0, ph_i);
  }
}

// EXTRAPOLATEONFACE of Alg. 1 (L232): P_face = P_i + phi_i (grad P_i . (x_f - x_i))
inline void extrapolate(const double* Pc, const double* g, const double* phi, double dx, double dy,
                        double* Pf) {
  for (int v = 0; v < NEQ; ++v) Pf[v] = Pc[v] + phi[v] * (g[2 * v] * dx + g[2 * v + 1] * dy);
}

inline int local_face(const tfo_mesh& m, int64_t cell, int32_t f) {
  for (int k = 0; k < m.nv(cell); ++k)
    if (m.cell_faces[m.cptr[cell] + k] == f) return k;
  return -1;
}

// Ghost state of a perfectly conducting slip wall (reading S24): the mirror image of the inner state, so that
// the face mean has B.n = 0, E_tangential = 0 and u_s.n = 0.  Vectors that must vanish normally flip their
// normal component (B, u_s); E flips its tangential components (z included); of each cleaning pair
// (B_n, Psi), (E_n, Phi) one member flips and the other is kept; rho_s and T_s are kept.
void wall_ghost(const double* P, double nx, double ny, double* G) {
  for (int v = 0; v < NEQ; ++v) G[v] = P[v];
  const double Bn = P[0] * nx + P[1] * ny;
  G[0] = P[0] - 2.0 * Bn * nx;
  G[1] = P[1] - 2.0 * Bn * ny;
  const double En = P[3] * nx + P[4] * ny;
  G[3] = -P[3] + 2.0 * En * nx;
  G[4] = -P[4] + 2.0 * En * ny;
  G[5] = -P[5];
  G[7] = -P[7];
  for (int s = 0; s < 2; ++s) {
    const double un = P[i_u(s)] * nx + P[i_u(s) + 1] * ny;
    G[i_u(s)] = P[i_u(s)] - 2.0 * un * nx;
    G[i_u(s) + 1] = P[i_u(s) + 1] - 2.0 * un * ny;
  }
}

// The boundary loop of L260: the state on the far side of boundary face f, given the reconstructed inner state.
//   TFO_BC_TRANSMISSIVE  P_R := P_L                                        (S9)
//   TFO_BC_GHOST         P_R := the caller's ghost state of that face      (does not move with P_L)
//   TFO_BC_WALL          P_R := wall_ghost(P_L, n)                         (S24)
void boundary_state(const tfo_mesh& m, int32_t f, const double* PL, double nx, double ny, double* PR) {
  const int32_t b = m.bface_of[f];
  const int tag = m.bc_tag[b];
  if (tag == TFO_BC_GHOST) for (int v = 0; v < NEQ; ++v) PR[v] = m.ghost[(size_t)NEQ * b + v];
  else if (tag == TFO_BC_WALL) wall_ghost(PL, nx, ny, PR);
  else for (int v = 0; v < NEQ; ++v) PR[v] = PL[v];
}

// perturbation size (S7): eps_k = delta * max(|P_cell,k|, ref_k), made representable
inline double fd_eps(const tfo_numerics& nu, double Pk, int k, double* Pk_pert) {
  const double e = nu.fd_delta * std::max(std::fabs(Pk), nu.fd_ref[k]);
  const double t = Pk + e;
  *Pk_pert = t;
  return t - Pk;
}

struct GradSource {
  // frozen gradient / limiter: either precomputed arrays or computed on demand for a row subset
  const double* grad = nullptr;   // [nc][18][2]
  const double* phi = nullptr;    // [nc][18]
};

// One row of Alg. 1 for cell i.  rhs_row[18], scale_row[18], blocks: the row's [18][18] blocks in BSR order.
void assemble_row(const tfo_mesh& m, const tfo_physics& ph, const tfo_numerics& nu, const double* P,
                  const double* Pn, const double* Pnm1, double dt, int64_t i, const double* g_all,
                  const double* phi_all, const int32_t* gmap /*cell -> slot in g_all or NULL*/,
                  double* rhs_row, double* scale_row, double* blocks /*or NULL*/) {
  auto slot = [&](int64_t c) -> int64_t { return gmap ? gmap[c] : c; };
  double Rt[NEQ], A[NEQ];
  for (int r = 0; r < NEQ; ++r) Rt[r] = A[r] = 0.0;
  const int32_t rb = m.bsr_rowptr[i], re = m.bsr_rowptr[i + 1];
  const int nblk = re - rb;
  if (blocks)
    for (int q = 0; q < nblk * NEQ * NEQ; ++q) blocks[q] = 0.0;
  auto block_of = [&](int32_t col) -> double* {
    for (int32_t q = rb; q < re; ++q)
      if (m.bsr_col[q] == col) return blocks + (int64_t)(q - rb) * NEQ * NEQ;
    return nullptr;
  };
  const bool do_flux = nu.term_mask & 1, do_src = nu.term_mask & 2, do_time = nu.term_mask & 4;
  const double vol = m.vol[i];

  // ---- loop over the faces of the cell (L230-244) ----
  if (do_flux)
    for (int k = 0; k < m.nv(i); ++k) {
      const int32_t f = m.cell_faces[m.cptr[i] + k];
      const int64_t cL = m.face_cells[2 * f], cR = m.face_cells[2 * f + 1];
      const bool own_is_L = (cL == i);
      const double s_if = own_is_L ? 1.0 : -1.0;
      const int kL = local_face(m, cL, f);
      // normal, length and midpoint offset from the L cell; R's offset from R's own corners
      const int64_t eL = m.cptr[cL] + kL;
      const double nx = m.fnrm[2 * eL], ny = m.fnrm[2 * eL + 1];
      const double len = m.flen[eL];
      const double dLx = m.fmid_off[2 * eL], dLy = m.fmid_off[2 * eL + 1];
      double dRx = 0, dRy = 0;
      if (cR >= 0) {
        const int64_t eR = m.cptr[cR] + local_face(m, cR, f);
        dRx = m.fmid_off[2 * eR];
        dRy = m.fmid_off[2 * eR + 1];
      }
      const double* gL = g_all + slot(cL) * NEQ * 2;
      const double* phL = phi_all + slot(cL) * NEQ;
      const double* gR = cR >= 0 ? g_all + slot(cR) * NEQ * 2 : nullptr;
      const double* phR = cR >= 0 ? phi_all + slot(cR) * NEQ : nullptr;
      double PL[NEQ], PR[NEQ], H[NEQ];
      extrapolate(P + NEQ * cL, gL, phL, dLx, dLy, PL);
      if (cR >= 0) extrapolate(P + NEQ * cR, gR, phR, dRx, dRy, PR);
      else boundary_state(m, f, PL, nx, ny, PR);                  // boundary face (L260; S9, S24)
      face_flux(ph, nu, PL, PR, nx, ny, H);
      for (int r = 0; r < NEQ; ++r) {
        Rt[r] += s_if * H[r] * len;
        A[r] += std::fabs(H[r] * len);
      }
      if (!blocks) continue;
      // perturb every variable of the L cell, then of the R cell (L235-243); frozen grad, phi (S8)
      for (int side = 0; side < 2; ++side) {
        const int64_t cX = side == 0 ? cL : cR;
        if (cX < 0) continue;
        double* blk = block_of((int32_t)cX);
        for (int v = 0; v < NEQ; ++v) {
          double Pc[NEQ], PLp[NEQ], PRp[NEQ], Hp[NEQ];
          for (int q = 0; q < NEQ; ++q) Pc[q] = P[NEQ * cX + q];
          const double eps = fd_eps(nu, Pc[v], v, &Pc[v]);
          if (side == 0) {
            extrapolate(Pc, gL, phL, dLx, dLy, PLp);
            if (cR >= 0) for (int q = 0; q < NEQ; ++q) PRp[q] = PR[q];
            else boundary_state(m, f, PLp, nx, ny, PRp);          // boundary: the far side follows its rule
          } else {
            for (int q = 0; q < NEQ; ++q) PLp[q] = PL[q];
            extrapolate(Pc, gR, phR, dRx, dRy, PRp);
          }
          face_flux(ph, nu, PLp, PRp, nx, ny, Hp);
          for (int r = 0; r < NEQ; ++r) blk[r * NEQ + v] += s_if * len * ((Hp[r] - H[r]) / eps);
        }
      }
    }
  double* diag = blocks ? block_of((int32_t)i) : nullptr;
  // ---- source (L245-253): one-point rule with the cell-centred value (L12) ----
  if (do_src) {
    double S[NEQ];
    source(ph, P + NEQ * i, S);
    for (int r = 0; r < NEQ; ++r) {
      Rt[r] -= S[r] * vol;
      A[r] += std::fabs(S[r] * vol);
    }
    if (blocks)
      for (int v = 0; v < NEQ; ++v) {
        double Pc[NEQ], Sp[NEQ];
        for (int q = 0; q < NEQ; ++q) Pc[q] = P[NEQ * i + q];
        const double eps = fd_eps(nu, Pc[v], v, &Pc[v]);
        source(ph, Pc, Sp);
        for (int r = 0; r < NEQ; ++r) diag[r * NEQ + v] -= vol * ((Sp[r] - S[r]) / eps);
      }
  }
  // ---- BDF2 time term (Eq. 13), Jacobian analytic (S15) ----
  if (do_time) {
    double U[NEQ], Un[NEQ], Unm1[NEQ];
    cons(ph, P + NEQ * i, U);
    cons(ph, Pn + NEQ * i, Un);
    cons(ph, Pnm1 + NEQ * i, Unm1);
    const double f = vol / (2.0 * dt);
    for (int r = 0; r < NEQ; ++r) {
      Rt[r] += f * (3.0 * U[r] - 4.0 * Un[r] + Unm1[r]);
      A[r] += f * (3.0 * std::fabs(U[r]) + 4.0 * std::fabs(Un[r]) + std::fabs(Unm1[r]));
    }
    if (blocks) {
      double D[NEQ * NEQ];
      dcons_dprim(ph, P + NEQ * i, D);
      for (int q = 0; q < NEQ * NEQ; ++q) diag[q] += 3.0 * f * D[q];
    }
  }
  for (int r = 0; r < NEQ; ++r) {
    rhs_row[r] = -Rt[r];   // Eq. 14 (L123): J dP = -R~
    if (scale_row) scale_row[r] = A[r];
  }
}

}  // namespace

// ==========================================================================================
// C entry points
// ==========================================================================================
extern "C" {

const char* tfo_last_error(void) { return g_err.c_str(); }

int tfo_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

#ifdef TFO_COUNT_OPS
#undef double
// out[0..6] = additions (incl. subtractions), multiplications, divisions, square roots, pow calls, comparisons,
// sign operations (fabs, negation) of the calling thread since the last reset
void tfo_opcount_get(int64_t* out) { for (int q = 0; q < tfo_count::N; ++q) out[q] = tfo_count::ops[q]; }
void tfo_opcount_reset(void) { for (int q = 0; q < tfo_count::N; ++q) tfo_count::ops[q] = 0; }
#define double tfo_count::real
#endif

void tfo_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

void tfo_default_physics(tfo_physics* p) {
  p->gamma_gas = 5.0 / 3.0;
  p->mass_ratio = 25.0;
  p->c = 20.0;
  p->gamma_psi = 1.0;
  p->chi_phi = 1.0;
  p->rusanov_alpha = 1.0;
}

void tfo_default_numerics(tfo_numerics* n, const tfo_physics* p) {
  n->fd_delta = 1e-6;
  for (int k = 0; k < NEQ; ++k) n->fd_ref[k] = 1.0;
  n->fd_ref[9] = 1.0 / p->mass_ratio;   // rho_e scale (S7)
  n->venkat_K = 1.0;
  n->lsq_weight_power = 2.0;
  n->ausm_Kp = 0.25;
  n->ausm_Ku = 0.75;
  n->ausm_sigma = 1.0;
  n->ausm_beta = 0.125;
  n->ausm_Minf[0] = n->ausm_Minf[1] = 0.1;
  n->term_mask = 7;
  n->pad_ = 0;
}

static int create_common(tfo_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                         const int32_t* cell_ptr /*NULL: triangles*/, const int32_t* cell_nodes,
                         const double* cell_xy) {
  if (!out || !cell_nodes || n_cells < 0 || n_nodes < 0 || (!node_xy && !cell_xy))
    return fail(-1, "tfo_mesh_create: bad argument");
  tfo_mesh* m = new tfo_mesh;
  m->nn = n_nodes;
  m->nc = n_cells;
  m->cptr.resize(n_cells + 1);
  for (int64_t i = 0; i <= n_cells; ++i) m->cptr[i] = cell_ptr ? cell_ptr[i] : (int32_t)(3 * i);
  if (m->cptr[0] != 0) { delete m; return fail(-1, "cell_ptr must start at 0"); }
  for (int64_t i = 0; i < n_cells; ++i)
    if (m->cptr[i + 1] - m->cptr[i] < 3 || m->cptr[i + 1] - m->cptr[i] > TFO_MAXV) {
      delete m;
      return fail(-2, "cell " + std::to_string(i) + " must have 3 or 4 corners");
    }
  const int64_t ncorn = m->cptr[n_cells];
  if (node_xy) m->node_xy.assign(node_xy, node_xy + 2 * n_nodes);
  m->cell_nodes.assign(cell_nodes, cell_nodes + ncorn);
  if (cell_xy) m->cell_xy.assign(cell_xy, cell_xy + 2 * ncorn);
  else {
    m->cell_xy.resize(2 * ncorn);
    for (int64_t i = 0; i < ncorn; ++i) {
      int32_t v = cell_nodes[i];
      if (v < 0 || v >= n_nodes) { delete m; return fail(-2, "node id out of range"); }
      m->cell_xy[2 * i] = node_xy[2 * v];
      m->cell_xy[2 * i + 1] = node_xy[2 * v + 1];
    }
  }
  m->perm.resize(n_cells);
  for (int64_t i = 0; i < n_cells; ++i) m->perm[i] = (int32_t)i;
  int rc = build(*m);
  if (rc) { delete m; return rc; }
  *out = m;
  return 0;
}

int tfo_mesh_create(tfo_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                    const int32_t* cell_nodes, const double* cell_xy) {
  return create_common(out, n_nodes, node_xy, n_cells, nullptr, cell_nodes, cell_xy);
}

int tfo_mesh_create_poly(tfo_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells,
                         const int32_t* cell_ptr, const int32_t* cell_nodes, const double* cell_xy) {
  if (!cell_ptr) return fail(-1, "tfo_mesh_create_poly: cell_ptr missing");
  return create_common(out, n_nodes, node_xy, n_cells, cell_ptr, cell_nodes, cell_xy);
}

int tfo_mesh_reorder(tfo_mesh* m, int kind, const int32_t* user_perm) {
  if (!m) return fail(-1, "null mesh");
  if (kind == 0) return 0;
  std::vector<int32_t> p;
  if (kind == 1) p = rcm_order(*m);
  else if (kind == 2) {
    if (!user_perm) return fail(-1, "user permutation missing");
    p.assign(user_perm, user_perm + m->nc);
    std::vector<char> hit(m->nc, 0);
    for (int64_t i = 0; i < m->nc; ++i) {
      if (p[i] < 0 || p[i] >= m->nc || hit[p[i]]) return fail(-1, "user permutation is not a bijection");
      hit[p[i]] = 1;
    }
  } else return fail(-1, "unknown reorder kind");
  std::vector<int32_t> cp(m->nc + 1, 0), cn, pm(m->nc);
  std::vector<double> cx;
  cn.reserve(m->cell_nodes.size());
  cx.reserve(m->cell_xy.size());
  for (int64_t i = 0; i < m->nc; ++i) {
    const int64_t o = p[i];
    for (int32_t q = m->cptr[o]; q < m->cptr[o + 1]; ++q) {
      cn.push_back(m->cell_nodes[q]);
      cx.push_back(m->cell_xy[2 * q]);
      cx.push_back(m->cell_xy[2 * q + 1]);
    }
    cp[i + 1] = (int32_t)cn.size();
    pm[i] = m->perm[o];
  }
  m->cptr.swap(cp);
  m->cell_nodes.swap(cn);
  m->cell_xy.swap(cx);
  m->perm.swap(pm);
  return build(*m);   // faces keep their ids (they are numbered by node pair), so the boundary tags stay valid
}

int tfo_mesh_info(const tfo_mesh* m, int32_t* max_faces, int64_t* n_bfaces) {
  if (!m) return fail(-1, "null mesh");
  if (max_faces) *max_faces = m->maxf;
  if (n_bfaces) *n_bfaces = (int64_t)m->bfaces.size();
  return 0;
}

int tfo_mesh_set_bc(tfo_mesh* m, const int32_t* tags, const double* ghost) {
  if (!m || !tags) return fail(-1, "null argument");
  const size_t nb = m->bfaces.size();
  bool need_ghost = false;
  for (size_t b = 0; b < nb; ++b) {
    if (tags[b] < 0 || tags[b] > TFO_BC_WALL) return fail(-1, "unknown boundary tag");
    need_ghost |= tags[b] == TFO_BC_GHOST;
  }
  if (need_ghost && !ghost) return fail(-1, "ghost states missing for TFO_BC_GHOST faces");
  m->bc_tag.assign(tags, tags + nb);
  if (ghost) m->ghost.assign(ghost, ghost + (size_t)NEQ * nb);
  else m->ghost.clear();
  return 0;
}

int tfo_mesh_sizes(const tfo_mesh* m, int64_t* n_cells, int64_t* n_faces, int64_t* nnzb, int64_t* n_stencil) {
  if (!m) return fail(-1, "null mesh");
  if (n_cells) *n_cells = m->nc;
  if (n_faces) *n_faces = m->nf;
  if (nnzb) *nnzb = (int64_t)m->bsr_col.size();
  if (n_stencil) *n_stencil = (int64_t)m->st_idx.size();
  return 0;
}

int tfo_mesh_get(const tfo_mesh* m, int which, void* dst, int64_t bytes) {
  if (!m || !dst) return fail(-1, "null argument");
  const void* src = nullptr;
  int64_t n = 0;
  std::vector<double> tmp;
  std::vector<int32_t> itmp;
  switch (which) {
    case TFO_FACE_CELLS: src = m->face_cells.data(); n = m->face_cells.size() * 4; break;
    case TFO_FACE_NODES: src = m->face_nodes.data(); n = m->face_nodes.size() * 4; break;
    case TFO_CELL_FACES: {   // [nc][maxf], -1 where a cell has fewer faces
      itmp.assign((size_t)m->nc * m->maxf, -1);
      for (int64_t i = 0; i < m->nc; ++i)
        for (int k = 0; k < m->nv(i); ++k) itmp[(size_t)i * m->maxf + k] = m->cell_faces[m->cptr[i] + k];
      src = itmp.data();
      n = itmp.size() * 4;
      break;
    }
    case TFO_BFACES: src = m->bfaces.data(); n = m->bfaces.size() * 4; break;
    case TFO_BC_TAGS: src = m->bc_tag.data(); n = m->bc_tag.size() * 4; break;
    case TFO_STENCIL_PTR: src = m->st_ptr.data(); n = m->st_ptr.size() * 4; break;
    case TFO_STENCIL_IDX: src = m->st_idx.data(); n = m->st_idx.size() * 4; break;
    case TFO_BSR_ROWPTR: src = m->bsr_rowptr.data(); n = m->bsr_rowptr.size() * 4; break;
    case TFO_BSR_COL: src = m->bsr_col.data(); n = m->bsr_col.size() * 4; break;
    case TFO_PERM: src = m->perm.data(); n = m->perm.size() * 4; break;
    case TFO_VOLUME: src = m->vol.data(); n = m->vol.size() * 8; break;
    case TFO_CENTROID: src = m->cen.data(); n = m->cen.size() * 8; break;
    case TFO_FACE_NORMAL_LEN: {   // [nf][3] = (nx, ny, len) taken from the L cell
      tmp.resize(3 * m->nf);
      for (int64_t f = 0; f < m->nf; ++f) {
        int64_t cL = m->face_cells[2 * f];
        int k = local_face(*m, cL, (int32_t)f);
        tmp[3 * f] = m->fnrm[2 * (m->cptr[cL] + k)];
        tmp[3 * f + 1] = m->fnrm[2 * (m->cptr[cL] + k) + 1];
        tmp[3 * f + 2] = m->flen[m->cptr[cL] + k];
      }
      src = tmp.data();
      n = tmp.size() * 8;
      break;
    }
    default: return fail(-1, "tfo_mesh_get: unknown item");
  }
  if (bytes != n) return fail(-1, "tfo_mesh_get: size mismatch, need " + std::to_string(n));
  if (n > 0) std::memcpy(dst, src, n);   // (an empty item has no storage: memcpy must not see its null pointer)
  return 0;
}

void tfo_mesh_destroy(tfo_mesh* m) { delete m; }

int tfo_gradients(const tfo_mesh* m, const tfo_numerics* nu, const double* state, double* grad, double* phi) {
  if (!m || !nu || !state || !grad || !phi) return fail(-1, "null argument");
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < m->nc; ++i) grad_cell(*m, *nu, state, i, grad + 2 * NEQ * i, phi + NEQ * i);
  return 0;
}

int tfo_assemble(const tfo_mesh* m, const tfo_physics* ph, const tfo_numerics* nu, const double* state,
                 const double* state_n, const double* state_nm1, double dt, double* rhs, double* scale,
                 double* vals, int64_t n_rows, const int32_t* rows) {
  if (!m || !ph || !nu || !state || !state_n || !state_nm1 || !rhs) return fail(-1, "null argument");
  if (!(dt > 0.0)) return fail(-1, "dt must be positive");
  const int64_t nc = m->nc;
  if (!rows) {
    std::vector<double> g(2 * NEQ * nc), phi(NEQ * nc);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < nc; ++i) grad_cell(*m, *nu, state, i, &g[2 * NEQ * i], &phi[NEQ * i]);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < nc; ++i)
      assemble_row(*m, *ph, *nu, state, state_n, state_nm1, dt, i, g.data(), phi.data(), nullptr,
                   rhs + NEQ * i, scale ? scale + NEQ * i : nullptr,
                   vals ? vals + (int64_t)m->bsr_rowptr[i] * NEQ * NEQ : nullptr);
    return 0;
  }
  // row subset: gradients only where needed (the rows and their face neighbours)
  std::vector<int32_t> gmap(nc, -1);
  std::vector<int32_t> need;
  for (int64_t r = 0; r < n_rows; ++r) {
    const int32_t i = rows[r];
    if (i < 0 || i >= nc) return fail(-1, "row out of range");
    for (int32_t q = m->bsr_rowptr[i]; q < m->bsr_rowptr[i + 1]; ++q) {
      const int32_t j = m->bsr_col[q];
      if (gmap[j] < 0) { gmap[j] = (int32_t)need.size(); need.push_back(j); }
    }
  }
  std::vector<double> g(2 * NEQ * need.size()), phi(NEQ * need.size());
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < (int64_t)need.size(); ++q)
    grad_cell(*m, *nu, state, need[q], &g[2 * NEQ * q], &phi[NEQ * q]);
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < n_rows; ++r) {
    const int64_t nb = (int64_t)(m->maxf + 1) * NEQ * NEQ;   // blocks per row, zero padded
    double* blk = vals ? vals + r * nb : nullptr;
    if (blk) for (int64_t q = 0; q < nb; ++q) blk[q] = 0.0;
    assemble_row(*m, *ph, *nu, state, state_n, state_nm1, dt, rows[r], g.data(), phi.data(), gmap.data(),
                 rhs + NEQ * r, scale ? scale + NEQ * r : nullptr, blk);
  }
  return 0;
}

int tfo_residual_frozen(const tfo_mesh* m, const tfo_physics* ph, const tfo_numerics* nu, const double* state,
                        const double* grad, const double* phi, const double* state_n, const double* state_nm1,
                        double dt, double* rhs) {
  if (!m || !ph || !nu || !state || !grad || !phi || !rhs) return fail(-1, "null argument");
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < m->nc; ++i)
    assemble_row(*m, *ph, *nu, state, state_n, state_nm1, dt, i, grad, phi, nullptr, rhs + NEQ * i, nullptr,
                 nullptr);
  return 0;
}

void tfo_flux_maxwell(const tfo_physics* ph, const double* UL, const double* UR, double nx, double ny, double* H8) {
  maxwell_flux(*ph, UL, UR, nx, ny, H8);
}
void tfo_flux_ausm(const tfo_physics* ph, const tfo_numerics* nu, int species, const double* PL5, const double* PR5,
                   double nx, double ny, double* H5) {
  ausm_flux(*ph, *nu, species, PL5, PR5, nx, ny, H5);
}
void tfo_flux_face(const tfo_physics* ph, const tfo_numerics* nu, const double* PL18, const double* PR18, double nx,
                   double ny, double* H18) {
  face_flux(*ph, *nu, PL18, PR18, nx, ny, H18);
}
// physical flux F(U).n of Eq. 3/5 (L56, L63) — what consistency (L85) compares against
void tfo_phys_flux(const tfo_physics* ph, const double* P, double nx, double ny, double* F) {
  maxwell_physical_flux(*ph, P, nx, ny, F);
  for (int s = 0; s < 2; ++s) {
    const double Rs = R_s(*ph, s), g = ph->gamma_gas;
    const double rho = P[i_rho(s)], T = P[i_T(s)];
    const double* u = P + i_u(s);
    const double un = u[0] * nx + u[1] * ny;
    const double p = rho * Rs * T;
    const double Ht = g * Rs / (g - 1.0) * T + 0.5 * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
    F[i_rho(s)] = rho * un;
    F[i_u(s)] = rho * un * u[0] + p * nx;
    F[i_u(s) + 1] = rho * un * u[1] + p * ny;
    F[i_u(s) + 2] = rho * un * u[2];
    F[i_T(s)] = rho * un * Ht;
  }
}
void tfo_ausm_split(double M, double alpha, double beta, double* o) {
  o[0] = M4p(M, beta);
  o[1] = M4m(M, beta);
  o[2] = P5p(M, alpha);
  o[3] = P5m(M, alpha);
}
void tfo_wall_ghost(const double* P18, double nx, double ny, double* G18) { wall_ghost(P18, nx, ny, G18); }
void tfo_source(const tfo_physics* ph, const double* P18, double* S18) { source(*ph, P18, S18); }
void tfo_cons(const tfo_physics* ph, const double* P18, double* U18) { cons(*ph, P18, U18); }
void tfo_dcons_dprim(const tfo_physics* ph, const double* P18, double* D) { dcons_dprim(*ph, P18, D); }

}  // extern "C"

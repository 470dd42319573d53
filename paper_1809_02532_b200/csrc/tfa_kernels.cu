// tfa_kernels.cu — steps a2..a7: gradient + limiter, and the fused residual/Jacobian assembly.
//
// Kernel design:
//  k_lsq_coef          once per (mesh, weight power): least-squares coefficient vectors c_ij so that
//                      grad P_i = sum_j c_ij (P_j - P_i)                                   (L74)
//  k_gradient_limiter  thread = (cell, variable): LS gradient + Venkatakrishnan phi      (L74, L208)
//  k_assemble          CTA = TILE cells; thread = one perturbed (or base) sub-flux evaluation
//                      (cell, species, which variable is perturbed) looping over the 3 faces;
//                      Jacobian columns are staged in shared memory and leave the SM as whole
//                      2592-byte blocks; no atomics, no memset, each face Jacobian stays on chip.
//                      Replaces Alg. 1's thread-per-cell loop (L221-256).
#include "tfa_common.cuh"
#include "tfa_physics.cuh"

namespace tfa {

// ================================================================================================
// a2: least-squares coefficients (once per mesh) and gradient + limiter (every assembly)
// ================================================================================================
__global__ void k_lsq_coef(int64_t nc, const int32_t* __restrict__ st_ptr, const double* __restrict__ st_d,
                           double power, double* __restrict__ coef) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  const int32_t b = st_ptr[i], e = st_ptr[i + 1];
  double a11 = 0, a12 = 0, a22 = 0;
  for (int32_t q = b; q < e; ++q) {
    const double dx = st_d[2 * (int64_t)q], dy = st_d[2 * (int64_t)q + 1];
    const double d2 = dx * dx + dy * dy;
    const double w = power == 2.0 ? 1.0 / d2 : pow(d2, -0.5 * power);
    a11 += w * dx * dx;
    a12 += w * dx * dy;
    a22 += w * dy * dy;
  }
  const double det = a11 * a22 - a12 * a12, tr = a11 + a22;
  const bool ok = det > 1e-12 * tr * tr;   // degenerate stencil -> zero gradient (first order)
  const double id = ok ? 1.0 / det : 0.0;
  for (int32_t q = b; q < e; ++q) {
    const double dx = st_d[2 * (int64_t)q], dy = st_d[2 * (int64_t)q + 1];
    const double d2 = dx * dx + dy * dy;
    const double w = power == 2.0 ? 1.0 / d2 : pow(d2, -0.5 * power);
    coef[2 * (int64_t)q] = id * w * (a22 * dx - a12 * dy);
    coef[2 * (int64_t)q + 1] = id * w * (a11 * dy - a12 * dx);
  }
}

constexpr int GL_CELLS = 16;               // cells per CTA
constexpr int GL_T = GL_CELLS * NEQ;       // 288 threads

// thread = (cell, variable): 18 consecutive lanes read one neighbour state (144 contiguous bytes)
__global__ void __launch_bounds__(GL_T) k_gradient_limiter(int64_t nc, const double* __restrict__ state,
                                                          const int32_t* __restrict__ st_ptr,
                                                          const int32_t* __restrict__ st_idx,
                                                          const double* __restrict__ coef,
                                                          const double* __restrict__ cgeo, double venkK,
                                                          double* __restrict__ lgrad, double* __restrict__ grad_out,
                                                          double* __restrict__ phi_out) {
  const int v = threadIdx.x % NEQ;
  const int64_t i = blockIdx.x * (int64_t)GL_CELLS + threadIdx.x / NEQ;
  if (i >= nc) return;
  const double Pi = state[NEQ * i + v];
  double gx = 0.0, gy = 0.0, umax = Pi, umin = Pi;
  const int32_t b = st_ptr[i], e = st_ptr[i + 1];
  for (int32_t q = b; q < e; ++q) {
    const int64_t j = st_idx[q];
    const double Pj = state[NEQ * j + v];
    const double dP = Pj - Pi;
    gx += coef[2 * (int64_t)q] * dP;
    gy += coef[2 * (int64_t)q + 1] * dP;
    umax = fmax(umax, Pj);
    umin = fmin(umin, Pj);
  }
  // Venkatakrishnan (L208; S13): eps^2 = (K h)^3, Delta2 sampled at the cell's three face midpoints
  const double* g = cgeo + CGEO * i;
  const double Kh = venkK * g[15];
  const double eps2 = Kh * Kh * Kh;
  double phi = 1.0;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const double d2 = gx * g[8 * k + 3] + gy * g[8 * k + 4];
    const double d1 = d2 > 0.0 ? umax - Pi : umin - Pi;
    const double num = d1 * d1 + eps2 + 2.0 * d1 * d2;
    const double den = d1 * d1 + 2.0 * d2 * d2 + d1 * d2 + eps2;
    const double pf = d2 != 0.0 ? num / den : 1.0;
    phi = fmin(phi, pf);
  }
  phi = fmin(phi, 1.0);
  if (lgrad) {
    lgrad[2 * (NEQ * i + v)] = phi * gx;
    lgrad[2 * (NEQ * i + v) + 1] = phi * gy;
  }
  if (grad_out) {
    grad_out[2 * (NEQ * i + v)] = gx;
    grad_out[2 * (NEQ * i + v) + 1] = gy;
    phi_out[NEQ * i + v] = phi;
  }
}

// ================================================================================================
// a3..a7: fused face flux + flux Jacobian + source + BDF2 + BSR write
// ================================================================================================
constexpr int TILE = 8;              // cells per CTA
constexpr int NA = 22 * TILE;        // AUSM tasks: (cell, species, {base, 5 own-side, 5 neighbour-side})
constexpr int NM = 17 * TILE;        // Maxwell tasks: (cell, {base, 8 own-side, 8 neighbour-side})
constexpr int AT = 192;              // threads per CTA (>= NA, multiple of 32)
static_assert(AT >= NA && AT >= NM, "thread count");

struct __align__(16) AsmSmem {
  double off[TILE][BLK];          // staged off-diagonal block of the current face (zeros persist)
  double diag[TILE][BLK];         // staged diagonal block
  double fbase[TILE][3][2][NEQ];  // reconstructed face states, canonical side 0 = L, 1 = R
  double fpert[TILE][3][2][NEQ];  // the same with variable v of that side's CELL perturbed
  double eps[TILE][4][NEQ];       // representable perturbation sizes: slot 0 own cell, 1..3 neighbour k
  double pc[TILE][NEQ];           // own cell-centre state
  double hbase[TILE][3][NEQ];     // base numerical flux of face k (canonical orientation)
  double fg[TILE][3][4];          // nx, ny, s_if * len, (unused)
  double vol[TILE];
  int32_t nbr[TILE][3];
  int32_t blk[TILE][4];           // BSR block index of (diag, nbr0, nbr1, nbr2); -1 if absent
};

__device__ __forceinline__ void st_global_v2(double* p, double a, double b) {
  asm volatile("st.global.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(a), "d"(b) : "memory");
}

// static-index access to the five rows/variables of species SP inside an 18-vector held in registers
template <int SP>
__device__ __forceinline__ void sp_get(const double* v18, double* v5) {
  v5[0] = v18[8 + SP];
  v5[1] = v18[10 + 3 * SP];
  v5[2] = v18[11 + 3 * SP];
  v5[3] = v18[12 + 3 * SP];
  v5[4] = v18[16 + SP];
}
template <int SP>
__device__ __forceinline__ void sp_put(double* v18, const double* v5) {
  v18[8 + SP] = v5[0];
  v18[10 + 3 * SP] = v5[1];
  v18[11 + 3 * SP] = v5[2];
  v18[12 + 3 * SP] = v5[3];
  v18[16 + SP] = v5[4];
}
// column v of (3 Omega / 2 dt) dU/dP for a species variable v (analytic, S15)
template <int SP>
__device__ __forceinline__ void time_column(const Consts& K, double* col, int v, const double* P, double ft) {
  constexpr int ir = 8 + SP, iu = 10 + 3 * SP, iT = 16 + SP;
  const double rho = P[ir], ux = P[iu], uy = P[iu + 1], uz = P[iu + 2], T = P[iT];
  if (v == ir) {
    col[ir] += ft;
    col[iu] += ft * ux;
    col[iu + 1] += ft * uy;
    col[iu + 2] += ft * uz;
    col[iT] += ft * (K.cv[SP] * T + 0.5 * (ux * ux + uy * uy + uz * uz));
  } else if (v == iT) {
    col[iT] += ft * rho * K.cv[SP];
  } else {
#pragma unroll
    for (int d = 0; d < 3; ++d)
      if (v == iu + d) {
        col[iu + d] += ft * rho;
        col[iT] += ft * rho * P[iu + d];
      }
  }
}

template <bool JAC>
__global__ void __launch_bounds__(AT, 3) k_assemble(int64_t nc, Consts K, const double* __restrict__ state,
                                                   const double* __restrict__ state_n,
                                                   const double* __restrict__ state_nm1, double inv2dt,
                                                   const double* __restrict__ lgrad,
                                                   const double* __restrict__ cgeo,
                                                   const int32_t* __restrict__ cell_nbr,
                                                   const int32_t* __restrict__ rowptr, double* __restrict__ rhs,
                                                   double* __restrict__ vals, int32_t* __restrict__ flags) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  AsmSmem& S = *reinterpret_cast<AsmSmem*>(smem_raw);
  const int tid = threadIdx.x;
  const int64_t cell0 = blockIdx.x * (int64_t)TILE;
  const bool do_flux = K.mask & 1, do_src = K.mask & 2, do_time = K.mask & 4;

  // ---- phase 0: topology of the tile, zero the off-diagonal staging ----
  if (tid < TILE) {
    const int64_t i = cell0 + tid;
    int32_t n[3] = {-1, -1, -1};
    if (i < nc) {
#pragma unroll
      for (int k = 0; k < 3; ++k) n[k] = cell_nbr[3 * i + k];
      const int32_t base = rowptr[i];
      const int32_t c[4] = {(int32_t)i, n[0], n[1], n[2]};
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        int rank = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b) rank += (c[b] >= 0 && c[b] < c[a]);
        S.blk[tid][a] = c[a] >= 0 ? base + rank : -1;
      }
      S.vol[tid] = cgeo[CGEO * i + 7];
    } else {
#pragma unroll
      for (int a = 0; a < 4; ++a) S.blk[tid][a] = -1;
      S.vol[tid] = 0.0;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) S.nbr[tid][k] = n[k];
  }
  if (tid < TILE * 3) {
    const int cl = tid / 3, k = tid % 3;
    const int64_t i = cell0 + cl;
    if (i < nc) {
      const double* g = cgeo + CGEO * i + 8 * k;
      const int32_t j = cell_nbr[3 * i + k];
      const bool own_is_L = j < 0 || i < j;
      S.fg[cl][k][0] = g[0];
      S.fg[cl][k][1] = g[1];
      S.fg[cl][k][2] = own_is_L ? g[2] : -g[2];
    }
  }
  if (JAC)
    for (int q = tid; q < TILE * BLK; q += AT) (&S.off[0][0])[q] = 0.0;

  // ---- phase A: reconstruct L/R face states and their perturbed counterparts (Alg. 1)
  for (int q = tid; q < TILE * 3 * 2 * NEQ; q += AT) {
    const int cl = q / (6 * NEQ), rem = q % (6 * NEQ);
    const int k = rem / (2 * NEQ), side = (rem / NEQ) % 2, v = rem % NEQ;
    const int64_t i = cell0 + cl;
    if (i >= nc) continue;
    const int32_t j = cell_nbr[3 * i + k];
    const bool own_is_L = j < 0 || i < j;
    const bool is_own = (j < 0) || (side == (own_is_L ? 0 : 1));   // boundary: P_R := P_L (S9)
    const int64_t X = is_own ? i : j;
    const double* g = cgeo + CGEO * i + 8 * k;
    const double dx = is_own ? g[3] : g[5], dy = is_own ? g[4] : g[6];
    const double Pc = state[NEQ * X + v];
    const double inc = lgrad[2 * (NEQ * X + v)] * dx + lgrad[2 * (NEQ * X + v) + 1] * dy;
    S.fbase[cl][k][side][v] = Pc + inc;
    // eps_k = delta * max(|P_cell,k|, ref_k), made representable (S7)
    const double t = Pc + K.delta * fmax(fabs(Pc), K.ref[v]);
    S.fpert[cl][k][side][v] = t + inc;
    const double e = t - Pc;
    if (is_own) {
      if (k == 0 && (side == 0 || j >= 0)) { S.eps[cl][0][v] = e; S.pc[cl][v] = Pc; }
    } else {
      S.eps[cl][1 + k][v] = e;
    }
  }
  __syncthreads();

  // ---- task decoding ----
  // AUSM task: a_cl cell, a_s species, a_p: 0 base, 1..5 own-side variable, 6..10 neighbour-side
  const bool a_on = tid < NA && cell0 + tid / 22 < nc;
  const int a_cl = a_on ? tid / 22 : 0, a_s = (tid % 22) / 11, a_p = tid % 11;
  const int a_j = a_p == 0 ? 0 : (a_p - 1) % 5;
  const int a_v = sp_idx(a_s, a_j);   // the variable this task perturbs
  int a_idx[5];
#pragma unroll
  for (int j = 0; j < 5; ++j) a_idx[j] = sp_idx(a_s, j);
  // Maxwell task: m_cl cell, m_p: 0 base, 1..8 own-side variable, 9..16 neighbour-side
  const bool m_on = tid < NM && cell0 + tid / 17 < nc;
  const int m_cl = m_on ? tid / 17 : 0, m_p = tid % 17;
  const int m_v = m_p == 0 ? 0 : (m_p - 1) % 8;

  double accA[5] = {0, 0, 0, 0, 0};                 // base: residual rows; own-side: diagonal column
  double accM[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  bool nonphys = false;

  // ---- phase B: faces (Alg. 1) ----
#pragma unroll 1
  for (int k = 0; k < 3; ++k) {
    double Ha[5], Hm[8];
    bool a_act = false, m_act = false;
    if (do_flux && a_on) {
      const int32_t j = S.nbr[a_cl][k];
      const bool own_is_L = S.fg[a_cl][k][2] > 0.0;
      const int own_side = own_is_L ? 0 : 1;
      const bool nbr_task = a_p >= 6;
      a_act = JAC ? !(nbr_task && j < 0) : a_p == 0;
      if (a_act) {
        double L[5], R[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          L[q] = S.fbase[a_cl][k][0][a_idx[q]];
          R[q] = S.fbase[a_cl][k][1][a_idx[q]];
        }
        if (a_p != 0) {
          const int side = nbr_task ? 1 - own_side : own_side;
          const double pv = S.fpert[a_cl][k][side][a_v];
          const bool both = j < 0;   // boundary: the perturbation moves both arguments (S9)
#pragma unroll
          for (int q = 0; q < 5; ++q)
            if (q == a_j) {
              if (side == 0 || both) L[q] = pv;
              if (side == 1 || both) R[q] = pv;
            }
        }
        const bool ok = ausm_flux(K, a_s, L, R, S.fg[a_cl][k][0], S.fg[a_cl][k][1], Ha);
        if (a_p == 0) {
          nonphys |= !ok;
          const double sl = S.fg[a_cl][k][2];
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            S.hbase[a_cl][k][a_idx[q]] = Ha[q];
            accA[q] += sl * Ha[q];
          }
        }
      }
    }
    if (do_flux && m_on) {
      const int32_t j = S.nbr[m_cl][k];
      const bool own_is_L = S.fg[m_cl][k][2] > 0.0;
      const int own_side = own_is_L ? 0 : 1;
      const bool nbr_task = m_p >= 9;
      m_act = JAC ? !(nbr_task && j < 0) : m_p == 0;
      if (m_act) {
        double L[8], R[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          L[q] = S.fbase[m_cl][k][0][q];
          R[q] = S.fbase[m_cl][k][1][q];
        }
        if (m_p != 0) {
          const int side = nbr_task ? 1 - own_side : own_side;
          const double pv = S.fpert[m_cl][k][side][m_v];
          const bool both = j < 0;
#pragma unroll
          for (int q = 0; q < 8; ++q)
            if (q == m_v) {
              if (side == 0 || both) L[q] = pv;
              if (side == 1 || both) R[q] = pv;
            }
        }
        maxwell_flux(K, L, R, S.fg[m_cl][k][0], S.fg[m_cl][k][1], Hm);
        if (m_p == 0) {
          const double sl = S.fg[m_cl][k][2];
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            S.hbase[m_cl][k][q] = Hm[q];
            accM[q] += sl * Hm[q];
          }
        }
      }
    }
    if (!JAC) continue;
    __syncthreads();
    // derivative columns (L239-241): (H_pert - H) / eps * s_if * Sigma
    if (a_act && a_p != 0) {
      const bool nbr_task = a_p >= 6;
      const double e = S.eps[a_cl][nbr_task ? 1 + k : 0][a_v];
      const double f = S.fg[a_cl][k][2] / e;
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        const double d = (Ha[q] - S.hbase[a_cl][k][a_idx[q]]) * f;
        if (nbr_task) S.off[a_cl][a_idx[q] * NEQ + a_v] = d;
        else accA[q] += d;
      }
    }
    if (m_act && m_p != 0) {
      const bool nbr_task = m_p >= 9;
      const double e = S.eps[m_cl][nbr_task ? 1 + k : 0][m_v];
      const double f = S.fg[m_cl][k][2] / e;
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const double d = (Hm[q] - S.hbase[m_cl][k][q]) * f;
        if (nbr_task) S.off[m_cl][q * NEQ + m_v] = d;
        else accM[q] += d;
      }
    }
    __syncthreads();
    // a7: the off-diagonal block of face k leaves the SM as one contiguous 2592-byte block
    for (int q = tid; q < TILE * (BLK / 2); q += AT) {
      const int cl = q / (BLK / 2), w = q % (BLK / 2);
      const int32_t b = S.blk[cl][1 + k];
      if (b >= 0) st_global_v2(vals + (int64_t)b * BLK + 2 * w, S.off[cl][2 * w], S.off[cl][2 * w + 1]);
    }
  }
  if (nonphys) atomicAdd(flags, 1);

  // ---- phase C: source (L245-253), BDF2 time term (Eq. 13), residual and diagonal block ----
  // residual rows: the base tasks own them (AUSM base: 5 species rows, Maxwell base: rows 0..7)
  if (a_on && a_p == 0) {
    const int64_t i = cell0 + a_cl;
    const double vol = S.vol[a_cl];
    double Ssrc[NEQ], S5[5];
    source_terms(K, S.pc[a_cl], Ssrc);
    if (a_s == 0) sp_get<0>(Ssrc, S5);
    else sp_get<1>(Ssrc, S5);
    double Q[5], Qn[5], Qm[5], U[5], Un[5], Um[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      Q[q] = S.pc[a_cl][a_idx[q]];
      Qn[q] = state_n[NEQ * i + a_idx[q]];
      Qm[q] = state_nm1[NEQ * i + a_idx[q]];
    }
    cons_species(K, a_s, Q, U);
    cons_species(K, a_s, Qn, Un);
    cons_species(K, a_s, Qm, Um);
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      double r = accA[q];
      if (do_src) r -= S5[q] * vol;
      if (do_time) r += vol * inv2dt * (3.0 * U[q] - 4.0 * Un[q] + Um[q]);
      rhs[NEQ * i + a_idx[q]] = -r;
    }
  }
  if (m_on && m_p == 0) {
    const int64_t i = cell0 + m_cl;
    const double vol = S.vol[m_cl];
    double Ssrc[NEQ];
    source_terms(K, S.pc[m_cl], Ssrc);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      double r = accM[q];
      if (do_src) r -= Ssrc[q] * vol;
      if (do_time) r += vol * inv2dt * (3.0 * S.pc[m_cl][q] - 4.0 * state_n[NEQ * i + q] + state_nm1[NEQ * i + q]);
      rhs[NEQ * i + q] = -r;
    }
  }
  if (!JAC) return;
  // diagonal block columns: own-side tasks (AUSM: variable a_idx[a_j]; Maxwell: variable m_v)
  const bool a_diag = a_on && a_p >= 1 && a_p <= 5;
  const bool m_diag = m_on && m_p >= 1 && m_p <= 8;
#pragma unroll 1
  for (int pass = 0; pass < 2; ++pass) {
    const bool on = pass == 0 ? a_diag : m_diag;
    if (!on) continue;
    const int cl = pass == 0 ? a_cl : m_cl;
    const int v = pass == 0 ? a_v : m_v;
    const double vol = S.vol[cl];
    double col[NEQ];
#pragma unroll
    for (int r = 0; r < NEQ; ++r) col[r] = 0.0;
    if (pass == 0) {
      if (a_s == 0) sp_put<0>(col, accA);
      else sp_put<1>(col, accA);
    } else {
#pragma unroll
      for (int q = 0; q < 8; ++q) col[q] = accM[q];
    }
    double P[NEQ];
#pragma unroll
    for (int r = 0; r < NEQ; ++r) P[r] = S.pc[cl][r];
    if (do_src) {
      double S0[NEQ], S1[NEQ];
      source_terms(K, P, S0);
      const double e = S.eps[cl][0][v];
      double Pp[NEQ];
#pragma unroll
      for (int r = 0; r < NEQ; ++r) Pp[r] = r == v ? P[r] + e : P[r];
      source_terms(K, Pp, S1);
      const double f = vol / e;
#pragma unroll
      for (int r = 0; r < NEQ; ++r) col[r] -= (S1[r] - S0[r]) * f;
    }
    if (do_time) {
      // analytic dU/dP (S15): identity on the field rows; species rows below
      const double ft = 3.0 * vol * inv2dt;
      if (pass == 1) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
          if (r == v) col[r] += ft;
      } else if (a_s == 0) time_column<0>(K, col, v, P, ft);
      else time_column<1>(K, col, v, P, ft);
    }
#pragma unroll
    for (int r = 0; r < NEQ; ++r) S.diag[cl][r * NEQ + v] = col[r];
  }
  __syncthreads();
  for (int q = tid; q < TILE * (BLK / 2); q += AT) {
    const int cl = q / (BLK / 2), w = q % (BLK / 2);
    const int32_t b = S.blk[cl][0];
    if (b >= 0) st_global_v2(vals + (int64_t)b * BLK + 2 * w, S.diag[cl][2 * w], S.diag[cl][2 * w + 1]);
  }
}

// ================================================================================================
// probes: roofline denominators measured in the same run
// ================================================================================================
__global__ void __launch_bounds__(256) k_probe_dfma(int iters, double* sink) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6,
         a7 = a0 + 7;
  const double b = 1.0000001, c = 1e-9;
  for (int it = 0; it < iters; ++it) {
    a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
    a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
  }
  const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) sink[0] = s;   // never true; keeps the loop alive
}

__global__ void __launch_bounds__(256) k_probe_copy(const double2* __restrict__ src, double2* __restrict__ dst,
                                                    int64_t n2) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n2; i += stride) dst[i] = src[i];
}

// ================================================================================================
// host-side launchers used by tfa_api.cu
// ================================================================================================
int launch_lsq_coef(const tfa_mesh& m, double power, double* coef, cudaStream_t st) {
  if (m.nc == 0) return 0;
  k_lsq_coef<<<cdiv(m.nc, 128), 128, 0, st>>>(m.nc, m.st_ptr.p, m.st_d.p, power, coef);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

int launch_gradient(const tfa_mesh& m, const double* state, const double* coef, double venkK, double* lgrad,
                    double* grad, double* phi, cudaStream_t st) {
  if (m.nc == 0) return 0;
  k_gradient_limiter<<<cdiv(m.nc, GL_CELLS), GL_T, 0, st>>>(m.nc, state, m.st_ptr.p, m.st_idx.p, coef, m.cgeo.p,
                                                           venkK, lgrad, grad, phi);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

int launch_assemble(const tfa_mesh& m, const Consts& K, const double* state, const double* state_n,
                    const double* state_nm1, double dt, const double* lgrad, double* rhs, double* vals,
                    int32_t* flags, cudaStream_t st) {
  if (m.nc == 0) return 0;
  static bool attr_done = false;
  const int smem = (int)sizeof(AsmSmem);
  if (!attr_done) {
    TFA_CUDA(cudaFuncSetAttribute(k_assemble<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    TFA_CUDA(cudaFuncSetAttribute(k_assemble<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    attr_done = true;
  }
  const unsigned grid = cdiv(m.nc, TILE);
  const double inv2dt = 1.0 / (2.0 * dt);
  if (vals)
    k_assemble<true><<<grid, AT, smem, st>>>(m.nc, K, state, state_n, state_nm1, inv2dt, lgrad, m.cgeo.p,
                                             m.cell_nbr.p, m.bsr_rowptr.p, rhs, vals, flags);
  else
    k_assemble<false><<<grid, AT, smem, st>>>(m.nc, K, state, state_n, state_nm1, inv2dt, lgrad, m.cgeo.p,
                                              m.cell_nbr.p, m.bsr_rowptr.p, rhs, vals, flags);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

int launch_probe_dfma(int grid, int iters, double* sink, cudaStream_t st) {
  k_probe_dfma<<<grid, 256, 0, st>>>(iters, sink);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

int launch_probe_copy(const double* src, double* dst, int64_t n, cudaStream_t st) {
  k_probe_copy<<<148 * 16, 256, 0, st>>>((const double2*)src, (double2*)dst, n / 2);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

}  // namespace tfa

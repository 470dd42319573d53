// tfa_assemble.cu — steps a3..a7 fused: face flux + flux Jacobian + source + BDF2 + BSR write.
//
// Design, replacing Alg. 1's thread-per-cell loop (L221-256):
//
//  * A persistent CTA walks tiles of T consecutive cells.  Cell i evaluates, for each of its three
//    faces, the base numerical flux and the fluxes with each variable of ITS OWN side perturbed
//    (Alg. 1).  The column (H_pert - H)/eps * s_if * Sigma_f is (a) accumulated into the
//    diagonal block (i,i) and (b) written, negated, as the block (j,i) of the NEIGHBOUR's row:
//    s_jf = -s_if, so d R_j / d P_i through the shared face is exactly minus cell i's own
//    contribution (same inputs, same code, bit-identical).  Every BSR block has exactly one
//    writer (cell i writes (i,i) and the (j,i)), so there are no atomics, no memset, and the
//    perturbed fluxes towards the other side are never evaluated: 6+6+9 = 21 flux evaluations per
//    cell-face instead of Alg. 1's 3*19 = 57 full ones.
//  * Lanes: an AUSM warp holds 5 groups of 6 lanes = (cell, species) x {base, 5 perturbed variables}
//    (Eq. 10); a Maxwell warp holds 3 groups of 9 lanes = cell x {base, 8 perturbed} (Eq. 9
//    L91).  The base flux reaches the group by warp shuffle; the flux Jacobian is block diagonal
//    (8x8, 5x5, 5x5), the source (Eq. 4/6) couples the blocks on the diagonal block only.
//  * 18x18 blocks are staged in shared memory (the structural zeros of the mirror blocks are
//    written once per CTA) and leave the SM as 2592-byte TMA bulk stores
//    (cp.async.bulk.global.shared::cta), rhs as one bulk store per tile.
#include "tfa_common.cuh"
#include "tfa_physics.cuh"

namespace tfa {

// ------------------------------------------------------------------------------------------------
// TMA bulk-store helpers (PTX ISA: cp.async.bulk, bulk async-groups, async proxy fence)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void bulk_store(void* gdst, const void* ssrc, uint32_t bytes) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(ssrc);
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(s), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// all bulk stores of this thread have finished READING shared memory (the staging may be reused)
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// make generic-proxy shared-memory writes visible to the async proxy (TMA) before the barrier
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ------------------------------------------------------------------------------------------------
template <int T>
struct AsmCfg {
  static_assert(T % 5 == 0, "tile must hold whole AUSM warps (5 cells per species warp)");
  static constexpr int AW = 2 * (T / 5);        // AUSM warps: warp w -> species w&1, cells 5*(w>>1)..+4
  static constexpr int MW = (T + 2) / 3;        // Maxwell warps: 3 cells each
  static constexpr int NT = 32 * (AW + MW);
};

template <int T>
struct __align__(128) AsmSmem {
  double mir[T][BLK];          // staged mirror block (j,i) of the current face; zeros persist
  double diag[T][BLK];         // staged diagonal block (i,i)
  double fb[T][3][2][NEQ];     // reconstructed face states, canonical side 0 = L, 1 = R
  double fpert[T][3][NEQ];     // own-side face state with variable v of the CELL perturbed
  double eps[T][NEQ];          // representable perturbation sizes of the own cell (S7)
  double pc[T][NEQ];           // own cell-centre state
  double s0[T][NEQ];           // source S(P_i)
  double rs[T][NEQ];           // non-flux part of R~: Omega (BDF2 term) - Omega S
  double rhs[T][NEQ];          // staged -R~
  double fg[T][3][4];          // nx, ny, s_if * Sigma_f, unused
  double vol[T];
  double ref[NEQ];
  alignas(16) int32_t blk[T][4];   // BSR block index of (i,i), (nbr0,i), (nbr1,i), (nbr2,i); -1 if absent
  int32_t nbr[T][3];
};

// conservative variables of one species from (rho, u, v, w, T)
__device__ __forceinline__ void cons5(double cv, const double* Q, double* U) {
  U[0] = Q[0];
  U[1] = Q[0] * Q[1];
  U[2] = Q[0] * Q[2];
  U[3] = Q[0] * Q[3];
  U[4] = Q[0] * (cv * Q[4] + 0.5 * (Q[1] * Q[1] + Q[2] * Q[2] + Q[3] * Q[3]));
}

template <int T, bool JAC>
__global__ void __launch_bounds__(AsmCfg<T>::NT) k_assemble(
    int64_t nc, Consts K, const double* __restrict__ state, const double* __restrict__ state_n,
    const double* __restrict__ state_nm1, double inv2dt, const double* __restrict__ lgrad,
    const double* __restrict__ cgeo, const int32_t* __restrict__ cell_nbr, const int32_t* __restrict__ blk4,
    double* __restrict__ rhs, double* __restrict__ vals, int32_t* __restrict__ flags) {
  using C = AsmCfg<T>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  AsmSmem<T>& S = *reinterpret_cast<AsmSmem<T>*>(smem_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool do_flux = K.mask & 1, do_src = K.mask & 2, do_time = K.mask & 4;
  const int64_t ntiles = (nc + T - 1) / T;

  // ---- role of this lane (tile independent) ----
  const bool is_ausm = warp < C::AW;
  int cl, p, sp = 0, base_lane;
  bool lane_ok;
  if (is_ausm) {
    const int g = lane / 6;
    p = lane - 6 * g;
    sp = warp & 1;
    cl = 5 * (warp >> 1) + g;
    lane_ok = lane < 30;
    base_lane = 6 * g;
  } else {
    const int g = lane / 9;
    p = lane - 9 * g;
    cl = 3 * (warp - C::AW) + g;
    lane_ok = lane < 27 && cl < T;
    base_lane = 9 * g;
  }
  if (!lane_ok) cl = 0;   // idle lanes shadow cell 0 (they take part in the shuffles, never store)
  // rows = variables of this lane's group; a_v / m_v = the variable this lane perturbs
  const int ir = 8 + sp, iu = 10 + 3 * sp, iT = 16 + sp;
  const int pj = p > 0 ? p - 1 : 0;
  const int v = is_ausm ? (pj == 0 ? ir : (pj == 4 ? iT : iu + pj - 1)) : pj;
  // species constants (warp uniform)
  const double cRs = K.Rs[sp], cgR = K.gR[sp], ccp = K.cp[sp], cMinf2 = K.Minf2[sp];

  if (JAC)
    for (int q = tid; q < T * BLK; q += C::NT) (&S.mir[0][0])[q] = 0.0;
  if (tid < NEQ) S.ref[tid] = K.ref[tid];
  __syncthreads();

  bool nonphys = false;

#pragma unroll 1
  for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int64_t cell0 = tile * T;
    const int ncell = (int)min((int64_t)T, nc - cell0);

    // ---- phase 0: topology and face geometry of the tile ----
    if (tid < 3 * T) {
      const int c = tid / 3, k = tid - 3 * c;
      const int64_t i = cell0 + c;
      if (c < ncell) {
        const double* g = cgeo + CGEO * i + 8 * k;
        const int32_t j = cell_nbr[3 * i + k];
        const bool own_is_L = j < 0 || i < j;
        S.nbr[c][k] = j;
        S.fg[c][k][0] = g[0];
        S.fg[c][k][1] = g[1];
        S.fg[c][k][2] = own_is_L ? g[2] : -g[2];
        if (k == 0) S.vol[c] = g[7];
      }
    }
    // S.blk[t] is written and read (when the bulk stores are issued) by thread t only
    if (tid < ncell) *reinterpret_cast<int4*>(&S.blk[tid][0]) = *reinterpret_cast<const int4*>(blk4 + 4 * (cell0 + tid));
    // ---- phase A: reconstruct L/R face states and the own-side perturbed ones (Alg. 1)
    for (int q = tid; q < ncell * (6 * NEQ); q += C::NT) {
      const int c = q / (6 * NEQ), rem = q - c * (6 * NEQ);
      const int k = rem / (2 * NEQ), rem2 = rem - k * (2 * NEQ);
      const int side = rem2 / NEQ, w = rem2 - side * NEQ;
      const int64_t i = cell0 + c;
      const int32_t j = cell_nbr[3 * i + k];
      const bool own_is_L = j < 0 || i < j;
      const bool is_own = (j < 0) || (side == (own_is_L ? 0 : 1));   // boundary: P_R := P_L (S9)
      const int64_t X = is_own ? i : j;
      const double* g = cgeo + CGEO * i + 8 * k;
      const double dx = is_own ? g[3] : g[5], dy = is_own ? g[4] : g[6];
      const double Pc = state[NEQ * X + w];
      const double2 lg = *reinterpret_cast<const double2*>(lgrad + 2 * (NEQ * X + w));
      const double inc = lg.x * dx + lg.y * dy;
      S.fb[c][k][side][w] = Pc + inc;
      if (is_own && (side == 0 || j >= 0)) {
        // eps_k = delta * max(|P_cell,k|, ref_k), made representable (S7)
        const double t = Pc + K.delta * fmax(fabs(Pc), S.ref[w]);
        S.fpert[c][k][w] = t + inc;
        if (k == 0) {
          S.eps[c][w] = t - Pc;
          S.pc[c][w] = Pc;
        }
      }
    }
    // ---- phase A2: the non-flux part of the residual (source L245, BDF2 Eq. 13), per (cell, group)
    if (tid >= C::NT - 3 * T) {
      const int q = tid - (C::NT - 3 * T);
      const int c = q / 3, grp = q - 3 * c;   // 0 fields, 1 ions, 2 electrons
      const int64_t i = cell0 + c;
      if (c < ncell) {
        double P[NEQ], Ss[NEQ];
#pragma unroll
        for (int r = 0; r < NEQ; r += 2) {
          const double2 t2 = *reinterpret_cast<const double2*>(state + NEQ * i + r);
          P[r] = t2.x;
          P[r + 1] = t2.y;
        }
        source_terms(K, P, Ss);
        const double vol = cgeo[CGEO * i + 7];
        const double ft = vol * inv2dt;
        if (grp == 0) {
#pragma unroll
          for (int r = 0; r < 8; ++r) {
            double a = 0.0;
            if (do_src) a -= Ss[r] * vol;
            if (do_time) a += ft * (3.0 * P[r] - 4.0 * state_n[NEQ * i + r] + state_nm1[NEQ * i + r]);
            S.rs[c][r] = a;
            S.s0[c][r] = Ss[r];
          }
        } else {
          const int s = grp - 1;
          const int rows[5] = {8 + s, 10 + 3 * s, 11 + 3 * s, 12 + 3 * s, 16 + s};
          double Q[5], Qn[5], Qm[5], U[5], Un[5], Um[5], S5[5];
          if (s == 0) { sp_get<0>(P, Q); sp_get<0>(Ss, S5); } else { sp_get<1>(P, Q); sp_get<1>(Ss, S5); }
#pragma unroll
          for (int r = 0; r < 5; ++r) {
            Qn[r] = state_n[NEQ * i + rows[r]];
            Qm[r] = state_nm1[NEQ * i + rows[r]];
          }
          const double cv = K.cv[s];
          cons5(cv, Q, U);
          cons5(cv, Qn, Un);
          cons5(cv, Qm, Um);
#pragma unroll
          for (int r = 0; r < 5; ++r) {
            double a = 0.0;
            if (do_src) a -= S5[r] * vol;
            if (do_time) a += ft * (3.0 * U[r] - 4.0 * Un[r] + Um[r]);
            S.rs[c][rows[r]] = a;
            S.s0[c][rows[r]] = S5[r];
          }
        }
      }
    }
    __syncthreads();   // B0: tile inputs staged

    const bool cell_ok = lane_ok && cl < ncell;
    const bool pert = p != 0;
    double acc[8];     // base lane: residual rows; perturbed lane: its column of the diagonal block
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = 0.0;
    const double inv_e = (JAC && pert) ? 1.0 / S.eps[cl][v] : 0.0;

    // ---- phase B: faces (Alg. 1) ----
#pragma unroll 1
    for (int k = 0; k < 3; ++k) {
      const int32_t j = S.nbr[cl][k];
      const double nx = S.fg[cl][k][0], ny = S.fg[cl][k][1], sl = S.fg[cl][k][2];
      const bool own_is_L = sl > 0.0, bnd = j < 0;
      const bool run = do_flux && (JAC || !pert);
      double d[8];
      if (is_ausm) {
        double H[5];
        if (run) {
          double L[5], R[5];
          L[0] = S.fb[cl][k][0][ir]; R[0] = S.fb[cl][k][1][ir];
#pragma unroll
          for (int q = 0; q < 3; ++q) { L[1 + q] = S.fb[cl][k][0][iu + q]; R[1 + q] = S.fb[cl][k][1][iu + q]; }
          L[4] = S.fb[cl][k][0][iT]; R[4] = S.fb[cl][k][1][iT];
          if (pert) {
            const double pv = S.fpert[cl][k][v];
            const bool pl = own_is_L || bnd, pr = !own_is_L || bnd;   // boundary: both arguments move (S9)
#pragma unroll
            for (int q = 0; q < 5; ++q)
              if (q == pj) {
                if (pl) L[q] = pv;
                if (pr) R[q] = pv;
              }
          }
          const bool ok = ausm_flux(cRs, cgR, ccp, cMinf2, K, L, R, nx, ny, H);
          if (!pert && cell_ok) nonphys |= !ok;
        } else {
#pragma unroll
          for (int q = 0; q < 5; ++q) H[q] = 0.0;
        }
        const double f = pert ? sl * inv_e : sl;
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const double hb = __shfl_sync(0xffffffffu, H[q], base_lane);
          // explicit rounding: the residual must not depend on JAC through FMA contraction
          d[q] = __dmul_rn(pert ? H[q] - hb : H[q], f);
          acc[q] = __dadd_rn(acc[q], d[q]);
        }
      } else {
        double H[8];
        if (run) {
          double L[8], R[8];
#pragma unroll
          for (int q = 0; q < 8; ++q) { L[q] = S.fb[cl][k][0][q]; R[q] = S.fb[cl][k][1][q]; }
          if (pert) {
            const double pv = S.fpert[cl][k][v];
            const bool pl = own_is_L || bnd, pr = !own_is_L || bnd;
#pragma unroll
            for (int q = 0; q < 8; ++q)
              if (q == pj) {
                if (pl) L[q] = pv;
                if (pr) R[q] = pv;
              }
          }
          maxwell_flux(K, L, R, nx, ny, H);
        } else {
#pragma unroll
          for (int q = 0; q < 8; ++q) H[q] = 0.0;
        }
        const double f = pert ? sl * inv_e : sl;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const double hb = __shfl_sync(0xffffffffu, H[q], base_lane);
          // explicit rounding: the residual must not depend on JAC through FMA contraction
          d[q] = __dmul_rn(pert ? H[q] - hb : H[q], f);
          acc[q] = __dadd_rn(acc[q], d[q]);
        }
      }
      if (!JAC) continue;
      // the staging of the previous face / tile has been read by the TMA
      if (tid < T) bulk_wait_read();
      __syncthreads();   // B1
      if (pert && cell_ok && !bnd) {
        if (is_ausm) {
          S.mir[cl][ir * NEQ + v] = -d[0];
#pragma unroll
          for (int q = 0; q < 3; ++q) S.mir[cl][(iu + q) * NEQ + v] = -d[1 + q];
          S.mir[cl][iT * NEQ + v] = -d[4];
        } else {
#pragma unroll
          for (int q = 0; q < 8; ++q) S.mir[cl][q * NEQ + v] = -d[q];
        }
      }
      fence_async_smem();
      __syncthreads();   // B2
      // a7: the block (j,i) leaves the SM as one 2592-byte bulk store
      if (tid < ncell) {
        const int32_t b = S.blk[tid][1 + k];
        if (b >= 0) {
          bulk_store(vals + (int64_t)b * BLK, &S.mir[tid][0], BLK * 8);
          bulk_commit();
        }
      }
    }

    // ---- phase C: residual, source Jacobian (L245-253), BDF2 diagonal (Eq. 13), diagonal block ----
    if (!JAC) {
      if (tid < T) bulk_wait_read();
      __syncthreads();
    }
    if (cell_ok && !pert) {
      if (is_ausm) {
        S.rhs[cl][ir] = -(acc[0] + S.rs[cl][ir]);
#pragma unroll
        for (int q = 0; q < 3; ++q) S.rhs[cl][iu + q] = -(acc[1 + q] + S.rs[cl][iu + q]);
        S.rhs[cl][iT] = -(acc[4] + S.rs[cl][iT]);
      } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) S.rhs[cl][q] = -(acc[q] + S.rs[cl][q]);
      }
    }
    if (JAC && cell_ok && pert) {
      const double vol = S.vol[cl];
      double col[NEQ];
#pragma unroll
      for (int r = 0; r < NEQ; ++r) col[r] = 0.0;
      if (is_ausm) {
        // flux part: rows of this species (static indices per species keep col[] in registers)
        if (sp == 0) sp_put<0>(col, acc); else sp_put<1>(col, acc);
      } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) col[q] = acc[q];
      }
      double P[NEQ];
#pragma unroll
      for (int r = 0; r < NEQ; ++r) P[r] = S.pc[cl][r];
      if (do_time) {
        // analytic dU/dP (S15): identity on the field rows; species rows below
        const double ft = 3.0 * vol * inv2dt;
        if (!is_ausm) {
#pragma unroll
          for (int r = 0; r < 8; ++r)
            if (r == v) col[r] += ft;
        } else if (sp == 0) time_column<0>(K, col, v, P, ft);
        else time_column<1>(K, col, v, P, ft);
      }
      if (do_src) {
        const double e = S.eps[cl][v];
#pragma unroll
        for (int r = 0; r < NEQ; ++r)
          if (r == v) P[r] += e;
        double S1[NEQ];
        source_terms(K, P, S1);
        const double f = vol * inv_e;
        // rows 0,1,2 (B), 6 (Psi), 8,9 (mass) have no source: S1 - S0 = 0 exactly
#pragma unroll
        for (int r = 0; r < NEQ; ++r)
          if (!(r < 3 || r == 6 || r == 8 || r == 9)) col[r] -= (S1[r] - S.s0[cl][r]) * f;
      }
#pragma unroll
      for (int r = 0; r < NEQ; ++r) S.diag[cl][r * NEQ + v] = col[r];
    }
    fence_async_smem();
    __syncthreads();   // B3
    if (tid < ncell && JAC) {
      bulk_store(vals + (int64_t)S.blk[tid][0] * BLK, &S.diag[tid][0], BLK * 8);
      bulk_commit();
    }
    if (tid == T - 1) {
      bulk_store(rhs + NEQ * cell0, &S.rhs[0][0], (uint32_t)ncell * NEQ * 8);
      bulk_commit();
    }
  }
  if (tid < T) bulk_wait_all();
  if (nonphys) atomicAdd(flags, 1);
}

// ================================================================================================
int launch_assemble(const tfa_mesh& m, const Consts& K, const double* state, const double* state_n,
                    const double* state_nm1, double dt, const double* lgrad, double* rhs, double* vals,
                    int32_t* flags, cudaStream_t st) {
  if (m.nc == 0) return 0;
  constexpr int T = 10;
  using C = AsmCfg<T>;
  static int ctas_per_sm = 0, n_sm = 0;
  const int smem = (int)sizeof(AsmSmem<T>);
  if (!ctas_per_sm) {
    TFA_CUDA(cudaFuncSetAttribute(k_assemble<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    TFA_CUDA(cudaFuncSetAttribute(k_assemble<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int dev = 0, occ = 0;
    TFA_CUDA(cudaGetDevice(&dev));
    TFA_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    TFA_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_assemble<T, true>, C::NT, smem));
    if (occ < 1) return set_error(TFA_ECUDA, "k_assemble does not fit on an SM");
    ctas_per_sm = occ;
  }
  const int64_t ntiles = (m.nc + T - 1) / T;
  const unsigned grid = (unsigned)std::min<int64_t>(ntiles, (int64_t)n_sm * ctas_per_sm);
  const double inv2dt = 1.0 / (2.0 * dt);
  if (vals)
    k_assemble<T, true><<<grid, C::NT, smem, st>>>(m.nc, K, state, state_n, state_nm1, inv2dt, lgrad, m.cgeo.p,
                                                   m.cell_nbr.p, m.blk4.p, rhs, vals, flags);
  else
    k_assemble<T, false><<<grid, C::NT, smem, st>>>(m.nc, K, state, state_n, state_nm1, inv2dt, lgrad, m.cgeo.p,
                                                    m.cell_nbr.p, m.blk4.p, rhs, vals, flags);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

}  // namespace tfa

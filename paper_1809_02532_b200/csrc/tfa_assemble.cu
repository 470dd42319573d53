// tfa_assemble.cu — steps a3..a7 fused: face flux + flux Jacobian + source + BDF2 + BSR write.
//
// Design, replacing Alg. 1's thread-per-cell loop (L221-256):
//
//  * A persistent CTA walks tiles of T consecutive cells.  Cell i evaluates, for each of its three
//    faces, the numerical flux through the face in ITS OWN outward frame (own state first, outward
//    normal) and the fluxes with each variable of its own side perturbed (Alg. 1).  The
//    column (H_pert - H)/eps * Sigma_f is (a) accumulated into the diagonal block (i,i) and (b)
//    written, negated, as the block (j,i) of the NEIGHBOUR's row: the face enters R_j with the
//    opposite sign, so d R_j / d P_i through it is exactly minus cell i's own contribution.  Every
//    BSR block has exactly one writer, so there are no atomics and no memset, and the perturbed
//    fluxes towards the other side are never evaluated: 6+6+9 = 21 flux evaluations per cell-face
//    instead of Alg. 1's 3*19 = 57 full ones.
//  * Lanes: an AUSM warp holds 5 groups of 6 lanes = (cell, species) x {base, 5 perturbed variables}
//    (Eq. 10); a Maxwell warp holds 3 groups of 9 lanes = cell x {base, 8 perturbed} (Eq. 9
//    L91).  The reconstructed face states (L232: P + phi grad P . dx) of both sides come from the
//    gradient kernel's face-state array (every lane of a group reads the same addresses; the
//    perturbation is added to the own-side value), staged one tile ahead into shared memory by TMA
//    bulk loads; the base flux reaches the group by warp shuffle; the flux Jacobian is block diagonal
//    (8x8, 5x5, 5x5), the source (Eq. 4/6) couples the blocks on the diagonal block only.
//  * 18x18 blocks are staged in shared memory (their structural zeros are written once per CTA)
//    and leave the SM as 2592-byte TMA bulk stores (cp.async.bulk.global.shared::cta).
//  * The TFA_ASM_* constants below were tuned by measurement (DESIGN.md 6.3 lists what was tried).
#include <cstdlib>

#include "tfa_common.cuh"
#include "tfa_physics.cuh"
#include "tfa_tma.cuh"

#ifndef TFA_ASM_EARLY2
#define TFA_ASM_EARLY2 1   // bit 0: AUSM lanes, bit 1: Maxwell lanes evaluate all three faces before the first barrier
#endif
#ifndef TFA_ASM_BLKP
#define TFA_ASM_BLKP 330   // doubles between staged blocks (324 = dense)
#endif
#ifndef TFA_ASM_T
#define TFA_ASM_T 10      // cells per tile (multiple of 5)
#endif
#ifndef TFA_ASM_NM
#define TFA_ASM_NM 2   // mirror staging buffers per tile (the barrier sequence is written for 2)
#endif

namespace tfa {

constexpr int BLKP = TFA_ASM_BLKP;
// Packed Jacobian (second option; tfa_assemble_packed): an off-diagonal block holds only its 114
// structural non-zeros -- fields 8x8, ions 5x5, electrons 5x5, each row-major, in that order -- and the diagonal
// blocks sit in an array of their own.  Staged 118 doubles apart (odd number of 16-byte units, as BLKP).
constexpr int PKB = TFA_PACKED_BLOCK;   // 114
constexpr int PKP = 118;


// ------------------------------------------------------------------------------------------------
template <int T>
struct AsmCfg {
  static_assert(T % 5 == 0, "tile must hold whole AUSM warps (5 cells per species warp)");
  static constexpr int AW = 2 * (T / 5);        // AUSM warps: warp w -> species w&1, cells 5*(w>>1)..+4
  static constexpr int MW = (T + 2) / 3;        // Maxwell warps: 3 cells each
  static constexpr int NT = 32 * (AW + MW);
};

// Inputs of one tile, fetched by TMA one tile ahead (read latency under the Jacobian's write stream is
// long): own-side and other-side face states of every (cell, face), geometry records, cell-centre states.
// NF = face slots per cell: 3 (triangle meshes) or 4 (meshes with quadrilaterals).
template <int T, int NF>
struct __align__(16) AsmIn {
  double fx[T][NF][NEQ];  // other side of face k of cell c: the neighbour's face state; on a boundary face the
                          // cell's own row again, or the caller's ghost state (TFA_BC_GHOST)
  double fo[T][NF][NEQ];  // own side
  double cg[T][8 * NF];
  double st[T][NEQ];
  int32_t nf[T][NF];      // packed neighbour (tfa_common.cuh): 4 * neighbour + its local face, or < 0 on the boundary
  int32_t pad_[4 - (T * NF) % 4];   // keeps the struct a multiple of 16 bytes
};

template <int T, int NM, int NF, bool PK>
struct __align__(128) AsmSmem {
  static constexpr int MP = PK ? PKP : BLKP;
  AsmIn<T, NF> in[2];
  uint64_t full[2];        // mbarriers: stage s has landed
  // staged blocks: a stride of BLKP doubles (16-byte multiple, odd number of 16-byte units) spreads the
  // column stores of different cells over the banks
  double mir[NM][T][MP];    // mirror blocks (j,i), face k in buffer k % NM; structural zeros persist
  double diag[T][BLKP];     // diagonal block (i,i); structural zeros persist
  double rs[T][NEQ];     // non-flux part of R~: Omega (BDF2 term) - Omega S
  double s0[T][8];       // Lorentz-force and Joule-heating rows of S(P_i): equations 10..17
};

// roles: 0 = ion AUSM lanes, 1 = electron AUSM lanes, 2 = Maxwell lanes (k_residual; k_assemble runs both
// species through the role-0 code with the species at run time, which keeps its hot code small).
// index of the q-th variable of the role's group inside the 18-vector
template <int ROLE>
__device__ __forceinline__ constexpr int vidx(int q) {
  return ROLE == 2 ? q : (q == 0 ? 8 + ROLE : (q == 4 ? 16 + ROLE : 9 + 3 * ROLE + q));
}

// Momentum and energy source rows of one species (Eq. 6; S5) with the rounding sequence
// pinned, so that the base values kept in shared memory and the perturbed re-evaluations of the
// source Jacobian (Alg. 1) agree bit for bit wherever the perturbed variable does not enter.
__device__ __forceinline__ void lorentz_rows(double qn, const double* E, const double* B, double u, double v,
                                             double w, double* out4) {
  double t;
  t = __dmul_rn(w, B[1]); t = __fma_rn(v, B[2], -t); out4[0] = __dmul_rn(qn, __dadd_rn(E[0], t));
  t = __dmul_rn(u, B[2]); t = __fma_rn(w, B[0], -t); out4[1] = __dmul_rn(qn, __dadd_rn(E[1], t));
  t = __dmul_rn(v, B[0]); t = __fma_rn(u, B[1], -t); out4[2] = __dmul_rn(qn, __dadd_rn(E[2], t));
  t = __dmul_rn(u, E[0]); t = __fma_rn(v, E[1], t); t = __fma_rn(w, E[2], t); out4[3] = __dmul_rn(qn, t);
}

// conservative variables of one species from (rho, u, v, w, T)
__device__ __forceinline__ void cons5(double cv, const double* Q, double* U) {
  U[0] = Q[0];
  U[1] = Q[0] * Q[1];
  U[2] = Q[0] * Q[2];
  U[3] = Q[0] * Q[3];
  U[4] = Q[0] * (cv * Q[4] + 0.5 * (Q[1] * Q[1] + Q[2] * Q[2] + Q[3] * Q[3]));
}

// ------------------------------------------------------------------------------------------------
// Non-flux part of the residual of one (cell, group): source (Alg. 1) and BDF2 term (Eq. 13).
// grp 0 = field rows 0..7, 1 = ion rows, 2 = electron rows.  P, Pn, Pm: the cell's 18 values at the three time
// levels.  Writes the group's rows of rs[18] and (species) its four entries of s0[8].
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cell_group_rest(const int grp, const Consts& K, const double* __restrict__ P,
                                                const double* __restrict__ Pn, const double* __restrict__ Pm,
                                                double vol, double inv2dt, double* __restrict__ rs,
                                                double* __restrict__ s0) {
  const bool do_src = K.mask & 2, do_time = K.mask & 4;
  const double ft = vol * inv2dt;
  if (grp == 0) {
    // S_E = -c^2 sum_s q_s n_s u_s, S_Phi = c^2 sum_s q_s n_s  (Eq. 4; eps0 = 1/c^2)
    const double qi = K.qm[0] * P[8], qe = K.qm[1] * P[9];
    double Sf[8];
    Sf[0] = Sf[1] = Sf[2] = Sf[6] = 0.0;
    Sf[3] = -K.c2 * (qi * P[10] + qe * P[13]);
    Sf[4] = -K.c2 * (qi * P[11] + qe * P[14]);
    Sf[5] = -K.c2 * (qi * P[12] + qe * P[15]);
    Sf[7] = K.c2 * (qi + qe);
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      double a = 0.0;
      if (do_src) a -= Sf[r] * vol;
      if (do_time) a += ft * (3.0 * P[r] - 4.0 * Pn[r] + Pm[r]);
      rs[r] = a;
    }
  } else {
    const int s = grp - 1;
    const int rows[5] = {8 + s, 10 + 3 * s, 11 + 3 * s, 12 + 3 * s, 16 + s};
    double Q[5], Qn[5], Qm[5], U[5], Un[5], Um[5], S5[5], E[3], B[3];
#pragma unroll
    for (int r = 0; r < 5; ++r) {
      Q[r] = P[rows[r]];
      Qn[r] = Pn[rows[r]];
      Qm[r] = Pm[rows[r]];
    }
#pragma unroll
    for (int r = 0; r < 3; ++r) { B[r] = P[r]; E[r] = P[3 + r]; }
    S5[0] = 0.0;
    lorentz_rows(K.qm[s] * Q[0], E, B, Q[1], Q[2], Q[3], S5 + 1);
    const double cv = K.cv[s];
    cons5(cv, Q, U);
    cons5(cv, Qn, Un);
    cons5(cv, Qm, Um);
#pragma unroll
    for (int r = 0; r < 5; ++r) {
      double a = 0.0;
      if (do_src) a -= S5[r] * vol;
      if (do_time) a += ft * (3.0 * U[r] - 4.0 * Un[r] + Um[r]);
      rs[rows[r]] = a;
    }
    s0[3 * s] = S5[1];
    s0[3 * s + 1] = S5[2];
    s0[3 * s + 2] = S5[3];
    s0[6 + s] = S5[4];
  }
}

// ------------------------------------------------------------------------------------------------
// One warp fetches the inputs of the tile starting at cell cellN (nN cells) into a stage: lane l handles the
// (cell, face) pairs l and l + 32 (nfN[0], nfN[1] = their packed neighbours) and copies each pair's other-side row.
// ------------------------------------------------------------------------------------------------
template <int T, int NF>
__device__ __forceinline__ void stage_inputs(AsmIn<T, NF>& in, uint64_t* bar, int lane, const int32_t (&nfN)[2],
                                             int64_t cellN, int nN, const double* __restrict__ state,
                                             const double* __restrict__ fown, const double* __restrict__ cgeo,
                                             const double* __restrict__ ghost, int32_t* __restrict__ flags,
                                             const Limits& lim) {
  static_assert(NF * T <= 64, "two (cell, face) pairs per lane");
  if (lane == 0)
    mbar_arrive_expect_tx(bar, (uint32_t)nN * (NF * NEQ * 8 + NF * NEQ * 8 + 8 * NF * 8 + NEQ * 8));
#pragma unroll
  for (int h = 0; h < (NF * T > 32 ? 2 : 1); ++h) {
    const int l = lane + 32 * h;
    if (l < NF * nN) {
      const int32_t nf = nfN[h];
      const double* src;
      TFA_BOUND(flags, nf >= 0 ? (nf >> 2) < lim.n_cells && (nf & 3) < NF
                               : (bc_tag_of(nf) != TFA_BC_GHOST || (ghost != nullptr && bc_face_of(nf) < lim.n_ghost)));
      TFA_BOUND(flags, cellN >= 0 && cellN + nN <= lim.n_cells && l < NF * T);
      if (nf >= 0) src = fown + (NF * (int64_t)(nf >> 2) + (nf & 3)) * NEQ;          // the neighbour's face state
      else if (bc_tag_of(nf) == TFA_BC_GHOST) src = ghost + bc_face_of(nf) * NEQ;     // the caller's ghost state
      else src = fown + (NF * cellN + l) * NEQ;                                       // the cell's own row (S9, S24)
      bulk_load(&in.fx[0][0][0] + l * NEQ, src, NEQ * 8, bar);
      (&in.nf[0][0])[l] = nf;
    }
  }
  if (lane == 31) bulk_load(&in.fo[0][0][0], fown + NF * NEQ * cellN, (uint32_t)nN * NF * NEQ * 8, bar);
  if (lane == 30) bulk_load(&in.cg[0][0], cgeo + 8 * NF * cellN, (uint32_t)nN * 8 * NF * 8, bar);
  if (lane == 29) bulk_load(&in.st[0][0], state + NEQ * cellN, (uint32_t)nN * NEQ * 8, bar);
}

// ------------------------------------------------------------------------------------------------
// The tile loop of one warp role.  All roles execute the same sequence of CTA barriers.
// ------------------------------------------------------------------------------------------------
template <int T, int NM, int NF, bool PK, int ROLE>
__device__ __forceinline__ void role_loop(AsmSmem<T, NM, NF, PK>& S, const bool JAC, const int64_t nc, const Consts& K,
                                          const double* __restrict__ state, const double* __restrict__ state_n,
                                          const double* __restrict__ state_nm1, const double inv2dt,
                                          const double* __restrict__ fown, const double* __restrict__ cgeo,
                                          const int32_t* __restrict__ nbrf, const int32_t* __restrict__ blkmap,
                                          const double* __restrict__ ghost, double* __restrict__ rhs,
                                          double* __restrict__ vals, double* __restrict__ vals_o,
                                          int32_t* __restrict__ flags, const Limits& lim) {
  using C = AsmCfg<T>;
  constexpr int BS = blk_stride(NF);
  // where a mirror block goes: the BSR value array (324 doubles per block), or the packed off-diagonal array
  constexpr int MBLK = PK ? PKB : BLK;
  double* __restrict__ const mvals = PK ? vals_o : vals;
  constexpr int NV = ROLE == 2 ? 8 : 5;   // variables (= rows) of the role's group
  constexpr int GL = NV + 1;              // lanes per group: base + NV perturbed
  constexpr int NG = ROLE == 2 ? 3 : 5;   // groups per warp
  // AUSM lanes: one code path for both species (halves the kernel's hot code), the species at run time
  const int SPC = ROLE == 2 ? 0 : ((threadIdx.x >> 5) & 1);
  auto vx = [&](const int q) { return ROLE == 2 ? q : (q == 0 ? 8 + SPC : (q == 4 ? 16 + SPC : 9 + 3 * SPC + q)); };
  // warp issuing the end-of-tile bulk stores: the first Maxwell warp (it has slack at the top of the next tile;
  // measured against warp 1 and the last warp)
  constexpr int WB = C::AW;
  static_assert(T <= 32, "one issuing lane per tile cell");
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool do_flux = K.mask & 1, do_src = K.mask & 2, do_time = K.mask & 4;
  const int64_t ntiles = (nc + T - 1) / T;

  const int g = lane / GL, p = lane - GL * g;
  int cl = ROLE == 2 ? 3 * (warp - C::AW) + g : 5 * (warp >> 1) + g;
  const bool lane_ok = lane < GL * NG && cl < T;
  if (!lane_ok) cl = 0;   // idle lanes shadow the tile's first cell (they join the shuffles, never store)
  const int base_lane = GL * g;
  const bool pert = p != 0;
  const int pj = p - 1;   // perturbed variable of the group; -1 on the base lane
  const int v = ROLE == 2 ? max(pj, 0) : (pj <= 0 ? 8 + SPC : (pj == 4 ? 16 + SPC : 9 + 3 * SPC + pj));
  const bool run = do_flux && (JAC || !pert);
  const double pm = pert ? 1.0 : 0.0;
  bool nonphys = false;

  const bool loader = ROLE == 2 && warp == C::AW + C::MW - 1;   // the (lightly loaded) last warp fetches inputs
  int it = 0;
#pragma unroll 1
  for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
    const int64_t cell0 = tile * T;
    const int ncell = (int)min((int64_t)T, nc - cell0);
    const bool act = lane_ok && cl < ncell;
    const int ca = act ? cl : 0;
    const int64_t i = cell0 + ca;
    // this tile's inputs were requested one tile ago (kernel prologue for the first one)
    const AsmIn<T, NF>& in = S.in[it & 1];
    mbar_wait(&S.full[it & 1], (it >> 1) & 1);
    const double* __restrict__ cg = in.cg[ca];
    const double* __restrict__ sO = in.st[ca];

    // ---- the non-flux part of the residual, one thread per (cell, group) ----
    // (two paths, fields and species: one warp each, so that neither warp runs both)
    if (ROLE == 2 && warp >= C::AW + C::MW - 2) {
      const bool fields = warp == C::AW + C::MW - 1;
      const int c = fields ? lane : lane >> 1, grp = fields ? 0 : 1 + (lane & 1);
      if (lane < (fields ? T : 2 * T) && c < ncell) {
        const double* Pn_ = state_n + NEQ * (cell0 + c);
        const double* Pm_ = state_nm1 + NEQ * (cell0 + c);
        cell_group_rest(grp, K, in.st[c], Pn_, Pm_, in.cg[c][7], inv2dt, S.rs[c], S.s0[c]);
      }
    }
    // the next tile of this CTA: its packed neighbours (needed to request its inputs after face 0), and
    // the lines its non-TMA reads touch, towards L2
    const int64_t cellN = cell0 + (int64_t)gridDim.x * T;
    const int nN = cellN < nc ? (int)min((int64_t)T, nc - cellN) : 0;
    int32_t nfN[2] = {-1, -1};
    if (loader) {
      if (lane < NF * nN) nfN[0] = nbrf[NF * cellN + lane];
      if (NF * T > 32 && lane + 32 < NF * nN) nfN[1] = nbrf[NF * cellN + lane + 32];
    }
    if (warp == 0 && nN > 0) {
      const char* base;
      int l, bytes;
      if (lane < 26) {
        l = lane % 13;
        base = reinterpret_cast<const char*>((lane < 13 ? state_n : state_nm1) + NEQ * cellN);
        bytes = nN * NEQ * 8;
      } else if (lane < 29) {
        l = lane - 26;
        base = reinterpret_cast<const char*>(blkmap + BS * cellN);
        bytes = nN * BS * 4;
      } else {
        l = lane - 29;   // the tile after the next one
        base = reinterpret_cast<const char*>(nbrf + NF * (cellN + (int64_t)gridDim.x * T));
        bytes = cellN + (int64_t)gridDim.x * T + T <= nc ? T * NF * 4 : 0;
      }
      if (l * 128 < bytes + 127 && bytes > 0) prefetch_l2(base + min(l * 128, bytes - 1));
    }
    int32_t nbk[NF];
#pragma unroll
    for (int k = 0; k < NF; ++k) nbk[k] = in.nf[ca][k];

    // where this tile's blocks go: thread t < ncell issues the bulk stores of cell t
    int4 b4 = make_int4(-1, -1, -1, -1);
    int32_t b5 = -1;   // block of the fourth face (quadrilaterals)
    // bulk stores are issued by lane c (cell c) of warp 0 for the faces 0, 1 and of warp 1 for the diagonal block
    // and face 2, so that neither warp carries all 4 T requests of a tile (about 70 cycles each)
    const bool issuer = JAC && (warp == 0 || warp == WB) && lane < ncell;
    if (issuer) {
      b4 = *reinterpret_cast<const int4*>(blkmap + BS * (cell0 + lane));
      if (NF == 4) b5 = blkmap[BS * (cell0 + lane) + 4];
    }

    // eps_k = delta * max(|P_cell,k|, ref_k), made representable (S7)
    const double Pcv = sO[v];
    const double tv = Pcv + K.delta * fmax(fabs(Pcv), K.ref[v]);
    const double eps = tv - Pcv;
    const double inv_e = 1.0 / eps;

    // this lane's perturbation of the group's variables (Alg. 1): eps on its own one, 0 elsewhere
    double me[NV];
#pragma unroll
    for (int q = 0; q < NV; ++q) me[q] = q == pj ? eps : 0.0;

    double acc[NV];   // base lane: residual rows; perturbed lane: its column of the diagonal block

    // ---- one face (Alg. 1): d = this lane's scaled flux (base lane) or flux-Jacobian column ----
    auto face = [&](const int k, double* __restrict__ d) -> bool {
      const int32_t nf = nbk[k];   // packed neighbour: 4 * neighbour + its local face, or < 0 on the boundary
      const double2 g01 = *reinterpret_cast<const double2*>(cg + 8 * k);   // outward unit normal
      const double len = cg[8 * k + 2];                                    // Sigma_f
      const bool bnd = nf < 0;
      const double nx = g01.x, ny = g01.y;
      // own-side and other-side face states of this face (L232), written by k_gradient_limiter, staged by TMA
      const double* __restrict__ fo = in.fo[ca][k];
      const double* __restrict__ fx = in.fx[ca][k];

      const bool any_bnd = __any_sync(0xffffffffu, bnd);   // warp-uniform; boundary faces are rare
      double H[NV];
      if (run) {
        // the perturbed variable enters at the cell centre and is re-extrapolated with the frozen
        // limited gradient (L236-237; S8): (P + eps) + phi grad P . dx = face state + eps
        double own[NV], oth[NV];
        if (ROLE == 2) {
#pragma unroll
          for (int q = 0; q < NV; q += 2) {
            const double2 o2 = *reinterpret_cast<const double2*>(fo + q);
            const double2 x2 = *reinterpret_cast<const double2*>(fx + q);
            own[q] = o2.x + me[q];
            own[q + 1] = o2.y + me[q + 1];
            oth[q] = x2.x;
            oth[q + 1] = x2.y;
          }
        } else {
#pragma unroll
          for (int q = 0; q < NV; ++q) {
            own[q] = fo[vx(q)] + me[q];
            oth[q] = fx[vx(q)];
          }
        }
        if (any_bnd) {
          // boundary face (L260): the far side follows the face's rule; under the transmissive and the wall rule
          // it is a function of the own side, so the perturbation moves both arguments (S9, S24)
          if (bnd) {
            if (ROLE == 2) bc_fields(bc_tag_of(nf), own, nx, ny, oth);
            else bc_species(bc_tag_of(nf), own, nx, ny, oth);
          }
        }
        if (ROLE == 2) {
          maxwell_flux(K, own, oth, nx, ny, H);
        } else {
          const bool ok = ausm_flux(K.Rs[SPC], K.gR[SPC], K.cp[SPC], K.Minf2[SPC], K.Minf[SPC], K, own, oth, nx, ny, H);
          if (!pert && act) nonphys |= !ok;
        }
      } else {
#pragma unroll
        for (int q = 0; q < NV; ++q) H[q] = 0.0;
      }
      const double f = pert ? len * inv_e : len;
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        const double hb = __shfl_sync(0xffffffffu, H[q], base_lane);
        // perturbed lane: (H_pert - H) Sigma_f / eps; base lane: H Sigma_f  (pm = 1 or 0, exact)
        d[q] = __dmul_rn(__fma_rn(-hb, pm, H[q]), f);
      }
      return bnd;
    };
    // block (j,i) of the neighbour across a face: minus this cell's own column (staged, structural zeros persist)
    auto stage_mirror = [&](const int buf, const double* __restrict__ d, const bool bnd) {
      if (JAC && pert && act && !bnd) {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
          // packed: entry (row q, column pj) of the group's dense sub-block; BSR: entry (vx(q), v) of the 18 x 18 block
          const int e = PK ? (ROLE == 2 ? 8 * q + pj : 64 + 25 * SPC + 5 * q + pj) : vx(q) * NEQ + v;
          S.mir[buf][cl][e] = -d[q];
        }
      }
    };
    static_assert(NM == 2, "the barrier sequence below is written for two mirror buffers");
    constexpr bool EARLY2 = TFA_ASM_EARLY2 & (ROLE == 2 ? 2 : 1);   // evaluate face 2 together with faces 0, 1

    // faces 0, 1 go out first (mirror buffers 0, 1), then face 2 -- and face 3 of a quadrilateral -- reuse them
    double d0[NV], d1[NV], d2[NV], d3[NF == 4 ? NV : 1];
    const bool bnd0 = face(0, d0);
    const bool bnd1 = face(1, d1);
    bool bnd2 = false, bnd3 = false;
    if (EARLY2) {
      bnd2 = face(2, d2);
      if constexpr (NF == 4) bnd3 = face(3, d3);
    }
    if (loader && nN > 0) {
      // request the next tile's inputs into the other stage (every read of that stage ended before the
      // previous tile's closing barrier) — here, while this Maxwell warp would wait for the AUSM warps
      stage_inputs<T, NF>(S.in[(it + 1) & 1], &S.full[(it + 1) & 1], lane, nfN, cellN, nN, state, fown, cgeo, ghost, flags,
                          lim);
    }
    // both mirror buffers and the diagonal staging are free: the previous tile's bulk stores have read
    // them.  This barrier also publishes S.rs / S.s0 of the tile.
    if ((warp == 0 || warp == WB) && lane < T) bulk_wait_read();
    cta_sync();   // A
    stage_mirror(0, d0, bnd0);
    stage_mirror(1, d1, bnd1);
    fence_async_smem();
    cta_sync();   // 1
    // a7: each block leaves the SM as one 2592-byte bulk store
    if (issuer) {
      TFA_BOUND(flags, b4.x < lim.n_blocks && b4.y < lim.n_mirror_blocks && b4.z < lim.n_mirror_blocks &&
                           b4.w < lim.n_mirror_blocks && b5 < lim.n_mirror_blocks && cell0 + lane < lim.n_cells);
    }
    if (issuer && warp == 0) {
      if (b4.y >= 0) bulk_store(mvals + (int64_t)b4.y * MBLK, &S.mir[0][lane][0], MBLK * 8);
      if (b4.z >= 0) bulk_store(mvals + (int64_t)b4.z * MBLK, &S.mir[1][lane][0], MBLK * 8);
      bulk_commit();
    }
    if (!EARLY2) {   // (the Maxwell lanes: while the bulk stores read the buffers)
      bnd2 = face(2, d2);
      if constexpr (NF == 4) bnd3 = face(3, d3);
    }
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      acc[q] = __dadd_rn(__dadd_rn(d0[q], d1[q]), d2[q]);
      if constexpr (NF == 4) acc[q] = __dadd_rn(acc[q], d3[q]);
    }

    // ---- residual, source Jacobian (L245-253), BDF2 diagonal (Eq. 13), diagonal block ----
    if (act && !pert) {
#pragma unroll
      for (int q = 0; q < NV; ++q) rhs[NEQ * i + vx(q)] = -(acc[q] + S.rs[cl][vx(q)]);
    }
    if (JAC) {
      if (act && pert) {
        const double vol = cg[7];
        const double ft = 3.0 * vol * inv2dt;
        const double fs = vol * inv_e;
        if (ROLE == 2) {
          // column v = pj of the field variables: flux rows 0..7 (+ BDF2 identity, S15) and, for B and E,
          // the Lorentz / Joule rows of both species
          if (do_time) {
#pragma unroll
            for (int q = 0; q < 8; ++q)
              if (q == pj) acc[q] += ft;
          }
#pragma unroll
          for (int q = 0; q < 8; ++q) S.diag[cl][q * NEQ + v] = acc[q];
          double E[3], B[3];
#pragma unroll
          for (int r = 0; r < 3; ++r) {
            B[r] = r == pj ? tv : sO[r];
            E[r] = 3 + r == pj ? tv : sO[3 + r];
          }
#pragma unroll
          for (int s = 0; s < 2; ++s) {
            double S1[4];
            lorentz_rows(K.qm[s] * sO[8 + s], E, B, sO[10 + 3 * s], sO[11 + 3 * s], sO[12 + 3 * s], S1);
#pragma unroll
            for (int r = 0; r < 3; ++r)
              S.diag[cl][(10 + 3 * s + r) * NEQ + v] = do_src ? -(S1[r] - S.s0[cl][3 * s + r]) * fs : 0.0;
            S.diag[cl][(16 + s) * NEQ + v] = do_src ? -(S1[3] - S.s0[cl][6 + s]) * fs : 0.0;
          }
        } else {
          // column v of species ROLE: own flux rows (+ BDF2 dU/dP, analytic, S15), own Lorentz / Joule
          // rows, and the current / charge rows of E and Phi
          double Q[5], Qp[5], E[3], B[3];
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            Q[q] = sO[vx(q)];
            Qp[q] = q == pj ? tv : Q[q];
          }
#pragma unroll
          for (int r = 0; r < 3; ++r) { B[r] = sO[r]; E[r] = sO[3 + r]; }
          if (do_time) {
            const double cv = K.cv[SPC];
            if (pj == 0) {
              acc[0] += ft;
              acc[1] += ft * Q[1];
              acc[2] += ft * Q[2];
              acc[3] += ft * Q[3];
              acc[4] += ft * (cv * Q[4] + 0.5 * (Q[1] * Q[1] + Q[2] * Q[2] + Q[3] * Q[3]));
            } else if (pj == 4) {
              acc[4] += ft * Q[0] * cv;
            } else {
#pragma unroll
              for (int dd = 1; dd <= 3; ++dd)
                if (pj == dd) {
                  acc[dd] += ft * Q[0];
                  acc[4] += ft * Q[0] * Q[dd];
                }
            }
          }
          const double qn = K.qm[SPC] * Q[0], qnp = K.qm[SPC] * Qp[0];
          double S1[4];
          lorentz_rows(qnp, E, B, Qp[1], Qp[2], Qp[3], S1);
          if (do_src) {
#pragma unroll
            for (int r = 0; r < 3; ++r) acc[1 + r] -= (S1[r] - S.s0[cl][3 * SPC + r]) * fs;
            acc[4] -= (S1[3] - S.s0[cl][6 + SPC]) * fs;
          }
#pragma unroll
          for (int q = 0; q < 5; ++q) S.diag[cl][vx(q) * NEQ + v] = acc[q];
          // S_E = -c^2 sum_s q_s n_s u_s and S_Phi = c^2 sum_s q_s n_s: only this species' term moves
#pragma unroll
          for (int r = 0; r < 3; ++r)
            S.diag[cl][(3 + r) * NEQ + v] = do_src ? K.c2 * (qnp * Qp[1 + r] - qn * Q[1 + r]) * fs : 0.0;
          S.diag[cl][7 * NEQ + v] = do_src ? -K.c2 * (qnp - qn) * fs : 0.0;
        }
      }
    }
    // the mirror buffers have been read by the bulk stores of faces 0, 1: faces 2 (and 3) take them
    if (warp == 0 && lane < T) bulk_wait_read();
    cta_sync();   // 2
    stage_mirror(0, d2, bnd2);
    if constexpr (NF == 4) stage_mirror(1, d3, bnd3);
    fence_async_smem();
    cta_sync();   // B: every block of the tile is staged
    if (issuer && warp == WB) {
      if (b4.x >= 0) bulk_store(vals + (int64_t)b4.x * BLK, &S.diag[lane][0], BLK * 8);   // (-1: a shard's ghost cell)
      if (b4.w >= 0) bulk_store(mvals + (int64_t)b4.w * MBLK, &S.mir[0][lane][0], MBLK * 8);
      if (NF == 4 && b5 >= 0) bulk_store(mvals + (int64_t)b5 * MBLK, &S.mir[1][lane][0], MBLK * 8);
      bulk_commit();
    }
  }
  if (JAC && (warp == 0 || warp == WB) && lane < T) bulk_wait_all();
  if (nonphys) atomicAdd(flags, 1);
}

template <int T, int NM, int NF, bool PK>
__global__ void __launch_bounds__(AsmCfg<T>::NT, T >= 10 ? 2 : 4) k_assemble(
    const int64_t nc, const __grid_constant__ Consts K, const double* __restrict__ state,
    const double* __restrict__ state_n, const double* __restrict__ state_nm1, const double inv2dt,
    const double* __restrict__ fown, const double* __restrict__ cgeo, const int32_t* __restrict__ nbrf,
    const int32_t* __restrict__ blkmap, const double* __restrict__ ghost, double* __restrict__ rhs,
    double* __restrict__ vals, double* __restrict__ vals_o, int32_t* __restrict__ flags,
    const __grid_constant__ Limits lim) {
  using C = AsmCfg<T>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  AsmSmem<T, NM, NF, PK>& S = *reinterpret_cast<AsmSmem<T, NM, NF, PK>*>(smem_raw);
  // (residual-only calls go to k_residual; the JAC = false path here is kept for completeness)
  const bool JAC = vals != nullptr;
  const int warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) {
    mbar_init(&S.full[0], 1);
    mbar_init(&S.full[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (JAC) {   // structural zeros of the staged blocks, once per CTA
    for (int q = threadIdx.x; q < NM * T * AsmSmem<T, NM, NF, PK>::MP; q += C::NT) (&S.mir[0][0][0])[q] = 0.0;
    for (int q = threadIdx.x; q < T * BLKP; q += C::NT) (&S.diag[0][0])[q] = 0.0;
  }
  __syncthreads();
  if (warp == C::AW + C::MW - 1) {
    // prologue: request the inputs of this CTA's first tile
    const int lane = threadIdx.x & 31;
    const int64_t cellF = (int64_t)blockIdx.x * T;
    const int nF = cellF < nc ? (int)min((int64_t)T, nc - cellF) : 0;
    if (nF > 0) {
      int32_t nfF[2] = {-1, -1};
      if (lane < NF * nF) nfF[0] = nbrf[NF * cellF + lane];
      if (NF * T > 32 && lane + 32 < NF * nF) nfF[1] = nbrf[NF * cellF + lane + 32];
      stage_inputs<T, NF>(S.in[0], &S.full[0], lane, nfF, cellF, nF, state, fown, cgeo, ghost, flags, lim);
    }
  }
  __syncthreads();   // the prologue's neighbour table (plain stores) is visible
  // packed output: the AUSM warpgroup takes 8 registers per thread from the Maxwell one (136 / 120, no spills in
  // either role); measured 1.91 against 1.96 ms at c4b.  The BSR kernel, bound by its store stream, does not move
  // (2.18 against 2.17 ms) and keeps the even split; 152 / 104 and 168 / 88 spill in the Maxwell role and lose.
  if constexpr (PK && C::AW == 4 && C::MW == 4) {
    if (warp >= C::AW) asm volatile("setmaxnreg.dec.sync.aligned.u32 120;");
    else asm volatile("setmaxnreg.inc.sync.aligned.u32 136;");
  }
  if (warp >= C::AW)
    role_loop<T, NM, NF, PK, 2>(S, JAC, nc, K, state, state_n, state_nm1, inv2dt, fown, cgeo, nbrf, blkmap, ghost, rhs,
                                vals, vals_o, flags, lim);
  else
    role_loop<T, NM, NF, PK, 0>(S, JAC, nc, K, state, state_n, state_nm1, inv2dt, fown, cgeo, nbrf, blkmap, ghost, rhs,
                                vals, vals_o, flags, lim);
}

// ================================================================================================
// Residual only (tfa_assemble with bsr_vals = NULL; the matrix-free operator's evaluations): no Jacobian, so
// no staging, no perturbed lanes — thread = (cell, group), one warp per 32 cells and group (ions, electrons,
// fields), the three faces in sequence, face states straight from the gradient kernel's array.
// ================================================================================================
constexpr int RES_CELLS = 32;
template <int ROLE, int NF>
__device__ __forceinline__ void residual_rows(const int64_t i, const Consts& K, const double* __restrict__ state,
                                              const double* __restrict__ state_n, const double* __restrict__ state_nm1,
                                              const double inv2dt, const double* __restrict__ fown,
                                              const double* __restrict__ cgeo, const int32_t* __restrict__ nbrf,
                                              const double* __restrict__ ghost, double* __restrict__ rhs,
                                              bool& nonphys, int32_t* __restrict__ flags, const Limits& lim) {
  constexpr int NV = ROLE == 2 ? 8 : 5;
  constexpr int SPC = ROLE == 2 ? 0 : ROLE;
  const double* __restrict__ cg = cgeo + 8 * NF * i;
  double acc[NV];
#pragma unroll
  for (int q = 0; q < NV; ++q) acc[q] = 0.0;
  if (K.mask & 1) {
#pragma unroll 1
    for (int k = 0; k < NF; ++k) {
      const int32_t nf = nbrf[NF * i + k];
      const double nx = cg[8 * k], ny = cg[8 * k + 1], len = cg[8 * k + 2];
      const double* __restrict__ fo = fown + (NF * i + k) * NEQ;
      const int tag = nf < 0 ? bc_tag_of(nf) : 0;
      TFA_BOUND(flags, nf >= 0 ? (nf >> 2) < lim.n_cells && (nf & 3) < NF
                               : (tag != TFA_BC_GHOST || (ghost != nullptr && bc_face_of(nf) < lim.n_ghost)));
      const double* __restrict__ fx = nf >= 0 ? fown + (NF * (int64_t)(nf >> 2) + (nf & 3)) * NEQ
                                              : (tag == TFA_BC_GHOST ? ghost + bc_face_of(nf) * NEQ : fo);
      double own[NV], oth[NV], H[NV];
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        own[q] = fo[vidx<ROLE>(q)];
        oth[q] = fx[vidx<ROLE>(q)];
      }
      if (nf < 0) {   // boundary face (L260): the far side follows the face's rule
        if (ROLE == 2) bc_fields(tag, own, nx, ny, oth);
        else bc_species(tag, own, nx, ny, oth);
      }
      if (ROLE == 2) maxwell_flux(K, own, oth, nx, ny, H);
      else nonphys |= !ausm_flux(K.Rs[SPC], K.gR[SPC], K.cp[SPC], K.Minf2[SPC], K.Minf[SPC], K, own, oth, nx, ny, H);
#pragma unroll
      for (int q = 0; q < NV; ++q) acc[q] = __dadd_rn(acc[q], __dmul_rn(H[q], len));
    }
  }
  double rs[NEQ], s0[8];
  cell_group_rest(ROLE == 2 ? 0 : ROLE + 1, K, state + NEQ * i, state_n + NEQ * i, state_nm1 + NEQ * i, cg[7], inv2dt,
                  rs, s0);
#pragma unroll
  for (int q = 0; q < NV; ++q) rhs[NEQ * i + vidx<ROLE>(q)] = -(acc[q] + rs[vidx<ROLE>(q)]);
}

template <int NF>
__global__ void __launch_bounds__(3 * RES_CELLS) k_residual(
    const int64_t nc, const __grid_constant__ Consts K, const double* __restrict__ state,
    const double* __restrict__ state_n, const double* __restrict__ state_nm1, const double inv2dt,
    const double* __restrict__ fown, const double* __restrict__ cgeo, const int32_t* __restrict__ nbrf,
    const double* __restrict__ ghost, double* __restrict__ rhs, int32_t* __restrict__ flags,
    const __grid_constant__ Limits lim) {
  const int role = threadIdx.x >> 5;   // warp 0 ions, 1 electrons, 2 fields
  const int64_t i = blockIdx.x * (int64_t)RES_CELLS + (threadIdx.x & 31);
  if (i >= nc) return;
  bool nonphys = false;
  if (role == 0)
    residual_rows<0, NF>(i, K, state, state_n, state_nm1, inv2dt, fown, cgeo, nbrf, ghost, rhs, nonphys, flags, lim);
  else if (role == 1)
    residual_rows<1, NF>(i, K, state, state_n, state_nm1, inv2dt, fown, cgeo, nbrf, ghost, rhs, nonphys, flags, lim);
  else
    residual_rows<2, NF>(i, K, state, state_n, state_nm1, inv2dt, fown, cgeo, nbrf, ghost, rhs, nonphys, flags, lim);
  if (nonphys) atomicAdd(flags, 1);
}

// ================================================================================================
namespace {
template <int T, int NM, int NF, bool PK>
int launch_nm(const tfa_mesh& m, const Consts& K, const double* state, const double* state_n,
              const double* state_nm1, double dt, const double* fown, const double* ghost, double* rhs, double* vals,
              double* vals_o, int32_t* flags, int* resident_ctas, cudaStream_t st) {
  using C = AsmCfg<T>;
  const int smem = (int)sizeof(AsmSmem<T, NM, NF, PK>);
  if (*resident_ctas <= 0) {   // once per context (= per device): CTAs that fit the GPU at once
    TFA_CUDA(cudaFuncSetAttribute(k_assemble<T, NM, NF, PK>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int dev = 0, occ = 0, n_sm = 0;
    TFA_CUDA(cudaGetDevice(&dev));
    TFA_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    TFA_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_assemble<T, NM, NF, PK>, C::NT, smem));
    if (occ < 1) return set_error(TFA_ECUDA, "k_assemble does not fit on an SM");
    *resident_ctas = n_sm * occ;
  }
  const int64_t ntiles = (m.nc + T - 1) / T;
  const unsigned grid = (unsigned)std::min<int64_t>(ntiles, (int64_t)*resident_ctas);
  const double inv2dt = 1.0 / (2.0 * dt);
  const Limits lim{m.nc, (int64_t)m.F * m.nc, PK ? m.nc : m.nnzb, PK ? m.nnzb - m.nc : m.nnzb, m.nb, m.nst};
  // packed: the block map is the packed one (diagonal slot = the cell, mirror slots index the off-diagonal array)
  k_assemble<T, NM, NF, PK><<<grid, C::NT, smem, st>>>(m.nc, K, state, state_n, state_nm1, inv2dt, fown, m.cgeo.p,
                                                       m.nbrf.p, PK ? m.pblkmap.p : m.blkmap.p, ghost, rhs, vals,
                                                       vals_o, flags, lim);
  TFA_CUDA(cudaGetLastError());
  return 0;
}
}  // namespace

// vals_o == NULL: vals is the BSR value array.  Else packed output: vals = diagonal blocks [nc][324], vals_o =
// off-diagonal blocks [nnzb - nc][114].  resident_ctas: 4 slots, (F - 3) + 2 * packed.
int launch_assemble(const tfa_mesh& m, const Consts& K, const double* state, const double* state_n,
                    const double* state_nm1, double dt, const double* fown, const double* ghost, double* rhs,
                    double* vals, double* vals_o, int32_t* flags, int* resident_ctas, cudaStream_t st) {
  if (m.nc == 0) return 0;
  if (!vals) {
    const double inv2dt = 1.0 / (2.0 * dt);
    const Limits lim{m.nc, (int64_t)m.F * m.nc, 0, 0, m.nb, m.nst};
    if (m.F == 3)
      k_residual<3><<<cdiv(m.nc, RES_CELLS), 3 * RES_CELLS, 0, st>>>(m.nc, K, state, state_n, state_nm1, inv2dt, fown,
                                                                   m.cgeo.p, m.nbrf.p, ghost, rhs, flags, lim);
    else
      k_residual<4><<<cdiv(m.nc, RES_CELLS), 3 * RES_CELLS, 0, st>>>(m.nc, K, state, state_n, state_nm1, inv2dt, fown,
                                                                   m.cgeo.p, m.nbrf.p, ghost, rhs, flags, lim);
    TFA_CUDA(cudaGetLastError());
    return 0;
  }
#define TFA_LAUNCH(NF_, PK_, SLOT_)                                                                              \
  return launch_nm<TFA_ASM_T, 2, NF_, PK_>(m, K, state, state_n, state_nm1, dt, fown, ghost, rhs, vals, vals_o, \
                                           flags, resident_ctas + SLOT_, st)
  if (!vals_o) {
    if (m.F == 3) TFA_LAUNCH(3, false, 0);
    TFA_LAUNCH(4, false, 1);
  }
  if (m.F == 3) TFA_LAUNCH(3, true, 2);
  TFA_LAUNCH(4, true, 3);
#undef TFA_LAUNCH
}

}  // namespace tfa

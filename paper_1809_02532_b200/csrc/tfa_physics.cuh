// tfa_physics.cuh — device functions of the two-fluid model and its numerical fluxes.
//
// Written for the GPU path only (no code shared with oracle/): reciprocals are hoisted, FMA
// contraction is left to nvcc, branches are selects.  Citations: PAPER.md lines "L<n>".
#pragma once
#include "tfa_common.cuh"

#ifndef TFA_FAST_MATH64
#define TFA_FAST_MATH64 1   // 1: Newton-refined sqrt / reciprocal in the AUSM flux; 0: IEEE library sequences
#endif
#if TFA_FAST_MATH64
#define TFA_SQRT(x) nsqrt(x)
#define TFA_RCP(x) nrcp(x)
#else
#define TFA_SQRT(x) sqrt(x)
#define TFA_RCP(x) (1.0 / (x))
#endif

namespace tfa {

// Derived constants, computed once on the host and passed by value as a kernel parameter
// (the paper's "dco" device-config-option structs, L177/L195, flattened into one POD).
struct Consts {
  double c, c2;            // speed of light, c^2 (= 1/eps0 with mu0 = 1)
  double gp2;              // gamma_psi^2            (Eq. 2: gamma^2 Psi)
  double xc2;              // (chi c)^2              (Eq. 2: (chi c)^2 Phi)
  double gpc, xc;          // gamma_psi c, chi c     (cleaning wave speeds)
  double half_alpha;       // 0.5 * rusanov_alpha    (Eq. 9)
  double Rs[2];            // k_B/m_s
  double qm[2];            // q_s/m_s
  double gR[2];            // gamma R_s  (a^2 = gamma R T)
  double cp[2], cv[2];
  double Minf2[2];
  double Kp, Ku, sigma, beta16;
  double delta;
  double ref[NEQ];
  double venkK;
  int mask;
};

__host__ inline Consts make_consts(const tfa_physics& ph, const tfa_numerics& nu) {
  Consts K;
  K.c = ph.c;
  K.c2 = ph.c * ph.c;
  K.gp2 = ph.gamma_psi * ph.gamma_psi;
  K.xc = ph.chi_phi * ph.c;
  K.xc2 = K.xc * K.xc;
  K.gpc = ph.gamma_psi * ph.c;
  K.half_alpha = 0.5 * ph.rusanov_alpha;
  for (int s = 0; s < 2; ++s) {
    K.Rs[s] = s == 0 ? 1.0 : ph.mass_ratio;
    K.qm[s] = s == 0 ? 1.0 : -ph.mass_ratio;
    K.gR[s] = ph.gamma_gas * K.Rs[s];
    K.cv[s] = K.Rs[s] / (ph.gamma_gas - 1.0);
    K.cp[s] = ph.gamma_gas * K.Rs[s] / (ph.gamma_gas - 1.0);
    K.Minf2[s] = nu.ausm_Minf[s] * nu.ausm_Minf[s];
  }
  K.Kp = nu.ausm_Kp;
  K.Ku = nu.ausm_Ku;
  K.sigma = nu.ausm_sigma;
  K.beta16 = 16.0 * nu.ausm_beta;
  K.delta = nu.fd_delta;
  for (int k = 0; k < NEQ; ++k) K.ref[k] = nu.fd_ref[k];
  K.venkK = nu.venkat_K;
  K.mask = nu.term_mask;
  return K;
}

// index of the j-th variable (rho, u, v, w, T) of species s in the 18-vector
__device__ __forceinline__ int sp_idx(int s, int j) {
  return j == 0 ? 8 + s : (j == 4 ? 16 + s : 9 + 3 * s + j);
}

// Modified Rusanov flux of the Maxwell + cleaning rows (Eq. 9; F.n of Eq. 2).
// |A_n|dU = c dU_t + (cleaning speed) dU_n for B and E, (cleaning speed) dPsi/dPhi (S3).
__device__ __forceinline__ void maxwell_flux(const Consts& K, const double* L, const double* R, double nx,
                                             double ny, double* H) {
  double s[8], d[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    s[r] = L[r] + R[r];
    d[r] = R[r] - L[r];
  }
  const double dBn = d[0] * nx + d[1] * ny;
  const double dEn = d[3] * nx + d[4] * ny;
  const double kB = (K.gpc - K.c) * dBn;   // c(dB - dBn n) + gpc dBn n = c dB + (gpc - c) dBn n
  const double kE = (K.xc - K.c) * dEn;
  const double h = 0.5, a = K.half_alpha;
  // n x V = (ny Vz, -nx Vz, nx Vy - ny Vx)
  H[0] = h * (ny * s[5] + K.gp2 * s[6] * nx) - a * (K.c * d[0] + kB * nx);
  H[1] = h * (-nx * s[5] + K.gp2 * s[6] * ny) - a * (K.c * d[1] + kB * ny);
  H[2] = h * (nx * s[4] - ny * s[3]) - a * (K.c * d[2]);
  H[3] = h * (-K.c2 * (ny * s[2]) + K.xc2 * s[7] * nx) - a * (K.c * d[3] + kE * nx);
  H[4] = h * (K.c2 * (nx * s[2]) + K.xc2 * s[7] * ny) - a * (K.c * d[4] + kE * ny);
  H[5] = h * (-K.c2 * (nx * s[1] - ny * s[0])) - a * (K.c * d[5]);
  H[6] = h * (K.c2 * (s[0] * nx + s[1] * ny)) - a * (K.gpc * d[6]);
  H[7] = h * (s[3] * nx + s[4] * ny) - a * (K.xc * d[7]);
}

// Square root and reciprocal for the flux: a single-precision hardware seed (MUFU.RSQ / MUFU.RCP, 23
// bits) refined by two Newton steps in FP64 (fused multiply-adds only) -- about half the instructions
// and latency of the correctly rounded library sequences, error below 1 ulp.  Arguments are the
// positive, O(1)-scaled quantities of a physical state (a non-physical one is reported by the
// rho, T > 0 test, whatever these return).
__device__ __forceinline__ double nsqrt(double x) {
  const double y = (double)rsqrtf((float)x);
  double g = x * y, h = 0.5 * y;
  double r = fma(-g, h, 0.5);
  g = fma(g, r, g);
  h = fma(h, r, h);
  r = fma(-g, h, 0.5);
  g = fma(g, r, g);
  h = fma(h, r, h);
  return fma(fma(-g, g, x), h, g);   // last correction: g + (x - g^2) / (2 g)
}
__device__ __forceinline__ double nrcp(double d) {
  double y = (double)__frcp_rn((float)d);
  double e = fma(-d, y, 1.0);
  y = fma(y, e, y);
  e = fma(-d, y, 1.0);
  y = fma(y, e, y);
  e = fma(-d, y, 1.0);
  return fma(y, e, y);
}

// max / min as one compare and one select (fmax / fmin cost several instructions for their NaN rules; a NaN
// here can only come from a non-physical state, which is reported separately)
__device__ __forceinline__ double sel_max(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double sel_min(double a, double b) { return a < b ? a : b; }

// Multi-fluid AUSM+-up for one species (Eq. 10; Liou's scheme = ref. [30]; S4).
// L, R = (rho, u, v, w, T).  Returns true if the states are physical.
// Rs, gR, cp, Minf2: the species' constants (K.Rs[s], ...), passed in registers (warp uniform).
__device__ __forceinline__ bool ausm_flux(double Rs, double gR, double cp, double Minf2, const Consts& K,
                                          const double* L, const double* R, double nx, double ny, double* H) {
  const double rL = L[0], rR = R[0], TL = L[4], TR = R[4];
  const bool ok = (rL > 0.0) & (rR > 0.0) & (TL > 0.0) & (TR > 0.0);
  const double aL = TFA_SQRT(gR * TL), aR = TFA_SQRT(gR * TR);
  const double pL = rL * Rs * TL, pR = rR * Rs * TR;
  const double unL = L[1] * nx + L[2] * ny, unR = R[1] * nx + R[2] * ny;
  const double HtL = cp * TL + 0.5 * (L[1] * L[1] + L[2] * L[2] + L[3] * L[3]);
  const double HtR = cp * TR + 0.5 * (R[1] * R[1] + R[2] * R[2] + R[3] * R[3]);
  const double a12 = 0.5 * (aL + aR);
  const double ia = TFA_RCP(a12);
  const double ML = unL * ia, MR = unR * ia;
  const double Mb2 = 0.5 * (unL * unL + unR * unR) * (ia * ia);
  const double Mo = TFA_SQRT(sel_min(1.0, sel_max(Mb2, Minf2)));
  const double fa = Mo * (2.0 - Mo);
  const double al16 = 3.0 * (5.0 * fa * fa - 4.0);             // 16 alpha, alpha = 3/16 (-4 + 5 fa^2)
  // split Mach numbers and pressures; for |M| >= 1:  M4+ = max(M,0), P5+ = (M > 0), etc.
  const double m2pL = 0.25 * (ML + 1.0) * (ML + 1.0), m2mL = -0.25 * (ML - 1.0) * (ML - 1.0);
  const double m2pR = 0.25 * (MR + 1.0) * (MR + 1.0), m2mR = -0.25 * (MR - 1.0) * (MR - 1.0);
  const bool supL = fabs(ML) >= 1.0, supR = fabs(MR) >= 1.0;
  const double M4p = supL ? sel_max(ML, 0.0) : m2pL * (1.0 - K.beta16 * m2mL);
  const double M4m = supR ? sel_min(MR, 0.0) : m2mR * (1.0 + K.beta16 * m2pR);
  const double P5p = supL ? (ML > 0.0 ? 1.0 : 0.0) : m2pL * ((2.0 - ML) - al16 * ML * m2mL);
  const double P5m = supR ? (MR < 0.0 ? 1.0 : 0.0) : m2mR * ((-2.0 - MR) + al16 * MR * m2pR);
  const double rsum = rL + rR;
  const double Mp = -K.Kp * sel_max(1.0 - K.sigma * Mb2, 0.0) * (pR - pL) * (ia * ia) * TFA_RCP(fa * 0.5 * rsum);
  const double M12 = M4p + M4m + Mp;
  const bool up = M12 > 0.0;
  const double mdot = a12 * M12 * (up ? rL : rR);
  const double pu = -K.Ku * P5p * P5m * rsum * (fa * a12) * (unR - unL);
  const double p12 = P5p * pL + P5m * pR + pu;
  const bool upm = mdot > 0.0;
  H[0] = mdot;
  H[1] = mdot * (upm ? L[1] : R[1]) + p12 * nx;
  H[2] = mdot * (upm ? L[2] : R[2]) + p12 * ny;
  H[3] = mdot * (upm ? L[3] : R[3]);
  H[4] = mdot * (upm ? HtL : HtR);
  return ok;
}

// Two-fluid source (Eq. 4, Eq. 6; charge density rho_s q_s/m_s, S5; eps0 = 1/c^2)
__device__ __forceinline__ void source_terms(const Consts& K, const double* P, double* S) {
  const double qi = K.qm[0] * P[8], qe = K.qm[1] * P[9];   // q_s n_s
  const double Bx = P[0], By = P[1], Bz = P[2], Ex = P[3], Ey = P[4], Ez = P[5];
  const double ux = P[10], uy = P[11], uz = P[12], vx = P[13], vy = P[14], vz = P[15];
  S[0] = S[1] = S[2] = 0.0;
  S[3] = -K.c2 * (qi * ux + qe * vx);
  S[4] = -K.c2 * (qi * uy + qe * vy);
  S[5] = -K.c2 * (qi * uz + qe * vz);
  S[6] = 0.0;
  S[7] = K.c2 * (qi + qe);
  S[8] = S[9] = 0.0;
  S[10] = qi * (Ex + (uy * Bz - uz * By));
  S[11] = qi * (Ey + (uz * Bx - ux * Bz));
  S[12] = qi * (Ez + (ux * By - uy * Bx));
  S[13] = qe * (Ex + (vy * Bz - vz * By));
  S[14] = qe * (Ey + (vz * Bx - vx * Bz));
  S[15] = qe * (Ez + (vx * By - vy * Bx));
  S[16] = qi * (ux * Ex + uy * Ey + uz * Ez);
  S[17] = qe * (vx * Ex + vy * Ey + vz * Ez);
}

// conservative variables of one species, U = (rho, rho u, rho (c_v T + u^2/2))  (Eq. 5)
__device__ __forceinline__ void cons_species(const Consts& K, int s, const double* Q, double* U) {
  const double rho = Q[0];
  U[0] = rho;
  U[1] = rho * Q[1];
  U[2] = rho * Q[2];
  U[3] = rho * Q[3];
  U[4] = rho * (K.cv[s] * Q[4] + 0.5 * (Q[1] * Q[1] + Q[2] * Q[2] + Q[3] * Q[3]));
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

}  // namespace tfa

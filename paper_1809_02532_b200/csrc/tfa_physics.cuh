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
  double Minf2[2], Minf[2];
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
    K.Minf[s] = nu.ausm_Minf[s];
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
// and latency of the correctly rounded library sequences, error below 1 ulp (tests: tfa_probe_math).
// Precondition: the argument lies in the normal single-precision range (about 1e-38 .. 3e38) and is positive:
// zero, negative, subnormal-in-float or huge arguments give NaN / Inf, not the IEEE result.  The callers pass
// gamma R T, a_1/2, f_a rho of a physical state, O(1e-3 .. 1e3) in the normalised units; a non-physical state
// (rho <= 0 or T <= 0) is reported by the separate test, whatever these return.  TFA_FAST_MATH64 = 0 compiles
// the IEEE sequences instead.
// Error budget: the seed is good to 2^-22; one coupled Newton step squares that (2^-44), and the closing
// correction squares it again, below the last bit; a second full step before the correction (round 1 had one) only
// cost three FMAs on the flux's critical path.  Likewise two steps suffice for the reciprocal (2^-23 -> 2^-46 -> 2^-92).
__device__ __forceinline__ double nsqrt(double x) {
  const double y = (double)rsqrtf((float)x);
  double g = x * y, h = 0.5 * y;
  const double r = fma(-g, h, 0.5);
  g = fma(g, r, g);
  h = fma(h, r, h);
  return fma(fma(-g, g, x), h, g);   // last correction: g + (x - g^2) / (2 g)
}
__device__ __forceinline__ double nrcp(double d) {
  double y = (double)__frcp_rn((float)d);
  double e = fma(-d, y, 1.0);
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
__device__ __forceinline__ bool ausm_flux(double Rs, double gR, double cp, double Minf2, double Minf, const Consts& K,
                                          const double* L, const double* R, double nx, double ny, double* H) {
  const double rL = L[0], rR = R[0], TL = L[4], TR = R[4];
  const bool ok = (rL > 0.0) & (rR > 0.0) & (TL > 0.0) & (TR > 0.0);
  const double aL = TFA_SQRT(gR * TL), aR = TFA_SQRT(gR * TR);
  const double pL = rL * Rs * TL, pR = rR * Rs * TR;
  const double unL = L[1] * nx + L[2] * ny, unR = R[1] * nx + R[2] * ny;
  const double a12 = 0.5 * (aL + aR);
  const double ia = TFA_RCP(a12);
  const double ML = unL * ia, MR = unR * ia;
  const double Mb2 = 0.5 * (unL * unL + unR * unR) * (ia * ia);
  // M_o = sqrt(min(1, max(Mbar^2, M_inf^2))): below the cut-off it is M_inf itself (per lane, so that a result never
  // depends on which lanes share the warp); the square root is skipped when the whole warp is below it -- every face
  // of the GEM configurations, whose in-plane velocities vanish
  const bool low = Mb2 <= Minf2;
  double Mo = Minf;
  if (!__all_sync(__activemask(), low)) Mo = low ? Minf : TFA_SQRT(sel_min(1.0, Mb2));
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
  // the upwind side's velocity and total enthalpy H = c_p T + u^2 / 2 (only that side's is needed)
  const bool upm = mdot > 0.0;
  const double uu = upm ? L[1] : R[1], uv = upm ? L[2] : R[2], uw = upm ? L[3] : R[3], uT = upm ? TL : TR;
  H[0] = mdot;
  H[1] = mdot * uu + p12 * nx;
  H[2] = mdot * uv + p12 * ny;
  H[3] = mdot * uw;
  H[4] = mdot * (cp * uT + 0.5 * (uu * uu + uv * uv + uw * uw));
  return ok;
}

// Far side of a boundary face, per group of variables (the boundary loop of L260 folded into the face lanes;
// include/tfa.h TFA_BC_*).  TRANSMISSIVE: the own side again (S9).  WALL: its mirror image (S24): B and u_s flip
// their normal component, E its tangential ones (z included), Phi flips; Psi, rho_s, T_s are kept.  GHOST: `oth`
// already holds the caller's ghost state (fetched in place of a neighbour's face state) and is left alone.
__device__ __forceinline__ void bc_fields(int tag, const double* own, double nx, double ny, double* oth) {
  if (tag == TFA_BC_GHOST) return;
#pragma unroll
  for (int q = 0; q < 8; ++q) oth[q] = own[q];
  if (tag == TFA_BC_WALL) {
    const double Bn = own[0] * nx + own[1] * ny, En = own[3] * nx + own[4] * ny;
    oth[0] = own[0] - 2.0 * Bn * nx;
    oth[1] = own[1] - 2.0 * Bn * ny;
    oth[3] = 2.0 * En * nx - own[3];
    oth[4] = 2.0 * En * ny - own[4];
    oth[5] = -own[5];
    oth[7] = -own[7];
  }
}
__device__ __forceinline__ void bc_species(int tag, const double* own, double nx, double ny, double* oth) {
  if (tag == TFA_BC_GHOST) return;
#pragma unroll
  for (int q = 0; q < 5; ++q) oth[q] = own[q];
  if (tag == TFA_BC_WALL) {
    const double un = own[1] * nx + own[2] * ny;
    oth[1] = own[1] - 2.0 * un * nx;
    oth[2] = own[2] - 2.0 * un * ny;
  }
}
// tag of a boundary face from its packed neighbour entry (tfa_common.cuh): -1 - (4 b + tag)
__device__ __forceinline__ int bc_tag_of(int32_t packed) { return (-1 - packed) & 3; }
__device__ __forceinline__ int64_t bc_face_of(int32_t packed) { return (int64_t)((-1 - packed) >> 2); }

}  // namespace tfa

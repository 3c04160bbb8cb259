// sfh_device.cuh — device-side helpers of libsfh (sm_100a): TMA / mbarrier PTX wrappers and the
// per-face arithmetic of the scheme (limiter, primitive conversion, HLLC flux, eq. 16).
// Written from PAPER.md and DESIGN.md's readings; shares nothing with oracle/.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>

namespace sfh {

// ------------------------------------------------------------------------------------------------
// mbarrier + bulk-copy (TMA) wrappers.  One CTA-local mbarrier, phase 0 only (one block per CTA).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "SFH_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra SFH_DONE;\n"
      "bra SFH_WAIT;\n"
      "SFH_DONE:\n"
      "}\n" ::"r"(bar), "r"(parity)
      : "memory");
}
// contiguous global -> shared bulk copy (bytes multiple of 16, both addresses 16-byte aligned)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
// asynchronous prefetch of a contiguous global range into L2 (bytes multiple of 16)
__device__ __forceinline__ void prefetch_l2(const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// 4-D tiled tensor copy global -> shared; coordinates innermost first
__device__ __forceinline__ void tensor4_g2s(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(dst),
      "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

// ------------------------------------------------------------------------------------------------
// arithmetic of the scheme
// ------------------------------------------------------------------------------------------------

// minmod limiter (reading R12): 0 if the arguments differ in sign, else the one of smaller magnitude
__device__ __forceinline__ double minmod(double a, double b) {
  const double m = fmin(fabs(a), fabs(b));
  return (a * b <= 0.0) ? 0.0 : copysign(m, a);
}

// eq. (16)-(17): quadratic interpolation in time through U^n, U^{n+1/2}, U^{n+1}
__device__ __forceinline__ double time_interp(double U0, double Uh, double U1, double tau) {
  const double U1st = 2.0 * Uh - U0;                                   // eq. (17): first-order estimate of U^{n+1}
  return (U1 - U1st) * (tau * tau) + ((1.0 - tau) * U0 + tau * U1st);  // eq. (16)
}

// Arithmetic conventions of the CUDA path: the
// formulas are the oracle's, rearranged so that every fp64 division becomes ONE correctly rounded
// reciprocal (__drcp_rn, ~7 DFMA issue slots against ~12 for a division) shared by all quotients
// with that denominator, and sqrt(g P / rho) becomes (g P) rsqrt(g P rho) (~12 slots against ~25).
// Each rearrangement moves a result by a few ulp; nothing is approximated beyond rounding.

// conserved -> primitive (rho, vx, vy, vz, P), eq. (8); returns 1/rho
__device__ __forceinline__ double cons_to_prim(const double u[5], double gm1, double w[5]) {
  const double ir = __drcp_rn(u[0]);
  w[0] = u[0];
  w[1] = u[1] * ir;
  w[2] = u[2] * ir;
  w[3] = u[3] * ir;
  const double ke = (0.5 * (u[1] * u[1] + u[2] * u[2] + u[3] * u[3])) * ir;
  w[4] = gm1 * (u[4] - ke);
  return ir;
}

// primitive -> conserved (used where a stored half-step state W^{n+1/2} feeds eq. (16))
__device__ __forceinline__ void prim_to_cons(const double w[5], double igm1, double u[5]) {
  u[0] = w[0];
  u[1] = w[0] * w[1];
  u[2] = w[0] * w[2];
  u[3] = w[0] * w[3];
  u[4] = w[4] * igm1 + 0.5 * w[0] * (w[1] * w[1] + w[2] * w[2] + w[3] * w[3]);
}

// c_s = sqrt(gamma P / rho) as (gamma P) rsqrt(gamma P rho)
__device__ __forceinline__ double sound_speed(double gamma, double P, double rho) {
  const double gP = gamma * P;
  return gP * rsqrt(gP * rho);
}

// HLLC flux (Toro et al. 1994 as cited; Davis wave speeds, reading R6) in the face
// frame: u = normal velocity, v, w = the two tangential ones; Fn = (mass, normal momentum, tangential
// momenta, energy).  cL, cR = sound speeds of the two states; igm1 = 1/(gamma-1).
// Star state as in the oracle, U*_K = q_K (rho, rho S*, rho v, rho w, E + rho (S*-u)(S* + P/(rho (S_K-u))))_K
// with q_K = (S_K-u_K)/(S_K-S*); here 1/(S_K-S*) is formed once and the pressure term is carried as
// q rho (S*-u) P / (rho (S_K-u)) = P (S*-u)/(S_K-S*), which removes the third division.
// HAVE_E: the total energies of the two states are known (cell-centred states: the conserved E).
template <bool HAVE_E>
__device__ __forceinline__ void hllc_flux(double rL, double uL, double vL, double wL, double PL, double cL, double EL,
                                          double rR, double uR, double vR, double wR, double PR, double cR, double ER,
                                          double igm1, double Fn[5]) {
  const double SL = fmin(uL - cL, uR - cR);
  const double SR = fmax(uL + cL, uR + cR);
  double Ss = 0.0;
  const bool star = SL < 0.0 && SR > 0.0;
  if (star) {
    const double mL = rL * (SL - uL), mR = rR * (SR - uR);
    Ss = (PR - PL + mL * uL - mR * uR) * __drcp_rn(mL - mR);
  }
  const bool left = star ? (Ss >= 0.0) : (SL >= 0.0);
  const double r = left ? rL : rR, u = left ? uL : uR, v = left ? vL : vR, w = left ? wL : wR;
  const double P = left ? PL : PR, S = left ? SL : SR;
  const double E = HAVE_E ? (left ? EL : ER) : P * igm1 + 0.5 * r * (u * u + v * v + w * w);
  const double ru = r * u;
  Fn[0] = ru;
  Fn[1] = ru * u + P;
  Fn[2] = ru * v;
  Fn[3] = ru * w;
  Fn[4] = u * (E + P);
  if (star) {
    const double inv = __drcp_rn(S - Ss);
    const double q = (S - u) * inv;
    const double rv = r * v, rw = r * w, d = Ss - u;
    Fn[0] += S * (q * r - r);
    Fn[1] += S * (q * (r * Ss) - ru);
    Fn[2] += S * (q * rv - rv);
    Fn[3] += S * (q * rw - rw);
    Fn[4] += S * ((q * (E + (r * d) * Ss) + (P * d) * inv) - E);
  }
}

}  // namespace sfh

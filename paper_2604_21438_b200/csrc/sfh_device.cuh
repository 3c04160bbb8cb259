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

// conserved -> primitive (rho, vx, vy, vz, P), eq. (8)
__device__ __forceinline__ void cons_to_prim(const double u[5], double gm1, double w[5]) {
  const double rho = u[0];
  w[0] = rho;
  w[1] = u[1] / rho;
  w[2] = u[2] / rho;
  w[3] = u[3] / rho;
  const double ke = 0.5 * (u[1] * u[1] + u[2] * u[2] + u[3] * u[3]) / rho;
  w[4] = gm1 * (u[4] - ke);
}

// HLLC flux (Toro et al. 1994 as cited; Davis wave speeds, reading R6) in the face
// frame: u = normal velocity, v, w = the two tangential ones; Fn = (mass, normal momentum, tangential
// momenta, energy).  cL, cR = sound speeds of the two states.
__device__ __forceinline__ void hllc_flux(double rL, double uL, double vL, double wL, double PL, double cL, double rR,
                                          double uR, double vR, double wR, double PR, double cR, double gm1,
                                          double Fn[5]) {
  const double SL = fmin(uL - cL, uR - cR);
  const double SR = fmax(uL + cL, uR + cR);
  const double EL = PL / gm1 + 0.5 * rL * (uL * uL + vL * vL + wL * wL);
  const double ER = PR / gm1 + 0.5 * rR * (uR * uR + vR * vR + wR * wR);
  if (SL >= 0.0) {
    Fn[0] = rL * uL; Fn[1] = rL * uL * uL + PL; Fn[2] = rL * uL * vL; Fn[3] = rL * uL * wL; Fn[4] = uL * (EL + PL);
  } else if (SR <= 0.0) {
    Fn[0] = rR * uR; Fn[1] = rR * uR * uR + PR; Fn[2] = rR * uR * vR; Fn[3] = rR * uR * wR; Fn[4] = uR * (ER + PR);
  } else {
    const double mL = rL * (SL - uL), mR = rR * (SR - uR);
    const double Ss = (PR - PL + mL * uL - mR * uR) / (mL - mR);
    const bool left = Ss >= 0.0;
    const double r = left ? rL : rR, u = left ? uL : uR, v = left ? vL : vR, w = left ? wL : wR;
    const double P = left ? PL : PR, E = left ? EL : ER, S = left ? SL : SR, mk = left ? mL : mR;
    // U*_K = (S_K - u_K)/(S_K - S*) (rho, rho S*, rho v, rho w, E + rho (S* - u)(S* + P/(rho (S_K - u))))
    const double q = (S - u) / (S - Ss);
    const double ru = r * u;
    Fn[0] = ru + S * (q * r - r);
    Fn[1] = (ru * u + P) + S * (q * (r * Ss) - ru);
    Fn[2] = ru * v + S * (q * (r * v) - r * v);
    Fn[3] = ru * w + S * (q * (r * w) - r * w);
    Fn[4] = u * (E + P) + S * (q * (E + r * (Ss - u) * (Ss + P / mk)) - E);
  }
}

__device__ __forceinline__ double sound_speed(double gamma, double P, double rho) { return sqrt(gamma * P / rho); }

}  // namespace sfh

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

// minmod(a, b) / 2 without multiplying the arguments: the difference of smaller magnitude, times 1/2 if the signs
// agree and 0 if not (compare + select; the form the corrector's walk uses)
__device__ __forceinline__ double half_minmod(double a, double b) {
  const double m = fabs(a) < fabs(b) ? a : b;
  const bool same = (__double2hiint(a) ^ __double2hiint(b)) >= 0;
  return __hiloint2double(same ? 0x3fe00000 : 0, 0) * m;
}

// eq. (16)-(17): quadratic interpolation in time through U^n, U^{n+1/2}, U^{n+1}
__device__ __forceinline__ double time_interp(double U0, double Uh, double U1, double tau) {
  const double U1st = 2.0 * Uh - U0;                                   // eq. (17): first-order estimate of U^{n+1}
  return (U1 - U1st) * (tau * tau) + ((1.0 - tau) * U0 + tau * U1st);  // eq. (16)
}

// Arithmetic conventions of the stage kernels.
// The stage kernels are bound by the fp64 pipe and by instruction issue, so every formula of the
// oracle is evaluated in the form that needs the fewest fp64 instructions and no branches:
//  * 1/x and 1/sqrt(x) start from the hardware seed (MUFU.RCP64H / MUFU.RSQ64H, which read only the
//    upper 32 bits of x: relative error < 2^-19) followed by ONE third-order step (error ~ e^3 < 2^-57,
//    i.e. the result is within 1 ulp); no range checks: the arguments are ratios of positive, normal
//    densities, pressures and wave-speed differences (a non-positive rho or P is reported by sfh_status
//    and has no defined result on either side);
//  * min/max/minmod are compare+select (no NaN fix-ups);
//  * the HLLC star flux is written as F_K + S_K (U*_K - U_K) with U*_K - U_K expanded analytically.
// Each rearrangement moves a result by a few ulp; nothing is approximated beyond rounding.

__device__ __forceinline__ double rcp_fast(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);
  const double t = fma(e, e, e);
  return fma(y, t, y);                       // y (1 + e + e^2)
}
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y * y, 1.0);      // 1 - x y^2
  const double p = fma(e, 0.375, 0.5);
  return fma(p, y * e, y);                   // y (1 + e/2 + 3 e^2/8)
}
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

// conserved -> primitive (rho, vx, vy, vz, P), eq. (8); returns 1/rho
__device__ __forceinline__ double cons_to_prim(const double u[5], double gm1, double w[5]) {
  const double ir = rcp_fast(u[0]);
  w[0] = u[0];
  w[1] = u[1] * ir;
  w[2] = u[2] * ir;
  w[3] = u[3] * ir;
  const double m2 = fma(u[3], u[3], fma(u[2], u[2], u[1] * u[1]));
  const double ke = (0.5 * ir) * m2;
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
  return gP * rsqrt_fast(gP * rho);
}

// CFL speed of one cell (reading R16): max_d |v_d| + c_s, from the conserved state.  Every kernel that
// produces a block's maximum speed calls this, so the cached per-block maxima and the reduction over
// whole states agree bit for bit.
__device__ __forceinline__ double cell_speed(const double u[5], double gamma, double gm1) {
  // (max_d |m_d| + sqrt(gamma (gamma-1) (rho E - |m|^2 / 2))) / rho: c_s rho = sqrt(gamma P rho) without forming P
  // or the velocities (19 fp64 instructions instead of 26; the corrector's helpers evaluate this for every cell)
  const double m2 = fma(u[3], u[3], fma(u[2], u[2], u[1] * u[1]));
  const double x = (gamma * gm1) * fma(-0.5, m2, u[0] * u[4]);
  const double mm = fmax(fmax(fabs(u[1]), fabs(u[2])), fabs(u[3]));
  return fma(x, rsqrt_fast(x), mm) * rcp_fast(u[0]);
}

__device__ __forceinline__ double warp_max(double x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x = fmax(x, __shfl_xor_sync(0xffffffffu, x, o));
  return x;
}

// HLLC flux (Toro et al. 1994 as cited; Davis wave speeds, reading R6) in the face
// frame: u = normal velocity, v, w = the two tangential ones; Fn = (mass, normal momentum, tangential
// momenta, energy).  cL, cR = sound speeds of the two states; igm1 = 1/(gamma-1).
// Branch-free.  With K the upwind side (L if S* >= 0, else R: S_L < S* < S_R holds strictly for Davis speeds and
// positive rho, P, so S_L >= 0 implies S* > 0 and S_R <= 0 implies S* < 0),
//   F = F_K + s (U*_K - U_K),  s = S_K clipped at zero (min(S_L, 0) or max(S_R, 0): zero in the supersonic cases),
// and with d = S* - u_K, g = d/(S_K - S*), A = rho_K g the oracle's star state
//   U*_K = q (rho, rho S*, rho v, rho w, E + rho d (S* + P/(rho (S_K-u))))_K,  q = (S_K-u_K)/(S_K-S*) = 1 + g
// gives  U*_K - U_K = (A, rho d + A S*, A v, A w, g (E + P + rho d S*) + rho d S*).
// The denominator m_L - m_R of S* is strictly negative for positive rho (m_L < 0 < m_R), whatever
// the wave pattern, so S* is always finite, and S_K - S* never vanishes.
// HAVE_E: the total energies of the two states are known (cell-centred states: the conserved E).
template <bool HAVE_E>
__device__ __forceinline__ void hllc_flux(double rL, double uL, double vL, double wL, double PL, double cL, double EL,
                                          double rR, double uR, double vR, double wR, double PR, double cR, double ER,
                                          double igm1, double Fn[5]) {
  const double SL = dmin(uL - cL, uR - cR);
  const double SR = dmax(uL + cL, uR + cR);
  const double mL = rL * (SL - uL), mR = rR * (SR - uR);
  const double num = ((PR - PL) + mL * uL) - mR * uR, den = mL - mR;   // S* = num / den, den < 0
  const double Ss = num * rcp_fast(den);
  // S_L < S* < S_R strictly (Davis speeds, positive rho and P), so the upwind side is the sign of S* alone, and
  // clipping the chosen wave speed at zero drops the star term in the supersonic cases
  const bool left = !(num > 0.0);            // S* = num / den >= 0 with den < 0: known before the reciprocal lands
  const double r = left ? rL : rR, u = left ? uL : uR, v = left ? vL : vR, w = left ? wL : wR;
  const double P = left ? PL : PR, S = left ? SL : SR;
  const double E = HAVE_E ? (left ? EL : ER) : fma(P, igm1, (0.5 * r) * fma(w, w, fma(v, v, u * u)));
  const double ru = r * u, EP = E + P;
  const double inv = den * rcp_fast(fma(S, den, -num));   // 1 / (S - S*) = den / (S den - num): independent of the first reciprocal
  const bool in = left ? SL < 0.0 : SR > 0.0;
  const double s = in ? S : 0.0;
  const double d = Ss - u, g = d * inv, rd = r * d, A = rd * inv, rdS = rd * Ss;
  Fn[0] = fma(s, A, ru);
  Fn[1] = fma(s, fma(A, Ss, rd), fma(ru, u, P));
  Fn[2] = Fn[0] * v;                         // tangential momenta are carried by the mass flux
  Fn[3] = Fn[0] * w;
  Fn[4] = fma(s, fma(g, EP + rdS, rdS), u * EP);
}

// Roe flux ("the method of Roe (1981)"; reading R30) in the face frame, same conventions as
// hllc_flux.  Roe averages weighted by sqrt(rho) (1/sqrt(rho) from the hardware seed: sqrt(rho) = rho rsqrt(rho),
// sqrt(rho) H = (E + P) rsqrt(rho)); wave strengths alpha_k and eigenvectors K_k of the averaged state;
// Harten's entropy fix on the two acoustic waves, delta = c~/10;
//   F = ((F_L + F_R) - sum_k |lambda_k| alpha_k K_k) / 2,
// with the five dissipation components summed wave by wave: b_k = |lambda_k| alpha_k,
//   D = (b1+b2+b5, b1 (u-c) + b2 u + b5 (u+c), D0 v + b3, D0 w + b4, b1 (H - u c) + b2 q^2/2 + b3 v + b4 w + b5 (H + u c)).
// HAVE_E (cell-centred states): the total energies EL, ER and isL, isR = 1/sqrt(rho) are known.
template <bool HAVE_E>
__device__ __forceinline__ void roe_flux(double rL, double uL, double vL, double wL, double PL, double EL, double isL,
                                         double rR, double uR, double vR, double wR, double PR, double ER, double isR,
                                         double gm1, double igm1, double Fn[5]) {
  const double eL = HAVE_E ? EL : fma(PL, igm1, (0.5 * rL) * fma(wL, wL, fma(vL, vL, uL * uL)));
  const double eR = HAVE_E ? ER : fma(PR, igm1, (0.5 * rR) * fma(wR, wR, fma(vR, vR, uR * uR)));
  const double iL = HAVE_E ? isL : rsqrt_fast(rL), iR = HAVE_E ? isR : rsqrt_fast(rR);
  const double sL = rL * iL, sR = rR * iR;
  const double iw = rcp_fast(sL + sR);
  const double aL = sL * iw, aR = sR * iw;
  const double ut = fma(aL, uL, aR * uR), vt = fma(aL, vL, aR * vR), wt = fma(aL, wL, aR * wR);
  const double epL = eL + PL, epR = eR + PR;
  const double Ht = fma(epL, iL, epR * iR) * iw;
  const double q2 = fma(wt, wt, fma(vt, vt, ut * ut));
  const double c2 = gm1 * fma(-0.5, q2, Ht);
  const double ic = rsqrt_fast(c2), ct = c2 * ic, ic2 = ic * ic;
  const double rt = sL * sR;
  const double dr = rR - rL, du = uR - uL, dv = vR - vL, dw = wR - wL, dP = PR - PL;
  const double rcu = (rt * ct) * du, hic2 = 0.5 * ic2;
  const double a1 = (dP - rcu) * hic2, a5 = (dP + rcu) * hic2;
  const double a2 = fma(-dP, ic2, dr);
  const double delta = 0.1 * ct, idel = 10.0 * ic;
  const double lm = ut - ct, lp = ut + ct;
  const double fm = 0.5 * fma(lm * lm, idel, delta), fp = 0.5 * fma(lp * lp, idel, delta);
  const double l1 = fabs(lm) < delta ? fm : fabs(lm);
  const double l5 = fabs(lp) < delta ? fp : fabs(lp);
  const double l2 = fabs(ut);
  const double b1 = l1 * a1, b5 = l5 * a5, b2 = l2 * a2, b3 = l2 * (rt * dv), b4 = l2 * (rt * dw);
  const double D0 = (b1 + b2) + b5;
  const double D1 = fma(b5, lp, fma(b1, lm, b2 * ut));
  const double D2 = fma(D0, vt, b3), D3 = fma(D0, wt, b4);
  const double uc = ut * ct;
  const double D4 = fma(b5, Ht + uc, fma(b1, Ht - uc, fma(b2, 0.5 * q2, fma(b3, vt, b4 * wt))));
  const double mL = rL * uL, mR = rR * uR;
  Fn[0] = 0.5 * ((mL + mR) - D0);
  Fn[1] = 0.5 * ((fma(mL, uL, PL) + fma(mR, uR, PR)) - D1);
  Fn[2] = 0.5 * (fma(mL, vL, mR * vR) - D2);
  Fn[3] = 0.5 * (fma(mL, wL, mR * wR) - D3);
  Fn[4] = 0.5 * (fma(uL, epL, uR * epR) - D4);
}

}  // namespace sfh

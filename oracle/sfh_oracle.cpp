// sfh_oracle.cpp — CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, literal CPU implementation of the per-step hydrodynamics update on
// octree block-structured AMR grids of arxiv/paper_2604_21438 (SFUMATO#), written from
// PAPER.md and the readings R1..R20 listed in DESIGN.md ("Readings of the paper").
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this library.  It shares no code, header, table or helper with the CUDA
// path under paper_2604_21438_b200/csrc/ and neither includes the other.
//
// Structure (deliberately unlike the GPU path): every block stores a GHOSTED 12^3 array;
// ghost cells are filled by a global-index accessor get(level, I,J,K) that looks blocks up in
// a hash map and falls back to slope-limited prolongation from the next coarser level; there
// are no neighbour tables.  fp64 everywhere, compiled with
// -ffp-contract=off so every operation rounds once, as written.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"): exact Riemann solution of the Sod tube,
// HLLC identities, conservation to round-off on periodic AMR meshes with flux correction
// (and its failure with reflux switched off), uniform == fully refined bitwise, mirror
// symmetry, free-stream preservation, eq. (16) closed forms, eq. (14)-(15) table,
// prolong/restrict identities, 1-D invariance, contact advection, 2nd-order convergence; the time axis
// (tests/test_oracle_time_pins.py): linear advection exact to round-off on a sub-cycled AMR mesh (fixes
// the tau / tau_half schedule of advance_adaptive and the copies fill_ghosts_level reads), fill_ghosts at
// tau in {0, 1/4, 1/2, 3/4, 1} against the expanded eq. (16), the CFL step in closed form.
// Parity unpinned by the paper (any reasonable choice passes every pin; fixed only by
// DESIGN.md): Davis wave speeds (R6), first-order predictor (R8), primitive-variable
// reconstruction (R11), minmod limiter (R12), CFL speed definition (R16), the entropy-fix width of
// the Roe solver (R30; the Roe flux itself is pinned by tests/test_oracle_roe_pins.py).
//
// Passive scalars (eq. 12-13; reading R32): up to 8 extra conserved densities
// rho*s per cell, carried by the Riemann solver's mass flux, reconstructed, prolonged, restricted and refluxed like
// the hydro variables; pins in tests/test_oracle_scalar_pins.py.
//
// Passages followed: PAPER.md:39-44,58 (Euler equations, E of eq. 8); :96 (blocks, levels);
// :108-120 (time marching, eq. 14-15); :126 (MUSCL, predictor-corrector, HLLC);
// :128 (ghost interpolation in space and time, reflux); :142-148 (three stored time levels,
// eq. 16-17); :599 (correction between coarse and fine cells = restriction).

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <functional>
#include <set>
#include <unordered_map>
#include <vector>

namespace {

#ifndef SFH_ORACLE_N
#define SFH_ORACLE_N 8
#endif
constexpr int N = SFH_ORACLE_N;   // cells per block edge: 8; built a second time with 16
constexpr int NF = N * N;         // cells of a block face
constexpr int G = 2;    // ghost layers                    BASELINE.json configs
constexpr int M = N + 2 * G;
constexpr int NV = 5;   // rho, rho vx, rho vy, rho vz, rho E
constexpr int NSMAX = 8;          // passive scalars rho*s advected with the gas (eq. 12-13; reading R32)
constexpr int NVMAX = NV + NSMAX; // a mesh carries nv = NV + nscalar conserved variables per cell
constexpr int M3 = M * M * M;

struct Config {            // binary layout mirrored by the ctypes Structure in oracle/binding.py
  int32_t nb0[3];
  int32_t ncell, nghost;
  int32_t max_level;
  int32_t bc[3][2];        // 0 periodic, 1 outflow (zero gradient)
  double box_len[3];
  double gamma, cfl;
  int32_t nscalar;         // passive scalars carried besides the 5 hydro variables (0..NSMAX)
};

struct Src {               // how a block cell is read
  int mode;                // 0: copy `which`;  1: eq. (16) time interpolation at tau; -1: invalid
  int which;
  double tau;
};

struct Mesh {
  Config cfg;
  int64_t nb = 0;
  int nlev = 0;
  int nv = NV;             // conserved variables per cell: NV + cfg.nscalar
  int64_t blk = NV * M3;   // doubles per ghosted block: nv * 12^3
  std::vector<int> lev, bx, by, bz;
  std::vector<char> leaf;
  std::unordered_map<uint64_t, int> map;
  std::vector<std::vector<int>> of_level;
  double* U[3] = {nullptr, nullptr, nullptr};
  // flux registers (Berger & Colella as cited): per flagged (block, face)
  std::vector<int> rslot, fslot;     // [nb*6] -> slot or -1
  std::vector<double> R, FH;         // [slot][nv][N][N]
  int reflux_on = 1;
  int riemann = 0;                   // 0 HLLC, 1 Roe (PAPER.md:126 names both)
  char err[256] = {0};
};

inline uint64_t key(int l, int x, int y, int z) {
  return (uint64_t(l) << 60) | (uint64_t(uint32_t(x) & 0xFFFFF) << 40) |
         (uint64_t(uint32_t(y) & 0xFFFFF) << 20) | uint64_t(uint32_t(z) & 0xFFFFF);
}

inline int find(const Mesh& m, int l, int x, int y, int z) {
  auto it = m.map.find(key(l, x, y, z));
  return it == m.map.end() ? -1 : it->second;
}

inline int gidx(int v, int i, int j, int k) {  // i,j,k in [-G, N+G)
  return ((v * M + (k + G)) * M + (j + G)) * M + (i + G);
}

inline double h_of(const Mesh& m, int l) {
  return m.cfg.box_len[0] / (double(m.cfg.nb0[0]) * N * double(1 << l));
}

// ---------------------------------------------------------------- eq. (16)-(17)
inline double time_interp(double U0, double Uh, double U1, double tau) {
  const double U1st = 2.0 * Uh - U0;                                    // eq. (17)
  return (U1 - U1st) * (tau * tau) + ((1.0 - tau) * U0 + tau * U1st);   // eq. (16), tau=(t-t^n)/(t^{n+1}-t^n)
}

inline void cell_value(const Mesh& m, int b, int i, int j, int k, const Src& s, double out[NVMAX]) {
  for (int v = 0; v < m.nv; ++v) {
    const int64_t o = int64_t(b) * m.blk + gidx(v, i, j, k);
    if (s.mode == 0) out[v] = m.U[s.which][o];
    else out[v] = time_interp(m.U[0][o], m.U[1][o], m.U[2][o], s.tau);
  }
}

inline double minmod(double a, double b) {          // reading R12
  if (a * b <= 0.0) return 0.0;
  const double s = a > 0.0 ? 1.0 : -1.0;
  return s * std::min(std::fabs(a), std::fabs(b));
}

// Domain boundary rule applied to a global cell index of level l (reading R1).
inline bool apply_bc(const Mesh& m, int l, int idx[3]) {
  for (int d = 0; d < 3; ++d) {
    const int n = (m.cfg.nb0[d] * N) << l;
    if (idx[d] < 0) {
      if (m.cfg.bc[d][0] == 0) idx[d] += n; else idx[d] = 0;
    } else if (idx[d] >= n) {
      if (m.cfg.bc[d][1] == 0) idx[d] -= n; else idx[d] = n - 1;
    }
  }
  return true;
}

// Accessor: value of global cell (I,J,K) of level l (readings R1, R3).  srcs[lv] says how
// level lv's stored data are read.  Returns false on a nesting violation.
bool get(const Mesh& m, int l, int I, int J, int K, const Src* srcs, double out[NVMAX]) {
  int idx[3] = {I, J, K};
  apply_bc(m, l, idx);
  const int b = find(m, l, idx[0] / N, idx[1] / N, idx[2] / N);
  if (b >= 0) {
    if (srcs[l].mode < 0) return false;
    cell_value(m, b, idx[0] % N, idx[1] % N, idx[2] % N, srcs[l], out);
    return true;
  }
  if (l == 0) return false;
  // slope-limited linear prolongation from level l-1 (reading R3; PAPER.md:128 defers the
  // formula to a paper that is not available)
  const int c[3] = {idx[0] >> 1, idx[1] >> 1, idx[2] >> 1};
  double Q[NVMAX], Qp[NVMAX], Qm[NVMAX];
  if (!get(m, l - 1, c[0], c[1], c[2], srcs, Q)) return false;
  for (int v = 0; v < m.nv; ++v) out[v] = Q[v];
  for (int d = 0; d < 3; ++d) {
    int cp[3] = {c[0], c[1], c[2]}, cm[3] = {c[0], c[1], c[2]};
    cp[d] += 1; cm[d] -= 1;
    if (!get(m, l - 1, cp[0], cp[1], cp[2], srcs, Qp)) return false;
    if (!get(m, l - 1, cm[0], cm[1], cm[2], srcs, Qm)) return false;
    const double sigma = (idx[d] & 1) ? 1.0 : -1.0;
    for (int v = 0; v < m.nv; ++v) {
      const double slope = minmod(Qp[v] - Q[v], Q[v] - Qm[v]);
      out[v] = out[v] + sigma * 0.25 * slope;
    }
  }
  return true;
}

// ------------------------------------------------------------------ ghost fill (a2, a3, a5)
int fill_ghosts_level(Mesh& m, int l, int which, int interp, double tau) {
  std::vector<Src> srcs(m.nlev);
  for (int lv = 0; lv < m.nlev; ++lv) srcs[lv] = Src{0, which, 0.0};
  if (interp) {
    for (int lv = 0; lv < m.nlev; ++lv) srcs[lv] = Src{-1, 0, 0.0};
    srcs[l] = Src{0, which, 0.0};
    if (l > 0) srcs[l - 1] = Src{1, 0, tau};
  }
  const std::vector<int>& blocks = m.of_level[l];
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 8) reduction(+ : bad)
  for (int64_t t = 0; t < (int64_t)blocks.size(); ++t) {
    const int b = blocks[t];
    double* dst = m.U[which] + int64_t(b) * m.blk;
    double val[NVMAX];
    for (int k = -G; k < N + G; ++k)
      for (int j = -G; j < N + G; ++j)
        for (int i = -G; i < N + G; ++i) {
          if (i >= 0 && i < N && j >= 0 && j < N && k >= 0 && k < N) continue;
          if (!get(m, l, m.bx[b] * N + i, m.by[b] * N + j, m.bz[b] * N + k, srcs.data(), val)) { bad++; continue; }
          for (int v = 0; v < m.nv; ++v) dst[gidx(v, i, j, k)] = val[v];
        }
  }
  if (bad) { snprintf(m.err, sizeof m.err, "fill_ghosts: %d cells could not be resolved (nesting)", bad); return -2; }
  return 0;
}

// ------------------------------------------------------------------ primitives, eq. (8)
inline void cons_to_prim(const double U[NV], double gamma, double W[NV]) {
  const double rho = U[0];
  W[0] = rho;
  W[1] = U[1] / rho;
  W[2] = U[2] / rho;
  W[3] = U[3] / rho;
  const double ke = 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / rho;
  W[4] = (gamma - 1.0) * (U[4] - ke);
}

// ------------------------------------------------------------------ HLLC (reading R6)
// W = (rho, vx, vy, vz, P); flux through a face with normal along axis d.
void hllc(const double WLin[NV], const double WRin[NV], int d, double gamma, double F[NV]) {
  const int n = 1 + d, t1 = 1 + (d + 1) % 3, t2 = 1 + (d + 2) % 3;
  const double rL = WLin[0], uL = WLin[n], vL = WLin[t1], wL = WLin[t2], PL = WLin[4];
  const double rR = WRin[0], uR = WRin[n], vR = WRin[t1], wR = WRin[t2], PR = WRin[4];
  const double cL = std::sqrt(gamma * PL / rL);
  const double cR = std::sqrt(gamma * PR / rR);
  const double SL = std::min(uL - cL, uR - cR);   // Davis estimate
  const double SR = std::max(uL + cL, uR + cR);
  const double EL = PL / (gamma - 1.0) + 0.5 * rL * (uL * uL + vL * vL + wL * wL);
  const double ER = PR / (gamma - 1.0) + 0.5 * rR * (uR * uR + vR * vR + wR * wR);
  double Fn[NV];  // in the face frame: (mass, normal mom, t1 mom, t2 mom, energy)
  if (SL >= 0.0) {
    Fn[0] = rL * uL; Fn[1] = rL * uL * uL + PL; Fn[2] = rL * uL * vL; Fn[3] = rL * uL * wL; Fn[4] = uL * (EL + PL);
  } else if (SR <= 0.0) {
    Fn[0] = rR * uR; Fn[1] = rR * uR * uR + PR; Fn[2] = rR * uR * vR; Fn[3] = rR * uR * wR; Fn[4] = uR * (ER + PR);
  } else {
    const double mL = rL * (SL - uL), mR = rR * (SR - uR);
    const double Sstar = (PR - PL + mL * uL - mR * uR) / (mL - mR);
    double r, u, v, w, P, E, S, mk;
    if (Sstar >= 0.0) { r = rL; u = uL; v = vL; w = wL; P = PL; E = EL; S = SL; mk = mL; }
    else              { r = rR; u = uR; v = vR; w = wR; P = PR; E = ER; S = SR; mk = mR; }
    // U*_K = (S_K-u_K)/(S_K-S*) (rho, rho S*, rho v, rho w, E + rho (S*-u)(S* + P/(rho (S_K-u))))_K
    const double q = (S - u) / (S - Sstar);
    const double Us[NV] = {q * r, q * (r * Sstar), q * (r * v), q * (r * w),
                           q * (E + r * (Sstar - u) * (Sstar + P / mk))};
    const double Uk[NV] = {r, r * u, r * v, r * w, E};
    const double Fk[NV] = {r * u, r * u * u + P, r * u * v, r * u * w, u * (E + P)};
    for (int c = 0; c < NV; ++c) Fn[c] = Fk[c] + S * (Us[c] - Uk[c]);
  }
  F[0] = Fn[0]; F[n] = Fn[1]; F[t1] = Fn[2]; F[t2] = Fn[3]; F[4] = Fn[4];
}

// ------------------------------------------------------------------ Roe ("the method of Roe (1981)"; reading R30)
// Roe's linearised Riemann solver as in Roe (1981), written with the wave strengths and right
// eigenvectors of the Roe-averaged state (rho~ = sqrt(rhoL rhoR); u~, v~, w~, H~ weighted by sqrt(rho)):
//   F = (F_L + F_R)/2 - (1/2) sum_k |lambda_k| alpha_k K_k,
//   lambda = (u~ - c~, u~, u~, u~, u~ + c~),  c~^2 = (gamma-1)(H~ - |v~|^2/2),
//   alpha_1,5 = (dP -/+ rho~ c~ du)/(2 c~^2), alpha_2 = drho - dP/c~^2, alpha_3 = rho~ dv, alpha_4 = rho~ dw,
//   K_1,5 = (1, u~ -/+ c~, v~, w~, H~ -/+ u~ c~), K_2 = (1, u~, v~, w~, |v~|^2/2), K_3 = (0,0,1,0,v~), K_4 = (0,0,0,1,w~).
// The paper gives no entropy fix; reading R30: Harten's (1983) on the two acoustic waves,
// |lambda| -> (lambda^2 + delta^2)/(2 delta) where |lambda| < delta, delta = c~/10.  PARITY UNPINNED (delta).
void roe(const double WLin[NV], const double WRin[NV], int d, double gamma, double F[NV]) {
  const int n = 1 + d, t1 = 1 + (d + 1) % 3, t2 = 1 + (d + 2) % 3;
  const double rL = WLin[0], uL = WLin[n], vL = WLin[t1], wL = WLin[t2], PL = WLin[4];
  const double rR = WRin[0], uR = WRin[n], vR = WRin[t1], wR = WRin[t2], PR = WRin[4];
  const double EL = PL / (gamma - 1.0) + 0.5 * rL * (uL * uL + vL * vL + wL * wL);
  const double ER = PR / (gamma - 1.0) + 0.5 * rR * (uR * uR + vR * vR + wR * wR);
  const double HL = (EL + PL) / rL, HR = (ER + PR) / rR;
  const double sL = std::sqrt(rL), sR = std::sqrt(rR), sw = sL + sR;
  const double rt = sL * sR;
  const double ut = (sL * uL + sR * uR) / sw, vt = (sL * vL + sR * vR) / sw, wt = (sL * wL + sR * wR) / sw;
  const double Ht = (sL * HL + sR * HR) / sw;
  const double q2 = ut * ut + vt * vt + wt * wt;
  const double c2 = (gamma - 1.0) * (Ht - 0.5 * q2);
  const double ct = std::sqrt(c2);
  const double dr = rR - rL, du = uR - uL, dv = vR - vL, dw = wR - wL, dP = PR - PL;
  const double a1 = (dP - rt * ct * du) / (2.0 * c2);
  const double a2 = dr - dP / c2;
  const double a3 = rt * dv, a4 = rt * dw;
  const double a5 = (dP + rt * ct * du) / (2.0 * c2);
  const double delta = 0.1 * ct;
  auto fixed = [delta](double lam) {
    const double al = std::fabs(lam);
    return al < delta ? (lam * lam + delta * delta) / (2.0 * delta) : al;
  };
  const double l1 = fixed(ut - ct), l2 = std::fabs(ut), l5 = fixed(ut + ct);
  const double K1[NV] = {1.0, ut - ct, vt, wt, Ht - ut * ct};
  const double K2[NV] = {1.0, ut, vt, wt, 0.5 * q2};
  const double K3[NV] = {0.0, 0.0, 1.0, 0.0, vt};
  const double K4[NV] = {0.0, 0.0, 0.0, 1.0, wt};
  const double K5[NV] = {1.0, ut + ct, vt, wt, Ht + ut * ct};
  const double FL[NV] = {rL * uL, rL * uL * uL + PL, rL * uL * vL, rL * uL * wL, uL * (EL + PL)};
  const double FR[NV] = {rR * uR, rR * uR * uR + PR, rR * uR * vR, rR * uR * wR, uR * (ER + PR)};
  double Fn[NV];
  for (int c = 0; c < NV; ++c)
    Fn[c] = 0.5 * (FL[c] + FR[c]) -
            0.5 * (l1 * a1 * K1[c] + l2 * (a2 * K2[c] + a3 * K3[c] + a4 * K4[c]) + l5 * a5 * K5[c]);
  F[0] = Fn[0]; F[n] = Fn[1]; F[t1] = Fn[2]; F[t2] = Fn[3]; F[4] = Fn[4];
}

inline void riemann_flux(const Mesh& m, const double WL[NV], const double WR[NV], int d, double F[NV]) {
  if (m.riemann == 1) roe(WL, WR, d, m.cfg.gamma, F);
  else hllc(WL, WR, d, m.cfg.gamma, F);
}

inline int fidx(int v, int f, int a, int b) { return ((v * (N + 1) + f) * N + b) * N + a; }  // face f=0..N, tangential (a fastest)

inline void cell_of(int d, int c, int a, int b, int& i, int& j, int& k) {
  // c along d; (a,b) = the other two axes in increasing axis order
  if (d == 0) { i = c; j = a; k = b; }
  else if (d == 1) { i = a; j = c; k = b; }
  else { i = a; j = b; k = c; }
}

// ------------------------------------------------------------------ passive scalars (eq. 12-13; reading R32)
// A scalar is carried as the conserved density q = rho * s (y_i n_H of eq. 12, rho C_d T_d of eq. 13; source terms are
// not part of this path).  Its primitive is s = q / rho; its interface flux is the Riemann solver's mass flux times
// the interface value of s on the side the mass comes from:  F_q = F_rho * (F_rho >= 0 ? s_L : s_R).
inline void scalar_fluxes(int nv, const double WL[NVMAX], const double WR[NVMAX], double F[NVMAX]) {
  for (int v = NV; v < nv; ++v) F[v] = F[0] * (F[0] >= 0.0 ? WL[v] : WR[v]);
}
inline void all_prims(const Mesh& m, const double* U, int i, int j, int k, double w[NVMAX]) {
  double u[NV];
  for (int v = 0; v < NV; ++v) u[v] = U[gidx(v, i, j, k)];
  cons_to_prim(u, m.cfg.gamma, w);
  for (int v = NV; v < m.nv; ++v) w[v] = U[gidx(v, i, j, k)] / u[0];
}

// U_out = U^n - lam * ((dFx + dFy) + dFz) on the interior cells, all nv variables; F = [3][nv][N+1][N][N]
void flux_update(const Mesh& m, const double* Un, double* Uout, const std::vector<double>& F, double lam) {
  const int fs = m.nv * (N + 1) * N * N;
  const double* Fx = F.data(); const double* Fy = Fx + fs; const double* Fz = Fy + fs;
  for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i)
    for (int v = 0; v < m.nv; ++v) {
      const double sum = ((Fx[fidx(v, i + 1, j, k)] - Fx[fidx(v, i, j, k)]) +
                          (Fy[fidx(v, j + 1, i, k)] - Fy[fidx(v, j, i, k)])) +
                         (Fz[fidx(v, k + 1, i, j)] - Fz[fidx(v, k, i, j)]);
      Uout[gidx(v, i, j, k)] = Un[gidx(v, i, j, k)] - lam * sum;
    }
}

// ------------------------------------------------------------------ predictor (a4; reading R8)
void predictor_block(Mesh& m, int b, double dt) {
  const int nv = m.nv, fs = nv * (N + 1) * N * N;
  const double h = h_of(m, m.lev[b]);
  const double* Un = m.U[0] + int64_t(b) * m.blk;
  double* Uh = m.U[1] + int64_t(b) * m.blk;
  std::vector<double> W(m.blk), F(3 * fs);
  for (int k = -1; k <= N; ++k) for (int j = -1; j <= N; ++j) for (int i = -1; i <= N; ++i) {
    // only face-adjacent ghost cells are read below, but converting the whole 10^3 box is harmless
    double w[NVMAX];
    all_prims(m, Un, i, j, k, w);
    for (int v = 0; v < nv; ++v) W[gidx(v, i, j, k)] = w[v];
  }
  for (int d = 0; d < 3; ++d)
    for (int tb = 0; tb < N; ++tb) for (int ta = 0; ta < N; ++ta) for (int f = 0; f <= N; ++f) {
      int i0, j0, k0, i1, j1, k1;
      cell_of(d, f - 1, ta, tb, i0, j0, k0);
      cell_of(d, f, ta, tb, i1, j1, k1);
      double WL[NVMAX], WR[NVMAX], Ff[NVMAX];
      for (int v = 0; v < nv; ++v) { WL[v] = W[gidx(v, i0, j0, k0)]; WR[v] = W[gidx(v, i1, j1, k1)]; }
      riemann_flux(m, WL, WR, d, Ff);
      scalar_fluxes(nv, WL, WR, Ff);
      for (int v = 0; v < nv; ++v) F[d * fs + fidx(v, f, ta, tb)] = Ff[v];
    }
  flux_update(m, Un, Uh, F, 0.5 * dt / h);
}

// ------------------------------------------------------------------ corrector (a6, a7; readings R11-R14)
void corrector_block(Mesh& m, int b, double dt) {
  const int nv = m.nv, fs = nv * (N + 1) * N * N;
  const double h = h_of(m, m.lev[b]);
  const double* Un = m.U[0] + int64_t(b) * m.blk;
  const double* Uh = m.U[1] + int64_t(b) * m.blk;
  double* Unew = m.U[2] + int64_t(b) * m.blk;
  std::vector<double> W(m.blk), F(3 * fs);
  for (int k = -G; k < N + G; ++k) for (int j = -G; j < N + G; ++j) for (int i = -G; i < N + G; ++i) {
    double w[NVMAX];
    all_prims(m, Uh, i, j, k, w);
    for (int v = 0; v < nv; ++v) W[gidx(v, i, j, k)] = w[v];
  }
  for (int d = 0; d < 3; ++d)
    for (int tb = 0; tb < N; ++tb) for (int ta = 0; ta < N; ++ta) for (int f = 0; f <= N; ++f) {
      double WL[NVMAX], WR[NVMAX], Ff[NVMAX];
      for (int v = 0; v < nv; ++v) {
        double w[4];  // cells f-2, f-1, f, f+1 along d
        for (int s = 0; s < 4; ++s) { int i, j, k; cell_of(d, f - 2 + s, ta, tb, i, j, k); w[s] = W[gidx(v, i, j, k)]; }
        const double dl = minmod(w[2] - w[1], w[1] - w[0]);   // slope of the left cell  (f-1)
        const double dr = minmod(w[3] - w[2], w[2] - w[1]);   // slope of the right cell (f)
        WL[v] = w[1] + 0.5 * dl;
        WR[v] = w[2] - 0.5 * dr;
      }
      riemann_flux(m, WL, WR, d, Ff);
      scalar_fluxes(nv, WL, WR, Ff);
      for (int v = 0; v < nv; ++v) F[d * fs + fidx(v, f, ta, tb)] = Ff[v];
    }
  flux_update(m, Un, Unew, F, dt / h);
  // flux bookkeeping at coarse-fine faces (reading R14): fine side accumulates dt*F, the
  // coarse leaf stores its own flux.
  for (int d = 0; d < 3; ++d) for (int side = 0; side < 2; ++side) {
    const int face = 2 * d + side;
    const double* Fd = F.data() + d * fs;
    const int f = side ? N : 0;
    const int rs = m.rslot[int64_t(b) * 6 + face], fsl = m.fslot[int64_t(b) * 6 + face];
    for (int v = 0; v < nv; ++v) for (int tb = 0; tb < N; ++tb) for (int ta = 0; ta < N; ++ta) {
      const double val = Fd[fidx(v, f, ta, tb)];
      if (rs >= 0) m.R[(int64_t(rs) * nv + v) * NF + tb * N + ta] += dt * val;
      if (fsl >= 0) m.FH[(int64_t(fsl) * nv + v) * NF + tb * N + ta] = val;
    }
  }
}

// ------------------------------------------------------------------ restriction (a8; reading R15)
void restrict_level(Mesh& m, int lc, int src_copy, int dst_copy) {   // level lc+1 -> lc
  if (lc + 1 >= m.nlev) return;
  const std::vector<int>& blocks = m.of_level[lc];
#pragma omp parallel for schedule(dynamic, 8)
  for (int64_t t = 0; t < (int64_t)blocks.size(); ++t) {
    const int b = blocks[t];
    if (m.leaf[b]) continue;
    double* dst = m.U[dst_copy] + int64_t(b) * m.blk;
    for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i) {
      const int I = 2 * (m.bx[b] * N + i), J = 2 * (m.by[b] * N + j), K = 2 * (m.bz[b] * N + k);
      for (int v = 0; v < m.nv; ++v) {
        double sum = 0.0;
        for (int c = 0; c < 8; ++c) {   // fixed child-cell order c = cx + 2 cy + 4 cz
          const int fi = I + (c & 1), fj = J + ((c >> 1) & 1), fk = K + ((c >> 2) & 1);
          const int fb = find(m, lc + 1, fi / N, fj / N, fk / N);
          sum += m.U[src_copy][int64_t(fb) * m.blk + gidx(v, fi % N, fj % N, fk % N)];
        }
        dst[gidx(v, i, j, k)] = 0.125 * sum;
      }
    }
  }
}

// ------------------------------------------------------------------ reflux (a9)
void reflux_level(Mesh& m, int lc, int copy, double dt_coarse) {
  if (lc + 1 >= m.nlev || !m.reflux_on) return;
  const double h = h_of(m, lc);
  const std::vector<int>& blocks = m.of_level[lc];
  const int nfx = (m.cfg.nb0[0] * N) << (lc + 1), nfy = (m.cfg.nb0[1] * N) << (lc + 1), nfz = (m.cfg.nb0[2] * N) << (lc + 1);
  const int nf[3] = {nfx, nfy, nfz};
#pragma omp parallel for schedule(dynamic, 8)
  for (int64_t t = 0; t < (int64_t)blocks.size(); ++t) {
    const int b = blocks[t];
    double* U = m.U[copy] + int64_t(b) * m.blk;
    for (int face = 0; face < 6; ++face) {   // fixed order x-, x+, y-, y+, z-, z+
      const int fs = m.fslot[int64_t(b) * 6 + face];
      if (fs < 0) continue;
      const int d = face >> 1, side = face & 1;
      const double s = side ? 1.0 : -1.0;
      for (int tb = 0; tb < N; ++tb) for (int ta = 0; ta < N; ++ta) {
        int i, j, k;
        cell_of(d, side ? N - 1 : 0, ta, tb, i, j, k);
        const int gc[3] = {m.bx[b] * N + i, m.by[b] * N + j, m.bz[b] * N + k};
        for (int v = 0; v < m.nv; ++v) {
          double sumR = 0.0;
          for (int q = 0; q < 4; ++q) {   // 2x2 fine faces, first tangential index fastest
            int ff[3];
            int tq = 0;
            for (int dd = 0; dd < 3; ++dd) {
              if (dd == d) ff[dd] = side ? 2 * gc[dd] + 2 : 2 * gc[dd] - 1;   // first fine cell beyond the face
              else { ff[dd] = 2 * gc[dd] + ((q >> tq) & 1); ++tq; }
              if (ff[dd] < 0) ff[dd] += nf[dd];
              if (ff[dd] >= nf[dd]) ff[dd] -= nf[dd];
            }
            const int fb = find(m, lc + 1, ff[0] / N, ff[1] / N, ff[2] / N);
            const int rs = m.rslot[int64_t(fb) * 6 + (2 * d + (1 - side))];
            int fa, fbb;
            if (d == 0) { fa = ff[1] % N; fbb = ff[2] % N; }
            else if (d == 1) { fa = ff[0] % N; fbb = ff[2] % N; }
            else { fa = ff[0] % N; fbb = ff[1] % N; }
            sumR += m.R[(int64_t(rs) * m.nv + v) * NF + fbb * N + fa];
          }
          const double FHv = m.FH[(int64_t(fs) * m.nv + v) * NF + tb * N + ta];
          U[gidx(v, i, j, k)] = U[gidx(v, i, j, k)] - (s / h) * (0.25 * sumR - dt_coarse * FHv);
        }
      }
    }
  }
}

// ------------------------------------------------------------------ CFL (a10; reading R16)
double max_speed_level(const Mesh& m, int l, int copy) {
  const std::vector<int>& blocks = m.of_level[l];
  double smax = 0.0;
#pragma omp parallel for schedule(static) reduction(max : smax)
  for (int64_t t = 0; t < (int64_t)blocks.size(); ++t) {
    const double* U = m.U[copy] + int64_t(blocks[t]) * m.blk;
    for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i) {
      double u[NV], w[NV];
      for (int v = 0; v < NV; ++v) u[v] = U[gidx(v, i, j, k)];
      cons_to_prim(u, m.cfg.gamma, w);
      const double cs = std::sqrt(m.cfg.gamma * w[4] / w[0]);
      const double s = std::max(std::max(std::fabs(w[1]), std::fabs(w[2])), std::fabs(w[3])) + cs;
      if (s > smax) smax = s;
    }
  }
  return smax;
}

double cfl_dt_level(const Mesh& m, int l, int copy) {
  if (m.of_level[l].empty()) return INFINITY;
  return m.cfg.cfl * h_of(m, l) / max_speed_level(m, l, copy);
}

void zero_registers(Mesh& m, int lc) {   // registers of the (lc, lc+1) interface
  for (int b : m.of_level[lc + 1]) for (int f = 0; f < 6; ++f) {
    const int rs = m.rslot[int64_t(b) * 6 + f];
    if (rs >= 0) std::fill_n(&m.R[int64_t(rs) * m.nv * NF], m.nv * NF, 0.0);
  }
  for (int b : m.of_level[lc]) for (int f = 0; f < 6; ++f) {
    const int fs = m.fslot[int64_t(b) * 6 + f];
    if (fs >= 0) std::fill_n(&m.FH[int64_t(fs) * m.nv * NF], m.nv * NF, 0.0);
  }
}

void copy_level(Mesh& m, int l, int src, int dst) {
  for (int b : m.of_level[l]) std::memcpy(m.U[dst] + int64_t(b) * m.blk, m.U[src] + int64_t(b) * m.blk, sizeof(double) * m.blk);
}

void for_blocks(Mesh& m, int l, double dt, void (*fn)(Mesh&, int, double)) {
  const std::vector<int>& blocks = m.of_level[l];
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t t = 0; t < (int64_t)blocks.size(); ++t) fn(m, blocks[t], dt);
}

// eq. (14)-(15), PAPER.md:114-118 (reading R18: N includes 0)
int substep_exponent(double dtH, double dt_cfl_h) {
  int n = 0;
  while (std::ldexp(dtH, -n) > dt_cfl_h && n < 30) ++n;
  return n;
}

// ------------------------------------------------------------------ drivers (a11)
int step_sync(Mesh& m, double dt) {
  for (int l = 0; l + 1 < m.nlev; ++l) zero_registers(m, l);
  for (int l = 0; l < m.nlev; ++l) if (int rc = fill_ghosts_level(m, l, 0, 0, 0.0)) return rc;
  for (int l = 0; l < m.nlev; ++l) for_blocks(m, l, dt, predictor_block);
  for (int l = 0; l < m.nlev; ++l) if (int rc = fill_ghosts_level(m, l, 1, 0, 0.0)) return rc;
  for (int l = 0; l < m.nlev; ++l) for_blocks(m, l, dt, corrector_block);
  for (int l = m.nlev - 2; l >= 0; --l) { restrict_level(m, l, 2, 2); reflux_level(m, l, 2, dt); }
  for (int l = 0; l < m.nlev; ++l) copy_level(m, l, 2, 0);
  return 0;
}

int advance_adaptive(Mesh& m, int l, double dt, double tau, double dt_parent, int64_t* nupd) {
  if (l + 1 < m.nlev) zero_registers(m, l);
  if (int rc = fill_ghosts_level(m, l, 0, 1, tau)) return rc;
  for_blocks(m, l, dt, predictor_block);
  const double tau_half = (l == 0) ? 0.0 : tau + 0.5 * (dt / dt_parent);
  if (int rc = fill_ghosts_level(m, l, 1, 1, tau_half)) return rc;
  for_blocks(m, l, dt, corrector_block);
  if (nupd) nupd[l] += 1;
  if (l + 1 < m.nlev && !m.of_level[l + 1].empty()) {
    const double dtc = cfl_dt_level(m, l + 1, 0);
    const int n = substep_exponent(dt, dtc);
    const double dtf = std::ldexp(dt, -n);
    const int nsub = 1 << n;
    for (int s = 0; s < nsub; ++s)
      if (int rc = advance_adaptive(m, l + 1, dtf, double(s) / double(nsub), dt, nupd)) return rc;
    restrict_level(m, l, 0, 2);
    reflux_level(m, l, 2, dt);
  }
  copy_level(m, l, 2, 0);
  return 0;
}

}  // namespace

// ====================================================================== C interface (ctypes)
extern "C" {

int orc_create_mesh(const Config* cfg, int64_t nblocks, const int32_t* level, const int32_t* ijk, Mesh** out) {
  if (!cfg || !out || cfg->ncell != N || cfg->nghost != G || cfg->nscalar < 0 || cfg->nscalar > NSMAX) return -1;
  Mesh* m = new Mesh;
  m->cfg = *cfg;
  m->nv = NV + cfg->nscalar;
  m->blk = int64_t(m->nv) * M3;
  m->nb = nblocks;
  m->nlev = cfg->max_level + 1;
  m->lev.resize(nblocks); m->bx.resize(nblocks); m->by.resize(nblocks); m->bz.resize(nblocks);
  m->of_level.resize(m->nlev);
  for (int64_t b = 0; b < nblocks; ++b) {
    m->lev[b] = level[b]; m->bx[b] = ijk[3 * b]; m->by[b] = ijk[3 * b + 1]; m->bz[b] = ijk[3 * b + 2];
    if (level[b] < 0 || level[b] >= m->nlev) { delete m; return -2; }
    if (!m->map.emplace(key(level[b], m->bx[b], m->by[b], m->bz[b]), int(b)).second) { delete m; return -2; }
    m->of_level[level[b]].push_back(int(b));
  }
  m->leaf.assign(nblocks, 1);
  for (int64_t b = 0; b < nblocks; ++b)
    if (m->lev[b] + 1 < m->nlev && find(*m, m->lev[b] + 1, 2 * m->bx[b], 2 * m->by[b], 2 * m->bz[b]) >= 0) m->leaf[b] = 0;
  // flag faces.  Fine side: a face whose same-level neighbour is absent inside the domain
  // (periodic wrap applied).  Coarse side: a leaf whose neighbour across the face is not a leaf.
  m->rslot.assign(nblocks * 6, -1); m->fslot.assign(nblocks * 6, -1);
  int nr = 0, nf = 0;
  for (int64_t b = 0; b < nblocks; ++b) for (int face = 0; face < 6; ++face) {
    const int d = face >> 1, side = face & 1, l = m->lev[b];
    int c[3] = {m->bx[b], m->by[b], m->bz[b]};
    c[d] += side ? 1 : -1;
    const int n = m->cfg.nb0[d] << l;
    if (c[d] < 0) { if (m->cfg.bc[d][0] != 0) continue; c[d] += n; }
    if (c[d] >= n) { if (m->cfg.bc[d][1] != 0) continue; c[d] -= n; }
    const int nbk = find(*m, l, c[0], c[1], c[2]);
    if (nbk < 0) { if (l > 0) m->rslot[b * 6 + face] = nr++; }
    else if (m->leaf[b] && !m->leaf[nbk]) m->fslot[b * 6 + face] = nf++;
  }
  m->R.assign(int64_t(nr) * m->nv * NF, 0.0);
  m->FH.assign(int64_t(nf) * m->nv * NF, 0.0);
  *out = m;
  return 0;
}

void orc_destroy_mesh(Mesh* m) { delete m; }
const char* orc_last_error(Mesh* m) { return m->err; }
int64_t orc_state_doubles(const Mesh* m) { return m->nb * m->blk; }

int orc_bind(Mesh* m, double* U0, double* U1, double* U2) { m->U[0] = U0; m->U[1] = U1; m->U[2] = U2; return 0; }
void orc_set_reflux(Mesh* m, int on) { m->reflux_on = on; }
int orc_set_riemann(Mesh* m, int solver) { if (solver != 0 && solver != 1) return -1; m->riemann = solver; return 0; }
int orc_is_leaf(const Mesh* m, int64_t b) { return m->leaf[b]; }
double orc_cell_width(const Mesh* m, int l) { return h_of(*m, l); }
int64_t orc_num_registers(const Mesh* m, int which) {
  int64_t n = 0;
  for (int v : (which ? m->fslot : m->rslot)) n += (v >= 0);
  return n;
}

int orc_fill_ghosts(Mesh* m, int level, int which, int interp, double tau) {
  for (int l = 0; l < m->nlev; ++l)
    if (level < 0 || level == l) if (int rc = fill_ghosts_level(*m, l, which, interp, tau)) return rc;
  return 0;
}
int orc_predictor(Mesh* m, int level, double dt) {
  for (int l = 0; l < m->nlev; ++l) if (level < 0 || level == l) for_blocks(*m, l, dt, predictor_block);
  return 0;
}
int orc_corrector(Mesh* m, int level, double dt) {
  for (int l = 0; l < m->nlev; ++l) if (level < 0 || level == l) for_blocks(*m, l, dt, corrector_block);
  return 0;
}
int orc_zero_registers(Mesh* m, int coarse_level) {
  for (int l = 0; l + 1 < m->nlev; ++l) if (coarse_level < 0 || coarse_level == l) zero_registers(*m, l);
  return 0;
}
int orc_restrict(Mesh* m, int coarse_level, int src_copy, int dst_copy) { restrict_level(*m, coarse_level, src_copy, dst_copy); return 0; }
int orc_reflux(Mesh* m, int coarse_level, int copy, double dt_coarse) { reflux_level(*m, coarse_level, copy, dt_coarse); return 0; }
int orc_copy_level(Mesh* m, int level, int src, int dst) {
  for (int l = 0; l < m->nlev; ++l) if (level < 0 || level == l) copy_level(*m, l, src, dst);
  return 0;
}
double orc_cfl_dt(Mesh* m, int level, int copy) {
  double dt = INFINITY;
  for (int l = 0; l < m->nlev; ++l) if (level < 0 || level == l) dt = std::min(dt, cfl_dt_level(*m, l, copy));
  return dt;
}
double orc_max_speed(Mesh* m, int level, int copy) { return max_speed_level(*m, level, copy); }
int orc_substep_exponent(double dtH, double dt_cfl_h) { return substep_exponent(dtH, dt_cfl_h); }
double orc_time_interp(double U0, double Uh, double U1, double tau) { return time_interp(U0, Uh, U1, tau); }
void orc_hllc(const double* WL, const double* WR, int d, double gamma, double* F) { hllc(WL, WR, d, gamma, F); }
void orc_roe(const double* WL, const double* WR, int d, double gamma, double* F) { roe(WL, WR, d, gamma, F); }
double orc_minmod(double a, double b) { return minmod(a, b); }
int orc_get(Mesh* m, int level, int I, int J, int K, int which, double* out) {   // sync-mode accessor
  std::vector<Src> srcs(m->nlev, Src{0, which, 0.0});
  double val[NVMAX];
  if (!get(*m, level, I, J, K, srcs.data(), val)) return -2;
  for (int v = 0; v < m->nv; ++v) out[v] = val[v];      // out: nv = 5 + nscalar doubles
  return 0;
}

// mode 0: synchronous, dt_fixed>0 overrides the CFL step; mode 1: adaptive
// (PAPER.md:108-120).  t accumulates elapsed time; nupd[level] counts level updates.
int orc_advance(Mesh* m, int nsteps, int mode, double dt_fixed, double* t, int64_t* nupd) {
  for (int s = 0; s < nsteps; ++s) {
    if (mode == 0) {
      double dt = dt_fixed;
      if (!(dt > 0.0)) { dt = INFINITY; for (int l = 0; l < m->nlev; ++l) dt = std::min(dt, cfl_dt_level(*m, l, 0)); }
      if (int rc = step_sync(*m, dt)) return rc;
      if (nupd) for (int l = 0; l < m->nlev; ++l) nupd[l] += 1;
      if (t) *t += dt;
    } else {
      const double dt = dt_fixed > 0.0 ? dt_fixed : cfl_dt_level(*m, 0, 0);
      if (int rc = advance_adaptive(*m, 0, dt, 0.0, dt, nupd)) return rc;
      if (t) *t += dt;
    }
  }
  return 0;
}

int64_t orc_status(Mesh* m, int copy) {   // cells with rho<=0 or P<=0 (or NaN), interior, all blocks
  int64_t bad = 0;
  for (int64_t b = 0; b < m->nb; ++b) {
    const double* U = m->U[copy] + b * m->blk;
    for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i) {
      double u[NV], w[NV];
      for (int v = 0; v < NV; ++v) u[v] = U[gidx(v, i, j, k)];
      cons_to_prim(u, m->cfg.gamma, w);
      if (!(w[0] > 0.0) || !(w[4] > 0.0)) ++bad;
    }
  }
  return bad;
}

// ------------------------------------------------------------------ refinement indicators
// criterion 0, eq. (33)-(34) PAPER.md:277-285: per block, max over interior cells of max(E(rho), E(P)),
//   E(q) = |d2x q + d2y q + d2z q| h^2 / q  with centred second differences (the h^2 cancels);
//   a block is refined where this is >= 1e-2 (the comparison is the caller's).
// criterion 1, "the Jeans length is resolved by at least 8 cells": per block, max over
//   interior cells of h / lambda_J, lambda_J = c_s sqrt(pi / (G rho)), c_s^2 = gamma P / rho (reading R31);
//   a block is refined where this is > 1/8.
// Reads the ghost cells (one layer, faces) of copy `which`: call orc_fill_ghosts first.
int orc_refine_indicator(Mesh* m, int which, int criterion, double G, double* out) {
  if (which < 0 || which > 2 || (criterion != 0 && criterion != 1)) return -1;
  const double gamma = m->cfg.gamma;
  const double pi = 3.14159265358979323846;
  for (int64_t b = 0; b < m->nb; ++b) {
    const double* U = m->U[which] + b * m->blk;
    const double h = h_of(*m, m->lev[b]);
    auto prim = [&](int i, int j, int k, double& rho, double& P) {
      double u[NV], w[NV];
      for (int v = 0; v < NV; ++v) u[v] = U[gidx(v, i, j, k)];
      cons_to_prim(u, gamma, w);
      rho = w[0]; P = w[4];
    };
    double best = 0.0;
    for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i) {
      double r0, P0;
      prim(i, j, k, r0, P0);
      double val;
      if (criterion == 0) {
        double lr = 0.0, lP = 0.0;
        for (int d = 0; d < 3; ++d) {
          double rp, Pp, rm, Pm;
          prim(i + (d == 0), j + (d == 1), k + (d == 2), rp, Pp);
          prim(i - (d == 0), j - (d == 1), k - (d == 2), rm, Pm);
          lr += (rp - 2.0 * r0) + rm;
          lP += (Pp - 2.0 * P0) + Pm;
        }
        val = std::max(std::fabs(lr) / r0, std::fabs(lP) / P0);
      } else {
        const double cs = std::sqrt(gamma * P0 / r0);
        val = h / (cs * std::sqrt(pi / (G * r0)));
      }
      if (val > best) best = val;
    }
    out[b] = best;
  }
  return 0;
}

// ------------------------------------------------------------------ regrid: state transfer
// The state of a NEW mesh from an OLD one after a regrid ("blocks are refined ... subdivided into
// eight child blocks"): every interior cell of every block of `dst` is the value of that cell in the old
// hierarchy, get(src, level, I, J, K): a copy where the block existed, the slope-limited conservative
// prolongation of reading R3 from the old coarser level(s) where it is new.  Blocks that disappear are
// dropped: their parents exist in both meshes and already hold the restricted data.
int orc_transfer_state(const Mesh* src, int src_which, Mesh* dst, int dst_which) {
  if (src_which < 0 || src_which > 2 || dst_which < 0 || dst_which > 2) return -1;
  for (int d = 0; d < 3; ++d)
    if (src->cfg.nb0[d] != dst->cfg.nb0[d] || src->cfg.bc[d][0] != dst->cfg.bc[d][0] ||
        src->cfg.bc[d][1] != dst->cfg.bc[d][1]) return -1;
  if (src->nv != dst->nv) return -1;
  std::vector<Src> srcs(std::max(src->nlev, dst->nlev), Src{0, src_which, 0.0});
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 8) reduction(+ : bad)
  for (int64_t b = 0; b < dst->nb; ++b) {
    const int l = dst->lev[b];
    double* out = dst->U[dst_which] + b * dst->blk;
    double val[NVMAX];
    for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i) {
      if (!get(*src, l, dst->bx[b] * N + i, dst->by[b] * N + j, dst->bz[b] * N + k, srcs.data(), val)) { bad++; continue; }
      for (int v = 0; v < dst->nv; ++v) out[gidx(v, i, j, k)] = val[v];
    }
  }
  if (bad) { snprintf(dst->err, sizeof dst->err, "transfer_state: %d cells could not be resolved", bad); return -2; }
  return 0;
}

// ------------------------------------------------------------------ regrid: the new block list
// PAPER.md:96 ("a block is refined ... subdivided into eight child blocks"), :277-285 (eq. 33-34), :641 (Jeans), :100
// (lists built on the host).  The new tree, from the indicator of copy `which` (ghosts filled here):
//   * every root block;
//   * the 8 children of every block B of level < max_level that is in the OLD mesh, is in the NEW tree, and is
//     flagged: its indicator is >= threshold (eq. 33 is written with >=) or one of its descendants in the old mesh is
//     flagged -- so a regrid deepens the tree by at most one level anywhere, drops the children of blocks that are
//     no longer flagged, and keeps the refinement above every flagged block;
//   * closed under proper nesting (reading R25): every one of the 26 neighbour positions of a level-l block that lies
//     inside the domain (periodic wrap applied; positions beyond an outflow face are skipped) is covered at level
//     l-1; missing blocks are created with their 7 siblings and, recursively, their ancestors.
// The new mesh lists its blocks level by level, (bx, by, bz) lexicographic within a level, and carries the same
// configuration.  The state is then moved with orc_transfer_state.
int orc_regrid(Mesh* m, int which, int criterion, double Gc, double threshold, Mesh** out) {
  if (!out) return -1;
  *out = nullptr;
  for (int l = 0; l < m->nlev; ++l) if (int rc = fill_ghosts_level(*m, l, which, 0, 0.0)) return rc;
  std::vector<double> ind(m->nb);
  if (int rc = orc_refine_indicator(m, which, criterion, Gc, ind.data())) return rc;
  typedef std::array<int, 3> C3;
  std::vector<std::set<C3>> tree(m->nlev);
  for (int64_t b = 0; b < m->nb; ++b) if (m->lev[b] == 0) tree[0].insert(C3{m->bx[b], m->by[b], m->bz[b]});
  // a block counts as flagged when its own indicator is >= threshold or when any of its descendants in the OLD mesh
  // is flagged (reading R33: a feature smaller than a coarse cell is invisible in the restricted data of the coarse
  // block above it, and must not lose its refinement for that)
  std::vector<char> flag(m->nb);
  for (int64_t b = 0; b < m->nb; ++b) flag[b] = ind[b] >= threshold;
  for (int l = m->nlev - 1; l >= 1; --l)
    for (int b : m->of_level[l])
      if (flag[b]) flag[find(*m, l - 1, m->bx[b] >> 1, m->by[b] >> 1, m->bz[b] >> 1)] = 1;
  for (int l = 0; l + 1 < m->nlev; ++l)
    for (int b : m->of_level[l]) {
      const C3 c{m->bx[b], m->by[b], m->bz[b]};
      if (!tree[l].count(c) || !flag[b]) continue;
      for (int q = 0; q < 8; ++q) tree[l + 1].insert(C3{2 * c[0] + (q & 1), 2 * c[1] + ((q >> 1) & 1), 2 * c[2] + ((q >> 2) & 1)});
    }
  // make the octet that holds block c of level l exist (and its ancestors)
  std::function<void(int, C3)> ensure = [&](int l, C3 c) {
    if (l == 0 || tree[l].count(c)) return;
    const C3 par{c[0] >> 1, c[1] >> 1, c[2] >> 1};
    ensure(l - 1, par);
    for (int q = 0; q < 8; ++q) tree[l].insert(C3{2 * par[0] + (q & 1), 2 * par[1] + ((q >> 1) & 1), 2 * par[2] + ((q >> 2) & 1)});
  };
  bool changed = true;
  while (changed) {
    changed = false;
    for (int l = m->nlev - 1; l >= 2; --l) {
      const std::vector<C3> blocks(tree[l].begin(), tree[l].end());
      for (const C3& x : blocks)
        for (int dz = -1; dz <= 1; ++dz) for (int dy = -1; dy <= 1; ++dy) for (int dx = -1; dx <= 1; ++dx) {
          int pos[3] = {x[0] + dx, x[1] + dy, x[2] + dz};
          bool outside = false;
          for (int d = 0; d < 3; ++d) {
            const int n = m->cfg.nb0[d] << l;
            if (pos[d] < 0) { if (m->cfg.bc[d][0] != 0) outside = true; else pos[d] += n; }
            else if (pos[d] >= n) { if (m->cfg.bc[d][1] != 0) outside = true; else pos[d] -= n; }
          }
          if (outside) continue;
          const C3 c{pos[0] >> 1, pos[1] >> 1, pos[2] >> 1};
          if (!tree[l - 1].count(c)) { ensure(l - 1, c); changed = true; }
        }
    }
  }
  std::vector<int32_t> level, ijk;
  for (int l = 0; l < m->nlev; ++l)
    for (const C3& c : tree[l]) { level.push_back(l); ijk.push_back(c[0]); ijk.push_back(c[1]); ijk.push_back(c[2]); }
  return orc_create_mesh(&m->cfg, int64_t(level.size()), level.data(), ijk.data(), out);
}

int64_t orc_num_blocks(const Mesh* m) { return m->nb; }
void orc_block_list(const Mesh* m, int32_t* level, int32_t* ijk) {
  for (int64_t b = 0; b < m->nb; ++b) {
    level[b] = m->lev[b];
    ijk[3 * b] = m->bx[b]; ijk[3 * b + 1] = m->by[b]; ijk[3 * b + 2] = m->bz[b];
  }
}

}  // extern "C"

// sfh_stage.cuh — the stage kernels of libsfh for sm_100a (B200): predictor (a4) and corrector
// (a6 + a7 of SURVEY.md section 8(a)).
//
// One persistent CTA of 512 threads per SM, warps specialised:
//   * 12 WALKER warps never leave the flux loop.  Walker thread (D, half, pencil) owns half of one of
//     the 64 pencils of axis D of the current 8^3 block: it computes the 5 face fluxes of its 4 cells,
//     each once, and stores the 4 flux differences to shared memory.  (The pencil walk with flux reuse
//     is the paper's mapping, Fig. 1; halving the pencils doubles the independent fp64
//     streams per block at the price of one duplicated face out of nine.)
//   * 4 HELPER warps run the rest of the pipeline around the walkers: their first lanes stage the block
//     after next with TMA (the ghost "fill" of same-level faces is this gather out of the neighbours'
//     interiors), all of them convert a staged block to primitives in place (predictor), fill the halo
//     of outflow faces, and turn the finished flux differences of the previous block into the updated
//     state (coalesced global loads/stores of U^n and the result).
// Staging is double buffered; the stages hand over through mbarriers only (no CTA-wide barrier), so
// the fp64 pipe sees walkers all the time while staging, conversion and update of the neighbouring
// blocks of the pipeline overlap them.
//
// Staged block ("landing" layout, both kernels): 10 tiles of [var][128 cells], variable stride 128:
//   tiles 0..5  the z column: z-plane pairs k = (-2,-1), (0,1), ..., (6,7), (8,9), 128-byte swizzled by
//               TMA (zs_pos): the low z halo, the interior, the high z halo;
//   tile 6, 7   the x-low / x-high halo  [k][j][ll]   (ll = layer, index increasing with x)
//   tile 8, 9   the y-low / y-high halo  [ll][k][i]
// Every pencil read of a half-warp is bank-conflict free in this layout (x pencils read cell PAIRS with
// 128-bit loads).  The predictor's tiles carry two more variables (P, c_s) written by the conversion; the total
// energy stays where it landed.
#pragma once

#include <cmath>

#include "sfh_device.cuh"
#include "sfh_kernels.cuh"

namespace sfh {

constexpr int WALK_WARPS = 12, HELP_WARPS = 4;
constexpr int WALK_THREADS = 32 * WALK_WARPS, HELP_THREADS = 32 * HELP_WARPS;
constexpr int STAGE_THREADS = WALK_THREADS + HELP_THREADS;   // 512 threads of 128 registers: the register file of one SM
constexpr int CVS = NG * FACE;                // variable stride of every tile (128 cells)
constexpr int NTILE = 10;
constexpr int T_XLO = 6, T_XHI = 7, T_YLO = 8, T_YHI = 9;
constexpr int DF_DOUBLES = 3 * BLK;           // flux differences of one block: [axis][5][512]
constexpr int HC = NC / HELP_THREADS;         // cells per helper thread in the update (4)

template <int STAGE>
struct Cfg {
  static constexpr int NVW = STAGE == 0 ? 7 : 5;      // staged variables per cell
  static constexpr int TS = NVW * CVS;                // tile stride (doubles): 896 / 640, a multiple of 1 KB
  static constexpr int LAND = NTILE * TS;             // one staged block
  static constexpr int NDF = STAGE == 0 ? 1 : 2;      // flux-difference buffers that fit beside the staging
  static constexpr int SMEM = (2 * LAND + NDF * DF_DOUBLES) * 8 + 384 + 1024;   // + barriers, + alignment slack
};
static_assert(Cfg<0>::SMEM <= 232448 && Cfg<1>::SMEM <= 232448, "shared memory of one SM");
static_assert((Cfg<0>::TS * 8) % 1024 == 0 && (Cfg<1>::TS * 8) % 1024 == 0, "swizzled tiles start on 1 KB");

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// ---- positions in the landing layout -----------------------------------------------------------------
template <int TS>
__device__ __forceinline__ int pos_zcol(int i, int j, int k) { return ((k + 2) >> 1) * TS + zs_pos(k & 1, j, i); }

// position of cell c in [-2, 10) of pencil (a, b) along axis D
template <int TS, int D>
__device__ __forceinline__ int cell_pos(int c, int a, int b) {
  if (D == 2) return pos_zcol<TS>(a, b, c);
  if (D == 0) {   // a = j, b = k
    const int in = pos_zcol<TS>(c, a, b);
    const int lo = T_XLO * TS + (b * 8 + a) * 2 + (c + 2);
    const int hi = T_XHI * TS + (b * 8 + a) * 2 + (c - N);
    return c < 0 ? lo : c >= N ? hi : in;
  }
  const int in = pos_zcol<TS>(a, c, b);   // a = i, b = k
  const int lo = T_YLO * TS + (c + 2) * 64 + b * 8 + a;
  const int hi = T_YHI * TS + (c - N) * 64 + b * 8 + a;
  return c < 0 ? lo : c >= N ? hi : in;
}

// one cell in the face frame of axis D: corrector (rho, normal v, tangential v's, P), predictor (rho, normal v,
// tangential v's, E, P, c_s)
template <int NVW, int D>
__device__ __forceinline__ void load_cell(const double* __restrict__ Wl, int o, double w[NVW]) {
  constexpr int vn = 1 + D, vt1 = 1 + (D + 1) % 3, vt2 = 1 + (D + 2) % 3;
  w[0] = Wl[o]; w[1] = Wl[o + vn * CVS]; w[2] = Wl[o + vt1 * CVS]; w[3] = Wl[o + vt2 * CVS]; w[4] = Wl[o + 4 * CVS];
  if (NVW == 7) { w[5] = Wl[o + 5 * CVS]; w[6] = Wl[o + 6 * CVS]; }
}
// cells c and c + 1 of the pencil, c even.  x pencils read the pair with one 128-bit load per variable.
template <int STAGE, int D>
__device__ __forceinline__ void load_two(const double* __restrict__ Wl, int c, int a, int b, double w0[], double w1[]) {
  constexpr int NVW = Cfg<STAGE>::NVW, TS = Cfg<STAGE>::TS;
  if (D == 0) {
    const int o = cell_pos<TS, 0>(c, a, b);
#pragma unroll
    for (int v = 0; v < NVW; ++v) {
      const double2 t = *reinterpret_cast<const double2*>(Wl + o + v * CVS);
      w0[v] = t.x; w1[v] = t.y;
    }
  } else {
    load_cell<NVW, D>(Wl, cell_pos<TS, D>(c, a, b), w0);
    load_cell<NVW, D>(Wl, cell_pos<TS, D>(c + 1, a, b), w1);
  }
}

// dF of cell c of the pencil = F(face c+1) - F(face c), in the FACE frame (the update un-permutes).
// Layouts (bank-conflict free for the walkers' stores and for the update's loads):
//   x: row (k, j) of 8, i XOR-swizzled with (j >> 1) | (k & 1) << 2;  y: [k][(j, i) ^ (k & 1) << 3];  z: [k][j][i]
__device__ __forceinline__ int dfx_idx(int i, int j, int k) { return (k * 8 + j) * 8 + (i ^ ((j >> 1) | ((k & 1) << 2))); }
__device__ __forceinline__ int dfy_idx(int i, int j, int k) { return BLK + k * 64 + ((j * 8 + i) ^ ((k & 1) << 3)); }
__device__ __forceinline__ int dfz_idx(int i, int j, int k) { return 2 * BLK + (k * 8 + j) * 8 + i; }
template <int D>
__device__ __forceinline__ void store_df(double* __restrict__ dF, int c, int a, int b, const double Fa[5],
                                         const double Fb[5]) {
  const int ci = D == 0 ? dfx_idx(c, a, b) : D == 1 ? dfy_idx(a, c, b) : dfz_idx(a, b, c);
#pragma unroll
  for (int q = 0; q < 5; ++q) dF[ci + q * NC] = Fa[q] - Fb[q];
}

// flux registers at coarse-fine faces (a7; reading R14); Fn in the face frame.  src / fs: the face's
// halo source and its coarse-side register slot (loaded at the start of the walk, so the walker never waits for
// them).  Every register entry has one contributor per launch: the accumulation is a fire-and-forget reduction
// (RED.ADD.F64) with the same result as a read-modify-write.
__device__ __forceinline__ void store_regs(int src, int fs, double* R, double* FH, int D, int t, const double Fn[5],
                                           double dt) {
  const int vn = 1 + D, vt1 = 1 + (D + 1) % 3, vt2 = 1 + (D + 2) % 3;
  if (src <= -2) {   // fine side of a coarse-fine face: accumulate dt * F
    double* r = R + size_t(-2 - src) * REG + t;
    atomicAdd(r, dt * Fn[0]); atomicAdd(r + vn * FACE, dt * Fn[1]); atomicAdd(r + vt1 * FACE, dt * Fn[2]);
    atomicAdd(r + vt2 * FACE, dt * Fn[3]); atomicAdd(r + 4 * FACE, dt * Fn[4]);
  }
  if (fs >= 0) {     // coarse leaf next to a covered block: keep its own flux
    double* r = FH + size_t(fs) * REG + t;
    r[0] = Fn[0]; r[vn * FACE] = Fn[1]; r[vt1 * FACE] = Fn[2]; r[vt2 * FACE] = Fn[3]; r[4 * FACE] = Fn[4];
  }
}

// ---- the walks ---------------------------------------------------------------------------------------
// A half pencil: faces f0 .. f0+4 and cells f0 .. f0+3, f0 = 0 or 4.  Face f lies between cells f-1 and f.
// The loops are unrolled by two so that the carried cell/face state ping-pongs between registers.

// flux of the cell-centred states w0 | w1 = (rho, u, v, w, E, P, c_s or 1/sqrt(rho)) with Riemann solver RS (0 HLLC, 1 Roe)
template <int RS>
__device__ __forceinline__ void cell_flux(const double w0[7], const double w1[7], double gm1, double igm1, double F[5]) {
  if (RS == 0)
    hllc_flux<true>(w0[0], w0[1], w0[2], w0[3], w0[5], w0[6], w0[4], w1[0], w1[1], w1[2], w1[3], w1[5], w1[6], w1[4], igm1, F);
  else
    roe_flux<true>(w0[0], w0[1], w0[2], w0[3], w0[5], w0[4], w0[6], w1[0], w1[1], w1[2], w1[3], w1[5], w1[4], w1[6], gm1,
                   igm1, F);
}

// predictor: first-order fluxes of the cell-centred states (reading R8)
// mf (MFX): mass flux of face f of this pencil goes to mf[f * 64]
template <int RS, int D, bool MFX>
__device__ __forceinline__ void walk_predictor(const double* __restrict__ Wl, double* __restrict__ dF, int a, int b,
                                               int f0, double gm1, double igm1, uint32_t bar_empty,
                                               uint32_t par_empty, bool wait_empty, double* __restrict__ mf) {
  constexpr int TS = Cfg<0>::TS;
  double w0[7], w1[7], wn[7], F0[5], F1[5];
  if (D == 0) {
    load_two<0, 0>(Wl, f0 - 2, a, b, wn, w0);       // cell f0-1
    load_two<0, 0>(Wl, f0, a, b, w1, wn);           // cells f0, f0+1
  } else {
    load_cell<7, D>(Wl, cell_pos<TS, D>(f0 - 1, a, b), w0);
    load_cell<7, D>(Wl, cell_pos<TS, D>(f0, a, b), w1);
  }
  cell_flux<RS>(w0, w1, gm1, igm1, F0);             // face f0
  if (MFX) mf[f0 * 64] = F0[0];
  if (wait_empty) mbar_wait(bar_empty, par_empty);  // the update of the block before has read dF
#pragma unroll
  for (int f = f0 + 1; f < f0 + 4; f += 2) {        // faces f (cells f-1 | f) and f+1 (cells f | f+1)
    if (D == 0) {
#pragma unroll
      for (int v = 0; v < 7; ++v) w0[v] = wn[v];
    } else {
      load_cell<7, D>(Wl, cell_pos<TS, D>(f, a, b), w0);
    }
    cell_flux<RS>(w1, w0, gm1, igm1, F1);
    if (MFX) mf[f * 64] = F1[0];
    store_df<D>(dF, f - 1, a, b, F1, F0);
    if (D == 0) load_two<0, 0>(Wl, f + 1, a, b, w1, wn);
    else load_cell<7, D>(Wl, cell_pos<TS, D>(f + 1, a, b), w1);
    cell_flux<RS>(w0, w1, gm1, igm1, F0);
    if (MFX) mf[(f + 1) * 64] = F0[0];
    store_df<D>(dF, f, a, b, F0, F1);
  }
}

// corrector: minmod-limited linear reconstruction of the primitives (readings R11, R12) + HLLC.
// Slope of the cell with value wc from its two one-sided differences; returns the right state of the
// cell's lower face in R and the left state of its upper face in Lnext:  W -/+ minmod/2
__device__ __forceinline__ void limited_states(const double wc[5], const double dn[5], const double dm[5], double R[5],
                                               double Lnext[5]) {
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    // minmod(dn, dm)/2 = k m with m the difference of smaller magnitude, k = 1/2 if the signs agree
    const double m = fabs(dn[v]) < fabs(dm[v]) ? dn[v] : dm[v];
    const bool same = (__double2hiint(dn[v]) ^ __double2hiint(dm[v])) >= 0;
    const double k = __hiloint2double(same ? 0x3fe00000 : 0, 0);
    R[v] = fma(-k, m, wc[v]);
    Lnext[v] = fma(k, m, wc[v]);
  }
}
template <int RS>
__device__ __forceinline__ void corrector_flux(const double WLs[5], const double WRs[5], double gamma, double igm1,
                                               double Fn[5]) {
  if (RS == 0) {
    const double cL = sound_speed(gamma, WLs[4], WLs[0]);
    const double cR = sound_speed(gamma, WRs[4], WRs[0]);
    hllc_flux<false>(WLs[0], WLs[1], WLs[2], WLs[3], WLs[4], cL, 0.0, WRs[0], WRs[1], WRs[2], WRs[3], WRs[4], cR, 0.0,
                     igm1, Fn);
  } else {
    roe_flux<false>(WLs[0], WLs[1], WLs[2], WLs[3], WLs[4], 0.0, 0.0, WRs[0], WRs[1], WRs[2], WRs[3], WRs[4], 0.0, 0.0,
                    gamma - 1.0, igm1, Fn);
  }
}

// ---- direction-generic corrector walk ------------------------------------------------------------------
// The corrector walk with every direction-dependent quantity (the positions of the thread's 8 cells in the
// landing layout, the variable offsets of the face frame, the positions of its 4 flux differences) held
// in registers, so that the twelve walker warps run ONE straight-line body: a third of the instruction
// footprint of three direction instantiations, and no loop-carried register rotation.
struct WalkGeom {
  int cp[12];    // cells -2 .. 9 of the pencil (a half pencil reads -2 .. 4 or 2 .. 9)
  int ov[3];     // offsets of the normal and the two tangential velocities
  int di[8];     // flux-difference positions of cells 0 .. 7
};
template <int STAGE, int D>
__device__ __forceinline__ void walk_geom(int a, int b, WalkGeom& g) {
  constexpr int TS = Cfg<STAGE>::TS;
#pragma unroll
  for (int cc = 0; cc < 12; ++cc) g.cp[cc] = cell_pos<TS, D>(cc - 2, a, b);
  g.ov[0] = (1 + D) * CVS; g.ov[1] = (1 + (D + 1) % 3) * CVS; g.ov[2] = (1 + (D + 2) % 3) * CVS;
#pragma unroll
  for (int cc = 0; cc < 8; ++cc) g.di[cc] = D == 0 ? dfx_idx(cc, a, b) : D == 1 ? dfy_idx(a, cc, b) : dfz_idx(a, b, cc);
}
__device__ __forceinline__ void load_cell_g(const double* __restrict__ Wl, int o, const int ov[3], double w[5]) {
  w[0] = Wl[o]; w[1] = Wl[o + ov[0]]; w[2] = Wl[o + ov[1]]; w[3] = Wl[o + ov[2]]; w[4] = Wl[o + 4 * CVS];
}
// REGS: the level has flux-register faces
template <int RS, bool REGS, bool MFX>
__device__ __forceinline__ void walk_corrector_generic(const double* __restrict__ Wl, double* __restrict__ dF,
                                                       const WalkGeom& g, int D, int a, int b, double gamma,
                                                       double igm1, const StageParams& p, int blk, double dt,
                                                       uint32_t bar_empty, uint32_t par_empty, bool wait_empty,
                                                       double* __restrict__ mf, bool upper, uint32_t bar_pair,
                                                       uint32_t par_pair) {
  double wp[5], wc[5], wn[5], dp[5], dn[5], L[5], Ln[5], R[5], Fa[5], Fb[5];
  const int f0 = upper ? 4 : 0;                               // faces f0 .. f0+4 (upper) or f0 .. f0+3 (lower)
  int cp[8], di[4];                                           // cells f0-2 .. f0+5, flux-difference slots of cells f0 .. f0+3
#pragma unroll
  for (int cc = 0; cc < 8; ++cc) cp[cc] = upper ? g.cp[cc + 4] : g.cp[cc];
#pragma unroll
  for (int cc = 0; cc < 4; ++cc) di[cc] = upper ? g.di[cc + 4] : g.di[cc];
  const int ds = g.di[3];                                     // cell 3's slot: face 4 goes through it to the lower half
  int rsrc = 0, rfs = -1;                                     // my boundary face: halo source, coarse-side register
  if (REGS) {
    const int f = blk * 6 + 2 * D + (f0 != 0);
    rsrc = p.face_src[f];
    rfs = p.fslot[f];
  }
  load_cell_g(Wl, cp[0], g.ov, wp);
  load_cell_g(Wl, cp[1], g.ov, wc);
  load_cell_g(Wl, cp[2], g.ov, wn);
#pragma unroll
  for (int v = 0; v < 5; ++v) { dp[v] = wc[v] - wp[v]; dn[v] = wn[v] - wc[v]; }
  limited_states(wc, dn, dp, R, L);                           // L = left state of face f0
#pragma unroll
  for (int ff = 0; ff < 5; ++ff) {                            // face f0+ff, between cells cc = ff+1 and ff+2
    if (ff == 4 && !upper) break;                             // face 4 comes from the upper half pencil (warp-uniform)
#pragma unroll
    for (int v = 0; v < 5; ++v) { wc[v] = wn[v]; dp[v] = dn[v]; }
    load_cell_g(Wl, cp[ff + 3], g.ov, wn);
#pragma unroll
    for (int v = 0; v < 5; ++v) dn[v] = wn[v] - wc[v];
    limited_states(wc, dn, dp, R, Ln);                        // right state of this face, left state of the next
    corrector_flux<RS>(L, R, gamma, igm1, (ff & 1) ? Fb : Fa);
    if (MFX) mf[(f0 + ff) * 64] = (ff & 1) ? Fb[0] : Fa[0];
#pragma unroll
    for (int v = 0; v < 5; ++v) L[v] = Ln[v];
    if (ff == 0) {
      if (REGS && f0 == 0 && (rsrc <= -2 || rfs >= 0)) store_regs(rsrc, rfs, p.R, p.FH, D, b * 8 + a, Fa, dt);
      if (wait_empty) mbar_wait(bar_empty, par_empty);        // the update two blocks back has read this dF buffer
      if (upper) {                                            // face 4: hand the flux to the lower half through cell 3's slot
#pragma unroll
        for (int q = 0; q < 5; ++q) dF[ds + q * NC] = Fa[q];
        __syncwarp();
        if ((threadIdx.x & 31) == 0) mbar_arrive(bar_pair);
      }
    } else {
#pragma unroll
      for (int q = 0; q < 5; ++q) dF[di[ff - 1] + q * NC] = (ff & 1) ? Fb[q] - Fa[q] : Fa[q] - Fb[q];
    }
  }
  if (REGS && f0 != 0 && (rsrc <= -2 || rfs >= 0)) store_regs(rsrc, rfs, p.R, p.FH, D, b * 8 + a, Fa, dt);
  if (!upper) {                                               // cell 3: F(face 4) - F(face 3), face 3 is in Fb
    mbar_wait(bar_pair, par_pair);
#pragma unroll
    for (int q = 0; q < 5; ++q) dF[ds + q * NC] = dF[ds + q * NC] - Fb[q];
  }
}

// ---- helpers: staging ----------------------------------------------------------------------------------
// Stages block `blk` into buffer L with TMA.  Lane 0 of helper warp hw issues a quarter of the copies
// (one thread issuing all eleven takes longer than the copies take to land); warp 0 also publishes the
// face sources and arms the barrier with the byte count (the count may go negative in between).
// No proxy fence here: the buffer's last generic-proxy accesses are the walkers' reads, ordered by the
// `full` barrier, and the helpers' own writes, each followed by the writer's fence (prepare()).
template <int STAGE>
__device__ __forceinline__ void issue_loads(const TensorMaps& tm, const StageParams& p, int blk, const int s[6],
                                            int hw, double* L, int* fsrc, uint32_t bar) {
  constexpr int TS = Cfg<STAGE>::TS;
  auto face = [&](int f) {
    const int axis = f >> 1, side = f & 1;
    const int tile = axis == 2 ? side * 5 : axis == 0 ? T_XLO + side : T_YLO + side;
    const uint32_t dst = smem_u32(L + tile * TS);
    if (s[f] >= 0) {
      // my low-side ghost layers are the neighbour's two highest layers, and vice versa
      const int lo = side ? 0 : N - NG;
      if (axis == 2) tensor4_g2s(dst, &tm.zs, 0, 0, lo, s[f] * NV, bar);
      else if (axis == 0) tensor4_g2s(dst, &tm.ax, lo, 0, 0, s[f] * NV, bar);
      else tensor4_g2s(dst, &tm.ay, 0, 0, lo, s[f] * NV, bar);         // map dims (i, k, j, var)
    } else if (s[f] <= -2) {
      bulk_g2s(dst, p.ghost + size_t(-2 - s[f]) * SLAB, SLAB * 8, bar);  // slabs come in the landing layout
    }
  };
  if (hw == 0) {
    uint32_t bytes = 4 * SLAB * 8;
    int any_out = 0;
#pragma unroll
    for (int f = 0; f < 6; ++f) {
      fsrc[f] = s[f];
      bytes += (s[f] != SRC_OUTFLOW) ? SLAB * 8 : 0;
      any_out |= s[f] == SRC_OUTFLOW;
    }
    fsrc[6] = any_out;
    mbar_expect_tx(bar, bytes);             // (release: publishes fsrc to the threads that see the phase complete)
    tensor4_g2s(smem_u32(L + 1 * TS), &tm.zs, 0, 0, 0, blk * NV, bar);   // interior: 4 z-plane pairs
    tensor4_g2s(smem_u32(L + 2 * TS), &tm.zs, 0, 0, 2, blk * NV, bar);
  } else if (hw == 1) {
    tensor4_g2s(smem_u32(L + 3 * TS), &tm.zs, 0, 0, 4, blk * NV, bar);
    tensor4_g2s(smem_u32(L + 4 * TS), &tm.zs, 0, 0, 6, blk * NV, bar);
    face(4);
  } else if (hw == 2) {
    face(5); face(0); face(1);
  } else {
    face(2); face(3);
  }
}

// staged conserved cells -> primitives + c_s + E, in place (predictor): the 512 interior cells and the
// ONE halo layer next to each face (the predictor is first order) = 896 cells.  The WALKERS convert the
// next block between two walks (12 warps finish it in a fraction of the time the 4 helper warps need,
// and the helpers' chain staging -> conversion -> ready was what the walkers waited for): walker thread
// t converts items t, t + 384 and (t < 128) t + 768 of the list [512 interior | z | x | y halo layers].
// Staged cell after the conversion: (rho, vx, vy, vz, E, P, x) with x what the solver needs once per cell: c_s
// (HLLC, RS = 0) or 1/sqrt(rho) (Roe's weights, RS = 1).
template <int RS>
__device__ __forceinline__ void convert_cell(double* __restrict__ c, double gamma, double gm1) {
  double u[5], w[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) u[v] = c[v * CVS];
  const double ir = cons_to_prim(u, gm1, w);
#pragma unroll
  for (int v = 1; v < 4; ++v) c[v * CVS] = w[v];
  // slot 4 keeps the total energy of the cell as it landed (eq. 8); the pressure goes to slot 5
  c[5 * CVS] = w[4];
  const double c2 = (gamma * w[4]) * ir;                   // c_s^2 = gamma P / rho
  c[6 * CVS] = RS == 0 ? c2 * rsqrt_fast(c2) : rsqrt_fast(u[0]);
}
// halo item h in [0, 384): group g = h >> 7 (z, x, y), side = bit 6, x = h & 63.
//   z: tile 0 layer kl = 1 (positions 64..127) / tile 5 layer kl = 0;  x: tile 6 odd positions (ll = 1) /
//   tile 7 even positions;  y: tile 8 layer ll = 1 (positions 64..127) / tile 9 layer ll = 0
template <int RS>
__device__ __forceinline__ void convert_halo_item(double* __restrict__ L, const int* __restrict__ fsrc, int h,
                                                  double gamma, double gm1) {
  constexpr int TS = Cfg<0>::TS;
  const int g = h >> 7, hi = (h >> 6) & 1, x = h & 63;     // g, hi: warp-uniform
  const int f = (g == 0 ? 4 : g == 1 ? 0 : 2) + hi;
  if (fsrc[f] == SRC_OUTFLOW) return;                      // nothing was staged there
  const int pos = g == 0 ? (hi ? 5 * TS + x : 64 + x)
                : g == 1 ? (T_XLO + hi) * TS + 2 * x + (hi ? 0 : 1)
                         : (T_YLO + hi) * TS + (hi ? x : 64 + x);
  convert_cell<RS>(L + pos, gamma, gm1);
}
template <int RS>
__device__ __forceinline__ void convert_share(double* __restrict__ L, const int* __restrict__ fsrc, double gamma,
                                              double gm1, int tid) {
  constexpr int TS = Cfg<0>::TS;
  convert_cell<RS>(L + (1 + (tid >> 7)) * TS + (tid & 127), gamma, gm1);          // interior tiles 1..3
  if (tid < 128) {
    convert_cell<RS>(L + 4 * TS + tid, gamma, gm1);                                // interior tile 4
    convert_halo_item<RS>(L, fsrc, tid + 256, gamma, gm1);                         // y halos
  } else {
    convert_halo_item<RS>(L, fsrc, tid - 128, gamma, gm1);                         // z and x halos
  }
}

// halo of an outflow face (reading R1): copies of the block's own edge layer
template <int STAGE>
__device__ __forceinline__ void fill_outflow(double* __restrict__ L, const int* __restrict__ fsrc, int hid) {
  constexpr int TS = Cfg<STAGE>::TS, NVW = Cfg<STAGE>::NVW;
#pragma unroll 1
  for (int q = hid; q < 6 * CVS; q += HELP_THREADS) {
    const int f = q >> 7, r = q & 127, axis = f >> 1, side = f & 1;
    if (fsrc[f] != SRC_OUTFLOW) continue;
    const int t = r & 63, ta = t & 7, tb = t >> 3, ll = r >> 6, edge = side ? N - 1 : 0;
    int src, dst;
    if (axis == 0) { src = pos_zcol<TS>(edge, ta, tb); dst = (T_XLO + side) * TS + t * 2 + ll; }
    else if (axis == 1) { src = pos_zcol<TS>(ta, edge, tb); dst = (T_YLO + side) * TS + ll * 64 + tb * 8 + ta; }
    else { src = pos_zcol<TS>(ta, tb, edge); dst = side * 5 * TS + zs_pos(ll, tb, ta); }
#pragma unroll
    for (int v = 0; v < NVW; ++v) L[dst + v * CVS] = L[src + v * CVS];
  }
}

// ---- helpers: update -----------------------------------------------------------------------------------
// U_out = U^n - lambda ((dFx + dFy) + dFz), lambda = dt/(2h) (predictor) or dt/h (corrector).
// The flux differences are stored in the face frame (mass, normal, tangential 1, tangential 2,
// energy): variable v of axis D is entry q with 1 + (D + q - 1) % 3 == v, q = 1..3.
// PRIM_OUT: store primitives (the half-step state).
// Two steps, so that the flux-difference buffer goes back to the walkers as early as possible:
// combine_fluxes turns un into the updated conserved cells (the only shared-memory reads), store_block
// writes them out (PRIM_OUT: as primitives, the half-step state).
__device__ __forceinline__ void combine_fluxes(const double* __restrict__ dF, double un[HC][NV], double lam, int hid) {
#pragma unroll
  for (int r = 0; r < HC; ++r) {
    const int cell = hid + r * HELP_THREADS;
    const int i = cell & 7, j = (cell >> 3) & 7, k = cell >> 6;
    const int cx = dfx_idx(i, j, k), cy = dfy_idx(i, j, k), cz = dfz_idx(i, j, k);
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const int qx = v, qy = (v == 0 || v == 4) ? v : 1 + (v + 1) % 3, qz = (v == 0 || v == 4) ? v : 1 + v % 3;
      const double sum = (dF[qx * NC + cx] + dF[qy * NC + cy]) + dF[qz * NC + cz];
      un[r][v] = un[r][v] - lam * sum;
    }
  }
}
template <bool PRIM_OUT>
__device__ __forceinline__ void store_block(const double u[HC][NV], double gm1, double* __restrict__ Uo, int hid) {
#pragma unroll
  for (int r = 0; r < HC; ++r) {
    const int cell = hid + r * HELP_THREADS;
    if (PRIM_OUT) {
      double w[NV];
      cons_to_prim(u[r], gm1, w);
#pragma unroll
      for (int v = 0; v < NV; ++v) Uo[v * NC + cell] = w[v];
    } else {
#pragma unroll
      for (int v = 0; v < NV; ++v) Uo[v * NC + cell] = u[r][v];
    }
  }
}

// ---- the stage kernel ------------------------------------------------------------------------------------
// CTA c handles blocks c, c + gridDim.x, ... of the level ("iterations" it = 0, 1, ...).  Barriers:
//   landed[s]  the TMA copies of the block staged in buffer s = it & 1 are complete (transaction count)
//   conv[s]    predictor: the walkers have converted buffer s to primitives (their share each)
//   ready[s]   buffer s is prepared (conversion by the walkers, outflow halos by the helpers): walk it
//   full[d]    all walkers have stored the flux differences into buffer d = it % NDF (and are done with
//              the staging buffer, which the helpers then re-stage)
//   empty[d]   the helpers have consumed flux-difference buffer d
// MFX: also export the mass flux of every face to p.mf (the passive-scalar kernels read it)
template <int STAGE, int RS, bool REGS, bool MFX>
__global__ void __launch_bounds__(STAGE_THREADS, 1) stage_kernel(const __grid_constant__ TensorMaps tm,
                                                                  const StageParams p) {
  using C = Cfg<STAGE>;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* L0 = reinterpret_cast<double*>(smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u));
  double* dF0 = L0 + 2 * C::LAND;
  uint64_t* bars = reinterpret_cast<uint64_t*>(dF0 + C::NDF * DF_DOUBLES);
  int* fsrc0 = reinterpret_cast<int*>(bars + 10);           // [2][8]
  double* hmax = reinterpret_cast<double*>(bars + 20);      // [2][4] per-helper-warp maximum speed, double buffered
  const uint32_t bar0 = smem_u32(bars);
  auto landed = [&](int s) { return bar0 + 8u * s; };
  auto ready = [&](int s) { return bar0 + 16u + 8u * s; };
  auto full = [&](int d) { return bar0 + 32u + 8u * d; };
  auto empty = [&](int d) { return bar0 + 48u + 8u * d; };
  auto conv = [&](int s) { return bar0 + 64u + 8u * s; };   // predictor: the walkers have converted buffer s
  // pair[P][it & 1]: the upper half pencils of (axis, pencil half) P have stored face 4 of block it.  Two per pair: the
  // upper warp may be a block ahead of the lower one, never two (the staging of block it + 2 waits for `full` of block it).
  auto pair = [&](int P, int it) { return bar0 + 224u + 8u * (2 * P + (it & 1)); };

  const int tid = threadIdx.x;
  const int stride = gridDim.x;
  const int blk0 = p.first + blockIdx.x;
  const int n = (p.count - int(blockIdx.x) + stride - 1) / stride;    // my iterations
  if (tid == 0) {
    for (int s = 0; s < 2; ++s) {
      mbar_init(landed(s), 1);
      mbar_init(ready(s), STAGE == 0 ? WALK_WARPS + HELP_WARPS : HELP_WARPS);
      mbar_init(conv(s), WALK_WARPS);
      mbar_init(full(s), WALK_WARPS);
      mbar_init(empty(s), HELP_WARPS);
    }
    for (int P = 0; P < 12; ++P) mbar_init(bar0 + 224u + 8u * P, 1);
    fence_mbar_init();
  }
  __syncthreads();
  const double gamma = p.gamma, gm1 = p.gamma - 1.0;
  const double dt = p.dt_dev ? *p.dt_dev : p.dt;

  if (tid < WALK_THREADS) {
    // ------------------------------------------------------------------------------ walkers

    const double igm1 = 1.0 / gm1;
    // Predictor: thread (D, half, pencil) walks faces 4 half .. 4 half + 4 (face 4 twice: its single flux-difference
    // buffer makes the walkers meet at every block anyway, measured: sharing face 4 loses 4 % there).
    // Corrector: no face is computed twice.  Warp w owns (axis D, pencils 32 q .. 32 q + 31) and one HALF: the upper half
    // computes faces 4..8 and hands face 4 to the lower half through cell 3's flux-difference slot, the lower half
    // computes faces 0..3.  The halves change hands every block, so that every warp averages 4.5 faces per block (its
    // two flux-difference buffers let a warp run up to a block ahead of the others), and they are dealt so that each
    // sub-partition (warp & 3) carries 14 or 13 faces per pencil at any time instead of 15.
    const int wp = tid >> 5, sub = wp & 3, slot = wp >> 2;
    const int P = STAGE == 0 ? (wp >> 2) + 3 * (wp & 1) : (sub >> 1) * 3 + slot;      // P = D + 3 q
    const int D = P % 3;
    const bool upper0 = STAGE == 0 ? ((wp >> 1) & 1) != 0 : ((sub & 1) ? slot == 2 : slot < 2);
    const int f0 = upper0 ? 4 : 0, pen = (P / 3) * 32 + (tid & 31), a = pen & 7, b = pen >> 3;
    WalkGeom geom;
    if (STAGE == 1) {
      if (D == 0) walk_geom<1, 0>(a, b, geom);
      else if (D == 1) walk_geom<1, 1>(a, b, geom);
      else walk_geom<1, 2>(a, b, geom);
    }
    auto convert_next = [&](int it) {                  // predictor: my share of block it, then both arrivals
      const int s = it & 1;
      mbar_wait(landed(s), (it >> 1) & 1);
      convert_share<RS>(L0 + s * C::LAND, fsrc0 + 8 * s, gamma, gm1, tid);
      fence_proxy_async();                             // my generic-proxy writes, before a later TMA overwrites them
      __syncwarp();
      if ((tid & 31) == 0) { mbar_arrive(conv(s)); mbar_arrive(ready(s)); }
    };
    if (STAGE == 0) convert_next(0);
    for (int it = 0; it < n; ++it) {
      const int s = it & 1, d = it % C::NDF;
      const double* Wl = L0 + s * C::LAND;
      double* dF = dF0 + d * DF_DOUBLES;
      const bool we = it >= C::NDF;
      const uint32_t pe = ((it / C::NDF) - 1) & 1;
      mbar_wait(ready(s), (it >> 1) & 1);
      const int blk = blk0 + it * stride;
      // mass fluxes of the block: [axis][face 0..8][pencil]
      double* mf = MFX ? p.mf + (size_t(blk) * 3 + D) * (9 * FACE) + pen : nullptr;
      if (STAGE == 0) {
        if (D == 0) walk_predictor<RS, 0, MFX>(Wl, dF, a, b, f0, gm1, igm1, empty(d), pe, we, mf);
        else if (D == 1) walk_predictor<RS, 1, MFX>(Wl, dF, a, b, f0, gm1, igm1, empty(d), pe, we, mf);
        else walk_predictor<RS, 2, MFX>(Wl, dF, a, b, f0, gm1, igm1, empty(d), pe, we, mf);
      } else {
        walk_corrector_generic<RS, REGS, MFX>(Wl, dF, geom, D, a, b, gamma, igm1, p, blk, dt, empty(d), pe, we, mf,
                                              upper0 != bool(it & 1), pair(P, it), (it >> 1) & 1);
      }
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(full(d));
      if (STAGE == 0 && it + 1 < n) convert_next(it + 1);
    }
  } else {
    // ------------------------------------------------------------------------------ helpers
    const int hid = tid - WALK_THREADS, hw = hid >> 5;
    const bool lane0 = (tid & 31) == 0;
    const double lam = (STAGE == 0 ? 0.5 : 1.0) * dt / p.h;
    auto prepare = [&](int it) {
      const int s = it & 1;
      double* L = L0 + s * C::LAND;
      const int* fsrc = fsrc0 + 8 * s;
      mbar_wait(landed(s), (it >> 1) & 1);
      if (fsrc[6]) {                                   // block-uniform: some face is an outflow face
        if (STAGE == 0) mbar_wait(conv(s), (it >> 1) & 1);   // the edge layers are converted
        fill_outflow<STAGE>(L, fsrc, hid);
        fence_proxy_async();                           // my generic-proxy writes, before a later TMA overwrites them
      }
      __syncwarp();
      if (lane0) mbar_arrive(ready(s));
    };
    auto load_src = [&](int it, int s[6]) {            // face sources of my it-th block
#pragma unroll
      for (int f = 0; f < 6; ++f) s[f] = p.face_src[(blk0 + it * stride) * 6 + f];
    };
    if (lane0) {
      for (int it = 0; it < 2 && it < n; ++it) {
        int s[6];
        load_src(it, s);
        issue_loads<STAGE>(tm, p, blk0 + it * stride, s, hw, L0 + it * C::LAND, fsrc0 + 8 * it, landed(it));
      }
      if (hw == 3 && n > 2) {
        prefetch_l2(p.Usrc + size_t(blk0 + 2 * stride) * BLK, BLK * 8);
        if (STAGE == 1) prefetch_l2(p.Un + size_t(blk0 + 2 * stride) * BLK, BLK * 8);
      }
    }
    __syncwarp();
    for (int it = 0; it < 2 && it < n; ++it) prepare(it);
    for (int it = 0; it < n; ++it) {
      const int s = it & 1, d = it % C::NDF;
      const int blk = blk0 + it * stride;
      // U^n of the block and the face sources of the block after next: in flight while the walkers finish
      double un[HC][NV];
      const double* Un = p.Un + size_t(blk) * BLK;
#pragma unroll
      for (int r = 0; r < HC; ++r)
#pragma unroll
        for (int v = 0; v < NV; ++v) un[r][v] = Un[v * NC + hid + r * HELP_THREADS];
      int snext[6];
      if (lane0 && it + 2 < n) load_src(it + 2, snext);
      mbar_wait(full(d), (it / C::NDF) & 1);
      if (lane0 && it + 2 < n) {                       // the walkers are done with staging buffer s as well
        issue_loads<STAGE>(tm, p, blk + 2 * stride, snext, hw, L0 + s * C::LAND, fsrc0 + 8 * s, landed(s));
        if (hw == 3 && it + 3 < n) {
          prefetch_l2(p.Usrc + size_t(blk + 3 * stride) * BLK, BLK * 8);
          if (STAGE == 1) prefetch_l2(p.Un + size_t(blk + 3 * stride) * BLK, BLK * 8);
        }
      }
      __syncwarp();
      combine_fluxes(dF0 + d * DF_DOUBLES, un, lam, hid);
      __syncwarp();
      if (lane0) mbar_arrive(empty(d));                // the walkers may store the next flux differences
      store_block<STAGE == 0>(un, gm1, p.Udst + size_t(blk) * BLK, hid);
      if (STAGE == 0 && it + 2 < n) prepare(it + 2);
      if (STAGE == 1 && p.bmax) {
        // The block's maximum CFL speed for the next step's dt (reading R16) from the updated cells still in
        // registers, after everything the walkers wait for has been handed over.  (Measured: these 26 fp64
        // instructions per cell cost the corrector 10 %: the stage kernels are bound by the instructions the SM
        // sub-partitions can dispatch, whichever warp they come from.)
        double sp[HC];
#pragma unroll
        for (int r = 0; r < HC; ++r) sp[r] = cell_speed(un[r], gamma, gm1);   // four independent chains
        const double s = warp_max(fmax(fmax(sp[0], sp[1]), fmax(sp[2], sp[3])));
        double* hm = hmax + 4 * (it & 1);
        if (lane0) hm[hw] = s;
        asm volatile("bar.sync 1, %0;" ::"n"(HELP_THREADS) : "memory");
        if (hid == 0) p.bmax[blk] = fmax(fmax(hm[0], hm[1]), fmax(hm[2], hm[3]));
      }
      // (corrector: after the block maximum, whose arithmetic covers the landing of the copies issued above)
      if (STAGE == 1 && it + 2 < n) prepare(it + 2);
    }
  }
}

// ---- host side: one set of instantiations per MFX value (sfh_kernels.cu: false, sfh_kernels_mf.cu: true) ------
template <int STAGE, int RS, bool REGS, bool MFX>
static cudaError_t configure_one() {
  return cudaFuncSetAttribute(stage_kernel<STAGE, RS, REGS, MFX>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              Cfg<STAGE>::SMEM);
}
template <bool MFX>
static cudaError_t configure_stage_kernels() {
  cudaError_t e;
  if ((e = configure_one<0, 0, false, MFX>()) != cudaSuccess || (e = configure_one<0, 1, false, MFX>()) != cudaSuccess ||
      (e = configure_one<1, 0, false, MFX>()) != cudaSuccess || (e = configure_one<1, 0, true, MFX>()) != cudaSuccess ||
      (e = configure_one<1, 1, false, MFX>()) != cudaSuccess || (e = configure_one<1, 1, true, MFX>()) != cudaSuccess)
    return e;
  return cudaSuccess;
}
template <int STAGE, int RS, bool REGS, bool MFX>
static void launch_one(int grid, const TensorMaps& tm, const StageParams& p, cudaStream_t st) {
  stage_kernel<STAGE, RS, REGS, MFX><<<grid, STAGE_THREADS, Cfg<STAGE>::SMEM, st>>>(tm, p);
}
// The corrector of a level with flux-register faces is its own instantiation: the register code costs the
// uniform-grid walk a few per cent even when it never runs (measured).
template <bool MFX>
static cudaError_t launch_stage_impl(int stage, const TensorMaps& tm, const StageParams& p, int sms, cudaStream_t st) {
  if (p.count <= 0) return cudaSuccess;
  const int grid = p.count < sms ? p.count : sms;
  const bool roe = p.riemann != 0;
  if (stage == 0) {
    if (roe) launch_one<0, 1, false, MFX>(grid, tm, p, st); else launch_one<0, 0, false, MFX>(grid, tm, p, st);
  } else if (p.use_regs) {
    if (roe) launch_one<1, 1, true, MFX>(grid, tm, p, st); else launch_one<1, 0, true, MFX>(grid, tm, p, st);
  } else {
    if (roe) launch_one<1, 1, false, MFX>(grid, tm, p, st); else launch_one<1, 0, false, MFX>(grid, tm, p, st);
  }
  return cudaGetLastError();
}

}  // namespace sfh

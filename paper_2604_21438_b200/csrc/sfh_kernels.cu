// sfh_kernels.cu — CUDA kernels of libsfh for sm_100a (B200).
//
// Stage kernels (predictor a4, corrector a6+a7 of SURVEY.md section 8(a)): one CTA of 192 threads
// per 8^3 block.  Thread 0 issues the TMA copies that stage the block and its 6 two-layer face
// halos in shared memory: one contiguous bulk copy for the interior, and per face either a 4-D
// tiled tensor copy straight out of the same-level neighbour's interior (the ghost "fill" is this
// gather), or a bulk copy of the coarse-fine ghost slab written by the prolongation kernel, or
// nothing for an outflow face.  All threads convert the 1280 staged cells to primitive variables
// into a second shared array laid out for conflict-free pencil walks, then 64 threads per axis walk
// the 64 pencils of that axis (x, y and z concurrently, two warps each), computing each face flux
// once and writing flux differences to shared memory (the staging area, now dead, is reused), and
// finally all threads combine U - lambda (dFx + dFy + dFz) with coalesced global loads/stores.
// The pencil walk with flux reuse is the paper's own mapping (Fig. 1); running the
// three axes side by side and staging through TMA is this design's.
#include <cmath>

#include "sfh_device.cuh"
#include "sfh_kernels.cuh"

namespace sfh {

constexpr int STAGE_THREADS = 192;
constexpr int LAND_INT = 0;                 // landing area (doubles): interior [5][8][8][8]
constexpr int LAND_HALO = BLK;              // then 6 slabs of SLAB doubles, face f = 2*axis + side
constexpr int LAND_DOUBLES = BLK + 6 * SLAB;  // 6400
constexpr int DF_DOUBLES = 3 * BLK;           // 7680, aliases the landing area
constexpr int W_DOUBLES = 6720;               // the primitive array (both stages)
constexpr int STAGE_SMEM = (W_DOUBLES + DF_DOUBLES) * 8 + 16 + 32;   // 115248 B (+1 KB reserved) -> 2 CTAs per SM

// Primitive-array layout for a stage with H halo layers and NVW stored variables: W[var][pos], every
// variable with the same stride VS, so that a cell's variables sit at compile-time offsets from the
// cell's position.  Positions: 64 x rows of 8+2H cells (+1 pad: odd stride, conflict-free x pencils),
// then the two y slabs [side][k][h][i], then the two z slabs [side][h][j][i].
template <int H, int NVW>
struct WLayout {
  static constexpr int RS = N + 2 * H + 1;          // x-row stride
  static constexpr int YS = N * H * N;              // one y slab
  static constexpr int ZS = H * N * N;              // one z slab
  static constexpr int Y0 = 64 * RS;
  static constexpr int Z0 = Y0 + 2 * YS;
  static constexpr int VS = Z0 + 2 * ZS;            // variable stride
  static constexpr int TOTAL = NVW * VS;
};

// ---- conversion of the staged conserved cells to primitives --------------------------------------
template <int STAGE>
__device__ __forceinline__ void convert_cell(const double* __restrict__ L, double* __restrict__ W, int src, int svs,
                                             int dst, double gamma, double gm1) {
  constexpr int H = STAGE == 0 ? 1 : 2;
  constexpr int NVW = STAGE == 0 ? 7 : 5;
  using WL = WLayout<H, NVW>;
  double u[5], w[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) u[v] = L[src + v * svs];
  const double ir = cons_to_prim(u, gm1, w);
#pragma unroll
  for (int v = 0; v < 5; ++v) W[dst + v * WL::VS] = w[v];
  if (STAGE == 0) {
    const double c2 = (gamma * w[4]) * ir;         // c_s^2 = gamma P / rho
    W[dst + 5 * WL::VS] = c2 * rsqrt_fast(c2);
    W[dst + 6 * WL::VS] = u[4];                    // total energy of the cell (eq. 8)
  }
}

// Interior: 512 cells in 3 rounds.  Halo: the H layers next to each of the 6 faces, 64 H cells per
// face; a warp covers 32 consecutive cells of ONE face, so the per-axis branches are warp-uniform.
// An outflow face (reading R1) has no staged slab: its halo cells copy the block's own edge layer.
template <int STAGE>
__device__ __forceinline__ void convert_block(const double* __restrict__ L, double* __restrict__ W,
                                              const int* __restrict__ fsrc, double gamma, double gm1, int tid) {
  constexpr int H = STAGE == 0 ? 1 : 2;
  constexpr int NVW = STAGE == 0 ? 7 : 5;
  using WL = WLayout<H, NVW>;
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    const int cell = tid + r * STAGE_THREADS;
    if (cell < NC) convert_cell<STAGE>(L, W, LAND_INT + cell, NC, (cell >> 3) * WL::RS + (cell & 7) + H, gamma, gm1);
  }
  constexpr int PER_FACE = H * FACE;               // 64 or 128
#pragma unroll
  for (int r = 0; r < 6 * PER_FACE / STAGE_THREADS; ++r) {
    const int q = tid + r * STAGE_THREADS;
    const int f = q / PER_FACE, rr = q % PER_FACE, axis = f >> 1, side = f & 1;
    const int t = rr & 63, ta = t & 7, tb = t >> 3;
    const int hh = rr >> 6;                        // layer within the H halo layers, outwards-increasing index c
    const int ll = side ? hh : hh + NG - H;        // layer within the staged 2-layer slab
    const bool outflow = fsrc[f] == SRC_OUTFLOW;
    const int edge = side ? N - 1 : 0;
    int src, dst;
    if (axis == 0) {          // ta = j, tb = k; slab [v][k][j][ll]
      src = outflow ? LAND_INT + t * 8 + edge : LAND_HALO + f * SLAB + t * 2 + ll;
      dst = t * WL::RS + (side ? N + H + hh : hh);
    } else if (axis == 1) {   // ta = i, tb = k; slab [v][k][ll][i]
      src = outflow ? LAND_INT + tb * 64 + edge * 8 + ta : LAND_HALO + f * SLAB + tb * 16 + ll * 8 + ta;
      dst = WL::Y0 + side * WL::YS + (tb * H + hh) * 8 + ta;
    } else {                  // ta = i, tb = j; slab [v][ll][j][i]
      src = outflow ? LAND_INT + edge * 64 + t : LAND_HALO + f * SLAB + ll * 64 + t;
      dst = WL::Z0 + side * WL::ZS + hh * 64 + t;
    }
    convert_cell<STAGE>(L, W, src, outflow ? NC : NG * FACE, dst, gamma, gm1);
  }
}

// ---- pencil walks ----------------------------------------------------------------------------------
// One thread per pencil; 64 pencils per axis; the three axes run side by side in different warps but
// through the SAME loop body (run-time positions and strides), so the instruction footprint is one
// flux body per stage.  Face f = 0..8 of a pencil lies between cells f-1 and f; each flux is computed
// once and used by both adjacent cells (the paper's mapping).  A pencil is three runs of
// positions in W: cells -H..-1 (low halo), 0..7 (interior x row), 8..7+H (high halo); the walk keeps
// one running position that is re-seated when it enters the next run.  Loops are unrolled by two so
// that the carried cell/face state ping-pongs between registers instead of being moved.
template <int H, int NVW>
struct Pencil {
  using WL = WLayout<H, NVW>;
  int lo0, lo_cs;          // cell c < 0 at lo0 + (c + H) * lo_cs
  int mid0, mid_cs;        // cell 0..7 at mid0 + c * mid_cs
  int hi0, hi_cs;          // cell c >= 8 at hi0 + (c - 8) * hi_cs
  int on, ot1, ot2;        // offsets of the normal / tangential velocity variables
  int df0, df_cs, df_swz;  // flux-difference index of cell c: df0 + ((c ^ df_swz) * df_cs)
  __device__ __forceinline__ Pencil(int D, int a, int b) {
    on = (1 + D) * WL::VS; ot1 = (1 + (D + 1) % 3) * WL::VS; ot2 = (1 + (D + 2) % 3) * WL::VS;
    if (D == 0) {
      lo0 = (b * 8 + a) * WL::RS; lo_cs = 1;
      mid0 = lo0 + H; mid_cs = 1;
      hi0 = mid0 + N; hi_cs = 1;
      df0 = (b * 8 + a) * 8; df_cs = 1; df_swz = a;      // x rows are XOR swizzled (bank spread)
    } else if (D == 1) {
      lo0 = WL::Y0 + b * H * 8 + a; lo_cs = 8;
      mid0 = b * 8 * WL::RS + a + H; mid_cs = WL::RS;
      hi0 = lo0 + WL::YS; hi_cs = 8;
      df0 = D * BLK + b * 64 + a; df_cs = 8; df_swz = 0;
    } else {
      lo0 = WL::Z0 + b * 8 + a; lo_cs = 64;
      mid0 = b * WL::RS + a + H; mid_cs = 8 * WL::RS;
      hi0 = lo0 + WL::ZS; hi_cs = 64;
      df0 = D * BLK + b * 8 + a; df_cs = 64; df_swz = 0;
    }
  }
  // the cell at position o, in the face frame (rho, normal v, tangential v's, P[, c_s, E])
  __device__ __forceinline__ void load(const double* __restrict__ W, int o, double w[NVW]) const {
    w[0] = W[o]; w[1] = W[o + on]; w[2] = W[o + ot1]; w[3] = W[o + ot2]; w[4] = W[o + 4 * WL::VS];
    if (NVW == 7) { w[5] = W[o + 5 * WL::VS]; w[6] = W[o + 6 * WL::VS]; }
  }
  // dF of cell c = F(face c+1) - F(face c), stored in the FACE frame (the update un-permutes)
  __device__ __forceinline__ void store_df(double* __restrict__ dF, int c, const double Fa[5], const double Fb[5]) const {
    const int ci = df0 + ((c ^ df_swz) * df_cs);
#pragma unroll
    for (int q = 0; q < 5; ++q) dF[ci + q * NC] = Fa[q] - Fb[q];
  }
};

// flux registers at coarse-fine faces (a7; reading R14); Fn in the face frame
__device__ __noinline__ void store_regs(const int32_t* face_src, const int32_t* fslot, double* R, double* FH, int blk,
                                        int D, int side, int t, double F0, double F1, double F2, double F3, double F4,
                                        double dt) {
  const double Fn[5] = {F0, F1, F2, F3, F4};
  const int f = 2 * D + side;
  const int src = face_src[blk * 6 + f];
  const int fs = fslot[blk * 6 + f];
  const int vn = 1 + D, vt1 = 1 + (D + 1) % 3, vt2 = 1 + (D + 2) % 3;
  if (src <= -2) {   // fine side of a coarse-fine face: accumulate dt * F
    double* r = R + size_t(-2 - src) * REG + t;
    r[0] += dt * Fn[0]; r[vn * FACE] += dt * Fn[1]; r[vt1 * FACE] += dt * Fn[2]; r[vt2 * FACE] += dt * Fn[3];
    r[4 * FACE] += dt * Fn[4];
  }
  if (fs >= 0) {     // coarse leaf next to a covered block: keep its own flux
    double* r = FH + size_t(fs) * REG + t;
    r[0] = Fn[0]; r[vn * FACE] = Fn[1]; r[vt1 * FACE] = Fn[2]; r[vt2 * FACE] = Fn[3]; r[4 * FACE] = Fn[4];
  }
}

// predictor: first-order HLLC on the cell-centred states (reading R8)
__device__ __forceinline__ void walk_predictor(const double* __restrict__ W, double* __restrict__ dF, int D, int a, int b,
                                               double igm1) {
  const Pencil<1, 7> pc(D, a, b);
  double w0[7], w1[7], F0[5], F1[5];
  pc.load(W, pc.lo0, w0);                     // cell -1
  pc.load(W, pc.mid0, w1);                    // cell 0
  hllc_flux<true>(w0[0], w0[1], w0[2], w0[3], w0[4], w0[5], w0[6], w1[0], w1[1], w1[2], w1[3], w1[4], w1[5], w1[6],
                  igm1, F0);                  // face 0
  int o = pc.mid0;
#pragma unroll 1
  for (int f = 1; f < N; f += 2) {            // faces f (cells f-1 | f) and f+1 (cells f | f+1)
    o += pc.mid_cs;
    pc.load(W, o, w0);                        // cell f
    hllc_flux<true>(w1[0], w1[1], w1[2], w1[3], w1[4], w1[5], w1[6], w0[0], w0[1], w0[2], w0[3], w0[4], w0[5], w0[6],
                    igm1, F1);
    pc.store_df(dF, f - 1, F1, F0);
    o = (f + 1 == N) ? pc.hi0 : o + pc.mid_cs;
    pc.load(W, o, w1);                        // cell f+1
    hllc_flux<true>(w0[0], w0[1], w0[2], w0[3], w0[4], w0[5], w0[6], w1[0], w1[1], w1[2], w1[3], w1[4], w1[5], w1[6],
                    igm1, F0);
    pc.store_df(dF, f, F0, F1);
  }
}

// corrector: minmod-limited linear reconstruction of the primitives (readings R11, R12) + HLLC
// slope of the cell with value wc from its two one-sided differences; returns the right state of the
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
__device__ __forceinline__ void corrector_flux(const double WLs[5], const double WRs[5], double gamma, double igm1,
                                               double Fn[5]) {
  const double cL = sound_speed(gamma, WLs[4], WLs[0]);
  const double cR = sound_speed(gamma, WRs[4], WRs[0]);
  hllc_flux<false>(WLs[0], WLs[1], WLs[2], WLs[3], WLs[4], cL, 0.0, WRs[0], WRs[1], WRs[2], WRs[3], WRs[4], cR, 0.0,
                   igm1, Fn);
}

// ---- corrector: landing layout and walk -------------------------------------------------------------
// The half-step state is stored as primitives, so the corrector needs no
// conversion: the pencils walk the staged tiles where TMA put them.  Landing area (doubles), every
// tile [v][128 cells] (variable stride 128):
//   z column: 6 z-plane pairs of 640 doubles: the low z halo, the 4 interior pairs, the high z halo,
//             each 128-byte swizzled (zs_pos), so a cell (i, j, k), k in [-2, 10), sits at
//             ((k + 2) >> 1) * 640 + zs_pos(k & 1, j, i);
//   then the x-low, x-high, y-low, y-high slabs, dense: x [v][k][j][ll], y [v][k][ll][i].
constexpr int C_ZCOL = 0, C_XLO = 6 * SLAB, C_XHI = 7 * SLAB, C_YLO = 8 * SLAB, C_YHI = 9 * SLAB;
constexpr int C_LAND = 10 * SLAB;                    // 6400 doubles
constexpr int CORR_SMEM = (C_LAND + DF_DOUBLES) * 8 + 16 + 32 + 1024;   // 113712 B (1 KB alignment slack) -> 2 CTAs per SM
constexpr int CVS = NG * FACE;                       // variable stride of every tile (128)

__device__ __forceinline__ int c_pos_zcol(int i, int j, int k) { return ((k + 2) >> 1) * SLAB + zs_pos(k & 1, j, i); }

// position of cell c in [-2, 10) of the pencil (a, b) along axis D
template <int D>
__device__ __forceinline__ int c_pos(int c, int a, int b) {
  if (D == 2) return c_pos_zcol(a, b, c);
  if (D == 0) {
    if (c < 0) return C_XLO + (b * 8 + a) * 2 + c + 2;
    if (c >= N) return C_XHI + (b * 8 + a) * 2 + c - N;
    return c_pos_zcol(c, a, b);
  }
  if (c < 0) return C_YLO + b * 16 + (c + 2) * 8 + a;
  if (c >= N) return C_YHI + b * 16 + (c - N) * 8 + a;
  return c_pos_zcol(a, c, b);
}

template <int D>
__device__ __forceinline__ void c_load(const double* __restrict__ Wl, int o, double w[5]) {
  constexpr int vn = 1 + D, vt1 = 1 + (D + 1) % 3, vt2 = 1 + (D + 2) % 3;
  w[0] = Wl[o]; w[1] = Wl[o + vn * CVS]; w[2] = Wl[o + vt1 * CVS]; w[3] = Wl[o + vt2 * CVS]; w[4] = Wl[o + 4 * CVS];
}

// dF of cell c of the pencil = F(face c+1) - F(face c), in the FACE frame (the update un-permutes)
template <int D>
__device__ __forceinline__ void c_store_df(double* __restrict__ dF, int c, int a, int b, const double Fa[5],
                                           const double Fb[5]) {
  const int ci = D == 0 ? (b * 8 + a) * 8 + (c ^ a) : D == 1 ? BLK + b * 64 + c * 8 + a : 2 * BLK + c * 64 + b * 8 + a;
#pragma unroll
  for (int q = 0; q < 5; ++q) dF[ci + q * NC] = Fa[q] - Fb[q];
}

template <int D>
__device__ __forceinline__ void walk_corrector(const double* __restrict__ Wl, double* __restrict__ dF, int a, int b,
                                               double gamma, double igm1, const StageParams& p, int blk, double dt) {
  double wa[5], wb[5], da[5], db[5], La[5], Lb[5], R[5], F0[5], F1[5];
  // cells -2, -1, 0: slope of cell -1 -> left state of face 0
  c_load<D>(Wl, c_pos<D>(-2, a, b), wa);
  c_load<D>(Wl, c_pos<D>(-1, a, b), wb);
#pragma unroll
  for (int v = 0; v < 5; ++v) da[v] = wb[v] - wa[v];          // W_-1 - W_-2
  c_load<D>(Wl, c_pos<D>(0, a, b), wa);
#pragma unroll
  for (int v = 0; v < 5; ++v) db[v] = wa[v] - wb[v];          // W_0 - W_-1
  limited_states(wb, db, da, R, La);                          // La = left state of face 0
  // face 0: cell 1 gives the slope of cell 0
  c_load<D>(Wl, c_pos<D>(1, a, b), wb);
#pragma unroll
  for (int v = 0; v < 5; ++v) da[v] = wb[v] - wa[v];          // W_1 - W_0
  limited_states(wa, da, db, R, Lb);                          // R = right state of face 0, Lb = left of face 1
  corrector_flux(La, R, gamma, igm1, F0);
  if (p.use_regs) store_regs(p.face_src, p.fslot, p.R, p.FH, blk, D, 0, b * 8 + a, F0[0], F0[1], F0[2], F0[3], F0[4], dt);
  // invariant at the top of a trip (f odd): wb = W_f, da = W_f - W_{f-1}, Lb = left state of face f,
  // F0 = flux of face f-1
#pragma unroll 1
  for (int f = 1; f < N; f += 2) {
    c_load<D>(Wl, c_pos<D>(f + 1, a, b), wa);                 // cell f+1
#pragma unroll
    for (int v = 0; v < 5; ++v) db[v] = wa[v] - wb[v];
    limited_states(wb, db, da, R, La);                        // right state of face f, left of face f+1
    corrector_flux(Lb, R, gamma, igm1, F1);                   // face f
    c_store_df<D>(dF, f - 1, a, b, F1, F0);
    c_load<D>(Wl, c_pos<D>(f + 2, a, b), wb);                 // cell f+2
#pragma unroll
    for (int v = 0; v < 5; ++v) da[v] = wb[v] - wa[v];
    limited_states(wa, da, db, R, Lb);                        // right state of face f+1, left of face f+2
    corrector_flux(La, R, gamma, igm1, F0);                   // face f+1
    c_store_df<D>(dF, f, a, b, F0, F1);
  }
  if (p.use_regs) store_regs(p.face_src, p.fslot, p.R, p.FH, blk, D, 1, b * 8 + a, F0[0], F0[1], F0[2], F0[3], F0[4], dt);
}

// ---- the stage kernels -------------------------------------------------------------------------------
// Both are persistent: CTA c of the grid handles blocks c, c + gridDim.x, ... of the level, thread 0
// stages each block with TMA and everybody waits on ONE mbarrier whose phase alternates per block.
// The block after the one being staged is pulled into L2 at the same time, so the TMA copies hit L2
// instead of paying the DRAM latency on the critical path.

// U_out = U^n - lambda ((dFx + dFy) + dFz), lambda = dt/(2h) (predictor) or dt/h (corrector).
// The flux differences are stored in the face frame (mass, normal, tangential 1, tangential 2,
// energy): variable v of axis D is entry q with 1 + (D + q - 1) % 3 == v, q = 1..3.
// 3 rounds of cells, all 5 variables each.  PRIM_OUT: store primitives (the half-step state).
constexpr int CR = (NC + STAGE_THREADS - 1) / STAGE_THREADS;
__device__ __forceinline__ void load_un(const double* __restrict__ Un, int tid, double un[CR][NV]) {
#pragma unroll
  for (int r = 0; r < CR; ++r) {
    const int cell = tid + r * STAGE_THREADS;
#pragma unroll
    for (int v = 0; v < NV; ++v) un[r][v] = cell < NC ? Un[v * NC + cell] : 0.0;
  }
}
template <bool PRIM_OUT>
__device__ __forceinline__ void update_block(const double* __restrict__ dF, const double un[CR][NV], double lam,
                                             double gm1, double* __restrict__ Uo, int tid) {
#pragma unroll
  for (int r = 0; r < CR; ++r) {
    const int cell = tid + r * STAGE_THREADS;
    if (cell < NC) {
      const int row = cell >> 3, i = cell & 7;
      const int cx = row * 8 + (i ^ (row & 7));
      double u[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const int qx = v, qy = (v == 0 || v == 4) ? v : 1 + (v + 1) % 3, qz = (v == 0 || v == 4) ? v : 1 + v % 3;
        const double sum = (dF[qx * NC + cx] + dF[BLK + qy * NC + cell]) + dF[2 * BLK + qz * NC + cell];
        u[v] = un[r][v] - lam * sum;
      }
      if (PRIM_OUT) {
        double w[NV];
        cons_to_prim(u, gm1, w);
#pragma unroll
        for (int v = 0; v < NV; ++v) Uo[v * NC + cell] = w[v];
      } else {
#pragma unroll
        for (int v = 0; v < NV; ++v) Uo[v * NC + cell] = u[v];
      }
    }
  }
}

// ---- predictor: stage conserved U^n -> convert -> walks -> update, stores W^{n+1/2} (primitives) ----
__device__ __forceinline__ void issue_predictor_loads(const TensorMaps& tm, const StageParams& p, int blk, double* L,
                                                      int* fsrc, uint32_t bar_a) {
  int s[6];
#pragma unroll
  for (int f = 0; f < 6; ++f) s[f] = p.face_src[blk * 6 + f];
  uint32_t bytes = BLK * 8;
#pragma unroll
  for (int f = 0; f < 6; ++f) {
    fsrc[f] = s[f];
    bytes += (s[f] != SRC_OUTFLOW) ? SLAB * 8 : 0;
  }
  fence_proxy_async();                    // the landing area was last written through the generic proxy
  mbar_expect_tx(bar_a, bytes);           // (release: publishes fsrc to the threads that see the phase complete)
  bulk_g2s(smem_u32(L + LAND_INT), p.Usrc + size_t(blk) * BLK, BLK * 8, bar_a);
#pragma unroll
  for (int f = 0; f < 6; ++f) {
    const uint32_t dst = smem_u32(L + LAND_HALO + f * SLAB);
    if (s[f] >= 0) {
      // my low-side ghost layers are the neighbour's two highest layers, and vice versa
      const int axis = f >> 1, lo = (f & 1) ? 0 : N - NG;
      tensor4_g2s(dst, &tm.ax[axis], axis == 0 ? lo : 0, axis == 1 ? lo : 0, axis == 2 ? lo : 0, s[f] * NV, bar_a);
    } else if (s[f] <= -2) {
      bulk_g2s(dst, p.ghost + size_t(-2 - s[f]) * SLAB, SLAB * 8, bar_a);
    }
  }
}

__global__ void __launch_bounds__(STAGE_THREADS, 2)
predictor_kernel(const __grid_constant__ TensorMaps tm, const StageParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* W = reinterpret_cast<double*>(smem_raw);
  double* L = W + W_DOUBLES;                       // landing area, later the flux differences
  uint64_t* bar = reinterpret_cast<uint64_t*>(L + DF_DOUBLES);
  int* fsrc = reinterpret_cast<int*>(bar + 2);     // halo source of the 6 faces

  const int tid = threadIdx.x;
  const int last = p.first + p.count;
  const int stride = gridDim.x;
  int blk = p.first + blockIdx.x;
  const uint32_t bar_a = smem_u32(bar);
  if (tid == 0) {
    mbar_init(bar_a, 1);
    fence_mbar_init();
    issue_predictor_loads(tm, p, blk, L, fsrc, bar_a);
    if (blk + stride < last) prefetch_l2(p.Usrc + size_t(blk + stride) * BLK, BLK * 8);
  }
  __syncthreads();
  const double gamma = p.gamma, gm1 = p.gamma - 1.0, igm1 = 1.0 / gm1;
  const double dt = p.dt_dev ? *p.dt_dev : p.dt;
  const double lam = 0.5 * dt / p.h;
  const int pen = tid & 63, pa = pen & 7, pb = pen >> 3, D = tid >> 6;
  uint32_t parity = 0;

  for (; blk < last; blk += stride) {
    mbar_wait(bar_a, parity);
    parity ^= 1;
    convert_block<0>(L, W, fsrc, gamma, gm1, tid);
    __syncthreads();
    walk_predictor(W, L, D, pa, pb, igm1);
    double un[CR][NV];
    load_un(p.Un + size_t(blk) * BLK, tid, un);   // in flight while the other walkers finish
    __syncthreads();
    update_block<true>(L, un, lam, gm1, p.Udst + size_t(blk) * BLK, tid);
    __syncthreads();                              // the landing area is free again
    if (tid == 0 && blk + stride < last) {
      issue_predictor_loads(tm, p, blk + stride, L, fsrc, bar_a);
      if (blk + 2 * stride < last) prefetch_l2(p.Usrc + size_t(blk + 2 * stride) * BLK, BLK * 8);
    }
  }
}

// ---- corrector: stage W^{n+1/2} (primitives) -> walks -> update with U^n, stores U^{n+1} ------------
// fsrc[6] = 1 if any face of the block is an outflow face
__device__ __forceinline__ void issue_corrector_loads(const TensorMaps& tm, const StageParams& p, int blk, double* Wl,
                                                      int* fsrc, uint32_t bar_a) {
  int s[6];
#pragma unroll
  for (int f = 0; f < 6; ++f) s[f] = p.face_src[blk * 6 + f];
  uint32_t bytes = BLK * 8;
  int any_out = 0;
#pragma unroll
  for (int f = 0; f < 6; ++f) {
    fsrc[f] = s[f];
    bytes += (s[f] != SRC_OUTFLOW) ? SLAB * 8 : 0;
    any_out |= s[f] == SRC_OUTFLOW;
  }
  fsrc[6] = any_out;
  mbar_expect_tx(bar_a, bytes);           // (release: publishes fsrc to the threads that see the phase complete)
#pragma unroll
  for (int kk = 0; kk < 4; ++kk)          // interior: 4 z-plane pairs
    tensor4_g2s(smem_u32(Wl + C_ZCOL + (1 + kk) * SLAB), &tm.zs, 0, 0, 2 * kk, blk * NV, bar_a);
#pragma unroll
  for (int f = 0; f < 6; ++f) {
    const int axis = f >> 1, side = f & 1;
    const uint32_t dst = smem_u32(Wl + (axis == 2 ? C_ZCOL + side * 5 * SLAB : axis == 0 ? C_XLO + side * SLAB
                                                                                           : C_YLO + side * SLAB));
    if (s[f] >= 0) {
      const int lo = side ? 0 : N - NG;
      if (axis == 2) tensor4_g2s(dst, &tm.zs, 0, 0, lo, s[f] * NV, bar_a);
      else tensor4_g2s(dst, &tm.ax[axis], axis == 0 ? lo : 0, axis == 1 ? lo : 0, 0, s[f] * NV, bar_a);
    } else if (s[f] <= -2) {
      bulk_g2s(dst, p.ghost + size_t(-2 - s[f]) * SLAB, SLAB * 8, bar_a);   // z slabs come pre-swizzled
    }
  }
}

// halo of an outflow face (reading R1): copies of the block's own edge layer
__device__ __forceinline__ void fill_outflow_slabs(double* __restrict__ Wl, const int* __restrict__ fsrc, int tid) {
#pragma unroll 1
  for (int q = tid; q < 6 * CVS; q += STAGE_THREADS) {
    const int f = q >> 7, r = q & 127, axis = f >> 1, side = f & 1;
    if (fsrc[f] != SRC_OUTFLOW) continue;
    const int t = r & 63, ta = t & 7, tb = t >> 3, ll = r >> 6, edge = side ? N - 1 : 0;
    int src, dst;
    if (axis == 0) { src = c_pos_zcol(edge, ta, tb); dst = (side ? C_XHI : C_XLO) + t * 2 + ll; }
    else if (axis == 1) { src = c_pos_zcol(ta, edge, tb); dst = (side ? C_YHI : C_YLO) + tb * 16 + ll * 8 + ta; }
    else { src = c_pos_zcol(ta, tb, edge); dst = C_ZCOL + side * 5 * SLAB + zs_pos(ll, tb, ta); }
#pragma unroll
    for (int v = 0; v < NV; ++v) Wl[dst + v * CVS] = Wl[src + v * CVS];
  }
}

__global__ void __launch_bounds__(STAGE_THREADS, 2)
corrector_kernel(const __grid_constant__ TensorMaps tm, const StageParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  // staged primitives, 1024-byte aligned (swizzle atoms)
  double* Wl = reinterpret_cast<double*>(smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u));
  double* dF = Wl + C_LAND;
  uint64_t* bar = reinterpret_cast<uint64_t*>(dF + DF_DOUBLES);
  int* fsrc = reinterpret_cast<int*>(bar + 2);

  const int tid = threadIdx.x;
  const int last = p.first + p.count;
  const int stride = gridDim.x;
  int blk = p.first + blockIdx.x;
  const uint32_t bar_a = smem_u32(bar);
  if (tid == 0) {
    mbar_init(bar_a, 1);
    fence_mbar_init();
    issue_corrector_loads(tm, p, blk, Wl, fsrc, bar_a);
    prefetch_l2(p.Un + size_t(blk) * BLK, BLK * 8);
    if (blk + stride < last) {
      prefetch_l2(p.Usrc + size_t(blk + stride) * BLK, BLK * 8);
      prefetch_l2(p.Un + size_t(blk + stride) * BLK, BLK * 8);
    }
  }
  __syncthreads();
  const double gamma = p.gamma, gm1 = p.gamma - 1.0, igm1 = 1.0 / gm1;
  const double dt = p.dt_dev ? *p.dt_dev : p.dt;
  const double lam = dt / p.h;
  const int pen = tid & 63, pa = pen & 7, pb = pen >> 3, D = tid >> 6;
  uint32_t parity = 0;

  for (; blk < last; blk += stride) {
    mbar_wait(bar_a, parity);
    parity ^= 1;
    if (fsrc[6]) {                                // block-uniform
      fill_outflow_slabs(Wl, fsrc, tid);
      __syncthreads();
    }
    if (D == 0) walk_corrector<0>(Wl, dF, pa, pb, gamma, igm1, p, blk, dt);
    else if (D == 1) walk_corrector<1>(Wl, dF, pa, pb, gamma, igm1, p, blk, dt);
    else walk_corrector<2>(Wl, dF, pa, pb, gamma, igm1, p, blk, dt);
    double un[CR][NV];
    load_un(p.Un + size_t(blk) * BLK, tid, un);   // in flight while the other walkers finish
    __syncthreads();                              // the staged primitives are dead, the flux differences complete
    if (tid == 0 && blk + stride < last) {        // the next block lands while this one is updated
      if (fsrc[6]) fence_proxy_async();           // outflow slabs were written through the generic proxy
      issue_corrector_loads(tm, p, blk + stride, Wl, fsrc, bar_a);
      if (blk + 2 * stride < last) {
        prefetch_l2(p.Usrc + size_t(blk + 2 * stride) * BLK, BLK * 8);
        prefetch_l2(p.Un + size_t(blk + 2 * stride) * BLK, BLK * 8);
      }
    }
    update_block<false>(dF, un, lam, gm1, p.Udst + size_t(blk) * BLK, tid);
    __syncthreads();                              // the flux differences are consumed
  }
}

static_assert(WLayout<1, 7>::TOTAL <= W_DOUBLES, "primitive array too small");
static_assert(LAND_DOUBLES <= DF_DOUBLES, "landing area must fit in the flux-difference area");
static_assert((W_DOUBLES * 8) % 128 == 0 && (SLAB * 8) % 1024 == 0 && (BLK * 8) % 128 == 0,
              "TMA destinations: 128 B, swizzled tiles 1024 B");

static int g_stage_ctas = 2 * 148;   // persistent grid: resident CTAs per SM x SMs (set by configure_kernels)

cudaError_t configure_kernels() {
  cudaError_t e = cudaFuncSetAttribute(predictor_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGE_SMEM);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(corrector_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, CORR_SMEM);
  if (e != cudaSuccess) return e;
  cudaFuncSetAttribute(predictor_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
  cudaFuncSetAttribute(corrector_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
  int dev = 0, sms = 0, per_sm = 0;
  if (cudaGetDevice(&dev) == cudaSuccess &&
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0) {
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, predictor_kernel, STAGE_THREADS, STAGE_SMEM) !=
            cudaSuccess || per_sm < 1)
      per_sm = 1;
    g_stage_ctas = sms * per_sm;
  }
  return cudaSuccess;
}

cudaError_t launch_stage(int stage, const TensorMaps& tm, const StageParams& p, cudaStream_t st) {
  if (p.count <= 0) return cudaSuccess;
  const int grid = p.count < g_stage_ctas ? p.count : g_stage_ctas;
  if (stage == 0) predictor_kernel<<<grid, STAGE_THREADS, STAGE_SMEM, st>>>(tm, p);
  else corrector_kernel<<<grid, STAGE_THREADS, CORR_SMEM, st>>>(tm, p);
  return cudaGetLastError();
}

}  // namespace sfh

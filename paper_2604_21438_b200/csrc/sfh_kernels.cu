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
constexpr int W_DOUBLES = 6720;               // max over stages of the primitive array
constexpr int STAGE_SMEM = (W_DOUBLES + DF_DOUBLES) * 8 + 16 + 32;   // 115248 B (+1 KB reserved) -> 2 CTAs per SM

// Primitive-array layout for a stage with H halo layers and NVW stored variables.
template <int H, int NVW>
struct WLayout {
  static constexpr int RS = N + 2 * H + 1;          // x-row stride (odd: conflict-free x pencils)
  static constexpr int XV = 64 * RS;                // variable stride of the x-row array
  static constexpr int X0 = 0;
  static constexpr int YV = N * H * N;              // variable stride of a y slab [k][h][i]
  static constexpr int Y0 = NVW * XV;               // two y slabs (low, high)
  static constexpr int ZV = H * N * N;              // z slab [h][j][i]
  static constexpr int Z0 = Y0 + 2 * NVW * YV;
  static constexpr int TOTAL = Z0 + 2 * NVW * ZV;
  // offset of variable 0 and variable stride of the cell at position c in [-H, 8+H) along axis D
  // of the pencil (a, b) = the two other axes in increasing order
  template <int D>
  __device__ static __forceinline__ int off(int c, int a, int b) {
    if (D == 0) return X0 + (b * 8 + a) * RS + c + H;
    if (D == 1) {
      if (c < 0) return Y0 + (b * H + (c + H)) * 8 + a;
      if (c >= N) return Y0 + NVW * YV + (b * H + (c - N)) * 8 + a;
      return X0 + (b * 8 + c) * RS + a + H;
    }
    if (c < 0) return Z0 + ((c + H) * 8 + b) * 8 + a;
    if (c >= N) return Z0 + NVW * ZV + ((c - N) * 8 + b) * 8 + a;
    return X0 + (c * 8 + b) * RS + a + H;
  }
  template <int D>
  __device__ static __forceinline__ int vs(int c) {
    if (D == 0) return XV;
    if (D == 1) return (c < 0 || c >= N) ? YV : XV;
    return (c < 0 || c >= N) ? ZV : XV;
  }
};

// ---- conversion of the staged conserved cells to primitives --------------------------------------
template <int STAGE>
__device__ __forceinline__ void convert_block(const double* __restrict__ L, double* __restrict__ W,
                                              const int* __restrict__ fsrc, double gamma, double gm1, int tid) {
  constexpr int H = STAGE == 0 ? 1 : 2;
  constexpr int NVW = STAGE == 0 ? 7 : 5;
  using WL = WLayout<H, NVW>;
  for (int idx = tid; idx < NC + 6 * NG * FACE; idx += STAGE_THREADS) {
    int src, svs, dst, dvs;
    if (idx < NC) {
      const int i = idx & 7, j = (idx >> 3) & 7, k = idx >> 6;
      src = LAND_INT + idx; svs = NC;
      dst = WL::X0 + (k * 8 + j) * WL::RS + i + H; dvs = WL::XV;
    } else {
      const int q = idx - NC, f = q >> 7, r = q & 127, axis = f >> 1, side = f & 1;
      const bool outflow = fsrc[f] == SRC_OUTFLOW;
      const int edge = side ? 7 : 0;
      int ll;
      if (axis == 0) {
        ll = r & 1;
        const int j = (r >> 1) & 7, k = r >> 4;
        const int c = side ? N + ll : ll - NG;
        if (c < -H || c >= N + H) continue;
        src = outflow ? LAND_INT + k * 64 + j * 8 + edge : LAND_HALO + f * SLAB + r;
        dst = WL::X0 + (k * 8 + j) * WL::RS + c + H; dvs = WL::XV;
      } else if (axis == 1) {
        const int i = r & 7, k = r >> 4;
        ll = (r >> 3) & 1;
        const int c = side ? N + ll : ll - NG;
        if (c < -H || c >= N + H) continue;
        const int hh = side ? c - N : c + H;
        src = outflow ? LAND_INT + k * 64 + edge * 8 + i : LAND_HALO + f * SLAB + r;
        dst = WL::Y0 + side * NVW * WL::YV + (k * H + hh) * 8 + i; dvs = WL::YV;
      } else {
        const int i = r & 7, j = (r >> 3) & 7;
        ll = r >> 6;
        const int c = side ? N + ll : ll - NG;
        if (c < -H || c >= N + H) continue;
        const int hh = side ? c - N : c + H;
        src = outflow ? LAND_INT + edge * 64 + j * 8 + i : LAND_HALO + f * SLAB + r;
        dst = WL::Z0 + side * NVW * WL::ZV + (hh * 8 + j) * 8 + i; dvs = WL::ZV;
      }
      svs = outflow ? NC : NG * FACE;
    }
    double u[5], w[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) u[v] = L[src + v * svs];
    const double ir = cons_to_prim(u, gm1, w);
#pragma unroll
    for (int v = 0; v < 5; ++v) W[dst + v * dvs] = w[v];
    if (STAGE == 0) {
      const double c2 = (gamma * w[4]) * ir;         // c_s^2 = gamma P / rho
      W[dst + 5 * dvs] = c2 * rsqrt(c2);
      W[dst + 6 * dvs] = u[4];                       // total energy of the cell (eq. 8)
    }
  }
}

// ---- pencil walks ----------------------------------------------------------------------------------
// One thread per pencil; 64 pencils per axis; the three axes run side by side in different warps but
// through the SAME rolled loop (runtime strides), so the instruction footprint is one flux body per
// stage.  Face f = 0..8 of a pencil lies between cells f-1 and f; each flux is computed once and used
// by both adjacent cells (the paper's mapping).
template <int H, int NVW>
struct Pencil {
  using WL = WLayout<H, NVW>;
  int lo0, lo_cs, lo_vs;   // cells c < 0:   offset lo0 + (c + H) * lo_cs, variable stride lo_vs
  int mid0, mid_cs;        // cells 0..7:    offset mid0 + c * mid_cs,     variable stride XV
  int hi0, hi_cs, hi_vs;   // cells c >= 8:  offset hi0 + (c - 8) * hi_cs
  int vn, vt1, vt2;        // variable slots of the normal / tangential velocities (momenta)
  int df0, df_cs, df_swz;  // flux-difference index of cell c: df0 + ((c ^ df_swz) * df_cs)
  __device__ __forceinline__ Pencil(int D, int a, int b) {
    vn = 1 + D; vt1 = 1 + (D + 1) % 3; vt2 = 1 + (D + 2) % 3;
    if (D == 0) {
      lo0 = (b * 8 + a) * WL::RS; lo_cs = 1; lo_vs = WL::XV;
      mid0 = lo0 + H; mid_cs = 1;
      hi0 = mid0 + N; hi_cs = 1; hi_vs = WL::XV;
      df0 = (b * 8 + a) * 8; df_cs = 1; df_swz = a;      // x rows are XOR swizzled (bank spread)
    } else if (D == 1) {
      lo0 = WL::Y0 + b * H * 8 + a; lo_cs = 8; lo_vs = WL::YV;
      mid0 = b * 8 * WL::RS + a + H; mid_cs = WL::RS;
      hi0 = lo0 + NVW * WL::YV; hi_cs = 8; hi_vs = WL::YV;
      df0 = D * BLK + b * 64 + a; df_cs = 8; df_swz = 0;
    } else {
      lo0 = WL::Z0 + b * 8 + a; lo_cs = 64; lo_vs = WL::ZV;
      mid0 = b * WL::RS + a + H; mid_cs = 8 * WL::RS;
      hi0 = lo0 + NVW * WL::ZV; hi_cs = 64; hi_vs = WL::ZV;
      df0 = D * BLK + b * 8 + a; df_cs = 64; df_swz = 0;
    }
  }
  // loads cell c >= 0 in the face frame (rho, normal v, tangential v's, P[, c_s])
  __device__ __forceinline__ void load(const double* __restrict__ W, int c, double w[NVW]) const {
    const bool hi = c >= N;
    const int o = hi ? hi0 + (c - N) * hi_cs : mid0 + c * mid_cs;
    const int s = hi ? hi_vs : WL::XV;
    w[0] = W[o]; w[1] = W[o + vn * s]; w[2] = W[o + vt1 * s]; w[3] = W[o + vt2 * s]; w[4] = W[o + 4 * s];
    if (NVW == 7) { w[5] = W[o + 5 * s]; w[NVW - 1] = W[o + 6 * s]; }
  }
  __device__ __forceinline__ void load_lo(const double* __restrict__ W, int c, double w[NVW]) const {
    const int o = lo0 + (c + H) * lo_cs, s = lo_vs;
    w[0] = W[o]; w[1] = W[o + vn * s]; w[2] = W[o + vt1 * s]; w[3] = W[o + vt2 * s]; w[4] = W[o + 4 * s];
    if (NVW == 7) { w[5] = W[o + 5 * s]; w[NVW - 1] = W[o + 6 * s]; }
  }
  // dF of cell c = F(face c+1) - F(face c), stored in the global variable order
  __device__ __forceinline__ void store_df(double* __restrict__ dF, int c, const double Fa[5], const double Fb[5]) const {
    const int ci = df0 + ((c ^ df_swz) * df_cs);
    dF[ci] = Fa[0] - Fb[0];
    dF[ci + vn * NC] = Fa[1] - Fb[1];
    dF[ci + vt1 * NC] = Fa[2] - Fb[2];
    dF[ci + vt2 * NC] = Fa[3] - Fb[3];
    dF[ci + 4 * NC] = Fa[4] - Fb[4];
  }
};

// flux registers at coarse-fine faces (a7; reading R14); Fn in the face frame
__device__ __forceinline__ void store_regs(const StageParams& p, int blk, int D, int side, int t, int vn, int vt1,
                                           int vt2, const double Fn[5], double dt) {
  const int f = 2 * D + side;
  const int src = p.face_src[blk * 6 + f];
  const int fs = p.fslot[blk * 6 + f];
  if (src <= -2) {   // fine side of a coarse-fine face: accumulate dt * F
    double* r = p.R + size_t(-2 - src) * REG + t;
    r[0] += dt * Fn[0]; r[vn * FACE] += dt * Fn[1]; r[vt1 * FACE] += dt * Fn[2]; r[vt2 * FACE] += dt * Fn[3];
    r[4 * FACE] += dt * Fn[4];
  }
  if (fs >= 0) {     // coarse leaf next to a covered block: keep its own flux
    double* r = p.FH + size_t(fs) * REG + t;
    r[0] = Fn[0]; r[vn * FACE] = Fn[1]; r[vt1 * FACE] = Fn[2]; r[vt2 * FACE] = Fn[3]; r[4 * FACE] = Fn[4];
  }
}

__device__ __forceinline__ void walk_predictor(const double* __restrict__ W, double* __restrict__ dF, int D, int a, int b,
                                               double igm1) {
  const Pencil<1, 7> pc(D, a, b);
  double wl[7], Fp[5];
  pc.load_lo(W, -1, wl);
#pragma unroll 1
  for (int f = 0; f <= N; ++f) {
    double wr[7], Fn[5];
    pc.load(W, f, wr);
    hllc_flux<true>(wl[0], wl[1], wl[2], wl[3], wl[4], wl[5], wl[6], wr[0], wr[1], wr[2], wr[3], wr[4], wr[5], wr[6],
                    igm1, Fn);
    if (f > 0) pc.store_df(dF, f - 1, Fn, Fp);
#pragma unroll
    for (int v = 0; v < 5; ++v) Fp[v] = Fn[v];
#pragma unroll
    for (int v = 0; v < 7; ++v) wl[v] = wr[v];
  }
}

__device__ __forceinline__ void walk_corrector(const double* __restrict__ W, double* __restrict__ dF, int D, int a, int b,
                                               double gamma, double igm1, const StageParams& p, int blk, double dt) {
  const Pencil<2, 5> pc(D, a, b);
  // cells -2, -1: the left face state of face 0 needs the slope of cell -1
  double wm[5], wc[5], dm[5], WLs[5], Fp[5];
  pc.load_lo(W, -2, wm);
  pc.load_lo(W, -1, wc);
#pragma unroll
  for (int v = 0; v < 5; ++v) { dm[v] = wc[v] - wm[v]; WLs[v] = 0.0; Fp[v] = 0.0; }
  // invariant at the top of iteration c (c = 0..9): wc = W_{c-1}, dm = W_{c-1} - W_{c-2};
  // for c >= 1, WLs = left state of face c-1 (= W_{c-2} + slope_{c-2}/2)
#pragma unroll 1
  for (int c = 0; c <= N + 1; ++c) {
    double wn[5], dn[5], sl[5];
    pc.load(W, c, wn);
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      dn[v] = wn[v] - wc[v];
      sl[v] = minmod(dn[v], dm[v]);      // slope of cell c-1 (reading R12), primitives (R11)
    }
    if (c >= 1) {
      // face f = c-1 between cells c-2 and c-1: right state from cell c-1
      double WRs[5], Fn[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) WRs[v] = wc[v] - 0.5 * sl[v];
      const double cL = sound_speed(gamma, WLs[4], WLs[0]);
      const double cR = sound_speed(gamma, WRs[4], WRs[0]);
      hllc_flux<false>(WLs[0], WLs[1], WLs[2], WLs[3], WLs[4], cL, 0.0, WRs[0], WRs[1], WRs[2], WRs[3], WRs[4], cR, 0.0,
                       igm1, Fn);
      const int f = c - 1;
      if (f > 0) pc.store_df(dF, f - 1, Fn, Fp);
      if (p.use_regs && (f == 0 || f == N)) store_regs(p, blk, D, f == N, b * 8 + a, pc.vn, pc.vt1, pc.vt2, Fn, dt);
#pragma unroll
      for (int v = 0; v < 5; ++v) Fp[v] = Fn[v];
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      WLs[v] = wc[v] + 0.5 * sl[v];      // left state of face c
      wc[v] = wn[v];
      dm[v] = dn[v];
    }
  }
}

// ---- the stage kernel --------------------------------------------------------------------------------
template <int STAGE>
__global__ void __launch_bounds__(STAGE_THREADS, 2)
stage_kernel(const __grid_constant__ TensorMaps tm, const StageParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* W = reinterpret_cast<double*>(smem_raw);
  double* L = W + W_DOUBLES;                       // landing area, later the flux differences
  uint64_t* bar = reinterpret_cast<uint64_t*>(L + DF_DOUBLES);
  int* fsrc = reinterpret_cast<int*>(bar + 2);     // halo source of the 6 faces

  const int tid = threadIdx.x;
  const int blk = p.first + blockIdx.x;
  const uint32_t bar_a = smem_u32(bar);
  if (tid < 6) fsrc[tid] = p.face_src[blk * 6 + tid];
  if (tid == 0) {
    mbar_init(bar_a, 1);
    fence_mbar_init();
  }
  __syncthreads();
  if (tid == 0) {
    uint32_t bytes = BLK * 8;
#pragma unroll
    for (int f = 0; f < 6; ++f) bytes += (fsrc[f] != SRC_OUTFLOW) ? SLAB * 8 : 0;
    mbar_expect_tx(bar_a, bytes);
    bulk_g2s(smem_u32(L + LAND_INT), p.Usrc + size_t(blk) * BLK, BLK * 8, bar_a);
#pragma unroll
    for (int f = 0; f < 6; ++f) {
      const int s = fsrc[f];
      const uint32_t dst = smem_u32(L + LAND_HALO + f * SLAB);
      if (s >= 0) {
        // my low-side ghost layers are the neighbour's two highest layers, and vice versa
        const int axis = f >> 1, lo = (f & 1) ? 0 : N - NG;
        tensor4_g2s(dst, &tm.ax[axis], axis == 0 ? lo : 0, axis == 1 ? lo : 0, axis == 2 ? lo : 0, s * NV, bar_a);
      } else if (s <= -2) {
        bulk_g2s(dst, p.ghost + size_t(-2 - s) * SLAB, SLAB * 8, bar_a);
      }
    }
    // U^n of this block is read again in the update at the end: pull it towards L2 now
    if (STAGE == 1) prefetch_l2(p.Un + size_t(blk) * BLK, BLK * 8);
  }
  const double gamma = p.gamma, gm1 = p.gamma - 1.0, igm1 = __drcp_rn(gm1);
  const double dt = p.dt_dev ? *p.dt_dev : p.dt;
  mbar_wait(bar_a, 0);

  convert_block<STAGE>(L, W, fsrc, gamma, gm1, tid);
  __syncthreads();

  {
    const int pen = tid & 63, a = pen & 7, b = pen >> 3, D = tid >> 6;
    if (STAGE == 0) walk_predictor(W, L, D, a, b, igm1);
    else walk_corrector(W, L, D, a, b, gamma, igm1, p, blk, dt);
  }
  __syncthreads();

  // U_out = U^n - lambda ((dFx + dFy) + dFz), lambda = dt/(2h) (predictor) or dt/h (corrector)
  const double lam = (STAGE == 0 ? 0.5 * dt : dt) / p.h;
  const double* __restrict__ Un = p.Un + size_t(blk) * BLK;
  double* __restrict__ Uo = p.Udst + size_t(blk) * BLK;
  constexpr int ROUNDS = (BLK + STAGE_THREADS - 1) / STAGE_THREADS;
  double un[ROUNDS];
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r) {          // all loads in flight before the first use
    const int idx = tid + r * STAGE_THREADS;
    un[r] = idx < BLK ? Un[idx] : 0.0;
  }
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r) {
    const int idx = tid + r * STAGE_THREADS;
    if (idx < BLK) {
      const int cell = idx & (NC - 1), v = idx >> 9, row = cell >> 3, i = cell & 7;
      const double dfx = L[v * NC + row * 8 + (i ^ (row & 7))];
      const double sum = (dfx + L[BLK + idx]) + L[2 * BLK + idx];
      Uo[idx] = un[r] - lam * sum;
    }
  }
}

static_assert(WLayout<2, 5>::TOTAL <= W_DOUBLES && WLayout<1, 7>::TOTAL <= W_DOUBLES, "primitive array too small");
static_assert(LAND_DOUBLES <= DF_DOUBLES, "landing area must fit in the flux-difference area");
static_assert((W_DOUBLES * 8) % 128 == 0 && (SLAB * 8) % 128 == 0 && (BLK * 8) % 128 == 0, "TMA destinations: 128 B");

cudaError_t configure_kernels() {
  cudaError_t e = cudaFuncSetAttribute(stage_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGE_SMEM);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(stage_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGE_SMEM);
  if (e != cudaSuccess) return e;
  cudaFuncSetAttribute(stage_kernel<0>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
  cudaFuncSetAttribute(stage_kernel<1>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
  return cudaSuccess;
}

cudaError_t launch_stage(int stage, const TensorMaps& tm, const StageParams& p, cudaStream_t st) {
  if (p.count <= 0) return cudaSuccess;
  if (stage == 0) stage_kernel<0><<<p.count, STAGE_THREADS, STAGE_SMEM, st>>>(tm, p);
  else stage_kernel<1><<<p.count, STAGE_THREADS, STAGE_SMEM, st>>>(tm, p);
  return cudaGetLastError();
}

}  // namespace sfh

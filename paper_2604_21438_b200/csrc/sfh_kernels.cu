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

// index of cell (position c along D, pencil (a,b)) in a flux-difference array; x rows are XOR
// swizzled so that the x walkers' stores spread over the banks
template <int D>
__device__ __forceinline__ int df_index(int c, int a, int b) {
  if (D == 0) return (b * 8 + a) * 8 + (c ^ a);
  if (D == 1) return b * 64 + c * 8 + a;
  return c * 64 + b * 8 + a;
}

// ---- conversion of the staged conserved cells to primitives --------------------------------------
template <int STAGE>
__device__ __forceinline__ void convert_block(const double* __restrict__ L, double* __restrict__ W,
                                              const int* __restrict__ fsrc, double gamma, double gm1, int tid) {
  constexpr int H = STAGE == 0 ? 1 : 2;
  constexpr int NVW = STAGE == 0 ? 6 : 5;
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
    cons_to_prim(u, gm1, w);
#pragma unroll
    for (int v = 0; v < 5; ++v) W[dst + v * dvs] = w[v];
    if (STAGE == 0) W[dst + 5 * dvs] = sound_speed(gamma, w[4], w[0]);
  }
}

// ---- pencil walks ----------------------------------------------------------------------------------
// Face f = 0..8 of a pencil lies between cells f-1 and f.  Flux components are returned in the
// global variable order; n, t1, t2 = normal and tangential momentum slots as in F[1+D], ...
template <int D>
__device__ __forceinline__ void store_regs(const StageParams& p, int blk, int side, int a, int b, const double F[5],
                                           double dt) {
  const int f = 2 * D + side;
  const int src = p.face_src[blk * 6 + f];
  const int fs = p.fslot[blk * 6 + f];
  const int t = b * 8 + a;
  if (src <= -2) {   // fine side of a coarse-fine face: accumulate dt * F (reading R14)
    double* r = p.R + size_t(-2 - src) * REG + t;
#pragma unroll
    for (int v = 0; v < 5; ++v) r[v * FACE] += dt * F[v];
  }
  if (fs >= 0) {     // coarse leaf next to a covered block: keep its own flux
    double* r = p.FH + size_t(fs) * REG + t;
#pragma unroll
    for (int v = 0; v < 5; ++v) r[v * FACE] = F[v];
  }
}

template <int D>
__device__ __forceinline__ void walk_predictor(const double* __restrict__ W, double* __restrict__ dF, int a, int b,
                                               double gm1) {
  using WL = WLayout<1, 6>;
  constexpr int n = 1 + D, t1 = 1 + (D + 1) % 3, t2 = 1 + (D + 2) % 3;
  double wl[6], Fp[5];
  {
    const int o = WL::template off<D>(-1, a, b), s = WL::template vs<D>(-1);
#pragma unroll
    for (int v = 0; v < 6; ++v) wl[v] = W[o + v * s];
  }
#pragma unroll
  for (int f = 0; f <= N; ++f) {
    double wr[6], Fn[5], F[5];
    const int o = WL::template off<D>(f, a, b), s = WL::template vs<D>(f);
#pragma unroll
    for (int v = 0; v < 6; ++v) wr[v] = W[o + v * s];
    hllc_flux(wl[0], wl[n], wl[t1], wl[t2], wl[4], wl[5], wr[0], wr[n], wr[t1], wr[t2], wr[4], wr[5], gm1, Fn);
    F[0] = Fn[0]; F[n] = Fn[1]; F[t1] = Fn[2]; F[t2] = Fn[3]; F[4] = Fn[4];
    if (f > 0) {
      const int ci = df_index<D>(f - 1, a, b);
#pragma unroll
      for (int v = 0; v < 5; ++v) dF[D * BLK + v * NC + ci] = F[v] - Fp[v];
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) Fp[v] = F[v];
#pragma unroll
    for (int v = 0; v < 6; ++v) wl[v] = wr[v];
  }
}

template <int D>
__device__ __forceinline__ void walk_corrector(const double* __restrict__ W, double* __restrict__ dF, int a, int b,
                                               double gamma, double gm1, const StageParams& p, int blk, double dt) {
  using WL = WLayout<2, 5>;
  constexpr int n = 1 + D, t1 = 1 + (D + 1) % 3, t2 = 1 + (D + 2) % 3;
  // cells -2, -1: difference and the left face state of face 0 need the slope of cell -1
  double wm[5], wc[5], dm[5], WLs[5], Fp[5];
  {
    const int o0 = WL::template off<D>(-2, a, b), s0 = WL::template vs<D>(-2);
    const int o1 = WL::template off<D>(-1, a, b), s1 = WL::template vs<D>(-1);
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      wm[v] = W[o0 + v * s0];
      wc[v] = W[o1 + v * s1];
      dm[v] = wc[v] - wm[v];
    }
  }
  // invariant at the top of iteration c (c = 0..9): wc = W_{c-1}, dm = W_{c-1} - W_{c-2};
  // for c >= 1, WLs = left state of face c-1 (= W_{c-2} + slope_{c-2}/2)
#pragma unroll
  for (int c = 0; c <= N + 1; ++c) {
    double wn[5], dn[5], sl[5];
    const int o = WL::template off<D>(c, a, b), s = WL::template vs<D>(c);
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      wn[v] = W[o + v * s];
      dn[v] = wn[v] - wc[v];
      sl[v] = minmod(dn[v], dm[v]);      // slope of cell c-1 (reading R12), primitives (R11)
    }
    if (c >= 1) {
      // face f = c-1 between cells c-2 and c-1: right state from cell c-1
      double WRs[5], Fn[5], F[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) WRs[v] = wc[v] - 0.5 * sl[v];
      const double cL = sound_speed(gamma, WLs[4], WLs[0]);
      const double cR = sound_speed(gamma, WRs[4], WRs[0]);
      hllc_flux(WLs[0], WLs[n], WLs[t1], WLs[t2], WLs[4], cL, WRs[0], WRs[n], WRs[t1], WRs[t2], WRs[4], cR, gm1, Fn);
      F[0] = Fn[0]; F[n] = Fn[1]; F[t1] = Fn[2]; F[t2] = Fn[3]; F[4] = Fn[4];
      const int f = c - 1;
      if (f > 0) {
        const int ci = df_index<D>(f - 1, a, b);
#pragma unroll
        for (int v = 0; v < 5; ++v) dF[D * BLK + v * NC + ci] = F[v] - Fp[v];
      }
      if (p.use_regs && (f == 0 || f == N)) store_regs<D>(p, blk, f == N, a, b, F, dt);
#pragma unroll
      for (int v = 0; v < 5; ++v) Fp[v] = F[v];
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
  }
  const double gamma = p.gamma, gm1 = p.gamma - 1.0;
  const double dt = p.dt_dev ? *p.dt_dev : p.dt;
  mbar_wait(bar_a, 0);

  convert_block<STAGE>(L, W, fsrc, gamma, gm1, tid);
  __syncthreads();

  {
    const int pen = tid & 63, a = pen & 7, b = pen >> 3, D = tid >> 6;
    if (STAGE == 0) {
      if (D == 0) walk_predictor<0>(W, L, a, b, gm1);
      else if (D == 1) walk_predictor<1>(W, L, a, b, gm1);
      else walk_predictor<2>(W, L, a, b, gm1);
    } else {
      if (D == 0) walk_corrector<0>(W, L, a, b, gamma, gm1, p, blk, dt);
      else if (D == 1) walk_corrector<1>(W, L, a, b, gamma, gm1, p, blk, dt);
      else walk_corrector<2>(W, L, a, b, gamma, gm1, p, blk, dt);
    }
  }
  __syncthreads();

  // U_out = U^n - lambda ((dFx + dFy) + dFz), lambda = dt/(2h) (predictor) or dt/h (corrector)
  const double lam = (STAGE == 0 ? 0.5 * dt : dt) / p.h;
  const double* __restrict__ Un = p.Un + size_t(blk) * BLK;
  double* __restrict__ Uo = p.Udst + size_t(blk) * BLK;
  for (int idx = tid; idx < BLK; idx += STAGE_THREADS) {
    const int cell = idx & (NC - 1), v = idx >> 9, row = cell >> 3, i = cell & 7;
    const double dfx = L[v * NC + row * 8 + (i ^ (row & 7))];
    const double sum = (dfx + L[BLK + idx]) + L[2 * BLK + idx];
    Uo[idx] = Un[idx] - lam * sum;
  }
}

static_assert(WLayout<2, 5>::TOTAL <= W_DOUBLES && WLayout<1, 6>::TOTAL <= W_DOUBLES, "primitive array too small");
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

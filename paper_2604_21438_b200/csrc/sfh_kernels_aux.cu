// sfh_kernels_aux.cu — the smaller kernels of libsfh (sm_100a): coarse-fine ghost prolongation (a3),
// restriction (a8), reflux (a9), CFL reduction (a10), status, layout permutation, ghosted export.
#include <cmath>

#include "sfh_device.cuh"
#include "sfh_kernels.cuh"

namespace sfh {

// maximum over the CTA (NW warps); the result is valid in thread 0.  wm: NW doubles of shared memory
template <int NW>
__device__ __forceinline__ double cta_max(double x, double* wm) {
  x = warp_max(x);
  if ((threadIdx.x & 31) == 0) wm[threadIdx.x >> 5] = x;
  __syncthreads();
  if (threadIdx.x < 32) {
    x = threadIdx.x < NW ? wm[threadIdx.x] : 0.0;
    x = warp_max(x);
  }
  return x;
}


// =====================================================================================================
// a3: ghost slabs of coarse-fine faces.  One CTA of 128 threads per slab (2 layers x 8 x 8 fine cells
// behind one coarse layer of 4 x 4 cells).  Step 1: the 68 coarse cells any of the 7-point stencils
// touches -- the coarse layer with a one-cell rim (6 x 6, corners unused) and the 4 x 4 cells on either
// side of it along the face normal -- are gathered once, interpolated in time (eq. 16) and, where the
// coarse copy holds primitives, converted back to conserved variables, into shared memory.  Step 2: one
// thread per fine ghost cell: minmod slopes of the coarse cell and the fine value
// Q + sum_d (+-1/4) slope_d (reading R3).
// =====================================================================================================
constexpr int PR_RIM = 36, PR_CELLS = PR_RIM + 2 * 16;   // [6 x 6 layer | 4 x 4 below | 4 x 4 above]

__global__ void __launch_bounds__(128) prolong_kernel(const ProlongParams p) {
  __shared__ double q[PR_CELLS][NV];
  __shared__ double q1[PR_CELLS][NV];      // dual fill: the same cells at tau1
  __shared__ int missing;
  const int slot = p.first + blockIdx.x;
  const int F = p.cf_block[slot], f = p.cf_face[slot], axis = f >> 1, side = f & 1;
  const int P = p.parent[F];
  const int t1ax = axis == 0 ? 1 : 0, t2ax = axis == 2 ? 1 : 2;    // the two in-face axes, lower first
  int oct[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) oct[d] = p.coord[3 * F + d] & 1;
  const int r = threadIdx.x;
  if (r == 0) missing = 0;
  __syncthreads();
  const double gm1 = p.gamma - 1.0, igm1 = 1.0 / gm1;

  // ---- step 1: thread r < 68 gathers coarse cell r of the stencil region
  if (r < PR_CELLS) {
    int ca, c1, c2;                       // offsets from (coarse layer, first coarse cell of the octant)
    bool needed = true;
    if (r < PR_RIM) {
      ca = 0; c1 = r % 6 - 1; c2 = r / 6 - 1;
      needed = !((c1 < 0 || c1 > 3) && (c2 < 0 || c2 > 3));
    } else {
      const int e = (r - PR_RIM) & 15;
      ca = r < PR_RIM + 16 ? -1 : 1; c1 = e & 3; c2 = e >> 2;
    }
    if (needed) {
      int c[3], rg[3];
      c[axis] = (side ? oct[axis] * 4 + 4 : oct[axis] * 4 - 1) + ca;
      c[t1ax] = oct[t1ax] * 4 + c1;
      c[t2ax] = oct[t2ax] * 4 + c2;
      const int32_t* nb = p.nbr27 + size_t(P) * 27;
      // does the parent touch an outflow boundary?  (face-region codes)
      const bool out_lo[3] = {nb[12] == NBR_OUTSIDE, nb[10] == NBR_OUTSIDE, nb[4] == NBR_OUTSIDE};
      const bool out_hi[3] = {nb[14] == NBR_OUTSIDE, nb[16] == NBR_OUTSIDE, nb[22] == NBR_OUTSIDE};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        rg[d] = 0;
        if (c[d] < 0) { if (out_lo[d]) c[d] = 0; else { rg[d] = -1; c[d] += N; } }
        else if (c[d] >= N) { if (out_hi[d]) c[d] = N - 1; else { rg[d] = 1; c[d] -= N; } }
      }
      const int Q = nb[(rg[2] + 1) * 9 + (rg[1] + 1) * 3 + (rg[0] + 1)];
      if (Q < 0) {
        missing = 1;                      // (a mesh sfh_create_mesh accepts never gets here)
      } else {
        const size_t o = size_t(Q) * BLK + (c[2] * 8 + c[1]) * 8 + c[0];
        double u0[NV], u1[NV], u2[NV], t[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) u0[v] = p.C0[o + v * NC];
        if (p.interp) {
#pragma unroll
          for (int v = 0; v < NV; ++v) { u1[v] = p.C1[o + v * NC]; u2[v] = p.C2[o + v * NC]; }
        }
        if (p.c0_prim) {
          prim_to_cons(u0, igm1, t);
#pragma unroll
          for (int v = 0; v < NV; ++v) u0[v] = t[v];
        }
        if (p.interp) {
          if (p.c1_prim) {
            prim_to_cons(u1, igm1, t);
#pragma unroll
            for (int v = 0; v < NV; ++v) u1[v] = t[v];
          }
          if (p.ghost1) {
#pragma unroll
            for (int v = 0; v < NV; ++v) q1[r][v] = time_interp(u0[v], u1[v], u2[v], p.tau1);
          }
#pragma unroll
          for (int v = 0; v < NV; ++v) u0[v] = time_interp(u0[v], u1[v], u2[v], p.tau);
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) q[r][v] = u0[v];
      }
    }
  }
  __syncthreads();

  // ---- step 2: thread r computes fine ghost cell r of the slab (slab layouts as staged by the stage kernels)
  int fc[3];
  if (axis == 0) {
    const int ll = r & 1;
    fc[0] = side ? N + ll : ll - NG; fc[1] = (r >> 1) & 7; fc[2] = r >> 4;
  } else if (axis == 1) {
    const int ll = (r >> 3) & 1;
    fc[0] = r & 7; fc[1] = side ? N + ll : ll - NG; fc[2] = r >> 4;
  } else {
    const int ll = r >> 6;
    fc[0] = r & 7; fc[1] = (r >> 3) & 7; fc[2] = side ? N + ll : ll - NG;
  }
  const int c1 = fc[t1ax] >> 1, c2 = fc[t2ax] >> 1;
  const int ctr = (c2 + 1) * 6 + (c1 + 1);
  int nbp[3], nbm[3];                     // stencil neighbours +d / -d, per axis d
  nbp[axis] = PR_RIM + 16 + c2 * 4 + c1; nbm[axis] = PR_RIM + c2 * 4 + c1;
  nbp[t1ax] = ctr + 1; nbm[t1ax] = ctr - 1;
  nbp[t2ax] = ctr + 6; nbm[t2ax] = ctr - 6;
  const int ll = fc[axis] < 0 ? fc[axis] + NG : fc[axis] - N;
  const int rout = slab_pos(axis, ll, fc[axis == 0 ? 1 : 0], fc[axis == 2 ? 1 : 2]);
  auto fine_value = [&](const double (*qq)[NV], bool prim, double* __restrict__ ghost) {
    double val[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const double q0 = qq[ctr][v];
      val[v] = q0;
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const double sig = (fc[d] & 1) ? 0.25 : -0.25;
        val[v] = val[v] + sig * minmod(qq[nbp[d]][v] - q0, q0 - qq[nbm[d]][v]);
      }
    }
    if (missing) {
#pragma unroll
      for (int v = 0; v < NV; ++v) val[v] = nan("");
    }
    if (prim) {               // the corrector stages primitives
      double w[NV];
      cons_to_prim(val, gm1, w);
#pragma unroll
      for (int v = 0; v < NV; ++v) val[v] = w[v];
    }
    // the slab is written in the staging layout of the stage kernels
    double* out = ghost + size_t(slot) * SLAB + rout;
#pragma unroll
    for (int v = 0; v < NV; ++v) out[v * NG * FACE] = val[v];
  };
  fine_value(q, p.out_prim != 0, p.ghost);
  if (p.ghost1) fine_value(q1, true, p.ghost1);
}

cudaError_t launch_prolong(const ProlongParams& p, cudaStream_t st) {
  if (p.count <= 0) return cudaSuccess;
  prolong_kernel<<<p.count, 128, 0, st>>>(p);
  return cudaGetLastError();
}

// =====================================================================================================
// a8: restriction.  One CTA per covered block, one thread per coarse cell: mean of the 8 fine cells
// in the fixed order cx fastest (reading R15).
// =====================================================================================================
__global__ void __launch_bounds__(NC) restrict_kernel(const double* __restrict__ Uf, double* __restrict__ Uc,
                                                      const int32_t* __restrict__ list,
                                                      const int32_t* __restrict__ child0, double gamma,
                                                      double* __restrict__ bmax) {
  const int b = list[blockIdx.x];
  const int t = threadIdx.x, i = t & 7, j = (t >> 3) & 7, k = t >> 6;
  const int child = child0[b] + (i >> 2) + 2 * (j >> 2) + 4 * (k >> 2);
  const int fi = 2 * (i & 3), fj = 2 * (j & 3), fk = 2 * (k & 3);
  const double* src = Uf + size_t(child) * BLK;
  double* dst = Uc + size_t(b) * BLK + t;
  double u[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    double sum = 0.0;
#pragma unroll
    for (int c = 0; c < 8; ++c)
      sum += src[v * NC + ((fk + ((c >> 2) & 1)) * 8 + fj + ((c >> 1) & 1)) * 8 + fi + (c & 1)];
    u[v] = 0.125 * sum;
    dst[v * NC] = u[v];
  }
  if (bmax) {                       // the block's cached maximum speed follows its new contents
    __shared__ double wm[NC / 32];
    const double s = cta_max<NC / 32>(cell_speed(u, gamma, gamma - 1.0), wm);
    if (t == 0) bmax[b] = s;
  }
}

cudaError_t launch_restrict(const double* Ufine, double* Ucoarse, const int32_t* list, const int32_t* child0, int count,
                            double gamma, double* bmax, cudaStream_t st) {
  if (count <= 0) return cudaSuccess;
  restrict_kernel<<<count, NC, 0, st>>>(Ufine, Ucoarse, list, child0, gamma, bmax);
  return cudaGetLastError();
}

// =====================================================================================================
// a9: reflux (Berger & Colella 1989 as cited).  One CTA of 64 threads per coarse
// leaf block that owns corrected faces; faces in the fixed order x-, x+, y-, y+, z-, z+, one thread per
// face cell, fine-face sum in fixed order: deterministic, no atomics.
// =====================================================================================================
__global__ void __launch_bounds__(FACE) reflux_kernel(double* __restrict__ U, const double* __restrict__ R,
                                                      const double* __restrict__ FH,
                                                      const int32_t* __restrict__ list,
                                                      const int32_t* __restrict__ fslot,
                                                      const int32_t* __restrict__ fh_src, double h, double dt_host,
                                                      const double* __restrict__ dt_dev, double gamma,
                                                      double* __restrict__ bmax) {
  const int b = list[blockIdx.x];
  const int t = threadIdx.x, ta = t & 7, tb = t >> 3;
  const double dt = dt_dev ? *dt_dev : dt_host;
  double* Ub = U + size_t(b) * BLK;
  for (int f = 0; f < 6; ++f) {
    const int fs = fslot[b * 6 + f];
    if (fs >= 0) {
      const int d = f >> 1, side = f & 1, c = side ? N - 1 : 0;
      const double s = side ? 1.0 : -1.0;
      const int cell = d == 0 ? (tb * 8 + ta) * 8 + c : d == 1 ? (tb * 8 + c) * 8 + ta : (c * 8 + tb) * 8 + ta;
      const int slot = fh_src[fs * 4 + (ta >> 2) + 2 * (tb >> 2)];
      const int fa = 2 * (ta & 3), fb = 2 * (tb & 3);
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const double* r = R + size_t(slot) * REG + v * FACE;
        double sumR = 0.0;
#pragma unroll
        for (int q = 0; q < 4; ++q) sumR += r[(fb + (q >> 1)) * 8 + fa + (q & 1)];
        const double FHv = FH[size_t(fs) * REG + v * FACE + t];
        Ub[v * NC + cell] = Ub[v * NC + cell] - (s / h) * (0.25 * sumR - dt * FHv);
      }
    }
    __syncthreads();
  }
  if (bmax) {                       // the block's cached maximum speed follows its corrected cells
    const double gm1 = gamma - 1.0;
    double smax = 0.0;
#pragma unroll
    for (int c = t; c < NC; c += FACE) {
      double u[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) u[v] = Ub[v * NC + c];
      smax = fmax(smax, cell_speed(u, gamma, gm1));
    }
    __shared__ double wm[FACE / 32];
    smax = cta_max<FACE / 32>(smax, wm);
    if (t == 0) bmax[b] = smax;
  }
}

cudaError_t launch_reflux(double* U, const double* R, const double* FH, const int32_t* list, const int32_t* fslot,
                          const int32_t* fh_src, int count, double h, double dt, const double* dt_dev,
                          double gamma, double* bmax, cudaStream_t st) {
  if (count <= 0) return cudaSuccess;
  reflux_kernel<<<count, FACE, 0, st>>>(U, R, FH, list, fslot, fh_src, h, dt, dt_dev, gamma, bmax);
  return cudaGetLastError();
}

// =====================================================================================================
// a10: CFL reduction ("grid-level reductions"; reading R16).  Per-thread running max,
// warp-shuffle max, one atomicMax per CTA on the bit pattern (positive doubles order like integers).
// =====================================================================================================
__global__ void __launch_bounds__(256) max_speed_kernel(const double* __restrict__ U, int first, int count, double gamma,
                                                        unsigned long long* smax_bits) {
  const double gm1 = gamma - 1.0;
  double smax = 0.0;
  for (int b = blockIdx.x; b < count; b += gridDim.x) {
    const double* Ub = U + size_t(first + b) * BLK;
#pragma unroll
    for (int c = threadIdx.x; c < NC; c += 256) {
      double u[5];
#pragma unroll
      for (int v = 0; v < NV; ++v) u[v] = Ub[v * NC + c];
      const double s = cell_speed(u, gamma, gm1);
      if (s > smax) smax = s;
    }
  }
  __shared__ double wm[8];
  smax = cta_max<8>(smax, wm);
  if (threadIdx.x == 0) atomicMax(smax_bits, (unsigned long long)__double_as_longlong(smax));
}

// the same maximum from the per-block maxima the corrector, the restriction and the reflux leave behind
__global__ void __launch_bounds__(256) max_cached_kernel(const double* __restrict__ bmax, int first, int count,
                                                         unsigned long long* smax_bits) {
  double smax = 0.0;
  for (int b = blockIdx.x * 256 + threadIdx.x; b < count; b += gridDim.x * 256) smax = fmax(smax, bmax[first + b]);
  __shared__ double wm[8];
  smax = cta_max<8>(smax, wm);
  if (threadIdx.x == 0) atomicMax(smax_bits, (unsigned long long)__double_as_longlong(smax));
}

cudaError_t launch_max_cached(const double* bmax, int first, int count, unsigned long long* smax_bits, int sms,
                              cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(smax_bits, 0, sizeof(unsigned long long), st);
  if (e != cudaSuccess || count <= 0) return e;
  const int need = (count + 2047) / 2048;
  max_cached_kernel<<<need < sms ? need : sms, 256, 0, st>>>(bmax, first, count, smax_bits);
  return cudaGetLastError();
}

cudaError_t launch_max_speed(const double* U, int first, int count, double gamma, unsigned long long* smax_bits,
                             int sms, cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(smax_bits, 0, sizeof(unsigned long long), st);
  if (e != cudaSuccess || count <= 0) return e;
  const int grid = count < sms * 8 ? count : sms * 8;
  max_speed_kernel<<<grid, 256, 0, st>>>(U, first, count, gamma, smax_bits);
  return cudaGetLastError();
}

__global__ void dt_finalize_kernel(const unsigned long long* smax_bits, LevelInfo li, double cfl, double* dt_dev,
                                   double* t_dev) {
  double dt = INFINITY;
  for (int l = 0; l < li.nlev; ++l)
    if (li.has[l]) dt = fmin(dt, cfl * li.h[l] / __longlong_as_double((long long)smax_bits[l]));
  *dt_dev = dt;
  *t_dev += dt;
}

cudaError_t launch_dt_finalize(const unsigned long long* smax_bits, const LevelInfo& li, double cfl, double* dt_dev,
                               double* t_dev, cudaStream_t st) {
  dt_finalize_kernel<<<1, 1, 0, st>>>(smax_bits, li, cfl, dt_dev, t_dev);
  return cudaGetLastError();
}

// =====================================================================================================
// status: cells with rho <= 0, P <= 0 or NaN (reading R28: reported, never floored)
// =====================================================================================================
__global__ void __launch_bounds__(256) count_bad_kernel(const double* __restrict__ U, int first, int count, double gamma,
                                                        int prim, unsigned long long* nbad) {
  const double gm1 = gamma - 1.0;
  unsigned int bad = 0;
  for (int b = blockIdx.x; b < count; b += gridDim.x) {
    const double* Ub = U + size_t(first + b) * BLK;
    for (int c = threadIdx.x; c < NC; c += 256) {
      double u[5], w[5];
#pragma unroll
      for (int v = 0; v < NV; ++v) u[v] = Ub[v * NC + c];
      if (prim) { w[0] = u[0]; w[4] = u[4]; }
      else cons_to_prim(u, gm1, w);
      if (!(w[0] > 0.0) || !(w[4] > 0.0)) ++bad;
    }
  }
  bad = __reduce_add_sync(0xffffffffu, bad);
  if ((threadIdx.x & 31) == 0 && bad) atomicAdd(nbad, (unsigned long long)bad);
}

cudaError_t launch_count_bad(const double* U, int first, int count, double gamma, int prim, unsigned long long* nbad,
                             int sms, cudaStream_t st) {
  if (count <= 0) return cudaSuccess;
  const int grid = count < sms * 8 ? count : sms * 8;
  count_bad_kernel<<<grid, 256, 0, st>>>(U, first, count, gamma, prim, nbad);
  return cudaGetLastError();
}

// =====================================================================================================
// caller layout <-> internal layout: block permutation (both are interior-only [5][8][8][8]); role 1 is
// held as primitives internally, so its copies convert on the way in and out.
// =====================================================================================================
__global__ void __launch_bounds__(256) permute_kernel(const double2* __restrict__ src, double2* __restrict__ dst,
                                                      const int64_t* __restrict__ perm, int first, int to_internal,
                                                      int ns, int bs16) {
  const int s = first + blockIdx.x;
  const int64_t e = perm[s];
  const size_t a = size_t(s) * (BLK / 2);
  for (int t = threadIdx.x; t < BLK / 2; t += 256) {
    const size_t b = caller_pos2(e, t / (NC / 2), t % (NC / 2), NV + ns, bs16);
    if (to_internal) dst[a + t] = src[b];
    else dst[b] = src[a + t];
  }
}

__global__ void __launch_bounds__(256) permute_prim_kernel(const double* __restrict__ src, double* __restrict__ dst,
                                                           const int64_t* __restrict__ perm, int first, int to_internal,
                                                           double gamma, int ns, int bs16) {
  const int s = first + blockIdx.x;
  const int64_t e = perm[s];
  const size_t a = size_t(s) * BLK;
  const double gm1 = gamma - 1.0, igm1 = 1.0 / gm1;
  for (int c = threadIdx.x; c < NC; c += 256) {
    double x[NV], y[NV];
    size_t b[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) b[v] = 2 * caller_pos2(e, v, c >> 1, NV + ns, bs16) + (c & 1);
#pragma unroll
    for (int v = 0; v < NV; ++v) x[v] = to_internal ? src[b[v]] : src[a + v * NC + c];
    if (to_internal) cons_to_prim(x, gm1, y);
    else prim_to_cons(x, igm1, y);
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      if (to_internal) dst[a + v * NC + c] = y[v];
      else dst[b[v]] = y[v];
    }
  }
}

cudaError_t launch_permute(const double* src, double* dst, const int64_t* perm, int first, int count, int to_internal,
                           int prim, double gamma, int ns, int bs16, cudaStream_t st) {
  if (count <= 0) return cudaSuccess;
  if (prim) permute_prim_kernel<<<count, 256, 0, st>>>(src, dst, perm, first, to_internal, gamma, ns, bs16);
  else permute_kernel<<<count, 256, 0, st>>>(reinterpret_cast<const double2*>(src), reinterpret_cast<double2*>(dst), perm,
                                             first, to_internal, ns, bs16);
  return cudaGetLastError();
}

// =====================================================================================================
// ghosted export (parity tests of the ghost fill): what the stage kernels stage, as 12^3 blocks
// =====================================================================================================
__global__ void __launch_bounds__(256) ghosted_kernel(const double* __restrict__ U, const double* __restrict__ ghost,
                                                      const int32_t* __restrict__ face_src,
                                                      const int64_t* __restrict__ perm, int first, int prim,
                                                      double gamma, double* __restrict__ G) {
  constexpr int M = N + 2 * NG;
  const int s = first + blockIdx.x;
  double* out = G + size_t(perm[s]) * NV * M * M * M;
  const double igm1 = 1.0 / (gamma - 1.0);
  for (int c = threadIdx.x; c < M * M * M; c += 256) {
    const int i = c % M - NG, j = (c / M) % M - NG, k = c / (M * M) - NG;
    const int o[3] = {i < 0 ? -1 : i >= N ? 1 : 0, j < 0 ? -1 : j >= N ? 1 : 0, k < 0 ? -1 : k >= N ? 1 : 0};
    const int nout = (o[0] != 0) + (o[1] != 0) + (o[2] != 0);
    const double* from = nullptr;   // variable 0 of the source cell
    int vs = NC;
    if (nout == 0) from = U + size_t(s) * BLK + (k * 8 + j) * 8 + i;
    else if (nout == 1) {
      const int axis = o[0] ? 0 : o[1] ? 1 : 2, side = o[axis] > 0;
      const int src = face_src[s * 6 + 2 * axis + side];
      int q[3] = {i, j, k};
      if (src == SRC_OUTFLOW) {
        q[axis] = side ? N - 1 : 0;
        from = U + size_t(s) * BLK + (q[2] * 8 + q[1]) * 8 + q[0];
      } else if (src >= 0) {
        q[axis] += side ? -N : N;
        from = U + size_t(src) * BLK + (q[2] * 8 + q[1]) * 8 + q[0];
      } else {
        const int ll = side ? q[axis] - N : q[axis] + NG;
        const int r = slab_pos(axis, ll, axis == 0 ? j : i, axis == 2 ? j : k);
        from = ghost + size_t(-2 - src) * SLAB + r;
        vs = NG * FACE;
      }
    }
    double x[NV], y[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) x[v] = from ? from[v * vs] : nan("");
    if (prim && from) prim_to_cons(x, igm1, y);
    else {
#pragma unroll
      for (int v = 0; v < NV; ++v) y[v] = x[v];
    }
#pragma unroll
    for (int v = 0; v < NV; ++v) out[v * M * M * M + c] = y[v];
  }
}

cudaError_t launch_ghosted(const double* U, const double* ghost, const int32_t* face_src, const int64_t* perm, int first,
                           int count, int prim, double gamma, double* G, cudaStream_t st) {
  if (count <= 0) return cudaSuccess;
  ghosted_kernel<<<count, 256, 0, st>>>(U, ghost, face_src, perm, first, prim, gamma, G);
  return cudaGetLastError();
}

// =====================================================================================================
// Refinement indicators.  One CTA of 256 threads per block: density and pressure of
// the block and of one ghost layer behind each face (gathered like the stage kernels do: the neighbour's
// interior, the block's own edge layer at an outflow face, the prolonged slab at a coarse-fine face) go to
// shared memory; then per interior cell
//   criterion 0, eq. (33)-(34) PAPER.md:277-285:  max(E(rho), E(P)),  E(q) = |sum_d (q_+d - 2 q + q_-d)| / q
//   criterion 1, PAPER.md:641 (reading R31):      h / lambda_J = h rho sqrt(G / (pi gamma P))
// and the maximum over the block, written in caller order.
// =====================================================================================================
__global__ void __launch_bounds__(256) refine_indicator_kernel(const double* __restrict__ U,
                                                               const double* __restrict__ ghost,
                                                               const int32_t* __restrict__ face_src,
                                                               const int64_t* __restrict__ perm, int first, int prim,
                                                               double gamma, int criterion, double G, double h,
                                                               double* __restrict__ out) {
  constexpr int M1 = N + 2;                    // one ghost layer
  __shared__ double rho[M1 * M1 * M1], prs[M1 * M1 * M1];
  __shared__ double wm[8];
  const int s = first + blockIdx.x;
  const double gm1 = gamma - 1.0;
  for (int c = threadIdx.x; c < M1 * M1 * M1; c += 256) {
    const int i = c % M1 - 1, j = (c / M1) % M1 - 1, k = c / (M1 * M1) - 1;
    const int o[3] = {i < 0 ? -1 : i >= N ? 1 : 0, j < 0 ? -1 : j >= N ? 1 : 0, k < 0 ? -1 : k >= N ? 1 : 0};
    const int nout = (o[0] != 0) + (o[1] != 0) + (o[2] != 0);
    if (nout > 1) continue;                    // edges and corners: no stencil reads them
    const double* from;
    int vs = NC;
    if (nout == 0) from = U + size_t(s) * BLK + (k * 8 + j) * 8 + i;
    else {
      const int axis = o[0] ? 0 : o[1] ? 1 : 2, side = o[axis] > 0;
      const int src = face_src[s * 6 + 2 * axis + side];
      int q[3] = {i, j, k};
      if (src == SRC_OUTFLOW) {
        q[axis] = side ? N - 1 : 0;
        from = U + size_t(s) * BLK + (q[2] * 8 + q[1]) * 8 + q[0];
      } else if (src >= 0) {
        q[axis] += side ? -N : N;
        from = U + size_t(src) * BLK + (q[2] * 8 + q[1]) * 8 + q[0];
      } else {
        const int ll = side ? 0 : NG - 1;      // the slab layer next to the face
        from = ghost + size_t(-2 - src) * SLAB + slab_pos(axis, ll, axis == 0 ? j : i, axis == 2 ? j : k);
        vs = NG * FACE;
      }
    }
    double x[NV], w[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) x[v] = from[v * vs];
    if (prim) { w[0] = x[0]; w[4] = x[4]; }
    else cons_to_prim(x, gm1, w);
    rho[c] = w[0];
    prs[c] = w[4];
  }
  __syncthreads();
  double best = 0.0;
  for (int c = threadIdx.x; c < NC; c += 256) {
    const int i = c & 7, j = (c >> 3) & 7, k = c >> 6;
    const int m = ((k + 1) * M1 + (j + 1)) * M1 + (i + 1);
    const double r0 = rho[m], P0 = prs[m];
    double val;
    if (criterion == 0) {
      double lr = 0.0, lP = 0.0;
      const int st[3] = {1, M1, M1 * M1};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        lr += (rho[m + st[d]] - 2.0 * r0) + rho[m - st[d]];
        lP += (prs[m + st[d]] - 2.0 * P0) + prs[m - st[d]];
      }
      val = fmax(fabs(lr) / r0, fabs(lP) / P0);
    } else {
      const double cs = sqrt(gamma * P0 / r0);
      val = h / (cs * sqrt(3.14159265358979323846 / (G * r0)));
    }
    best = fmax(best, val);
  }
  best = cta_max<8>(best, wm);
  if (threadIdx.x == 0) out[perm[s]] = best;
}

cudaError_t launch_refine_indicator(const double* U, const double* ghost, const int32_t* face_src, const int64_t* perm,
                                    int first, int count, int prim, double gamma, int criterion, double G, double h,
                                    double* out, cudaStream_t st) {
  if (count <= 0) return cudaSuccess;
  refine_indicator_kernel<<<count, 256, 0, st>>>(U, ghost, face_src, perm, first, prim, gamma, criterion, G, h, out);
  return cudaGetLastError();
}

// =====================================================================================================
// Regrid: state of a new mesh from an old one.  One CTA per block of
// the new mesh.  tsrc[d] >= 0: the block exists in the old mesh, slot tsrc[d]: copy.  tsrc[d] <= -2: it is
// new; its parent is old slot -2 - tsrc[d]: every fine cell is the slope-limited conservative prolongation
// (reading R3) of the parent's cell and its six neighbours, which lie in the parent, in its same-level
// neighbour, behind an outflow face (zero gradient) or in the old mesh's prolonged ghost slab.  tsrc[d] == -1:
// the parent is new as well (created one level earlier by the same transfer): the same prolongation from the
// NEW mesh's buffers, so a regrid may deepen the tree by any number of levels.
// =====================================================================================================
__global__ void __launch_bounds__(256) transfer_kernel(const TransferParams p) {
  const int d = blockIdx.x;
  const int t = p.tsrc[d];
  double* out = p.Ud + size_t(d) * BLK;
  if (t >= 0) {
    const double2* from = reinterpret_cast<const double2*>(p.Uc + size_t(t) * BLK);
    double2* to = reinterpret_cast<double2*>(out);
    for (int q = threadIdx.x; q < BLK / 2; q += 256) to[q] = from[q];
    return;
  }
  // the parent: in the old mesh (t <= -2) or in the new one (t == -1)
  const bool in_new = t == -1;
  const int P = in_new ? p.parent_n[d] : -2 - t;
  const double* Us = in_new ? p.Un : p.Us;
  const double* ghost = in_new ? p.ghost_n : p.ghost_s;
  const int32_t* face_src = in_new ? p.face_src_n : p.face_src_s;
  const int oct[3] = {p.coord_d[3 * d] & 1, p.coord_d[3 * d + 1] & 1, p.coord_d[3 * d + 2] & 1};
  const double* Up = Us + size_t(P) * BLK;
  auto fetch = [&](int c0, int c1, int c2, double q[NV]) {       // coarse cell of the parent's neighbourhood
    int c[3] = {c0, c1, c2};
    const double* from;
    int vs = NC;
    const int axis = (c0 < 0 || c0 >= N) ? 0 : (c1 < 0 || c1 >= N) ? 1 : (c2 < 0 || c2 >= N) ? 2 : -1;
    if (axis < 0) from = Up + (c[2] * 8 + c[1]) * 8 + c[0];
    else {
      const int side = c[axis] >= N;
      const int src = face_src[P * 6 + 2 * axis + side];
      if (src == SRC_OUTFLOW) {
        c[axis] = side ? N - 1 : 0;
        from = Up + (c[2] * 8 + c[1]) * 8 + c[0];
      } else if (src >= 0) {
        c[axis] += side ? -N : N;
        from = Us + size_t(src) * BLK + (c[2] * 8 + c[1]) * 8 + c[0];
      } else {
        from = ghost + size_t(-2 - src) * SLAB +
               slab_pos(axis, side ? 0 : NG - 1, axis == 0 ? c[1] : c[0], axis == 2 ? c[1] : c[2]);
        vs = NG * FACE;
      }
    }
#pragma unroll
    for (int v = 0; v < NV; ++v) q[v] = from[v * vs];
  };
  for (int cell = threadIdx.x; cell < NC; cell += 256) {
    const int f[3] = {cell & 7, (cell >> 3) & 7, cell >> 6};
    const int c[3] = {oct[0] * 4 + (f[0] >> 1), oct[1] * 4 + (f[1] >> 1), oct[2] * 4 + (f[2] >> 1)};
    double Q[NV], Qp[NV], Qm[NV], val[NV];
    fetch(c[0], c[1], c[2], Q);
#pragma unroll
    for (int v = 0; v < NV; ++v) val[v] = Q[v];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      fetch(c[0] + (a == 0), c[1] + (a == 1), c[2] + (a == 2), Qp);
      fetch(c[0] - (a == 0), c[1] - (a == 1), c[2] - (a == 2), Qm);
      const double sig = (f[a] & 1) ? 0.25 : -0.25;
#pragma unroll
      for (int v = 0; v < NV; ++v) val[v] = val[v] + sig * minmod(Qp[v] - Q[v], Q[v] - Qm[v]);
    }
#pragma unroll
    for (int v = 0; v < NV; ++v) out[v * NC + cell] = val[v];
  }
}

cudaError_t launch_transfer(const TransferParams& p, int count, cudaStream_t st) {
  if (count <= 0) return cudaSuccess;
  transfer_kernel<<<count, 256, 0, st>>>(p);
  return cudaGetLastError();
}

// =====================================================================================================
// fp64 issue-rate microbenchmark (the "alu" roofline denominator of bench.py): every thread runs CHAINS
// independent DFMA chains; with 1024 threads per SM the fp64 pipe is saturated whatever the dependent
// latency.  Returns nothing useful in `sink` (it only keeps the compiler from dropping the loop).
// =====================================================================================================
template <int CHAINS>
__global__ void __launch_bounds__(1024) dfma_rate_kernel(int iters, double seed, double* __restrict__ sink) {
  double x[CHAINS];
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) x[c] = seed + 1e-3 * (threadIdx.x + c);
  const double a = 1.0 - 1e-9, b = 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 16; ++r)
#pragma unroll
      for (int c = 0; c < CHAINS; ++c) x[c] = fma(x[c], a, b);
  }
  double t = 0.0;
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) t += x[c];
  if (t == 123.456) sink[0] = t;
}

// thread-level DFMA instructions per launch = ctas * 1024 * iters * 16 * chains
cudaError_t launch_dfma_rate(int chains, int ctas, int iters, double* sink, cudaStream_t st) {
  if (chains == 1) dfma_rate_kernel<1><<<ctas, 1024, 0, st>>>(iters, 0.5, sink);
  else if (chains == 2) dfma_rate_kernel<2><<<ctas, 1024, 0, st>>>(iters, 0.5, sink);
  else if (chains == 4) dfma_rate_kernel<4><<<ctas, 1024, 0, st>>>(iters, 0.5, sink);
  else dfma_rate_kernel<8><<<ctas, 1024, 0, st>>>(iters, 0.5, sink);
  return cudaGetLastError();
}

}  // namespace sfh

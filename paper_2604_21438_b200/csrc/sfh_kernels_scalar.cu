// sfh_kernels_scalar.cu — passive scalars on the hydro sweep (eq. 12-13, PAPER.md:80-88;
// DESIGN.md reading R32).  A scalar is carried as the conserved density q = rho * s; its interface flux is the
// Riemann solver's mass flux (exported by the stage kernels, StageParams::mf) times the interface value of s on the
// side the mass comes from, F_q = F_rho * (F_rho >= 0 ? s_L : s_R); s is cell-centred in the predictor and
// minmod-limited linear in the corrector, like the other primitives (R11, R12).  The scalars live behind the hydro
// part of every state buffer, Q[nb][ns][8][8][8] (conserved in all three roles), with their own coarse-fine ghost
// slabs and flux registers; prolongation, eq. (16), restriction and reflux act on them exactly as on the hydro
// variables.  These kernels move 40 B per scalar and cell-update and do a handful of flops: plain gather kernels.
#include <cmath>

#include "sfh_device.cuh"
#include "sfh_kernels.cuh"

namespace sfh {

constexpr int M12 = N + 2 * NG;      // ghosted edge
// The ghosted block in shared memory: rows of 12 cells at a stride of 24 doubles, so that the two rows a half warp
// reads (8 cells of row j, 8 of row j + 1) fall on disjoint banks (a stride of 12 gives two-way conflicts: measured
// 43 % of the kernel's shared-memory wavefronts).
constexpr int ROW = 24, PLANE = M12 * ROW + 2;   // (+ 2: the x-halo stores, one cell per (j, k), spread over the banks)
constexpr int G3 = M12 * PLANE;
__device__ __forceinline__ int gpos(int i, int j, int k) { return (k + NG) * PLANE + (j + NG) * ROW + (i + NG); }

// Source of one variable of ghosted cell (i, j, k) of block s: the block itself, the same-level neighbour, the block's
// own edge layer (outflow) or the coarse-fine slab.  Edge / corner ghosts (no stage reads them): returns null.
// U: array [nb][nvar][512] (+ v * NC selects the variable); slab: [ncf][nslabvar][128] (+ v * 128); fsrc6: the six
// face sources of block s.
__device__ __forceinline__ const double* ghost_src(const double* __restrict__ U, int nvar, const double* __restrict__ slab,
                                                   int nslabvar, const int32_t* __restrict__ fsrc6, int s, int i, int j,
                                                   int k, int* vstride) {
  const int o[3] = {i < 0 ? -1 : i >= N ? 1 : 0, j < 0 ? -1 : j >= N ? 1 : 0, k < 0 ? -1 : k >= N ? 1 : 0};
  const int nout = (o[0] != 0) + (o[1] != 0) + (o[2] != 0);
  *vstride = NC;
  if (nout == 0) return U + size_t(s) * nvar * NC + (k * 8 + j) * 8 + i;
  if (nout > 1) return nullptr;
  const int axis = o[0] ? 0 : o[1] ? 1 : 2, side = o[axis] > 0;
  const int src = fsrc6[2 * axis + side];
  int q[3] = {i, j, k};
  if (src == SRC_OUTFLOW) {
    q[axis] = side ? N - 1 : 0;
    return U + size_t(s) * nvar * NC + (q[2] * 8 + q[1]) * 8 + q[0];
  }
  if (src >= 0) {
    q[axis] += side ? -N : N;
    return U + size_t(src) * nvar * NC + (q[2] * 8 + q[1]) * 8 + q[0];
  }
  const int ll = side ? q[axis] - N : q[axis] + NG;
  *vstride = NG * FACE;
  return slab + size_t(-2 - src) * nslabvar * (NG * FACE) + slab_pos(axis, ll, axis == 0 ? j : i, axis == 2 ? j : k);
}

// =====================================================================================================
// Scalar stage: one CTA of 256 threads per block.  1 / rho and s = q / rho of the block and its two-layer face halos
// go to shared memory (gathered like the stage kernels gather: neighbour interiors, outflow copies, coarse-fine
// slabs; every thread resolves the sources of its up to seven ghosted cells ONCE, for all scalars), and so do the
// block's mass fluxes (read coalesced, stored face-fastest / row-contiguous so that the cells of a warp read them
// without bank conflicts).  Every thread then updates two cells per scalar: the six face fluxes of a cell (each
// face is evaluated by both its cells, a few flops), dF in the order (x + y) + z, q_out = q^n - lambda dF.
// STAGE 1 also feeds the scalar flux registers of coarse-fine faces (fine side += dt F, coarse leaf side = F; one
// contributor per entry: no atomics needed).
// =====================================================================================================
// mass fluxes of one block in shared memory: x faces [k][j][9], y faces [k][9][i], z faces [9][j][i]
__device__ __forceinline__ int mfs_pos(int d, int f, int ta, int tb) {   // face f of pencil (ta, tb) (lower axis first)
  return d == 0 ? (tb * 8 + ta) * 9 + f : d == 1 ? 576 + (tb * 9 + f) * 8 + ta : 1152 + (f * 8 + tb) * 8 + ta;
}

template <int STAGE>
__global__ void __launch_bounds__(256, 4) scalar_stage_kernel(const ScalarStageParams p) {
  __shared__ double sv[G3];                // s = q / rho on the ghosted block (edges and corners are never read)
  __shared__ double mfs[3 * 9 * FACE];
  const int s = p.first + blockIdx.x;
  const int t = threadIdx.x;
  const double dt = p.dt_dev ? *p.dt_dev : p.dt;
  const double lam = (STAGE == 0 ? 0.5 : 1.0) * dt / p.h;
  __shared__ int fsrc6[6];                 // the face sources first: the gathers below must not wait for them one by one
  __shared__ int fslot6[6];
  if (t < 6) { fsrc6[t] = p.face_src[s * 6 + t]; fslot6[t] = STAGE == 1 ? p.fslot[s * 6 + t] : -1; }
  // the block's mass fluxes [axis][face 0..8][pencil]: coalesced read, transposed store; warp pair w2 = t >> 6 takes
  // the (axis, face) rows w2, w2 + 4, ...
  const double* mf = p.mf + size_t(s) * 3 * 9 * FACE;
#pragma unroll
  for (int rr = 0; rr < 7; ++rr) {
    const int row = (t >> 6) + 4 * rr, pen = t & (FACE - 1);
    if (row < 27) mfs[mfs_pos(row / 9, row % 9, pen & 7, pen >> 3)] = mf[row * FACE + pen];
  }
  __syncthreads();
  // My five cells of the ghosted block: interior cells t and t + 256, and items t, t + 256, t + 512 of the six
  // two-layer face halos (item h: face h >> 7 -- warp-uniform --, layer (h >> 6) & 1, in-face position h & 63).  For
  // each: where it goes in the 12^3 arrays, and where variable 0 of rho / of the scalars comes from (the block itself,
  // the same-level neighbour, the block's own edge layer at an outflow face, or the coarse-fine slab).
  constexpr int NI = 5;
  int dst[NI];
  const double* qsrc[NI];
  const double* hsrc[NI];
  unsigned slabbed = 0;                    // bit r: the source is a coarse-fine slab (variable stride 128, not 512)
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int cell = t + 256 * r;
    dst[r] = gpos(cell & 7, (cell >> 3) & 7, cell >> 6);
    hsrc[r] = p.Hsrc + size_t(s) * NV * NC + cell;
    qsrc[r] = p.Qsrc + size_t(s) * p.ns * NC + cell;
  }
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    const int h = t + 256 * r, f = h >> 7, axis = f >> 1, side = f & 1, ll = (h >> 6) & 1, ta = h & 7, tb = (h >> 3) & 7;
    const int src = fsrc6[f];
    int q[3];                              // the ghost cell, block-local
    q[axis] = side ? N + ll : ll - NG;
    q[axis == 0 ? 1 : 0] = ta;
    q[axis == 2 ? 1 : 2] = tb;
    dst[2 + r] = gpos(q[0], q[1], q[2]);
    if (src <= -2) {                       // coarse-fine slab
      const int pos = slab_pos(axis, ll, ta, tb);
      hsrc[2 + r] = p.ghostH + size_t(-2 - src) * NV * (NG * FACE) + pos;
      qsrc[2 + r] = p.ghostS + size_t(-2 - src) * p.ns * (NG * FACE) + pos;
      slabbed |= 1u << (2 + r);
    } else {
      const int blk = src >= 0 ? src : s;  // same-level neighbour, or the block's own edge layer (outflow)
      q[axis] = src >= 0 ? q[axis] + (side ? -N : N) : (side ? N - 1 : 0);
      const int cell = (q[2] * 8 + q[1]) * 8 + q[0];
      hsrc[2 + r] = p.Hsrc + size_t(blk) * NV * NC + cell;
      qsrc[2 + r] = p.Qsrc + size_t(blk) * p.ns * NC + cell;
    }
  }
  // All loads of the first scalar are in flight together with those of rho; the loads of scalar v + 1 are issued
  // before scalar v is computed (one memory latency per block instead of one per phase).
  double rh[NI], qv[NI];
  auto load_q = [&](int v) {
#pragma unroll
    for (int r = 0; r < NI; ++r) qv[r] = qsrc[r][v * ((slabbed >> r) & 1 ? NG * FACE : NC)];
  };
#pragma unroll
  for (int r = 0; r < NI; ++r) rh[r] = hsrc[r][0];                 // variable 0 of both copies is rho
  load_q(0);
  double ir[NI];
#pragma unroll
  for (int r = 0; r < NI; ++r) ir[r] = rcp_fast(rh[r]);
  // my two cells (i, j, k0) and (i, j, k0 + 4): positions in the ghosted array and of their lower faces' mass fluxes
  // (the upper faces and the second cell are constant offsets away)
  const int ci = t & 7, cj = (t >> 3) & 7, ck0 = t >> 6;
  const int m00 = gpos(ci, cj, ck0);
  const int fpos[3] = {mfs_pos(0, ci, cj, ck0), mfs_pos(1, cj, ci, ck0), mfs_pos(2, ck0, ci, cj)};
  constexpr int st[3] = {1, ROW, PLANE};
  constexpr int fup[3] = {1, 8, FACE};                                  // next face along the pencil
  constexpr int fk4[3] = {4 * 8 * 9, 4 * 9 * 8, 4 * FACE};              // the same pencil position four planes up
  for (int v = 0; v < p.ns; ++v) {
    __syncthreads();                         // the previous scalar's sv is no longer read
#pragma unroll
    for (int r = 0; r < NI; ++r) sv[dst[r]] = qv[r] * ir[r];
    if (v + 1 < p.ns) load_q(v + 1);
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int cell = t + 256 * r, m0 = m00 + 4 * r * PLANE;
      const int ijk[3] = {ci, cj, ck0 + 4 * r};
      const size_t o = (size_t(s) * p.ns + v) * NC + cell;
      const double qn = p.Qn[o];
      double dF[3];
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const int c = ijk[d];
        // s of the cells c-1, c, c+1 (and c-2, c+2 for the corrector's three limited slopes): each slope once
        const double s0 = sv[m0], sm = sv[m0 - st[d]], sp = sv[m0 + st[d]];
        double sL[2] = {sm, s0}, sR[2] = {s0, sp};            // left / right states of the lower and the upper face
        if (STAGE == 1) {
          const double smm = sv[m0 - 2 * st[d]], spp = sv[m0 + 2 * st[d]];
          const double d1 = sm - smm, d2 = s0 - sm, d3 = sp - s0, d4 = spp - sp;
          const double hm = half_minmod(d2, d1), h0 = half_minmod(d3, d2), hp = half_minmod(d4, d3);
          sL[0] = sm + hm; sR[0] = s0 - h0; sL[1] = s0 + h0; sR[1] = sp - hp;
        }
        double F[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {        // the cell's lower (e = 0) and upper face: face index c + e
          const double fm = mfs[fpos[d] + r * fk4[d] + e * fup[d]];
          F[e] = fm * (fm >= 0.0 ? sL[e] : sR[e]);
        }
        dF[d] = F[1] - F[0];
        if (STAGE == 1 && (c == 0 || c == N - 1)) {        // flux registers (a7 for the scalars)
          const int ta = d == 0 ? ijk[1] : ijk[0], tb = d == 2 ? ijk[1] : ijk[2];
          const int e = c == 0 ? 0 : 1, f = 2 * d + e;
          const int src = fsrc6[f], fs = fslot6[f];
          if (src <= -2) {
            double* rg = p.RS + (size_t(-2 - src) * p.ns + v) * FACE + tb * 8 + ta;
            *rg = *rg + dt * F[e];
          }
          if (fs >= 0) p.FHS[(size_t(fs) * p.ns + v) * FACE + tb * 8 + ta] = F[e];
        }
      }
      p.Qdst[o] = qn - lam * ((dF[0] + dF[1]) + dF[2]);
    }
  }
}

cudaError_t launch_scalar_stage(int stage, const ScalarStageParams& p, cudaStream_t st) {
  if (p.count <= 0 || p.ns <= 0) return cudaSuccess;
  if (stage == 0) scalar_stage_kernel<0><<<p.count, 256, 0, st>>>(p);
  else scalar_stage_kernel<1><<<p.count, 256, 0, st>>>(p);
  return cudaGetLastError();
}

// =====================================================================================================
// Coarse-fine ghost slabs of the scalars: the geometry of prolong_kernel (sfh_kernels_aux.cu), one variable at a
// time, conserved values throughout (no primitive copies).  interp: eq. (16) at tau (and at tau1 into ghost1).
// =====================================================================================================
constexpr int PR_RIM = 36, PR_CELLS = PR_RIM + 2 * 16;

__global__ void __launch_bounds__(128) prolong_scalar_kernel(const ProlongScalarParams p) {
  __shared__ double q[PR_CELLS], q1[PR_CELLS];
  __shared__ int missing;
  const int slot = p.first + blockIdx.x;
  const int F = p.cf_block[slot], f = p.cf_face[slot], axis = f >> 1, side = f & 1;
  const int P = p.parent[F];
  const int t1ax = axis == 0 ? 1 : 0, t2ax = axis == 2 ? 1 : 2;
  int oct[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) oct[d] = p.coord[3 * F + d] & 1;
  const int r = threadIdx.x;
  if (r == 0) missing = 0;
  // ---- which coarse cell thread r < 68 gathers (the same for every variable)
  size_t src_off = 0;
  bool gather = false;
  if (r < PR_CELLS) {
    int ca, c1, c2;
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
      const bool out_lo[3] = {nb[12] == NBR_OUTSIDE, nb[10] == NBR_OUTSIDE, nb[4] == NBR_OUTSIDE};
      const bool out_hi[3] = {nb[14] == NBR_OUTSIDE, nb[16] == NBR_OUTSIDE, nb[22] == NBR_OUTSIDE};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        rg[d] = 0;
        if (c[d] < 0) { if (out_lo[d]) c[d] = 0; else { rg[d] = -1; c[d] += N; } }
        else if (c[d] >= N) { if (out_hi[d]) c[d] = N - 1; else { rg[d] = 1; c[d] -= N; } }
      }
      const int Q = nb[(rg[2] + 1) * 9 + (rg[1] + 1) * 3 + (rg[0] + 1)];
      if (Q < 0) missing = 1;
      else { gather = true; src_off = size_t(Q) * p.ns * NC + (c[2] * 8 + c[1]) * 8 + c[0]; }
    }
  }
  // ---- which fine ghost cell thread r computes
  int fc[3];
  if (axis == 0) { const int ll = r & 1; fc[0] = side ? N + ll : ll - NG; fc[1] = (r >> 1) & 7; fc[2] = r >> 4; }
  else if (axis == 1) { const int ll = (r >> 3) & 1; fc[0] = r & 7; fc[1] = side ? N + ll : ll - NG; fc[2] = r >> 4; }
  else { const int ll = r >> 6; fc[0] = r & 7; fc[1] = (r >> 3) & 7; fc[2] = side ? N + ll : ll - NG; }
  const int c1 = fc[t1ax] >> 1, c2 = fc[t2ax] >> 1;
  const int ctr = (c2 + 1) * 6 + (c1 + 1);
  int nbp[3], nbm[3];
  nbp[axis] = PR_RIM + 16 + c2 * 4 + c1; nbm[axis] = PR_RIM + c2 * 4 + c1;
  nbp[t1ax] = ctr + 1; nbm[t1ax] = ctr - 1;
  nbp[t2ax] = ctr + 6; nbm[t2ax] = ctr - 6;
  const int ll = fc[axis] < 0 ? fc[axis] + NG : fc[axis] - N;
  const int rout = slab_pos(axis, ll, fc[axis == 0 ? 1 : 0], fc[axis == 2 ? 1 : 2]);
  for (int v = 0; v < p.ns; ++v) {
    __syncthreads();
    if (gather) {
      const size_t o = src_off + size_t(v) * NC;
      const double u0 = p.C0[o];
      if (p.interp) {
        const double u1 = p.C1[o], u2 = p.C2[o];
        q[r] = time_interp(u0, u1, u2, p.tau);
        if (p.ghost1) q1[r] = time_interp(u0, u1, u2, p.tau1);
      } else {
        q[r] = u0;
      }
    }
    __syncthreads();
    auto fine_value = [&](const double* qq, double* __restrict__ ghost) {
      const double q0 = qq[ctr];
      double val = q0;
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const double sig = (fc[d] & 1) ? 0.25 : -0.25;
        val = val + sig * minmod(qq[nbp[d]] - q0, q0 - qq[nbm[d]]);
      }
      if (missing) val = nan("");
      ghost[(size_t(slot) * p.ns + v) * (NG * FACE) + rout] = val;
    };
    fine_value(q, p.ghost);
    if (p.ghost1) fine_value(q1, p.ghost1);
  }
}

cudaError_t launch_prolong_scalar(const ProlongScalarParams& p, cudaStream_t st) {
  if (p.count <= 0 || p.ns <= 0) return cudaSuccess;
  prolong_scalar_kernel<<<p.count, 128, 0, st>>>(p);
  return cudaGetLastError();
}

// =====================================================================================================
// Restriction and reflux of the scalars: restrict_kernel / reflux_kernel (sfh_kernels_aux.cu) on Q, RS, FHS.
// =====================================================================================================
__global__ void __launch_bounds__(NC) restrict_scalar_kernel(const double* __restrict__ Qf, double* __restrict__ Qc,
                                                             const int32_t* __restrict__ list,
                                                             const int32_t* __restrict__ child0, int ns) {
  const int b = list[blockIdx.x];
  const int t = threadIdx.x, i = t & 7, j = (t >> 3) & 7, k = t >> 6;
  const int child = child0[b] + (i >> 2) + 2 * (j >> 2) + 4 * (k >> 2);
  const int fi = 2 * (i & 3), fj = 2 * (j & 3), fk = 2 * (k & 3);
  for (int v = 0; v < ns; ++v) {
    const double* src = Qf + (size_t(child) * ns + v) * NC;
    double sum = 0.0;
#pragma unroll
    for (int c = 0; c < 8; ++c) sum += src[((fk + ((c >> 2) & 1)) * 8 + fj + ((c >> 1) & 1)) * 8 + fi + (c & 1)];
    Qc[(size_t(b) * ns + v) * NC + t] = 0.125 * sum;
  }
}

cudaError_t launch_restrict_scalar(const double* Qfine, double* Qcoarse, const int32_t* list, const int32_t* child0,
                                   int count, int ns, cudaStream_t st) {
  if (count <= 0 || ns <= 0) return cudaSuccess;
  restrict_scalar_kernel<<<count, NC, 0, st>>>(Qfine, Qcoarse, list, child0, ns);
  return cudaGetLastError();
}

__global__ void __launch_bounds__(FACE) reflux_scalar_kernel(double* __restrict__ Q, const double* __restrict__ RS,
                                                             const double* __restrict__ FHS,
                                                             const int32_t* __restrict__ list,
                                                             const int32_t* __restrict__ fslot,
                                                             const int32_t* __restrict__ fh_src, int ns, double h,
                                                             double dt_host, const double* __restrict__ dt_dev) {
  const int b = list[blockIdx.x];
  const int t = threadIdx.x, ta = t & 7, tb = t >> 3;
  const double dt = dt_dev ? *dt_dev : dt_host;
  for (int f = 0; f < 6; ++f) {
    const int fs = fslot[b * 6 + f];
    if (fs >= 0) {
      const int d = f >> 1, side = f & 1, c = side ? N - 1 : 0;
      const double s = side ? 1.0 : -1.0;
      const int cell = d == 0 ? (tb * 8 + ta) * 8 + c : d == 1 ? (tb * 8 + c) * 8 + ta : (c * 8 + tb) * 8 + ta;
      const int slot = fh_src[fs * 4 + (ta >> 2) + 2 * (tb >> 2)];
      const int fa = 2 * (ta & 3), fb = 2 * (tb & 3);
      for (int v = 0; v < ns; ++v) {
        const double* r = RS + (size_t(slot) * ns + v) * FACE;
        double sumR = 0.0;
#pragma unroll
        for (int q = 0; q < 4; ++q) sumR += r[(fb + (q >> 1)) * 8 + fa + (q & 1)];
        const double FHv = FHS[(size_t(fs) * ns + v) * FACE + t];
        double* u = Q + (size_t(b) * ns + v) * NC + cell;
        *u = *u - (s / h) * (0.25 * sumR - dt * FHv);
      }
    }
    __syncthreads();
  }
}

cudaError_t launch_reflux_scalar(double* Q, const double* RS, const double* FHS, const int32_t* list,
                                 const int32_t* fslot, const int32_t* fh_src, int count, int ns, double h, double dt,
                                 const double* dt_dev, cudaStream_t st) {
  if (count <= 0 || ns <= 0) return cudaSuccess;
  reflux_scalar_kernel<<<count, FACE, 0, st>>>(Q, RS, FHS, list, fslot, fh_src, ns, h, dt, dt_dev);
  return cudaGetLastError();
}

// =====================================================================================================
// caller layout [nb][5 + ns][512] <-> internal scalar part [slot][ns][512]
// =====================================================================================================
__global__ void __launch_bounds__(256) permute_scalar_kernel(const double2* __restrict__ src, double2* __restrict__ dst,
                                                             const int64_t* __restrict__ perm, int first, int ns,
                                                             int to_internal, int bs16) {
  const int s = first + blockIdx.x;
  const int64_t e = perm[s];
  const size_t in = size_t(s) * ns * (NC / 2);                               // internal: scalars only
  for (int t = threadIdx.x; t < ns * (NC / 2); t += 256) {
    // caller: behind the 5 hydro variables
    const size_t ca = caller_pos2(e, NV + t / (NC / 2), t % (NC / 2), NV + ns, bs16);
    if (to_internal) dst[in + t] = src[ca];
    else dst[ca] = src[in + t];
  }
}

cudaError_t launch_permute_scalar(const double* src, double* dst, const int64_t* perm, int first, int count, int ns,
                                  int to_internal, int bs16, cudaStream_t st) {
  if (count <= 0 || ns <= 0) return cudaSuccess;
  permute_scalar_kernel<<<count, 256, 0, st>>>(reinterpret_cast<const double2*>(src), reinterpret_cast<double2*>(dst),
                                               perm, first, ns, to_internal, bs16);
  return cudaGetLastError();
}

// =====================================================================================================
// Regrid: scalars of a new mesh from an old one (transfer_kernel of sfh_kernels_aux.cu on Q and the scalar slabs)
// =====================================================================================================
__global__ void __launch_bounds__(256) transfer_scalar_kernel(const TransferParams p, int ns) {
  const int d = blockIdx.x;
  const int t = p.tsrc[d];
  double* out = p.Ud + size_t(d) * ns * NC;
  if (t >= 0) {
    const double2* from = reinterpret_cast<const double2*>(p.Uc + size_t(t) * ns * NC);
    double2* to = reinterpret_cast<double2*>(out);
    for (int q = threadIdx.x; q < ns * NC / 2; q += 256) to[q] = from[q];
    return;
  }
  const bool in_new = t == -1;
  const int P = in_new ? p.parent_n[d] : -2 - t;
  const double* Qs = in_new ? p.Un : p.Us;
  const double* ghost = in_new ? p.ghost_n : p.ghost_s;
  const int32_t* face_src = in_new ? p.face_src_n : p.face_src_s;
  const int oct[3] = {p.coord_d[3 * d] & 1, p.coord_d[3 * d + 1] & 1, p.coord_d[3 * d + 2] & 1};
  for (int v = 0; v < ns; ++v)
    for (int cell = threadIdx.x; cell < NC; cell += 256) {
      const int f[3] = {cell & 7, (cell >> 3) & 7, cell >> 6};
      const int c[3] = {oct[0] * 4 + (f[0] >> 1), oct[1] * 4 + (f[1] >> 1), oct[2] * 4 + (f[2] >> 1)};
      auto fetch = [&](int c0, int c1, int c2) {       // one ghost layer is reached at most: the slab layer next to the face
        int vs;
        const double* from = ghost_src(Qs, ns, ghost, ns, face_src + P * 6, P, c0, c1, c2, &vs);
        return from[v * vs];
      };
      const double Q = fetch(c[0], c[1], c[2]);
      double val = Q;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        const double Qp = fetch(c[0] + (a == 0), c[1] + (a == 1), c[2] + (a == 2));
        const double Qm = fetch(c[0] - (a == 0), c[1] - (a == 1), c[2] - (a == 2));
        const double sig = (f[a] & 1) ? 0.25 : -0.25;
        val = val + sig * minmod(Qp - Q, Q - Qm);
      }
      out[size_t(v) * NC + cell] = val;
    }
}

cudaError_t launch_transfer_scalar(const TransferParams& p, int count, int ns, cudaStream_t st) {
  if (count <= 0 || ns <= 0) return cudaSuccess;
  transfer_scalar_kernel<<<count, 256, 0, st>>>(p, ns);
  return cudaGetLastError();
}

}  // namespace sfh

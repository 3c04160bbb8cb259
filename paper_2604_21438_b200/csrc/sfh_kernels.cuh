// sfh_kernels.cuh — launch wrappers of the CUDA kernels of libsfh (defined in sfh_kernels.cu).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

#include "sfh_internal.h"

namespace sfh {

struct StageParams {
  const double* Usrc;   // state the stage differentiates: U^n (predictor) or U^{n+1/2} (corrector)
  const double* Un;     // U^n, the state that is updated
  double* Udst;         // U^{n+1/2} (predictor) or U^{n+1} (corrector)
  const double* ghost;  // coarse-fine ghost slabs [ncf][5][2 layers x 64]
  double* R;            // fine-side flux registers  [ncf][5][64]
  double* FH;           // coarse-side flux registers [nfh][5][64]
  const int32_t* face_src;
  const int32_t* fslot;
  const double* dt_dev;  // if non-null the step is read from device memory
  double dt;
  double h;
  double gamma;
  int first, count;      // slot range of the level
  int use_regs;          // corrector: the level has flux-register faces
  int riemann;           // 0 HLLC, 1 Roe
  double* bmax;          // corrector: per-block maximum CFL speed of U^{n+1} (or null)
  double* mf;            // if non-null: mass flux of every face, [blocks of the level][3 axes][9 faces][64 pencils], base shifted so that slots index it (passive scalars)
};

struct TensorMaps {      // tensor maps of ONE state buffer seen as [5 nb][8][8][8]
  CUtensorMap ax;        // x-face slab: box {2,8,8,5} over (i, j, k, var), dense in smem: [var][k][j][ll]
  CUtensorMap ay;        // y-face slab: box {8,8,2,5} over the PERMUTED view (i, k, j, var), dense: [var][ll][k][i]
  CUtensorMap zs;        // box {8,8,2,5} (a pair of z planes of all 5 variables), 128-byte swizzled in smem
};

// Positions inside a coarse-fine ghost slab [var][128] (variable stride 128) = the staging layout of
// the stage kernels (sfh_kernels.cu): ll = layer (index increasing with the coordinate), (ta, tb) = the
// two in-face coordinates, lower axis first.
__host__ __device__ inline int slab_pos(int axis, int ll, int ta, int tb);

// Position of cell (kl, j, i) of a z-plane pair inside a 128-byte-swizzled slab [v][kl][j][i] of fp64
// (variable stride 128): the TMA swizzle XORs byte-address bits [4,7) with bits [7,10), i.e. the
// 16-byte chunk (i >> 1, j & 1) with (j >> 1, kl).
__host__ __device__ inline int zs_pos(int kl, int j, int i) { return (kl << 6) | ((j ^ kl) << 3) | (i ^ (j & 6)); }
__host__ __device__ inline int slab_pos(int axis, int ll, int ta, int tb) {
  return axis == 0 ? (tb * 8 + ta) * 2 + ll : axis == 1 ? ll * 64 + tb * 8 + ta : zs_pos(ll, tb, ta);
}

struct ProlongParams {
  const double* C0;      // coarse level: role `which` (interp = 0) or role 0 (interp = 1)
  const double* C1;      // coarse role 1 (interp = 1)
  const double* C2;      // coarse role 2 (interp = 1)
  double* ghost;
  const int32_t* cf_block;
  const int32_t* cf_face;
  const int32_t* parent;
  const int32_t* coord;
  const int32_t* nbr27;
  int first, count;      // slab range of the fine level
  int interp;
  double tau;
  int c0_prim, c1_prim;  // the coarse copy C0 / C1 holds primitives (the half-step state)
  int out_prim;          // write primitives (half-step fill)
  double gamma;
  // dual fill (interp = 1 only): the same gather also yields the half-step slab at tau1, as primitives
  double* ghost1;        // or null
  double tau1;
};

// sms: SM count of the device (configure_kernels): the persistent grid is min(count, sms) CTAs
cudaError_t launch_stage(int stage, const TensorMaps& tm, const StageParams& p, int sms, cudaStream_t st);
cudaError_t launch_prolong(const ProlongParams& p, cudaStream_t st);
// bmax (nullable): per-block maximum CFL speed, rewritten for the blocks the kernel changes
cudaError_t launch_restrict(const double* Ufine, double* Ucoarse, const int32_t* list, const int32_t* child0,
                            int count, double gamma, double* bmax, cudaStream_t st);
cudaError_t launch_reflux(double* U, const double* R, const double* FH, const int32_t* list, const int32_t* fslot,
                          const int32_t* fh_src, int count, double h, double dt, const double* dt_dev,
                          double gamma, double* bmax, cudaStream_t st);
cudaError_t launch_max_speed(const double* U, int first, int count, double gamma, unsigned long long* smax_bits,
                             int sms, cudaStream_t st);
cudaError_t launch_max_cached(const double* bmax, int first, int count, unsigned long long* smax_bits, int sms,
                              cudaStream_t st);
struct LevelInfo {
  double h[MAX_LEVELS];
  int has[MAX_LEVELS];
  int nlev;
};
// dt = min_l cfl*h_l/smax_l over levels with blocks; *dt_dev = dt; *t_dev += dt
cudaError_t launch_dt_finalize(const unsigned long long* smax_bits, const LevelInfo& li, double cfl, double* dt_dev,
                               double* t_dev, cudaStream_t st);
cudaError_t launch_count_bad(const double* U, int first, int count, double gamma, int prim, unsigned long long* nbad,
                             int sms, cudaStream_t st);
// Position (in double2 units) of cell pair t2 = cell / 2 of variable v of caller entry e, in a caller array with nvt
// variables per cell.  Blocks of 8^3 cells: [e][nvt][512].  Blocks of 16^3 cells (bs16): the
// library handles a 16^3 block as its eight 8^3 octants, e = 8 * block + octant (octant c = cx + 2 cy + 4 cz), and
// the caller's array is [block][nvt][16][16][16]: an octant's rows of 8 cells are contiguous.
__host__ __device__ inline size_t caller_pos2(int64_t e, int v, int t2, int nvt, int bs16) {
  if (!bs16) return (size_t(e) * nvt + v) * (NC / 2) + t2;
  const int c = int(e & 7), i = 2 * (t2 & 3), j = (t2 >> 2) & 7, k = t2 >> 5;
  const size_t row = ((size_t(e >> 3) * nvt + v) * 16 + 8 * (c >> 2) + k) * 16 + 8 * ((c >> 1) & 1) + j;
  return (row * 16 + 8 * (c & 1) + i) / 2;
}
// dst[slot][...] = src[perm[slot]][...] (to_internal) or the inverse, for slots [first, first+count)
// prim: the internal copy holds primitives (role 1); the caller's copy is always conserved
// ns: passive scalars per cell: the caller's blocks are [5 + ns][512], the internal hydro blocks [5][512]
cudaError_t launch_permute(const double* src, double* dst, const int64_t* perm, int first, int count, int to_internal,
                           int prim, double gamma, int ns, int bs16, cudaStream_t st);
cudaError_t launch_ghosted(const double* U, const double* ghost, const int32_t* face_src, const int64_t* perm,
                           int first, int count, int prim, double gamma, double* G, cudaStream_t st);
// per-block refinement indicator (criterion 0: eq. 33-34, 1: h / Jeans length) of slots [first, first+count), caller order
cudaError_t launch_refine_indicator(const double* U, const double* ghost, const int32_t* face_src, const int64_t* perm,
                                    int first, int count, int prim, double gamma, int criterion, double G, double h,
                                    double* out, cudaStream_t st);
// regrid: block d of the new mesh <- old slot tsrc[d] >= 0 (copy), prolongation from OLD parent -2 - tsrc[d]
// (tsrc[d] <= -2), or prolongation from its parent in the NEW mesh (tsrc[d] == -1; that parent was filled one level
// earlier by the same transfer).  The arrays are the hydro parts [.][5][512] or the scalar parts [.][ns][512].
struct TransferParams {
  const double* Uc;            // old buffer holding the block's own level (copies)
  const double* Us;            // old buffer holding the parent level
  const double* ghost_s;       // old mesh: coarse-fine slabs of that copy
  const int32_t* face_src_s;
  const double* Un;            // new buffer holding the parent level (or null at level 0)
  const double* ghost_n;       // new mesh: coarse-fine slabs
  const int32_t* face_src_n;
  const int32_t* parent_n;     // new mesh: parent slot per block of this launch
  const int32_t* tsrc;         // per block of this launch
  const int32_t* coord_d;
  double* Ud;                  // destination blocks of this launch
};
cudaError_t launch_transfer(const TransferParams& p, int count, cudaStream_t st);
cudaError_t configure_kernels(int* sm_count);

// ---- passive scalars (sfh_kernels_scalar.cu): Q[nb][ns][512] behind the hydro part of every state buffer ----------
struct ScalarStageParams {
  const double* Qsrc;    // scalars the stage differentiates: q^n (predictor) or q^{n+1/2} (corrector), conserved
  const double* Qn;      // q^n
  double* Qdst;          // q^{n+1/2} or q^{n+1}
  const double* Hsrc;    // hydro copy of the same state as Qsrc (variable 0 = rho in both its forms)
  const double* ghostH;  // its coarse-fine slabs
  const double* ghostS;  // coarse-fine slabs of Qsrc  [ncf][ns][128]
  const double* mf;      // mass fluxes written by the hydro stage  [blocks of the level][3][9][64], indexed by slot (shifted base)
  double* RS;            // fine-side scalar flux registers [ncf][ns][64]
  double* FHS;           // coarse-side                     [nfh][ns][64]
  const int32_t* face_src;
  const int32_t* fslot;
  const double* dt_dev;
  double dt, h;
  int first, count, ns;
};
struct ProlongScalarParams {
  const double *C0, *C1, *C2;   // scalar parts of the coarse level's copies (interp = 0: C0 only)
  double* ghost;
  double* ghost1;               // dual fill (interp only), or null
  const int32_t *cf_block, *cf_face, *parent, *coord, *nbr27;
  int first, count, ns, interp;
  double tau, tau1;
};
cudaError_t launch_scalar_stage(int stage, const ScalarStageParams& p, cudaStream_t st);
cudaError_t launch_prolong_scalar(const ProlongScalarParams& p, cudaStream_t st);
cudaError_t launch_restrict_scalar(const double* Qfine, double* Qcoarse, const int32_t* list, const int32_t* child0,
                                   int count, int ns, cudaStream_t st);
cudaError_t launch_reflux_scalar(double* Q, const double* RS, const double* FHS, const int32_t* list,
                                 const int32_t* fslot, const int32_t* fh_src, int count, int ns, double h, double dt,
                                 const double* dt_dev, cudaStream_t st);
cudaError_t launch_permute_scalar(const double* src, double* dst, const int64_t* perm, int first, int count, int ns,
                                  int to_internal, int bs16, cudaStream_t st);
cudaError_t launch_transfer_scalar(const TransferParams& p, int count, int ns, cudaStream_t st);
// fp64 issue-rate microbenchmark: `ctas` CTAs of 1024 threads, each thread `iters` x 16 x `chains` DFMAs
cudaError_t launch_dfma_rate(int chains, int ctas, int iters, double* sink, cudaStream_t st);

}  // namespace sfh

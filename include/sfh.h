/* sfh.h — C ABI of libsfh: the per-step hydrodynamics update on octree block-structured AMR grids
 * of arxiv/paper_2604_21438 (SFUMATO#), B200 (sm_100a) only.
 *
 * What the calls compute is defined by PAPER.md (cited per call as PAPER.md:<line>) and, where the
 * paper is silent, by the readings R1..R34 of DESIGN.md.  There is no CPU fallback: every call that
 * touches field data launches CUDA kernels on the caller's stream and returns SFH_ECUDA when no
 * device is usable.
 *
 * Conventions
 *   - Blocks: N^3 = 8^3 cells (16^3: see "Blocks of 16^3 cells" below); level l has cell width
 *     h_l = box_len[0] / (nb0[0]*8*2^l).  A block of level l has integer coordinates (bx,by,bz) in [0, nb0_d * 2^l);
 *     child c = cx + 2 cy + 4 cz of (bx,by,bz) is (2bx+cx, 2by+cy, 2bz+cz) at level l+1.
 *     EVERY block of every level holds data and is updated, covered (non-leaf) blocks too.
 *   - Conserved variables, in this order: rho, rho*vx, rho*vy, rho*vz, rho*E with
 *     rho*E = P/(gamma-1) + rho |v|^2 / 2 (eq. 1-3; eq. 8).  fp64.
 *   - Passive scalars (sfh_config.nscalar = NS > 0): conserved densities q = rho*s
 *     (y_i n_H of eq. 12, rho C_d T_d of eq. 13; source terms are not part of this
 *     path) follow the 5 hydro variables of every cell.  Their interface flux is the Riemann solver's
 *     mass flux times the interface value of s = q/rho on the side the mass comes from (cell-centred
 *     in the predictor, minmod-limited linear in the corrector; reading R32); ghost fill,
 *     eq. (16), restriction, flux registers and reflux treat them like the hydro variables.
 *   - "Caller layout" of a state: double U[nblocks][5 + NS][8][8][8], indexed [block][var][k][j][i]
 *     (i = x fastest), blocks in the order given to sfh_create_mesh, INTERIOR cells only.
 *   - Internal layout: interior-only blocks in the library's own order (level-major, Morton within
 *     a level); ghost values are never stored for same-level neighbours (the stage kernels gather
 *     them from the neighbours' interiors through the neighbour map); only ghost slabs on
 *     coarse-fine faces are materialised (in the work buffer) by sfh_fill_ghosts.
 *   - Three state copies ("roles"): 0 = U^n, 1 = U^{n+1/2}, 2 = U^{n+1} (values "at
 *     the current, previous, and half timesteps" are kept for temporal interpolation).  The library
 *     keeps role 1 as primitives (rho, v, P) internally; every copy crosses this interface as
 *     conserved variables.
 *   - Pointers: "host" = ordinary host memory, "device" = CUDA device memory of the current
 *     device.  `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls are
 *     asynchronous on that stream unless they return a host scalar (noted per call).
 *   - Ownership: the caller owns state and work buffers and the stream; the library owns the mesh
 *     tables (host and device).  A mesh is immutable after creation.
 *   - Errors: every int call returns SFH_OK (0) or a negative code; nothing throws or aborts
 *     across the ABI; sfh_last_error() returns a text for the calling thread's last failure.
 *     Non-positive density or pressure is reported by sfh_status, never floored (reading R28).
 */
#ifndef SFH_H_
#define SFH_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SFH_OK 0
#define SFH_EINVAL (-1) /* bad argument                                   */
#define SFH_EMESH (-2)  /* block list is not a valid, properly nested octree */
#define SFH_ENOMEM (-3) /* host or device allocation failed                */
#define SFH_ECUDA (-4)  /* CUDA runtime/driver error (text in sfh_last_error) */
#define SFH_ESTATE (-5) /* mesh not bound to state/work buffers            */

typedef struct sfh_mesh sfh_mesh; /* opaque, library-owned */

typedef struct {
  int32_t nb0[3];     /* root (level-0) blocks per axis */
  int32_t ncell;      /* cells per block edge: 8 or 16, see below */
  int32_t nghost;     /* ghost layers; only 2 is supported     */
  int32_t max_level;  /* finest level that may hold blocks (0 = uniform grid)                    */
  int32_t bc[3][2];   /* per axis, low/high face: 0 periodic, 1 outflow (zero gradient, R1)      */
  double box_len[3];  /* physical size; cells are cubes of h_0 = box_len[0]/(nb0[0]*8)           */
  double gamma;       /* ideal-gas exponent of eq. (8)      */
  double cfl;         /* CFL number used by sfh_cfl_dt / sfh_advance                             */
  int32_t nscalar;    /* passive scalars advected with the gas, 0..SFH_MAX_SCALARS   PAPER.md:80-88 (eq. 12-13) */
} sfh_config;
#define SFH_MAX_SCALARS 8

/* Blocks of 16^3 cells (ncell = 16; the paper's faster GPU variant, Table 5).
 * The scheme does not depend on how cells are grouped into blocks, and this library never stores ghost cells, so
 * the halo-to-interior argument for larger blocks does not apply to it: a 16^3 block (l; I, J, K) is handled as its
 * eight 8^3 octants (l; 2I + cx, 2J + cy, 2K + cz), octant c = cx + 2 cy + 4 cz, of a root grid of 2 nb0 blocks.
 * What changes is the CALLER'S layout: every state array that crosses this interface (sfh_set_state,
 * sfh_get_state, sfh_advance_host) is double [nblocks][5 + nscalar][16][16][16], and nb0, `level`, `ijk` of
 * sfh_create_mesh count 16^3 blocks.  Everything that is counted or indexed per block elsewhere in this header
 * (sfh_num_blocks, sfh_level_range, sfh_block_order, sfh_get_ghosted, sfh_refine_indicator, sfh_block_list, the
 * per-block arguments of sfh_regrid*) then refers to the octants: entry e = 8 * block + c.  A mesh that sfh_regrid
 * derives from a 16^3 mesh is a mesh of 8^3 blocks (refinement is decided per octant). */

/* ---- mesh: octree block table and neighbour map -------------------------- */

/* Builds the block table (level, coordinates, parent, first child), the 27-entry same-level
 * neighbour map, the per-face halo sources, and the flux-register maps on the HOST.  `level`
 * [nblocks] and `ijk` [nblocks][3] are host arrays.  Validates: levels/coordinates in range, no
 * duplicates, every block of level > 0 has its parent and all 7 siblings, and proper nesting over
 * all 26 neighbours (a neighbour position inside the domain holds a block of the same level or
 * its parent exists, reading R25); violations give SFH_EMESH.  Needs no GPU. */
int sfh_create_mesh(const sfh_config* cfg, int64_t nblocks, const int32_t* level, const int32_t* ijk,
                    sfh_mesh** out);
int sfh_destroy_mesh(sfh_mesh* m);

/* Riemann solver of the predictor and corrector fluxes: "either the HLLC scheme (Toro et al. 1994) or the
 * method of Roe (1981)".  SFH_RIEMANN_HLLC is the default (the paper's benchmarks use it,
 * PAPER.md:536); SFH_RIEMANN_ROE is Roe's linearised solver with Harten's entropy fix on the acoustic
 * waves (reading R30).  Host-side switch, takes effect at the next stage launch; any other
 * value gives SFH_EINVAL. */
#define SFH_RIEMANN_HLLC 0
#define SFH_RIEMANN_ROE 1
int sfh_set_riemann(sfh_mesh* m, int solver);

int64_t sfh_num_blocks(const sfh_mesh* m);
/* Blocks of `level` occupy library slots [first, first+count). */
int sfh_level_range(const sfh_mesh* m, int level, int64_t* first, int64_t* count);
/* perm[s] = caller index of the block stored in library slot s (host array [nblocks]). */
int sfh_block_order(const sfh_mesh* m, int64_t* perm);
/* Number of coarse-fine block faces (fine side; two ghost slabs -- of U^n and of the
 * half-step state -- and one flux register each) and of
 * coarse-leaf faces that receive a flux correction. */
int sfh_num_faces(const sfh_mesh* m, int64_t* n_fine_faces, int64_t* n_coarse_faces);
/* Cell width of a level. */
double sfh_cell_width(const sfh_mesh* m, int level);

/* Bytes of ONE state copy in the internal layout (hydro blocks, then the scalars' blocks), and of the
 * work buffer (coarse-fine ghost slabs, flux registers, per-block maximum speeds, reduction scratch;
 * with scalars also their slabs and registers and the mass fluxes of one stage). */
int64_t sfh_state_bytes(const sfh_mesh* m);
int64_t sfh_work_bytes(const sfh_mesh* m);

/* Attaches caller-owned DEVICE buffers (each state buffer >= sfh_state_bytes, work >=
 * sfh_work_bytes, all 256-byte aligned), uploads the mesh tables and creates the TMA tensor maps
 * of the three state buffers.  Synchronous.  The work buffer is zeroed. */
int sfh_bind(sfh_mesh* m, void* d_state0, void* d_state1, void* d_state2, void* d_work);

/* Copies a DEVICE state in caller layout into / out of role `which` (0,1,2) of every level.
 * sfh_get_state(which=0) after sfh_advance returns U at the new time. */
int sfh_set_state(sfh_mesh* m, int which, const double* d_U, void* stream);
int sfh_get_state(sfh_mesh* m, int which, double* d_U, void* stream);

/* ---- the hot path ------------------------------------------------------------------------------ */

/* Ghost fill of role `which` on `level` (-1: every level, coarse to fine).
 * Same-level ("sibling") ghosts and outflow ghosts are not stored: the hydro stage kernels gather
 * them.  This call computes the ghost slabs of every block face of the level whose neighbour is
 * one level coarser: slope-limited linear prolongation of the coarse data (reading R3), which are
 *   interp = 0: role `which` of level-1 (synchronous mode: both levels at the same time);
 *   interp = 1: the quadratic time interpolation of eq. (16)-(17) of roles
 *               0, 1, 2 of level-1 at tau = (t - t^n)/(t^{n+1} - t^n) of the COARSE step.
 * Asynchronous. */
int sfh_fill_ghosts(sfh_mesh* m, int level, int which, int interp, double tau, void* stream);

/* Writes ghosted blocks double G[nblocks][5][12][12][12] (caller block order, DEVICE; the 5 hydro
 * variables only) of role `which`: interiors, and the 6 face halos exactly as the stage kernels see them (same-level
 * gather, outflow copy, or the coarse-fine slabs last written by sfh_fill_ghosts); edge and
 * corner ghost cells, which no stage reads, are set to NaN.  For parity tests of the ghost fill. */
int sfh_get_ghosted(sfh_mesh* m, int which, double* d_G, void* stream);

/* Refinement indicators, one double per block in CALLER order to d_out (device,
 * [nblocks]); sfh_regrid thresholds them and builds the new mesh.
 *   SFH_REFINE_CURVATURE  eq. (33)-(34): max over the block's interior cells of
 *                         max(E(rho), E(P)), E(q) = |d2x q + d2y q + d2z q| h^2 / q with centred second
 *                         differences (the paper refines where this is >= 1e-2);
 *   SFH_REFINE_JEANS      PAPER.md:641: max over the cells of h / lambda_J, lambda_J = c_s sqrt(pi / (G rho))
 *                         (the paper refines where the Jeans length spans fewer than 8 cells: > 1/8).
 * Reads one ghost layer of state copy `which`: same-level and outflow halos are gathered, coarse-fine
 * halos are prolonged from the same copy of the coarser level first (the call refills the slabs of `which`
 * itself, as sfh_fill_ghosts(-1, which, 0, 0) would).  Asynchronous on `stream`.  SFH_EINVAL for an unknown criterion or G <= 0 with the Jeans criterion. */
#define SFH_REFINE_CURVATURE 0
#define SFH_REFINE_JEANS 1
int sfh_refine_indicator(sfh_mesh* m, int which, int criterion, double G, double* d_out, void* stream);

/* Regrid, step 1: builds the NEW mesh of a regrid from the
 * state of `m` (bound).  The refinement indicator of copy `which` (sfh_refine_indicator: criterion, G) is evaluated
 * on the device and brought to the host, where the library builds the new block list (the lists are
 * managed on the hosts):
 *   - every root block;
 *   - the 8 children of every block of level < max_level that is in `m`, is in the new tree, and is flagged: its
 *     indicator is >= threshold (eq. 33 is written with >=) or one of its descendants in `m` is flagged (a feature
 *     smaller than a coarse cell does not show in the restricted data of the blocks above it).  A regrid deepens the
 *     tree by at most one level anywhere and drops the children of blocks that are no longer flagged;
 *   - closed under proper nesting over the 26 neighbours (reading R25): missing blocks are added with their 7
 *     siblings and, recursively, their ancestors.
 * *out is a new, UNBOUND mesh with the same configuration and Riemann solver (destroy it with sfh_destroy_mesh); its
 * caller order is level-major, (bx, by, bz) lexicographic within a level (sfh_block_list).  The caller allocates its
 * buffers (sfh_state_bytes / sfh_work_bytes), binds it and moves the state with sfh_transfer_state.  Synchronises
 * `stream`. */
int sfh_regrid(sfh_mesh* m, int which, int criterion, double G, double threshold, sfh_mesh** out, void* stream);

/* The host half of sfh_regrid: the new mesh from an indicator the caller supplies (host array [nblocks], caller
 * order; any criterion of the caller's own), same rules.  Needs no GPU and no binding. */
int sfh_regrid_from_indicator(const sfh_mesh* m, const double* h_indicator, double threshold, sfh_mesh** out);

/* The block list of a mesh in caller order: level[nblocks], ijk[nblocks][3] (host arrays). */
int sfh_block_list(const sfh_mesh* m, int32_t* level, int32_t* ijk);

/* Regrid, step 2: fills state copy dst_which of the NEW mesh `dst` from copy src_which of the OLD
 * mesh `src` (both bound, same domain, same number of scalars): a block present in both is copied; a new block is
 * created from its parent by the slope-limited conservative prolongation of reading R3 (so restricting the new
 * children gives the parent back) -- from its parent in the old mesh where that exists, else from its parent in the
 * new mesh, which the same call created one level earlier (any number of new levels); blocks that disappear are
 * dropped (their parents hold the restricted data).  A new root block gives SFH_EMESH.  Only the conserved copies
 * (0 and 2).  Refills the old mesh's coarse-fine ghost slabs from src_which itself (the prolongation stencils of
 * new blocks next to an old coarse-fine face read them).
 * `dst` comes from sfh_regrid or from sfh_create_mesh.  Synchronous (it uploads a block map built on the host
 * into a table allocated at sfh_bind, and waits for the copy). */
int sfh_transfer_state(sfh_mesh* src, int src_which, sfh_mesh* dst, int dst_which, void* stream);

/* CFL time step (reading R16): dt = cfl * h_l / max over all cells of level l of
 * (max_d |v_d| + c_s), c_s = sqrt(gamma P / rho), from role 0; level = -1: minimum over levels
 * ("grid-level reductions").  Warp-shuffle + atomic-max reduction
 * (exact).  Returns the value in *dt_host: synchronises the stream.  SFH_ESTATE if the step is not finite and
 * positive (a level without a single finite positive speed: see sfh_status). */
int sfh_cfl_dt(sfh_mesh* m, int level, double* dt_host, void* stream);

/* The CFL step of ONE level without any allocation, for callers that cannot call cudaMalloc: a program whose
 * memory pool already owns the device (an allocation from inside this library would fail or fragment the pool), a
 * time-critical loop in which cudaMalloc / cudaFree would stall every stream of the device, a plug-in whose host
 * forbids allocations after start-up.  Such callers cannot use sfh_cfl_dt, because that needs a bound mesh and
 * sfh_bind allocates the device copy of the mesh tables.  This call needs no mesh:
 *   d_U      DEVICE, double [nblocks][5][8][8][8] ([block][var][k][j][i], the 5 hydro variables, conserved): the
 *            blocks of one level, any order; read only;
 *   h        cell width of that level; gamma, cfl as in sfh_config;
 *   d_out    DEVICE, double[2], written: d_out[0] = cfl * h / s, d_out[1] = s = max over all cells of
 *            max_d |v_d| + c_s (reading R16; the same arithmetic as sfh_cfl_dt).  Cells with a NaN speed
 *            are ignored as in sfh_cfl_dt; if no cell has a positive speed, s = 0 and d_out[0] = inf (this call cannot
 *            report that as SFH_ESTATE: it does not wait for the result).
 * The per-block maxima and the running maximum, which every other path keeps in the caller's work buffer, live in an
 * array built into the library image: SFH_NOALLOC_MAX_BLOCKS * 8 + 256 bytes (512.25 KB) of device memory on every
 * GPU that loads libsfh.so, held until the process exits.  nblocks > SFH_NOALLOC_MAX_BLOCKS gives SFH_EINVAL (use
 * sfh_cfl_dt with a work buffer of your own), as do nblocks < 1, null pointers, gamma <= 1, cfl <= 0, h <= 0.
 * The first call on each device looks up the array's device address (the device must be current, as for every call
 * here): make that first call before any stream capture.  All calls share the array and it keeps the previous
 * call's contents; each call clears what it needs on `stream` first, so calls on one stream (or ordered by events)
 * are independent, while calls that may run on the GPU at the same time -- two streams, two host threads --
 * race on it and return garbage.  Asynchronous on `stream`; calls no cudaMalloc, cudaFree or allocating routine. */
#define SFH_NOALLOC_MAX_BLOCKS 65536
int sfh_cfl_dt_noalloc(const double* d_U, int64_t nblocks, double gamma, double cfl, double h, double* d_out,
                       void* stream);

/* One predictor-corrector update of `level` (-1: every level) by dt   (R8-R14):
 *   zero the flux registers of the (level, level+1) interface;
 *   predictor: U^{n+1/2} = U^n - dt/(2h) sum_d dF_d, first-order HLLC fluxes      (role 0 -> 1);
 *   sfh_fill_ghosts(level, which=1, interp, tau + dtau/2);
 *   corrector: minmod-limited linear reconstruction of primitives of U^{n+1/2}, HLLC flux
 *              (PAPER.md:126), U^{n+1} = U^n - dt/h sum_d dF_d                    (roles 0,1 -> 2);
 *   flux-register accumulate: fine side += dt*F, coarse leaf side stores F.
 * The caller must have called sfh_fill_ghosts(level, 0, interp, tau) before.  tau = time fraction
 * of the start of this step within the parent-level step, dtau = dt/dt_parent (both ignored when
 * interp = 0).  Asynchronous.  Does not rotate the roles (see sfh_end_step). */
int sfh_hydro_step(sfh_mesh* m, int level, double dt, int interp, double tau, double dtau, void* stream);

/* Flux correction of `coarse_level` after level+1 has reached the same time:
 *   restriction: every covered cell of role 2 of coarse_level = mean of its 8 children (role 0 of
 *                level+1, i.e. after that level's sfh_end_step);
 *   reflux: each leaf cell of coarse_level on a coarse-fine face gets
 *           U -= (s/h) (1/4 sum_{2x2} R_fine - dt_coarse F_coarse), s = +1/-1 for its upper/lower face.
 * Fixed summation order, no floating-point atomics.  Asynchronous. */
int sfh_flux_correct(sfh_mesh* m, int coarse_level, double dt_coarse, void* stream);

/* Restriction alone (a8): covered cells of role `dst_role` of coarse_level = mean of the 8 children
 * in role `src_role` of coarse_level+1.  Used to make initial data consistent.  Asynchronous. */
int sfh_restrict(sfh_mesh* m, int coarse_level, int src_role, int dst_role, void* stream);

/* Ends the step of `level` (-1: all): role 0 <-> role 2 (U^n := U^{n+1}).  Host-side pointer
 * rotation, no data movement. */
int sfh_end_step(sfh_mesh* m, int level);

/* Level driver.  mode 0 = synchronous: all levels advance with a common dt =
 * dt_fixed if > 0 else the minimum CFL step over levels, computed on the device without a host
 * round trip.  mode 1 = adaptive: Berger-Colella recursion; the step of level l+1 is
 * dt_l 2^-n with n = min{m >= 0 : dt_l 2^-m <= dt_CFL^{l+1}} (eq. 14-15); level 0 uses dt_fixed if
 * > 0 else its CFL step.  Adds the elapsed time to *t_host and the number of updates of each level
 * to nupd_host[0..max_level] (either may be NULL).  Synchronises the stream before returning.  SFH_ESTATE if
 * a CFL step is not finite and positive or a level would need more than 2^20 sub-steps of its parent (both
 * mean the state holds bad cells, reading R28; the state is left as it was when that was detected). */
int sfh_advance(sfh_mesh* m, int ncoarse_steps, int mode, double dt_fixed, double* t_host,
                int64_t* nupd_host, void* stream);

/* End-to-end convenience: h_in (HOST, caller layout) -> device role 0, sfh_advance, role 0 -> h_out
 * (HOST).  Host buffers should be pinned for full PCIe speed.  t_host, nupd_host as in sfh_advance.
 * Synchronous. */
int sfh_advance_host(sfh_mesh* m, const double* h_in, double* h_out, int ncoarse_steps, int mode,
                     double dt_fixed, double* t_host, int64_t* nupd_host, void* stream);

/* Number of interior cells of role `which` with rho <= 0, P <= 0 or NaN (all blocks).  Synchronises. */
int sfh_status(sfh_mesh* m, int which, int64_t* n_bad_cells, void* stream);

/* Kernels launched by this library since the mesh was created (for bench.py's gpu_launches). */
int64_t sfh_launch_count(const sfh_mesh* m);

/* Per-kernel device timing for roofline reports.  While enabled, every launch of a hot-path kernel
 * is bracketed by two CUDA events on the caller's stream.  Kernel classes: 0 predictor stage (a4),
 * 1 corrector stage (a6+a7), 2 coarse-fine ghost prolongation (a3), 3 restriction (a8), 4 reflux
 * (a9), 5 CFL reduction (a10), 6 the passive-scalar kernels (stage, prolongation, restriction,
 * reflux).  sfh_kernel_times synchronises on the recorded events, ADDS the elapsed milliseconds and
 * launch counts since the last call to ms[7] / count[7] (host arrays) and forgets them. */
#define SFH_NUM_KERNEL_CLASSES 7
int sfh_profile(sfh_mesh* m, int enable);
int sfh_kernel_times(sfh_mesh* m, double* ms, int64_t* count);

/* Measurement support (bench.py's "alu" roofline denominator; SURVEY.md 8(d) "verify by microbenchmark"): the
 * rate at which this device issues fp64 fused multiply-adds, in thread-level DFMA instructions per second
 * (x2 = FLOP/s).  `chains` (1, 2, 4 or 8) independent dependent chains per thread, 2 CTAs of 1024 threads per
 * SM: 8 measures the pipe's peak, 1 the rate a fully dependent instruction stream reaches at full occupancy.
 * Best of three timed launches (CUDA events on `stream`).  Synchronous.  Needs no mesh. */
int sfh_measure_fp64_rate(int chains, double* dfma_per_second, void* stream);

const char* sfh_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SFH_H_ */

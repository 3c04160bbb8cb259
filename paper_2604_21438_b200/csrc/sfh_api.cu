// sfh_api.cu — the C ABI of libsfh (include/sfh.h): mesh handle, role rotation, level drivers.
// Every step of the hot path runs in the kernels of sfh_kernels*.cu; this file only sequences them.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <unordered_map>
#include <vector>

#include "sfh_kernels.cuh"

using namespace sfh;

namespace sfh {
static thread_local std::string g_err;
void set_error(const std::string& s) { g_err = s; }
}  // namespace sfh

struct sfh_mesh {
  HostMesh hm;
  bool bound = false;
  int sms = 1;                          // SM count of the device (persistent grids: one CTA per SM)
  int riemann = SFH_RIEMANN_HLLC;
  char* dev_tables = nullptr;
  int32_t *d_face_src = nullptr, *d_fslot = nullptr, *d_nbr27 = nullptr, *d_parent = nullptr, *d_child0 = nullptr,
          *d_coord = nullptr, *d_cf_block = nullptr, *d_cf_face = nullptr, *d_fh_src = nullptr,
          *d_restrict_list = nullptr, *d_reflux_list = nullptr;
  int64_t* d_perm = nullptr;
  int32_t* d_tsrc = nullptr;            // regrid: per block of THIS (new) mesh, where its data come from (sfh_transfer_state)
  double* d_ind = nullptr;              // regrid: refinement indicator per block, library order scratch (sfh_regrid)
  double* state[3] = {nullptr, nullptr, nullptr};
  double *ghost = nullptr, *ghost1 = nullptr, *R = nullptr, *FH = nullptr;   // ghost: slabs of U^n, ghost1: of U^{n+1/2}
  // passive scalars (ns = cfg.nscalar > 0): slabs of q^n / q^{n+1/2}, flux registers, the stage kernels' mass fluxes
  int ns = 0;
  double *ghostS = nullptr, *ghostS1 = nullptr, *RS = nullptr, *FHS = nullptr, *MF = nullptr;
  unsigned long long* smax = nullptr;   // [MAX_LEVELS] bit patterns of the per-level maximum speed
  double *dt_dev = nullptr, *t_dev = nullptr;
  unsigned long long* nbad = nullptr;
  // per-block maximum CFL speed: written by the corrector for U^{n+1} (role 2), rewritten by the restriction and
  // the reflux for the blocks they change.  pending[l]: the entries of level l describe its role-2 state;
  // valid[l]: they describe its role-0 state (after the rotation), so the CFL reduction need not re-read it.
  double* bmax = nullptr;
  bool bmax_pending[MAX_LEVELS] = {false}, bmax_valid[MAX_LEVELS] = {false};
  int role[MAX_LEVELS][3];              // role -> physical state buffer, per level
  TensorMaps tm[3];                     // per physical state buffer
  int64_t launches = 0;
  // eq. (15) needs the finer level's CFL step on the host once per parent step.  The reduction does not depend on the
  // parent's own update, so it is enqueued BEFORE the parent's stage kernels, copied to pinned memory, and the host
  // waits on an event that has long fired when it gets there: the device never idles for the round trip.
  unsigned long long* h_smax = nullptr;  // pinned, [MAX_LEVELS]
  cudaEvent_t ev_smax[MAX_LEVELS] = {nullptr};
  // optional per-kernel-class timing (sfh_profile / sfh_kernel_times)
  bool profiling = false;
  struct Span { int cls; cudaEvent_t a, b; };
  std::vector<Span> spans;
  std::vector<cudaEvent_t> event_pool;
};

namespace {

constexpr size_t ALIGN = 256;
inline size_t up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

struct WorkLayout {
  size_t ghost, R, FH, bmax, ghostS, RS, FHS, MF, scalars, total;
};
WorkLayout work_layout(const HostMesh& hm) {
  WorkLayout w;
  const size_t ncf = hm.cf_block.size(), ns = size_t(hm.cfg.nscalar);
  w.ghost = 0;
  w.R = up(w.ghost + 2 * ncf * SLAB * 8);      // two slab sets: the fill of U^n and of the half-step state
  w.FH = up(w.R + ncf * REG * 8);
  w.bmax = up(w.FH + size_t(hm.nfh) * REG * 8);
  w.ghostS = up(w.bmax + size_t(hm.nb) * 8);   // passive scalars: two slab sets, registers, mass fluxes
  w.RS = up(w.ghostS + 2 * ncf * ns * NG * FACE * 8);
  w.FHS = up(w.RS + ncf * ns * FACE * 8);
  w.MF = up(w.FHS + size_t(hm.nfh) * ns * FACE * 8);
  // mass fluxes of ONE stage of ONE level (consumed by the scalar kernel right after the stage that wrote them):
  // sized by the largest level, indexed by (slot - first slot of the level)
  int64_t widest = 0;
  for (int l = 0; l < hm.nlev; ++l) widest = hm.lev_count[l] > widest ? hm.lev_count[l] : widest;
  w.scalars = up(w.MF + (ns ? size_t(widest) * 3 * 9 * FACE * 8 : 0));
  w.total = w.scalars + 4096;
  return w;
}

int fail(int code, const std::string& what) {
  set_error(what);
  return code;
}
int cuda_fail(cudaError_t e, const char* where) {
  set_error(std::string(where) + ": " + cudaGetErrorString(e));
  return SFH_ECUDA;
}
#define CU(call, where)                                    \
  do {                                                     \
    cudaError_t e_ = (call);                               \
    if (e_ != cudaSuccess) return cuda_fail(e_, where);    \
  } while (0)

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// Tensor maps of one state buffer seen as a 4-D fp64 tensor [5*nb][8][8][8] (innermost = x): the
// two-layer x-face slab {2,8,8,5}; the two-layer y-face slab over the view with j and k exchanged
// (dimensions (i, k, j, var), box {8,8,2,5}) so that it lands as [var][ll][k][i]; and the z-plane pair.
int make_tensor_maps(void* base, int64_t nb, TensorMaps& out) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  CU(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres), "cudaGetDriverEntryPoint");
  if (!fn || qres != cudaDriverEntryPointSuccess) return fail(SFH_ECUDA, "cuTensorMapEncodeTiled not available");
  EncodeTiledFn encode = reinterpret_cast<EncodeTiledFn>(fn);
  const cuuint64_t nvb = cuuint64_t(NV) * cuuint64_t(nb);
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  CUresult r[3];
  {
    const cuuint64_t dims[4] = {N, N, N, nvb};
    const cuuint64_t strides[3] = {N * 8, N * N * 8, N * N * N * 8};
    const cuuint32_t box[4] = {NG, N, N, NV};
    r[0] = encode(&out.ax, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  }
  {
    const cuuint64_t dims[4] = {N, N, N, nvb};                        // (i, k, j, var)
    const cuuint64_t strides[3] = {N * N * 8, N * 8, N * N * N * 8};  // of k, j, var
    const cuuint32_t box[4] = {N, N, NG, NV};
    r[1] = encode(&out.ay, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  }
  {
    // 128-byte swizzle wants 128-byte rows (a 64-byte inner box would be padded to 128-byte lines,
    // measured): view two consecutive x rows (j, j+1) as one row of 16 doubles -> [5 nb][8][4][16]
    const cuuint64_t dims2[4] = {2 * N, N / 2, N, nvb};
    const cuuint64_t strides2[3] = {2 * N * 8, N * N * 8, N * N * N * 8};
    const cuuint32_t box2[4] = {2 * N, N / 2, NG, NV};
    r[2] = encode(&out.zs, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims2, strides2, box2, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  }
  for (int q = 0; q < 3; ++q)
    if (r[q] != CUDA_SUCCESS) {
      char buf[96];
      snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (map %d, CUresult %d)", q, int(r[q]));
      return fail(SFH_ECUDA, buf);
    }
  return SFH_OK;
}

inline cudaStream_t S(void* s) { return reinterpret_cast<cudaStream_t>(s); }

// Brackets one kernel launch with two events when profiling is on.
struct Timed {
  sfh_mesh* m;
  cudaStream_t st;
  cudaEvent_t a = nullptr, b = nullptr;
  int cls;
  static cudaEvent_t take(sfh_mesh* m) {
    cudaEvent_t e = nullptr;
    if (!m->event_pool.empty()) { e = m->event_pool.back(); m->event_pool.pop_back(); }
    else if (cudaEventCreate(&e) != cudaSuccess) e = nullptr;
    return e;
  }
  Timed(sfh_mesh* m_, int cls_, cudaStream_t st_) : m(m_), st(st_), cls(cls_) {
    if (!m->profiling) return;
    a = take(m);
    b = take(m);
    if (a) cudaEventRecord(a, st);
  }
  ~Timed() {
    if (!a || !b) return;
    cudaEventRecord(b, st);
    m->spans.push_back({cls, a, b});
  }
};
inline double* role_buf(const sfh_mesh* m, int l, int r) { return m->state[m->role[l][r]]; }
// scalar part of the same copy: Q[nb][ns][512] behind the hydro blocks
inline double* role_q(const sfh_mesh* m, int l, int r) { return m->state[m->role[l][r]] + size_t(m->hm.nb) * BLK; }

int check_bound(const sfh_mesh* m) {
  if (!m) return fail(SFH_EINVAL, "null mesh");
  if (!m->bound) return fail(SFH_ESTATE, "mesh is not bound to state/work buffers (sfh_bind)");
  return SFH_OK;
}
int check_level(const sfh_mesh* m, int level) {
  if (level < -1 || level >= m->hm.nlev) return fail(SFH_EINVAL, "level out of range");
  return SFH_OK;
}

struct Dt {   // a step known on the host, or to be read from device memory
  double host;
  const double* dev;
};

// which = 1 fills the half-step slabs (ghost1), else the U^n slabs.  dual (interp only): one gather fills both,
// the U^n slabs at tau and the half-step slabs at tau1.
int fill_level(sfh_mesh* m, int l, int which, int interp, double tau, cudaStream_t st, bool dual = false,
               double tau1 = 0.0) {
  const HostMesh& hm = m->hm;
  if (l == 0 || hm.cf_count[l] == 0) return SFH_OK;
  ProlongParams p;
  if (interp) { p.C0 = role_buf(m, l - 1, 0); p.C1 = role_buf(m, l - 1, 1); p.C2 = role_buf(m, l - 1, 2); }
  else { p.C0 = p.C1 = p.C2 = role_buf(m, l - 1, which); }
  p.ghost = which == 1 ? m->ghost1 : m->ghost;
  p.ghost1 = dual ? m->ghost1 : nullptr;
  p.tau1 = tau1;
  p.cf_block = m->d_cf_block; p.cf_face = m->d_cf_face; p.parent = m->d_parent; p.coord = m->d_coord;
  p.nbr27 = m->d_nbr27;
  p.first = int(hm.cf_first[l]); p.count = int(hm.cf_count[l]);
  p.interp = interp; p.tau = tau;
  // role 1 (the half-step state) is stored as primitives
  p.c0_prim = !interp && which == 1;
  p.c1_prim = 1;
  p.out_prim = which == 1;
  p.gamma = hm.cfg.gamma;
  {
    Timed tmr(m, 2, st);
    CU(launch_prolong(p, st), "prolong_kernel");
  }
  m->launches += 1;
  if (m->ns > 0) {      // the scalars' slabs: same gather, conserved values in every copy
    ProlongScalarParams q;
    if (interp) { q.C0 = role_q(m, l - 1, 0); q.C1 = role_q(m, l - 1, 1); q.C2 = role_q(m, l - 1, 2); }
    else { q.C0 = q.C1 = q.C2 = role_q(m, l - 1, which); }
    q.ghost = which == 1 ? m->ghostS1 : m->ghostS;
    q.ghost1 = dual ? m->ghostS1 : nullptr;
    q.cf_block = m->d_cf_block; q.cf_face = m->d_cf_face; q.parent = m->d_parent; q.coord = m->d_coord;
    q.nbr27 = m->d_nbr27;
    q.first = p.first; q.count = p.count; q.ns = m->ns; q.interp = interp; q.tau = tau; q.tau1 = tau1;
    Timed tmr(m, 6, st);
    CU(launch_prolong_scalar(q, st), "prolong_scalar_kernel");
    m->launches += 1;
  }
  return SFH_OK;
}

int stage_level(sfh_mesh* m, int l, int stage, Dt dt, cudaStream_t st) {
  const HostMesh& hm = m->hm;
  if (hm.lev_count[l] == 0) return SFH_OK;
  StageParams p;
  const int src_role = stage == 0 ? 0 : 1;
  p.Usrc = role_buf(m, l, src_role);
  p.Un = role_buf(m, l, 0);
  p.Udst = role_buf(m, l, stage == 0 ? 1 : 2);
  p.ghost = stage == 0 ? m->ghost : m->ghost1; p.R = m->R; p.FH = m->FH;
  p.face_src = m->d_face_src; p.fslot = m->d_fslot;
  p.dt_dev = dt.dev; p.dt = dt.host; p.h = hm.h[l]; p.gamma = hm.cfg.gamma;
  p.first = int(hm.lev_first[l]); p.count = int(hm.lev_count[l]);
  p.use_regs = stage == 1 && (hm.cf_count[l] > 0 || hm.reflux_count[l] > 0);
  p.riemann = m->riemann;
  p.bmax = stage == 1 ? m->bmax : nullptr;
  // the kernels index the mass fluxes by slot: shift the base so that the level's first block lands at MF[0]
  double* const mf_level = m->ns > 0 ? m->MF - size_t(hm.lev_first[l]) * (3 * 9 * FACE) : nullptr;
  p.mf = mf_level;
  // the corrector overwrites the level's cached maxima with those of U^{n+1}: they stop describing U^n now
  if (stage == 1) { m->bmax_pending[l] = true; m->bmax_valid[l] = false; }
  {
    Timed tmr(m, stage, st);
    CU(launch_stage(stage, m->tm[m->role[l][src_role]], p, m->sms, st), "stage_kernel");
  }
  m->launches += 1;
  if (m->ns > 0) {      // the scalars ride on the mass fluxes the stage has just exported
    ScalarStageParams q;
    q.Qsrc = role_q(m, l, src_role); q.Qn = role_q(m, l, 0); q.Qdst = role_q(m, l, stage == 0 ? 1 : 2);
    q.Hsrc = p.Usrc; q.ghostH = p.ghost; q.ghostS = stage == 0 ? m->ghostS : m->ghostS1; q.mf = mf_level;
    q.RS = m->RS; q.FHS = m->FHS; q.face_src = m->d_face_src; q.fslot = m->d_fslot;
    q.dt_dev = dt.dev; q.dt = dt.host; q.h = hm.h[l]; q.first = p.first; q.count = p.count; q.ns = m->ns;
    Timed tmr(m, 6, st);
    CU(launch_scalar_stage(stage, q, st), "scalar_stage_kernel");
    m->launches += 1;
  }
  return SFH_OK;
}

int zero_fine_registers(sfh_mesh* m, int coarse_level, cudaStream_t st) {   // registers of (l, l+1)
  const HostMesh& hm = m->hm;
  const int lf = coarse_level + 1;
  if (lf >= hm.nlev || hm.cf_count[lf] == 0) return SFH_OK;
  CU(cudaMemsetAsync(m->R + size_t(hm.cf_first[lf]) * REG, 0, size_t(hm.cf_count[lf]) * REG * 8, st), "memset R");
  if (m->ns > 0)
    CU(cudaMemsetAsync(m->RS + size_t(hm.cf_first[lf]) * m->ns * FACE, 0, size_t(hm.cf_count[lf]) * m->ns * FACE * 8, st),
       "memset RS");
  return SFH_OK;
}

int hydro_level(sfh_mesh* m, int l, Dt dt, int interp, double tau, double dtau, cudaStream_t st,
                bool half_filled = false) {
  int rc;
  if ((rc = zero_fine_registers(m, l, st))) return rc;
  if ((rc = stage_level(m, l, 0, dt, st))) return rc;
  if (!half_filled && (rc = fill_level(m, l, 1, interp, tau + 0.5 * dtau, st))) return rc;
  return stage_level(m, l, 1, dt, st);
}

int flux_correct_level(sfh_mesh* m, int lc, Dt dt, cudaStream_t st) {
  const HostMesh& hm = m->hm;
  if (lc + 1 >= hm.nlev || hm.lev_count[lc + 1] == 0) return SFH_OK;
  m->bmax_valid[lc] = false;      // restriction and reflux rewrite entries with the maxima of role 2
  {
    Timed tmr(m, 3, st);
    CU(launch_restrict(role_buf(m, lc + 1, 0), role_buf(m, lc, 2), m->d_restrict_list + hm.restrict_first[lc],
                       m->d_child0, int(hm.restrict_count[lc]), hm.cfg.gamma, m->bmax, st), "restrict_kernel");
  }
  m->launches += hm.restrict_count[lc] > 0;
  {
    Timed tmr(m, 4, st);
    CU(launch_reflux(role_buf(m, lc, 2), m->R, m->FH, m->d_reflux_list + hm.reflux_first[lc], m->d_fslot,
                     m->d_fh_src, int(hm.reflux_count[lc]), hm.h[lc], dt.host, dt.dev, hm.cfg.gamma, m->bmax, st),
       "reflux_kernel");
  }
  m->launches += hm.reflux_count[lc] > 0;
  if (m->ns > 0) {
    Timed tmr(m, 6, st);
    CU(launch_restrict_scalar(role_q(m, lc + 1, 0), role_q(m, lc, 2), m->d_restrict_list + hm.restrict_first[lc],
                              m->d_child0, int(hm.restrict_count[lc]), m->ns, st), "restrict_scalar_kernel");
    CU(launch_reflux_scalar(role_q(m, lc, 2), m->RS, m->FHS, m->d_reflux_list + hm.reflux_first[lc], m->d_fslot,
                            m->d_fh_src, int(hm.reflux_count[lc]), m->ns, hm.h[lc], dt.host, dt.dev, st),
       "reflux_scalar_kernel");
    m->launches += (hm.restrict_count[lc] > 0) + (hm.reflux_count[lc] > 0);
  }
  return SFH_OK;
}

void rotate(sfh_mesh* m, int l) {
  std::swap(m->role[l][0], m->role[l][2]);
  m->bmax_valid[l] = m->bmax_pending[l];     // the old U^n becomes scratch
  m->bmax_pending[l] = false;
}

int max_speed_level(sfh_mesh* m, int l, cudaStream_t st) {
  const HostMesh& hm = m->hm;
  Timed tmr(m, 5, st);
  if (m->bmax_valid[l])
    CU(launch_max_cached(m->bmax, int(hm.lev_first[l]), int(hm.lev_count[l]), m->smax + l, m->sms, st),
       "max_cached_kernel");
  else
    CU(launch_max_speed(role_buf(m, l, 0), int(hm.lev_first[l]), int(hm.lev_count[l]), hm.cfg.gamma, m->smax + l,
                        m->sms, st), "max_speed_kernel");
  m->launches += hm.lev_count[l] > 0;
  return SFH_OK;
}

int cfl_host(sfh_mesh* m, int level, double* dt_out, cudaStream_t st) {
  const HostMesh& hm = m->hm;
  int rc;
  for (int l = 0; l < hm.nlev; ++l)
    if ((level < 0 || level == l) && (rc = max_speed_level(m, l, st))) return rc;
  unsigned long long bits[MAX_LEVELS];
  CU(cudaMemcpyAsync(bits, m->smax, sizeof bits, cudaMemcpyDeviceToHost, st), "memcpy smax");
  CU(cudaStreamSynchronize(st), "cudaStreamSynchronize");
  double dt = INFINITY;
  for (int l = 0; l < hm.nlev; ++l)
    if ((level < 0 || level == l) && hm.lev_count[l] > 0) {
      double s;
      std::memcpy(&s, &bits[l], 8);
      const double dtl = hm.cfg.cfl * hm.h[l] / s;
      // a NaN speed never wins the device's max (R28: bad cells are reported, not floored), so s = 0 or inf here
      // means the level holds no finite positive speed at all
      if (!(dtl > 0.0) || !std::isfinite(dtl)) {
        char buf[128];
        snprintf(buf, sizeof buf, "CFL step of level %d is not finite and positive (max speed %g): bad cells? (sfh_status)", l, s);
        return fail(SFH_ESTATE, buf);
      }
      dt = std::fmin(dt, dtl);
    }
  *dt_out = dt;
  return SFH_OK;
}

// The CFL step of level l in two halves: request (reduction + copy to pinned memory + event, all on the stream) and
// fetch (wait for the event, form the step).  Between the two the caller may enqueue work that does not change role 0
// of level l.
int cfl_request(sfh_mesh* m, int l, cudaStream_t st) {
  int rc;
  if (!m->h_smax) {
    CU(cudaHostAlloc(reinterpret_cast<void**>(&m->h_smax), sizeof(unsigned long long) * MAX_LEVELS, cudaHostAllocDefault),
       "cudaHostAlloc");
  }
  if (!m->ev_smax[l]) CU(cudaEventCreateWithFlags(&m->ev_smax[l], cudaEventDisableTiming), "cudaEventCreate");
  if ((rc = max_speed_level(m, l, st))) return rc;
  CU(cudaMemcpyAsync(m->h_smax + l, m->smax + l, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st), "memcpy smax");
  CU(cudaEventRecord(m->ev_smax[l], st), "cudaEventRecord");
  return SFH_OK;
}
int cfl_fetch(sfh_mesh* m, int l, double* dt_out) {
  CU(cudaEventSynchronize(m->ev_smax[l]), "cudaEventSynchronize");
  double s;
  std::memcpy(&s, m->h_smax + l, 8);
  const double dtl = m->hm.cfg.cfl * m->hm.h[l] / s;
  if (!(dtl > 0.0) || !std::isfinite(dtl)) {
    char buf[128];
    snprintf(buf, sizeof buf, "CFL step of level %d is not finite and positive (max speed %g): bad cells? (sfh_status)", l, s);
    return fail(SFH_ESTATE, buf);
  }
  *dt_out = dtl;
  return SFH_OK;
}

// eq. (14)-(15): smallest n >= 0 with dtH 2^-n <= dt_cfl (reading R18)
constexpr int MAX_SUBSTEP_EXPONENT = 20;   // 2^20 sub-steps of one parent step: beyond any sane hierarchy
int substep_exponent(double dtH, double dt_cfl) {
  int n = 0;
  while (n <= MAX_SUBSTEP_EXPONENT && std::ldexp(dtH, -n) > dt_cfl) ++n;
  return n;
}

int advance_adaptive(sfh_mesh* m, int l, double dt, double tau, double dtau, int64_t* nupd, cudaStream_t st) {
  const HostMesh& hm = m->hm;
  const int interp = l > 0;
  int rc;
  // the coarser level has finished its step: its three time copies give both ghost fills in one gather
  const bool has_finer = l + 1 < hm.nlev && hm.lev_count[l + 1] > 0;
  // the finer level's CFL step (for eq. 15 below) does not depend on this level's update: ask for it first
  if (has_finer && (rc = cfl_request(m, l + 1, st))) return rc;
  if ((rc = fill_level(m, l, 0, interp, tau, st, interp != 0, tau + 0.5 * dtau))) return rc;
  if ((rc = hydro_level(m, l, Dt{dt, nullptr}, interp, tau, dtau, st, interp != 0))) return rc;
  if (nupd) nupd[l] += 1;
  if (has_finer) {
    double dtc;
    if ((rc = cfl_fetch(m, l + 1, &dtc))) return rc;
    const int n = substep_exponent(dt, dtc);
    if (n > MAX_SUBSTEP_EXPONENT) {
      char buf[160];
      snprintf(buf, sizeof buf, "level %d would need more than 2^%d sub-steps of its parent (dt %g, CFL step %g): bad cells?",
               l + 1, MAX_SUBSTEP_EXPONENT, dt, dtc);
      return fail(SFH_ESTATE, buf);
    }
    const double dtf = std::ldexp(dt, -n);
    const int nsub = 1 << n;
    for (int s = 0; s < nsub; ++s)
      if ((rc = advance_adaptive(m, l + 1, dtf, double(s) / double(nsub), dtf / dt, nupd, st))) return rc;
    if ((rc = flux_correct_level(m, l, Dt{dt, nullptr}, st))) return rc;
  }
  rotate(m, l);
  return SFH_OK;
}

int step_sync(sfh_mesh* m, double dt_fixed, cudaStream_t st) {
  const HostMesh& hm = m->hm;
  int rc;
  Dt dt{dt_fixed, nullptr};
  if (!(dt_fixed > 0.0)) {
    LevelInfo li;
    li.nlev = hm.nlev;
    for (int l = 0; l < hm.nlev; ++l) {
      li.h[l] = hm.h[l];
      li.has[l] = hm.lev_count[l] > 0;
      if ((rc = max_speed_level(m, l, st))) return rc;
    }
    CU(launch_dt_finalize(m->smax, li, hm.cfg.cfl, m->dt_dev, m->t_dev, st), "dt_finalize_kernel");
    m->launches += 1;
    dt = Dt{0.0, m->dt_dev};
  }
  for (int l = 0; l < hm.nlev; ++l) if ((rc = zero_fine_registers(m, l, st))) return rc;
  for (int l = 0; l < hm.nlev; ++l) if ((rc = fill_level(m, l, 0, 0, 0.0, st))) return rc;
  for (int l = 0; l < hm.nlev; ++l) if ((rc = stage_level(m, l, 0, dt, st))) return rc;
  for (int l = 0; l < hm.nlev; ++l) if ((rc = fill_level(m, l, 1, 0, 0.0, st))) return rc;
  for (int l = 0; l < hm.nlev; ++l) if ((rc = stage_level(m, l, 1, dt, st))) return rc;
  for (int l = hm.nlev - 1; l >= 0; --l) {
    if ((rc = flux_correct_level(m, l, dt, st))) return rc;
    rotate(m, l);
  }
  return SFH_OK;
}

}  // namespace

// =====================================================================================================
extern "C" {

const char* sfh_last_error(void) { return g_err.c_str(); }

int sfh_create_mesh(const sfh_config* cfg, int64_t nblocks, const int32_t* level, const int32_t* ijk,
                    sfh_mesh** out) {
  if (!cfg || !out) return fail(SFH_EINVAL, "null argument");
  *out = nullptr;
  sfh_mesh* m = new (std::nothrow) sfh_mesh;
  if (!m) return fail(SFH_ENOMEM, "out of host memory");
  std::string err;
  int rc;
  try {
    rc = build_host_mesh(*cfg, nblocks, level, ijk, m->hm, err);
  } catch (const std::bad_alloc&) {
    delete m;
    return fail(SFH_ENOMEM, "out of host memory");
  }
  if (rc != SFH_OK) {
    delete m;
    return fail(rc, err);
  }
  for (int l = 0; l < MAX_LEVELS; ++l) for (int r = 0; r < 3; ++r) m->role[l][r] = r;
  m->ns = cfg->nscalar;
  *out = m;
  return SFH_OK;
}

int sfh_destroy_mesh(sfh_mesh* m) {
  if (!m) return SFH_OK;
  for (auto& sp : m->spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
  for (cudaEvent_t e : m->event_pool) cudaEventDestroy(e);
  for (cudaEvent_t e : m->ev_smax) if (e) cudaEventDestroy(e);
  if (m->h_smax) cudaFreeHost(m->h_smax);
  if (m->dev_tables) cudaFree(m->dev_tables);
  delete m;
  return SFH_OK;
}

int sfh_set_riemann(sfh_mesh* m, int solver) {
  if (!m) return fail(SFH_EINVAL, "null mesh");
  if (solver != SFH_RIEMANN_HLLC && solver != SFH_RIEMANN_ROE) return fail(SFH_EINVAL, "unknown Riemann solver");
  m->riemann = solver;
  return SFH_OK;
}

int64_t sfh_num_blocks(const sfh_mesh* m) { return m ? m->hm.nb : 0; }

int sfh_level_range(const sfh_mesh* m, int level, int64_t* first, int64_t* count) {
  if (!m || level < 0 || level >= m->hm.nlev) return fail(SFH_EINVAL, "level out of range");
  if (first) *first = m->hm.lev_first[level];
  if (count) *count = m->hm.lev_count[level];
  return SFH_OK;
}

int sfh_block_order(const sfh_mesh* m, int64_t* perm) {
  if (!m || !perm) return fail(SFH_EINVAL, "null argument");
  std::memcpy(perm, m->hm.perm.data(), sizeof(int64_t) * size_t(m->hm.nb));
  return SFH_OK;
}

int sfh_num_faces(const sfh_mesh* m, int64_t* n_fine_faces, int64_t* n_coarse_faces) {
  if (!m) return fail(SFH_EINVAL, "null mesh");
  if (n_fine_faces) *n_fine_faces = int64_t(m->hm.cf_block.size());
  if (n_coarse_faces) *n_coarse_faces = m->hm.nfh;
  return SFH_OK;
}

double sfh_cell_width(const sfh_mesh* m, int level) {
  if (!m || level < 0 || level >= m->hm.nlev) return 0.0;
  return m->hm.h[level];
}

int64_t sfh_state_bytes(const sfh_mesh* m) { return m ? int64_t(up(size_t(m->hm.nb) * (NV + m->ns) * NC * 8)) : 0; }
int64_t sfh_work_bytes(const sfh_mesh* m) { return m ? int64_t(work_layout(m->hm).total) : 0; }
int64_t sfh_launch_count(const sfh_mesh* m) { return m ? m->launches : 0; }

int sfh_bind(sfh_mesh* m, void* d_state0, void* d_state1, void* d_state2, void* d_work) {
  if (!m || !d_state0 || !d_state1 || !d_state2 || !d_work) return fail(SFH_EINVAL, "null argument");
  void* ptrs[4] = {d_state0, d_state1, d_state2, d_work};
  for (void* p : ptrs)
    if (reinterpret_cast<uintptr_t>(p) % ALIGN) return fail(SFH_EINVAL, "buffers must be 256-byte aligned");
  int ndev = 0;
  CU(cudaGetDeviceCount(&ndev), "cudaGetDeviceCount");
  if (ndev == 0) return fail(SFH_ECUDA, "no CUDA device");
  const HostMesh& hm = m->hm;
  if (!m->dev_tables) {
    // one allocation for all tables
    struct Item { const void* src; size_t bytes; void** dst; };
    const Item items[] = {
        {hm.face_src.data(), hm.face_src.size() * 4, (void**)&m->d_face_src},
        {hm.fslot.data(), hm.fslot.size() * 4, (void**)&m->d_fslot},
        {hm.nbr27.data(), hm.nbr27.size() * 4, (void**)&m->d_nbr27},
        {hm.parent.data(), hm.parent.size() * 4, (void**)&m->d_parent},
        {hm.child0.data(), hm.child0.size() * 4, (void**)&m->d_child0},
        {hm.coord.data(), hm.coord.size() * 4, (void**)&m->d_coord},
        {hm.cf_block.data(), hm.cf_block.size() * 4, (void**)&m->d_cf_block},
        {hm.cf_face.data(), hm.cf_face.size() * 4, (void**)&m->d_cf_face},
        {hm.fh_src.data(), hm.fh_src.size() * 4, (void**)&m->d_fh_src},
        {hm.restrict_list.data(), hm.restrict_list.size() * 4, (void**)&m->d_restrict_list},
        {hm.reflux_list.data(), hm.reflux_list.size() * 4, (void**)&m->d_reflux_list},
        {hm.perm.data(), hm.perm.size() * 8, (void**)&m->d_perm},
        {nullptr, size_t(hm.nb) * 4, (void**)&m->d_tsrc},
        {nullptr, size_t(hm.nb) * 8, (void**)&m->d_ind},
    };
    size_t total = 0;
    for (const Item& it : items) total += up(it.bytes + 1);
    cudaError_t e = cudaMalloc((void**)&m->dev_tables, total);
    if (e != cudaSuccess) { m->dev_tables = nullptr; set_error("cudaMalloc of mesh tables failed"); return SFH_ENOMEM; }
    size_t off = 0;
    for (const Item& it : items) {
      *it.dst = m->dev_tables + off;
      if (it.bytes && it.src) e = cudaMemcpy(m->dev_tables + off, it.src, it.bytes, cudaMemcpyHostToDevice);
      if (e != cudaSuccess) break;
      off += up(it.bytes + 1);
    }
    if (e == cudaSuccess) e = configure_kernels(&m->sms);
    if (e != cudaSuccess) {          // never keep half-uploaded tables: the next sfh_bind starts over
      cudaFree(m->dev_tables);
      m->dev_tables = nullptr;
      return cuda_fail(e, "upload of the mesh tables / kernel configuration");
    }
  }
  m->state[0] = static_cast<double*>(d_state0);
  m->state[1] = static_cast<double*>(d_state1);
  m->state[2] = static_cast<double*>(d_state2);
  const WorkLayout w = work_layout(hm);
  char* wb = static_cast<char*>(d_work);
  CU(cudaMemset(wb, 0, w.total), "zero work buffer");
  m->ghost = reinterpret_cast<double*>(wb + w.ghost);
  m->ghost1 = m->ghost + hm.cf_block.size() * SLAB;
  m->R = reinterpret_cast<double*>(wb + w.R);
  m->FH = reinterpret_cast<double*>(wb + w.FH);
  m->bmax = reinterpret_cast<double*>(wb + w.bmax);
  m->ghostS = reinterpret_cast<double*>(wb + w.ghostS);
  m->ghostS1 = m->ghostS + hm.cf_block.size() * size_t(m->ns) * NG * FACE;
  m->RS = reinterpret_cast<double*>(wb + w.RS);
  m->FHS = reinterpret_cast<double*>(wb + w.FHS);
  m->MF = reinterpret_cast<double*>(wb + w.MF);
  for (int l = 0; l < MAX_LEVELS; ++l) m->bmax_pending[l] = m->bmax_valid[l] = false;
  m->smax = reinterpret_cast<unsigned long long*>(wb + w.scalars);
  m->dt_dev = reinterpret_cast<double*>(wb + w.scalars + 256);
  m->t_dev = reinterpret_cast<double*>(wb + w.scalars + 512);
  m->nbad = reinterpret_cast<unsigned long long*>(wb + w.scalars + 768);
  for (int b = 0; b < 3; ++b) {
    const int rc = make_tensor_maps(m->state[b], hm.nb, m->tm[b]);
    if (rc) return rc;
  }
  for (int l = 0; l < MAX_LEVELS; ++l) for (int r = 0; r < 3; ++r) m->role[l][r] = r;
  // the uploads and the memset above ran on the legacy stream: the caller's (non-blocking) streams see them done
  CU(cudaDeviceSynchronize(), "cudaDeviceSynchronize");
  m->bound = true;
  return SFH_OK;
}

int sfh_set_state(sfh_mesh* m, int which, const double* d_U, void* stream) {
  int rc = check_bound(m);
  if (rc) return rc;
  if (which < 0 || which > 2 || !d_U) return fail(SFH_EINVAL, "bad argument");
  for (int l = 0; l < m->hm.nlev; ++l) {
    if (which == 0) m->bmax_valid[l] = false;
    if (which == 2) m->bmax_pending[l] = false;
    CU(launch_permute(d_U, role_buf(m, l, which), m->d_perm, int(m->hm.lev_first[l]), int(m->hm.lev_count[l]), 1,
                      which == 1, m->hm.cfg.gamma, m->ns, m->hm.bs16, S(stream)), "permute_kernel");
    CU(launch_permute_scalar(d_U, role_q(m, l, which), m->d_perm, int(m->hm.lev_first[l]), int(m->hm.lev_count[l]),
                             m->ns, 1, m->hm.bs16, S(stream)), "permute_scalar_kernel");
    m->launches += (m->hm.lev_count[l] > 0) * (1 + (m->ns > 0));
  }
  return SFH_OK;
}

int sfh_get_state(sfh_mesh* m, int which, double* d_U, void* stream) {
  int rc = check_bound(m);
  if (rc) return rc;
  if (which < 0 || which > 2 || !d_U) return fail(SFH_EINVAL, "bad argument");
  for (int l = 0; l < m->hm.nlev; ++l) {
    CU(launch_permute(role_buf(m, l, which), d_U, m->d_perm, int(m->hm.lev_first[l]), int(m->hm.lev_count[l]), 0,
                      which == 1, m->hm.cfg.gamma, m->ns, m->hm.bs16, S(stream)), "permute_kernel");
    CU(launch_permute_scalar(role_q(m, l, which), d_U, m->d_perm, int(m->hm.lev_first[l]), int(m->hm.lev_count[l]),
                             m->ns, 0, m->hm.bs16, S(stream)), "permute_scalar_kernel");
    m->launches += (m->hm.lev_count[l] > 0) * (1 + (m->ns > 0));
  }
  return SFH_OK;
}

int sfh_fill_ghosts(sfh_mesh* m, int level, int which, int interp, double tau, void* stream) {
  int rc = check_bound(m);
  if (rc || (rc = check_level(m, level))) return rc;
  if (which < 0 || which > 2) return fail(SFH_EINVAL, "which must be 0, 1 or 2");
  for (int l = 0; l < m->hm.nlev; ++l)
    if ((level < 0 || level == l) && (rc = fill_level(m, l, which, interp, tau, S(stream)))) return rc;
  return SFH_OK;
}

int sfh_get_ghosted(sfh_mesh* m, int which, double* d_G, void* stream) {
  int rc = check_bound(m);
  if (rc) return rc;
  if (which < 0 || which > 2 || !d_G) return fail(SFH_EINVAL, "bad argument");
  for (int l = 0; l < m->hm.nlev; ++l) {
    CU(launch_ghosted(role_buf(m, l, which), which == 1 ? m->ghost1 : m->ghost, m->d_face_src, m->d_perm, int(m->hm.lev_first[l]),
                      int(m->hm.lev_count[l]), which == 1, m->hm.cfg.gamma, d_G, S(stream)), "ghosted_kernel");
    m->launches += m->hm.lev_count[l] > 0;
  }
  return SFH_OK;
}

int sfh_refine_indicator(sfh_mesh* m, int which, int criterion, double G, double* d_out, void* stream) {
  int rc = check_bound(m);
  if (rc) return rc;
  if (which < 0 || which > 2 || !d_out) return fail(SFH_EINVAL, "bad argument");
  if (criterion != SFH_REFINE_CURVATURE && criterion != SFH_REFINE_JEANS) return fail(SFH_EINVAL, "unknown criterion");
  if (criterion == SFH_REFINE_JEANS && !(G > 0.0)) return fail(SFH_EINVAL, "G must be positive");
  // the coarse-fine slabs may hold anything (time-interpolated values of the last sub-step): refill them
  for (int l = 1; l < m->hm.nlev; ++l)
    if ((rc = fill_level(m, l, which, 0, 0.0, S(stream)))) return rc;
  for (int l = 0; l < m->hm.nlev; ++l) {
    CU(launch_refine_indicator(role_buf(m, l, which), which == 1 ? m->ghost1 : m->ghost, m->d_face_src, m->d_perm,
                               int(m->hm.lev_first[l]), int(m->hm.lev_count[l]), which == 1, m->hm.cfg.gamma, criterion,
                               G, m->hm.h[l], d_out, S(stream)), "refine_indicator_kernel");
    m->launches += m->hm.lev_count[l] > 0;
  }
  return SFH_OK;
}

int sfh_transfer_state(sfh_mesh* src, int src_which, sfh_mesh* dst, int dst_which, void* stream) {
  int rc = check_bound(src);
  if (rc || (rc = check_bound(dst))) return rc;
  if ((src_which != 0 && src_which != 2) || (dst_which != 0 && dst_which != 2))
    return fail(SFH_EINVAL, "state transfer works on the conserved copies (roles 0 and 2)");
  const HostMesh &hs = src->hm, &hd = dst->hm;
  for (int d = 0; d < 3; ++d)
    if (hs.cfg.nb0[d] != hd.cfg.nb0[d] || hs.cfg.bc[d][0] != hd.cfg.bc[d][0] || hs.cfg.bc[d][1] != hd.cfg.bc[d][1] ||
        hs.cfg.box_len[d] != hd.cfg.box_len[d])
      return fail(SFH_EINVAL, "the two meshes describe different domains");
  if (src->ns != dst->ns) return fail(SFH_EINVAL, "the two meshes carry different numbers of passive scalars");
  auto key = [](int l, const int32_t* c) {
    return (uint64_t(l) << 60) | (uint64_t(uint32_t(c[0]) & 0xFFFFF) << 40) | (uint64_t(uint32_t(c[1]) & 0xFFFFF) << 20) |
           uint64_t(uint32_t(c[2]) & 0xFFFFF);
  };
  // tsrc[b] of new block b: >= 0 copy of old slot; <= -2 prolongation from OLD parent slot -2 - tsrc; -1 prolongation
  // from its parent in the NEW mesh (a block more than one level below anything the old mesh holds there: the parent
  // was itself created by this transfer, one level earlier)
  std::vector<int32_t> tsrc;
  std::vector<char> from_new(size_t(hd.nlev), 0);
  try {
    std::unordered_map<uint64_t, int32_t> old;
    old.reserve(size_t(hs.nb) * 2);
    for (int64_t b = 0; b < hs.nb; ++b) old.emplace(key(hs.lev[b], &hs.coord[3 * b]), int32_t(b));
    tsrc.resize(size_t(hd.nb));
    for (int64_t b = 0; b < hd.nb; ++b) {
      const int l = hd.lev[b];
      auto it = old.find(key(l, &hd.coord[3 * b]));
      if (it != old.end()) { tsrc[b] = it->second; continue; }
      const int32_t pc[3] = {hd.coord[3 * b] >> 1, hd.coord[3 * b + 1] >> 1, hd.coord[3 * b + 2] >> 1};
      it = l > 0 ? old.find(key(l - 1, pc)) : old.end();
      if (it != old.end()) { tsrc[b] = -2 - it->second; continue; }
      if (l == 0) return fail(SFH_EMESH, "a root block of the new mesh is not in the old mesh");
      tsrc[b] = -1;
      from_new[size_t(l)] = 1;
    }
  } catch (const std::bad_alloc&) {
    return fail(SFH_ENOMEM, "out of host memory");
  }
  cudaStream_t st = S(stream);
  // the prolongation stencils read the old mesh's coarse-fine slabs: refill them from src_which
  for (int l = 1; l < hs.nlev; ++l)
    if ((rc = fill_level(src, l, src_which, 0, 0.0, st))) return rc;
  CU(cudaMemcpyAsync(dst->d_tsrc, tsrc.data(), tsrc.size() * 4, cudaMemcpyHostToDevice, st), "upload of the transfer table");
  // a new block of level l reads old level l (copy), old level l-1 (prolongation) or new level l-1; the roles rotate
  // per level, so these may sit in different physical buffers
  for (int l = 0; l < hd.nlev; ++l) {
    const int lc = l < hs.nlev ? l : hs.nlev - 1, lp = l > 0 ? (l - 1 < hs.nlev ? l - 1 : hs.nlev - 1) : 0;
    const int64_t first = hd.lev_first[l], count = hd.lev_count[l];
    if (from_new[size_t(l)] && (rc = fill_level(dst, l - 1, dst_which, 0, 0.0, st))) return rc;   // slabs of the new parents
    TransferParams tp;
    tp.Uc = role_buf(src, lc, src_which); tp.Us = role_buf(src, lp, src_which); tp.ghost_s = src->ghost;
    tp.face_src_s = src->d_face_src;
    tp.Un = l > 0 ? role_buf(dst, l - 1, dst_which) : nullptr; tp.ghost_n = dst->ghost; tp.face_src_n = dst->d_face_src;
    tp.parent_n = dst->d_parent + first;
    tp.tsrc = dst->d_tsrc + first; tp.coord_d = dst->d_coord + 3 * first;
    tp.Ud = role_buf(dst, l, dst_which) + size_t(first) * BLK;
    CU(launch_transfer(tp, int(count), st), "transfer_kernel");
    if (dst->ns > 0) {
      tp.Uc = role_q(src, lc, src_which); tp.Us = role_q(src, lp, src_which); tp.ghost_s = src->ghostS;
      tp.Un = l > 0 ? role_q(dst, l - 1, dst_which) : nullptr; tp.ghost_n = dst->ghostS;
      tp.Ud = role_q(dst, l, dst_which) + size_t(first) * dst->ns * NC;
      CU(launch_transfer_scalar(tp, int(count), dst->ns, st), "transfer_scalar_kernel");
    }
    dst->launches += (count > 0) * (1 + (dst->ns > 0));
  }
  CU(cudaStreamSynchronize(st), "cudaStreamSynchronize");      // tsrc (host vector) must outlive the upload
  for (int l = 0; l < hd.nlev; ++l) {
    if (dst_which == 0) dst->bmax_valid[l] = false;
    else dst->bmax_pending[l] = false;
  }
  return SFH_OK;
}

int sfh_regrid(sfh_mesh* m, int which, int criterion, double G, double threshold, sfh_mesh** out, void* stream) {
  if (!out) return fail(SFH_EINVAL, "null argument");
  *out = nullptr;
  int rc = check_bound(m);
  if (rc) return rc;
  const HostMesh& hm = m->hm;
  std::vector<double> ind(size_t(hm.nb));
  if ((rc = sfh_refine_indicator(m, which, criterion, G, m->d_ind, stream))) return rc;       // caller order
  CU(cudaMemcpyAsync(ind.data(), m->d_ind, ind.size() * 8, cudaMemcpyDeviceToHost, S(stream)), "download of the indicator");
  CU(cudaStreamSynchronize(S(stream)), "cudaStreamSynchronize");
  return sfh_regrid_from_indicator(m, ind.data(), threshold, out);
}

int sfh_regrid_from_indicator(const sfh_mesh* m, const double* h_indicator, double threshold, sfh_mesh** out) {
  if (!m || !h_indicator || !out) return fail(SFH_EINVAL, "null argument");
  *out = nullptr;
  const HostMesh& hm = m->hm;
  std::vector<int32_t> level, ijk;
  int rc;
  try {
    std::vector<double> ind_slot(size_t(hm.nb));      // caller order -> library order
    for (int64_t s = 0; s < hm.nb; ++s) ind_slot[size_t(s)] = h_indicator[size_t(hm.perm[size_t(s)])];
    if ((rc = regrid_block_list(hm, ind_slot.data(), threshold, level, ijk))) return rc;
  } catch (const std::bad_alloc&) {
    return fail(SFH_ENOMEM, "out of host memory");
  }
  sfh_mesh* nm = nullptr;
  if ((rc = sfh_create_mesh(&hm.cfg, int64_t(level.size()), level.data(), ijk.data(), &nm))) return rc;
  nm->riemann = m->riemann;
  *out = nm;
  return SFH_OK;
}

int sfh_block_list(const sfh_mesh* m, int32_t* level, int32_t* ijk) {
  if (!m || !level || !ijk) return fail(SFH_EINVAL, "null argument");
  const HostMesh& hm = m->hm;
  for (int64_t s = 0; s < hm.nb; ++s) {
    const int64_t b = hm.perm[size_t(s)];
    level[b] = hm.lev[size_t(s)];
    for (int d = 0; d < 3; ++d) ijk[3 * b + d] = hm.coord[size_t(3 * s + d)];
  }
  return SFH_OK;
}

int sfh_cfl_dt(sfh_mesh* m, int level, double* dt_host, void* stream) {
  int rc = check_bound(m);
  if (rc || (rc = check_level(m, level))) return rc;
  if (!dt_host) return fail(SFH_EINVAL, "null dt_host");
  return cfl_host(m, level, dt_host, S(stream));
}

int sfh_hydro_step(sfh_mesh* m, int level, double dt, int interp, double tau, double dtau, void* stream) {
  int rc = check_bound(m);
  if (rc || (rc = check_level(m, level))) return rc;
  if (!(dt > 0.0)) return fail(SFH_EINVAL, "dt must be positive");
  const Dt d{dt, nullptr};
  cudaStream_t st = S(stream);
  if (level >= 0) return hydro_level(m, level, d, interp, tau, dtau, st);
  // all levels, stage by stage (synchronous mode)
  for (int l = 0; l < m->hm.nlev; ++l) if ((rc = zero_fine_registers(m, l, st))) return rc;
  for (int l = 0; l < m->hm.nlev; ++l) if ((rc = stage_level(m, l, 0, d, st))) return rc;
  for (int l = 0; l < m->hm.nlev; ++l) if ((rc = fill_level(m, l, 1, interp, tau + 0.5 * dtau, st))) return rc;
  for (int l = 0; l < m->hm.nlev; ++l) if ((rc = stage_level(m, l, 1, d, st))) return rc;
  return SFH_OK;
}

int sfh_flux_correct(sfh_mesh* m, int coarse_level, double dt_coarse, void* stream) {
  int rc = check_bound(m);
  if (rc) return rc;
  if (coarse_level < 0 || coarse_level >= m->hm.nlev) return fail(SFH_EINVAL, "level out of range");
  return flux_correct_level(m, coarse_level, Dt{dt_coarse, nullptr}, S(stream));
}

int sfh_restrict(sfh_mesh* m, int coarse_level, int src_role, int dst_role, void* stream) {
  int rc = check_bound(m);
  if (rc) return rc;
  const HostMesh& hm = m->hm;
  if (coarse_level < 0 || coarse_level >= hm.nlev || src_role < 0 || src_role > 2 || dst_role < 0 || dst_role > 2)
    return fail(SFH_EINVAL, "bad argument");
  if (src_role == 1 || dst_role == 1)
    return fail(SFH_EINVAL, "the half-step state (role 1) is never restricted (DESIGN.md reading R10)");
  if (coarse_level + 1 >= hm.nlev || hm.restrict_count[coarse_level] == 0) return SFH_OK;
  // the cached block maxima follow a restriction into U^{n+1} (role 2); one into U^n invalidates them
  m->bmax_valid[coarse_level] = false;     // (into role 2: the entries are rewritten with role-2 maxima)
  CU(launch_restrict(role_buf(m, coarse_level + 1, src_role), role_buf(m, coarse_level, dst_role),
                     m->d_restrict_list + hm.restrict_first[coarse_level], m->d_child0,
                     int(hm.restrict_count[coarse_level]), hm.cfg.gamma, dst_role == 2 ? m->bmax : nullptr, S(stream)),
     "restrict_kernel");
  CU(launch_restrict_scalar(role_q(m, coarse_level + 1, src_role), role_q(m, coarse_level, dst_role),
                            m->d_restrict_list + hm.restrict_first[coarse_level], m->d_child0,
                            int(hm.restrict_count[coarse_level]), m->ns, S(stream)), "restrict_scalar_kernel");
  m->launches += 1 + (m->ns > 0);
  return SFH_OK;
}

int sfh_end_step(sfh_mesh* m, int level) {
  int rc = check_bound(m);
  if (rc || (rc = check_level(m, level))) return rc;
  for (int l = 0; l < m->hm.nlev; ++l) if (level < 0 || level == l) rotate(m, l);
  return SFH_OK;
}

int sfh_advance(sfh_mesh* m, int ncoarse_steps, int mode, double dt_fixed, double* t_host, int64_t* nupd_host,
                void* stream) {
  int rc = check_bound(m);
  if (rc) return rc;
  if (ncoarse_steps < 0 || (mode != 0 && mode != 1)) return fail(SFH_EINVAL, "bad argument");
  cudaStream_t st = S(stream);
  const HostMesh& hm = m->hm;
  double t = 0.0;
  if (mode == 0) {
    CU(cudaMemsetAsync(m->t_dev, 0, 8, st), "memset t");
    for (int s = 0; s < ncoarse_steps; ++s) {
      if ((rc = step_sync(m, dt_fixed, st))) return rc;
      if (dt_fixed > 0.0) t += dt_fixed;
      if (nupd_host) for (int l = 0; l < hm.nlev; ++l) nupd_host[l] += hm.lev_count[l] > 0;
    }
    double tdev = 0.0;
    CU(cudaMemcpyAsync(&tdev, m->t_dev, 8, cudaMemcpyDeviceToHost, st), "memcpy t");
    CU(cudaStreamSynchronize(st), "cudaStreamSynchronize");
    t += tdev;
  } else {
    for (int s = 0; s < ncoarse_steps; ++s) {
      double dt = dt_fixed;
      if (!(dt > 0.0) && (rc = cfl_host(m, 0, &dt, st))) return rc;
      if ((rc = advance_adaptive(m, 0, dt, 0.0, 0.0, nupd_host, st))) return rc;
      t += dt;
    }
    CU(cudaStreamSynchronize(st), "cudaStreamSynchronize");
  }
  if (t_host) *t_host += t;
  return SFH_OK;
}

int sfh_advance_host(sfh_mesh* m, const double* h_in, double* h_out, int ncoarse_steps, int mode, double dt_fixed,
                     double* t_host, int64_t* nupd_host, void* stream) {
  int rc = check_bound(m);
  if (rc) return rc;
  if (!h_in || !h_out) return fail(SFH_EINVAL, "null host buffer");
  cudaStream_t st = S(stream);
  const size_t bytes = size_t(m->hm.nb) * (NV + m->ns) * NC * 8;
  // role 1 (U^{n+1/2}) of level 0 is scratch between steps: use its buffer for staging in caller order
  double* stage = m->state[m->role[0][1]];
  for (int l = 1; l < m->hm.nlev; ++l)
    if (m->role[l][1] != m->role[0][1]) return fail(SFH_ESTATE, "internal: role 1 buffers differ between levels");
  CU(cudaMemcpyAsync(stage, h_in, bytes, cudaMemcpyHostToDevice, st), "H2D");
  if ((rc = sfh_set_state(m, 0, stage, stream))) return rc;
  if ((rc = sfh_advance(m, ncoarse_steps, mode, dt_fixed, t_host, nupd_host, stream))) return rc;
  if ((rc = sfh_get_state(m, 0, stage, stream))) return rc;
  CU(cudaMemcpyAsync(h_out, stage, bytes, cudaMemcpyDeviceToHost, st), "D2H");
  CU(cudaStreamSynchronize(st), "cudaStreamSynchronize");
  return SFH_OK;
}

int sfh_profile(sfh_mesh* m, int enable) {
  if (!m) return fail(SFH_EINVAL, "null mesh");
  m->profiling = enable != 0;
  return SFH_OK;
}

int sfh_kernel_times(sfh_mesh* m, double* ms, int64_t* count) {
  if (!m || !ms || !count) return fail(SFH_EINVAL, "null argument");
  for (auto& sp : m->spans) {
    CU(cudaEventSynchronize(sp.b), "cudaEventSynchronize");
    float t = 0.f;
    CU(cudaEventElapsedTime(&t, sp.a, sp.b), "cudaEventElapsedTime");
    ms[sp.cls] += double(t);
    count[sp.cls] += 1;
    m->event_pool.push_back(sp.a);
    m->event_pool.push_back(sp.b);
  }
  m->spans.clear();
  return SFH_OK;
}

int sfh_measure_fp64_rate(int chains, double* dfma_per_second, void* stream) {
  if (!dfma_per_second || (chains != 1 && chains != 2 && chains != 4 && chains != 8))
    return fail(SFH_EINVAL, "chains must be 1, 2, 4 or 8");
  int dev = 0, sms = 0;
  CU(cudaGetDevice(&dev), "cudaGetDevice");
  CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute");
  cudaStream_t st = S(stream);
  double* sink = nullptr;
  if (cudaMalloc((void**)&sink, 8) != cudaSuccess) return fail(SFH_ENOMEM, "cudaMalloc failed");
  cudaEvent_t a = nullptr, b = nullptr;
  cudaError_t e = cudaEventCreate(&a);
  if (e == cudaSuccess) e = cudaEventCreate(&b);
  const int ctas = 2 * sms, iters = 4096;
  double best = 0.0;
  for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {        // the first launch warms up
    cudaEventRecord(a, st);
    e = launch_dfma_rate(chains, ctas, iters, sink, st);
    cudaEventRecord(b, st);
    if (e == cudaSuccess) e = cudaEventSynchronize(b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    const double rate = double(ctas) * 1024.0 * iters * 16.0 * chains / (double(ms) * 1e-3);
    if (rep > 0 && rate > best) best = rate;
  }
  if (a) cudaEventDestroy(a);
  if (b) cudaEventDestroy(b);
  cudaFree(sink);
  if (e != cudaSuccess) return cuda_fail(e, "dfma_rate_kernel");
  *dfma_per_second = best;
  return SFH_OK;
}

int sfh_status(sfh_mesh* m, int which, int64_t* n_bad_cells, void* stream) {
  int rc = check_bound(m);
  if (rc) return rc;
  if (which < 0 || which > 2 || !n_bad_cells) return fail(SFH_EINVAL, "bad argument");
  cudaStream_t st = S(stream);
  CU(cudaMemsetAsync(m->nbad, 0, 8, st), "memset");
  for (int l = 0; l < m->hm.nlev; ++l) {
    CU(launch_count_bad(role_buf(m, l, which), int(m->hm.lev_first[l]), int(m->hm.lev_count[l]), m->hm.cfg.gamma,
                        which == 1, m->nbad, m->sms, st), "count_bad_kernel");
    m->launches += m->hm.lev_count[l] > 0;
  }
  unsigned long long n = 0;
  CU(cudaMemcpyAsync(&n, m->nbad, 8, cudaMemcpyDeviceToHost, st), "memcpy");
  CU(cudaStreamSynchronize(st), "cudaStreamSynchronize");
  *n_bad_cells = int64_t(n);
  return SFH_OK;
}

}  // extern "C"

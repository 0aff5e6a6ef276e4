// mhd_api.cu -- the C ABI of include/mhd.h: solver object, slice scheduling, kernel dispatch, stream-overlapped
// host path.  No CPU fallback anywhere: every entry point that computes needs a CUDA device.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/mhd.h"
#include "mhd_kernels3.cuh"

using namespace mhd;

namespace {

thread_local std::string g_cuda_err = "no CUDA error recorded";

inline int cuda_fail(cudaError_t e, const char* where) {
  g_cuda_err = std::string(where) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? MHD_ENOMEM : MHD_ECUDA;
}
#define CU(call)                                         \
  do {                                                   \
    cudaError_t e_ = (call);                             \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);  \
  } while (0)

constexpr int kMaxStreams = 8;

struct HostLane {            // one stream of mhd_advance_host with its staging buffers and workspace
  cudaStream_t stream = nullptr;
  void *Ui = nullptr, *Bi = nullptr, *Uo = nullptr, *Bo = nullptr, *fo = nullptr, *eo = nullptr, *ws = nullptr;
};

}  // namespace

struct mhd_solver {
  mhd_config cfg;
  int N, g, T, S, narr;
  size_t esz;                               // bytes per element
  size_t nUi, nBi, nUo, nBo, nF, nE;        // elements per group
  size_t S3;
  int slice_groups;                         // groups whose working set is kept L2-resident per sweep of the stages
  void* ws = nullptr;                       // slice_groups * narr * S3 elements
  unsigned long long* d_stats = nullptr;    // 3 counters
  unsigned long long* d_red = nullptr;      // dt reduction cell
  unsigned long long launches = 0;
  HostLane lanes[kMaxStreams];
  int lane_groups = 0, lane_count = 0;
  // optional per-stage timing (mhd_set_profiling): pairs of events around every stage launch
  bool prof_on = false;
  std::vector<cudaEvent_t> prof_ev;         // 2 per recorded launch
  std::vector<int> prof_stage;              // stage id per recorded launch
  size_t prof_used = 0;
};

namespace {

template <class R>
KParams<R> make_params(const mhd_solver* s, const void* Ui, const void* Bi, void* Uo, void* Bo, void* fo, void* eo,
                       void* ws, int first, double dt, double dh) {
  KParams<R> p;
  p.Uin = static_cast<const R*>(Ui) + (size_t)first * s->nUi;
  p.Bin = static_cast<const R*>(Bi) + (size_t)first * s->nBi;
  p.Uout = static_cast<R*>(Uo) + (size_t)first * s->nUo;
  p.Bout = static_cast<R*>(Bo) + (size_t)first * s->nBo;
  p.fout = fo ? static_cast<R*>(fo) + (size_t)first * s->nF : nullptr;
  p.eout = eo ? static_cast<R*>(eo) + (size_t)first * s->nE : nullptr;
  p.ws = static_cast<R*>(ws);
  p.stats = s->d_stats;
  p.N = s->N; p.g = s->g; p.T = s->T; p.S = s->S; p.S2 = s->S * s->S; p.S3 = (int)s->S3; p.narr = s->narr;
  p.nUi = (long long)s->nUi; p.nBi = (long long)s->nBi; p.nUo = (long long)s->nUo; p.nBo = (long long)s->nBo;
  p.nF = (long long)s->nF; p.nE = (long long)s->nE;
  p.gam = (R)s->cfg.gamma; p.gm1 = (R)(s->cfg.gamma - 1.0); p.gm1inv = (R)(1.0 / (s->cfg.gamma - 1.0));
  p.dt = (R)dt; p.dh = (R)dh; p.min_dens = (R)s->cfg.min_dens; p.min_pres = (R)s->cfg.min_pres;
  p.tie = (R)(s->cfg.emf_tie * dh / dt);
  return p;
}

#define SOLVER_SWITCH(sol, CALL)          \
  switch (sol) {                           \
    case MHD_HLLE: { constexpr int SOLVER = kHLLE; CALL; } break; \
    case MHD_HLLD: { constexpr int SOLVER = kHLLD; CALL; } break; \
    default:       { constexpr int SOLVER = kROE;  CALL; } break; \
  }

enum Stage : int { ST_LOAD = 0, ST_RECON, ST_FLUX1, ST_EMF1, ST_HALF, ST_CORR, ST_FLUX2, ST_EMF2, ST_FINAL, ST_PLANES, ST_DT, ST_COUNT };
const char* const kStageNames[ST_COUNT] = { "load_prim", "recon_ctu", "flux_pass1", "emf_pass1", "half_step", "ctu_corr",
                                            "flux_pass2", "emf_pass2", "final_update", "planes", "dt_reduce" };
constexpr size_t kProfMaxLaunches = 16384;

inline void prof_begin(mhd_solver* s, int stage, cudaStream_t st) {
  if (!s->prof_on || s->prof_used >= kProfMaxLaunches) return;
  if (s->prof_ev.size() < 2 * (s->prof_used + 1)) {
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    s->prof_ev.push_back(a); s->prof_ev.push_back(b); s->prof_stage.push_back(stage);
  }
  s->prof_stage[s->prof_used] = stage;
  cudaEventRecord(s->prof_ev[2 * s->prof_used], st);
}
inline void prof_end(mhd_solver* s, cudaStream_t st) {
  if (!s->prof_on || s->prof_used >= kProfMaxLaunches) return;
  cudaEventRecord(s->prof_ev[2 * s->prof_used + 1], st);
  s->prof_used++;
}
#define LAUNCH(stage, ...)        \
  do {                            \
    prof_begin(s, stage, st);     \
    __VA_ARGS__;                  \
    prof_end(s, st);              \
    s->launches++;                \
  } while (0)

// all stages of one slice of groups, in the paper's step order
template <class R>
int run_slice(mhd_solver* s, const KParams<R>& p, int ng, cudaStream_t st) {
  const int TPB = 256;
  const dim3 blk(TPB);
  const unsigned nb = (unsigned)((s->S3 + TPB - 1) / TPB);
  const dim3 g1(nb, 1, ng), g3(nb, 3, ng);
  const int T = s->T, sol = s->cfg.riemann, lim = s->cfg.limvar;
  LAUNCH(ST_LOAD, (k_load_prim<R><<<g1, blk, 0, st>>>(p)));
  if (s->cfg.scheme == MHD_VL) {
    LAUNCH(ST_FLUX1, SOLVER_SWITCH(sol, (k_flux1_vl<R, SOLVER><<<g3, blk, 0, st>>>(p))));          // step 1
    LAUNCH(ST_EMF1, (k_emf<R><<<g1, blk, 0, st>>>(p, A_W, 1, T - 1, 0, T)));                       // step 2
    LAUNCH(ST_HALF, (k_half<R><<<g1, blk, 0, st>>>(p, 1, T - 1)));                                 // step 3
    if (lim == MHD_LIM_PRIM) LAUNCH(ST_FLUX2, SOLVER_SWITCH(sol, (k_flux2_vl<R, SOLVER, kLimPrim><<<g3, blk, 0, st>>>(p))));
    else LAUNCH(ST_FLUX2, SOLVER_SWITCH(sol, (k_flux2_vl<R, SOLVER, kLimChar><<<g3, blk, 0, st>>>(p))));   // steps 4+5
    LAUNCH(ST_EMF2, (k_emf<R><<<g1, blk, 0, st>>>(p, A_WH, 3, T - 3, 1, T - 1)));                  // step 6
  } else {
    const int r = s->cfg.recon == MHD_PLM ? 1 : 2;
    if (s->cfg.recon == MHD_PLM) {
      if (lim == MHD_LIM_PRIM) LAUNCH(ST_RECON, (k_recon_ctu<R, kPLM, kLimPrim><<<g3, blk, 0, st>>>(p)));
      else LAUNCH(ST_RECON, (k_recon_ctu<R, kPLM, kLimChar><<<g3, blk, 0, st>>>(p)));
    } else {
      if (lim == MHD_LIM_PRIM) LAUNCH(ST_RECON, (k_recon_ctu<R, kPPM, kLimPrim><<<g3, blk, 0, st>>>(p)));
      else LAUNCH(ST_RECON, (k_recon_ctu<R, kPPM, kLimChar><<<g3, blk, 0, st>>>(p)));
    }                                                                                              // step 1
    LAUNCH(ST_FLUX1, SOLVER_SWITCH(sol, (k_flux_lr<R, SOLVER><<<g3, blk, 0, st>>>(p, A_B, r + 1, T - r, 0, T))));   // step 2
    LAUNCH(ST_EMF1, (k_emf<R><<<g1, blk, 0, st>>>(p, A_W, r + 1, T - 1 - r, 0, T)));               // step 3
    LAUNCH(ST_HALF, (k_half<R><<<g1, blk, 0, st>>>(p, r + 1, T - 1 - r)));                         // step 4
    LAUNCH(ST_CORR, (k_ctu_corr<R><<<g3, blk, 0, st>>>(p, r)));                                    // step 5
    LAUNCH(ST_FLUX2, SOLVER_SWITCH(sol, (k_flux_lr<R, SOLVER><<<g3, blk, 0, st>>>(p, A_BH, r + 1, T - r, r + 1, T - 1 - r))));  // step 6
    LAUNCH(ST_EMF2, (k_emf<R><<<g1, blk, 0, st>>>(p, A_WH, r + 2, T - 2 - r, r + 1, T - 1 - r)));  // step 7
  }
  LAUNCH(ST_FINAL, (k_final<R><<<g1, blk, 0, st>>>(p)));                                           // step 7 / 8
  if (p.fout || p.eout) {
    const int M = s->N + 1;
    LAUNCH(ST_PLANES, (k_planes<R><<<dim3((9 * M * M + TPB - 1) / TPB, 1, ng), blk, 0, st>>>(p)));
  }
  CU(cudaGetLastError());
  return MHD_OK;
}

template <class R>
int advance_dev(mhd_solver* s, const void* Ui, const void* Bi, void* Uo, void* Bo, void* fo, void* eo, void* ws,
                int ngroups, double dt, double dh, cudaStream_t st) {
  for (int first = 0; first < ngroups; first += s->slice_groups) {
    const int ng = std::min(s->slice_groups, ngroups - first);
    KParams<R> p = make_params<R>(s, Ui, Bi, Uo, Bo, fo, eo, ws, first, dt, dh);
    int rc = run_slice<R>(s, p, ng, st);
    if (rc != MHD_OK) return rc;
  }
  return MHD_OK;
}

int check_config(const mhd_config* c) {
  if (!c) return MHD_EINVAL;
  if (c->ps2 < 8 || c->ps2 > 64 || (c->ps2 & 1)) return MHD_EINVAL;
  if (c->scheme != MHD_VL && c->scheme != MHD_CTU) return MHD_EINVAL;
  if (c->recon != MHD_PLM && c->recon != MHD_PPM) return MHD_EINVAL;
  if (c->riemann < MHD_HLLE || c->riemann > MHD_ROE) return MHD_EINVAL;
  if (c->limvar != MHD_LIM_PRIM && c->limvar != MHD_LIM_CHAR) return MHD_EINVAL;
  if (c->prec != MHD_FP32 && c->prec != MHD_FP64) return MHD_EINVAL;
  if (c->scheme == MHD_VL && c->recon == MHD_PPM) return MHD_EINVAL;
  const int need = c->recon == MHD_PPM ? 4 : 3;     // DESIGN.md R8
  if (c->nghost < need || c->nghost > 8) return MHD_EINVAL;
  if (!(c->gamma > 1.0) || !std::isfinite(c->gamma)) return MHD_EINVAL;
  if (!(c->min_dens >= 0.0) || !(c->min_pres >= 0.0)) return MHD_EINVAL;
  if (c->max_groups < 1 || c->device < 0) return MHD_EINVAL;
  return MHD_OK;
}

}  // namespace

extern "C" {

int mhd_create(const mhd_config* cfg, mhd_solver** out) {
  if (!out) return MHD_EINVAL;
  *out = nullptr;
  int rc = check_config(cfg);
  if (rc != MHD_OK) return rc;
  int ndev = 0;
  CU(cudaGetDeviceCount(&ndev));
  if (cfg->device >= ndev) return MHD_EINVAL;
  CU(cudaSetDevice(cfg->device));
  mhd_solver* s = new (std::nothrow) mhd_solver();
  if (!s) return MHD_ENOMEM;
  s->cfg = *cfg;
  if (!(s->cfg.emf_tie > 0.0)) s->cfg.emf_tie = cfg->prec == MHD_FP32 ? 1e-5 : 1e-12;
  s->N = cfg->ps2; s->g = cfg->nghost; s->T = s->N + 2 * s->g; s->S = s->T + 1;
  s->S3 = (size_t)s->S * s->S * s->S;
  s->narr = cfg->scheme == MHD_VL ? A_VL_END : A_CTU_END;
  s->esz = cfg->prec == MHD_FP32 ? 4 : 8;
  const size_t N = s->N, T = s->T;
  s->nUi = 5 * T * T * T; s->nBi = 3 * T * T * (T + 1);
  s->nUo = 5 * N * N * N; s->nBo = 3 * N * N * (N + 1);
  s->nF = 9 * 5 * N * N; s->nE = 9 * 2 * (N + 1) * N;
  // slice = as many groups as keep workspace + their input and output inside a budget well below the 126 MB L2
  double budget_mb = 72.0;
  if (const char* e = getenv("MHD_SLICE_MB")) { double v = atof(e); if (v > 0) budget_mb = v; }
  const size_t per_group = ((size_t)s->narr * s->S3 + s->nUi + s->nBi + s->nUo + s->nBo + s->nF + s->nE) * s->esz;
  long sg = (long)(budget_mb * 1048576.0 / (double)per_group);
  if (const char* e = getenv("MHD_SLICE_GROUPS")) { long v = atol(e); if (v > 0) sg = v; }
  if (sg < 1) sg = 1;
  if (sg > cfg->max_groups) sg = cfg->max_groups;
  s->slice_groups = (int)sg;
  cudaError_t e = cudaMalloc(&s->ws, (size_t)s->slice_groups * s->narr * s->S3 * s->esz);
  if (e == cudaSuccess) e = cudaMalloc((void**)&s->d_stats, 4 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMemset(s->d_stats, 0, 4 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMemset(s->ws, 0, (size_t)s->slice_groups * s->narr * s->S3 * s->esz);
  if (e != cudaSuccess) { int r = cuda_fail(e, "mhd_create allocation"); mhd_destroy(s); return r; }
  s->d_red = s->d_stats + 3;
  *out = s;
  return MHD_OK;
}

static void free_lanes(mhd_solver* s) {
  for (int l = 0; l < kMaxStreams; ++l) {
    HostLane& L = s->lanes[l];
    if (L.stream) cudaStreamDestroy(L.stream);
    cudaFree(L.Ui); cudaFree(L.Bi); cudaFree(L.Uo); cudaFree(L.Bo); cudaFree(L.fo); cudaFree(L.eo); cudaFree(L.ws);
    L = HostLane();
  }
  s->lane_groups = 0; s->lane_count = 0;
}

int mhd_destroy(mhd_solver* s) {
  if (!s) return MHD_EINVAL;
  cudaSetDevice(s->cfg.device);
  free_lanes(s);
  for (cudaEvent_t e : s->prof_ev) cudaEventDestroy(e);
  cudaFree(s->ws);
  cudaFree(s->d_stats);
  delete s;
  return MHD_OK;
}

int mhd_sizes(const mhd_solver* s, size_t* a, size_t* b, size_t* c, size_t* d, size_t* e, size_t* f) {
  if (!s) return MHD_EINVAL;
  if (a) *a = s->nUi; if (b) *b = s->nBi; if (c) *c = s->nUo; if (d) *d = s->nBo; if (e) *e = s->nF; if (f) *f = s->nE;
  return MHD_OK;
}

int mhd_advance(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out, void* flux_out,
                void* emf_out, int ngroups, double dt, double dh, void* cuda_stream) {
  if (!s || !U_in || !B_in || !U_out || !B_out) return MHD_EINVAL;
  if (ngroups < 0 || ngroups > s->cfg.max_groups) return MHD_EINVAL;
  if (!(dt > 0.0) || !(dh > 0.0) || !std::isfinite(dt) || !std::isfinite(dh)) return MHD_EINVAL;
  if (ngroups == 0) return MHD_OK;
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  return s->cfg.prec == MHD_FP32
             ? advance_dev<float>(s, U_in, B_in, U_out, B_out, flux_out, emf_out, s->ws, ngroups, dt, dh, st)
             : advance_dev<double>(s, U_in, B_in, U_out, B_out, flux_out, emf_out, s->ws, ngroups, dt, dh, st);
}

}  // extern "C"

#include "mhd_api_host.inl"

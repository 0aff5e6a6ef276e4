// mhd_api.cu -- the C ABI of include/mhd.h: solver object, slice scheduling over concurrent streams, kernel dispatch,
// stream-overlapped host path.  No CPU fallback anywhere: every entry point that computes needs a CUDA device.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/mhd.h"
#include "mhd_kernels3.cuh"
#include "mhd_grid.cuh"
#include "mhd_amr.cuh"
#include "mhd_prolong.cuh"
#include "mhd_ctu_pass1.cuh"
#include "mhd_vl_pass1.cuh"
#include "mhd_march.h"

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

struct DevLane {             // one internal stream of mhd_advance with its workspace
  cudaStream_t stream = nullptr;
  cudaEvent_t done = nullptr;
  void* ws = nullptr;
};

}  // namespace

struct mhd_solver {
  mhd_config cfg;
  int N, g, T, S, narr;
  size_t esz;                               // bytes per element
  size_t nUi, nBi, nUo, nBo, nF, nE;        // elements per group
  size_t S3;
  int slice_groups;                         // groups per slice (one slice = one pass of all stages on one lane)
  int nlanes;                               // concurrent slices of mhd_advance
  bool slice_fixed = false;                 // MHD_SLICE_GROUPS given: slices exactly as asked (experiments, tests)
  DevLane dev[kMaxStreams];
  cudaEvent_t fork = nullptr;
  unsigned long long* d_stats = nullptr;    // 3 counters
  unsigned long long* d_red = nullptr;      // dt reduction cell
  unsigned long long launches = 0;
  HostLane lanes[kMaxStreams];
  int lane_groups = 0, lane_count = 0;
  // optional per-stage timing (mhd_set_profiling): pairs of events around every stage launch; slices then run
  // one after the other on the caller's stream so that the stage times do not overlap
  bool no_fused_pass1 = false;              // MHD_NO_FUSED_PASS1=1: the staged CTU steps 1 + 2 also for the standard group (tests)
  bool no_march = false;                    // MHD_NO_MARCH=1 (or MHD_NO_FUSED_PASS1): VL without the plane-marching kernels (tests, A/B runs)
  bool prof_on = false;
  std::vector<cudaEvent_t> prof_ev;         // 2 per recorded launch
  std::vector<int> prof_stage;              // stage id per recorded launch
  size_t prof_used = 0;
  // staging buffers of mhd_grid_advance (ghost-zoned groups of the whole grid), allocated on first use
  void *gUi = nullptr, *gBi = nullptr, *gUo = nullptr, *gBo = nullptr;
  int grid_groups = 0;
};

namespace {

template <class R>
KParams<R> make_params(const mhd_solver* s, const void* Ui, const void* Bi, void* Uo, void* Bo, void* fo, void* eo,
                       void* ws, int first, double dt, double dh, unsigned long long* red) {
  KParams<R> p;
  p.Uin = static_cast<const R*>(Ui) + (size_t)first * s->nUi;
  p.Bin = static_cast<const R*>(Bi) + (size_t)first * s->nBi;
  p.Uout = static_cast<R*>(Uo) + (size_t)first * s->nUo;
  p.Bout = static_cast<R*>(Bo) + (size_t)first * s->nBo;
  p.fout = fo ? static_cast<R*>(fo) + (size_t)first * s->nF : nullptr;
  p.eout = eo ? static_cast<R*>(eo) + (size_t)first * s->nE : nullptr;
  p.ws = static_cast<R*>(ws);
  p.stats = s->d_stats;
  p.red = red;                       // non-null: the final update also reduces the CFL speed of the state it writes (S9)
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

#define LIM_SWITCH(lim, CALL)             \
  switch (lim) {                           \
    case 0: { constexpr int LIM = 0; CALL; } break; \
    case 1: { constexpr int LIM = 1; CALL; } break; \
    case 2: { constexpr int LIM = 2; CALL; } break; \
    case 3: { constexpr int LIM = 3; CALL; } break; \
    case 4: { constexpr int LIM = 4; CALL; } break; \
    default: { constexpr int LIM = 5; CALL; } break; \
  }

enum Stage : int { ST_LOAD = 0, ST_RECON, ST_FLUX1, ST_EMF1, ST_HALF, ST_CORR, ST_FLUX2, ST_EMF2, ST_FINAL, ST_DT, ST_PASS1, ST_MARCH1, ST_MARCH2, ST_COUNT };
const char* const kStageNames[ST_COUNT] = { "load_prim", "recon_ctu", "flux_pass1", "emf_pass1", "half_step", "ctu_corr",
                                            "flux_pass2", "emf_pass2", "final_update", "dt_reduce", "pass1_fused", "march_pass1", "march_pass2" };
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

// ---- index boxes: [lo, hi) per axis ---------------------------------------------------------
inline Box3 box(int x0, int x1, int y0, int y1, int z0, int z1) {
  Box3 b; b.lo[0] = x0; b.lo[1] = y0; b.lo[2] = z0; b.n[0] = x1 - x0; b.n[1] = y1 - y0; b.n[2] = z1 - z0;
  for (int a = 0; a < 2; ++a) b.m[a] = b.n[a] > 1 ? (unsigned)(0x100000000ULL / (unsigned)b.n[a]) + 1u : 0u;   // n >= 2 always (ps2 >= 8)
  return b;
}
// per sweep direction d: normal index in [n0, n1), both transverse indices in [t0, t1)
inline Box3x3 dir_boxes(int n0, int n1, int t0, int t1) {
  Box3x3 bx;
  for (int d = 0; d < 3; ++d) {
    int lo[3] = { t0, t0, t0 }, hi[3] = { t1, t1, t1 };
    lo[d] = n0; hi[d] = n1;
    bx.b[d] = box(lo[0], hi[0], lo[1], hi[1], lo[2], hi[2]);
  }
  return bx;
}
// edges along c: the two transverse indices in [a0, a1], the index along the edge in [c0, c1)
inline Box3x3 edge_boxes(int a0, int a1, int c0, int c1) {
  Box3x3 bx;
  for (int c = 0; c < 3; ++c) {
    int lo[3] = { a0, a0, a0 }, hi[3] = { a1 + 1, a1 + 1, a1 + 1 };
    lo[c] = c0; hi[c] = c1;
    bx.b[c] = box(lo[0], hi[0], lo[1], hi[1], lo[2], hi[2]);
  }
  return bx;
}
inline unsigned blocks_for(const Box3& b, int tpb) { return (unsigned)((b.n[0] * b.n[1] * b.n[2] + tpb - 1) / tpb); }
inline unsigned blocks_for(const Box3x3& bx, int tpb) {
  return std::max(blocks_for(bx.b[0], tpb), std::max(blocks_for(bx.b[1], tpb), blocks_for(bx.b[2], tpb)));
}

// all stages of one slice of groups, in the paper's step order
template <class R, int SC>
int run_slice_sc(mhd_solver* s, const KParams<R>& p0, int ng, cudaStream_t st) {
  const KParamsSC<R, SC> p(p0);
  const int TPB = 256;
  const dim3 blk(TPB);
  const int T = s->T, S = s->S, N = s->N, g = s->g, sol = s->cfg.riemann;
  const int lim = s->cfg.limvar + 2 * s->cfg.limiter;     // template parameter LIM of the slope kernels
#define GRID1(b) dim3(blocks_for(b, TPB), 1, ng)
#define GRID3(b) dim3(blocks_for(b, TPB), 3, ng)
  // standard VL + PLM group: the whole step as two plane-marching kernels with the intermediates on chip (mhd_vl_march.cuh)
  if constexpr (SC == 23) {
    if (s->cfg.scheme == MHD_VL && s->cfg.recon == MHD_PLM && N == 16 && g == 3 && !s->no_march && vl_march_supports<R>(sol)) {
      cudaError_t e1 = cudaSuccess, e2 = cudaSuccess;
      LAUNCH(ST_MARCH1, e1 = launch_vl_march<R>(p0, ng, sol, lim, 1, st));
      LAUNCH(ST_MARCH2, e2 = launch_vl_march<R>(p0, ng, sol, lim, 2, st));
      if (e1 != cudaSuccess) return cuda_fail(e1, "k_vl_march1");
      if (e2 != cudaSuccess) return cuda_fail(e2, "k_vl_march2");
      return MHD_OK;
    }
  }
  int f2 = A_F;                                   // where the pass-2 fluxes are
  const Box3 ball = box(0, S, 0, S, 0, S);
  // standard VL group with HLLD or Roe: S0 + S1 + S2 in one kernel (mhd_vl_pass1.cuh)
  bool fusedv = false;
  if constexpr (SC == 23) {
    fusedv = s->cfg.scheme == MHD_VL && N == 16 && g == 3 && sol != MHD_HLLE && !s->no_fused_pass1;
    const dim3 gv((kV1T + kV1Chunk - 1) / kV1Chunk, 1, ng);
    if (fusedv && sol == MHD_HLLD) LAUNCH(ST_PASS1, (k_vl_pass1<R, kHLLD, SC><<<gv, kV1Threads, 0, st>>>(p)));
    if constexpr (sizeof(R) == 4) {      // Roe in FP64 spills at 128 registers: 2.30 ms against 2.17 ms staged
      if (fusedv && sol == MHD_ROE) LAUNCH(ST_PASS1, (k_vl_pass1<R, kROE, SC><<<gv, kV1Threads, 0, st>>>(p)));
    } else if (sol == MHD_ROE) fusedv = false;
  }
  if (!fusedv) LAUNCH(ST_LOAD, (k_load_prim<R, SC><<<GRID1(ball), blk, 0, st>>>(p, ball)));
  if (s->cfg.scheme == MHD_VL) {
    // pass-1 edge EMFs only where the half step reads them: transverse indices 1 .. T-1, along the edge 1 .. T-2
    const Box3x3 bf1 = dir_boxes(1, T, 0, T), be1 = edge_boxes(1, T - 1, 1, T - 1);
    const Box3 bh = box(1, T - 1, 1, T - 1, 1, T - 1);
    // pass 2 only where the final update needs it: faces n in [g, g+N], t in [g-1, g+N]; edges of the interior faces
    const Box3x3 bf2 = dir_boxes(g, g + N + 1, g - 1, g + N + 1), be2 = edge_boxes(g, g + N, g, g + N);
    if (!fusedv) LAUNCH(ST_FLUX1, SOLVER_SWITCH(sol, (k_flux1_vl<R, SOLVER, SC><<<GRID3(bf1), blk, 0, st>>>(p, bf1))));          // step 1
    LAUNCH(ST_EMF1, (k_emf<R, A_F, SC><<<GRID3(be1), blk, 0, st>>>(p, be1, A_W)));                                      // step 2
    LAUNCH(ST_HALF, (k_half<R, SC><<<GRID1(bh), blk, 0, st>>>(p, bh, 1)));                                         // step 3
    if (s->cfg.recon == MHD_PLM && s->cfg.hcorr) {
      // R19: eta of the pass-2 faces and of the transverse faces around them (one face further along the normal), then Roe with eta^H
      const Box3x3 bet = dir_boxes(g - 1, g + N + 2, g - 1, g + N + 1);
      LIM_SWITCH(lim, LAUNCH(ST_RECON, (k_eta2_vl<R, LIM, SC><<<GRID3(bet), blk, 0, st>>>(p, bet))));
      LIM_SWITCH(lim, LAUNCH(ST_FLUX2, (k_flux2_vl<R, kROE, LIM, SC, true><<<GRID3(bf2), blk, 0, st>>>(p, bf2))));
    } else if (s->cfg.recon == MHD_PLM) {
      LIM_SWITCH(lim, LAUNCH(ST_FLUX2, SOLVER_SWITCH(sol, (k_flux2_vl<R, SOLVER, LIM, SC><<<GRID3(bf2), blk, 0, st>>>(p, bf2)))));   // steps 4+5
    } else {
      // VL + PPM (NEXT-4): limited slopes of the half-step primitives (parked in the dead pass-1 flux arrays), the
      // monotonised parabola's interface values as L/R states, then the plain L/R Riemann kernel of CTU
      // (H-correction: eta also on the faces one further along the normal, hence states and slopes of one more cell)
      const int hp = s->cfg.hcorr ? 1 : 0;
      const Box3x3 bsl = dir_boxes(g - 2 - hp, g + N + 2 + hp, g - 1, g + N + 1), brc = dir_boxes(g - 1 - hp, g + N + 1 + hp, g - 1, g + N + 1);
      LIM_SWITCH(lim, LAUNCH(ST_RECON, (k_slope_ctu<R, LIM, SC><<<GRID3(bsl), blk, 0, st>>>(p, bsl, A_WH))));
      LIM_SWITCH(lim, LAUNCH(ST_RECON, (k_recon_ctu<R, kPPMNoTrace, LIM, SC><<<GRID3(brc), blk, 0, st>>>(p, brc, A_WH))));
      if (hp) {
        const Box3x3 bet = dir_boxes(g - 1, g + N + 2, g - 1, g + N + 1);
        LAUNCH(ST_RECON, (k_flux_lr<R, kROE, SC, kHcEta><<<GRID3(bet), blk, 0, st>>>(p, bet, A_BH)));
        LAUNCH(ST_FLUX2, (k_flux_lr<R, kROE, SC, kHcOn><<<GRID3(bf2), blk, 0, st>>>(p, bf2, A_BH)));
      } else
      LAUNCH(ST_FLUX2, SOLVER_SWITCH(sol, (k_flux_lr<R, SOLVER, SC><<<GRID3(bf2), blk, 0, st>>>(p, bf2, A_BH))));
    }
    LAUNCH(ST_EMF2, (k_emf<R, A_F, SC><<<GRID3(be2), blk, 0, st>>>(p, be2, A_WH)));                                     // step 6
  } else {
    // everything is derived from the cells whose half-step state the second pass needs, [lo, hi)^3 = interior + 1:
    // pass-1 fluxes on their faces and on the faces their edge EMFs touch, face states one cell further, PPM slopes
    // one more (the oracle evaluates these stages on the whole tile; what it computes outside is never used)
    // (H-correction, R19: eta of the corrected states also on the transverse faces around the pass-2 faces: everything of the first
    // pass one cell further out, which is the one more ghost cell the switch asks for)
    const int hp = s->cfg.hcorr ? 1 : 0;
    const int lo = g - 1 - hp, hi = g + N + 1 + hp;
    const Box3x3 brc = dir_boxes(lo - 1, hi + 1, lo - 1, hi + 1), bf1 = dir_boxes(lo, hi + 1, lo - 1, hi + 1);
    const Box3x3 be1 = edge_boxes(lo, hi, lo, hi);
    const Box3 bh = box(lo, hi, lo, hi, lo, hi);
    const Box3x3 bco = dir_boxes(g - 1, g + N + 1, g - 1, g + N + 1), bf2 = dir_boxes(g, g + N + 1, g - 1, g + N + 1);
    const Box3x3 be2 = edge_boxes(g, g + N, g, g + N);
    // standard patch group in FP32 with PPM, MC limiter in characteristic variables and HLLD: steps 1 + 2 in one kernel
    // (mhd_ctu_pass1.cuh); everything else: slopes -> states -> Riemann solve as three kernels
    bool fused1 = false;
    if constexpr (SC == 25 && sizeof(R) == 4) {
      fused1 = N == 16 && g == 4 && s->cfg.recon == MHD_PPM && lim == 1 && sol == MHD_HLLD && !s->no_fused_pass1;
      if (fused1) {
        constexpr int ACROSS = kP1Across;
        const size_t shm = (size_t)21 * kP1Along * ACROSS * sizeof(R);
        const dim3 grd(kP1Across * (kP1Across / ACROSS), 3, ng);
        LAUNCH(ST_PASS1, (k_ctu_pass1<R, kHLLD, 1, ACROSS, SC><<<grd, kP1Along * ACROSS, shm, st>>>(p)));
      }
    }
    if (!fused1) {
      if (s->cfg.recon == MHD_PLM) {
        LIM_SWITCH(lim, LAUNCH(ST_RECON, (k_recon_ctu<R, kPLM, LIM, SC><<<GRID3(brc), blk, 0, st>>>(p, brc, A_W))));
      } else {
        const Box3x3 bsl = dir_boxes(lo - 2, hi + 2, lo - 1, hi + 1);
        LIM_SWITCH(lim, LAUNCH(ST_RECON, (k_slope_ctu<R, LIM, SC><<<GRID3(bsl), blk, 0, st>>>(p, bsl, A_W))));
        LIM_SWITCH(lim, LAUNCH(ST_RECON, (k_recon_ctu<R, kPPM, LIM, SC><<<GRID3(brc), blk, 0, st>>>(p, brc, A_W))));
      }                                                                                                        // step 1
      LAUNCH(ST_FLUX1, SOLVER_SWITCH(sol, (k_flux_lr<R, SOLVER, SC><<<GRID3(bf1), blk, 0, st>>>(p, bf1, A_B))));    // step 2
    }
    LAUNCH(ST_EMF1, (k_emf<R, A_F, SC><<<GRID3(be1), blk, 0, st>>>(p, be1, A_W)));                                      // step 3
    LAUNCH(ST_HALF, (k_half<R, SC><<<GRID1(bh), blk, 0, st>>>(p, bh, 0)));                                         // step 4
    if (hp) {
      const Box3x3 bet = dir_boxes(g - 1, g + N + 2, g - 1, g + N + 1);
      LAUNCH(ST_RECON, (k_flux2_ctu<R, kROE, SC, kHcEta><<<GRID3(bet), blk, 0, st>>>(p, bet)));
      LAUNCH(ST_FLUX2, (k_flux2_ctu<R, kROE, SC, kHcOn><<<GRID3(bf2), blk, 0, st>>>(p, bf2)));
    } else
    LAUNCH(ST_FLUX2, SOLVER_SWITCH(sol, (k_flux2_ctu<R, SOLVER, SC><<<GRID3(bf2), blk, 0, st>>>(p, bf2))));        // steps 5 + 6
    LAUNCH(ST_EMF2, (k_emf<R, A_F2, SC><<<GRID3(be2), blk, 0, st>>>(p, be2, A_WH)));                               // step 7
    f2 = A_F2;
  }
  const Box3 bin = box(g, g + N, g, g + N, g, g + N);
  const unsigned nbf = std::max(blocks_for(bin, TPB), (unsigned)((9 * (N + 1) * (N + 1) + TPB - 1) / TPB));
  const dim3 gfin(nbf, 1, ng);                                                                                   // step 7 / 8
  if (p.red) {                                                                                                   // + S9 (mhd_advance_dt)
    if (f2 == A_F) LAUNCH(ST_FINAL, (k_final<R, A_F, SC, true><<<gfin, blk, 0, st>>>(p, bin)));
    else LAUNCH(ST_FINAL, (k_final<R, A_F2, SC, true><<<gfin, blk, 0, st>>>(p, bin)));
  } else {
    if (f2 == A_F) LAUNCH(ST_FINAL, (k_final<R, A_F, SC, false><<<gfin, blk, 0, st>>>(p, bin)));
    else LAUNCH(ST_FINAL, (k_final<R, A_F2, SC, false><<<gfin, blk, 0, st>>>(p, bin)));
  }
#undef GRID1
#undef GRID3
  CU(cudaGetLastError());
  return MHD_OK;
}

// the kernels are instantiated for the two tile pitches of the standard patch group (N = 16: S = 23 with 3 ghost cells,
// S = 25 with 4) and for a run-time pitch (everything else)
template <class R>
int run_slice(mhd_solver* s, const KParams<R>& p, int ng, cudaStream_t st) {
  switch (s->S) {
    case 23: return run_slice_sc<R, 23>(s, p, ng, st);
    case 25: return run_slice_sc<R, 25>(s, p, ng, st);
    default: return run_slice_sc<R, 0>(s, p, ng, st);
  }
}

// a batch that needs several slices is cut into equal ones (no small last slice whose launches cannot fill the GPU)
// A batch that fits one slice is still cut into one slice per lane when every slice keeps >= kMinSliceGroups groups:
// each stage kernel ends in a partial wave of blocks (10.4 waves of k_vl_pass1 at 512 groups), and the other lane's
// kernels fill the SMs it leaves idle.  Measured (B200, 512 groups, VL+PLM+HLLD): 0.973 against 1.000 ms per step in
// FP32, 1.876 against 1.917 ms in FP64; slices are bitwise independent of the cut (tests/test_gpu_api.py).
constexpr int kMinSliceGroups = 128;
inline int balanced_slice(const mhd_solver* s, int ngroups, int cap) {
  int nslices = (ngroups + cap - 1) / cap;
  if (nslices < s->nlanes && ngroups >= kMinSliceGroups * s->nlanes && !s->slice_fixed) nslices = s->nlanes;
  return (ngroups + nslices - 1) / nslices;
}

// slices of one batch on ONE stream with ONE workspace (host path, profiling)
template <class R>
int advance_serial(mhd_solver* s, const void* Ui, const void* Bi, void* Uo, void* Bo, void* fo, void* eo, void* ws,
                   int ngroups, double dt, double dh, cudaStream_t st, unsigned long long* red, int slice_cap) {
  const int per = balanced_slice(s, ngroups, slice_cap);
  for (int first = 0; first < ngroups; first += per) {
    const int ng = std::min(per, ngroups - first);
    KParams<R> p = make_params<R>(s, Ui, Bi, Uo, Bo, fo, eo, ws, first, dt, dh, red);
    int rc = run_slice<R>(s, p, ng, st);
    if (rc != MHD_OK) return rc;
  }
  return MHD_OK;
}

// slices round-robin over the internal lanes, forked from and joined back into the caller's stream
template <class R>
int advance_lanes(mhd_solver* s, const void* Ui, const void* Bi, void* Uo, void* Bo, void* fo, void* eo,
                  int ngroups, double dt, double dh, cudaStream_t user, unsigned long long* red) {
  const int per = balanced_slice(s, ngroups, s->slice_groups);
  const int nslices = (ngroups + per - 1) / per;
  const int nl = std::min(s->nlanes, nslices);
  if (s->prof_on || nl <= 1) return advance_serial<R>(s, Ui, Bi, Uo, Bo, fo, eo, s->dev[0].ws, ngroups, dt, dh, user, red, s->slice_groups);
  CU(cudaEventRecord(s->fork, user));
  for (int l = 0; l < nl; ++l) CU(cudaStreamWaitEvent(s->dev[l].stream, s->fork, 0));
  int i = 0, rc = MHD_OK;
  for (int first = 0; first < ngroups && rc == MHD_OK; first += per, ++i) {
    const int ng = std::min(per, ngroups - first);
    DevLane& L = s->dev[i % nl];
    KParams<R> p = make_params<R>(s, Ui, Bi, Uo, Bo, fo, eo, L.ws, first, dt, dh, red);
    rc = run_slice<R>(s, p, ng, L.stream);
  }
  // also on an error: what the lanes have been given is joined back into the caller's stream
  for (int l = 0; l < nl; ++l) {
    cudaError_t e = cudaEventRecord(s->dev[l].done, s->dev[l].stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(user, s->dev[l].done, 0);
    if (e != cudaSuccess && rc == MHD_OK) rc = cuda_fail(e, "mhd_advance join");
  }
  return rc;
}

// largest signal speed from the bit pattern the kernels reduced; MHD_ESTATE if it is not finite and positive (a NaN or infinite
// state: the kernels encode a NaN speed as +inf so that the maximum cannot drop it)
inline int speed_to_dt(const mhd_solver* s, unsigned long long bits, double cfl, double dh, double* dt_out, double* maxspeed_out) {
  double smax;
  if (s->cfg.prec == MHD_FP32) { unsigned int b32 = (unsigned int)(bits & 0xffffffffu); float f; memcpy(&f, &b32, 4); smax = f; }
  else memcpy(&smax, &bits, 8);
  if (maxspeed_out) *maxspeed_out = smax;
  *dt_out = cfl * dh / smax;
  return (std::isfinite(smax) && smax > 0.0) ? MHD_OK : MHD_ESTATE;
}

int advance_impl(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out, void* flux_out, void* emf_out,
                 int ngroups, double dt, double dh, void* cuda_stream, unsigned long long* red) {
  if (!s || !U_in || !B_in || !U_out || !B_out) return MHD_EINVAL;
  if (ngroups < 0 || ngroups > s->cfg.max_groups) return MHD_EINVAL;
  if (!(dt > 0.0) || !(dh > 0.0) || !std::isfinite(dt) || !std::isfinite(dh)) return MHD_EINVAL;
  if (ngroups == 0) return MHD_OK;
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  return s->cfg.prec == MHD_FP32
             ? advance_lanes<float>(s, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, st, red)
             : advance_lanes<double>(s, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, st, red);
}

int check_config(const mhd_config* c) {
  if (!c) return MHD_EINVAL;
  if (c->ps2 < 8 || c->ps2 > 64 || (c->ps2 & 1)) return MHD_EINVAL;
  if (c->scheme != MHD_VL && c->scheme != MHD_CTU) return MHD_EINVAL;
  if (c->recon != MHD_PLM && c->recon != MHD_PPM) return MHD_EINVAL;
  if (c->riemann < MHD_HLLE || c->riemann > MHD_ROE) return MHD_EINVAL;
  if (c->limvar != MHD_LIM_PRIM && c->limvar != MHD_LIM_CHAR) return MHD_EINVAL;
  if (c->prec != MHD_FP32 && c->prec != MHD_FP64) return MHD_EINVAL;
  if (c->limiter < MHD_LIMITER_MC || c->limiter > MHD_LIMITER_VANLEER) return MHD_EINVAL;
  int need = c->recon == MHD_PPM ? 4 : 3;           // DESIGN.md R8
  if (c->hcorr != 0 && c->hcorr != 1) return MHD_EINVAL;
  if (c->hcorr) {                                   // DESIGN.md R19: Roe only, one more ghost cell
    if (c->riemann != MHD_ROE) return MHD_EINVAL;
    need += 1;
  }
  if (c->nghost < need || c->nghost > 8) return MHD_EINVAL;
  if (!(c->gamma > 1.0) || !std::isfinite(c->gamma)) return MHD_EINVAL;
  if (!(c->min_dens >= 0.0) || !(c->min_pres >= 0.0)) return MHD_EINVAL;
  if (c->max_groups < 1 || c->device < 0) return MHD_EINVAL;
  return MHD_OK;
}

}  // namespace

static void free_lanes(mhd_solver* s) {
  for (int l = 0; l < kMaxStreams; ++l) {
    HostLane& L = s->lanes[l];
    if (L.stream) cudaStreamDestroy(L.stream);
    cudaFree(L.Ui); cudaFree(L.Bi); cudaFree(L.Uo); cudaFree(L.Bo); cudaFree(L.fo); cudaFree(L.eo); cudaFree(L.ws);
    L = HostLane();
  }
  s->lane_groups = 0; s->lane_count = 0;
}

// for the other translation units of the library (mhd_noalloc.cu): a CUDA failure recorded for mhd_strerror(MHD_ECUDA)
namespace mhd {
int note_cuda_failure(cudaError_t e, const char* where) { return cuda_fail(e, where); }
}

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
  s->no_fused_pass1 = getenv("MHD_NO_FUSED_PASS1") != nullptr;
  s->no_march = s->no_fused_pass1 || getenv("MHD_NO_MARCH") != nullptr;
  s->narr = (cfg->scheme == MHD_VL && cfg->recon == MHD_PLM) ? A_VL_END : A_CTU_END;   // face-state arrays: CTU, VL + PPM
  if (cfg->scheme == MHD_CTU && cfg->hcorr) s->narr = A_CTU_HC_END;                     // + eta of the pass-2 faces
  s->esz = cfg->prec == MHD_FP32 ? 4 : 8;
  const size_t N = s->N, T = s->T;
  s->nUi = 5 * T * T * T; s->nBi = 3 * T * T * (T + 1);
  s->nUo = 5 * N * N * N; s->nBo = 3 * N * N * (N + 1);
  s->nF = 9 * 5 * N * N; s->nE = 9 * 2 * (N + 1) * N;
  // Lanes x slice: nlanes slices are in flight at once; a slice holds as many groups as fit the per-lane share of
  // the workspace budget.  Measured on B200: time per group falls monotonically with the slice size even far beyond
  // the L2 capacity, so slices only bound the workspace memory (MHD_LANES / MHD_SLICE_MB /
  // MHD_SLICE_GROUPS override for experiments)
  int nl = 2;
  if (const char* e = getenv("MHD_LANES")) { int v = atoi(e); if (v >= 1) nl = v; }
  s->nlanes = std::min(nl, kMaxStreams);
  double budget_mb = 6144.0;
  if (const char* e = getenv("MHD_SLICE_MB")) { double v = atof(e); if (v > 0) budget_mb = v; }
  const size_t per_group = ((size_t)s->narr * s->S3 + s->nUi + s->nBi + s->nUo + s->nBo + s->nF + s->nE) * s->esz;
  long sg = (long)(budget_mb * 1048576.0 / s->nlanes / (double)per_group);
  if (const char* e = getenv("MHD_SLICE_GROUPS")) { long v = atol(e); if (v > 0) { sg = v; s->slice_fixed = true; } }
  if (sg < 1) sg = 1;
  if (sg > cfg->max_groups) sg = cfg->max_groups;
  s->slice_groups = (int)sg;
  const size_t ws_bytes = (size_t)s->slice_groups * s->narr * s->S3 * s->esz;
  cudaError_t e = cudaMalloc((void**)&s->d_stats, 4 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMemset(s->d_stats, 0, 4 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->fork, cudaEventDisableTiming);
  for (int l = 0; l < s->nlanes && e == cudaSuccess; ++l) {
    e = cudaStreamCreateWithFlags(&s->dev[l].stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->dev[l].done, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaMalloc(&s->dev[l].ws, ws_bytes);
    // MHD_POISON=1 fills the workspace with NaN bit patterns: a stage that read a value no earlier stage wrote would
    // poison the output (tests/test_gpu_api.py compares a poisoned run bitwise with a normal one)
    if (e == cudaSuccess) e = cudaMemset(s->dev[l].ws, getenv("MHD_POISON") ? 0xFF : 0, ws_bytes);
  }
  if (e != cudaSuccess) { int r = cuda_fail(e, "mhd_create allocation"); mhd_destroy(s); return r; }
  s->d_red = s->d_stats + 3;
  *out = s;
  return MHD_OK;
}

int mhd_destroy(mhd_solver* s) {
  if (!s) return MHD_EINVAL;
  cudaSetDevice(s->cfg.device);
  cudaDeviceSynchronize();
  free_lanes(s);
  for (cudaEvent_t e : s->prof_ev) cudaEventDestroy(e);
  for (int l = 0; l < kMaxStreams; ++l) {
    if (s->dev[l].stream) cudaStreamDestroy(s->dev[l].stream);
    if (s->dev[l].done) cudaEventDestroy(s->dev[l].done);
    cudaFree(s->dev[l].ws);
  }
  if (s->fork) cudaEventDestroy(s->fork);
  cudaFree(s->gUi); cudaFree(s->gBi); cudaFree(s->gUo); cudaFree(s->gBo);
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
  return advance_impl(s, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, cuda_stream, nullptr);
}

// mhd_advance with the CFL reduction (S9) of its own output fused into the final update (S8)
int mhd_advance_dt(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out, void* flux_out,
                   void* emf_out, int ngroups, double dt, double dh, double cfl, double* dt_out, double* maxspeed_out,
                   void* cuda_stream) {
  if (!s || !dt_out || ngroups < 1 || !(cfl > 0.0)) return MHD_EINVAL;
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  CU(cudaMemsetAsync(s->d_red, 0, sizeof(unsigned long long), st));
  const int rc = advance_impl(s, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, cuda_stream, s->d_red);
  if (rc != MHD_OK) return rc;
  unsigned long long bits = 0;
  CU(cudaMemcpyAsync(&bits, s->d_red, sizeof bits, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  return speed_to_dt(s, bits, cfl, dh, dt_out, maxspeed_out);
}

}  // extern "C"

#include "mhd_api_host.inl"
#include "mhd_api_grid.inl"
#include "mhd_api_amr.inl"

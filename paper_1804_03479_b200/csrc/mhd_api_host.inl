// mhd_api_host.inl -- included by mhd_api.cu: stream-overlapped host path, dt reduction,
// counters, FMA-peak probe, error strings.

namespace {

int ensure_lanes(mhd_solver* s, int nstreams, int chunk_groups) {
  if (s->lane_count >= nstreams && s->lane_groups >= chunk_groups) return MHD_OK;
  free_lanes(s);
  const size_t e = s->esz, cg = (size_t)chunk_groups;
  const size_t wsg = (size_t)std::min(s->slice_groups, chunk_groups);
  for (int l = 0; l < nstreams; ++l) {
    HostLane& L = s->lanes[l];
    CU(cudaStreamCreateWithFlags(&L.stream, cudaStreamNonBlocking));
    CU(cudaMalloc(&L.Ui, cg * s->nUi * e)); CU(cudaMalloc(&L.Bi, cg * s->nBi * e));
    CU(cudaMalloc(&L.Uo, cg * s->nUo * e)); CU(cudaMalloc(&L.Bo, cg * s->nBo * e));
    CU(cudaMalloc(&L.fo, cg * s->nF * e)); CU(cudaMalloc(&L.eo, cg * s->nE * e));
    CU(cudaMalloc(&L.ws, wsg * s->narr * s->S3 * e));
    CU(cudaMemsetAsync(L.ws, 0, wsg * s->narr * s->S3 * e, L.stream));
  }
  s->lane_count = nstreams; s->lane_groups = chunk_groups;
  return MHD_OK;
}

// red != nullptr: the final update of every chunk also reduces the CFL speed into *red (zeroed on lane 0 before any chunk)
int advance_host_impl(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out, void* flux_out,
                      void* emf_out, int ngroups, double dt, double dh, int chunk_groups, int nstreams, unsigned long long* red) {
  if (!s || !U_in || !B_in || !U_out || !B_out) return MHD_EINVAL;
  if (ngroups < 0 || nstreams < 1 || nstreams > kMaxStreams) return MHD_EINVAL;
  if (chunk_groups < 1 || chunk_groups > s->cfg.max_groups) return MHD_EINVAL;
  if (!(dt > 0.0) || !(dh > 0.0) || !std::isfinite(dt) || !std::isfinite(dh)) return MHD_EINVAL;
  if (ngroups == 0) return MHD_OK;
  CU(cudaSetDevice(s->cfg.device));
  int rc = ensure_lanes(s, nstreams, chunk_groups);
  if (rc != MHD_OK) return rc;
  const size_t e = s->esz;
  const char* hUi = static_cast<const char*>(U_in); const char* hBi = static_cast<const char*>(B_in);
  char* hUo = static_cast<char*>(U_out); char* hBo = static_cast<char*>(B_out);
  char* hf = static_cast<char*>(flux_out); char* he = static_cast<char*>(emf_out);
  // the lane's slice size must not exceed its workspace
  const int slice_cap = std::min(s->slice_groups, chunk_groups);
  if (red) {
    CU(cudaMemsetAsync(red, 0, sizeof(unsigned long long), s->lanes[0].stream));
    CU(cudaEventRecord(s->fork, s->lanes[0].stream));
    for (int l = 1; l < nstreams; ++l) CU(cudaStreamWaitEvent(s->lanes[l].stream, s->fork, 0));
  }
  int c = 0;
  for (int first = 0; first < ngroups && rc == MHD_OK; first += chunk_groups, ++c) {
    const size_t ng = (size_t)std::min(chunk_groups, ngroups - first), f = (size_t)first;
    HostLane& L = s->lanes[c % nstreams];
    cudaError_t ce = cudaMemcpyAsync(L.Ui, hUi + f * s->nUi * e, ng * s->nUi * e, cudaMemcpyHostToDevice, L.stream);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(L.Bi, hBi + f * s->nBi * e, ng * s->nBi * e, cudaMemcpyHostToDevice, L.stream);
    if (ce != cudaSuccess) { rc = cuda_fail(ce, "mhd_advance_host H2D"); break; }
    rc = s->cfg.prec == MHD_FP32
             ? advance_serial<float>(s, L.Ui, L.Bi, L.Uo, L.Bo, hf ? L.fo : nullptr, he ? L.eo : nullptr, L.ws, (int)ng, dt, dh, L.stream, red, slice_cap)
             : advance_serial<double>(s, L.Ui, L.Bi, L.Uo, L.Bo, hf ? L.fo : nullptr, he ? L.eo : nullptr, L.ws, (int)ng, dt, dh, L.stream, red, slice_cap);
    if (rc != MHD_OK) break;
    ce = cudaMemcpyAsync(hUo + f * s->nUo * e, L.Uo, ng * s->nUo * e, cudaMemcpyDeviceToHost, L.stream);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(hBo + f * s->nBo * e, L.Bo, ng * s->nBo * e, cudaMemcpyDeviceToHost, L.stream);
    if (ce == cudaSuccess && hf) ce = cudaMemcpyAsync(hf + f * s->nF * e, L.fo, ng * s->nF * e, cudaMemcpyDeviceToHost, L.stream);
    if (ce == cudaSuccess && he) ce = cudaMemcpyAsync(he + f * s->nE * e, L.eo, ng * s->nE * e, cudaMemcpyDeviceToHost, L.stream);
    if (ce != cudaSuccess) rc = cuda_fail(ce, "mhd_advance_host D2H");
  }
  // also on an error: no copy into the caller's host buffers is left in flight when this call returns
  for (int l = 0; l < nstreams; ++l) {
    const cudaError_t ce = cudaStreamSynchronize(s->lanes[l].stream);
    if (ce != cudaSuccess && rc == MHD_OK) rc = cuda_fail(ce, "mhd_advance_host synchronize");
  }
  return rc;
}

}  // namespace

extern "C" {

int mhd_advance_host(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out, void* flux_out,
                     void* emf_out, int ngroups, double dt, double dh, int chunk_groups, int nstreams) {
  return advance_host_impl(s, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, chunk_groups, nstreams, nullptr);
}

int mhd_advance_host_dt(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out, void* flux_out,
                        void* emf_out, int ngroups, double dt, double dh, int chunk_groups, int nstreams, double cfl,
                        double* dt_out, double* maxspeed_out) {
  if (!s || !dt_out || ngroups < 1 || !(cfl > 0.0)) return MHD_EINVAL;
  const int rc = advance_host_impl(s, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, chunk_groups, nstreams, s->d_red);
  if (rc != MHD_OK) return rc;
  unsigned long long bits = 0;
  CU(cudaMemcpy(&bits, s->d_red, sizeof bits, cudaMemcpyDeviceToHost));      // every lane is synchronised
  return speed_to_dt(s, bits, cfl, dh, dt_out, maxspeed_out);
}

int mhd_dt_reduce(mhd_solver* s, const void* U, const void* B, int ngroups, int nghost_of_arrays, double dh, double cfl,
                  double* dt_out, double* maxspeed_out, void* cuda_stream) {
  if (!s || !U || !B || !dt_out || ngroups < 1) return MHD_EINVAL;
  if (nghost_of_arrays != 0 && nghost_of_arrays != s->g) return MHD_EINVAL;
  if (!(dh > 0.0) || !(cfl > 0.0)) return MHD_EINVAL;
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int N = s->N, ng = nghost_of_arrays, T = N + 2 * ng;
  const long long nU = 5LL * T * T * T, nB = 3LL * T * T * (T + 1);
  CU(cudaMemsetAsync(s->d_red, 0, sizeof(unsigned long long), st));
  const dim3 grid((N * N * N + 255) / 256, 1, ngroups), blk(256);
  if (s->cfg.prec == MHD_FP32)
    LAUNCH(ST_DT, (k_dt<float><<<grid, blk, 0, st>>>(static_cast<const float*>(U), static_cast<const float*>(B), N, ng, nU, nB,
                                       (float)s->cfg.gamma, (float)s->cfg.min_dens, (float)s->cfg.min_pres, s->d_red)));
  else
    LAUNCH(ST_DT, (k_dt<double><<<grid, blk, 0, st>>>(static_cast<const double*>(U), static_cast<const double*>(B), N, ng, nU, nB,
                                        s->cfg.gamma, s->cfg.min_dens, s->cfg.min_pres, s->d_red)));
  CU(cudaGetLastError());
  unsigned long long bits = 0;
  CU(cudaMemcpyAsync(&bits, s->d_red, sizeof bits, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  return speed_to_dt(s, bits, cfl, dh, dt_out, maxspeed_out);
}

int mhd_get_stats(mhd_solver* s, unsigned long long* fd, unsigned long long* fp, unsigned long long* fb) {
  if (!s) return MHD_EINVAL;
  CU(cudaSetDevice(s->cfg.device));
  CU(cudaDeviceSynchronize());
  unsigned long long h[3];
  CU(cudaMemcpy(h, s->d_stats, sizeof h, cudaMemcpyDeviceToHost));
  if (fd) *fd = h[0]; if (fp) *fp = h[1]; if (fb) *fb = h[2];
  return MHD_OK;
}

unsigned long long mhd_launch_count(const mhd_solver* s) { return s ? s->launches : 0ULL; }

int mhd_set_profiling(mhd_solver* s, int on) {
  if (!s) return MHD_EINVAL;
  s->prof_on = on != 0;
  s->prof_used = 0;
  return MHD_OK;
}

int mhd_get_profile(mhd_solver* s, double* ms_per_stage, unsigned long long* launches_per_stage, int nstages) {
  if (!s || !ms_per_stage || !launches_per_stage || nstages < ST_COUNT) return MHD_EINVAL;
  CU(cudaSetDevice(s->cfg.device));
  CU(cudaDeviceSynchronize());
  for (int i = 0; i < nstages; ++i) { ms_per_stage[i] = 0.0; launches_per_stage[i] = 0; }
  for (size_t l = 0; l < s->prof_used; ++l) {
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, s->prof_ev[2 * l], s->prof_ev[2 * l + 1]));
    ms_per_stage[s->prof_stage[l]] += ms;
    launches_per_stage[s->prof_stage[l]]++;
  }
  return ST_COUNT;
}

const char* mhd_profile_stage_name(int stage) { return (stage >= 0 && stage < ST_COUNT) ? kStageNames[stage] : ""; }

int mhd_measure_fma_peak(int device, int prec, double* tflops_out) {
  if (!tflops_out || (prec != MHD_FP32 && prec != MHD_FP64)) return MHD_EINVAL;
  CU(cudaSetDevice(device));
  cudaDeviceProp prop;
  CU(cudaGetDeviceProperties(&prop, device));
  void* out = nullptr;
  CU(cudaMalloc(&out, 64));
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  const int blocks = prop.multiProcessorCount * 8, iters = prec == MHD_FP32 ? 4096 : 2048;
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {
    CU(cudaEventRecord(e0));
    if (prec == MHD_FP32) k_fma_peak<float><<<blocks, 256>>>(static_cast<float*>(out), iters);
    else k_fma_peak<double><<<blocks, 256>>>(static_cast<double*>(out), iters);
    CU(cudaEventRecord(e1));
    CU(cudaEventSynchronize(e1));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, e0, e1));
    const double flops = 2.0 * 64.0 * iters * 256.0 * blocks;
    if (rep > 0) best = std::max(best, flops / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
  *tflops_out = best;
  return MHD_OK;
}

const char* mhd_strerror(int code) {
  switch (code) {
    case MHD_OK: return "ok";
    case MHD_EINVAL: return "invalid argument or configuration";
    case MHD_ECUDA: return g_cuda_err.c_str();
    case MHD_ENOMEM: return "out of device memory";
    case MHD_ESTATE: return "the state has no finite positive signal speed (NaN or infinite values): no time step";
    case MHD_ELIMIT: return "size beyond the fixed capacity of a no-allocation entry point (MHD_NOALLOC_MAX_BLOCKS, include/mhd.h)";
    default: return "unknown error code";
  }
}

}  // extern "C"

// mhd_api_grid.inl -- included by mhd_api.cu: device-side preparation / closing for a uniform periodic grid
// and the grid-resident step built from them.

namespace {

int grid_dims(const mhd_solver* s, int nx, int ny, int nz, GridDims* d) {
  const int N = s->N;
  if (nx < N || ny < N || nz < N || nx % N || ny % N || nz % N) return MHD_EINVAL;
  // the periodic ghost fill wraps at most once around the domain
  if (s->g > nx || s->g > ny || s->g > nz) return MHD_EINVAL;
  d->nx = nx; d->ny = ny; d->nz = nz; d->mx = nx / N; d->my = ny / N; d->mz = nz / N;
  const long long G = (long long)d->mx * d->my * d->mz;
  if (G > s->cfg.max_groups || G > 65535) return MHD_EINVAL;   // one grid.z slot per group
  return MHD_OK;
}

template <class R>
int grid_pack_t(mhd_solver* s, const void* U, const void* bx, const void* by, const void* bz, const GridDims& d, int ng,
                void* Uin, void* Bin, cudaStream_t st) {
  const int T = s->N + 2 * ng, S = T + 1, G = d.mx * d.my * d.mz;
  k_grid_pack<R><<<dim3((S * S * S + 255) / 256, 1, G), 256, 0, st>>>(
      static_cast<const R*>(U), static_cast<const R*>(bx), static_cast<const R*>(by), static_cast<const R*>(bz), d, s->N, ng,
      static_cast<R*>(Uin), static_cast<R*>(Bin));
  s->launches++;
  CU(cudaGetLastError());
  return MHD_OK;
}

template <class R>
int grid_unpack_t(mhd_solver* s, const void* Uout, const void* Bout, const GridDims& d, void* U, void* bx, void* by, void* bz,
                  cudaStream_t st) {
  const int N = s->N, G = d.mx * d.my * d.mz;
  k_grid_unpack<R><<<dim3((N * N * N + 255) / 256, 1, G), 256, 0, st>>>(
      static_cast<const R*>(Uout), static_cast<const R*>(Bout), d, N, static_cast<R*>(U), static_cast<R*>(bx),
      static_cast<R*>(by), static_cast<R*>(bz));
  s->launches++;
  CU(cudaGetLastError());
  return MHD_OK;
}

}  // namespace

extern "C" {

int mhd_grid_pack(mhd_solver* s, const void* U, const void* bx, const void* by, const void* bz, int nx, int ny, int nz,
                  void* U_in, void* B_in, void* cuda_stream) {
  if (!s || !U || !bx || !by || !bz || !U_in || !B_in) return MHD_EINVAL;
  GridDims d;
  int rc = grid_dims(s, nx, ny, nz, &d);
  if (rc != MHD_OK) return rc;
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  return s->cfg.prec == MHD_FP32 ? grid_pack_t<float>(s, U, bx, by, bz, d, s->g, U_in, B_in, st)
                                 : grid_pack_t<double>(s, U, bx, by, bz, d, s->g, U_in, B_in, st);
}

int mhd_grid_unpack(mhd_solver* s, const void* U_out, const void* B_out, int nx, int ny, int nz, void* U, void* bx, void* by,
                    void* bz, void* cuda_stream) {
  if (!s || !U || !bx || !by || !bz || !U_out || !B_out) return MHD_EINVAL;
  GridDims d;
  int rc = grid_dims(s, nx, ny, nz, &d);
  if (rc != MHD_OK) return rc;
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  return s->cfg.prec == MHD_FP32 ? grid_unpack_t<float>(s, U_out, B_out, d, U, bx, by, bz, st)
                                 : grid_unpack_t<double>(s, U_out, B_out, d, U, bx, by, bz, st);
}

}  // extern "C"

// pack -> all stages -> unpack; red != nullptr: the final update also reduces the CFL speed into *red
static int grid_advance_impl(mhd_solver* s, void* U, void* bx, void* by, void* bz, int nx, int ny, int nz, double dt, double dh,
                             unsigned long long* red, void* cuda_stream) {
  if (!s || !U || !bx || !by || !bz) return MHD_EINVAL;
  if (!(dt > 0.0) || !(dh > 0.0) || !std::isfinite(dt) || !std::isfinite(dh)) return MHD_EINVAL;
  GridDims d;
  int rc = grid_dims(s, nx, ny, nz, &d);
  if (rc != MHD_OK) return rc;
  CU(cudaSetDevice(s->cfg.device));
  const int G = d.mx * d.my * d.mz;
  if (s->grid_groups < G) {
    CU(cudaDeviceSynchronize());
    cudaFree(s->gUi); cudaFree(s->gBi); cudaFree(s->gUo); cudaFree(s->gBo);
    s->gUi = s->gBi = s->gUo = s->gBo = nullptr; s->grid_groups = 0;
    CU(cudaMalloc(&s->gUi, (size_t)G * s->nUi * s->esz)); CU(cudaMalloc(&s->gBi, (size_t)G * s->nBi * s->esz));
    CU(cudaMalloc(&s->gUo, (size_t)G * s->nUo * s->esz)); CU(cudaMalloc(&s->gBo, (size_t)G * s->nBo * s->esz));
    s->grid_groups = G;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (red) CU(cudaMemsetAsync(red, 0, sizeof(unsigned long long), st));
  if (s->cfg.prec == MHD_FP32) {
    rc = grid_pack_t<float>(s, U, bx, by, bz, d, s->g, s->gUi, s->gBi, st);
    if (rc == MHD_OK) rc = advance_lanes<float>(s, s->gUi, s->gBi, s->gUo, s->gBo, nullptr, nullptr, G, dt, dh, st, red);
    if (rc == MHD_OK) rc = grid_unpack_t<float>(s, s->gUo, s->gBo, d, U, bx, by, bz, st);
  } else {
    rc = grid_pack_t<double>(s, U, bx, by, bz, d, s->g, s->gUi, s->gBi, st);
    if (rc == MHD_OK) rc = advance_lanes<double>(s, s->gUi, s->gBi, s->gUo, s->gBo, nullptr, nullptr, G, dt, dh, st, red);
    if (rc == MHD_OK) rc = grid_unpack_t<double>(s, s->gUo, s->gBo, d, U, bx, by, bz, st);
  }
  return rc;
}

extern "C" {

int mhd_grid_advance(mhd_solver* s, void* U, void* bx, void* by, void* bz, int nx, int ny, int nz, double dt, double dh,
                     void* cuda_stream) {
  return grid_advance_impl(s, U, bx, by, bz, nx, ny, nz, dt, dh, nullptr, cuda_stream);
}

int mhd_grid_advance_dt(mhd_solver* s, void* U, void* bx, void* by, void* bz, int nx, int ny, int nz, double dt, double dh,
                        double cfl, double* dt_out, double* maxspeed_out, void* cuda_stream) {
  if (!s || !dt_out || !(cfl > 0.0)) return MHD_EINVAL;
  const int rc = grid_advance_impl(s, U, bx, by, bz, nx, ny, nz, dt, dh, s->d_red, cuda_stream);
  if (rc != MHD_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  unsigned long long bits = 0;
  CU(cudaMemcpyAsync(&bits, s->d_red, sizeof bits, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  return speed_to_dt(s, bits, cfl, dh, dt_out, maxspeed_out);
}

int mhd_grid_dt(mhd_solver* s, const void* U, const void* bx, const void* by, const void* bz, int nx, int ny, int nz, double dh,
                double cfl, double* dt_out, double* maxspeed_out, void* cuda_stream) {
  if (!s || !U || !bx || !by || !bz || !dt_out) return MHD_EINVAL;
  if (nx < 1 || ny < 1 || nz < 1 || !(dh > 0.0) || !(cfl > 0.0)) return MHD_EINVAL;
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  GridDims d; d.nx = nx; d.ny = ny; d.nz = nz; d.mx = d.my = d.mz = 1;
  const size_t n3 = (size_t)nx * ny * nz;
  CU(cudaMemsetAsync(s->d_red, 0, sizeof(unsigned long long), st));
  const dim3 grid((unsigned)((n3 + 255) / 256)), blk(256);
  if (s->cfg.prec == MHD_FP32)
    LAUNCH(ST_DT, (k_dt_grid<float><<<grid, blk, 0, st>>>(static_cast<const float*>(U), static_cast<const float*>(bx),
                   static_cast<const float*>(by), static_cast<const float*>(bz), d, (float)s->cfg.gamma, (float)s->cfg.min_dens,
                   (float)s->cfg.min_pres, s->d_red)));
  else
    LAUNCH(ST_DT, (k_dt_grid<double><<<grid, blk, 0, st>>>(static_cast<const double*>(U), static_cast<const double*>(bx),
                   static_cast<const double*>(by), static_cast<const double*>(bz), d, s->cfg.gamma, s->cfg.min_dens,
                   s->cfg.min_pres, s->d_red)));
  CU(cudaGetLastError());
  unsigned long long bits = 0;
  CU(cudaMemcpyAsync(&bits, s->d_red, sizeof bits, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  return speed_to_dt(s, bits, cfl, dh, dt_out, maxspeed_out);
}

}  // extern "C"

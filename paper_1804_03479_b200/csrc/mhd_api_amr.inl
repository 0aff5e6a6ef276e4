// mhd_api_amr.inl -- included by mhd_api.cu: the AMR correction operation on a static two-level mesh
// (PAPER.md:205-207).

namespace {

int amr_geom(const mhd_solver* s, const int* lo, const int* hi, int nx, int ny, int nz, Amr* a) {
  if (!lo || !hi) return MHD_EINVAL;
  const int N = s->N, h = N / 2, n[3] = { nx, ny, nz };
  a->N = N; a->h = h;
  for (int d = 0; d < 3; ++d) {
    if (n[d] < N || n[d] % N) return MHD_EINVAL;
    // patch-aligned, non-empty, at least one patch away from the periodic boundary
    if (lo[d] % h || hi[d] % h || lo[d] < h || hi[d] > n[d] - h || lo[d] >= hi[d]) return MHD_EINVAL;
    // the box must be tiled by whole fine patch groups
    if ((hi[d] - lo[d]) % h) return MHD_EINVAL;
    a->n.set(d, n[d]); a->mg.set(d, n[d] / N); a->lo.set(d, lo[d]); a->hi.set(d, hi[d]); a->mf.set(d, (hi[d] - lo[d]) / h);
  }
  return MHD_OK;
}

}  // namespace

extern "C" {

int mhd_amr_restrict(mhd_solver* s, const void* U_f, const void* B_f, const int* lo, const int* hi, void* Uc, void* bxc,
                     void* byc, void* bzc, int nx, int ny, int nz, void* cuda_stream) {
  if (!s || !U_f || !B_f || !Uc || !bxc || !byc || !bzc) return MHD_EINVAL;
  Amr a;
  int rc = amr_geom(s, lo, hi, nx, ny, nz, &a);
  if (rc != MHD_OK) return rc;
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int npts = (a.hi[0] - a.lo[0] + 1) * (a.hi[1] - a.lo[1] + 1) * (a.hi[2] - a.lo[2] + 1);
  const dim3 grid((npts + 255) / 256), blk(256);
  if (s->cfg.prec == MHD_FP32)
    k_amr_restrict<float><<<grid, blk, 0, st>>>(static_cast<const float*>(U_f), static_cast<const float*>(B_f), a, static_cast<float*>(Uc),
                                                static_cast<float*>(bxc), static_cast<float*>(byc), static_cast<float*>(bzc));
  else
    k_amr_restrict<double><<<grid, blk, 0, st>>>(static_cast<const double*>(U_f), static_cast<const double*>(B_f), a, static_cast<double*>(Uc),
                                                 static_cast<double*>(bxc), static_cast<double*>(byc), static_cast<double*>(bzc));
  s->launches++;
  CU(cudaGetLastError());
  return MHD_OK;
}

int mhd_amr_fixup(mhd_solver* s, const void* flux_c, const void* emf_c, const void* flux_f, const void* emf_f, const int* lo,
                  const int* hi, double dt, double dh_c, double w_c, double w_f, void* Uc, void* bxc, void* byc, void* bzc,
                  int nx, int ny, int nz, void* cuda_stream) {
  if (!s || !flux_c || !emf_c || !flux_f || !emf_f || !Uc || !bxc || !byc || !bzc) return MHD_EINVAL;
  if (!(dt > 0.0) || !(dh_c > 0.0) || !std::isfinite(w_c) || !std::isfinite(w_f)) return MHD_EINVAL;
  Amr a;
  int rc = amr_geom(s, lo, hi, nx, ny, nz, &a);
  if (rc != MHD_OK) return rc;
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int nb[3] = { a.hi[0] - a.lo[0], a.hi[1] - a.lo[1], a.hi[2] - a.lo[2] };
  const int nfaces = 2 * (nb[1] * nb[2] + nb[2] * nb[0] + nb[0] * nb[1]);
  const int ncand = (nb[0] + 3) * (nb[1] + 3) * (nb[2] + 3);
  const dim3 blk(256), gf((nfaces + 255) / 256), ge((ncand + 255) / 256, 3);
  const double q = dt / dh_c;
  if (s->cfg.prec == MHD_FP32) {
    k_amr_flux_fixup<float><<<gf, blk, 0, st>>>(static_cast<const float*>(flux_c), static_cast<const float*>(flux_f), a, (float)q, (float)w_c,
                                                (float)w_f, static_cast<float*>(Uc));
    k_amr_emf_fixup<float><<<ge, blk, 0, st>>>(static_cast<const float*>(emf_c), static_cast<const float*>(emf_f), a, (float)q, (float)w_c,
                                               (float)w_f, static_cast<float*>(bxc), static_cast<float*>(byc), static_cast<float*>(bzc));
  } else {
    k_amr_flux_fixup<double><<<gf, blk, 0, st>>>(static_cast<const double*>(flux_c), static_cast<const double*>(flux_f), a, q, w_c, w_f,
                                                 static_cast<double*>(Uc));
    k_amr_emf_fixup<double><<<ge, blk, 0, st>>>(static_cast<const double*>(emf_c), static_cast<const double*>(emf_f), a, q, w_c, w_f,
                                                static_cast<double*>(bxc), static_cast<double*>(byc), static_cast<double*>(bzc));
  }
  s->launches += 2;
  CU(cudaGetLastError());
  return MHD_OK;
}

int mhd_amr_prolong(mhd_solver* s, const void* Uc, const void* bxc, const void* byc, const void* bzc, int nx, int ny, int nz,
                    const int* lo, const int* hi, void* U_f, void* bx_f, void* by_f, void* bz_f, void* cuda_stream) {
  if (!s || !Uc || !bxc || !byc || !bzc || !U_f || !bx_f || !by_f || !bz_f || !lo || !hi) return MHD_EINVAL;
  const int n[3] = { nx, ny, nz };
  ProlongGeom g;
  long long npts = 1;
  for (int d = 0; d < 3; ++d) {
    if (n[d] < 2 || lo[d] < 0 || lo[d] >= hi[d] || hi[d] > n[d]) return MHD_EINVAL;
    g.n.set(d, n[d]); g.lo.set(d, lo[d]); g.hi.set(d, hi[d]);
    npts *= hi[d] - lo[d] + 1;
  }
  CU(cudaSetDevice(s->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const dim3 grid((unsigned)((npts + 127) / 128)), blk(128);
  if (s->cfg.prec == MHD_FP32)
    k_amr_prolong<float><<<grid, blk, 0, st>>>(static_cast<const float*>(Uc), static_cast<const float*>(bxc), static_cast<const float*>(byc),
                                               static_cast<const float*>(bzc), g, static_cast<float*>(U_f), static_cast<float*>(bx_f),
                                               static_cast<float*>(by_f), static_cast<float*>(bz_f));
  else
    k_amr_prolong<double><<<grid, blk, 0, st>>>(static_cast<const double*>(Uc), static_cast<const double*>(bxc), static_cast<const double*>(byc),
                                                static_cast<const double*>(bzc), g, static_cast<double*>(U_f), static_cast<double*>(bx_f),
                                                static_cast<double*>(by_f), static_cast<double*>(bz_f));
  s->launches++;
  CU(cudaGetLastError());
  return MHD_OK;
}

}  // extern "C"

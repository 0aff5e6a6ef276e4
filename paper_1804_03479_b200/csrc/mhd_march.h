// mhd_march.h -- launchers of the plane-marching VL kernels (mhd_vl_march.cuh), compiled in their own translation unit
#pragma once
#include <cuda_runtime.h>
#include "mhd_kernels.cuh"

namespace mhd {

// pass = 1: S0-S4 (k_vl_march1), pass = 2: S5-S8 and, if p.red is set, S9 (k_vl_march2).  solver: kHLLD or kROE (Roe: FP32 only);
// lim = limvar + 2 * limiter.  Standard VL group only (N = 16, 3 ghost cells, PLM).  Returns the launch error.
template <class R> cudaError_t launch_vl_march(const KParams<R>& p, int ngroups, int solver, int lim, int pass, cudaStream_t st);
// whether the fused path serves this solver in this precision
template <class R> bool vl_march_supports(int solver);

}  // namespace mhd

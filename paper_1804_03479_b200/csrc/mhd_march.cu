// mhd_march.cu -- instantiations and launchers of the plane-marching VL kernels (mhd_vl_march.cuh)
#include <algorithm>
#include <cstdlib>
#include "mhd_march.h"
#include "mhd_vl_march.cuh"

namespace mhd {

namespace {

// block slots of the marching kernels on one B200 (two resident blocks on each of 148 SMs in FP32 with HLLD); MHD_MARCH_SLOTS overrides (tests: 1 = never
// chunk, a large value = always the finest chunks)
// one_per_sm: FP64 and Roe run one block per SM
inline int march_slots(bool one_per_sm) {
  const char* e = getenv("MHD_MARCH_SLOTS");
  const int v = e ? atoi(e) : 0;
  return v > 0 ? v : (one_per_sm ? 148 : 296);
}
#define kMarchSlots march_slots(sizeof(R) == 8 || SOLVER == kROE)

template <class K> cudaError_t big_smem(K kernel, size_t bytes) {
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

template <class R, int SOLVER, int LIM>
cudaError_t launch2(const KParamsSC<R, 23>& p, int ng, cudaStream_t st) {
  cudaError_t e = big_smem(k_vl_march2<R, SOLVER, LIM>, march2_smem<R>());
  if (e != cudaSuccess) return e;
  // chunks of the 16 interior planes: as many as keep the grid within one wave of the 2 x 148 block slots (see k_vl_march1)
  const int chunks = std::max(1, std::min(8, kMarchSlots / ng)), per = (16 + chunks - 1) / chunks;
  k_vl_march2<R, SOLVER, LIM><<<dim3(ng, (16 + per - 1) / per), kM2P, march2_smem<R>(), st>>>(p, per);
  return cudaGetLastError();
}

template <class R, int SOLVER>
cudaError_t launch_solver(const KParamsSC<R, 23>& p, int ng, int lim, int pass, cudaStream_t st) {
  if (pass == 1) {
    // bulk copies need 16-byte aligned planes: the group strides are multiples of 16 bytes, the base pointers must be
    const bool no_tma = getenv("MHD_NO_TMA") != nullptr;      // read at every launch (tests switch it within one process)
    const bool tma = !no_tma && ((reinterpret_cast<size_t>(p.Uin) | reinterpret_cast<size_t>(p.Bin)) & 15) == 0;
    const int chunks = std::max(1, std::min(10, kMarchSlots / ng)), per = (20 + chunks - 1) / chunks;   // 20 half-step planes
    cudaError_t e;
    if (tma) {
      if ((e = big_smem(k_vl_march1<R, SOLVER, true>, march1_smem<R, true>())) != cudaSuccess) return e;
      k_vl_march1<R, SOLVER, true><<<dim3(ng, (20 + per - 1) / per), kMP, march1_smem<R, true>(), st>>>(p, per);
    } else {
      if ((e = big_smem(k_vl_march1<R, SOLVER, false>, march1_smem<R, false>())) != cudaSuccess) return e;
      k_vl_march1<R, SOLVER, false><<<dim3(ng, (20 + per - 1) / per), kMP, march1_smem<R, false>(), st>>>(p, per);
    }
    return cudaGetLastError();
  }
  switch (lim) {
    case 0: return launch2<R, SOLVER, 0>(p, ng, st);
    case 1: return launch2<R, SOLVER, 1>(p, ng, st);
    case 2: return launch2<R, SOLVER, 2>(p, ng, st);
    case 3: return launch2<R, SOLVER, 3>(p, ng, st);
    case 4: return launch2<R, SOLVER, 4>(p, ng, st);
    default: return launch2<R, SOLVER, 5>(p, ng, st);
  }
}

}  // namespace

// Roe: FP32 only (in FP64 the solver alone needs ~220 registers, a 484-thread block has 128 per thread); MHD_MARCH_ROE=0 keeps the
// fused first pass + staged kernels of round 1 for A/B runs
template <class R> bool vl_march_supports(int solver) {
  if (solver == kHLLD) return true;
  if (solver == kROE && sizeof(R) == 4) { const char* e = getenv("MHD_MARCH_ROE"); return !(e && e[0] == '0'); }
  return false;
}

template <class R>
cudaError_t launch_vl_march(const KParams<R>& p0, int ng, int solver, int lim, int pass, cudaStream_t st) {
  const KParamsSC<R, 23> p(p0);
  if (solver == kHLLD) return launch_solver<R, kHLLD>(p, ng, lim, pass, st);
  if constexpr (sizeof(R) == 4) {
    if (solver == kROE) return launch_solver<R, kROE>(p, ng, lim, pass, st);
  }
  return cudaErrorInvalidValue;
}

template cudaError_t launch_vl_march<float>(const KParams<float>&, int, int, int, int, cudaStream_t);
template cudaError_t launch_vl_march<double>(const KParams<double>&, int, int, int, int, cudaStream_t);
template bool vl_march_supports<float>(int);
template bool vl_march_supports<double>(int);

}  // namespace mhd

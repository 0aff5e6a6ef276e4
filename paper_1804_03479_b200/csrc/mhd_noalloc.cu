// mhd_noalloc.cu -- mhd_dt_reduce_noalloc (include/mhd.h): the CFL reduction S9 (R13) for callers that
// cannot allocate: no solver object, no cudaMalloc / cudaFree, no host synchronisation, the result stays on the device.
//
// The scratch memory of the reduction (one partial maximum per block and an arrival counter) is the file-scope array below: a fixed
// part of the library's device image, present on every GPU that loads libmhd.so until the process exits (kScratchBytes = 513 KB).
// In HOST code the array's name is a host-side stand-in, not a device address: the address the kernel gets comes from
// cudaGetSymbolAddress, asked once per device with that device current (scratch_of_current_device).
//
// Two-stage reduction in one launch: every block writes the largest speed of its 256 cells into its own slot, the block that
// arrives last (counter) takes the maximum of all slots and writes { dt, maxspeed } as doubles.  Maxima are exact, so the result
// has the bits of mhd_dt_reduce (one atomicMax per block on a solver-owned cell) whatever the arrival order.
// All calls share the array: the counter is cleared on the caller's stream before every launch (a memset node, not an allocation),
// the slots need no clearing (the last block reads only the slots this launch wrote).  Two calls that overlap on the GPU (different
// streams, or graphs replayed concurrently) race on the counter and the slots: serialise them.
#include <mutex>

#include "../../include/mhd.h"
#include "mhd_kernels3.cuh"

namespace mhd {
int note_cuda_failure(cudaError_t e, const char* where);      // mhd_api.cu: records the message mhd_strerror(MHD_ECUDA) returns
}

using namespace mhd;

namespace {

constexpr int kMaxBlocks = MHD_NOALLOC_MAX_BLOCKS;            // slots; a launch has ngroups * ceil(ps2^3 / 256) blocks
constexpr int kHead = 32;                                     // 256 bytes in front of the slots: [0] = arrival counter
constexpr size_t kScratchBytes = (size_t)(kHead + kMaxBlocks) * sizeof(unsigned long long);

static __device__ __align__(256) unsigned long long g_dt_scratch[kHead + kMaxBlocks];
static_assert(kScratchBytes == sizeof(unsigned long long) * (32 + 65536), "include/mhd.h states 513 KB");

constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned long long* g_scratch_addr[kMaxDevices] = {};         // device address of g_dt_scratch on each device, once asked

// device address of the scratch array on the CURRENT device (asked once per device)
int scratch_of_current_device(unsigned long long** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return note_cuda_failure(e, "mhd_dt_reduce_noalloc: cudaGetDevice");
  if (dev < 0 || dev >= kMaxDevices) return MHD_EINVAL;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    void* q = nullptr;
    e = cudaGetSymbolAddress(&q, g_dt_scratch);
    if (e != cudaSuccess) return note_cuda_failure(e, "mhd_dt_reduce_noalloc: cudaGetSymbolAddress(g_dt_scratch)");
    if (!q) return MHD_ECUDA;
    g_scratch_addr[dev] = static_cast<unsigned long long*>(q);
  }
  *out = g_scratch_addr[dev];
  return MHD_OK;
}

// largest value of the block's 256 threads, valid in thread 0
template <class R>
__device__ __forceinline__ R block_max256(R x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x = Num<R>::max(x, __shfl_xor_sync(0xffffffffu, x, o));
  __shared__ R part[8];
  __syncthreads();                                            // the second use in a kernel must not overtake the first one's reads
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = x;
  __syncthreads();
  R m = R(0);
  if (threadIdx.x < 32) {
    m = threadIdx.x < 8 ? part[threadIdx.x] : R(0);
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) m = Num<R>::max(m, __shfl_xor_sync(0xffffffffu, m, o));
  }
  return m;
}

// grid (ceil(N^3 / 256), 1, groups), 256 threads: the cell loop of k_dt (mhd_kernels3.cuh), the same cell_signal_speed
template <class R>
__global__ void __launch_bounds__(256) k_dt_noalloc(const R* __restrict__ U, const R* __restrict__ B, int N, int ng, long long nU,
                                                    long long nB, R gam, R min_dens, R min_pres, double cfl_dh,
                                                    unsigned long long* scratch, double* __restrict__ out) {
  const int T = N + 2 * ng;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  R smax = R(0);
  if (t < N * N * N) {
    const int i = t % N + ng, j = (t / N) % N + ng, k = t / (N * N) + ng;
    const R* u_ = U + (size_t)blockIdx.z * nU;
    const R* bx = B + (size_t)blockIdx.z * nB;
    const R* by = bx + (size_t)T * T * (T + 1);
    const R* bz = by + (size_t)T * T * (T + 1);
    const size_t T3 = (size_t)T * T * T, cq = ((size_t)k * T + j) * T + i;
    const size_t qx = ((size_t)k * T + j) * (T + 1) + i, qy = ((size_t)k * (T + 1) + j) * T + i;
    const R bl[3] = { bx[qx], by[qy], bz[cq] }, bu[3] = { bx[qx + 1], by[qy + T], bz[cq + (size_t)T * T] };
    const R u[5] = { u_[cq], u_[T3 + cq], u_[2 * T3 + cq], u_[3 * T3 + cq], u_[4 * T3 + cq] };
    smax = cell_signal_speed(u, bl, bu, gam, min_dens, min_pres);
  }
  const unsigned nblocks = gridDim.x * gridDim.z, me = blockIdx.z * gridDim.x + blockIdx.x;
  unsigned long long* slots = scratch + kHead;
  const R mine = block_max256(smax);
  __shared__ bool last;
  if (threadIdx.x == 0) {
    // speeds are >= 0 (or +inf for a NaN cell): their bit patterns order like the values (Bits, mhd_kernels3.cuh)
    slots[me] = (unsigned long long)Bits<R>::enc(mine);
    __threadfence();                                          // the slot is visible before the arrival is counted
    last = atomicAdd(scratch, 1ULL) == (unsigned long long)(nblocks - 1);
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  unsigned long long best = 0;
  for (unsigned b = threadIdx.x; b < nblocks; b += blockDim.x) best = max(best, __ldcg(slots + b));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
  __shared__ unsigned long long part[8];
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int w = 1; w < 8; ++w) best = max(best, part[w]);
    double s;
    if (sizeof(R) == 4) s = (double)__uint_as_float((unsigned)best); else s = __longlong_as_double((long long)best);
    out[0] = cfl_dh / s;                                      // dt = cfl * dh / maxspeed (the host path's expression)
    out[1] = s;
  }
}

template <class R>
cudaError_t launch(const void* U, const void* B, int N, int ng, int ngroups, double gamma, double min_dens, double min_pres,
                   double cfl_dh, unsigned long long* scratch, double* out, cudaStream_t st) {
  const int T = N + 2 * ng;
  const long long nU = 5LL * T * T * T, nB = 3LL * T * T * (T + 1);
  const dim3 grid((N * N * N + 255) / 256, 1, ngroups), blk(256);
  k_dt_noalloc<R><<<grid, blk, 0, st>>>(static_cast<const R*>(U), static_cast<const R*>(B), N, ng, nU, nB, (R)gamma, (R)min_dens,
                                         (R)min_pres, cfl_dh, scratch, out);
  return cudaGetLastError();
}

}  // namespace

extern "C" int mhd_dt_reduce_noalloc(int prec, const void* U, const void* B, int ngroups, int ps2, int nghost_of_arrays, double gamma,
                                     double min_dens, double min_pres, double dh, double cfl, double* dt_speed_out, void* cuda_stream) {
  if ((prec != MHD_FP32 && prec != MHD_FP64) || !U || !B || !dt_speed_out || ngroups < 1) return MHD_EINVAL;
  if (ps2 < 8 || ps2 > 64 || (ps2 & 1) || nghost_of_arrays < 0 || nghost_of_arrays > 8) return MHD_EINVAL;
  if (!(gamma > 1.0) || !(dh > 0.0) || !(cfl > 0.0)) return MHD_EINVAL;
  const long long per_group = ((long long)ps2 * ps2 * ps2 + 255) / 256;
  if ((long long)ngroups * per_group > kMaxBlocks || ngroups > 65535) return MHD_ELIMIT;      // beyond the fixed scratch array
  unsigned long long* scratch = nullptr;
  const int rc = scratch_of_current_device(&scratch);
  if (rc != MHD_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  cudaError_t e = cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), st);      // the arrival counter starts at zero
  if (e != cudaSuccess) return note_cuda_failure(e, "mhd_dt_reduce_noalloc: cudaMemsetAsync");
  const double cfl_dh = cfl * dh;
  e = prec == MHD_FP32 ? launch<float>(U, B, ps2, nghost_of_arrays, ngroups, gamma, min_dens, min_pres, cfl_dh, scratch, dt_speed_out, st)
                       : launch<double>(U, B, ps2, nghost_of_arrays, ngroups, gamma, min_dens, min_pres, cfl_dh, scratch, dt_speed_out, st);
  if (e != cudaSuccess) return note_cuda_failure(e, "k_dt_noalloc");
  return MHD_OK;
}

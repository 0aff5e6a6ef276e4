// mhd_kernels3.cuh -- stage kernels, part 3: full update with the coarse-fine boundary planes
// (PAPER.md:207), and the CFL reduction.  See mhd_kernels.cuh for the layout.
#pragma once
#include "mhd_kernels2.cuh"

namespace mhd {

// ---- S8: U^{n+1} = U^n - dt/dh sum dF2 (Eq. 10) on the N^3 interior cells, b^{n+1} by Eq. 13 on their faces;
// epilogue: time-centred fluxes and edge EMFs on the lower / mid / upper face planes of each
// direction, copied by the first 9 (N+1)^2 threads of the group (one per plane point (a2, a1), a1, a2 in [0, N]) -------
template <class R, int FBASE, class KP>
__device__ __forceinline__ void copy_planes(const KP& p, int grp, int t) {
  const int N = p.N, M = N + 1, g = p.g;
  if (t >= 9 * M * M) return;
  const int a1 = t % M, a2 = (t / M) % M, pl = t / (M * M);
  const int d = pl / 3, s = pl - 3 * d, t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  const int fi = (s == 0 ? 0 : (s == 1 ? N / 2 : N)) + g, c1 = a1 + g, c2 = a2 + g;
  // flat index with idx[d] = fi, idx[t1] = c1, idx[t2] = c2
  const int ix = d == 0 ? fi : (t1 == 0 ? c1 : c2), iy = d == 1 ? fi : (t1 == 1 ? c1 : c2), iz = d == 2 ? fi : (t1 == 2 ? c1 : c2);
  const int q = (iz * p.S + iy) * p.S + ix;
  const R* w = p.ws + (size_t)grp * p.narr * p.S3;
  if (p.fout && a1 < N && a2 < N) {
    const R* F = w + (size_t)(FBASE + 7 * d) * p.S3;
    const R f0 = F[q], fn = F[(size_t)p.S3 + q], f1 = F[(size_t)2 * p.S3 + q], f2 = F[(size_t)3 * p.S3 + q], f4 = F[(size_t)4 * p.S3 + q];
    R* fo = p.fout + (size_t)grp * p.nF + (size_t)pl * 5 * N * N + (size_t)a2 * N + a1;
    const size_t NN = (size_t)N * N;
    fo[0] = f0; fo[(size_t)(1 + d) * NN] = fn; fo[(size_t)(1 + t1) * NN] = f1; fo[(size_t)(1 + t2) * NN] = f2; fo[4 * NN] = f4;
  }
  if (p.eout) {
    R* e0 = p.eout + (size_t)grp * p.nE + (size_t)pl * 2 * M * N;
    R* e1 = e0 + (size_t)M * N;
    if (a1 < N) e0[(size_t)a2 * N + a1] = w[(size_t)(A_E + t1) * p.S3 + q];
    if (a2 < N) e1[(size_t)a2 * M + a1] = w[(size_t)(A_E + t2) * p.S3 + q];
  }
}

// largest signal speed of a cell (R13) from its conserved data and its six face fields
template <class R>
__device__ __forceinline__ R cell_signal_speed(const R (&u)[5], const R (&bl)[3], const R (&bu)[3], R gam, R min_dens, R min_pres) {
  const R Bc[3] = { R(0.5) * (bl[0] + bu[0]), R(0.5) * (bl[1] + bu[1]), R(0.5) * (bl[2] + bu[2]) };
  const R rho = Num<R>::max(u[0], min_dens);
  const R v[3] = { u[1] / rho, u[2] / rho, u[3] / rho };
  const R b2 = Bc[0] * Bc[0] + Bc[1] * Bc[1] + Bc[2] * Bc[2];
  R P = (gam - R(1)) * (u[4] - R(0.5) * rho * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]) - R(0.5) * b2);
  P = Num<R>::max(P, min_pres);
  R smax = R(0);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const R bn2 = Bc[d] * Bc[d];
    smax = Num<R>::max(smax, Num<R>::abs(v[d]) + fast_speed(rho, P, bn2, b2 - bn2, gam));
  }
  // fmax drops a NaN operand, and a NaN density / energy is replaced by the floors above: a cell with any NaN input reports an
  // infinite speed, which survives every maximum and makes the reducing call fail with MHD_ESTATE instead of returning a finite dt
  const R chk = ((u[0] + u[1]) + (u[2] + u[3])) + (u[4] + b2);
  return (chk == chk && smax == smax) ? smax : R(INFINITY);
}
// speeds are >= 0, so their IEEE bit patterns order like unsigned integers: one atomicMax per block
template <class R> struct Bits;
template <> struct Bits<float> {
  typedef unsigned int U;
  static __device__ __forceinline__ U enc(float x) { return __float_as_uint(x); }
};
template <> struct Bits<double> {
  typedef unsigned long long U;
  static __device__ __forceinline__ U enc(double x) { return (U)__double_as_longlong(x); }
};
// block of 256 threads, every thread calls
template <class R>
__device__ __forceinline__ void block_max_to(R smax, unsigned long long* out) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) smax = Num<R>::max(smax, __shfl_xor_sync(0xffffffffu, smax, o));
  __shared__ R red[8];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = smax;
  __syncthreads();
  if (threadIdx.x < 32) {
    R m = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : R(0);
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) m = Num<R>::max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (threadIdx.x == 0) atomicMax(reinterpret_cast<typename Bits<R>::U*>(out), Bits<R>::enc(m));
  }
}

// DT (mhd_advance_dt): S9 on the cell's own new state in the same kernel -- the thread also evaluates the upper faces of
// its cell (the same expression as the neighbour's lower face, hence the same bits) and the block reduces the speeds
template <class R, int FBASE, int SC, bool DT>
__global__ void __launch_bounds__(256, OccFinal<R>::minb) k_final(const KParamsSC<R, SC> p, const Box3 box) {
  typedef KParamsSC<R, SC> KP;
  Ctx<R, KP> c(p, box);
  if (p.fout || p.eout) copy_planes<R, FBASE>(p, blockIdx.z, blockIdx.x * blockDim.x + threadIdx.x);
  if (!DT && !c.ok) return;
  R smax = R(0);
  if (c.ok) {
    const int g = p.g, N = p.N;
    const int ii = c.i - g, jj = c.j - g, kk = c.k - g;
    const R qh = p.dt / p.dh;
    R u[5], dU[5];
    load_U_in(p, c, u);
    flux_div<FBASE>(c, dU);
    R* Uo = p.Uout + (size_t)c.grp * p.nUo;
    const size_t N3 = (size_t)N * N * N, cq = ((size_t)kk * N + jj) * N + ii;
#pragma unroll
    for (int v = 0; v < 5; ++v) { u[v] = u[v] - qh * dU[v]; Uo[v * N3 + cq] = u[v]; }
    R* Bx = p.Bout + (size_t)c.grp * p.nBo;
    R* By = Bx + (size_t)N * N * (N + 1);
    R* Bz = By + (size_t)N * N * (N + 1);
    const int q = c.q;
    R bl[3], bu[3];
    bl[0] = ct_face<R, 0>(c, c.arr(A_B + 0), q, qh);
    bl[1] = ct_face<R, 1>(c, c.arr(A_B + 1), q, qh);
    bl[2] = ct_face<R, 2>(c, c.arr(A_B + 2), q, qh);
    Bx[((size_t)kk * N + jj) * (N + 1) + ii] = bl[0];
    By[((size_t)kk * (N + 1) + jj) * N + ii] = bl[1];
    Bz[((size_t)kk * N + jj) * N + ii] = bl[2];
    if (DT || ii == N - 1) bu[0] = ct_face<R, 0>(c, c.arr(A_B + 0), q + 1, qh);
    if (DT || jj == N - 1) bu[1] = ct_face<R, 1>(c, c.arr(A_B + 1), q + p.S, qh);
    if (DT || kk == N - 1) bu[2] = ct_face<R, 2>(c, c.arr(A_B + 2), q + p.S2, qh);
    if (ii == N - 1) Bx[((size_t)kk * N + jj) * (N + 1) + N] = bu[0];
    if (jj == N - 1) By[((size_t)kk * (N + 1) + N) * N + ii] = bu[1];
    if (kk == N - 1) Bz[((size_t)N * N + jj) * N + ii] = bu[2];
    if (DT) {
#pragma unroll
      for (int v = 0; v < 5; ++v) opaque(u[v]);
#pragma unroll
      for (int v = 0; v < 3; ++v) { opaque(bl[v]); opaque(bu[v]); }
      smax = cell_signal_speed(u, bl, bu, p.gam, p.min_dens, p.min_pres);
    }
  }
  if (DT) block_max_to(smax, p.red);
}

// ---- S9: CFL (R13): max over interior cells and directions of |v_d| + c_f,d -------------------
template <class R>
__global__ void __launch_bounds__(256) k_dt(const R* __restrict__ U, const R* __restrict__ B, int N, int ng, long long nU,
                                            long long nB, R gam, R min_dens, R min_pres, unsigned long long* out) {
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
  block_max_to(smax, out);
}

// ---- register-only FMA chains: measured FP32 / FP64 FMA peak (ALU roofline denominator) ----------------
template <class R>
__global__ void __launch_bounds__(256) k_fma_peak(R* out, int iters) {
  R a[8], x = R(1.0000001), y = R(1e-9) * threadIdx.x;
#pragma unroll
  for (int v = 0; v < 8; ++v) a[v] = R(v) + y;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int v = 0; v < 8; ++v) a[v] = a[v] * x + y;
  }
  R s = R(0);
#pragma unroll
  for (int v = 0; v < 8; ++v) s += a[v];
  if (s == R(-1)) out[0] = s;
}

}  // namespace mhd

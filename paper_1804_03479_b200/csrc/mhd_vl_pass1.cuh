// mhd_vl_pass1.cuh -- VL steps S0 + S1 + S2 of the standard patch group (N = 16, 3 ghost cells) in ONE kernel
// (PAPER.md:191): stage the tile, primitives, first-order fluxes with the face-centred normal field.
//
// The staged path writes the primitives (k_load_prim) and reads them back twice per direction (k_flux1_vl).  Here one
// block owns the x-y plane of the tile (22 x 22 cells, one thread per cell) and marches over a chunk of planes along z:
// the primitives of the plane go to shared memory for the x- and y-neighbours, the plane below stays in registers for
// the z-face, so every Riemann solve takes its left state from shared memory or registers and its right state from
// registers.  Of the primitives only the density goes to memory (the EMF kernel reads it beside the reference EMFs).
// Same device functions and operands as the staged kernels; values the staged path rounds by storing pass through an
// empty asm (no multiply of one stage contracted with an add of the next); last-bit differences to the staged kernels
// remain (see mhd_ctu_pass1.cuh).  Measured (B200, 512 groups, HLLD): FP32 0.32 ms against 0.16 + 0.29 ms for
// k_load_prim + k_flux1_vl, FP64 0.69 ms against 0.30 + 0.56 ms; Roe FP32 (one block, 128 registers) 0.55 ms against
// 0.16 + 0.57 ms; Roe FP64 spills (2.30 ms against 2.17 ms) and keeps the staged kernels.
#pragma once
#include "mhd_ctu_pass1.cuh"

namespace mhd {

constexpr int kV1T = 22;                     // tile width of the standard VL group
constexpr int kV1Threads = kV1T * kV1T;      // 484
#ifndef MHD_V1_CHUNK
#define MHD_V1_CHUNK 4
#endif
constexpr int kV1Chunk = MHD_V1_CHUNK;       // planes per block (+ one recomputed plane of primitives below the chunk)

// generic 1-D state of direction D from the 8 primitives (rho, vx, vy, vz, P, Bcx, Bcy, Bcz)
template <class R, int D>
__device__ __forceinline__ void gen_from_prim(const R (&W)[8], R (&w)[7]) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  w[0] = W[0]; w[1] = W[1 + D]; w[2] = W[1 + T1]; w[3] = W[1 + T2]; w[4] = W[4]; w[5] = W[5 + T1]; w[6] = W[5 + T2];
}
template <class R, int D>
__device__ __forceinline__ void gen_from_smem(const R* __restrict__ sW, int t, R (&w)[7]) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  w[0] = sW[t]; w[1] = sW[(1 + D) * kV1Threads + t]; w[2] = sW[(1 + T1) * kV1Threads + t]; w[3] = sW[(1 + T2) * kV1Threads + t];
  w[4] = sW[4 * kV1Threads + t]; w[5] = sW[(5 + T1) * kV1Threads + t]; w[6] = sW[(5 + T2) * kV1Threads + t];
}

template <class R, bool COUNT, class KP>
__device__ __forceinline__ void v1_load_prim(const KP& p, const R* __restrict__ U, const R* __restrict__ Bx, const R* __restrict__ By,
                                             const R* __restrict__ Bz, int i, int j, int k, R (&bl)[3], R (&W)[8]) {
  constexpr int T = kV1T;
  R bu[3], u[5];
  bl[0] = Bx[(k * T + j) * (T + 1) + i]; bu[0] = Bx[(k * T + j) * (T + 1) + i + 1];
  bl[1] = By[(k * (T + 1) + j) * T + i]; bu[1] = By[(k * (T + 1) + j + 1) * T + i];
  bl[2] = Bz[(k * T + j) * T + i];       bu[2] = Bz[((k + 1) * T + j) * T + i];
  const int cq = (k * T + j) * T + i;
#pragma unroll
  for (int v = 0; v < 5; ++v) u[v] = U[v * T * T * T + cq];
  cons_to_prim<COUNT>(p, u, bl, bu, W);
#pragma unroll
  for (int v = 0; v < 8; ++v) opaque(W[v]);
}

// grid: (ceil(22 / kV1Chunk) chunks, 1, groups); 484 threads; static shared memory 2 x 8 x 484 values.
// (Tried: staging the next plane's 11 inputs per thread through shared memory with cp.async while the solves run --
// slower, 0.46 against 0.39 ms: eleven 4-byte asynchronous copies per thread cost more than the latency they hide.)
// FP32 HLLD: two resident blocks (64 registers), the plane buffer double-buffered (one barrier per plane); FP64 and Roe:
// one block (up to 128 registers); FP64 with a single buffer inside the 48 KB of static shared memory and a second
// barrier per plane
template <class R, int SOLVER, int SC>
__global__ void __launch_bounds__(kV1Threads, (sizeof(R) == 4 && SOLVER != kROE) ? 2 : 1) k_vl_pass1(const KParamsSC<R, SC> p) {
  constexpr int T = kV1T;
  constexpr int NBUF = sizeof(R) == 4 ? 2 : 1;
  __shared__ R sWbuf[NBUF * 8 * kV1Threads];
  const int t = threadIdx.x, i = t % T, j = t / T, grp = blockIdx.z;
  const int k0 = blockIdx.x * kV1Chunk, k1 = min(k0 + kV1Chunk, T);
  const int S = p.S, S3 = p.S3;
  R* w = p.ws + (size_t)grp * p.narr * S3;
  auto arr = [&](int x) { return w + (size_t)x * S3; };
  const R* U = p.Uin + (size_t)grp * p.nUi;
  const R* Bx = p.Bin + (size_t)grp * p.nBi;
  const R* By = Bx + T * T * (T + 1);
  const R* Bz = By + T * T * (T + 1);
  R Wp[8], bl[3];
  if (k0 > 0) v1_load_prim<R, false>(p, U, Bx, By, Bz, i, j, k0 - 1, bl, Wp);     // plane below the chunk: primitives only
  for (int k = k0; k < k1; ++k) {
    R* sW = sWbuf + (NBUF == 2 ? (k & 1) : 0) * 8 * kV1Threads;
    R W[8];
    v1_load_prim<R, true>(p, U, Bx, By, Bz, i, j, k, bl, W);
    const int q = (k * S + j) * S + i;
    // of the primitives only the density is read again (by the EMF kernel, beside the reference EMFs): the rest of W
    // lives in shared memory and registers for the solves below and never goes to memory
    arr(A_W)[q] = W[0];
#pragma unroll
    for (int v = 0; v < 8; ++v) sW[v * kV1Threads + t] = W[v];
    arr(A_EC + 0)[q] = W[3] * W[6] - W[2] * W[7];
    arr(A_EC + 1)[q] = W[1] * W[7] - W[3] * W[5];
    arr(A_EC + 2)[q] = W[2] * W[5] - W[1] * W[6];
    arr(A_B + 0)[q] = bl[0]; arr(A_B + 1)[q] = bl[1]; arr(A_B + 2)[q] = bl[2];
    __syncthreads();                       // the other buffer is free again: every thread left plane k-1 before this barrier
    R wl[7], wr[7], F[7];
    if (i >= 1) {
      gen_from_smem<R, 0>(sW, t - 1, wl); gen_from_prim<R, 0>(W, wr);
      if (riemann<R, SOLVER>(wl, wr, bl[0], p.gam, p.gm1inv, F)) count_event(p.stats + 2);
#pragma unroll
      for (int v = 0; v < 7; ++v) arr(A_F + v)[q] = F[v];
    }
    if (j >= 1) {
      gen_from_smem<R, 1>(sW, t - T, wl); gen_from_prim<R, 1>(W, wr);
      if (riemann<R, SOLVER>(wl, wr, bl[1], p.gam, p.gm1inv, F)) count_event(p.stats + 2);
#pragma unroll
      for (int v = 0; v < 7; ++v) arr(A_F + 7 + v)[q] = F[v];
    }
    if (k >= 1) {
      gen_from_prim<R, 2>(Wp, wl); gen_from_prim<R, 2>(W, wr);
      if (riemann<R, SOLVER>(wl, wr, bl[2], p.gam, p.gm1inv, F)) count_event(p.stats + 2);
#pragma unroll
      for (int v = 0; v < 7; ++v) arr(A_F + 14 + v)[q] = F[v];
    }
#pragma unroll
    for (int v = 0; v < 8; ++v) Wp[v] = W[v];
    if (NBUF == 1) __syncthreads();        // single buffer: everybody has read plane k before it is overwritten
  }
}

}  // namespace mhd

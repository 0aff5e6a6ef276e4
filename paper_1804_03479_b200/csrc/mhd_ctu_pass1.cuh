// mhd_ctu_pass1.cuh -- CTU steps 1 + 2 of the standard patch group (N = 16, 4 ghost cells, PPM) in ONE kernel
// (PAPER.md:176-177): limited slopes, PPM parabola + half-step tracing + primitive source terms, pass-1 Riemann solve.
//
// The staged path runs three kernels (k_slope_ctu -> k_recon_ctu -> k_flux_lr) that hand 21 slope arrays and 42 state
// arrays to each other through HBM.  All three are one-dimensional along the sweep direction D, so a thread block that
// owns complete PENCILS along D needs nothing from any other block: one block = one plane of the tile that contains D
// (24 cells along D x 20 across, one thread per cell, x always the fastest thread index so that rows stay coalesced);
// slopes and upper states travel to the neighbour along D through shared memory.  Nothing is computed twice; the
// states still go to memory once (step 5 needs them), the slopes never do, and the Riemann solve reads its left state
// from shared memory and its right state from registers.  Same device functions as the staged kernels, same operands;
// the values that the staged path rounds by storing them (slopes, states) pass through an empty asm here, so that no
// multiply of one stage is contracted with an add of the next.  The result still differs from the staged kernels in
// the last bit of some values (the compiler orders and contracts the arithmetic inside a stage differently when the
// stages share one function: measured <= 1e-7 of max|U|, 5e-7 of the fluxes, 3e-6 of the edge EMFs in FP32); the parity
// tests against the oracle run through this kernel, and tests/test_gpu_api.py bounds the difference to the staged path.
// Measured (B200, 512 groups, HLLD): FP32 0.74 ms against 1.14 ms for the three kernels (two resident 480-thread blocks, 64
// registers).  FP64 needs 128 registers: one 480-thread block 2.18 ms, two half-plane blocks (ACROSS = 10) 1.95 ms on one
// box and 2.15 ms on another against 2.16 ms staged; Roe needs ~110 FP32 registers: 1.29 ms against 1.29 ms staged.
// FP64, Roe, other limiters, PLM and other group sizes keep the staged kernels.
#pragma once
#include "mhd_kernels2.cuh"

namespace mhd {

// opaque(): mhd_kernels.cuh

constexpr int kP1Along = 24;                       // cells along D: the whole tile, T = 24
constexpr int kP1Across = 20;                      // cells across: g-2 .. g+N+1
// a block covers ACROSS of the 20 cells across (20: the whole plane, 480 threads; 10: half of it, 240 threads)

template <class R, int SOLVER, int LIM, int ACROSS, int D, class KP>
__device__ __forceinline__ void ctu_pass1_plane(const KP& p, R* __restrict__ sm, int grp, int plane, int part) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  constexpr int kP1Threads = kP1Along * ACROSS;
  constexpr int sD = D == 0 ? 1 : ACROSS;          // distance of the neighbour along D in the block
  const int t = threadIdx.x;
  const int g = p.g, lo = g - 1;
  // a: index along D (0 .. 23 <-> tile cell a), b: in-plane index across, plane: the third axis
  int a, b;
  if (D == 0) { a = t % kP1Along; b = t / kP1Along; } else { b = t % ACROSS; a = t / ACROSS; }
  const int ta = lo - 1 + part * ACROSS + b, tp = lo - 1 + plane;  // tile indices across / of the plane
  const int i = D == 0 ? a : ta, j = D == 1 ? a : (D == 0 ? ta : tp), k = D == 2 ? a : tp;
  const int S = p.S, S2 = p.S2, S3 = p.S3;
  const int q = (k * S + j) * S + i;
  const int od = D == 0 ? 1 : (D == 1 ? S : S2), o1 = T1 == 0 ? 1 : (T1 == 1 ? S : S2), o2 = T2 == 0 ? 1 : (T2 == 1 ? S : S2);
  R* w = p.ws + (size_t)grp * p.narr * S3;
  auto arr = [&](int x) { return w + (size_t)x * S3; };
  R* sW = sm;                                       // [7][480] primitives
  R* sS = sm + 7 * kP1Threads;                      // [7][480] limited slopes
  R* sU = sm + 14 * kP1Threads;                     // [7][480] upper-face states
  // ---- phase 1: primitives of the pencil ----
  R w0[7];
  load_gen<R, D>(arr(A_W), S3, q, w0);
  const R bnc = arr(A_W + 5 + D)[q];
#pragma unroll
  for (int v = 0; v < 7; ++v) sW[v * kP1Threads + t] = w0[v];
  __syncthreads();
  // ---- phase 2: limited slopes (cells 1 .. 22) ----
  R wm[7], wp[7], s0[7];
  const bool has_nb = a >= 1 && a <= kP1Along - 2;
  if (has_nb) {
#pragma unroll
    for (int v = 0; v < 7; ++v) { wm[v] = sW[v * kP1Threads + t - sD]; wp[v] = sW[v * kP1Threads + t + sD]; }
    slope3<R, LIM>(wm, w0, wp, bnc, p.gam, s0);
#pragma unroll
    for (int v = 0; v < 7; ++v) { opaque(s0[v]); sS[v * kP1Threads + t] = s0[v]; }
  }
  __syncthreads();
  // ---- phase 3: parabola, tracing, source terms (cells 2 .. 21): the states go to memory and the upper one to the block ----
  R wlo[7], wup[7];
  const bool rec = a >= 2 && a <= kP1Along - 3;
  if (rec) {
    R sm_[7], sp_[7];
#pragma unroll
    for (int v = 0; v < 7; ++v) { sm_[v] = sS[v * kP1Threads + t - sD]; sp_[v] = sS[v * kP1Threads + t + sD]; }
    const R sig = p.dt / p.dh, hdt = R(0.5) * p.dt;
    ppm_trace(wm, w0, wp, sm_, s0, sp_, bnc, p.gam, sig, wlo, wup);
    const R* bn_ = arr(A_B + D); const R* b1_ = arr(A_B + T1); const R* b2_ = arr(A_B + T2);
    const R idh = R(1) / p.dh;
    const R dbn = (bn_[q + od] - bn_[q]) * idh;
    const R db1 = (b1_[q + o1] - b1_[q]) * idh;
    const R db2 = (b2_[q + o2] - b2_[q]) * idh;
    const R s1 = hdt * w0[2] * lim_minmod(dbn, -db1), s2 = hdt * w0[3] * lim_minmod(dbn, -db2);
    wlo[5] += s1; wup[5] += s1; wlo[6] += s2; wup[6] += s2;
    apply_floors(p, wlo); apply_floors(p, wup);
    // step 5 + 6 reads the lower state of cells g .. g+N and the upper state of cells g-1 .. g+N-1 along D, across
    // g-1 .. g+N: only those go to memory (the pass-1 solve below takes its states from the block)
    const bool keep = ta >= g - 1 && ta <= g + p.N && tp >= g - 1 && tp <= g + p.N;
    const bool keep_lo = keep && a >= g && a <= g + p.N, keep_up = keep && a >= g - 1 && a <= g + p.N - 1;
#pragma unroll
    for (int v = 0; v < 7; ++v) {
      opaque(wlo[v]); opaque(wup[v]);
      if (keep_lo) arr(A_LO + 7 * D + v)[q] = wlo[v];
      if (keep_up) arr(A_UP + 7 * D + v)[q] = wup[v];
      sU[v * kP1Threads + t] = wup[v];
    }
  }
  __syncthreads();
  // ---- phase 4: pass-1 Riemann solve on the lower face of cells 3 .. 21 ----
  if (a >= 3 && a <= kP1Along - 3) {
    R wl[7], F[7];
#pragma unroll
    for (int v = 0; v < 7; ++v) wl[v] = sU[v * kP1Threads + t - sD];
    const bool fb = riemann<R, SOLVER>(wl, wlo, arr(A_B + D)[q], p.gam, p.gm1inv, F);
    if (fb) count_event(p.stats + 2);
#pragma unroll
    for (int v = 0; v < 7; ++v) arr(A_F + 7 * D + v)[q] = F[v];
  }
}

// grid: (20 planes x 20 / ACROSS parts, 3 directions, groups); 24 * ACROSS threads; dynamic shared memory 21 * threads * sizeof(R)
// resident blocks per SM asked from ptxas: FP32 HLLD fits the 68 registers that two 480-thread blocks leave (64, no spill)
template <class R, int SOLVER> struct OccPass1 { static constexpr int minb = 2; };

template <class R, int SOLVER, int LIM, int ACROSS, int SC>
__global__ void __launch_bounds__(kP1Along * ACROSS, OccPass1<R, SOLVER>::minb) k_ctu_pass1(const KParamsSC<R, SC> p) {
  extern __shared__ unsigned char smem_raw[];
  R* sm = reinterpret_cast<R*>(smem_raw);
  constexpr int parts = kP1Across / ACROSS;
  const int plane = blockIdx.x / parts, part = blockIdx.x - plane * parts;
  switch (blockIdx.y) {
    case 0: ctu_pass1_plane<R, SOLVER, LIM, ACROSS, 0>(p, sm, blockIdx.z, plane, part); break;
    case 1: ctu_pass1_plane<R, SOLVER, LIM, ACROSS, 1>(p, sm, blockIdx.z, plane, part); break;
    default: ctu_pass1_plane<R, SOLVER, LIM, ACROSS, 2>(p, sm, blockIdx.z, plane, part); break;
  }
}

}  // namespace mhd

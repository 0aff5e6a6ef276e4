// mhd_grid.cuh -- device-side preparation and closing steps for a uniform periodic grid.
//
// The paper's host layer copies patch data into ghost-zoned patch groups before the solver call ("preparation",
// PAPER.md:236-244) and stores the results back afterwards ("closing").  For a uniform periodic grid both are pure
// data movement; doing them on the device keeps multi-step runs (BASELINE configs 3, 4) entirely in HBM.
//
// Grid layout (as paper_1804_03479_b200/inputs.py): U[5][nz][ny][nx], bx[nz][ny][nx+1], by[nz][ny+1][nx],
// bz[nz+1][ny][nx], x fastest; the last face of each periodic direction duplicates the first.
// Group g = (gz*my + gy)*mx + gx (gx fastest) covers cells [gx*N, (gx+1)*N) x ... plus `ng` ghost cells per side.
#pragma once
#include "mhd_kernels3.cuh"

namespace mhd {

struct GridDims { int nx, ny, nz, mx, my, mz; };

__device__ __forceinline__ int wrap(int i, int n) { i %= n; return i < 0 ? i + n : i; }

// ---- preparation: one thread per point of the (T+1)^3 index space of a group -------------------------------------
template <class R>
__global__ void __launch_bounds__(256) k_grid_pack(const R* __restrict__ U, const R* __restrict__ bx, const R* __restrict__ by,
                                                   const R* __restrict__ bz, GridDims d, int N, int ng,
                                                   R* __restrict__ Uin, R* __restrict__ Bin) {
  const int T = N + 2 * ng, S = T + 1;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= S * S * S) return;
  const int i = t % S, j = (t / S) % S, k = t / (S * S);
  const int grp = blockIdx.z, gx = grp % d.mx, gy = (grp / d.mx) % d.my, gz = grp / (d.mx * d.my);
  // global cell / face indices of tile point (i,j,k); a face index f wraps like a cell index (face n == face 0)
  const int ix = wrap(gx * N + i - ng, d.nx), jy = wrap(gy * N + j - ng, d.ny), kz = wrap(gz * N + k - ng, d.nz);
  const size_t nUi = (size_t)5 * T * T * T, nf = (size_t)T * T * (T + 1);
  R* Bxo = Bin + (size_t)grp * 3 * nf;
  R* Byo = Bxo + nf;
  R* Bzo = Byo + nf;
  if (j < T && k < T) Bxo[((size_t)k * T + j) * (T + 1) + i] = bx[((size_t)kz * d.ny + jy) * (d.nx + 1) + ix];
  if (i < T && k < T) Byo[((size_t)k * (T + 1) + j) * T + i] = by[((size_t)kz * (d.ny + 1) + jy) * d.nx + ix];
  if (i < T && j < T) Bzo[((size_t)k * T + j) * T + i] = bz[((size_t)kz * d.ny + jy) * d.nx + ix];
  if (i < T && j < T && k < T) {
    const size_t n3 = (size_t)d.nx * d.ny * d.nz, src = ((size_t)kz * d.ny + jy) * d.nx + ix;
    const size_t T3 = (size_t)T * T * T, dst = ((size_t)k * T + j) * T + i;
    R* Uo = Uin + (size_t)grp * nUi;
#pragma unroll
    for (int v = 0; v < 5; ++v) Uo[v * T3 + dst] = U[v * n3 + src];
  }
}

// ---- closing: one thread per interior cell of a group; each cell owns its three lower faces ------------------------
template <class R>
__global__ void __launch_bounds__(256) k_grid_unpack(const R* __restrict__ Uout, const R* __restrict__ Bout, GridDims d, int N,
                                                     R* __restrict__ U, R* __restrict__ bx, R* __restrict__ by, R* __restrict__ bz) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= N * N * N) return;
  const int i = t % N, j = (t / N) % N, k = t / (N * N);
  const int grp = blockIdx.z, gx = grp % d.mx, gy = (grp / d.mx) % d.my, gz = grp / (d.mx * d.my);
  const int ix = gx * N + i, jy = gy * N + j, kz = gz * N + k;
  const size_t N3 = (size_t)N * N * N, nf = (size_t)N * N * (N + 1);
  const R* Ug = Uout + (size_t)grp * 5 * N3;
  const R* Bxg = Bout + (size_t)grp * 3 * nf;
  const R* Byg = Bxg + nf;
  const R* Bzg = Byg + nf;
  const size_t n3 = (size_t)d.nx * d.ny * d.nz, dst = ((size_t)kz * d.ny + jy) * d.nx + ix;
#pragma unroll
  for (int v = 0; v < 5; ++v) U[v * n3 + dst] = Ug[v * N3 + t];
  const R vx = Bxg[((size_t)k * N + j) * (N + 1) + i];
  const R vy = Byg[((size_t)k * (N + 1) + j) * N + i];
  const R vz = Bzg[((size_t)k * N + j) * N + i];
  bx[((size_t)kz * d.ny + jy) * (d.nx + 1) + ix] = vx;
  by[((size_t)kz * (d.ny + 1) + jy) * d.nx + ix] = vy;
  bz[((size_t)kz * d.ny + jy) * d.nx + ix] = vz;
  if (ix == 0) bx[((size_t)kz * d.ny + jy) * (d.nx + 1) + d.nx] = vx;          // periodic duplicate: face n == face 0
  if (jy == 0) by[((size_t)kz * (d.ny + 1) + d.ny) * d.nx + ix] = vy;
  if (kz == 0) bz[((size_t)d.nz * d.ny + jy) * d.nx + ix] = vz;
}

// ---- CFL reduction on the grid layout (same arithmetic as k_dt) ----------------------------------------------------
template <class R>
__global__ void __launch_bounds__(256) k_dt_grid(const R* __restrict__ U, const R* __restrict__ bx, const R* __restrict__ by,
                                                 const R* __restrict__ bz, GridDims d, R gam, R min_dens, R min_pres,
                                                 unsigned long long* out) {
  const size_t n3 = (size_t)d.nx * d.ny * d.nz;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  R smax = R(0);
  if (t < n3) {
    const int i = (int)(t % d.nx), j = (int)((t / d.nx) % d.ny), k = (int)(t / ((size_t)d.nx * d.ny));
    const size_t qx = ((size_t)k * d.ny + j) * (d.nx + 1) + i, qy = ((size_t)k * (d.ny + 1) + j) * d.nx + i;
    const R bl[3] = { bx[qx], by[qy], bz[t] }, bu[3] = { bx[qx + 1], by[qy + d.nx], bz[t + (size_t)d.nx * d.ny] };
    const R u[5] = { U[t], U[n3 + t], U[2 * n3 + t], U[3 * n3 + t], U[4 * n3 + t] };
    smax = cell_signal_speed(u, bl, bu, gam, min_dens, min_pres);
  }
  block_max_to(smax, out);
}

}  // namespace mhd

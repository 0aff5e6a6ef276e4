// mhd_vl_march.cuh -- the VL step of the standard patch group (N = 16, 3 ghost cells, PLM) as TWO plane-marching kernels
// with every intermediate of a pass on chip ("one CUDA thread block per patch group"):
//
//   k_vl_march1 : S0 + S1 + S2 + S3 + S4   tile -> primitives -> first-order fluxes -> edge EMFs -> half-step state
//   k_vl_march2 : S5 + S6 + S7 + S8 (+ S9) PLM at the half step -> fluxes -> edge EMFs -> full update, planes, CFL speed
//
// One block owns one patch group and marches along z; a thread owns the cell (i, j) of the current x-y plane.  At plane k
// it solves the Riemann problems of the cell's three LOWER faces (x, y in the plane, z between planes k-1 and k), puts
// the fluxes into shared memory, and after a barrier every thread has what the scheme needs from its neighbours:
//   * the flux differences of its cell in x and y (the z difference closes one plane later),
//   * the three edge EMFs through the cell's lowest corner: E_z in the plane, E_x and E_y on the level k-1/2 (they need the
//     y / x face data and the reference EMFs of plane k-1: four values carried in registers, the rest double-buffered),
//   * with them the CT update of the lower faces and, one plane behind, the finished cell (k-1).
// Nothing but the half-step primitives and face fields (11 arrays of 22^3 per group) goes to memory between the two
// kernels: the 21 flux arrays, 3 EMF arrays, 3 reference-EMF arrays and the copies of the face field of the staged path
// (mhd_kernels*.cuh), and the second read of all of them, are gone.  Same device functions as the staged kernels (solvers,
// slopes, upwind switch, con -> prim); the sums of Eq. 10 / Eq. 13 are associated as (in-plane part - lower z term) + upper
// z term, so results agree with the staged kernels to rounding, not bitwise (a uniform state is still an exact fixed point).
#pragma once
#include "mhd_vl_pass1.cuh"
#include "mhd_kernels3.cuh"

namespace mhd {

constexpr int kMT = 22, kMP = kMT * kMT;          // tile width, cells per plane (= threads of k_vl_march1)
constexpr int kM2W = 18, kM2P = kM2W * kM2W;      // pass 2 runs on cells [2, 20)^2 of the plane: 324 threads
enum : int { M_WH = 0, M_BH = 8, M_END = 11 };    // workspace of the fused path: arrays of 22^3 (pitch 22): Wh[8], bh[3]
constexpr int kMWS = M_END * kMT * kMT * kMT;     // values per group: a multiple of 4, so every plane of every group is 16-byte aligned

// SURVEY C6 / DESIGN.md R10, R10a for the edge through the lowest corner of cell q = (a, b); qa = (a-1, b), qb = (a, b-1),
// qab = (a-1, b-1).  Same expression, same order as emf_dir (mhd_kernels.cuh).
template <class R>
__device__ __forceinline__ R edge_emf(R Ea_q, R Ea_qb, R Eb_q, R Eb_qa, R ma_qb, R ma_q, R mb_qa, R mb_q, R ec_q, R ec_qa,
                                      R ec_qb, R ec_qab, R r_q, R r_qa, R r_qb, R r_qab, R ht) {
  R e = R(0.25) * (Ea_q + Ea_qb + Eb_q + Eb_qa);
  e += R(0.25) * (upwind(ma_qb, ht * (r_qab + r_qb), Eb_qa - ec_qab, Eb_q - ec_qb) - upwind(ma_q, ht * (r_qa + r_q), ec_qa - Eb_qa, ec_q - Eb_q));
  e += R(0.25) * (upwind(mb_qa, ht * (r_qab + r_qa), Ea_qb - ec_qab, Ea_q - ec_qa) - upwind(mb_q, ht * (r_qb + r_q), ec_qb - Ea_qb, ec_q - Ea_q));
  return e;
}

// The three edge EMFs through the lowest corner of the thread's cell from the flux planes in shared memory.
//   sF : [21][P] fluxes of the lower x / y / z faces of the plane's cells, generic component order (7 per direction)
//   Cc / Cp : [3][P] reference EMFs (x, y, z) of the cells of this plane / of the plane below; rc / rp : their densities
//   pF* : the thread's own x / y face data of the plane below (mass flux, E_y from the x face, mass flux, -E_x from the y face)
// t = index of the cell in the plane, ox / oy = offsets of the x / y neighbour
template <class R, int P>
__device__ __forceinline__ void march_emfs(const R* __restrict__ sF, const R* __restrict__ Cc, const R* __restrict__ Cp,
                                           const R* __restrict__ rc, const R* __restrict__ rp, int t, int ox, int oy, R pFx0, R pFx6,
                                           R pFy0, R pFy5, R ht, bool below, R& Ex, R& Ey, R& Ez) {
  const R* Fx = sF; const R* Fy = sF + 7 * P; const R* Fz = sF + 14 * P;
  // E_z at (i-1/2, j-1/2, k): a = x, b = y; from an x face E_z = -F[5], from a y face E_z = +F[6]
  Ez = edge_emf<R>(-Fx[5 * P + t], -Fx[5 * P + t - oy], Fy[6 * P + t], Fy[6 * P + t - ox], Fx[t - oy], Fx[t], Fy[t - ox], Fy[t],
                   Cc[2 * P + t], Cc[2 * P + t - ox], Cc[2 * P + t - oy], Cc[2 * P + t - ox - oy], rc[t], rc[t - ox], rc[t - oy], rc[t - ox - oy], ht);
  Ex = R(0); Ey = R(0);
  if (below) {
    // E_x at (i, j-1/2, k-1/2): a = y, b = z; from a y face E_x = -F[5], from a z face E_x = +F[6]
    Ex = edge_emf<R>(-Fy[5 * P + t], -pFy5, Fz[6 * P + t], Fz[6 * P + t - oy], pFy0, Fy[t], Fz[t - oy], Fz[t],
                     Cc[t], Cc[t - oy], Cp[t], Cp[t - oy], rc[t], rc[t - oy], rp[t], rp[t - oy], ht);
    // E_y at (i-1/2, j, k-1/2): a = z, b = x; from a z face E_y = -F[5], from an x face E_y = +F[6]
    Ey = edge_emf<R>(-Fz[5 * P + t], -Fz[5 * P + t - ox], Fx[6 * P + t], pFx6, Fz[t - ox], Fz[t], pFx0, Fx[t],
                     Cc[P + t], Cp[P + t], Cc[P + t - ox], Cp[P + t - ox], rc[t], rp[t], rc[t - ox], rp[t - ox], ht);
  }
}

// in-plane flux differences of the thread's cell in conserved order (rho, Mx, My, Mz, e), summed x then y (Eq. 10), and the
// flux through its lower z face in the same order
template <class R, int P>
__device__ __forceinline__ void march_fluxdiv(const R* __restrict__ sF, int t, int ox, int oy, R (&dxy)[5], R (&fz)[5]) {
  const R* Fx = sF; const R* Fy = sF + 7 * P; const R* Fz = sF + 14 * P;
  R dx[5], dy[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) { dx[v] = Fx[v * P + t + ox] - Fx[v * P + t]; dy[v] = Fy[v * P + t + oy] - Fy[v * P + t]; }
  // y faces carry (rho, My, Mz, Mx, e), z faces (rho, Mz, Mx, My, e)
  dxy[0] = dx[0] + dy[0]; dxy[1] = dx[1] + dy[3]; dxy[2] = dx[2] + dy[1]; dxy[3] = dx[3] + dy[2]; dxy[4] = dx[4] + dy[4];
  fz[0] = Fz[t]; fz[1] = Fz[2 * P + t]; fz[2] = Fz[3 * P + t]; fz[3] = Fz[P + t]; fz[4] = Fz[4 * P + t];
}

// ---- bulk asynchronous copies global -> shared memory (TMA engine, 1-D form: no tensor map) completing on an mbarrier ----
__device__ __forceinline__ unsigned smem_u32(const void* q) { return (unsigned)__cvta_generic_to_shared(q); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// dst, src 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void bulk_load(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
               "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok)
                 : "r"(smem_u32(bar)), "r"(parity)
                 : "memory");
  } while (!ok);
}

// ---------------------------------------------------------------------------------------------------------------------
// pass 1: grid = groups, 484 threads.  Dynamic shared memory in planes of 484 values: primitives + reference EMFs of planes
// k and k-1 (2 x 11), fluxes (21), edge EMFs (3), half-step x / y faces (2); with TMA the staged input planes: U (5), Bx and
// By (22 x 23 values + alignment slack each), Bz of levels k and k+1 (2), and one mbarrier.
// TMA: the input planes of a patch group are contiguous in memory (U[v][k][.][.], Bx[k][.][.], ...), so plane k+1 is
// fetched by eight 1-D bulk copies issued by one thread while the block works on plane k: no thread waits for its own
// eleven loads, and every byte of the tile is read from DRAM exactly once, in whole 16-byte units.
// ---------------------------------------------------------------------------------------------------------------------
constexpr int kMXP = 512;                          // values reserved for a staged Bx / By plane (506 + up to 3 of alignment slack)
template <class R, bool TMA> constexpr size_t march1_smem() {
  return (size_t)((2 * 11 + 21 + 3 + 2) * kMP + (TMA ? 7 * kMP + 2 * kMXP : 0)) * sizeof(R) + (TMA ? 16 : 0);
}

// grid = (groups, chunks): a small batch is cut along z into `chunks` blocks per group so that it still fills the GPU.  A chunk that
// owns the half-step planes [k0, k1) marches over the planes k0-1 .. k1: the first plane only sets up what the others carry (its
// primitives and x / y face data), so every chunk repeats two planes of solves; the values it produces are those of the whole march,
// bit for bit (same operations on the same operands), whatever the number of chunks.
template <class R, int SOLVER, bool TMA>
__global__ void __launch_bounds__(kMP, (sizeof(R) == 4 && SOLVER != kROE) ? 2 : 1) k_vl_march1(const KParamsSC<R, 23> p, const int per) {
  constexpr int T = kMT, P = kMP, T3 = T * T * T, XP = T * (T + 1);
  extern __shared__ __align__(16) unsigned char march_smem[];
  R* sW = reinterpret_cast<R*>(march_smem);     // [2][11][P]: primitives (8) and reference EMFs (3) of planes k, k-1
  R* sF = sW + 2 * 11 * P;                       // [21][P]
  R* sE = sF + 21 * P;                           // [3][P]: E_x, E_y, E_z of this plane's corners
  R* sX = sE + 3 * P;                            // [2][P]: half-step lower x / y faces of plane k-1
  R* sU = sX + 2 * P;                            // TMA: [5][P] conserved variables of the staged plane
  R* sBx = sU + 5 * P;                           //      [kMXP] x faces, [kMXP] y faces of the staged plane
  R* sBy = sBx + kMXP;
  R* sBz = sBy + kMXP;                           //      [2][P] z faces: level k in slot k & 1, level k+1 in the other
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(sBz + 2 * P);
  const int t = threadIdx.x, i = t % T, j = t / T, grp = blockIdx.x;
  R* ws = p.ws + (size_t)grp * kMWS;
  const R* U = p.Uin + (size_t)grp * p.nUi;
  const R* Bx = p.Bin + (size_t)grp * p.nBi;
  const R* By = Bx + T * XP;
  const R* Bz = By + T * XP;
  const R qh = (R(0.5) * p.dt) / p.dh, ht = R(0.5) * p.tie;
  const bool cell = i >= 1 && i < T - 1 && j >= 1 && j < T - 1;       // half-step cells of the plane
  const bool corner = i >= 1 && j >= 1;                                // edges through the lowest corner exist
  const bool fx = corner && j < T - 1, fy = corner && i < T - 1;       // lower x / y faces of half-step cells (and their upper rim)
  const int k0 = 1 + (int)blockIdx.y * per, k1 = min(T - 1, k0 + per), kb = k0 - 1;   // this block's half-step planes [k0, k1), first plane of the march
  // stage plane kn: U, Bx, By of plane kn and Bz of level kn+1 (the prologue also brings level 0).  A face plane of
  // 22 x 23 floats starts on an 8-byte boundary for odd kn: the copy starts at the 16-byte boundary below it
  auto stage = [&](int kn) {
    constexpr unsigned PB = P * sizeof(R);
    const unsigned mis = (unsigned)((size_t)kn * XP * sizeof(R)) & 15u;
    const unsigned XB = (unsigned)(XP * sizeof(R) + mis + 15u) & ~15u;
    mbar_expect_tx(bar, (kn == kb ? 7u : 6u) * PB + 2u * XB);
#pragma unroll
    for (int v = 0; v < 5; ++v) bulk_load(sU + v * P, U + v * T3 + kn * P, PB, bar);
    bulk_load(sBx, reinterpret_cast<const char*>(Bx + kn * XP) - mis, XB, bar);
    bulk_load(sBy, reinterpret_cast<const char*>(By + kn * XP) - mis, XB, bar);
    if (kn == kb) bulk_load(sBz + (kn & 1) * P, Bz + kn * P, PB, bar);
    bulk_load(sBz + ((kn + 1) & 1) * P, Bz + (kn + 1) * P, PB, bar);
  };
  if (TMA) {
    if (t == 0) { mbar_init(bar, 1); stage(kb); }
    __syncthreads();
  }
  R A[5] = { R(0), R(0), R(0), R(0), R(0) };                           // (x, y flux differences) - (lower z flux) of cell k
  R Cx = R(0), Cy = R(0), bzlo = R(0);                                 // open CT sums of the lower x / y faces; finished lower z face
  R pFx0 = R(0), pFx6 = R(0), pFy0 = R(0), pFy5 = R(0);                // x / y face data of the plane below
  for (int k = kb; k <= k1; ++k) {
    R* Wc = sW + (k & 1) * 11 * P;
    const R* Wp = sW + ((k & 1) ^ 1) * 11 * P;
    R bl[3], W[8];
    if (TMA) {
      mbar_wait(bar, (unsigned)(k - kb) & 1u);
      const int sh = (int)((((size_t)k * XP * sizeof(R)) & 15u) / sizeof(R));
      R u[5], bu[3];
#pragma unroll
      for (int v = 0; v < 5; ++v) u[v] = sU[v * P + t];
      bl[0] = sBx[sh + j * (T + 1) + i]; bu[0] = sBx[sh + j * (T + 1) + i + 1];
      bl[1] = sBy[sh + j * T + i];       bu[1] = sBy[sh + (j + 1) * T + i];
      bl[2] = sBz[(k & 1) * P + t];      bu[2] = sBz[((k + 1) & 1) * P + t];
      cons_to_prim<true>(p, u, bl, bu, W);
#pragma unroll
      for (int v = 0; v < 8; ++v) opaque(W[v]);
    } else {
      v1_load_prim<R, true>(p, U, Bx, By, Bz, i, j, k, bl, W);
    }
#pragma unroll
    for (int v = 0; v < 8; ++v) Wc[v * P + t] = W[v];
    Wc[8 * P + t] = W[3] * W[6] - W[2] * W[7];
    Wc[9 * P + t] = W[1] * W[7] - W[3] * W[5];
    Wc[10 * P + t] = W[2] * W[5] - W[1] * W[6];
    __syncthreads();
    if (TMA && t == 0 && k + 1 <= k1) stage(k + 1);        // every thread has taken plane k out of the staging buffers
    {
      R wl[7], wr[7], F[7];
      if (i >= 1) {
        gen_from_smem<R, 0>(Wc, t - 1, wl); gen_from_prim<R, 0>(W, wr);
        if (riemann<R, SOLVER>(wl, wr, bl[0], p.gam, p.gm1inv, F)) count_event(p.stats + 2);
#pragma unroll
        for (int v = 0; v < 7; ++v) sF[v * P + t] = F[v];
      }
      if (j >= 1) {
        gen_from_smem<R, 1>(Wc, t - T, wl); gen_from_prim<R, 1>(W, wr);
        if (riemann<R, SOLVER>(wl, wr, bl[1], p.gam, p.gm1inv, F)) count_event(p.stats + 2);
#pragma unroll
        for (int v = 0; v < 7; ++v) sF[(7 + v) * P + t] = F[v];
      }
      if (k > kb) {
        gen_from_smem<R, 2>(Wp, t, wl); gen_from_prim<R, 2>(W, wr);
        if (riemann<R, SOLVER>(wl, wr, bl[2], p.gam, p.gm1inv, F)) count_event(p.stats + 2);
#pragma unroll
        for (int v = 0; v < 7; ++v) sF[(14 + v) * P + t] = F[v];
      }
    }
    __syncthreads();
    // time-n data of cell (i, j, k-1) and its lower x / y faces, read a second time (L2): asked for here, used below
    R Uo[5] = { R(0), R(0), R(0), R(0), R(0) }, bxo = R(0), byo = R(0);
    if (k >= kb + 2) {
      const int cq = ((k - 1) * T + j) * T + i;
      if (cell) {
#pragma unroll
        for (int v = 0; v < 5; ++v) Uo[v] = U[v * T3 + cq];
      }
      if (fx) bxo = Bx[((k - 1) * T + j) * (T + 1) + i];
      if (fy) byo = By[((k - 1) * (T + 1) + j) * T + i];
    }
    // ---- edge EMFs: E_z of this plane, E_x / E_y of the level k-1/2 ----
    R Ex = R(0), Ey = R(0), Ez = R(0);
    if (corner) {
      march_emfs<R, P>(sF, Wc + 8 * P, Wp + 8 * P, Wc, Wp, t, 1, T, pFx0, pFx6, pFy0, pFy5, ht, k > kb, Ex, Ey, Ez);
      pFx0 = sF[t]; pFx6 = sF[6 * P + t]; pFy0 = sF[7 * P + t]; pFy5 = sF[12 * P + t];
    }
    sE[t] = Ex; sE[P + t] = Ey; sE[2 * P + t] = Ez;
    // ---- CT (Eq. 13 with dt/2) of the lower x / y faces of plane k-1: their open sums close with E_y / E_x of this level ----
    R bxh = R(0), byh = R(0);
    if (k >= kb + 2) {
      if (fx) { bxh = bxo - qh * (Cx - Ey); ws[(size_t)(M_BH + 0) * T3 + (k - 1) * P + t] = bxh; }
      if (fy) { byh = byo - qh * (Ex + Cy); ws[(size_t)(M_BH + 1) * T3 + (k - 1) * P + t] = byh; }
    }
    sX[t] = bxh; sX[P + t] = byh;
    // ---- flux differences of cell (i, j, k); U^{n+1/2} of cell (i, j, k-1) (Eq. 10 with dt/2) ----
    R Uh[5];
    if (cell) {
      R dxy[5], fz[5];
      march_fluxdiv<R, P>(sF, t, 1, T, dxy, fz);
#pragma unroll
      for (int v = 0; v < 5; ++v) { Uh[v] = Uo[v] - qh * (A[v] + fz[v]); A[v] = dxy[v] - fz[v]; }
    }
    __syncthreads();
    // ---- the lower z face of level k-1/2 is complete; open the sums of the lower x / y faces of plane k; cell (i, j, k-1) ----
    R bzh = R(0);
    if (cell && k > kb) {
      bzh = bl[2] - qh * ((sE[P + t + 1] - Ey) - (sE[t + T] - Ex));
      ws[(size_t)(M_BH + 2) * T3 + k * P + t] = bzh;
    }
    if (fx) Cx = (sE[2 * P + t + T] - Ez) + Ey;
    if (fy) Cy = -Ex - (sE[2 * P + t + 1] - Ez);
    if (cell && k >= kb + 2) {
      // the upper x / y faces of a cell are the lower faces of its neighbours
      const R blh[3] = { bxh, byh, bzlo }, buh[3] = { sX[t + 1], sX[P + t + T], bzh };
      R Wh[8];
      cons_to_prim(p, Uh, blh, buh, Wh);
#pragma unroll
      for (int v = 0; v < 8; ++v) ws[(size_t)(M_WH + v) * T3 + (k - 1) * P + t] = Wh[v];
    }
    bzlo = bzh;
  }
}

// ---------------------------------------------------------------------------------------------------------------------
// pass 2: grid = groups, 324 threads = cells [2, 20)^2 of the plane (the transverse range of the pass-2 faces, DESIGN.md
// section 6), marching over planes 2 .. 19.  Shared memory: planes of 324 values: reference EMFs + density of planes k, k-1
// (2 x 4), fluxes (21), edge EMFs (3), the upper z state of the cell below (7), new x / y faces for the CFL speed (2); and a
// ring of three whole 22 x 22 planes of the 8 half-step primitives (k-1, k, k+1), filled by 1-D bulk copies (TMA) one
// plane ahead: every slope operand comes from shared memory, and the plane is read from memory once.
// ---------------------------------------------------------------------------------------------------------------------
// FP32 also stages the time-n planes the update of cell plane k-1 reads (U, x / y faces of plane k-1, z faces of level k): 6 planes of
// 484 + 2 x 508 values; in FP64 the block is at the 227 KB limit without them and reads them from memory
template <class R> constexpr bool march2_stage_in() { return sizeof(R) == 4; }
constexpr int kMXS = 508;                          // 22 x 23 face values + 2 of alignment slack
template <class R> constexpr size_t march2_smem() {
  return (size_t)((2 * 4 + 21 + 3 + 7 + 2) * kM2P + 3 * 8 * kMP + (march2_stage_in<R>() ? 6 * kMP + 2 * kMXS : 0)) * sizeof(R) + 32;
}

#ifndef MHD_M2_MINB
#define MHD_M2_MINB 2
#endif
#ifndef MHD_M2_MINB_ROE
#define MHD_M2_MINB_ROE 1
#endif
// S9 (p.red set: mhd_advance_dt) is a run-time branch, not a template flag: the two instantiations compiled the energy flux of
// the Riemann solve to different last bits in FP32, and mhd_advance_dt must equal mhd_advance + mhd_dt_reduce bit for bit
template <class R, int SOLVER, int LIM>
__global__ void __launch_bounds__(kM2P, sizeof(R) == 4 ? (SOLVER != kROE ? MHD_M2_MINB : MHD_M2_MINB_ROE) : 1) k_vl_march2(const KParamsSC<R, 23> p, const int per) {
  constexpr int T = kMT, PT = kMT * kMT, T3 = T * T * T, P = kM2P, W = kM2W, N = 16, M = N + 1, g = 3;
  extern __shared__ __align__(16) unsigned char march_smem[];
  R* sR = reinterpret_cast<R*>(march_smem);     // [3][8][PT]: half-step primitives of planes k-1, k, k+1 (plane kp in slot kp % 3)
  R* sC = sR + 3 * 8 * PT;                       // [2][4][P]: ec_x, ec_y, ec_z, rho of the half-step state, planes k and k-1
  R* sF = sC + 2 * 4 * P;                        // [21][P]
  R* sE = sF + 21 * P;                           // [3][P]
  R* sZ = sE + 3 * P;                            // [7][P]: W(k-1) + slope_z(k-1)/2 of the thread's own column
  R* sX = sZ + 7 * P;                            // [2][P]: new lower x / y faces of plane k-1 (DT)
  constexpr bool SIN = march2_stage_in<R>();
  R* sUt = sX + 2 * P;                           // SIN: [5][PT] U of plane k-1, then x faces [kMXS], y faces [kMXS] of plane k-1, z faces [PT] of level k
  R* sBxt = sUt + 5 * PT;
  R* sByt = sBxt + kMXS;
  R* sBzt = sByt + kMXS;
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(SIN ? sBzt + PT : sX + 2 * P);
  unsigned long long* bar2 = bar + 1;
  const int t = threadIdx.x, i = t % W + 2, j = t / W + 2, grp = blockIdx.x;
  const int c = j * T + i;
  const R* ws = p.ws + (size_t)grp * kMWS;
  const R* Wh = ws + (size_t)M_WH * T3;
  const R* bh = ws + (size_t)M_BH * T3;
  const R* U = p.Uin + (size_t)grp * p.nUi;
  const R* Bx = p.Bin + (size_t)grp * p.nBi;
  const R* By = Bx + T * T * (T + 1);
  const R* Bz = By + T * T * (T + 1);
  R* Uo = p.Uout + (size_t)grp * p.nUo;
  R* Bxo = p.Bout + (size_t)grp * p.nBo;
  R* Byo = Bxo + N * N * (N + 1);
  R* Bzo = Byo + N * N * (N + 1);
  R* fo = p.fout ? p.fout + (size_t)grp * p.nF : nullptr;
  R* eo = p.eout ? p.eout + (size_t)grp * p.nE : nullptr;
  const R q = p.dt / p.dh, ht = R(0.5) * p.tie;
  const int ii = i - g, jj = j - g;                                     // interior indices
  const bool in = ii >= 0 && ii < N && jj >= 0 && jj < N;                // interior cell column
  const bool corner = ii >= 0 && jj >= 0;                                // i, j in [g, g+N]: the edges of the interior faces
  const bool fx = ii >= 0 && jj >= 0 && jj < N, fy = jj >= 0 && ii >= 0 && ii < N;
  const int sx = i == g ? 0 : (i == g + N / 2 ? 1 : (i == g + N ? 2 : -1));   // this thread's x / y faces lie on an output plane
  const int sy = j == g ? 0 : (j == g + N / 2 ? 1 : (j == g + N ? 2 : -1));
  R A[5] = { R(0), R(0), R(0), R(0), R(0) };
  R Cx = R(0), Cy = R(0), bzlo = R(0);
  R pFx0 = R(0), pFx6 = R(0), pFy0 = R(0), pFy5 = R(0);
  R smax = R(0);
  const bool DT = p.red != nullptr;
  const int k0 = g + (int)blockIdx.y * per, k1 = min(g + N, k0 + per), kb = k0 - 1;     // this block's interior planes [k0, k1) (see k_vl_march1)
  // stage the 8 primitives of plane kp into its ring slot
  auto stage = [&](int kp, bool arm) {
    constexpr unsigned PB = PT * sizeof(R);
    if (arm) mbar_expect_tx(bar, 8u * PB);
#pragma unroll
    for (int v = 0; v < 8; ++v) bulk_load(sR + ((kp % 3) * 8 + v) * PT, Wh + v * T3 + kp * PT, PB, bar);
  };
  // SIN: the time-n planes that iteration kn + 1 reads: U, x / y faces of plane kn, z faces of level kn + 1 (alignment as in pass 1)
  auto stage_in = [&](int kn) {
    constexpr unsigned PB = PT * sizeof(R);
    constexpr int XP = T * (T + 1);
    const unsigned mis = (unsigned)((size_t)kn * XP * sizeof(R)) & 15u;
    const unsigned XB = (unsigned)(XP * sizeof(R) + mis + 15u) & ~15u;
    mbar_expect_tx(bar2, 6u * PB + 2u * XB);
#pragma unroll
    for (int v = 0; v < 5; ++v) bulk_load(sUt + v * PT, U + v * T3 + kn * PT, PB, bar2);
    bulk_load(sBxt, reinterpret_cast<const char*>(Bx + kn * XP) - mis, XB, bar2);
    bulk_load(sByt, reinterpret_cast<const char*>(By + kn * XP) - mis, XB, bar2);
    bulk_load(sBzt, Bz + (kn + 1) * PT, PB, bar2);
  };
  const bool sin = SIN && ((reinterpret_cast<size_t>(p.Uin) | reinterpret_cast<size_t>(p.Bin)) & 15) == 0;   // bulk copies need 16-byte aligned planes
  if (t == 0) {
    mbar_init(bar, 1);
    if (SIN) mbar_init(bar2, 1);
    mbar_expect_tx(bar, 3u * 8u * PT * sizeof(R));
    stage(kb - 1, false); stage(kb, false); stage(kb + 1, false);
    if (sin) stage_in(kb);
  }
  __syncthreads();
  mbar_wait(bar, 0);
  R bhn[3] = { bh[kb * PT + c], bh[T3 + kb * PT + c], bh[2 * T3 + kb * PT + c] };   // normal fields of the lower faces of plane k
  for (int k = kb; k <= k1; ++k) {
    R* Cc = sC + (k & 1) * 4 * P;
    const R* Cp = sC + ((k & 1) ^ 1) * 4 * P;
    const R* Rk = sR + (k % 3) * 8 * PT;
    const int kk = k - g;
    {
      R W0[8];
#pragma unroll
      for (int v = 0; v < 8; ++v) W0[v] = Rk[v * PT + c];
      Cc[t] = W0[3] * W0[6] - W0[2] * W0[7];
      Cc[P + t] = W0[1] * W0[7] - W0[3] * W0[5];
      Cc[2 * P + t] = W0[2] * W0[5] - W0[1] * W0[6];
      Cc[3 * P + t] = W0[0];
      R wm[7], w0[7], wl[7], wr[7], sl[7], sr[7], F[7];
      // x face: PLM of cells i-1 and i, normal field = the half-step face value
      if (i >= g) {
        R wmm[7], wp[7];
        load_gen<R, 0>(Rk, PT, c - 2, wmm); load_gen<R, 0>(Rk, PT, c - 1, wm); gen_from_prim<R, 0>(W0, w0); load_gen<R, 0>(Rk, PT, c + 1, wp);
        slope3<R, LIM>(wmm, wm, w0, Rk[5 * PT + c - 1], p.gam, sl);
        slope3<R, LIM>(wm, w0, wp, W0[5], p.gam, sr);
#pragma unroll
        for (int v = 0; v < 7; ++v) { wl[v] = wm[v] + R(0.5) * sl[v]; wr[v] = w0[v] - R(0.5) * sr[v]; }
        apply_floors(p, wl); apply_floors(p, wr);
        if (riemann<R, SOLVER>(wl, wr, bhn[0], p.gam, p.gm1inv, F)) count_event(p.stats + 2);
#pragma unroll
        for (int v = 0; v < 7; ++v) sF[v * P + t] = F[v];
      }
      if (j >= g) {
        R wmm[7], wp[7];
        load_gen<R, 1>(Rk, PT, c - 2 * T, wmm); load_gen<R, 1>(Rk, PT, c - T, wm); gen_from_prim<R, 1>(W0, w0); load_gen<R, 1>(Rk, PT, c + T, wp);
        slope3<R, LIM>(wmm, wm, w0, Rk[6 * PT + c - T], p.gam, sl);
        slope3<R, LIM>(wm, w0, wp, W0[6], p.gam, sr);
#pragma unroll
        for (int v = 0; v < 7; ++v) { wl[v] = wm[v] + R(0.5) * sl[v]; wr[v] = w0[v] - R(0.5) * sr[v]; }
        apply_floors(p, wl); apply_floors(p, wr);
        if (riemann<R, SOLVER>(wl, wr, bhn[1], p.gam, p.gm1inv, F)) count_event(p.stats + 2);
#pragma unroll
        for (int v = 0; v < 7; ++v) sF[(7 + v) * P + t] = F[v];
      }
      // z face between planes k-1 and k: the upper state of the cell below was left in sZ one plane ago
      {
        R wp[7];
        if (k > kb) mbar_wait(bar, (unsigned)(k - kb) & 1u);                 // plane k+1 has landed (the first three with the prologue)
        load_gen<R, 2>(sR + ((k + 2) % 3) * 8 * PT, PT, c, wm); gen_from_prim<R, 2>(W0, w0); load_gen<R, 2>(sR + ((k + 1) % 3) * 8 * PT, PT, c, wp);
        slope3<R, LIM>(wm, w0, wp, W0[7], p.gam, sr);
        if (k > kb) {
#pragma unroll
          for (int v = 0; v < 7; ++v) { wl[v] = sZ[v * P + t]; wr[v] = w0[v] - R(0.5) * sr[v]; }
          apply_floors(p, wl); apply_floors(p, wr);
          if (riemann<R, SOLVER>(wl, wr, bhn[2], p.gam, p.gm1inv, F)) count_event(p.stats + 2);
#pragma unroll
          for (int v = 0; v < 7; ++v) sF[(14 + v) * P + t] = F[v];
        }
#pragma unroll
        for (int v = 0; v < 7; ++v) sZ[v * P + t] = w0[v] + R(0.5) * sr[v];
      }
    }
    __syncthreads();
    if (t == 0 && k + 2 <= k1 + 1) stage(k + 2, true);                    // into the slot of plane k-1: nobody reads it any more
    // time-n data of cell (i, j, k-1), its lower x / y faces and the lower z face of level k-1/2: asked for here, used below
    R Ut[5] = { R(0), R(0), R(0), R(0), R(0) }, bxo = R(0), byo = R(0), bzo = R(0);
    if (sin) {
      if (k > kb) {
        mbar_wait(bar2, (unsigned)(k - kb - 1) & 1u);
        const int sh = (int)((((size_t)(k - 1) * T * (T + 1) * sizeof(R)) & 15u) / sizeof(R));
#pragma unroll
        for (int v = 0; v < 5; ++v) Ut[v] = sUt[v * PT + c];
        bxo = sBxt[sh + j * (T + 1) + i]; byo = sByt[sh + c]; bzo = sBzt[c];
      }
    } else {
      if (k >= kb + 2) {
        const int cq = ((k - 1) * T + j) * T + i;
        if (in) {
#pragma unroll
          for (int v = 0; v < 5; ++v) Ut[v] = U[v * T3 + cq];
        }
        if (fx) bxo = Bx[((k - 1) * T + j) * (T + 1) + i];
        if (fy) byo = By[((k - 1) * (T + 1) + j) * T + i];
      }
      if (in && k > kb) bzo = Bz[(k * T + j) * T + i];
    }
    if (k < k1) {
      const int qn = (k + 1) * PT + c;
      bhn[0] = bh[qn]; bhn[1] = bh[T3 + qn]; bhn[2] = bh[2 * T3 + qn];
    }
    // ---- flux differences of cell (i, j, k); U^{n+1} of cell (i, j, k-1) (Eq. 10) ----
    R Un[5];
    if (in) {
      R dxy[5], fz[5];
      march_fluxdiv<R, P>(sF, t, 1, W, dxy, fz);
      if (k >= kb + 2) {
        const int oq = ((kk - 1) * N + jj) * N + ii;
#pragma unroll
        for (int v = 0; v < 5; ++v) { Un[v] = Ut[v] - q * (A[v] + fz[v]); Uo[v * N * N * N + oq] = Un[v]; }
      }
#pragma unroll
      for (int v = 0; v < 5; ++v) A[v] = dxy[v] - fz[v];
    }
    // ---- time-centred fluxes on the lower / mid / upper face planes (layout: include/mhd.h) ----
    if (fo) {
      const int NN = N * N;
      if (sx >= 0 && jj >= 0 && jj < N && kk >= 0 && kk < N) {           // x planes: [z][y], components (rho, Mn, Mt1, Mt2, e) -> (rho, Mx, My, Mz, e)
        R* f = fo + (size_t)(0 + sx) * 5 * NN + kk * N + jj;
        f[0] = sF[t]; f[NN] = sF[P + t]; f[2 * NN] = sF[2 * P + t]; f[3 * NN] = sF[3 * P + t]; f[4 * NN] = sF[4 * P + t];
      }
      if (sy >= 0 && ii >= 0 && ii < N && kk >= 0 && kk < N) {           // y planes: [x][z], y faces carry (rho, My, Mz, Mx, e)
        R* f = fo + (size_t)(3 + sy) * 5 * NN + ii * N + kk;
        f[0] = sF[7 * P + t]; f[2 * NN] = sF[8 * P + t]; f[3 * NN] = sF[9 * P + t]; f[NN] = sF[10 * P + t]; f[4 * NN] = sF[11 * P + t];
      }
      if (in && k > kb && (kk == 0 || kk == N / 2 || kk == N)) {         // z planes: [y][x], z faces carry (rho, Mz, Mx, My, e)
        R* f = fo + (size_t)(6 + (kk == 0 ? 0 : (kk == N ? 2 : 1))) * 5 * NN + jj * N + ii;
        f[0] = sF[14 * P + t]; f[3 * NN] = sF[15 * P + t]; f[NN] = sF[16 * P + t]; f[2 * NN] = sF[17 * P + t]; f[4 * NN] = sF[18 * P + t];
      }
    }
    // ---- edge EMFs ----
    R Ex = R(0), Ey = R(0), Ez = R(0);
    if (corner) {
      march_emfs<R, P>(sF, Cc, Cp, Cc + 3 * P, Cp + 3 * P, t, 1, W, pFx0, pFx6, pFy0, pFy5, ht, k > kb, Ex, Ey, Ez);
      pFx0 = sF[t]; pFx6 = sF[6 * P + t]; pFy0 = sF[7 * P + t]; pFy5 = sF[12 * P + t];
    }
    sE[t] = Ex; sE[P + t] = Ey; sE[2 * P + t] = Ez;
    if (eo && corner) {
      const int MN = M * N;
      const bool kf = k > kb, kc = kk >= 0 && kk < N;                      // kf: the EMFs of the level k-1/2 exist (an interior face level); kc: plane k is interior
      if (sx >= 0) {                                                     // x planes: E_y [z: N+1][y: N], E_z [z: N][y: N+1]
        R* e = eo + (size_t)(0 + sx) * 2 * MN;
        if (kf && jj < N) e[kk * N + jj] = Ey;
        if (kc) e[MN + kk * M + jj] = Ez;
      }
      if (sy >= 0) {                                                     // y planes: E_z [x: N+1][z: N], E_x [x: N][z: N+1]
        R* e = eo + (size_t)(3 + sy) * 2 * MN;
        if (kc) e[ii * N + kk] = Ez;
        if (kf && ii < N) e[MN + ii * M + kk] = Ex;
      }
      if (kf && (kk == 0 || kk == N / 2 || kk == N)) {                   // z planes: E_x [y: N+1][x: N], E_y [y: N][x: N+1]
        R* e = eo + (size_t)(6 + (kk == 0 ? 0 : (kk == N ? 2 : 1))) * 2 * MN;
        if (ii < N) e[jj * N + ii] = Ex;
        if (jj < N) e[MN + jj * M + ii] = Ey;
      }
    }
    __syncthreads();
    if (sin && t == 0 && k > kb && k + 1 <= k1) stage_in(k);               // every thread has taken the planes of this iteration
    // ---- CT (Eq. 13): lower z face of level k-1/2; lower x / y faces of plane k-1 ----
    R bzn = R(0), bxn = R(0), byn = R(0);
    if (in && k > kb) {
      bzn = bzo - q * ((sE[P + t + 1] - Ey) - (sE[t + W] - Ex));
      Bzo[(kk * N + jj) * N + ii] = bzn;
    }
    if (fx) {
      if (k >= kb + 2) {
        bxn = bxo - q * (Cx - Ey);
        Bxo[((kk - 1) * N + jj) * (N + 1) + ii] = bxn;
      }
      Cx = (sE[2 * P + t + W] - Ez) + Ey;
    }
    if (fy) {
      if (k >= kb + 2) {
        byn = byo - q * (Ex + Cy);
        Byo[((kk - 1) * (N + 1) + jj) * N + ii] = byn;
      }
      Cy = -Ex - (sE[2 * P + t + 1] - Ez);
    }
    if (DT && k >= kb + 2) {
      // S9 on the new state of cell (i, j, k-1): its upper x / y faces are the lower faces of the neighbours
      sX[t] = bxn; sX[P + t] = byn;
      __syncthreads();
      if (in) {
        R bl[3] = { bxn, byn, bzlo }, bu[3] = { sX[t + 1], sX[P + t + W], bzn };
#pragma unroll
        for (int v = 0; v < 5; ++v) opaque(Un[v]);
#pragma unroll
        for (int v = 0; v < 3; ++v) { opaque(bl[v]); opaque(bu[v]); }
        smax = Num<R>::max(smax, cell_signal_speed(Un, bl, bu, p.gam, p.min_dens, p.min_pres));
      }
    }
    bzlo = bzn;
  }
  if (DT) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smax = Num<R>::max(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    __syncthreads();
    if ((t & 31) == 0) sE[t >> 5] = smax;
    __syncthreads();
    if (t == 0) {
      R m = sE[0];
      for (int w = 1; w < (P + 31) / 32; ++w) m = Num<R>::max(m, sE[w]);
      atomicMax(reinterpret_cast<typename Bits<R>::U*>(p.red), Bits<R>::enc(m));
    }
  }
}

}  // namespace mhd

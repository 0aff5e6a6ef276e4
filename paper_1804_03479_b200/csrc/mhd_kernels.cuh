// mhd_kernels.cuh -- the stage kernels of the patch-group update (sm_100a), part 1: layout, staging, pass-1
// fluxes, edge EMFs, half step.
//
// Work decomposition: a batch is processed in SLICES of groups; inside a slice every stage of the scheme is one
// kernel over exactly the cells / faces / edges that stage needs (a compact index box per sweep direction, no
// masked-out threads), for all groups of the slice: blockIdx.z = group in slice, blockIdx.y = sweep direction
// where the stage has one, x-fastest thread order (coalesced rows).  Slices run concurrently on several streams
// (mhd_api.cu) so that the drain / ramp-up between dependent stages of one slice is filled by another slice.
//
// Workspace of one group: NARR arrays of S^3 Reals with the uniform strides (1, S, S^2), S = T+1, so that
// cell (i,j,k), its lower faces and its lower edges all share the flat index q = (k*S + j)*S + i:
//   b[d][q]  = field on the lower d-face of cell q            (Fig. 1)
//   F[d][c][q] = flux through that face, generic component order (rho, Mn, Mt1, Mt2, e, Bt1, Bt2), (n,t1,t2) cyclic
//   E[c][q]  = EMF on the edge along c through the cell's lowest corner, i.e. at (a-1/2, b-1/2), (a,b,c) cyclic
//   EC[c][q] = cell-centred reference EMF -(v x Bc)_c of cell q (time n, later overwritten by the half-step one)
#pragma once
#include "mhd_recon.cuh"

namespace mhd {

enum : int {
  A_W = 0,      // 8: rho, vx, vy, vz, P, Bcx, Bcy, Bcz at t^n
  A_B = 8,      // 3: face field at t^n
  A_F = 11,     // 21: F[d][c]
  A_E = 32,     // 3
  A_BH = 35,    // 3: face field at t^{n+1/2}
  A_WH = 38,    // 8: half-step primitives
  A_ETA = 1,    // 3: H-correction (R19): eta of the pass-2 faces of VL, in the arrays of the time-n velocities (dead after the half step)
  A_EC = 46,    // 3: cell-centred reference EMF
  A_VL_END = 49,
  A_LO = 49,    // 21: CTU state at the lower d-face of each cell, [d][v]
  A_UP = 70,    // 21: CTU state at the upper d-face
  A_F2 = 91,    // 21: CTU pass-2 fluxes (the fused correction + Riemann kernel still reads the pass-1 fluxes while it writes)
  A_CTU_END = 112,
  A_ETAC = 112, // 3: H-correction of CTU: eta of the pass-2 faces (the time-n velocities are still read by the correction step)
  A_CTU_HC_END = 115
};
// H-correction (R19) in the pass-2 face kernels: kHcOff the plain solver, kHcEta only eta of the face is written, kHcOn the solver
// with eta^H = max over the face and the eight transverse faces of its two cells
enum : int { kHcOff = 0, kHcEta = 1, kHcOn = 2 };
// eta^H of the D face q from the eta arrays at `base`
template <class R, int D, class C>
__device__ __forceinline__ R eta_h(const C& c, int base, int q) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  R etah = c.arr(base + D)[q];
  const R* e1 = c.arr(base + T1); const R* e2 = c.arr(base + T2);
  const int o1 = c.off(T1), o2 = c.off(T2), ql = q - c.off(D);
  etah = Num<R>::max(etah, Num<R>::max(Num<R>::max(e1[ql], e1[ql + o1]), Num<R>::max(e1[q], e1[q + o1])));
  etah = Num<R>::max(etah, Num<R>::max(Num<R>::max(e2[ql], e2[ql + o2]), Num<R>::max(e2[q], e2[q + o2])));
  return etah;
}

template <class R> struct KParams {
  const R* Uin; const R* Bin;       // first group of the slice
  R* Uout; R* Bout; R* fout; R* eout;
  R* ws;
  unsigned long long* stats;        // [0] density floors, [1] pressure floors, [2] Riemann fallbacks
  unsigned long long* red;          // mhd_advance_dt: cell of the fused CFL reduction (bit pattern of the largest speed), else null
  int N, g, T, S, S2, S3, narr;
  long long nUi, nBi, nUo, nBo, nF, nE;
  R gam, gm1, gm1inv, dt, dh, min_dens, min_pres;
  R tie;   // emf_tie * dh / dt (R10a)
};

// compact index box of one launch: cells lo[d] .. lo[d]+n[d]-1; Box3x3 = one box per sweep direction
// m[0], m[1] = floor(2^32 / n[0,1]) + 1: t / n = umulhi(t, m) exactly for t n < 2^32 (a thread index within one group)
struct Box3 { int lo[3], n[3]; unsigned m[2]; };
struct Box3x3 { Box3 b[3]; };

// KParams with the tile pitch known at compile time (SC = S = T + 1 > 0): S, S2, S3, T shadow the run-time members, so every
// array offset a * S3 and neighbour offset folds into the immediate field of the load / store.  SC = 0: run-time pitch.
template <class R, int SC> struct KParamsSC : KParams<R> {
  static constexpr int S = SC, S2 = SC * SC, S3 = SC * SC * SC, T = SC - 1;
  KParamsSC() = default;
  __host__ __device__ KParamsSC(const KParams<R>& b) : KParams<R>(b) {}
};
template <class R> struct KParamsSC<R, 0> : KParams<R> {
  KParamsSC() = default;
  __host__ __device__ KParamsSC(const KParams<R>& b) : KParams<R>(b) {}
};

template <class R, class KP> struct Ctx {
  const KP& p;
  int q, i, j, k, grp;
  bool ok;
  R* w;   // this group's workspace
  __device__ __forceinline__ Ctx(const KP& p_, const Box3& b) : p(p_) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    ok = t < b.n[0] * b.n[1] * b.n[2];
    const int r = (int)__umulhi((unsigned)t, b.m[0]);
    i = b.lo[0] + (t - r * b.n[0]);
    const int kk = (int)__umulhi((unsigned)r, b.m[1]);
    j = b.lo[1] + (r - kk * b.n[1]);
    k = b.lo[2] + kk;
    q = (k * p.S + j) * p.S + i;
    grp = blockIdx.z;
    w = p.ws + (size_t)grp * p.narr * p.S3;
  }
  __device__ __forceinline__ R* arr(int a) const { return w + (size_t)a * p.S3; }
  __device__ __forceinline__ int off(int d) const { return d == 0 ? 1 : (d == 1 ? p.S : p.S2); }
  __device__ __forceinline__ int idx(int d) const { return d == 0 ? i : (d == 1 ? j : k); }
};

__device__ __forceinline__ void count_event(unsigned long long* ctr) { atomicAdd(ctr, 1ULL); }

// a value the staged path rounds by storing it: the compiler must materialise it here (no contraction across stages)
__device__ __forceinline__ void opaque(float& x) { asm volatile("" : "+f"(x)); }
__device__ __forceinline__ void opaque(double& x) { asm volatile("" : "+d"(x)); }

// generic 1-D state of cell q for direction D from an 8-array primitive block
template <class R, int D>
__device__ __forceinline__ void load_gen(const R* Wb, int S3, int q, R (&w)[7]) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  w[0] = Wb[q];
  w[1] = Wb[(size_t)(1 + D) * S3 + q]; w[2] = Wb[(size_t)(1 + T1) * S3 + q]; w[3] = Wb[(size_t)(1 + T2) * S3 + q];
  w[4] = Wb[(size_t)4 * S3 + q];
  w[5] = Wb[(size_t)(5 + T1) * S3 + q]; w[6] = Wb[(size_t)(5 + T2) * S3 + q];
}

template <bool COUNT = true, class R, class KP>
__device__ __forceinline__ void apply_floors(const KP& p, R (&w)[7]) {
  if (w[0] < p.min_dens) { w[0] = p.min_dens; if (COUNT) count_event(p.stats + 0); }
  if (w[4] < p.min_pres) { w[4] = p.min_pres; if (COUNT) count_event(p.stats + 1); }
}

// conserved cell data + the six face fields of the cell -> primitives (Eq. 5; floors R9)
template <bool COUNT = true, class R, class KP>
__device__ __forceinline__ void cons_to_prim(const KP& p, const R (&u)[5], const R (&bl)[3], const R (&bu)[3], R (&W)[8]) {
  const R bcx = R(0.5) * (bl[0] + bu[0]), bcy = R(0.5) * (bl[1] + bu[1]), bcz = R(0.5) * (bl[2] + bu[2]);
  R rho = u[0];
  if (rho < p.min_dens) { rho = p.min_dens; if (COUNT) count_event(p.stats + 0); }
  const R ir = frcp(rho);
  const R vx = u[1] * ir, vy = u[2] * ir, vz = u[3] * ir;
  R P = p.gm1 * (u[4] - R(0.5) * rho * (vx * vx + vy * vy + vz * vz) - R(0.5) * (bcx * bcx + bcy * bcy + bcz * bcz));
  if (P < p.min_pres) { P = p.min_pres; if (COUNT) count_event(p.stats + 1); }
  W[0] = rho; W[1] = vx; W[2] = vy; W[3] = vz; W[4] = P; W[5] = bcx; W[6] = bcy; W[7] = bcz;
}

// primitives and the cell-centred reference EMF -(v x Bc) of a cell into the workspace
template <class R, class KP>
__device__ __forceinline__ void store_prim(const Ctx<R, KP>& c, int wbase, const R (&W)[8]) {
#pragma unroll
  for (int v = 0; v < 8; ++v) c.arr(wbase + v)[c.q] = W[v];
  c.arr(A_EC + 0)[c.q] = W[3] * W[6] - W[2] * W[7];
  c.arr(A_EC + 1)[c.q] = W[1] * W[7] - W[3] * W[5];
  c.arr(A_EC + 2)[c.q] = W[2] * W[5] - W[1] * W[6];
}

// ---- S0 + S1: stage the input tile: face fields into the workspace, primitives of all T^3 cells -----------------
template <class R, int SC>
__global__ void __launch_bounds__(256) k_load_prim(const KParamsSC<R, SC> p, const Box3 box) {
  typedef KParamsSC<R, SC> KP;
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  const int T = p.T, i = c.i, j = c.j, k = c.k, q = c.q;
  const R* Bx = p.Bin + (size_t)c.grp * p.nBi;
  const R* By = Bx + (size_t)T * T * (T + 1);
  const R* Bz = By + (size_t)T * T * (T + 1);
  // every load is issued before the first store: the compiler cannot prove that the workspace does not alias the
  // inputs, so a load placed after a store would wait for that store's data, i.e. for a full memory round trip
  const bool fx = j < T && k < T, fy = i < T && k < T, fz = i < T && j < T, cell = i < T && j < T && k < T;
  R bl[3] = { R(0), R(0), R(0) }, bu[3] = { R(0), R(0), R(0) }, u[5] = { R(1), R(0), R(0), R(0), R(1) };
  if (fx) bl[0] = Bx[((size_t)k * T + j) * (T + 1) + i];
  if (fy) bl[1] = By[((size_t)k * (T + 1) + j) * T + i];
  if (fz) bl[2] = Bz[((size_t)k * T + j) * T + i];
  if (cell) {
    bu[0] = Bx[((size_t)k * T + j) * (T + 1) + i + 1];
    bu[1] = By[((size_t)k * (T + 1) + j + 1) * T + i];
    bu[2] = Bz[((size_t)(k + 1) * T + j) * T + i];
    const R* U = p.Uin + (size_t)c.grp * p.nUi;
    const size_t T3 = (size_t)T * T * T, cq = ((size_t)k * T + j) * T + i;
#pragma unroll
    for (int v = 0; v < 5; ++v) u[v] = U[v * T3 + cq];
  }
  if (fx) c.arr(A_B + 0)[q] = bl[0];
  if (fy) c.arr(A_B + 1)[q] = bl[1];
  if (fz) c.arr(A_B + 2)[q] = bl[2];
  if (!cell) return;
  R W[8];
  cons_to_prim(p, u, bl, bu, W);
  store_prim(c, A_W, W);
}

// ---- VL step 1: first-order fluxes, normal B = face value ----------------------------------------
template <class R, int SOLVER, int D, class KP>
__device__ __forceinline__ void flux1_dir(const KP& p, const Box3& box) {
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  R wl[7], wr[7], F[7];
  load_gen<R, D>(c.arr(A_W), p.S3, c.q - c.off(D), wl);
  load_gen<R, D>(c.arr(A_W), p.S3, c.q, wr);
  const bool fb = riemann<R, SOLVER>(wl, wr, c.arr(A_B + D)[c.q], p.gam, p.gm1inv, F);
  if (fb) count_event(p.stats + 2);
#pragma unroll
  for (int v = 0; v < 7; ++v) c.arr(A_F + 7 * D + v)[c.q] = F[v];
}
template <class R, int SOLVER, int SC>
__global__ void __launch_bounds__(256, OccFlux<R, SOLVER>::minb) k_flux1_vl(const KParamsSC<R, SC> p, const Box3x3 bx) {
  switch (blockIdx.y) {
    case 0: flux1_dir<R, SOLVER, 0>(p, bx.b[0]); break;
    case 1: flux1_dir<R, SOLVER, 1>(p, bx.b[1]); break;
    default: flux1_dir<R, SOLVER, 2>(p, bx.b[2]); break;
  }
}

// ---- S3 / S7: upwinded edge EMFs (formula DESIGN.md R10) --------------------------------------
// edge along C at (a-1/2, b-1/2), (a,b,c) cyclic; face EMFs: from an a-face E_c = -F_a[B_t1], from a b-face E_c = +F_b[B_t2]
// upwind switch on the face mass flux m (R10).  R10a: |m| <= m0 (less than emf_tie of the cell mass crosses the face
// in dt) counts as zero -> centred mean; between m0 and 2 m0 a linear ramp to the upwind value keeps the EMF continuous
template <class R> __device__ __forceinline__ R upwind(R m, R m0, R qm, R qp) {
  const R am = Num<R>::abs(m), qu = m > R(0) ? qm : qp;
  if (am >= R(2) * m0) return qu;                      // plain upwinding: all but a vanishing fraction of the faces
  const R mean = R(0.5) * (qm + qp);
  if (am <= m0) return mean;
  const R w = fdiv(am - m0, m0);                       // weight of the upwind value on the ramp m0 < |m| < 2 m0
  return w * qu + (R(1) - w) * mean;
}
template <class R, int C, int FBASE, class KP>
__device__ __forceinline__ void emf_dir(const KP& p, const Box3& box, int rhobase) {
  constexpr int A = (C + 1) % 3, B = (C + 2) % 3;
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  const int q = c.q, qa = q - c.off(A), qb = q - c.off(B), qab = qa - c.off(B);
  const R* Fa5 = c.arr(FBASE + 7 * A + 5); const R* Fa0 = c.arr(FBASE + 7 * A + 0);
  const R* Fb6 = c.arr(FBASE + 7 * B + 6); const R* Fb0 = c.arr(FBASE + 7 * B + 0);
  const R* ec = c.arr(A_EC + C); const R* rho = c.arr(rhobase);
  const R Ea_q = -Fa5[q], Ea_qb = -Fa5[qb], Eb_q = Fb6[q], Eb_qa = Fb6[qa];
  const R ec_q = ec[q], ec_qa = ec[qa], ec_qb = ec[qb], ec_qab = ec[qab];
  const R ht = R(0.5) * p.tie, r_q = rho[q], r_qa = rho[qa], r_qb = rho[qb], r_qab = rho[qab];
  R e = R(0.25) * (Ea_q + Ea_qb + Eb_q + Eb_qa);
  e += R(0.25) * (upwind(Fa0[qb], ht * (r_qab + r_qb), Eb_qa - ec_qab, Eb_q - ec_qb) - upwind(Fa0[q], ht * (r_qa + r_q), ec_qa - Eb_qa, ec_q - Eb_q));
  e += R(0.25) * (upwind(Fb0[qa], ht * (r_qab + r_qa), Ea_qb - ec_qab, Ea_q - ec_qa) - upwind(Fb0[q], ht * (r_qb + r_q), ec_qb - Ea_qb, ec_q - Ea_q));
  c.arr(A_E + C)[q] = e;
}
template <class R, int FBASE, int SC>
__global__ void __launch_bounds__(256, OccEmf<R>::minb) k_emf(const KParamsSC<R, SC> p, const Box3x3 bx, int rhobase) {
  switch (blockIdx.y) {
    case 0: emf_dir<R, 0, FBASE>(p, bx.b[0], rhobase); break;
    case 1: emf_dir<R, 1, FBASE>(p, bx.b[1], rhobase); break;
    default: emf_dir<R, 2, FBASE>(p, bx.b[2], rhobase); break;
  }
}

// Eq. 13 for the lower D-face of cell x (flat index), step factor qh = tau/dh
template <class R, int D, class KP>
__device__ __forceinline__ R ct_face(const Ctx<R, KP>& c, const R* bsrc, int x, R qh) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  const R* E1 = c.arr(A_E + T1); const R* E2 = c.arr(A_E + T2);
  return bsrc[x] - qh * ((E2[x + c.off(T1)] - E2[x]) - (E1[x + c.off(T2)] - E1[x]));
}

// Eq. 10: sum over x, y, z (in this order) of the flux differences of cell q, conserved order
template <int FBASE, class R, class KP>
__device__ __forceinline__ void flux_div(const Ctx<R, KP>& c, R (&dU)[5]) {
#pragma unroll
  for (int v = 0; v < 5; ++v) dU[v] = R(0);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const int t1 = (d + 1) % 3, t2 = (d + 2) % 3, qu = c.q + c.off(d);
    const R* F = c.arr(FBASE + 7 * d);
    const size_t S3 = c.p.S3;
    dU[0] += F[qu] - F[c.q];
    dU[1 + d] += F[S3 + qu] - F[S3 + c.q];
    dU[1 + t1] += F[2 * S3 + qu] - F[2 * S3 + c.q];
    dU[1 + t2] += F[3 * S3 + qu] - F[3 * S3 + c.q];
    dU[4] += F[4 * S3 + qu] - F[4 * S3 + c.q];
  }
}

template <class R, class KP>
__device__ __forceinline__ void load_U_in(const KP& p, const Ctx<R, KP>& c, R (&u)[5]) {
  const int T = p.T;
  const R* U = p.Uin + (size_t)c.grp * p.nUi;
  const size_t T3 = (size_t)T * T * T, cq = ((size_t)c.k * T + c.j) * T + c.i;
#pragma unroll
  for (int v = 0; v < 5; ++v) u[v] = U[v * T3 + cq];
}

// ---- S4: half-step state: U^{n+1/2}, b^{n+1/2} on the faces of the cells, W^{n+1/2} -------
template <class R, int SC>
__global__ void __launch_bounds__(256, OccHalf<R>::minb) k_half(const KParamsSC<R, SC> p, const Box3 box, const int full) {
  typedef KParamsSC<R, SC> KP;
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  const R qh = (R(0.5) * p.dt) / p.dh;
  R u[5], dU[5];
  load_U_in(p, c, u);
  flux_div<A_F>(c, dU);
#pragma unroll
  for (int v = 0; v < 5; ++v) u[v] = u[v] - qh * dU[v];
  const int q = c.q;
  R bl[3], bu[3];
  bl[0] = ct_face<R, 0>(c, c.arr(A_B + 0), q, qh); bu[0] = ct_face<R, 0>(c, c.arr(A_B + 0), q + 1, qh);
  bl[1] = ct_face<R, 1>(c, c.arr(A_B + 1), q, qh); bu[1] = ct_face<R, 1>(c, c.arr(A_B + 1), q + p.S, qh);
  bl[2] = ct_face<R, 2>(c, c.arr(A_B + 2), q, qh); bu[2] = ct_face<R, 2>(c, c.arr(A_B + 2), q + p.S2, qh);
  c.arr(A_BH + 0)[q] = bl[0]; c.arr(A_BH + 1)[q] = bl[1]; c.arr(A_BH + 2)[q] = bl[2];
  if (c.i == box.lo[0] + box.n[0] - 1) c.arr(A_BH + 0)[q + 1] = bu[0];
  if (c.j == box.lo[1] + box.n[1] - 1) c.arr(A_BH + 1)[q + p.S] = bu[1];
  if (c.k == box.lo[2] + box.n[2] - 1) c.arr(A_BH + 2)[q + p.S2] = bu[2];
  R W[8];
  cons_to_prim(p, u, bl, bu, W);
  if (full) { store_prim(c, A_WH, W); return; }
  // CTU: only the density and the reference EMFs of the half-step state are read later (steps 5 + 6 take the half-step
  // normal field; the EMF kernel of step 7 takes rho and -(v x Bc))
  c.arr(A_WH)[q] = W[0];
  c.arr(A_EC + 0)[q] = W[3] * W[6] - W[2] * W[7];
  c.arr(A_EC + 1)[q] = W[1] * W[7] - W[3] * W[5];
  c.arr(A_EC + 2)[q] = W[2] * W[5] - W[1] * W[6];
}

}  // namespace mhd

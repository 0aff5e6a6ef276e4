// mhd_kernels2.cuh -- stage kernels, part 2: VL steps 4+5, CTU steps 1, 2/6 and 5.  See mhd_kernels.cuh for the layout.
#pragma once
#include "mhd_kernels.cuh"

namespace mhd {

// ---- VL steps 4+5: PLM at the half step + Riemann solve, normal B = half-step face value --------
// PLM states of a D face from the half-step primitives (shared by the flux kernel and the eta kernel of the H-correction)
template <class R, int LIMVAR, int D, bool COUNT, class KP>
__device__ __forceinline__ void plm_states_vl(const Ctx<R, KP>& c, const KP& p, R (&wl)[7], R (&wr)[7]) {
  const int o = c.off(D), q = c.q;
  const R* Wh = c.arr(A_WH);
  R wmm[7], wm[7], w0[7], wp[7], sl[7], sr[7];
  load_gen<R, D>(Wh, p.S3, q - 2 * o, wmm);
  load_gen<R, D>(Wh, p.S3, q - o, wm);
  load_gen<R, D>(Wh, p.S3, q, w0);
  load_gen<R, D>(Wh, p.S3, q + o, wp);
  slope3<R, LIMVAR>(wmm, wm, w0, Wh[(size_t)(5 + D) * p.S3 + q - o], p.gam, sl);
  slope3<R, LIMVAR>(wm, w0, wp, Wh[(size_t)(5 + D) * p.S3 + q], p.gam, sr);
#pragma unroll
  for (int v = 0; v < 7; ++v) { wl[v] = wm[v] + R(0.5) * sl[v]; wr[v] = w0[v] - R(0.5) * sr[v]; }
  apply_floors<COUNT>(p, wl); apply_floors<COUNT>(p, wr);
}
template <class R, int SOLVER, int LIMVAR, int D, bool HC, class KP>
__device__ __forceinline__ void flux2_vl_dir(const KP& p, const Box3& box) {
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  const int q = c.q;
  R wl[7], wr[7], F[7];
  plm_states_vl<R, LIMVAR, D, true>(c, p, wl, wr);
  // eta^H: this face and the lower / upper T1 and T2 faces of its two cells (k_eta2_vl wrote them on a box one face wider)
  const R etah = HC ? eta_h<R, D>(c, A_ETA, q) : R(0);
  const bool fb = riemann<R, SOLVER>(wl, wr, c.arr(A_BH + D)[q], p.gam, p.gm1inv, F, etah);
  if (fb) count_event(p.stats + 2);
#pragma unroll
  for (int v = 0; v < 7; ++v) c.arr(A_F + 7 * D + v)[q] = F[v];
}
template <class R, int SOLVER, int LIMVAR, int SC, bool HC = false>
__global__ void __launch_bounds__(256, OccFlux<R, SOLVER>::minb) k_flux2_vl(const KParamsSC<R, SC> p, const Box3x3 bx) {
  switch (blockIdx.y) {
    case 0: flux2_vl_dir<R, SOLVER, LIMVAR, 0, HC>(p, bx.b[0]); break;
    case 1: flux2_vl_dir<R, SOLVER, LIMVAR, 1, HC>(p, bx.b[1]); break;
    default: flux2_vl_dir<R, SOLVER, LIMVAR, 2, HC>(p, bx.b[2]); break;
  }
}
// H-correction (R19): eta of every pass-2 face and of the transverse faces around them (the same PLM states, floors not counted twice)
template <class R, int LIMVAR, int D, class KP>
__device__ __forceinline__ void eta2_vl_dir(const KP& p, const Box3& box) {
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  R wl[7], wr[7];
  plm_states_vl<R, LIMVAR, D, false>(c, p, wl, wr);
  c.arr(A_ETA + D)[c.q] = eta_face(wl, wr, c.arr(A_BH + D)[c.q], p.gam);
}
template <class R, int LIMVAR, int SC>
__global__ void __launch_bounds__(256, Occ<R>::minb) k_eta2_vl(const KParamsSC<R, SC> p, const Box3x3 bx) {
  switch (blockIdx.y) {
    case 0: eta2_vl_dir<R, LIMVAR, 0>(p, bx.b[0]); break;
    case 1: eta2_vl_dir<R, LIMVAR, 1>(p, bx.b[1]); break;
    default: eta2_vl_dir<R, LIMVAR, 2>(p, bx.b[2]); break;
  }
}

// ---- CTU step 1: reconstruction + half-step tracing + primitive MHD source terms ------------------
// PPM needs the limited slope of three cells per cell: the slopes are computed once per cell and direction by
// k_slope_ctu (parked in the flux arrays, which are free until step 2) and read back here.
template <class R, int LIMVAR, int D, class KP>
__device__ __forceinline__ void slope_ctu_dir(const KP& p, const Box3& box, int wbase) {
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  const int o = c.off(D), q = c.q, S3 = p.S3;
  const R* W = c.arr(wbase);
  R wm[7], w0[7], wp[7], dw[7];
  load_gen<R, D>(W, S3, q - o, wm);
  load_gen<R, D>(W, S3, q, w0);
  load_gen<R, D>(W, S3, q + o, wp);
  slope3<R, LIMVAR>(wm, w0, wp, W[(size_t)(5 + D) * S3 + q], p.gam, dw);
#pragma unroll
  for (int v = 0; v < 7; ++v) c.arr(A_F + 7 * D + v)[q] = dw[v];
}
template <class R, int LIMVAR, int SC>
__global__ void __launch_bounds__(256, Occ<R>::minb) k_slope_ctu(const KParamsSC<R, SC> p, const Box3x3 bx, int wbase) {
  switch (blockIdx.y) {
    case 0: slope_ctu_dir<R, LIMVAR, 0>(p, bx.b[0], wbase); break;
    case 1: slope_ctu_dir<R, LIMVAR, 1>(p, bx.b[1], wbase); break;
    default: slope_ctu_dir<R, LIMVAR, 2>(p, bx.b[2], wbase); break;
  }
}

template <class R, int RECON, int LIMVAR, int D, class KP>
__device__ __forceinline__ void recon_ctu_dir(const KP& p, const Box3& box, int wbase) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  const int o = c.off(D), q = c.q, S3 = p.S3;
  const R* W = c.arr(wbase);
  const R* Bn = W + (size_t)(5 + D) * S3;
  const R sig = p.dt / p.dh, hdt = R(0.5) * p.dt;
  R wm[7], w0[7], wp[7], wlo[7], wup[7];
  load_gen<R, D>(W, S3, q - o, wm);
  load_gen<R, D>(W, S3, q, w0);
  load_gen<R, D>(W, S3, q + o, wp);
  if (RECON == kPLM) {
    R dw[7];
    slope3<R, LIMVAR>(wm, w0, wp, Bn[q], p.gam, dw);
    plm_trace(w0, Bn[q], p.gam, sig, dw, wlo, wup);
  } else {
    R sm[7], s0[7], sp[7];
#pragma unroll
    for (int v = 0; v < 7; ++v) {
      const R* sl = c.arr(A_F + 7 * D + v);
      sm[v] = sl[q - o]; s0[v] = sl[q]; sp[v] = sl[q + o];
    }
    if (RECON == kPPMNoTrace) {
      // VL + PPM (NEXT-4): the parabola's interface values at the half step, no tracing, no source terms
      R W6[7];
      ppm_parabola(wm, w0, wp, sm, s0, sp, wlo, wup, W6);
      apply_floors(p, wlo); apply_floors(p, wup);
#pragma unroll
      for (int v = 0; v < 7; ++v) { c.arr(A_LO + 7 * D + v)[q] = wlo[v]; c.arr(A_UP + 7 * D + v)[q] = wup[v]; }
      return;
    }
    ppm_trace(wm, w0, wp, sm, s0, sp, Bn[q], p.gam, sig, wlo, wup);
  }
  const R* bn_ = c.arr(A_B + D); const R* b1_ = c.arr(A_B + T1); const R* b2_ = c.arr(A_B + T2);
  const R idh = R(1) / p.dh;
  const R dbn = (bn_[q + o] - bn_[q]) * idh;
  const R db1 = (b1_[q + c.off(T1)] - b1_[q]) * idh;
  const R db2 = (b2_[q + c.off(T2)] - b2_[q]) * idh;
  const R s1 = hdt * w0[2] * lim_minmod(dbn, -db1), s2 = hdt * w0[3] * lim_minmod(dbn, -db2);
  wlo[5] += s1; wup[5] += s1; wlo[6] += s2; wup[6] += s2;
  apply_floors(p, wlo); apply_floors(p, wup);
#pragma unroll
  for (int v = 0; v < 7; ++v) { c.arr(A_LO + 7 * D + v)[q] = wlo[v]; c.arr(A_UP + 7 * D + v)[q] = wup[v]; }
}
template <class R, int RECON, int LIMVAR, int SC>
__global__ void __launch_bounds__(256, Occ<R>::minb) k_recon_ctu(const KParamsSC<R, SC> p, const Box3x3 bx, int wbase) {
  switch (blockIdx.y) {
    case 0: recon_ctu_dir<R, RECON, LIMVAR, 0>(p, bx.b[0], wbase); break;
    case 1: recon_ctu_dir<R, RECON, LIMVAR, 1>(p, bx.b[1], wbase); break;
    default: recon_ctu_dir<R, RECON, LIMVAR, 2>(p, bx.b[2], wbase); break;
  }
}

// ---- CTU steps 2 and 6: Riemann solve between the upper state of cell i-1 and the lower of i ----
// HC (kHcOff / kHcEta / kHcOn) and etabase: H-correction of VL + PPM, whose pass 2 runs through this kernel
template <class R, int SOLVER, int D, int HC, class KP>
__device__ __forceinline__ void flux_lr_dir(const KP& p, const Box3& box, int bbase) {
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  const int q = c.q, ql = q - c.off(D);
  R wl[7], wr[7], F[7];
#pragma unroll
  for (int v = 0; v < 7; ++v) { wl[v] = c.arr(A_UP + 7 * D + v)[ql]; wr[v] = c.arr(A_LO + 7 * D + v)[q]; }
  if (HC == kHcEta) { c.arr(A_ETA + D)[q] = eta_face(wl, wr, c.arr(bbase + D)[q], p.gam); return; }
  const R etah = HC == kHcOn ? eta_h<R, D>(c, A_ETA, q) : R(0);
  const bool fb = riemann<R, SOLVER>(wl, wr, c.arr(bbase + D)[q], p.gam, p.gm1inv, F, etah);
  if (fb) count_event(p.stats + 2);
#pragma unroll
  for (int v = 0; v < 7; ++v) c.arr(A_F + 7 * D + v)[q] = F[v];
}
template <class R, int SOLVER, int SC, int HC = kHcOff>
__global__ void __launch_bounds__(256, OccFlux<R, SOLVER>::minb) k_flux_lr(const KParamsSC<R, SC> p, const Box3x3 bx, int bbase) {
  switch (blockIdx.y) {
    case 0: flux_lr_dir<R, SOLVER, 0, HC>(p, bx.b[0], bbase); break;
    case 1: flux_lr_dir<R, SOLVER, 1, HC>(p, bx.b[1], bbase); break;
    default: flux_lr_dir<R, SOLVER, 2, HC>(p, bx.b[2], bbase); break;
  }
}

// ---- CTU steps 5 + 6: transverse flux-gradient correction + conservative MHD source terms (R6) of
// the two states of a face, then the Riemann solve.  The corrected states never go to memory: the face reads the
// step-1 states of its two cells (upper state of cell i-1, lower state of cell i), everything the correction of each
// cell needs (pass-1 fluxes and edge EMFs of the transverse directions, time-n field gradients), and writes the pass-2
// flux into its own arrays (A_F2) because neighbouring faces still read the pass-1 fluxes.
// The part of the correction shared by the two faces of a cell:
template <class R> struct CtuCorr {
  R dF0, dF1, dF2, dF3, dF4;   // transverse flux differences in the generic order of D: (rho, M_D, M_T1, M_T2, e)
  R dB1, dB2;                  // CT update of the transverse field by the step-3 edge EMFs along D
  R dbn, m1, m2;               // dB_D/dD and the limited source factors
  R Bcn, Bc1, Bc2, v1, v2;     // time-n cell-centred field and transverse velocity
};
template <class R, int D, class KP>
__device__ __forceinline__ void ctu_corr_cell(const Ctx<R, KP>& c, const KP& p, int q, R qh, CtuCorr<R>& k) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  const int od = c.off(D), o1 = c.off(T1), o2 = c.off(T2);
  const size_t S3 = p.S3;
  R w0[7];
  load_gen<R, D>(c.arr(A_W), p.S3, q, w0);
  k.Bcn = c.arr(A_W + 5 + D)[q];
  // F[T1] is stored in generic order (T1, T2, D): its momentum slots (Mn, Mt1, Mt2) are (M_T1, M_T2, M_D);
  // F[T2] is in order (T2, D, T1): (M_T2, M_D, M_T1).  Permute into the generic order of D: (rho, M_D, M_T1, M_T2, e).
  const R* F1 = c.arr(A_F + 7 * T1); const R* F2 = c.arr(A_F + 7 * T2);
  auto d1 = [&](int comp) { return F1[comp * S3 + q + o1] - F1[comp * S3 + q]; };
  auto d2 = [&](int comp) { return F2[comp * S3 + q + o2] - F2[comp * S3 + q]; };
  k.dF0 = d1(0) + d2(0); k.dF1 = d1(3) + d2(2); k.dF2 = d1(1) + d2(3); k.dF3 = d1(2) + d2(1); k.dF4 = d1(4) + d2(4);
  const R* En = c.arr(A_E + D);
  const R Emm = En[q], Epm = En[q + o1], Emp = En[q + o2], Epp = En[q + o1 + o2];
  k.dB1 = -qh * R(0.5) * ((Emp - Emm) + (Epp - Epm));
  k.dB2 = qh * R(0.5) * ((Epm - Emm) + (Epp - Emp));
  const R* bn_ = c.arr(A_B + D); const R* b1_ = c.arr(A_B + T1); const R* b2_ = c.arr(A_B + T2);
  const R idh = R(1) / p.dh;
  k.dbn = (bn_[q + od] - bn_[q]) * idh;
  const R db1 = (b1_[q + o1] - b1_[q]) * idh, db2 = (b2_[q + o2] - b2_[q]) * idh;
  k.m1 = lim_minmod(k.dbn, -db2); k.m2 = lim_minmod(k.dbn, -db1);
  k.Bc1 = w0[5]; k.Bc2 = w0[6]; k.v1 = w0[2]; k.v2 = w0[3];
}
// one state w of the cell (at the face whose time-n normal field is bnn and half-step normal field bh): to conserved
// variables, correct, back to primitive variables with the floors of R9
template <bool COUNT = true, class R, class KP>
__device__ __forceinline__ void ctu_corr_apply(const KP& p, const CtuCorr<R>& k, R hdt, R qh, R bnn, R bh, R (&w)[7]) {
  R u[7];
  u[0] = w[0]; u[1] = w[0] * w[1]; u[2] = w[0] * w[2]; u[3] = w[0] * w[3];
  u[4] = w[4] * p.gm1inv + R(0.5) * w[0] * (sqr(w[1]) + sqr(w[2]) + sqr(w[3])) + R(0.5) * (sqr(bnn) + sqr(w[5]) + sqr(w[6]));
  u[5] = w[5]; u[6] = w[6];
  u[0] -= qh * k.dF0; u[1] -= qh * k.dF1; u[2] -= qh * k.dF2; u[3] -= qh * k.dF3; u[4] -= qh * k.dF4;
  u[5] += k.dB1; u[6] += k.dB2;
  u[1] += hdt * k.Bcn * k.dbn; u[2] += hdt * k.Bc1 * k.dbn; u[3] += hdt * k.Bc2 * k.dbn;
  u[5] += hdt * k.v1 * k.m1; u[6] += hdt * k.v2 * k.m2;
  u[4] += hdt * (k.Bc1 * k.v1 * k.m1 + k.Bc2 * k.v2 * k.m2);
  R rho = u[0];
  if (rho < p.min_dens) { rho = p.min_dens; if (COUNT) count_event(p.stats + 0); }
  const R ir = frcp(rho);
  w[0] = rho; w[1] = u[1] * ir; w[2] = u[2] * ir; w[3] = u[3] * ir; w[5] = u[5]; w[6] = u[6];
  w[4] = p.gm1 * (u[4] - R(0.5) * rho * (sqr(w[1]) + sqr(w[2]) + sqr(w[3])) - R(0.5) * (sqr(bh) + sqr(w[5]) + sqr(w[6])));
  if (w[4] < p.min_pres) { w[4] = p.min_pres; if (COUNT) count_event(p.stats + 1); }
}
// HC = kHcEta: the corrected states only, for eta of the face (floors not counted twice); kHcOn: the Roe solver with eta^H
template <class R, int SOLVER, int D, int HC, class KP>
__device__ __forceinline__ void flux2_ctu_dir(const KP& p, const Box3& box) {
  Ctx<R, KP> c(p, box);
  if (!c.ok) return;
  const int q = c.q, ql = q - c.off(D);
  const R hdt = R(0.5) * p.dt, qh = hdt / p.dh;
  R wl[7], wr[7], F[7];
#pragma unroll
  for (int v = 0; v < 7; ++v) { wl[v] = c.arr(A_UP + 7 * D + v)[ql]; wr[v] = c.arr(A_LO + 7 * D + v)[q]; }
  const R bnn = c.arr(A_B + D)[q], bh = c.arr(A_BH + D)[q];
  CtuCorr<R> k;
  ctu_corr_cell<R, D>(c, p, ql, qh, k);
  ctu_corr_apply<HC != kHcEta>(p, k, hdt, qh, bnn, bh, wl);
  ctu_corr_cell<R, D>(c, p, q, qh, k);
  ctu_corr_apply<HC != kHcEta>(p, k, hdt, qh, bnn, bh, wr);
  if (HC == kHcEta) { c.arr(A_ETAC + D)[q] = eta_face(wl, wr, bh, p.gam); return; }
  const R etah = HC == kHcOn ? eta_h<R, D>(c, A_ETAC, q) : R(0);
  const bool fb = riemann<R, SOLVER>(wl, wr, bh, p.gam, p.gm1inv, F, etah);
  if (fb) count_event(p.stats + 2);
#pragma unroll
  for (int v = 0; v < 7; ++v) c.arr(A_F2 + 7 * D + v)[q] = F[v];
}
template <class R, int SOLVER, int SC, int HC = kHcOff>
__global__ void __launch_bounds__(256, OccFlux<R, SOLVER>::minb) k_flux2_ctu(const KParamsSC<R, SC> p, const Box3x3 bx) {
  switch (blockIdx.y) {
    case 0: flux2_ctu_dir<R, SOLVER, 0, HC>(p, bx.b[0]); break;
    case 1: flux2_ctu_dir<R, SOLVER, 1, HC>(p, bx.b[1]); break;
    default: flux2_ctu_dir<R, SOLVER, 2, HC>(p, bx.b[2]); break;
  }
}

}  // namespace mhd

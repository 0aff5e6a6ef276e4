// mhd_eigen.cuh -- eigen-system based pieces: Roe and HLLE Riemann solvers, characteristic
// limiting and the primitive flux Jacobian used by the CTU tracing.  Formulas: DESIGN.md
// R4/R5/R7/R11/R18 (the paper defers them to Stone et al. 2008).  Waves are generated one at a time
// (left vector -> amplitude -> right vector) so that no 7x7 matrix is ever resident in registers.
#pragma once
#include "mhd_physics.cuh"

namespace mhd {

// magnetosonic speeds and the normalisation factors alpha_f/s, beta_1/2 shared by both eigen-systems
template <class R> struct WaveSet { R cf, cs, ca, af, as, b1, b2, S; };

template <class R>
__device__ __forceinline__ WaveSet<R> wave_set(R a2, R rho, R bn, R B1, R B2) {
  WaveSet<R> w;
  const R ir = frcp(rho);
  const R bt2 = B1 * B1 + B2 * B2;
  const R ca2 = bn * bn * ir, ct2 = bt2 * ir;
  const R sum = a2 + ca2 + ct2, dif = ca2 + ct2 - a2;
  const R cf2 = R(0.5) * (sum + Num<R>::sqrt(dif * dif + R(4) * a2 * ct2));
  R cs2 = (cf2 > R(0)) ? fdiv(a2 * ca2, cf2) : R(0);
  cs2 = (cs2 < R(0)) ? R(0) : cs2;
  w.cf = Num<R>::sqrt(cf2); w.cs = Num<R>::sqrt(cs2); w.ca = Num<R>::sqrt(ca2);
  const R den = cf2 - cs2;
  if (den <= R(0)) { w.af = R(1); w.as = R(0); }
  else {
    const R iden = frcp(den);
    R af2 = (a2 - cs2) * iden, as2 = (cf2 - a2) * iden;
    af2 = Num<R>::min(R(1), Num<R>::max(R(0), af2));
    as2 = Num<R>::min(R(1), Num<R>::max(R(0), as2));
    w.af = Num<R>::sqrt(af2); w.as = Num<R>::sqrt(as2);
  }
  const R bt = Num<R>::sqrt(bt2);
  if (bt == R(0)) { w.b1 = R(1); w.b2 = R(0); }
  else { const R ibt = frcp(bt); w.b1 = B1 * ibt; w.b2 = B2 * ibt; }
  w.S = (bn >= R(0)) ? R(1) : R(-1);
  return w;
}

// Roe average in total-enthalpy form with the single correction term X (R11)
template <class R> struct RoeAvg { R rho, vn, v1, v2, H, B1, B2, X, a2; };

template <class R>
__device__ __forceinline__ RoeAvg<R> roe_average(const R (&wl)[7], const R (&wr)[7], const Side<R>& L,
                                                 const Side<R>& Rr, R bn2, R gam) {
  RoeAvg<R> r;
  const R sl = Num<R>::sqrt(wl[0]), sr = Num<R>::sqrt(wr[0]);
  const R iw = frcp(sl + sr);
  const R HL = fdiv(L.U[4] + L.pT, wl[0]), HR = fdiv(Rr.U[4] + Rr.pT, wr[0]);
  r.rho = sl * sr;
  r.vn = (sl * wl[1] + sr * wr[1]) * iw;
  r.v1 = (sl * wl[2] + sr * wr[2]) * iw;
  r.v2 = (sl * wl[3] + sr * wr[3]) * iw;
  r.H = (sl * HL + sr * HR) * iw;
  r.B1 = (sr * wl[5] + sl * wr[5]) * iw;   // density weights swapped for the transverse field
  r.B2 = (sr * wl[6] + sl * wr[6]) * iw;
  r.X = (sqr(wl[5] - wr[5]) + sqr(wl[6] - wr[6])) * R(0.5) * iw * iw;
  const R irr = frcp(r.rho);
  const R ca2 = bn2 * irr, ct2 = (sqr(r.B1) + sqr(r.B2)) * irr;
  const R Hp = r.H - ca2 - ct2;
  const R v2 = sqr(r.vn) + sqr(r.v1) + sqr(r.v2);
  r.a2 = (gam - R(1)) * (Hp - R(0.5) * v2) - (gam - R(2)) * r.X;
  return r;
}

// HLLE with Einfeldt speeds; the Roe-average speeds take part only when a~^2 > 0 (R7)
template <class R>
__device__ __forceinline__ void hlle_flux(const R (&wl)[7], const R (&wr)[7], const Side<R>& L, const Side<R>& Rr,
                                          bool roe_ok, R roe_vn, R roe_cf, R (&F)[7]) {
  R bp = Num<R>::max(wr[1] + Rr.cf, R(0)), bm = Num<R>::min(wl[1] - L.cf, R(0));
  if (roe_ok) { bp = Num<R>::max(bp, roe_vn + roe_cf); bm = Num<R>::min(bm, roe_vn - roe_cf); }
  const R idb = frcp(bp - bm), bpm = bp * bm;
#pragma unroll
  for (int c = 0; c < 7; ++c) F[c] = (bp * L.F[c] - bm * Rr.F[c] + bpm * (Rr.U[c] - L.U[c])) * idb;
}

template <class R>
__device__ __forceinline__ void riemann_hlle(const R (&wl)[7], const R (&wr)[7], R bn, R gam, R gm1inv, R (&F)[7]) {
  const R bn2 = bn * bn;
  Side<R> L, Rr;
  side_setup(wl, bn, bn2, gm1inv, gam, L);
  side_setup(wr, bn, bn2, gm1inv, gam, Rr);
  const RoeAvg<R> r = roe_average(wl, wr, L, Rr, bn2, gam);
  const bool ok = r.a2 > R(0);
  R cf = R(0);
  if (ok) cf = wave_set(r.a2, r.rho, bn, r.B1, r.B2).cf;
  hlle_flux(wl, wr, L, Rr, ok, r.vn, cf, F);
}

// Roe: F = 1/2 (F_L + F_R) - 1/2 sum_k |lambda_k| (L_k . dU) R_k on the conserved eigen-system of the Roe average;
// HLLE where a~^2 <= 0 or an intermediate state has rho <= 0 or P <= 0.  Returns true if it fell back.
template <class R>
// etah (R19, H-correction): every wave speed of the dissipation term is max(|lam_k|, etah); 0: the plain solver
__device__ __forceinline__ bool riemann_roe(const R (&wl)[7], const R (&wr)[7], R bn, R gam, R gm1inv, R (&F)[7], R etah = R(0)) {
  const R bn2 = bn * bn;
  Side<R> L, Rr;
  side_setup(wl, bn, bn2, gm1inv, gam, L);
  side_setup(wr, bn, bn2, gm1inv, gam, Rr);
  const RoeAvg<R> r = roe_average(wl, wr, L, Rr, bn2, gam);
  const bool a2ok = r.a2 > R(0);
  const R a2 = r.a2, a = Num<R>::sqrt(a2), srho = Num<R>::sqrt(r.rho), isrho = frcp(srho);
  const WaveSet<R> w = wave_set(a2, r.rho, bn, r.B1, r.B2);
  const R irr = isrho * isrho;
  const R ca2 = bn2 * irr, bt2 = sqr(r.B1) + sqr(r.B2), ct2 = bt2 * irr;
  const R Hp = r.H - ca2 - ct2;
  const R vsq = sqr(r.vn) + sqr(r.v1) + sqr(r.v2);
  const R Qf = w.cf * w.af * w.S, Qs = w.cs * w.as * w.S;
  const R Afp = a * w.af * isrho, Asp = a * w.as * isrho;
  const R vb = r.v1 * w.b1 + r.v2 * w.b2, bt = Num<R>::sqrt(bt2);
  const R xt = fdiv((gam - R(2)) * r.X, gam - R(1));
  const R nn = fdiv(R(0.5), a2), g = (gam - R(1)) * nn;
  const R vxb = r.v1 * w.b2 - r.v2 * w.b1;
  const R lam[7] = { r.vn - w.cf, r.vn - w.ca, r.vn - w.cs, r.vn, r.vn + w.cs, r.vn + w.ca, r.vn + w.cf };

  R dU[7], Ui[7], diss[7];
#pragma unroll
  for (int c = 0; c < 7; ++c) { dU[c] = Rr.U[c] - L.U[c]; Ui[c] = L.U[c]; diss[c] = R(0); }
  bool bad = false;
#pragma unroll
  for (int k = 0; k < 7; ++k) {
    const R s = (k < 3) ? R(1) : R(-1);      // s = +1: the left-going ("-") wave, s = -1: the right-going one
    R Lk[7], Rk[7];
    if (k == 0 || k == 6) {                  // fast
      Lk[0] = g * w.af * (vsq - Hp) + nn * w.af * w.cf * (w.cf + s * r.vn) - s * nn * Qs * vb - nn * Asp * bt;
      Lk[1] = -g * w.af * r.vn - s * nn * w.af * w.cf;
      Lk[2] = -g * w.af * r.v1 + s * nn * Qs * w.b1;
      Lk[3] = -g * w.af * r.v2 + s * nn * Qs * w.b2;
      Lk[4] = g * w.af;
      Lk[5] = nn * Asp * r.rho * w.b1 - g * w.af * r.B1;
      Lk[6] = nn * Asp * r.rho * w.b2 - g * w.af * r.B2;
      Rk[0] = w.af; Rk[1] = w.af * (r.vn - s * w.cf);
      Rk[2] = w.af * r.v1 + s * Qs * w.b1; Rk[3] = w.af * r.v2 + s * Qs * w.b2;
      Rk[4] = w.af * (Hp - s * r.vn * w.cf) + s * Qs * vb + Asp * bt;
      Rk[5] = Asp * w.b1; Rk[6] = Asp * w.b2;
    } else if (k == 1 || k == 5) {           // Alfven
      Lk[0] = s * R(0.5) * vxb; Lk[1] = R(0); Lk[2] = -s * R(0.5) * w.b2; Lk[3] = s * R(0.5) * w.b1; Lk[4] = R(0);
      Lk[5] = -R(0.5) * srho * w.b2 * w.S; Lk[6] = R(0.5) * srho * w.b1 * w.S;
      Rk[0] = R(0); Rk[1] = R(0); Rk[2] = -s * w.b2; Rk[3] = s * w.b1; Rk[4] = -s * vxb;
      Rk[5] = -w.b2 * w.S * isrho; Rk[6] = w.b1 * w.S * isrho;
    } else if (k == 2 || k == 4) {           // slow
      Lk[0] = g * w.as * (vsq - Hp) + nn * w.as * w.cs * (w.cs + s * r.vn) + s * nn * Qf * vb + nn * Afp * bt;
      Lk[1] = -g * w.as * r.vn - s * nn * w.as * w.cs;
      Lk[2] = -g * w.as * r.v1 - s * nn * Qf * w.b1;
      Lk[3] = -g * w.as * r.v2 - s * nn * Qf * w.b2;
      Lk[4] = g * w.as;
      Lk[5] = -nn * Afp * r.rho * w.b1 - g * w.as * r.B1;
      Lk[6] = -nn * Afp * r.rho * w.b2 - g * w.as * r.B2;
      Rk[0] = w.as; Rk[1] = w.as * (r.vn - s * w.cs);
      Rk[2] = w.as * r.v1 - s * Qf * w.b1; Rk[3] = w.as * r.v2 - s * Qf * w.b2;
      Rk[4] = w.as * (Hp - s * r.vn * w.cs) - s * Qf * vb - Afp * bt;
      Rk[5] = -Afp * w.b1; Rk[6] = -Afp * w.b2;
    } else {                                  // entropy
      Lk[0] = R(1) - R(2) * g * (R(0.5) * vsq - xt);
      Lk[1] = R(2) * g * r.vn; Lk[2] = R(2) * g * r.v1; Lk[3] = R(2) * g * r.v2; Lk[4] = -R(2) * g;
      Lk[5] = R(2) * g * r.B1; Lk[6] = R(2) * g * r.B2;
      Rk[0] = R(1); Rk[1] = r.vn; Rk[2] = r.v1; Rk[3] = r.v2; Rk[4] = R(0.5) * vsq + xt; Rk[5] = R(0); Rk[6] = R(0);
    }
    R ak = R(0);
#pragma unroll
    for (int c = 0; c < 7; ++c) ak += Lk[c] * dU[c];
    const R wk = Num<R>::max(Num<R>::abs(lam[k]), etah) * ak;
#pragma unroll
    for (int c = 0; c < 7; ++c) { diss[c] += wk * Rk[c]; Ui[c] += ak * Rk[c]; }
    if (k < 6) {
      if (lam[k + 1] > lam[k]) {
        const R Pi = (gam - R(1)) * (Ui[4] - R(0.5) * fdiv(sqr(Ui[1]) + sqr(Ui[2]) + sqr(Ui[3]), Ui[0])
                                      - R(0.5) * (bn2 + sqr(Ui[5]) + sqr(Ui[6])));
        bad = bad || !(Ui[0] > R(0)) || !(Pi > R(0));
      }
    }
  }
  R Fh[7];
  hlle_flux(wl, wr, L, Rr, a2ok, r.vn, w.cf, Fh);
  const bool superL = lam[0] >= etah, superR = lam[6] <= -etah;     // R19: the shortcuts only where every wave is faster than etah
  const bool fallback = !a2ok || (!superL && !superR && bad);
#pragma unroll
  for (int c = 0; c < 7; ++c) {
    const R roe = R(0.5) * (L.F[c] + Rr.F[c]) - R(0.5) * diss[c];
    F[c] = fallback ? Fh[c] : (superL ? L.F[c] : (superR ? Rr.F[c] : roe));
  }
  return fallback;
}

template <class R, int SOLVER>
__device__ __forceinline__ bool riemann(const R (&wl)[7], const R (&wr)[7], R bn, R gam, R gm1inv, R (&F)[7], R etah = R(0)) {
  if (SOLVER == kHLLE) { riemann_hlle(wl, wr, bn, gam, gm1inv, F); return false; }
  else if (SOLVER == kHLLD) { riemann_hlld(wl, wr, bn, gam, gm1inv, F); return false; }
  else return riemann_roe(wl, wr, bn, gam, gm1inv, F, etah);
}
// R19: eta of a face = half the largest jump of the fast characteristic speeds v_n -+ c_f between its L and R states
template <class R>
__device__ __forceinline__ R eta_face(const R (&wl)[7], const R (&wr)[7], R bn, R gam) {
  const R bn2 = bn * bn;
  const R cl = fast_speed(wl[0], wl[4], bn2, wl[5] * wl[5] + wl[6] * wl[6], gam), cr = fast_speed(wr[0], wr[4], bn2, wr[5] * wr[5] + wr[6] * wr[6], gam);
  return R(0.5) * Num<R>::max(Num<R>::abs((wr[1] + cr) - (wl[1] + cl)), Num<R>::abs((wr[1] - cr) - (wl[1] - cl)));
}

}  // namespace mhd

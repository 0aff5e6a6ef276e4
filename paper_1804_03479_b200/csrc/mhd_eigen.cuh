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
// etah (R19, H-correction): every wave speed of the dissipation term is max(|lam_k|, etah); 0: the plain solver
//
// Evaluation: the left-going and the right-going wave of a family (fast, Alfven, slow) have left / right eigenvectors E +- O with a
// common even part E and an odd part O (the terms that carry the direction sign s).  The amplitudes L_k . dU are therefore E.dU +- O.dU
// with sums shared by all families (v.dM, B.dB, beta.dB, beta.dM), and the right vectors Re +- Ro are built once per family: no
// vector L_k is ever formed.  The intermediate states are still accumulated wave by wave in the order of the speeds (the
// positivity test of R7 needs them); their pressure test is the division-free rho (E - B^2/2) - M^2/2 > 0 (rho > 0 is tested first).
// The HLLE flux (and the fast speeds of the two sides it needs) is evaluated only where the solver falls back.
template <class R>
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
  // ---- amplitudes a_k = L_k . dU: even part + s * odd part, s = +1 for the left-going wave of a family ----
  R ak[7];
  {
    const R vdM = r.vn * dU[1] + r.v1 * dU[2] + r.v2 * dU[3];          // v . dM
    const R BdB = r.B1 * dU[5] + r.B2 * dU[6];                         // B_t . dB_t
    const R bdB = w.b1 * dU[5] + w.b2 * dU[6];                         // beta . dB_t
    const R bdM = w.b1 * dU[2] + w.b2 * dU[3];                         // beta . dM_t
    const R Y = dU[4] - vdM - BdB;
    const R G = g * ((vsq - Hp) * dU[0] + Y);
    const R Q = nn * (r.rho * bdB - bt * dU[0]);
    const R un = nn * (r.vn * dU[0] - dU[1]);
    const R tv = nn * (bdM - vb * dU[0]);
    const R Ef = w.af * (G + nn * w.cf * w.cf * dU[0]) + Asp * Q, Of = w.af * w.cf * un + Qs * tv;
    const R Es = w.as * (G + nn * w.cs * w.cs * dU[0]) - Afp * Q, Os = w.as * w.cs * un - Qf * tv;
    const R Ea = R(0.5) * srho * w.S * (w.b1 * dU[6] - w.b2 * dU[5]), Oa = R(0.5) * (vxb * dU[0] - w.b2 * dU[2] + w.b1 * dU[3]);
    ak[0] = Ef + Of; ak[6] = Ef - Of;
    ak[1] = Ea + Oa; ak[5] = Ea - Oa;
    ak[2] = Es + Os; ak[4] = Es - Os;
    ak[3] = dU[0] - R(2) * g * ((R(0.5) * vsq - xt) * dU[0] + Y);
  }
  // ---- right eigenvectors R_k = Re + s * Ro of each family (Ro has the components 1 .. 4 only) ----
  const R ReF[7] = { w.af, w.af * r.vn, w.af * r.v1, w.af * r.v2, w.af * Hp + Asp * bt, Asp * w.b1, Asp * w.b2 };
  const R RoF[4] = { -w.af * w.cf, Qs * w.b1, Qs * w.b2, Qs * vb - w.af * r.vn * w.cf };
  const R ReS[7] = { w.as, w.as * r.vn, w.as * r.v1, w.as * r.v2, w.as * Hp - Afp * bt, -Afp * w.b1, -Afp * w.b2 };
  const R RoS[4] = { -w.as * w.cs, -Qf * w.b1, -Qf * w.b2, -w.as * r.vn * w.cs - Qf * vb };
  const R ReA5 = -w.b2 * w.S * isrho, ReA6 = w.b1 * w.S * isrho;
  bool bad = false;
#pragma unroll
  for (int k = 0; k < 7; ++k) {
    const R s = (k < 3) ? R(1) : R(-1);
    R Rk[7];
    if (k == 0 || k == 6) {                  // fast
      Rk[0] = ReF[0]; Rk[5] = ReF[5]; Rk[6] = ReF[6];
#pragma unroll
      for (int c = 1; c < 5; ++c) Rk[c] = ReF[c] + s * RoF[c - 1];
    } else if (k == 1 || k == 5) {           // Alfven
      Rk[0] = R(0); Rk[1] = R(0); Rk[2] = -s * w.b2; Rk[3] = s * w.b1; Rk[4] = -s * vxb; Rk[5] = ReA5; Rk[6] = ReA6;
    } else if (k == 2 || k == 4) {           // slow
      Rk[0] = ReS[0]; Rk[5] = ReS[5]; Rk[6] = ReS[6];
#pragma unroll
      for (int c = 1; c < 5; ++c) Rk[c] = ReS[c] + s * RoS[c - 1];
    } else {                                  // entropy
      Rk[0] = R(1); Rk[1] = r.vn; Rk[2] = r.v1; Rk[3] = r.v2; Rk[4] = R(0.5) * vsq + xt; Rk[5] = R(0); Rk[6] = R(0);
    }
    const R wk = Num<R>::max(Num<R>::abs(lam[k]), etah) * ak[k];
#pragma unroll
    for (int c = 0; c < 7; ++c) { diss[c] += wk * Rk[c]; Ui[c] += ak[k] * Rk[c]; }
    if (k < 6) {
      if (lam[k + 1] > lam[k]) {
        // rho > 0 and P > 0 <=> rho (E - B^2/2) - M^2/2 > 0
        const R t = Ui[0] * (Ui[4] - R(0.5) * (bn2 + sqr(Ui[5]) + sqr(Ui[6]))) - R(0.5) * (sqr(Ui[1]) + sqr(Ui[2]) + sqr(Ui[3]));
        bad = bad || !(Ui[0] > R(0)) || !(t > R(0));
      }
    }
  }
  const bool superL = lam[0] >= etah, superR = lam[6] <= -etah;     // R19: the shortcuts only where every wave is faster than etah
  const bool fallback = !a2ok || (!superL && !superR && bad);
#pragma unroll
  for (int c = 0; c < 7; ++c) {
    const R roe = R(0.5) * (L.F[c] + Rr.F[c]) - R(0.5) * diss[c];
    F[c] = superL ? L.F[c] : (superR ? Rr.F[c] : roe);
  }
  if (fallback) hlle_flux(wl, wr, L, Rr, a2ok, r.vn, w.cf, F);
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

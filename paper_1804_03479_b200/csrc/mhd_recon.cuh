// mhd_recon.cuh -- limited slopes (primitive or characteristic variables), PLM / PPM face states and the
// half-step characteristic tracing of CTU step 1.  Formulas: DESIGN.md R4, R5.
#pragma once
#include "mhd_eigen.cuh"

namespace mhd {

// y = A(w0, bn) x : primitive-variable flux Jacobian of direction n, never formed as a matrix
template <class R>
__device__ __forceinline__ void jac_mul(const R (&w0)[7], R bn, R gam, R irho, const R (&x)[7], R (&y)[7]) {
  const R vn = w0[1];
  y[0] = vn * x[0] + w0[0] * x[1];
  y[1] = vn * x[1] + (x[4] + w0[5] * x[5] + w0[6] * x[6]) * irho;
  y[2] = vn * x[2] - bn * irho * x[5];
  y[3] = vn * x[3] - bn * irho * x[6];
  y[4] = vn * x[4] + gam * w0[4] * x[1];
  y[5] = vn * x[5] + w0[5] * x[1] - bn * x[2];
  y[6] = vn * x[6] + w0[6] * x[1] - bn * x[3];
}

// Limited slope of cell w0 from its two one-sided differences; LIMVAR = limvar + 2 * limiter.
// LIM_PRIM: componentwise.  LIM_CHAR: project on the left eigenvectors of (w0, bn), limit each characteristic
// amplitude, project back (wave order -f, -A, -s, entropy, +s, +A, +f).
template <class R, int LIMVAR>
__device__ __forceinline__ void limited_slope(const R (&w0)[7], R bn, R gam, const R (&dl)[7], const R (&dr)[7], R (&dw)[7]) {
  constexpr int LM = LIMVAR >> 1;
  if ((LIMVAR & 1) == kLimPrim) {
#pragma unroll
    for (int v = 0; v < 7; ++v) dw[v] = lim_sel<R, LM>(dl[v], dr[v]);
    return;
  }
  // The eigenvectors of SURVEY A1 are sparse and come in +/- pairs: the projections are written through the
  // components of the differences along and across beta = B_t/|B_t| (tv, tb / pv, pb), the pair sums and differences.
  const R rho = w0[0], irho = frcp(rho);
  const R a2 = gam * w0[4] * irho, a = Num<R>::sqrt(a2), srho = Num<R>::sqrt(rho), isrho = frcp(srho);
  const WaveSet<R> w = wave_set(a2, rho, bn, w0[5], w0[6]);
  const R Qf = w.cf * w.af * w.S, Qs = w.cs * w.as * w.S, Af = a * w.af * srho, As = a * w.as * srho;
  const R nn = fdiv(R(0.5), a2);
  R am[7];   // limited amplitudes in the wave order -f, -A, -s, entropy, +s, +A, +f
  {
    R amp[2][7];
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      const R (&d)[7] = side ? dr : dl;
      const R tv = w.b1 * d[2] + w.b2 * d[3], pv = w.b1 * d[3] - w.b2 * d[2];
      const R tb = w.b1 * d[5] + w.b2 * d[6], pb = w.b1 * d[6] - w.b2 * d[5];
      const R Pf = nn * irho * (w.af * d[4] + As * tb), Vf = nn * (w.cf * w.af * d[1] - Qs * tv);
      const R Ps = nn * irho * (w.as * d[4] - Af * tb), Vs = nn * (w.cs * w.as * d[1] + Qf * tv);
      const R Pa = R(0.5) * w.S * isrho * pb, Va = R(0.5) * pv;
      amp[side][0] = Pf - Vf; amp[side][6] = Pf + Vf;
      amp[side][2] = Ps - Vs; amp[side][4] = Ps + Vs;
      amp[side][1] = Pa + Va; amp[side][5] = Pa - Va;
      amp[side][3] = d[0] - R(2) * nn * d[4];
    }
#pragma unroll
    for (int k = 0; k < 7; ++k) am[k] = lim_sel<R, LM>(amp[0][k], amp[1][k]);
  }
  const R Fs = am[0] + am[6], Fd = am[0] - am[6], Ss = am[2] + am[4], Sd = am[2] - am[4];
  const R Asum = am[1] + am[5], Adif = am[1] - am[5];
  const R comp = w.af * Fs + w.as * Ss;                  // compressive part: density and pressure
  const R tv = Qs * Fd - Qf * Sd, tb = As * Fs - Af * Ss, pb = w.S * srho * Asum;
  dw[0] = rho * comp + am[3];
  dw[1] = -(w.cf * w.af * Fd + w.cs * w.as * Sd);
  dw[2] = w.b1 * tv - w.b2 * Adif;
  dw[3] = w.b2 * tv + w.b1 * Adif;
  dw[4] = rho * a2 * comp;
  dw[5] = w.b1 * tb - w.b2 * pb;
  dw[6] = w.b2 * tb + w.b1 * pb;
}

template <class R, int LIMVAR>
__device__ __forceinline__ void slope3(const R (&wm)[7], const R (&w0)[7], const R (&wp)[7], R bn, R gam, R (&dw)[7]) {
  R dl[7], dr[7];
#pragma unroll
  for (int v = 0; v < 7; ++v) { dl[v] = w0[v] - wm[v]; dr[v] = wp[v] - w0[v]; }
  limited_slope<R, LIMVAR>(w0, bn, gam, dl, dr, dw);
}

// CTU step 1, PLM: states at the lower / upper face of the cell at t^{n+1/2} (matrix-form tracing, all waves)
template <class R>
__device__ __forceinline__ void plm_trace(const R (&w0)[7], R bn, R gam, R sig, const R (&dw)[7], R (&wlo)[7], R (&wup)[7]) {
  R Ad[7];
  jac_mul(w0, bn, gam, frcp(w0[0]), dw, Ad);
#pragma unroll
  for (int v = 0; v < 7; ++v) {
    wup[v] = w0[v] + R(0.5) * dw[v] - R(0.5) * sig * Ad[v];
    wlo[v] = w0[v] - R(0.5) * dw[v] - R(0.5) * sig * Ad[v];
  }
}

// PPM parabola of a cell from the limited slopes of the cell and its two neighbours, monotonised (R4 i-iii):
// interface values Wl, Wr and W6
template <class R>
__device__ __forceinline__ void ppm_parabola(const R (&wm)[7], const R (&w0)[7], const R (&wp)[7], const R (&sm)[7],
                                             const R (&s0)[7], const R (&sp)[7], R (&Wl)[7], R (&Wr)[7], R (&W6)[7]) {
#pragma unroll
  for (int v = 0; v < 7; ++v) {
    R l = R(0.5) * (wm[v] + w0[v]) - (s0[v] - sm[v]) * R(1.0 / 6.0);
    R r = R(0.5) * (w0[v] + wp[v]) - (sp[v] - s0[v]) * R(1.0 / 6.0);
    if ((r - w0[v]) * (w0[v] - l) <= R(0)) { l = w0[v]; r = w0[v]; }
    const R d = r - l, w6 = R(6) * (w0[v] - R(0.5) * (l + r));
    R nl = l, nr = r;
    if (d * w6 > d * d) nl = R(3) * w0[v] - R(2) * r;
    if (d * w6 < -d * d) nr = R(3) * w0[v] - R(2) * l;
    l = Num<R>::max(Num<R>::min(w0[v], wm[v]), Num<R>::min(Num<R>::max(w0[v], wm[v]), nl));
    r = Num<R>::max(Num<R>::min(w0[v], wp[v]), Num<R>::min(Num<R>::max(w0[v], wp[v]), nr));
    Wl[v] = l; Wr[v] = r;
    W6[v] = R(6) * (w0[v] - R(0.5) * (l + r));
  }
}

// CTU step 1, PPM: the parabola traced with its first and second moments (matrix form, all waves).
template <class R>
__device__ __forceinline__ void ppm_trace(const R (&wm)[7], const R (&w0)[7], const R (&wp)[7], const R (&sm)[7],
                                          const R (&s0)[7], const R (&sp)[7], R bn, R gam, R sig, R (&wlo)[7], R (&wup)[7]) {
  R Wl[7], Wr[7], xu[7], xl[7], W6[7];
  ppm_parabola(wm, w0, wp, sm, s0, sp, Wl, Wr, W6);
#pragma unroll
  for (int v = 0; v < 7; ++v) {
    const R dd = Wr[v] - Wl[v];
    xu[v] = dd - W6[v]; xl[v] = dd + W6[v];
  }
  const R irho = frcp(w0[0]);
  R Au[7], Al[7], A6[7], AA6[7];
  jac_mul(w0, bn, gam, irho, xu, Au);
  jac_mul(w0, bn, gam, irho, xl, Al);
  jac_mul(w0, bn, gam, irho, W6, A6);
  jac_mul(w0, bn, gam, irho, A6, AA6);
#pragma unroll
  for (int v = 0; v < 7; ++v) {
    wup[v] = Wr[v] - R(0.5) * sig * Au[v] - sig * sig * AA6[v] * R(1.0 / 3.0);
    wlo[v] = Wl[v] - R(0.5) * sig * Al[v] - sig * sig * AA6[v] * R(1.0 / 3.0);
  }
}

}  // namespace mhd

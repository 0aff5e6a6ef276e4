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

// MC-limited slope of cell w0 from its two one-sided differences.
// LIM_PRIM: componentwise.  LIM_CHAR: project on the left eigenvectors of (w0, bn), limit each characteristic
// amplitude, project back (wave order -f, -A, -s, entropy, +s, +A, +f).
template <class R, int LIMVAR>
__device__ __forceinline__ void limited_slope(const R (&w0)[7], R bn, R gam, const R (&dl)[7], const R (&dr)[7], R (&dw)[7]) {
  if (LIMVAR == kLimPrim) {
#pragma unroll
    for (int v = 0; v < 7; ++v) dw[v] = lim_mc(dl[v], dr[v]);
    return;
  }
  const R rho = w0[0], irho = frcp(rho);
  const R a2 = gam * w0[4] * irho, a = Num<R>::sqrt(a2), srho = Num<R>::sqrt(rho), isrho = frcp(srho);
  const WaveSet<R> w = wave_set(a2, rho, bn, w0[5], w0[6]);
  const R Qf = w.cf * w.af * w.S, Qs = w.cs * w.as * w.S, Af = a * w.af * srho, As = a * w.as * srho;
  const R nn = fdiv(R(0.5), a2);
#pragma unroll
  for (int v = 0; v < 7; ++v) dw[v] = R(0);
#pragma unroll
  for (int k = 0; k < 7; ++k) {
    const R s = (k < 3) ? R(1) : R(-1);
    R Lk[7], Rk[7];
    if (k == 0 || k == 6) {
      Lk[0] = R(0); Lk[1] = -s * nn * w.cf * w.af; Lk[2] = s * nn * Qs * w.b1; Lk[3] = s * nn * Qs * w.b2;
      Lk[4] = nn * w.af * irho; Lk[5] = nn * As * w.b1 * irho; Lk[6] = nn * As * w.b2 * irho;
      Rk[0] = rho * w.af; Rk[1] = -s * w.cf * w.af; Rk[2] = s * Qs * w.b1; Rk[3] = s * Qs * w.b2;
      Rk[4] = rho * a2 * w.af; Rk[5] = As * w.b1; Rk[6] = As * w.b2;
    } else if (k == 1 || k == 5) {
      Lk[0] = R(0); Lk[1] = R(0); Lk[2] = -s * R(0.5) * w.b2; Lk[3] = s * R(0.5) * w.b1; Lk[4] = R(0);
      Lk[5] = -R(0.5) * w.b2 * w.S * isrho; Lk[6] = R(0.5) * w.b1 * w.S * isrho;
      Rk[0] = R(0); Rk[1] = R(0); Rk[2] = -s * w.b2; Rk[3] = s * w.b1; Rk[4] = R(0);
      Rk[5] = -w.b2 * w.S * srho; Rk[6] = w.b1 * w.S * srho;
    } else if (k == 2 || k == 4) {
      Lk[0] = R(0); Lk[1] = -s * nn * w.cs * w.as; Lk[2] = -s * nn * Qf * w.b1; Lk[3] = -s * nn * Qf * w.b2;
      Lk[4] = nn * w.as * irho; Lk[5] = -nn * Af * w.b1 * irho; Lk[6] = -nn * Af * w.b2 * irho;
      Rk[0] = rho * w.as; Rk[1] = -s * w.cs * w.as; Rk[2] = -s * Qf * w.b1; Rk[3] = -s * Qf * w.b2;
      Rk[4] = rho * a2 * w.as; Rk[5] = -Af * w.b1; Rk[6] = -Af * w.b2;
    } else {
      Lk[0] = R(1); Lk[1] = R(0); Lk[2] = R(0); Lk[3] = R(0); Lk[4] = -R(2) * nn; Lk[5] = R(0); Lk[6] = R(0);
      Rk[0] = R(1); Rk[1] = R(0); Rk[2] = R(0); Rk[3] = R(0); Rk[4] = R(0); Rk[5] = R(0); Rk[6] = R(0);
    }
    R al = R(0), ar = R(0);
#pragma unroll
    for (int v = 0; v < 7; ++v) { al += Lk[v] * dl[v]; ar += Lk[v] * dr[v]; }
    const R am = lim_mc(al, ar);
#pragma unroll
    for (int v = 0; v < 7; ++v) dw[v] += am * Rk[v];
  }
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

// CTU step 1, PPM: parabola from the limited slopes of the cell and its two neighbours, monotonised
// (R4 i-iii), then traced with the parabola's first and second moments.
template <class R>
__device__ __forceinline__ void ppm_trace(const R (&wm)[7], const R (&w0)[7], const R (&wp)[7], const R (&sm)[7],
                                          const R (&s0)[7], const R (&sp)[7], R bn, R gam, R sig, R (&wlo)[7], R (&wup)[7]) {
  R Wl[7], Wr[7], xu[7], xl[7], W6[7];
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
    const R dd = r - l;
    W6[v] = R(6) * (w0[v] - R(0.5) * (l + r));
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

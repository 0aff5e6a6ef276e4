// mhd_physics.cuh -- per-face / per-cell device arithmetic of the patch-group MHD update (sm_100a).
//
// Register-resident formulations of: the ideal-MHD flux (Eq. 7), the gamma-law total energy
// (Eq. 5), the HLLE / HLLD / Roe Riemann solvers the paper names, the MC-limited
// PLM and PPM reconstructions in primitive or characteristic variables, and the CTU
// characteristic tracing in matrix form (R5).  The formulas the paper leaves to its references are
// the readings of DESIGN.md (R1-R18).  Everything is a template on Real (float / double); divisions are
// turned into shared reciprocals and all branches of a solver are evaluated and selected at the end so that
// a warp never diverges on the wave pattern.
//
// Generic 1-D state of direction n: W = (rho, vn, vt1, vt2, P, Bt1, Bt2) with the normal field Bn passed
// separately; conserved U = (rho, Mn, Mt1, Mt2, e, Bt1, Bt2).
#pragma once
#include <cuda_runtime.h>

namespace mhd {

enum : int { kHLLE = 0, kHLLD = 1, kROE = 2 };

// resident 256-thread blocks per SM requested from ptxas for the ALU-bound (Riemann / reconstruction) kernels
#ifndef MHD_MINB32
#define MHD_MINB32 4
#endif
#ifndef MHD_MINB64
#define MHD_MINB64 2
#endif
#ifndef MHD_MINB64_FLUX
#define MHD_MINB64_FLUX 3
#endif
// latency-bound update kernels: resident 256-thread blocks per SM requested from ptxas, from sweeps on B200
// (uncapped, ptxas hoists every load of the FP64 half-step kernel into 158 registers: 11 % of the warps resident)
#ifndef MHD_OCC_HALF64
#define MHD_OCC_HALF64 2
#define MHD_OCC_HALF32 6
#define MHD_OCC_FINAL64 4
#define MHD_OCC_FINAL32 6
#define MHD_OCC_EMF64 5
#define MHD_OCC_EMF32 1
#endif
template <class R> struct OccHalf  { static constexpr int minb = sizeof(R) == 8 ? MHD_OCC_HALF64 : MHD_OCC_HALF32; };
template <class R> struct OccFinal { static constexpr int minb = sizeof(R) == 8 ? MHD_OCC_FINAL64 : MHD_OCC_FINAL32; };
template <class R> struct OccEmf   { static constexpr int minb = sizeof(R) == 8 ? MHD_OCC_EMF64 : MHD_OCC_EMF32; };
template <class R> struct Occ { static constexpr int minb = sizeof(R) == 8 ? MHD_MINB64 : MHD_MINB32; };          // reconstruction
// Riemann kernels (measured: HLLD FP64 3 > 2 > 4 blocks.  Roe, since the solver forms no left eigenvectors any more (mhd_eigen.cuh): FP64
// 2 blocks of 128 registers with ~220 bytes of spills beat 1 block of 190 registers, VL+PLM+Roe 5.5e8 -> 6.9e8; 3 blocks: 4.6e8.
// FP32 3 blocks of 85 registers beat 2 of 96, CTU+PPM+Roe 9.4e8 -> 1.00e9; 4 blocks: 9.0e8)
#ifndef MHD_OCC_ROE64
#define MHD_OCC_ROE64 2
#endif
#ifndef MHD_OCC_ROE32
#define MHD_OCC_ROE32 3
#endif
template <class R, int SOLVER> struct OccFlux {
  static constexpr int minb = SOLVER == 2 ? (sizeof(R) == 8 ? MHD_OCC_ROE64 : MHD_OCC_ROE32) : (sizeof(R) == 8 ? MHD_MINB64_FLUX : MHD_MINB32);
};
enum : int { kPLM = 0, kPPM = 1, kPPMNoTrace = 2 };   // kPPMNoTrace: the PPM parabola at the half step of VL (NEXT-4)
enum : int { kLimPrim = 0, kLimChar = 1 };   // kernels take LIM = limvar + 2 * limiter (limiter: 0 MC, 1 minmod, 2 van Leer)

template <class R> struct Num;
// -DMHD_IEEE32: control build (libmhd_ieee32.so, tests/fp32_controls.py): every FP32 division / square root IEEE-rounded
// instead of the SFU approximations, to separate their error from the rounding inherent to single precision
template <> struct Num<float> {
#ifdef MHD_IEEE32
  static __device__ __forceinline__ float sqrt(float x) { return __fsqrt_rn(x); }
#else
  static __device__ __forceinline__ float sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
#endif
  static __device__ __forceinline__ float abs(float x) { return fabsf(x); }
  static __device__ __forceinline__ float min(float a, float b) { return fminf(a, b); }
  static __device__ __forceinline__ float max(float a, float b) { return fmaxf(a, b); }
};
template <> struct Num<double> {
  static __device__ __forceinline__ double sqrt(double x) { return ::sqrt(x); }
  static __device__ __forceinline__ double abs(double x) { return fabs(x); }
  static __device__ __forceinline__ double min(double a, double b) { return fmin(a, b); }
  static __device__ __forceinline__ double max(double a, double b) { return fmax(a, b); }
};

template <class R> __device__ __forceinline__ R sqr(R x) { return x * x; }

// Divisions and square roots.  FP64: IEEE.  FP32: the SFU approximations (rcp.approx / sqrt.approx, <= 1-2 ulp), one
// or two instructions instead of the ~10-instruction IEEE sequences with a slow-path call; the FP32 parity bound
// (1e-4 after 10 steps) is four orders of magnitude above their error.
__device__ __forceinline__ double frcp(double x) { return 1.0 / x; }
__device__ __forceinline__ double fdiv(double a, double b) { return a / b; }
#ifdef MHD_IEEE32
__device__ __forceinline__ float frcp(float x) { return __frcp_rn(x); }
__device__ __forceinline__ float fdiv(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ float frsqrt(float x) { return __frcp_rn(__fsqrt_rn(x)); }
#else
__device__ __forceinline__ float frcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float fdiv(float a, float b) { return a * frcp(b); }
__device__ __forceinline__ float frsqrt(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
#endif
__device__ __forceinline__ double frsqrt(double x) { return rsqrt(x); }
// sqrt(x) and 1/sqrt(x): FP64 from one rsqrt (sqrt = x * rsqrt), FP32 from the two SFU approximations
__device__ __forceinline__ void sqrt_and_inverse(double x, double& s, double& is) { is = rsqrt(x); s = x * is; }
__device__ __forceinline__ void sqrt_and_inverse(float x, float& s, float& is) {
  s = Num<float>::sqrt(x);
  is = frcp(s);
}
// several reciprocals at once.  FP32: one SFU op each.  FP64: ONE division for the product and a few multiplications
// (a double division is ~10 DFMA-pipe instructions plus a slow-path call); all arguments must be finite and non-zero.
__device__ __forceinline__ void frcp2(float a, float b, float& ia, float& ib) { ia = frcp(a); ib = frcp(b); }
__device__ __forceinline__ void frcp2(double a, double b, double& ia, double& ib) {
  const double inv = 1.0 / (a * b);
  ia = b * inv; ib = a * inv;
}
__device__ __forceinline__ void frcp4(float a, float b, float c, float d, float& ia, float& ib, float& ic, float& id) {
  ia = frcp(a); ib = frcp(b); ic = frcp(c); id = frcp(d);
}
__device__ __forceinline__ void frcp4(double a, double b, double c, double d, double& ia, double& ib, double& ic, double& id) {
  const double ab = a * b, cd = c * d, inv = 1.0 / (ab * cd);
  const double iab = cd * inv, icd = ab * inv;
  ia = b * iab; ib = a * iab; ic = d * icd; id = c * icd;
}

// monotonised-central limiter (R5)
// FP32: the same value in 7 instructions instead of 13: min(|a|, |b|) with the sign sign(a) xor sign(b) in ONE instruction
// (min.xorsign.abs), so opposite signs give a value <= 0 that the clamp at zero removes (a zero operand gives 0 by itself);
// min(|s| / 2, 2 q) = 2 min(|s| / 4, q) exactly; the sign of the result is that of a (= that of a + b where the signs agree)
__device__ __forceinline__ float lim_mc(float a, float b) {
  float q;
  asm("min.xorsign.abs.f32 %0, %1, %2;" : "=f"(q) : "f"(a), "f"(b));
  const float r = fmaxf(fminf(q, 0.25f * fabsf(a + b)), 0.0f);
  return copysignf(r + r, a);
}
template <class R> __device__ __forceinline__ R lim_mc(R a, R b) {
  R s = a + b;
  R m = Num<R>::min(R(0.5) * Num<R>::abs(s), R(2) * Num<R>::min(Num<R>::abs(a), Num<R>::abs(b)));
  m = (s > R(0)) ? m : -m;
  return (a * b <= R(0)) ? R(0) : m;
}
// minmod of the CTU multidimensional MHD source terms (R6)
template <class R> __device__ __forceinline__ R lim_minmod(R a, R b) {
  R m = Num<R>::min(Num<R>::abs(a), Num<R>::abs(b));
  m = (a > R(0)) ? m : -m;
  return (a * b <= R(0)) ? R(0) : m;
}
// van Leer (harmonic-mean) limiter, NEXT-4 variant
template <class R> __device__ __forceinline__ R lim_vanleer(R a, R b) {
  const R ab = a * b;
  return (ab <= R(0)) ? R(0) : fdiv(R(2) * ab, a + b);
}
// slope limiter selected at compile time: 0 MC (R5), 1 minmod, 2 van Leer
template <class R, int LIMITER> __device__ __forceinline__ R lim_sel(R a, R b) {
  return LIMITER == 1 ? lim_minmod(a, b) : (LIMITER == 2 ? lim_vanleer(a, b) : lim_mc(a, b));
}

// ---- one side of a face: everything the solvers need from a primitive state -------------------------------
template <class R> struct Side {
  R U[7];   // conserved (Eq. 5)
  R F[7];   // physical flux (Eq. 7)
  R pT;     // P + B^2/2
  R vB;     // v.B
  R cf;     // fast speed along n
  R g;      // cf^2 - ca^2 >= 0, evaluated without cancellation (HLLD star-state denominators)
};

template <class R>
__device__ __forceinline__ void side_setup(const R (&w)[7], R bn, R bn2, R gm1inv, R gam, Side<R>& s) {
  R bt2 = w[5] * w[5] + w[6] * w[6];
  R pmag = R(0.5) * (bn2 + bt2);
  R v2 = w[1] * w[1] + w[2] * w[2] + w[3] * w[3];
  s.pT = w[4] + pmag;
  s.vB = bn * w[1] + w[5] * w[2] + w[6] * w[3];
  R mn = w[0] * w[1];
  s.U[0] = w[0]; s.U[1] = mn; s.U[2] = w[0] * w[2]; s.U[3] = w[0] * w[3];
  s.U[4] = w[4] * gm1inv + R(0.5) * w[0] * v2 + pmag;
  s.U[5] = w[5]; s.U[6] = w[6];
  s.F[0] = mn;
  s.F[1] = mn * w[1] + s.pT - bn2;
  s.F[2] = mn * w[2] - bn * w[5];
  s.F[3] = mn * w[3] - bn * w[6];
  s.F[4] = (s.U[4] + s.pT) * w[1] - bn * s.vB;
  s.F[5] = w[5] * w[1] - bn * w[2];
  s.F[6] = w[6] * w[1] - bn * w[3];
  // c_f^2 = 1/2 [ (a^2+ca^2+ct^2) + sqrt( (ca^2+ct^2-a^2)^2 + 4 a^2 ct^2 ) ]   (R1, R18)
  R ir = frcp(w[0]);
  R a2 = gam * w[4] * ir, ca2 = bn2 * ir, ct2 = bt2 * ir;
  R sum = a2 + ca2 + ct2, dif = ca2 + ct2 - a2;
  R root = Num<R>::sqrt(dif * dif + R(4) * a2 * ct2);
  s.cf = Num<R>::sqrt(R(0.5) * (sum + root));
  // cf^2 - ca^2 = 1/2 (x + root), x = a^2 + ct^2 - ca^2 (root^2 = x^2 + 4 ca^2 ct^2); rationalised where x < 0
  R x = a2 + ct2 - ca2;
  s.g = (x >= R(0)) ? R(0.5) * (x + root) : fdiv(R(2) * ca2 * ct2, root - x);
}

template <class R>
__device__ __forceinline__ R fast_speed(R rho, R P, R bn2, R bt2, R gam) {
  R ir = frcp(rho);
  R a2 = gam * P * ir, ca2 = bn2 * ir, ct2 = bt2 * ir;
  R sum = a2 + ca2 + ct2, dif = ca2 + ct2 - a2;
  return Num<R>::sqrt(R(0.5) * (sum + Num<R>::sqrt(dif * dif + R(4) * a2 * ct2)));
}

// ---- HLLD (Miyoshi & Kusano form; R7/R12) ------------------------------------------------
// Evaluation notes (all algebraic identities of the reading): the scalars of both sides first, the
// reciprocals of independent denominators batched (frcp2 / frcp4), sqrt(rho*) together with its reciprocal from one
// rsqrt, and the flux / conserved vectors only of the side the face turns out to lie on.
template <class R>
__device__ __forceinline__ void riemann_hlld(const R (&wl)[7], const R (&wr)[7], R bn, R gam, R gm1inv, R (&F)[7]) {
  const R bn2 = bn * bn;
  R irL, irR;
  frcp2(wl[0], wr[0], irL, irR);
  R pT[2], pmag[2], cf[2], root[2], a2[2], ca2[2], ct2[2];
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    const R (&w)[7] = a ? wr : wl;
    const R ir = a ? irR : irL;
    const R bt2 = w[5] * w[5] + w[6] * w[6];
    pmag[a] = R(0.5) * (bn2 + bt2);
    pT[a] = w[4] + pmag[a];
    // c_f^2 = 1/2 [ (a^2+ca^2+ct^2) + sqrt( (ca^2+ct^2-a^2)^2 + 4 a^2 ct^2 ) ]   (R1, R18)
    a2[a] = gam * w[4] * ir; ca2[a] = bn2 * ir; ct2[a] = bt2 * ir;
    const R sum = a2[a] + ca2[a] + ct2[a], dif = ca2[a] + ct2[a] - a2[a];
    root[a] = Num<R>::sqrt(dif * dif + R(4) * a2[a] * ct2[a]);
    cf[a] = Num<R>::sqrt(R(0.5) * (sum + root[a]));
  }
  const R uL = wl[1], uR = wr[1];
  const bool lmax = cf[0] >= cf[1];
  const R cmax = lmax ? cf[0] : cf[1];
  // cf^2 - ca^2 of the faster side = 1/2 (x + root), x = a^2 + ct^2 - ca^2 (root^2 = x^2 + 4 ca^2 ct^2); rationalised where x < 0
  R gm;
  {
    const R a2m = lmax ? a2[0] : a2[1], ca2m = lmax ? ca2[0] : ca2[1], ct2m = lmax ? ct2[0] : ct2[1], rootm = lmax ? root[0] : root[1];
    const R xx = a2m + ct2m - ca2m;
    const R gnum = R(2) * ca2m * ct2m;          // numerator of the rationalised form
    const R inv = frcp(xx < R(0) ? rootm - xx : R(1));
    gm = xx < R(0) ? gnum * inv : R(0.5) * (xx + rootm);
  }
  const R SL = Num<R>::min(uL, uR) - cmax, SR = Num<R>::max(uL, uR) + cmax;
  const R sL = (SL - uL) * wl[0], sR = (SR - uR) * wr[0];
  const R idn = frcp(sR - sL);
  // contact speed through the differences u_L - u_R and pT_R - pT_L taken directly from the inputs, so that slow
  // flows in a strong field keep their significant digits (the textbook quotient subtracts O(pT) terms)
  const R du = uL - uR;
  const R dp = (wr[4] - wl[4]) + R(0.5) * ((wr[5] - wl[5]) * (wr[5] + wl[5]) + (wr[6] - wl[6]) * (wr[6] + wl[6]));
  const R uLmSM = (sR * du + dp) * idn, uRmSM = (sL * du + dp) * idn;     // u_alpha - S_M
  const R SM = uL - uLmSM;
  const R pTs = (sR * pT[0] - sL * pT[1] + sL * sR * (uR - uL)) * idn;
  const R tiny = R(1e-12) * pTs;
  // the side of the contact the face lies on: S_L <= S*_L <= S_M in floating point too (S*_L = S_M - |Bn| / sqrt(rho*_L))
  const bool left = (SL >= R(0)) || (SM >= R(0));
  // rho (S-u)^2 - Bn^2 of each side without cancellation: (S-u)^2 = (cmax + delta)^2, cmax^2 = ca_m^2 + g_m
  const R delta = Num<R>::max(du, R(0));
  const R rhom = lmax ? wl[0] : wr[0], irm = lmax ? irL : irR;
  const R grow = gm + delta * (R(2) * cmax + delta);
  const R bfac = bn2 * irm;

  // star states of both sides (the double-star state needs both); total energy and v.B only of the side the face lies on
  const R dSML = (SL - uL) + uLmSM, dSMR = (SR - uR) + uRmSM;               // S_alpha - S_M
  const R NbL = wl[0] * grow + bfac * (wl[0] - rhom), NbR = wr[0] * grow + bfac * (wr[0] - rhom);   // rho (S-u)^2 - Bn^2
  const R DL = NbL + sL * uLmSM, DR = NbR + sR * uRmSM;                     // rho (S-u)(S-S_M) - Bn^2
  const bool degL = Num<R>::abs(DL) < tiny, degR = Num<R>::abs(DR) < tiny;
  R idSML, idSMR, iDL, iDR;
  frcp4(dSML, dSMR, degL ? R(1) : DL, degR ? R(1) : DR, idSML, idSMR, iDL, iDR);
  R rs[2], v1s[2], v2s[2], b1s[2], b2s[2], sq[2], isq[2];
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    const R (&w)[7] = a ? wr : wl;
    const R sa = a ? sR : sL, umSM = a ? uRmSM : uLmSM;
    const R idSM = a ? idSMR : idSML, iD = a ? iDR : iDL, Nb = a ? NbR : NbL;
    const bool degen = a ? degR : degL;
    rs[a] = sa * idSM;
    const R fv = degen ? R(0) : -bn * umSM * iD;
    const R fb = degen ? R(1) : Nb * iD;
    v1s[a] = w[2] - w[5] * fv; v2s[a] = w[3] - w[6] * fv;
    b1s[a] = w[5] * fb; b2s[a] = w[6] * fb;
    sqrt_and_inverse(rs[a], sq[a], isq[a]);
  }
  const R abn = Num<R>::abs(bn);
  // the chosen side: input state, conserved state and physical flux (Eq. 5, 7), star state
  R wa[7];
#pragma unroll
  for (int c = 0; c < 7; ++c) wa[c] = left ? wl[c] : wr[c];
  const R pTa = left ? pT[0] : pT[1], pma = left ? pmag[0] : pmag[1];
  const R Sa = left ? SL : SR, idSMa = left ? idSML : idSMR, isqa = left ? isq[0] : isq[1];
  const R r_s = left ? rs[0] : rs[1], sq_a = left ? sq[0] : sq[1];
  const R v1a = left ? v1s[0] : v1s[1], v2a = left ? v2s[0] : v2s[1];
  const R b1a = left ? b1s[0] : b1s[1], b2a = left ? b2s[0] : b2s[1];
  const R vBa0 = bn * wa[1] + wa[5] * wa[2] + wa[6] * wa[3];
  const R ena = wa[4] * gm1inv + R(0.5) * wa[0] * (wa[1] * wa[1] + wa[2] * wa[2] + wa[3] * wa[3]) + pma;
  const R vBa = bn * SM + b1a * v1a + b2a * v2a;
  const R esa = ((Sa - wa[1]) * ena - pTa * wa[1] + pTs * SM + bn * (vBa0 - vBa)) * idSMa;
  const R Ssa = left ? SM - abn * isqa : SM + abn * isqa;
  // region of that side: plain F_L / F_R, single star, double star
  const bool outer = left ? (SL >= R(0)) : !(SR >= R(0));
  const bool star = left ? (Ssa >= R(0)) : !(Ssa >= R(0));
  const R Us[7] = { r_s, r_s * SM, r_s * v1a, r_s * v2a, esa, b1a, b2a };
  // double-star state (transverse components and energy; U** = U* where Bn vanishes: no rotational waves)
  R Uss[7];
  {
    const R sg = bn > R(0) ? R(1) : R(-1);
    const R ir = frcp(sq[0] + sq[1]);
    const R v1 = (sq[0] * v1s[0] + sq[1] * v1s[1] + (b1s[1] - b1s[0]) * sg) * ir;
    const R v2 = (sq[0] * v2s[0] + sq[1] * v2s[1] + (b2s[1] - b2s[0]) * sg) * ir;
    const R b1 = (sq[0] * b1s[1] + sq[1] * b1s[0] + sq[0] * sq[1] * (v1s[1] - v1s[0]) * sg) * ir;
    const R b2 = (sq[0] * b2s[1] + sq[1] * b2s[0] + sq[0] * sq[1] * (v2s[1] - v2s[0]) * sg) * ir;
    const R vBss = bn * SM + b1 * v1 + b2 * v2;
    const R pm = left ? R(-1) : R(1);
    Uss[0] = Us[0]; Uss[1] = Us[1]; Uss[2] = r_s * v1; Uss[3] = r_s * v2;
    Uss[4] = esa + pm * sq_a * (vBa - vBss) * sg;
    Uss[5] = b1; Uss[6] = b2;
  }
  const R mn = wa[0] * wa[1];
  const R Ua[7] = { wa[0], mn, wa[0] * wa[2], wa[0] * wa[3], ena, wa[5], wa[6] };
  const R Fa[7] = { mn, mn * wa[1] + pTa - bn2, mn * wa[2] - bn * wa[5], mn * wa[3] - bn * wa[6],
                    (ena + pTa) * wa[1] - bn * vBa0, wa[5] * wa[1] - bn * wa[2], wa[6] * wa[1] - bn * wa[3] };
  // F* = F_a + S_a (U* - U_a);  F** = F_a + S* U** - (S* - S_a) U* - S_a U_a = F* + S* (U** - U*): one expression for both regions with
  // S* := 0 in the single-star region and where Bn vanishes (rho and the normal momentum are the same in U* and U**)
  const R Sse = (star || R(0.5) * bn2 < tiny) ? R(0) : Ssa;
#pragma unroll
  for (int c = 0; c < 7; ++c) {
    R f = Fa[c] + Sa * (Us[c] - Ua[c]);
    if (c >= 2) f += Sse * (Uss[c] - Us[c]);
    F[c] = outer ? Fa[c] : f;
  }
}

}  // namespace mhd

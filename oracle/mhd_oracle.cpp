// =====================================================================================
// mhd_oracle.cpp -- TEST INFRASTRUCTURE ONLY.  Plain, slow, scalar CPU restatement of the
// per-patch-group unsplit MHD update of GAMER-MHD (Zhang, Schive & Chiueh 2018), written
// from the paper text step by step.  It shares no code with the CUDA path
// (paper_1804_03479_b200/csrc) and must only be used by tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs.
//
// What it follows:
//   * equations: PAPER.md:40-74 (Eq. 1-9), Eq. 5 total energy, Eq. 7-9 fluxes
//   * staggering + CT: PAPER.md:82-168 (Eq. 10, 13, 16, Fig. 1)
//   * step order: PAPER.md:174-183 (CTU, 8 steps), PAPER.md:191-197 (VL, 7 steps)
//   * where the paper is silent (formulas of PLM/PPM, HLLE/HLLD/Roe, edge EMF, source
//     terms, floors) it follows the readings listed in DESIGN.md ("Readings", R1-R18).
// Every array is a whole-tile temporary with one uniform stride S=T+1; loops run over the
// maximal index range on which the inputs of a stage exist; temporaries start as NaN so a
// use of an uncomputed value poisons the output.  No tiling, fusion or reordering.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): eigen identities, Roe property, HLLD
// consistency, uniform state, conservation, div B, linear-wave convergence, ABC
// equilibrium convergence, field loop, symmetry, decomposition, Sod tube.  The absolute
// values of a nonlinear step have no external reference: "parity unpinned" beyond those.
//
// Build: g++ -O2 -fno-fast-math -ffp-contract=off -fopenmp -shared -fPIC
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstring>
#include <limits>
#include <vector>

extern "C" {
typedef struct {
  int ps2;      // N, interior cells per side
  int nghost;   // g
  double gamma;
  int scheme;   // 0 VL, 1 CTU
  int recon;    // 0 PLM, 1 PPM
  int riemann;  // 0 HLLE, 1 HLLD, 2 ROE
  int limvar;   // 0 primitive, 1 characteristic
  double min_dens, min_pres;
  double emf_tie;  // reading R10a: width of the linear blend of the CT upwind switch, in units of (mean cell density) * dh/dt
  int limiter;     // NEXT-4 variants: 0 MC (reading R5, the default), 1 minmod, 2 van Leer
  int minimal_ranges;  // 0: every stage on the maximal index range on which its inputs exist (the default); 1: every stage only
                       // where the final update of the N^3 interior cells needs it.  Same arithmetic per
                       // cell / face / edge; the outputs are bitwise the same (pinned), only the operation count differs
  int hcorr;           // NEXT-4 variant (reading R19): H-correction of the Roe solver (multidimensional entropy fix);
                       // needs riemann = Roe and one ghost cell more than the scheme alone; evaluated on the maximal ranges
} mhdref_config;
// measurement hook (oracle/count_ops.cpp): called with the number of the step that just finished inside one group's update
void (*mhdref_stage_hook)(int) = nullptr;
}

namespace {

typedef std::vector<double> Arr;
const double NaN = std::numeric_limits<double>::quiet_NaN();

struct Stats { unsigned long long fd = 0, fp = 0, fb = 0; };

inline double sq(double x) { return x * x; }

// MC limiter, reading R5: MC(a,b) = 0 if ab<=0 else sign(a+b) min(|a+b|/2, 2|a|, 2|b|)
inline double mc(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  double s = a + b;
  double m = std::min(0.5 * std::fabs(s), std::min(2.0 * std::fabs(a), 2.0 * std::fabs(b)));
  return s > 0.0 ? m : -m;
}
// NEXT-4 slope-limiter variants (PAPER.md:176 names none): the two other classical symmetric TVD limiters
// van Leer (harmonic mean): 2ab/(a+b) if ab > 0, else 0
inline double vanleer(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  return 2.0 * a * b / (a + b);
}
// minmod used by the CTU MHD source terms, reading R6 (and as the minmod slope limiter, limiter = 1)
inline double mm(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  double m = std::min(std::fabs(a), std::fabs(b));
  return a > 0.0 ? m : -m;
}

// ---------------------------------------------------------------------------------
// Generic 1-D state for direction n: W = (rho, vn, vt1, vt2, P, Bt1, Bt2), parameter Bn
// U = (rho, rho vn, rho vt1, rho vt2, e, Bt1, Bt2); Eq. 5
// ---------------------------------------------------------------------------------
void prim2cons(const double W[7], double Bn, double gam, double U[7]) {
  U[0] = W[0];
  U[1] = W[0] * W[1];
  U[2] = W[0] * W[2];
  U[3] = W[0] * W[3];
  U[4] = W[4] / (gam - 1.0) + 0.5 * W[0] * (sq(W[1]) + sq(W[2]) + sq(W[3])) + 0.5 * (sq(Bn) + sq(W[5]) + sq(W[6]));
  U[5] = W[5];
  U[6] = W[6];
}
// Eq. 7 with (x,y,z) -> (n,t1,t2); Eq. 8, 9 are its cyclic permutations
void physflux(const double W[7], double Bn, const double U[7], double F[7]) {
  double pT = W[4] + 0.5 * (sq(Bn) + sq(W[5]) + sq(W[6]));
  double vB = Bn * W[1] + W[5] * W[2] + W[6] * W[3];
  F[0] = U[1];
  F[1] = U[1] * W[1] + pT - Bn * Bn;
  F[2] = U[1] * W[2] - Bn * W[5];
  F[3] = U[1] * W[3] - Bn * W[6];
  F[4] = (U[4] + pT) * W[1] - Bn * vB;
  F[5] = W[5] * W[1] - Bn * W[2];
  F[6] = W[6] * W[1] - Bn * W[3];
}
// fast magnetosonic speed along n (reading R1/C1)
double fastspeed(const double W[7], double Bn, double gam) {
  // c_f^2 = 1/2[(a^2+b^2) + sqrt((a^2+b^2)^2 - 4 a^2 ca^2)]; the discriminant is evaluated in the algebraically
  // identical cancellation-free form (ca^2 + ct^2 - a^2)^2 + 4 a^2 ct^2 (reading R18)
  double a2 = gam * W[4] / W[0];
  double ca2 = sq(Bn) / W[0], ct2 = (sq(W[5]) + sq(W[6])) / W[0];
  double s = a2 + ca2 + ct2, td = ca2 + ct2 - a2;
  return std::sqrt(0.5 * (s + std::sqrt(td * td + 4.0 * a2 * ct2)));
}

// ---------------------------------------------------------------------------------
// A1: primitive eigen-system of direction n (used by characteristic limiting; the
// matrix A is used by the CTU tracing).  Order of waves: -f, -A, -s, entropy, +s, +A, +f
// ---------------------------------------------------------------------------------
void primA(const double W[7], double Bn, double gam, double A[7][7]) {
  for (int r = 0; r < 7; ++r) for (int c = 0; c < 7; ++c) A[r][c] = 0.0;
  double rho = W[0], vn = W[1], P = W[4], B1 = W[5], B2 = W[6];
  for (int r = 0; r < 7; ++r) A[r][r] = vn;
  A[0][1] = rho;
  A[1][4] = 1.0 / rho; A[1][5] = B1 / rho; A[1][6] = B2 / rho;
  A[2][5] = -Bn / rho;
  A[3][6] = -Bn / rho;
  A[4][1] = gam * P;
  A[5][1] = B1; A[5][2] = -Bn;
  A[6][1] = B2; A[6][3] = -Bn;
}
// shared pieces of A1 / A3: given a2 (sound speed^2), rho, Bn, Bt -> cf, cs, alphas, betas
struct WaveSet { double cf, cs, ca, af, as, b1, b2, S; };
WaveSet waveset(double a2, double rho, double Bn, double B1, double B2) {
  WaveSet w;
  double ca2 = Bn * Bn / rho, ct2 = (B1 * B1 + B2 * B2) / rho;
  double ts = a2 + ca2 + ct2, td = ca2 + ct2 - a2;
  double cf2 = 0.5 * (ts + std::sqrt(td * td + 4.0 * a2 * ct2));   // same discriminant as in fastspeed()
  double cs2 = (cf2 > 0.0) ? a2 * ca2 / cf2 : 0.0;
  if (cs2 < 0.0) cs2 = 0.0;
  w.cf = std::sqrt(cf2); w.cs = std::sqrt(cs2); w.ca = std::sqrt(ca2);
  double den = cf2 - cs2;
  if (den <= 0.0) { w.af = 1.0; w.as = 0.0; }
  else {
    double af2 = (a2 - cs2) / den, as2 = (cf2 - a2) / den;
    af2 = std::min(1.0, std::max(0.0, af2)); as2 = std::min(1.0, std::max(0.0, as2));
    w.af = std::sqrt(af2); w.as = std::sqrt(as2);
  }
  double bt = std::sqrt(B1 * B1 + B2 * B2);
  if (bt == 0.0) { w.b1 = 1.0; w.b2 = 0.0; } else { w.b1 = B1 / bt; w.b2 = B2 / bt; }
  w.S = (Bn >= 0.0) ? 1.0 : -1.0;
  return w;
}
void eig_prim(const double W[7], double Bn, double gam, double lam[7], double R[7][7], double L[7][7]) {
  double rho = W[0], vn = W[1], P = W[4];
  double a2 = gam * P / rho, a = std::sqrt(a2), sr = std::sqrt(rho);
  WaveSet w = waveset(a2, rho, Bn, W[5], W[6]);
  double Qf = w.cf * w.af * w.S, Qs = w.cs * w.as * w.S, Af = a * w.af * sr, As = a * w.as * sr;
  lam[0] = vn - w.cf; lam[1] = vn - w.ca; lam[2] = vn - w.cs; lam[3] = vn;
  lam[4] = vn + w.cs; lam[5] = vn + w.ca; lam[6] = vn + w.cf;
  double n = 0.5 / a2;
  // R[k][:] = k-th right eigenvector (a column of the usual matrix), L[k][:] = k-th left eigenvector
  for (int sgn = 0; sgn < 2; ++sgn) {
    double s = sgn == 0 ? 1.0 : -1.0;  // s=+1 : the "-" wave (upper signs), s=-1 : the "+" wave
    int kf = sgn == 0 ? 0 : 6, ka = sgn == 0 ? 1 : 5, ks = sgn == 0 ? 2 : 4;
    double Rf[7] = { rho * w.af, -s * w.cf * w.af, s * Qs * w.b1, s * Qs * w.b2, rho * a2 * w.af, As * w.b1, As * w.b2 };
    double Ra[7] = { 0, 0, -s * w.b2, s * w.b1, 0, -w.b2 * w.S * sr, w.b1 * w.S * sr };
    double Rs[7] = { rho * w.as, -s * w.cs * w.as, -s * Qf * w.b1, -s * Qf * w.b2, rho * a2 * w.as, -Af * w.b1, -Af * w.b2 };
    double Lf[7] = { 0, -s * n * w.cf * w.af, s * n * Qs * w.b1, s * n * Qs * w.b2, n * w.af / rho, n * As * w.b1 / rho, n * As * w.b2 / rho };
    double La[7] = { 0, 0, -s * 0.5 * w.b2, s * 0.5 * w.b1, 0, -0.5 * w.b2 * w.S / sr, 0.5 * w.b1 * w.S / sr };
    double Ls[7] = { 0, -s * n * w.cs * w.as, -s * n * Qf * w.b1, -s * n * Qf * w.b2, n * w.as / rho, -n * Af * w.b1 / rho, -n * Af * w.b2 / rho };
    for (int c = 0; c < 7; ++c) { R[kf][c] = Rf[c]; R[ka][c] = Ra[c]; R[ks][c] = Rs[c]; L[kf][c] = Lf[c]; L[ka][c] = La[c]; L[ks][c] = Ls[c]; }
  }
  double Re[7] = { 1, 0, 0, 0, 0, 0, 0 }, Le[7] = { 1, 0, 0, 0, -1.0 / a2, 0, 0 };
  for (int c = 0; c < 7; ++c) { R[3][c] = Re[c]; L[3][c] = Le[c]; }
}

// ---------------------------------------------------------------------------------
// A3: Roe average (enthalpy form) and conserved eigen-system
// ---------------------------------------------------------------------------------
struct RoeAvg { double rho, vn, v1, v2, H, B1, B2, X, a2; };
RoeAvg roe_average(const double WL[7], const double WR[7], double Bn, double gam) {
  RoeAvg r;
  double wl = std::sqrt(WL[0]), wr = std::sqrt(WR[0]), iw = 1.0 / (wl + wr);
  double UL[7], UR[7];
  prim2cons(WL, Bn, gam, UL); prim2cons(WR, Bn, gam, UR);
  double pTL = WL[4] + 0.5 * (sq(Bn) + sq(WL[5]) + sq(WL[6]));
  double pTR = WR[4] + 0.5 * (sq(Bn) + sq(WR[5]) + sq(WR[6]));
  double HL = (UL[4] + pTL) / WL[0], HR = (UR[4] + pTR) / WR[0];
  r.rho = wl * wr;
  r.vn = (wl * WL[1] + wr * WR[1]) * iw;
  r.v1 = (wl * WL[2] + wr * WR[2]) * iw;
  r.v2 = (wl * WL[3] + wr * WR[3]) * iw;
  r.H = (wl * HL + wr * HR) * iw;
  r.B1 = (wr * WL[5] + wl * WR[5]) * iw;   // weights swapped
  r.B2 = (wr * WL[6] + wl * WR[6]) * iw;
  r.X = (sq(WL[5] - WR[5]) + sq(WL[6] - WR[6])) * 0.5 * iw * iw;
  double ca2 = Bn * Bn / r.rho, ct2 = (sq(r.B1) + sq(r.B2)) / r.rho;
  double Hp = r.H - ca2 - ct2;
  double v2 = sq(r.vn) + sq(r.v1) + sq(r.v2);
  r.a2 = (gam - 1.0) * (Hp - 0.5 * v2) - (gam - 2.0) * r.X;
  return r;
}
void eig_cons(const RoeAvg& r, double Bn, double gam, double lam[7], double R[7][7], double L[7][7]) {
  double rho = r.rho, vn = r.vn, v1 = r.v1, v2_ = r.v2, a2 = r.a2, a = std::sqrt(a2), sr = std::sqrt(rho);
  WaveSet w = waveset(a2, rho, Bn, r.B1, r.B2);
  double ca2 = Bn * Bn / rho, ct2 = (sq(r.B1) + sq(r.B2)) / rho;
  double Hp = r.H - ca2 - ct2;
  double vsq = sq(vn) + sq(v1) + sq(v2_);
  double Qf = w.cf * w.af * w.S, Qs = w.cs * w.as * w.S, Afp = a * w.af / sr, Asp = a * w.as / sr;
  double vb = v1 * w.b1 + v2_ * w.b2, bt = std::sqrt(sq(r.B1) + sq(r.B2));
  double xt = (gam - 2.0) * r.X / (gam - 1.0);
  lam[0] = vn - w.cf; lam[1] = vn - w.ca; lam[2] = vn - w.cs; lam[3] = vn;
  lam[4] = vn + w.cs; lam[5] = vn + w.ca; lam[6] = vn + w.cf;
  double n = 0.5 / a2, g = (gam - 1.0) * n;
  for (int sgn = 0; sgn < 2; ++sgn) {
    double s = sgn == 0 ? 1.0 : -1.0;  // s=+1: "-" wave (upper signs)
    int kf = sgn == 0 ? 0 : 6, ka = sgn == 0 ? 1 : 5, ks = sgn == 0 ? 2 : 4;
    double Rf[7] = { w.af, w.af * (vn - s * w.cf), w.af * v1 + s * Qs * w.b1, w.af * v2_ + s * Qs * w.b2,
                     w.af * (Hp - s * vn * w.cf) + s * Qs * vb + Asp * bt, Asp * w.b1, Asp * w.b2 };
    double Ra[7] = { 0, 0, -s * w.b2, s * w.b1, -s * (v1 * w.b2 - v2_ * w.b1), -w.b2 * w.S / sr, w.b1 * w.S / sr };
    double Rs[7] = { w.as, w.as * (vn - s * w.cs), w.as * v1 - s * Qf * w.b1, w.as * v2_ - s * Qf * w.b2,
                     w.as * (Hp - s * vn * w.cs) - s * Qf * vb - Afp * bt, -Afp * w.b1, -Afp * w.b2 };
    double Lf[7] = { g * w.af * (vsq - Hp) + n * w.af * w.cf * (w.cf + s * vn) - s * n * Qs * vb - n * Asp * bt,
                     -g * w.af * vn - s * n * w.af * w.cf, -g * w.af * v1 + s * n * Qs * w.b1, -g * w.af * v2_ + s * n * Qs * w.b2,
                     g * w.af, n * Asp * rho * w.b1 - g * w.af * r.B1, n * Asp * rho * w.b2 - g * w.af * r.B2 };
    double La[7] = { s * 0.5 * (v1 * w.b2 - v2_ * w.b1), 0, -s * 0.5 * w.b2, s * 0.5 * w.b1, 0, -0.5 * sr * w.b2 * w.S, 0.5 * sr * w.b1 * w.S };
    double Ls[7] = { g * w.as * (vsq - Hp) + n * w.as * w.cs * (w.cs + s * vn) + s * n * Qf * vb + n * Afp * bt,
                     -g * w.as * vn - s * n * w.as * w.cs, -g * w.as * v1 - s * n * Qf * w.b1, -g * w.as * v2_ - s * n * Qf * w.b2,
                     g * w.as, -n * Afp * rho * w.b1 - g * w.as * r.B1, -n * Afp * rho * w.b2 - g * w.as * r.B2 };
    for (int c = 0; c < 7; ++c) { R[kf][c] = Rf[c]; R[ka][c] = Ra[c]; R[ks][c] = Rs[c]; L[kf][c] = Lf[c]; L[ka][c] = La[c]; L[ks][c] = Ls[c]; }
  }
  double Re[7] = { 1, vn, v1, v2_, 0.5 * vsq + xt, 0, 0 };
  double Le[7] = { 1.0 - 2.0 * g * (0.5 * vsq - xt), 2.0 * g * vn, 2.0 * g * v1, 2.0 * g * v2_, -2.0 * g, 2.0 * g * r.B1, 2.0 * g * r.B2 };
  for (int c = 0; c < 7; ++c) { R[3][c] = Re[c]; L[3][c] = Le[c]; }
}

// ---------------------------------------------------------------------------------
// Riemann solvers (PAPER.md:177 names them; formulas: readings R7/A2-A4)
// ---------------------------------------------------------------------------------
// A4 HLLE with Einfeldt speeds; the Roe-average term is dropped when a~^2 <= 0
void hlle(const double WL[7], const double WR[7], double Bn, double gam, double F[7]) {
  double UL[7], UR[7], FL[7], FR[7];
  prim2cons(WL, Bn, gam, UL); prim2cons(WR, Bn, gam, UR);
  physflux(WL, Bn, UL, FL); physflux(WR, Bn, UR, FR);
  double cfL = fastspeed(WL, Bn, gam), cfR = fastspeed(WR, Bn, gam);
  double bp = std::max(WR[1] + cfR, 0.0), bm = std::min(WL[1] - cfL, 0.0);
  RoeAvg r = roe_average(WL, WR, Bn, gam);
  if (r.a2 > 0.0) {
    WaveSet w = waveset(r.a2, r.rho, Bn, r.B1, r.B2);
    bp = std::max(bp, r.vn + w.cf); bm = std::min(bm, r.vn - w.cf);
  }
  for (int c = 0; c < 7; ++c) F[c] = (bp * FL[c] - bm * FR[c] + bp * bm * (UR[c] - UL[c])) / (bp - bm);
}

// A2 HLLD
void hlld(const double WL[7], const double WR[7], double Bn, double gam, double F[7]) {
  const double* W[2] = { WL, WR };
  double U[2][7], Fp[2][7], pT[2], cf[2];
  for (int a = 0; a < 2; ++a) {
    prim2cons(W[a], Bn, gam, U[a]); physflux(W[a], Bn, U[a], Fp[a]);
    pT[a] = W[a][4] + 0.5 * (sq(Bn) + sq(W[a][5]) + sq(W[a][6]));
    cf[a] = fastspeed(W[a], Bn, gam);
  }
  double uL = WL[1], uR = WR[1];
  double cmax = std::max(cf[0], cf[1]);
  double S[2] = { std::min(uL, uR) - cmax, std::max(uL, uR) + cmax };     // reading R12
  if (S[0] >= 0.0) { for (int c = 0; c < 7; ++c) F[c] = Fp[0][c]; return; }
  double s[2] = { (S[0] - uL) * WL[0], (S[1] - uR) * WR[0] };
  double SM = (s[1] * uR - s[0] * uL - pT[1] + pT[0]) / (s[1] - s[0]);
  double pTs = (s[1] * pT[0] - s[0] * pT[1] + s[0] * s[1] * (uR - uL)) / (s[1] - s[0]);
  double Us[2][7], Uss[2][7], rs[2], vBs[2], v1s[2], v2s[2];
  for (int a = 0; a < 2; ++a) {
    double rho_s = s[a] / (S[a] - SM);
    double D = s[a] * (S[a] - SM) - Bn * Bn;
    double v1, v2, B1, B2;
    if (std::fabs(D) < 1e-12 * pTs) { v1 = W[a][2]; v2 = W[a][3]; B1 = W[a][5]; B2 = W[a][6]; }
    else {
      double fv = Bn * (SM - W[a][1]) / D, fb = (s[a] * (S[a] - W[a][1]) - Bn * Bn) / D;
      v1 = W[a][2] - W[a][5] * fv; v2 = W[a][3] - W[a][6] * fv;
      B1 = W[a][5] * fb; B2 = W[a][6] * fb;
    }
    double vB = Bn * W[a][1] + W[a][5] * W[a][2] + W[a][6] * W[a][3];
    double vBstar = Bn * SM + B1 * v1 + B2 * v2;
    double es = ((S[a] - W[a][1]) * U[a][4] - pT[a] * W[a][1] + pTs * SM + Bn * (vB - vBstar)) / (S[a] - SM);
    Us[a][0] = rho_s; Us[a][1] = rho_s * SM; Us[a][2] = rho_s * v1; Us[a][3] = rho_s * v2; Us[a][4] = es; Us[a][5] = B1; Us[a][6] = B2;
    rs[a] = std::sqrt(rho_s); vBs[a] = vBstar; v1s[a] = v1; v2s[a] = v2;
  }
  double SsL = SM - std::fabs(Bn) / rs[0], SsR = SM + std::fabs(Bn) / rs[1];
  if (0.5 * Bn * Bn < 1e-12 * pTs) {
    for (int a = 0; a < 2; ++a) for (int c = 0; c < 7; ++c) Uss[a][c] = Us[a][c];
  } else {
    double sg = Bn > 0.0 ? 1.0 : -1.0, ir = 1.0 / (rs[0] + rs[1]);
    double v1 = (rs[0] * v1s[0] + rs[1] * v1s[1] + (Us[1][5] - Us[0][5]) * sg) * ir;
    double v2 = (rs[0] * v2s[0] + rs[1] * v2s[1] + (Us[1][6] - Us[0][6]) * sg) * ir;
    double B1 = (rs[0] * Us[1][5] + rs[1] * Us[0][5] + rs[0] * rs[1] * (v1s[1] - v1s[0]) * sg) * ir;
    double B2 = (rs[0] * Us[1][6] + rs[1] * Us[0][6] + rs[0] * rs[1] * (v2s[1] - v2s[0]) * sg) * ir;
    double vBss = Bn * SM + B1 * v1 + B2 * v2;
    for (int a = 0; a < 2; ++a) {
      double pm = a == 0 ? -1.0 : 1.0;
      Uss[a][0] = Us[a][0]; Uss[a][1] = Us[a][1]; Uss[a][2] = Us[a][0] * v1; Uss[a][3] = Us[a][0] * v2;
      Uss[a][4] = Us[a][4] + pm * rs[a] * (vBs[a] - vBss) * sg;
      Uss[a][5] = B1; Uss[a][6] = B2;
    }
  }
  if (SsL >= 0.0)      for (int c = 0; c < 7; ++c) F[c] = Fp[0][c] + S[0] * (Us[0][c] - U[0][c]);
  else if (SM >= 0.0)  for (int c = 0; c < 7; ++c) F[c] = Fp[0][c] + SsL * Uss[0][c] - (SsL - S[0]) * Us[0][c] - S[0] * U[0][c];
  else if (SsR >= 0.0) for (int c = 0; c < 7; ++c) F[c] = Fp[1][c] + SsR * Uss[1][c] - (SsR - S[1]) * Us[1][c] - S[1] * U[1][c];
  else if (S[1] >= 0.0) for (int c = 0; c < 7; ++c) F[c] = Fp[1][c] + S[1] * (Us[1][c] - U[1][c]);
  else                 for (int c = 0; c < 7; ++c) F[c] = Fp[1][c];
}

// Roe (reading R7/R11): 1/2(FL+FR) - 1/2 sum |lam_k| (L_k.dU) R_k, HLLE fallback
// returns 1 if it fell back to HLLE
// etah (reading R19, H-correction): every wave speed of the dissipation term is |lam_k| -> max(|lam_k|, etah); etah = 0: plain Roe
int roe(const double WL[7], const double WR[7], double Bn, double gam, double F[7], double etah = 0.0) {
  double UL[7], UR[7], FL[7], FR[7];
  prim2cons(WL, Bn, gam, UL); prim2cons(WR, Bn, gam, UR);
  physflux(WL, Bn, UL, FL); physflux(WR, Bn, UR, FR);
  RoeAvg r = roe_average(WL, WR, Bn, gam);
  if (!(r.a2 > 0.0)) { hlle(WL, WR, Bn, gam, F); return 1; }
  double lam[7], R[7][7], L[7][7], a[7], dU[7];
  eig_cons(r, Bn, gam, lam, R, L);
  // supersonic shortcuts; with the H-correction only where every wave is faster than etah, so that the flux stays a continuous
  // function of the states (for lam_min >= etah the dissipation formula below gives F_L exactly, as it does for plain Roe at lam_min >= 0)
  if (lam[0] >= etah) { for (int c = 0; c < 7; ++c) F[c] = FL[c]; return 0; }
  if (lam[6] <= -etah) { for (int c = 0; c < 7; ++c) F[c] = FR[c]; return 0; }
  for (int c = 0; c < 7; ++c) dU[c] = UR[c] - UL[c];
  for (int k = 0; k < 7; ++k) { a[k] = 0.0; for (int c = 0; c < 7; ++c) a[k] += L[k][c] * dU[c]; }
  // intermediate states U_L + sum_{k<=m} a_k R_k, m = 0..5, tested only where lam_{m+1} > lam_m
  double Ui[7];
  for (int c = 0; c < 7; ++c) Ui[c] = UL[c];
  for (int m = 0; m < 6; ++m) {
    for (int c = 0; c < 7; ++c) Ui[c] += a[m] * R[m][c];
    if (lam[m + 1] > lam[m]) {
      double P = (gam - 1.0) * (Ui[4] - 0.5 * (sq(Ui[1]) + sq(Ui[2]) + sq(Ui[3])) / Ui[0] - 0.5 * (sq(Bn) + sq(Ui[5]) + sq(Ui[6])));
      if (!(Ui[0] > 0.0) || !(P > 0.0)) { hlle(WL, WR, Bn, gam, F); return 1; }
    }
  }
  for (int c = 0; c < 7; ++c) {
    double d = 0.0;
    for (int k = 0; k < 7; ++k) d += std::max(std::fabs(lam[k]), etah) * a[k] * R[k][c];
    F[c] = 0.5 * (FL[c] + FR[c]) - 0.5 * d;
  }
  return 0;
}

int riemann(int solver, const double WL[7], const double WR[7], double Bn, double gam, double F[7], double etah = 0.0) {
  if (solver == 0) { hlle(WL, WR, Bn, gam, F); return 0; }
  if (solver == 1) { hlld(WL, WR, Bn, gam, F); return 0; }
  return roe(WL, WR, Bn, gam, F, etah);
}
// reading R19: eta of a face = half the largest jump of the two fast characteristic speeds v_n -+ c_f between its L and R states
double eta_face(const double WL[7], const double WR[7], double Bn, double gam) {
  double cl = fastspeed(WL, Bn, gam), cr = fastspeed(WR, Bn, gam);
  return 0.5 * std::max(std::fabs((WR[1] + cr) - (WL[1] + cl)), std::fabs((WR[1] - cr) - (WL[1] - cl)));
}

// ---------------------------------------------------------------------------------
// Edge EMF (readings R10, R10a = SURVEY C6 with the tie of DESIGN.md section 2.1)
// ---------------------------------------------------------------------------------
// upwind switch on the face mass flux m between the candidates qm (from the "-" side) and qp: qm if m > 0, qp if m < 0,
// the mean if m = 0.  R10a: "m = 0" means |m| <= m0 = tie * (mean density of the two cells rm, rp) [tie = emf_tie dh/dt],
// i.e. less than emf_tie of the cell mass crosses the face in dt; between m0 and 2 m0 the switch ramps linearly from
// the mean to the upwind value so that the EMF is a continuous function of m.  tie = 0 is the exact tie of SURVEY C6.
double emf_upwind(double tie, double m, double rm, double rp, double qm, double qp) {
  double m0 = tie * 0.5 * (rm + rp), am = std::fabs(m);
  if (am <= m0) return 0.5 * (qm + qp);
  if (am < 2.0 * m0) {
    double w = (am - m0) / m0;                       // 0..1: weight of the upwind value
    double qu = m > 0.0 ? qm : qp;
    return w * qu + (1.0 - w) * (0.5 * (qm + qp));
  }
  return m > 0.0 ? qm : qp;
}
// SURVEY C6 for the edge along c at (a-1/2, b-1/2), (a,b,c) cyclic.  Face EMFs (E_c from the face fluxes):
// Ea_lo = Ea(a-1/2, b-1), Ea_hi = Ea(a-1/2, b), Eb_lo = Eb(a-1, b-1/2), Eb_hi = Eb(a, b-1/2); mass fluxes through the same
// four faces; ec[4], rho[4] = reference EMF and density of the cells (a-1,b-1), (a,b-1), (a-1,b), (a,b)
double edge_emf_formula(double Ea_lo, double Ea_hi, double Eb_lo, double Eb_hi, double ma_lo, double ma_hi, double mb_lo,
                        double mb_hi, const double ec[4], const double rho[4], double tie) {
  double e = 0.25 * (Ea_hi + Ea_lo + Eb_hi + Eb_lo);
  e += 0.25 * (emf_upwind(tie, ma_lo, rho[0], rho[1], Eb_lo - ec[0], Eb_hi - ec[1]) - emf_upwind(tie, ma_hi, rho[2], rho[3], ec[2] - Eb_lo, ec[3] - Eb_hi));
  e += 0.25 * (emf_upwind(tie, mb_lo, rho[0], rho[2], Ea_lo - ec[0], Ea_hi - ec[2]) - emf_upwind(tie, mb_hi, rho[1], rho[3], ec[1] - Ea_lo, ec[3] - Ea_hi));
  return e;
}

// =====================================================================================
// one patch group
// =====================================================================================
struct Tile {
  int N, g, T, S;            // S = T+1 = uniform stride of every temporary
  size_t n3;
  inline size_t id(int i, int j, int k) const { return ((size_t)k * S + j) * S + i; }
};

// direction helpers: d=0,1,2 -> (n,t1,t2) cyclic; offsets of +1 along an axis
inline void cyc(int d, int& t1, int& t2) { t1 = (d + 1) % 3; t2 = (d + 2) % 3; }

struct Group {
  const mhdref_config& c;
  Tile t;
  double gam, dt, dh;
  Stats* st;
  // time-n data on the tile
  Arr U[5], b[3];           // conserved cell data, face fields (b[d] lower d-face of cell)
  Arr W[8];                 // rho, vx, vy, vz, P, Bcx, Bcy, Bcz
  Arr F[3][7];              // flux through the lower d-face of cell, generic component order
  Arr E[3];                 // edge EMF: E[0]=Ex at (i, j-1/2, k-1/2) etc.
  Arr Uh[5], bh[3], Wh[8];  // half-step data
  Arr Wlo[3][7], Wup[3][7]; // CTU: states at the lower / upper d-face of every cell (generic order)
  // H-correction (R19), in the pass whose fluxes update the solution (VL step 5, CTU step 6); the predictor pass keeps the plain
  // solver.  The pass over the faces runs twice, first recording eta of every face it visits, then solving with
  // eta^H = the largest eta among the face itself and the eight transverse faces of its two cells that were visited
  int hphase = 0;           // 0: no H-correction; 1: record eta; 2: solve with eta^H
  Arr eta[3];
  std::vector<char> etaok[3];

  Group(const mhdref_config& cfg, double dt_, double dh_, Stats* s) : c(cfg), gam(cfg.gamma), dt(dt_), dh(dh_), st(s) {
    t.N = cfg.ps2; t.g = cfg.nghost; t.T = t.N + 2 * t.g; t.S = t.T + 1; t.n3 = (size_t)t.S * t.S * t.S;
    auto mk = [&](Arr& a) { a.assign(t.n3, NaN); };
    for (auto& a : U) mk(a); for (auto& a : b) mk(a); for (auto& a : W) mk(a);
    for (auto& fd : F) for (auto& a : fd) mk(a);
    for (auto& a : E) mk(a); for (auto& a : Uh) mk(a); for (auto& a : bh) mk(a); for (auto& a : Wh) mk(a);
    if (cfg.scheme == 1) { for (auto& wd : Wlo) for (auto& a : wd) mk(a); for (auto& wd : Wup) for (auto& a : wd) mk(a); }
    if (cfg.hcorr) for (int d = 0; d < 3; ++d) { mk(eta[d]); etaok[d].assign(t.n3, 0); }
  }
  double etaH(int d, size_t q) const {
    int t1, t2; cyc(d, t1, t2);
    double e = eta[d][q];
    const int tt[2] = { t1, t2 };
    for (int s = 0; s < 2; ++s) {
      const int tdir = tt[s];
      const size_t ql = q - off(d), x[4] = { ql, ql + (size_t)off(tdir), q, q + (size_t)off(tdir) };   // lower / upper t-faces of the two cells
      for (int n = 0; n < 4; ++n) if (etaok[tdir][x[n]]) e = std::max(e, eta[tdir][x[n]]);
    }
    return e;
  }
  template <class Fn> void face_pass(Fn&& loops) {
    if (!c.hcorr) { loops(); return; }
    for (int d = 0; d < 3; ++d) { eta[d].assign(t.n3, NaN); etaok[d].assign(t.n3, 0); }
    hphase = 1; loops();
    hphase = 2; loops();
    hphase = 0;
  }
  inline int off(int d) const { return d == 0 ? 1 : (d == 1 ? t.S : t.S * t.S); }
  static inline void stage(int n) { if (mhdref_stage_hook) mhdref_stage_hook(n); }

  void load(const double* Uin, const double* Bin) {
    int T = t.T;
    for (int v = 0; v < 5; ++v)
      for (int k = 0; k < T; ++k) for (int j = 0; j < T; ++j) for (int i = 0; i < T; ++i)
        U[v][t.id(i, j, k)] = Uin[(((size_t)v * T + k) * T + j) * T + i];
    const double* bx = Bin; const double* by = bx + (size_t)T * T * (T + 1); const double* bz = by + (size_t)T * T * (T + 1);
    for (int k = 0; k < T; ++k) for (int j = 0; j < T; ++j) for (int i = 0; i <= T; ++i) b[0][t.id(i, j, k)] = bx[((size_t)k * T + j) * (T + 1) + i];
    for (int k = 0; k < T; ++k) for (int j = 0; j <= T; ++j) for (int i = 0; i < T; ++i) b[1][t.id(i, j, k)] = by[((size_t)k * (T + 1) + j) * T + i];
    for (int k = 0; k <= T; ++k) for (int j = 0; j < T; ++j) for (int i = 0; i < T; ++i) b[2][t.id(i, j, k)] = bz[((size_t)k * T + j) * T + i];
  }

  // S1 con -> prim on cells [lo,hi)^3 (Eq. 5; floors: reading R9)
  void con2prim(const Arr Uc[5], const Arr bf[3], Arr Wc[8], int lo, int hi) {
    for (int k = lo; k < hi; ++k) for (int j = lo; j < hi; ++j) for (int i = lo; i < hi; ++i) {
      size_t q = t.id(i, j, k);
      double Bc[3];
      for (int d = 0; d < 3; ++d) Bc[d] = 0.5 * (bf[d][q] + bf[d][q + off(d)]);
      double rho = Uc[0][q];
      if (rho < c.min_dens) { rho = c.min_dens; if (st) st->fd++; }
      double vx = Uc[1][q] / rho, vy = Uc[2][q] / rho, vz = Uc[3][q] / rho;
      double P = (gam - 1.0) * (Uc[4][q] - 0.5 * rho * (vx * vx + vy * vy + vz * vz) - 0.5 * (Bc[0] * Bc[0] + Bc[1] * Bc[1] + Bc[2] * Bc[2]));
      if (P < c.min_pres) { P = c.min_pres; if (st) st->fp++; }
      Wc[0][q] = rho; Wc[1][q] = vx; Wc[2][q] = vy; Wc[3][q] = vz; Wc[4][q] = P;
      Wc[5][q] = Bc[0]; Wc[6][q] = Bc[1]; Wc[7][q] = Bc[2];
    }
  }
  // generic 1-D state of a cell for direction d
  inline void gen(const Arr Wc[8], size_t q, int d, double w[7]) const {
    int t1, t2; cyc(d, t1, t2);
    w[0] = Wc[0][q]; w[1] = Wc[1 + d][q]; w[2] = Wc[1 + t1][q]; w[3] = Wc[1 + t2][q];
    w[4] = Wc[4][q]; w[5] = Wc[5 + t1][q]; w[6] = Wc[5 + t2][q];
  }
  void floors(double w[7]) {
    const bool count = st && hphase != 1;           // the eta-recording sweep of a pass repeats the states of the solving sweep
    if (w[0] < c.min_dens) { w[0] = c.min_dens; if (count) st->fd++; }
    if (w[4] < c.min_pres) { w[4] = c.min_pres; if (count) st->fp++; }
  }

  // reading R10: edge EMFs from the face fluxes F, cell-centred reference field from Wc (v, Bc).
  // Edge along c=(d) at (a-1/2, b-1/2), (a,b,c) cyclic.  Range: a,b in [alo,ahi], c in [clo,chi).
  void edge_emf(const Arr Wc[8], int alo, int ahi, int clo, int chi) {
    for (int cdir = 0; cdir < 3; ++cdir) {
      int a = (cdir + 1) % 3, bdir = (cdir + 2) % 3;   // (a,b,c) cyclic
      int oa = off(a), ob = off(bdir);
      // from an a-face (n=a,t1=b,t2=c): E_c = E_t2 = -F[B_t1] = -F[5]; from a b-face (n=b,t1=c,t2=a): E_c = E_t1 = +F[B_t2] = +F[6]
      auto Ea = [&](size_t q) { return -F[a][5][q]; };
      auto Eb = [&](size_t q) { return F[bdir][6][q]; };
      auto ec = [&](size_t q) { return Wc[1 + bdir][q] * Wc[5 + a][q] - Wc[1 + a][q] * Wc[5 + bdir][q]; };  // -(v x B)_c
      const double tie = c.emf_tie * dh / dt;               // R10a: m0 = tie * (mean density of the two cells)
      const Arr& rho = Wc[0];
      int idx[3];
      for (idx[cdir] = clo; idx[cdir] < chi; ++idx[cdir])
        for (idx[bdir] = alo; idx[bdir] <= ahi; ++idx[bdir])
          for (idx[a] = alo; idx[a] <= ahi; ++idx[a]) {
            size_t q = t.id(idx[0], idx[1], idx[2]);      // cell (a,b); its lower a-face is "a-1/2"
            size_t qa = q - oa, qb = q - ob, qab = q - oa - ob;
            double ma_lo = F[a][0][qb], ma_hi = F[a][0][q];       // mass flux through a-face (a-1/2, b-1) and (a-1/2, b)
            double mb_lo = F[bdir][0][qa], mb_hi = F[bdir][0][q]; // through b-face (a-1, b-1/2) and (a, b-1/2)
            // cells in the order (a-1,b-1), (a,b-1), (a-1,b), (a,b)
            const double ecs[4] = { ec(qab), ec(qb), ec(qa), ec(q) }, rhos[4] = { rho[qab], rho[qb], rho[qa], rho[q] };
            double e = edge_emf_formula(Ea(qb), Ea(q), Eb(qa), Eb(q), ma_lo, ma_hi, mb_lo, mb_hi, ecs, rhos, tie);
            E[cdir][q] = e;
          }
    }
  }
  // Eq. 13 on all faces of cells [lo,hi)^3 with step tau
  void ct_update(const Arr bin[3], Arr bout[3], double tau, int lo, int hi) {
    double qh = tau / dh;
    int ox = off(0), oy = off(1), oz = off(2);
    for (int k = lo; k < hi; ++k) for (int j = lo; j < hi; ++j) for (int i = lo; i <= hi; ++i) {
      size_t q = t.id(i, j, k);
      bout[0][q] = bin[0][q] - qh * ((E[2][q + oy] - E[2][q]) - (E[1][q + oz] - E[1][q]));
    }
    for (int k = lo; k < hi; ++k) for (int j = lo; j <= hi; ++j) for (int i = lo; i < hi; ++i) {
      size_t q = t.id(i, j, k);
      bout[1][q] = bin[1][q] - qh * ((E[0][q + oz] - E[0][q]) - (E[2][q + ox] - E[2][q]));
    }
    for (int k = lo; k <= hi; ++k) for (int j = lo; j < hi; ++j) for (int i = lo; i < hi; ++i) {
      size_t q = t.id(i, j, k);
      bout[2][q] = bin[2][q] - qh * ((E[1][q + ox] - E[1][q]) - (E[0][q + oy] - E[0][q]));
    }
  }
  // Eq. 10 on cells [lo,hi)^3 with step tau; flux-difference sums in the fixed order x, y, z
  void fv_update(Arr Uo[5], double tau, int lo, int hi) {
    double qh = tau / dh;
    for (int k = lo; k < hi; ++k) for (int j = lo; j < hi; ++j) for (int i = lo; i < hi; ++i) {
      size_t q = t.id(i, j, k);
      double dU[5] = { 0, 0, 0, 0, 0 };
      for (int d = 0; d < 3; ++d) {
        int t1, t2; cyc(d, t1, t2);
        size_t qu = q + off(d);
        dU[0] += F[d][0][qu] - F[d][0][q];
        dU[1 + d] += F[d][1][qu] - F[d][1][q];
        dU[1 + t1] += F[d][2][qu] - F[d][2][q];
        dU[1 + t2] += F[d][3][qu] - F[d][3][q];
        dU[4] += F[d][4][qu] - F[d][4][q];
      }
      for (int v = 0; v < 5; ++v) Uo[v][q] = U[v][q] - qh * dU[v];
    }
  }
  void solve_face(int d, size_t q, const double wl[7], const double wr[7], double bn, Arr (*Fout)[7] = nullptr) {
    if (hphase == 1) { eta[d][q] = eta_face(wl, wr, bn, gam); etaok[d][q] = 1; return; }
    double f[7];
    int fb = hphase == 2 ? riemann(c.riemann, wl, wr, bn, gam, f, etaH(d, q)) : riemann(c.riemann, wl, wr, bn, gam, f);
    if (fb && st) st->fb++;
    Arr (*Fo)[7] = Fout ? Fout : F;
    for (int v = 0; v < 7; ++v) Fo[d][v][q] = f[v];
  }

  // the slope limiter selected by the configuration (R5: MC; NEXT-4 variants: minmod, van Leer)
  double lim(double a, double b) const { return c.limiter == 1 ? mm(a, b) : (c.limiter == 2 ? vanleer(a, b) : mc(a, b)); }

  // PPM parabola of cell q in direction d (reading C4): interface values from the limited slopes of the cell and its
  // two neighbours, monotonised (i)-(iii); returns W_l, W_r, dW = W_r - W_l, W6
  void ppm_parabola(const Arr Wc[8], size_t q, int d, double Wl[7], double Wr[7], double dW[7], double W6[7]) const {
    int od = off(d);
    double sm[7], s0[7], sp[7], wm[7], w0[7], wp[7];
    slope(Wc, q - od, d, sm); slope(Wc, q, d, s0); slope(Wc, q + od, d, sp);
    gen(Wc, q - od, d, wm); gen(Wc, q, d, w0); gen(Wc, q + od, d, wp);
    for (int v = 0; v < 7; ++v) {
      Wl[v] = 0.5 * (wm[v] + w0[v]) - (s0[v] - sm[v]) / 6.0;
      Wr[v] = 0.5 * (w0[v] + wp[v]) - (sp[v] - s0[v]) / 6.0;
      // monotonise (C4 i-iii)
      if ((Wr[v] - w0[v]) * (w0[v] - Wl[v]) <= 0.0) { Wl[v] = w0[v]; Wr[v] = w0[v]; }
      double dw = Wr[v] - Wl[v], w6 = 6.0 * (w0[v] - 0.5 * (Wl[v] + Wr[v]));
      double nl = Wl[v], nr = Wr[v];
      if (dw * w6 > dw * dw) nl = 3.0 * w0[v] - 2.0 * Wr[v];
      if (dw * w6 < -dw * dw) nr = 3.0 * w0[v] - 2.0 * Wl[v];
      Wl[v] = nl; Wr[v] = nr;
      Wl[v] = std::max(std::min(w0[v], wm[v]), std::min(std::max(w0[v], wm[v]), Wl[v]));
      Wr[v] = std::max(std::min(w0[v], wp[v]), std::min(std::max(w0[v], wp[v]), Wr[v]));
      dW[v] = Wr[v] - Wl[v]; W6[v] = 6.0 * (w0[v] - 0.5 * (Wl[v] + Wr[v]));
    }
  }

  // limited slope of the generic state of cell q in direction d (R4/R5): primitive or characteristic
  void slope(const Arr Wc[8], size_t q, int d, double dWm[7]) const {
    double wm[7], w0[7], wp[7], dl[7], dr[7];
    gen(Wc, q - off(d), d, wm); gen(Wc, q, d, w0); gen(Wc, q + off(d), d, wp);
    for (int v = 0; v < 7; ++v) { dl[v] = w0[v] - wm[v]; dr[v] = wp[v] - w0[v]; }
    if (c.limvar == 0) { for (int v = 0; v < 7; ++v) dWm[v] = lim(dl[v], dr[v]); return; }
    double lam[7], R[7][7], L[7][7];
    eig_prim(w0, Wc[5 + d][q], gam, lam, R, L);
    for (int v = 0; v < 7; ++v) dWm[v] = 0.0;
    for (int k = 0; k < 7; ++k) {
      double al = 0.0, ar = 0.0;
      for (int v = 0; v < 7; ++v) { al += L[k][v] * dl[v]; ar += L[k][v] * dr[v]; }
      double am = lim(al, ar);
      for (int v = 0; v < 7; ++v) dWm[v] += am * R[k][v];
    }
  }

  // ------------------------------------------------------------------------------
  // VL, reading C2
  // ------------------------------------------------------------------------------
  void advance_vl() {
    int T = t.T;
    const bool mn = c.minimal_ranges != 0 && !c.hcorr;
    const int g = t.g, N = t.N;
    con2prim(U, b, W, 0, T);                                           // time-n primitives
    stage(1);
    // step 1: first-order fluxes, longitudinal B = face value; R19: the predictor pass uses the plain solver
    for (int d = 0; d < 3; ++d) {
      int lo[3] = { 0, 0, 0 }; lo[d] = 1;
      for (int k = lo[2]; k < T; ++k) for (int j = lo[1]; j < T; ++j) for (int i = lo[0]; i < T; ++i) {
        size_t q = t.id(i, j, k);
        double wl[7], wr[7];
        gen(W, q - off(d), d, wl); gen(W, q, d, wr);
        solve_face(d, q, wl, wr, b[d][q]);
      }
    }
    stage(2);
    edge_emf(W, 1, T - 1, mn ? 1 : 0, mn ? T - 1 : T);                 // step 2 (the half step reads edges along c only for c in [1, T-1))
    stage(3);
    fv_update(Uh, 0.5 * dt, 1, T - 1);                                 // step 3 (dt/2)
    ct_update(b, bh, 0.5 * dt, 1, T - 1);
    con2prim(Uh, bh, Wh, 1, T - 1);
    stage(4);
    for (auto& fd : F) for (auto& a : fd) a.assign(t.n3, NaN);           // pass-1 fluxes are dead from here on
    // step 4+5: PLM (or, NEXT-4 variant, the PPM parabola of C4) in primitive/characteristic variables at the half step,
    // no tracing (the half step supplies the time centring); Bn = bh(face).  Faces whose stencil lies inside the cells
    // that carry a half-step state: PLM cells i-2..i+1 -> faces 3..T-3; PPM cells i-3..i+2 -> faces 4..T-4
    const int r = c.recon == 0 ? 3 : 4;
    // minimal: the faces of the interior cells and of their transverse neighbours (the edge EMFs of the interior faces need those)
    const int tlo = mn ? g - 1 : 1, thi = mn ? g + N + 1 : T - 1, nlo = mn ? g : r, nhi = mn ? g + N : T - r;
    face_pass([&]() {
    for (int d = 0; d < 3; ++d) {
      int t1, t2; cyc(d, t1, t2);
      int idx[3];
      for (idx[t2] = tlo; idx[t2] < thi; ++idx[t2]) for (idx[t1] = tlo; idx[t1] < thi; ++idx[t1]) for (idx[d] = nlo; idx[d] <= nhi; ++idx[d]) {
        size_t q = t.id(idx[0], idx[1], idx[2]), ql = q - off(d);
        double wl[7], wr[7];
        if (c.recon == 0) {
          double sl[7], sr[7];
          gen(Wh, ql, d, wl); gen(Wh, q, d, wr);
          slope(Wh, ql, d, sl); slope(Wh, q, d, sr);
          for (int v = 0; v < 7; ++v) { wl[v] += 0.5 * sl[v]; wr[v] -= 0.5 * sr[v]; }
        } else {
          double lo_[7], dW[7], W6[7], up_[7];
          ppm_parabola(Wh, ql, d, lo_, wl, dW, W6);      // L state = W_r of the cell below the face
          ppm_parabola(Wh, q, d, wr, up_, dW, W6);       // R state = W_l of the cell above it
        }
        floors(wl); floors(wr);
        solve_face(d, q, wl, wr, bh[d][q]);
      }
    }
    });
    stage(5);
    if (mn) edge_emf(Wh, g, g + N, g, g + N); else edge_emf(Wh, r, T - r, 1, T - 1);   // step 6
    stage(6);
  }

  // ------------------------------------------------------------------------------
  // CTU, readings C3, C4
  // ------------------------------------------------------------------------------
  void advance_ctu() {
    int T = t.T;
    int r = c.recon == 0 ? 1 : 2;
    double sig = dt / dh, hdt = 0.5 * dt;
    const bool mn = c.minimal_ranges != 0 && !c.hcorr;
    // minimal: everything is derived from the cells whose half-step state the second pass needs, [lo, hi)^3 = interior + 1
    const int lo_ = t.g - 1, hi_ = t.g + t.N + 1;
    con2prim(U, b, W, 0, T);
    stage(1);
    // step 1: reconstruction + half-step tracing (matrix form, all waves) + primitive MHD source terms
    for (int d = 0; d < 3; ++d) {
      int t1, t2; cyc(d, t1, t2);
      int lo[3] = { 0, 0, 0 }, hi[3] = { T, T, T }; lo[d] = r; hi[d] = T - r;
      if (mn) for (int a = 0; a < 3; ++a) { lo[a] = lo_ - 1; hi[a] = hi_ + 1; }        // face states one cell beyond [lo, hi)^3
      for (int k = lo[2]; k < hi[2]; ++k) for (int j = lo[1]; j < hi[1]; ++j) for (int i = lo[0]; i < hi[0]; ++i) {
        size_t q = t.id(i, j, k);
        int od = off(d);
        double w0[7], A[7][7], wlo[7], wup[7];
        gen(W, q, d, w0);
        primA(w0, W[5 + d][q], gam, A);
        auto Ax = [&](const double x[7], double y[7]) { for (int a = 0; a < 7; ++a) { y[a] = 0.0; for (int e = 0; e < 7; ++e) y[a] += A[a][e] * x[e]; } };
        if (c.recon == 0) {
          double dWm[7], AdW[7];
          slope(W, q, d, dWm); Ax(dWm, AdW);
          for (int v = 0; v < 7; ++v) { wup[v] = w0[v] + 0.5 * dWm[v] - 0.5 * sig * AdW[v]; wlo[v] = w0[v] - 0.5 * dWm[v] - 0.5 * sig * AdW[v]; }
        } else {
          double Wl[7], Wr[7], dW[7], W6[7];
          ppm_parabola(W, q, d, Wl, Wr, dW, W6);
          double xu[7], xl[7], Au[7], Al[7], A6[7], AA6[7];
          for (int v = 0; v < 7; ++v) { xu[v] = dW[v] - W6[v]; xl[v] = dW[v] + W6[v]; }
          Ax(xu, Au); Ax(xl, Al); Ax(W6, A6); Ax(A6, AA6);
          for (int v = 0; v < 7; ++v) {
            wup[v] = Wr[v] - 0.5 * sig * Au[v] - sig * sig * AA6[v] / 3.0;
            wlo[v] = Wl[v] - 0.5 * sig * Al[v] - sig * sig * AA6[v] / 3.0;
          }
        }
        // primitive-stage MHD source terms (C3 step 1)
        double dbn = (b[d][q + od] - b[d][q]) / dh, db1 = (b[t1][q + off(t1)] - b[t1][q]) / dh, db2 = (b[t2][q + off(t2)] - b[t2][q]) / dh;
        double s1 = hdt * w0[2] * mm(dbn, -db1), s2 = hdt * w0[3] * mm(dbn, -db2);
        wlo[5] += s1; wup[5] += s1; wlo[6] += s2; wup[6] += s2;
        floors(wlo); floors(wup);
        for (int v = 0; v < 7; ++v) { Wlo[d][v][q] = wlo[v]; Wup[d][v][q] = wup[v]; }
      }
    }
    // step 2: F1 = Riemann(Wup(i-1), Wlo(i), b_n(face) at t^n); R19: the predictor pass uses the plain solver
    for (int d = 0; d < 3; ++d) {
      int lo[3] = { 0, 0, 0 }, hi[3] = { T, T, T }; lo[d] = r + 1; hi[d] = T - r;
      if (mn) { for (int a = 0; a < 3; ++a) { lo[a] = lo_ - 1; hi[a] = hi_ + 1; } lo[d] = lo_; }   // faces n in [lo, hi], t in [lo-1, hi]
      for (int k = lo[2]; k < hi[2]; ++k) for (int j = lo[1]; j < hi[1]; ++j) for (int i = lo[0]; i < hi[0]; ++i) {
        size_t q = t.id(i, j, k), ql = q - off(d);
        double wl[7], wr[7];
        for (int v = 0; v < 7; ++v) { wl[v] = Wup[d][v][ql]; wr[v] = Wlo[d][v][q]; }
        solve_face(d, q, wl, wr, b[d][q]);
      }
    }
    stage(2);
    if (mn) edge_emf(W, lo_, hi_, lo_, hi_); else edge_emf(W, r + 1, T - 1 - r, 0, T);   // step 3
    stage(3);
    fv_update(Uh, hdt, r + 1, T - 1 - r);                              // step 4
    ct_update(b, bh, hdt, r + 1, T - 1 - r);
    con2prim(Uh, bh, Wh, r + 1, T - 1 - r);
    stage(4);
    // step 5: transverse flux-gradient correction + conservative MHD source terms (C3 step 5)
    double qh = hdt / dh;
    for (int d = 0; d < 3; ++d) {
      int t1, t2; cyc(d, t1, t2);
      int od = off(d), o1 = off(t1), o2 = off(t2);
      int lo[3], hi[3];
      lo[t1] = lo[t2] = r + 1; hi[t1] = hi[t2] = T - 1 - r; lo[d] = r; hi[d] = T - r;
      if (mn) { lo[d] = lo_; hi[d] = hi_; }                            // the two cells of every pass-2 face
      for (int k = lo[2]; k < hi[2]; ++k) for (int j = lo[1]; j < hi[1]; ++j) for (int i = lo[0]; i < hi[0]; ++i) {
        size_t q = t.id(i, j, k);
        int cn = (d == 0 ? i : (d == 1 ? j : k));
        double w0[7]; gen(W, q, d, w0);
        double Bcn = W[5 + d][q];
        // transverse flux differences, permuted into the generic order of direction d:
        // F[t1] is in generic order (t1, t2, d): its (n,t1,t2) momentum slots are (M_t1, M_t2, M_d)
        double dF[5];
        dF[0] = (F[t1][0][q + o1] - F[t1][0][q]) + (F[t2][0][q + o2] - F[t2][0][q]);
        dF[1] = (F[t1][3][q + o1] - F[t1][3][q]) + (F[t2][2][q + o2] - F[t2][2][q]);   // M_d
        dF[2] = (F[t1][1][q + o1] - F[t1][1][q]) + (F[t2][3][q + o2] - F[t2][3][q]);   // M_t1
        dF[3] = (F[t1][2][q + o1] - F[t1][2][q]) + (F[t2][1][q + o2] - F[t2][1][q]);   // M_t2
        dF[4] = (F[t1][4][q + o1] - F[t1][4][q]) + (F[t2][4][q + o2] - F[t2][4][q]);
        // E_n on the four n-directed edges of the cell: E[d] at (t1-1/2,t2-1/2)=q, (t1+1/2,t2-1/2)=q+o1, ...
        double Emm = E[d][q], Epm = E[d][q + o1], Emp = E[d][q + o2], Epp = E[d][q + o1 + o2];
        double dB1 = -qh * 0.5 * ((Emp - Emm) + (Epp - Epm));
        double dB2 = qh * 0.5 * ((Epm - Emm) + (Epp - Emp));
        double dbn = (b[d][q + od] - b[d][q]) / dh, db1 = (b[t1][q + o1] - b[t1][q]) / dh, db2 = (b[t2][q + o2] - b[t2][q]) / dh;
        double m1 = mm(dbn, -db2), m2 = mm(dbn, -db1);
        double Bc1 = w0[5], Bc2 = w0[6], v1 = w0[2], v2 = w0[3];
        for (int side = 0; side < 2; ++side) {     // 0: Wlo (lower face cn), 1: Wup (upper face cn+1)
          int face = cn + side;
          if (face < r + 1 || face > T - 1 - r) continue;              // bh exists only there
          if (mn && (face < t.g || face > t.g + t.N)) continue;        // minimal: only the states of the interior faces
          size_t qf = q + (side ? od : 0);
          double w[7], u[7];
          for (int v = 0; v < 7; ++v) w[v] = side ? Wup[d][v][q] : Wlo[d][v][q];
          prim2cons(w, b[d][qf], gam, u);
          u[0] -= qh * dF[0]; u[1] -= qh * dF[1]; u[2] -= qh * dF[2]; u[3] -= qh * dF[3]; u[4] -= qh * dF[4];
          u[5] += dB1; u[6] += dB2;
          u[1] += hdt * Bcn * dbn; u[2] += hdt * Bc1 * dbn; u[3] += hdt * Bc2 * dbn;
          u[5] += hdt * v1 * m1; u[6] += hdt * v2 * m2;
          u[4] += hdt * (Bc1 * v1 * m1 + Bc2 * v2 * m2);
          double bn = bh[d][qf];
          double rho = u[0];
          if (rho < c.min_dens) { rho = c.min_dens; if (st) st->fd++; }
          w[0] = rho; w[1] = u[1] / rho; w[2] = u[2] / rho; w[3] = u[3] / rho;
          w[5] = u[5]; w[6] = u[6];
          w[4] = (gam - 1.0) * (u[4] - 0.5 * rho * (sq(w[1]) + sq(w[2]) + sq(w[3])) - 0.5 * (sq(bn) + sq(w[5]) + sq(w[6])));
          if (w[4] < c.min_pres) { w[4] = c.min_pres; if (st) st->fp++; }
          for (int v = 0; v < 7; ++v) (side ? Wup : Wlo)[d][v][q] = w[v];
        }
      }
    }
    // step 6: F2 = Riemann(corrected Wup(i-1), Wlo(i), bh_n)
    {
      Arr F2[3][7];
      for (int d = 0; d < 3; ++d) for (int v = 0; v < 7; ++v) F2[d][v].assign(t.n3, NaN);
      face_pass([&]() {
      for (int d = 0; d < 3; ++d) {
        int t1, t2; cyc(d, t1, t2);
        int lo[3], hi[3];
        lo[t1] = lo[t2] = r + 1; hi[t1] = hi[t2] = T - 1 - r; lo[d] = r + 1; hi[d] = T - r;
        if (mn) { lo[d] = t.g; hi[d] = t.g + t.N + 1; }
        for (int k = lo[2]; k < hi[2]; ++k) for (int j = lo[1]; j < hi[1]; ++j) for (int i = lo[0]; i < hi[0]; ++i) {
          size_t q = t.id(i, j, k), ql = q - off(d);
          double wl[7], wr[7];
          for (int v = 0; v < 7; ++v) { wl[v] = Wup[d][v][ql]; wr[v] = Wlo[d][v][q]; }
          solve_face(d, q, wl, wr, bh[d][q], F2);
        }
      }
      });
      for (int d = 0; d < 3; ++d) for (int v = 0; v < 7; ++v) F[d][v].swap(F2[d][v]);
    }
    stage(5);
    if (mn) edge_emf(Wh, t.g, t.g + t.N, t.g, t.g + t.N); else edge_emf(Wh, r + 2, T - 2 - r, r + 1, T - 1 - r);   // step 7
    stage(6);
  }

  void run(const double* Uin, const double* Bin, double* Uout, double* Bout, double* fout, double* eout) {
    load(Uin, Bin);
    stage(0);
    if (c.scheme == 0) advance_vl(); else advance_ctu();
    // step 7 (VL) / 8 (CTU): full update with F2 and the second edge EMFs; outputs
    int N = t.N, g = t.g;
    Arr Un[5], bn[3];
    for (auto& a : Un) a.assign(t.n3, NaN);
    for (auto& a : bn) a.assign(t.n3, NaN);
    fv_update(Un, dt, g, g + N);
    ct_update(b, bn, dt, g, g + N);
    stage(7);
    for (int v = 0; v < 5; ++v) for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i)
      Uout[(((size_t)v * N + k) * N + j) * N + i] = Un[v][t.id(i + g, j + g, k + g)];
    double* ox = Bout; double* oy = ox + (size_t)N * N * (N + 1); double* oz = oy + (size_t)N * N * (N + 1);
    for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i <= N; ++i) ox[((size_t)k * N + j) * (N + 1) + i] = bn[0][t.id(i + g, j + g, k + g)];
    for (int k = 0; k < N; ++k) for (int j = 0; j <= N; ++j) for (int i = 0; i < N; ++i) oy[((size_t)k * (N + 1) + j) * N + i] = bn[1][t.id(i + g, j + g, k + g)];
    for (int k = 0; k <= N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i) oz[((size_t)k * N + j) * N + i] = bn[2][t.id(i + g, j + g, k + g)];
    // boundary / mid-plane fluxes and EMFs (layout: reading R17)
    for (int d = 0; d < 3; ++d) {
      int t1, t2; cyc(d, t1, t2);
      for (int s = 0; s < 3; ++s) {
        int p = 3 * d + s, fi = (s == 0 ? 0 : (s == 1 ? N / 2 : N)) + g;
        int idx[3]; idx[d] = fi;
        if (fout) for (int a2 = 0; a2 < N; ++a2) for (int a1 = 0; a1 < N; ++a1) {
          idx[t1] = a1 + g; idx[t2] = a2 + g;
          size_t q = t.id(idx[0], idx[1], idx[2]);
          double fg[5]; fg[0] = F[d][0][q]; fg[1 + d] = F[d][1][q]; fg[1 + t1] = F[d][2][q]; fg[1 + t2] = F[d][3][q]; fg[4] = F[d][4][q];
          for (int v = 0; v < 5; ++v) fout[(((size_t)p * 5 + v) * N + a2) * N + a1] = fg[v];
        }
        if (eout) {
          double* e0 = eout + (size_t)p * 2 * (N + 1) * N; double* e1 = e0 + (size_t)(N + 1) * N;
          for (int a2 = 0; a2 <= N; ++a2) for (int a1 = 0; a1 < N; ++a1) {   // E_t1 at t2-1/2
            idx[t1] = a1 + g; idx[t2] = a2 + g;
            e0[(size_t)a2 * N + a1] = E[t1][t.id(idx[0], idx[1], idx[2])];
          }
          for (int a2 = 0; a2 < N; ++a2) for (int a1 = 0; a1 <= N; ++a1) {   // E_t2 at t1-1/2
            idx[t1] = a1 + g; idx[t2] = a2 + g;
            e1[(size_t)a2 * (N + 1) + a1] = E[t2][t.id(idx[0], idx[1], idx[2])];
          }
        }
      }
    }
  }
};

int check_cfg(const mhdref_config* c) {
  if (!c) return -1;
  if (c->ps2 < 2 || c->scheme < 0 || c->scheme > 1 || c->recon < 0 || c->recon > 1 || c->riemann < 0 || c->riemann > 2 || c->limvar < 0 || c->limvar > 1 || c->limiter < 0 || c->limiter > 2) return -1;
  int need = c->recon == 1 ? 4 : 3;                        // reading R8
  if (c->hcorr < 0 || c->hcorr > 1 || (c->hcorr && c->riemann != 2)) return -1;
  if (c->hcorr) need += 1;                                 // reading R19: eta of the transverse faces one cell further out
  if (c->nghost < need) return -1;
  if (!(c->gamma > 1.0)) return -1;
  if (!(c->emf_tie >= 0.0)) return -1;
  return 0;
}

}  // namespace

extern "C" {

// advance ngroups patch groups by dt (host pointers, double).  stats[3] += (density floors, pressure floors, Riemann fallbacks)
int mhdref_advance(const mhdref_config* cfg, const double* U_in, const double* B_in, double* U_out, double* B_out,
                   double* flux_out, double* emf_out, int ngroups, double dt, double dh, unsigned long long* stats, int force_ghost_ok) {
  if (!force_ghost_ok && check_cfg(cfg)) return -1;
  if (!U_in || !B_in || !U_out || !B_out || ngroups < 0) return -1;
  int N = cfg->ps2, T = N + 2 * cfg->nghost;
  size_t nUi = 5 * (size_t)T * T * T, nBi = 3 * (size_t)T * T * (T + 1), nUo = 5 * (size_t)N * N * N, nBo = 3 * (size_t)N * N * (N + 1);
  size_t nF = 9 * 5 * (size_t)N * N, nE = 9 * 2 * (size_t)(N + 1) * N;
  unsigned long long fd = 0, fp = 0, fb = 0;
#pragma omp parallel for schedule(dynamic) reduction(+ : fd, fp, fb)
  for (int gidx = 0; gidx < ngroups; ++gidx) {
    Stats s;
    Group G(*cfg, dt, dh, &s);
    G.run(U_in + gidx * nUi, B_in + gidx * nBi, U_out + gidx * nUo, B_out + gidx * nBo,
          flux_out ? flux_out + gidx * nF : nullptr, emf_out ? emf_out + gidx * nE : nullptr);
    fd += s.fd; fp += s.fp; fb += s.fb;
  }
  if (stats) { stats[0] += fd; stats[1] += fp; stats[2] += fb; }
  return 0;
}

// C8: dt = cfl*dh / max over interior cells and directions of |v_d| + c_f,d.  Arrays have `ng` ghost cells (0 or nghost).
int mhdref_dt(const mhdref_config* cfg, const double* U, const double* B, int ngroups, int ng, double dh, double cfl,
              double* dt_out, double* maxspeed_out) {
  if (!cfg || !U || !B || !dt_out) return -1;
  int N = cfg->ps2, T = N + 2 * ng;
  double gam = cfg->gamma;
  size_t nU = 5 * (size_t)T * T * T, nf = (size_t)T * T * (T + 1);
  double smax = 0.0;
  for (int gi = 0; gi < ngroups; ++gi) {
    const double* u = U + gi * nU; const double* bx = B + gi * 3 * nf; const double* by = bx + nf; const double* bz = by + nf;
    for (int k = ng; k < ng + N; ++k) for (int j = ng; j < ng + N; ++j) for (int i = ng; i < ng + N; ++i) {
      size_t q = ((size_t)k * T + j) * T + i, n3 = (size_t)T * T * T;
      double Bc[3] = { 0.5 * (bx[((size_t)k * T + j) * (T + 1) + i] + bx[((size_t)k * T + j) * (T + 1) + i + 1]),
                       0.5 * (by[((size_t)k * (T + 1) + j) * T + i] + by[((size_t)k * (T + 1) + j + 1) * T + i]),
                       0.5 * (bz[((size_t)k * T + j) * T + i] + bz[((size_t)(k + 1) * T + j) * T + i]) };
      double rho = std::max(u[q], cfg->min_dens);
      double v[3] = { u[n3 + q] / rho, u[2 * n3 + q] / rho, u[3 * n3 + q] / rho };
      double P = (gam - 1.0) * (u[4 * n3 + q] - 0.5 * rho * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]) - 0.5 * (Bc[0] * Bc[0] + Bc[1] * Bc[1] + Bc[2] * Bc[2]));
      P = std::max(P, cfg->min_pres);
      for (int d = 0; d < 3; ++d) {
        int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
        double w[7] = { rho, v[d], v[t1], v[t2], P, Bc[t1], Bc[t2] };
        smax = std::max(smax, std::fabs(v[d]) + fastspeed(w, Bc[d], gam));
      }
    }
  }
  if (maxspeed_out) *maxspeed_out = smax;
  *dt_out = cfl * dh / smax;
  return 0;
}

// ---- unit entry points for the pins (tests only) ----
int mhdref_riemann(int solver, const double* WL, const double* WR, double Bn, double gamma, double* F) { return riemann(solver, WL, WR, Bn, gamma, F); }
// Roe flux with every dissipation speed raised to at least etah (R19), and the eta of a face
int mhdref_roe_eta(const double* WL, const double* WR, double Bn, double gamma, double etah, double* F) { return roe(WL, WR, Bn, gamma, F, etah); }
double mhdref_eta_face(const double* WL, const double* WR, double Bn, double gamma) { return eta_face(WL, WR, Bn, gamma); }
void mhdref_prim2cons(const double* W, double Bn, double gamma, double* U) { prim2cons(W, Bn, gamma, U); }
void mhdref_physflux(const double* W, double Bn, double gamma, double* F) { double U[7]; prim2cons(W, Bn, gamma, U); physflux(W, Bn, U, F); }
double mhdref_fastspeed(const double* W, double Bn, double gamma) { return fastspeed(W, Bn, gamma); }
void mhdref_eig_prim(const double* W, double Bn, double gamma, double* lam, double* R, double* L, double* A) {
  double r[7][7], l[7][7], a[7][7];
  eig_prim(W, Bn, gamma, lam, r, l); primA(W, Bn, gamma, a);
  std::memcpy(R, r, sizeof r); std::memcpy(L, l, sizeof l); std::memcpy(A, a, sizeof a);
}
// Roe-average eigen-system; Uavg[9] = (rho, vn, v1, v2, H, B1, B2, X, a2).  returns -1 if a2 <= 0
int mhdref_eig_roe(const double* WL, const double* WR, double Bn, double gamma, double* lam, double* R, double* L, double* avg) {
  RoeAvg r = roe_average(WL, WR, Bn, gamma);
  double a[9] = { r.rho, r.vn, r.v1, r.v2, r.H, r.B1, r.B2, r.X, r.a2 };
  std::memcpy(avg, a, sizeof a);
  if (!(r.a2 > 0.0)) return -1;
  double rr[7][7], ll[7][7];
  eig_cons(r, Bn, gamma, lam, rr, ll);
  std::memcpy(R, rr, sizeof rr); std::memcpy(L, ll, sizeof ll);
  return 0;
}
// R10a unit entry points: the CT upwind switch (tie = emf_tie * dh / dt) and the C6 edge formula
double mhdref_emf_up(double m, double rm, double rp, double qm, double qp, double tie) { return emf_upwind(tie, m, rm, rp, qm, qp); }
double mhdref_edge_emf(const double* Eface /*Ea_lo, Ea_hi, Eb_lo, Eb_hi*/, const double* mface /*same order*/, const double* ec, const double* rho, double tie) {
  return edge_emf_formula(Eface[0], Eface[1], Eface[2], Eface[3], mface[0], mface[1], mface[2], mface[3], ec, rho, tie);
}
double mhdref_mc(double a, double b) { return mc(a, b); }
// slope limiter by index (0 MC, 1 minmod, 2 van Leer), for the limiter pins
double mhdref_limiter(int which, double a, double b) { return which == 1 ? mm(a, b) : (which == 2 ? vanleer(a, b) : mc(a, b)); }
}

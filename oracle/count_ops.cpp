// count_ops.cpp -- TEST / MEASUREMENT INFRASTRUCTURE ONLY.  Instantiates the oracle (mhd_oracle.cpp, unchanged) with an
// operation-counting scalar in place of `double` and prints the exact number of floating-point operations the
// algorithm, as the oracle states it, performs: per Riemann solve and per patch group.  These are the "algorithmic
// flops" of bench.py's ALU roofline; add, subtract, multiply, divide and square root count 1 each,
// comparisons / min / max / fabs are listed separately and not counted as flops.
//
// Build + run:  g++ -O1 -std=c++17 -o /tmp/count_ops oracle/count_ops.cpp && /tmp/count_ops
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <limits>
#include <vector>

typedef double real_t;
struct Tally { unsigned long long add = 0, mul = 0, div = 0, sqrt = 0, cmp = 0; };
static Tally g_t;

struct Counted {
  real_t v;
  Counted() : v(0) {}
  Counted(real_t x) : v(x) {}
  Counted(int x) : v(x) {}
  explicit operator real_t() const { return v; }
};
#define BINOP(op, field)                                                                             \
  inline Counted operator op(Counted a, Counted b) { g_t.field++; return Counted(a.v op b.v); }      \
  inline Counted operator op(Counted a, real_t b) { g_t.field++; return Counted(a.v op b); }         \
  inline Counted operator op(real_t a, Counted b) { g_t.field++; return Counted(a op b.v); }
BINOP(+, add) BINOP(-, add) BINOP(*, mul) BINOP(/, div)
#define CMPOP(op)                                                                 \
  inline bool operator op(Counted a, Counted b) { g_t.cmp++; return a.v op b.v; } \
  inline bool operator op(Counted a, real_t b) { g_t.cmp++; return a.v op b; }    \
  inline bool operator op(real_t a, Counted b) { g_t.cmp++; return a op b.v; }
CMPOP(<) CMPOP(>) CMPOP(<=) CMPOP(>=) CMPOP(==) CMPOP(!=)
inline Counted operator-(Counted a) { return Counted(-a.v); }
inline Counted& operator+=(Counted& a, Counted b) { g_t.add++; a.v += b.v; return a; }
inline Counted& operator-=(Counted& a, Counted b) { g_t.add++; a.v -= b.v; return a; }
inline Counted& operator*=(Counted& a, Counted b) { g_t.mul++; a.v *= b.v; return a; }
namespace std {
inline Counted sqrt(Counted a) { g_t.sqrt++; return Counted(std::sqrt(a.v)); }
inline Counted fabs(Counted a) { g_t.cmp++; return Counted(std::fabs(a.v)); }
inline Counted min(real_t a, Counted b) { g_t.cmp++; return Counted(a < b.v ? a : b.v); }
inline Counted min(Counted a, real_t b) { g_t.cmp++; return Counted(b < a.v ? b : a.v); }
inline Counted max(real_t a, Counted b) { g_t.cmp++; return Counted(a < b.v ? b.v : a); }
inline Counted max(Counted a, real_t b) { g_t.cmp++; return Counted(a.v < b ? b : a.v); }
template <> struct numeric_limits<Counted> { static Counted quiet_NaN() { return Counted(numeric_limits<real_t>::quiet_NaN()); } };
}  // namespace std

#define double Counted
#include "mhd_oracle.cpp"
#undef double

static Tally diff(const Tally& a, const Tally& b) { Tally d; d.add = a.add - b.add; d.mul = a.mul - b.mul; d.div = a.div - b.div; d.sqrt = a.sqrt - b.sqrt; d.cmp = a.cmp - b.cmp; return d; }
static void show(const char* what, const Tally& t, double per) {
  const double fl = (double)(t.add + t.mul + t.div + t.sqrt);
  std::printf("%-44s flops %12.1f  (add %.1f mul %.1f div %.1f sqrt %.1f; cmp/abs %.1f)\n", what, fl / per, t.add / per, t.mul / per,
              t.div / per, t.sqrt / per, t.cmp / per);
}

int main() {
  const real_t gam = 5.0 / 3.0;
  // a generic subsonic pair (double-star region of HLLD, no Roe fallback): the common case of every config
  Counted WL[7] = { 1.0, 0.10, -0.05, 0.07, 0.9, 0.6, -0.4 }, WR[7] = { 1.1, 0.05, 0.02, -0.03, 1.0, 0.5, -0.3 }, F[7];
  const char* names[3] = { "HLLE", "HLLD", "Roe" };
  for (int sol = 0; sol < 3; ++sol) {
    Tally t0 = g_t;
    mhdref_riemann(sol, WL, WR, Counted(0.7), Counted(gam), F);
    char buf[64]; std::snprintf(buf, sizeof buf, "per Riemann solve, %s", names[sol]);
    show(buf, diff(g_t, t0), 1.0);
  }
  // whole patch group, smooth seeded state (no floors), per interior cell-update; on the oracle's maximal index ranges and on the
  // minimal ones (every stage only where the final update needs it: the work the method itself requires, mhdref_config.minimal_ranges),
  // with the flops of each step (hook after every step of the group's update)
  struct V { const char* name; int scheme, recon, riemann, limvar, g; } vars[] = {
    { "VL+PLM+HLLD (g=3)", 0, 0, 1, 0, 3 }, { "VL+PLM+Roe (g=3)", 0, 0, 2, 0, 3 },
    { "CTU+PLM+HLLD char (g=3)", 1, 0, 1, 1, 3 }, { "CTU+PPM+HLLD char (g=4)", 1, 1, 1, 1, 4 },
    { "CTU+PPM+Roe char (g=4)", 1, 1, 2, 1, 4 } };
  const int N = 16;
  static Tally marks[8];
  mhdref_stage_hook = [](int n) { if (n >= 0 && n < 8) marks[n] = g_t; };
  const char* steps[8] = { "", "con->prim", "pass-1 fluxes (+ CTU reconstruction)", "EMF-1", "half step", "pass-2 states + fluxes", "EMF-2", "full update" };
  for (const V& v : vars) for (int mn = 0; mn < 2; ++mn) {
    const int T = N + 2 * v.g;
    mhdref_config cfg; cfg.ps2 = N; cfg.nghost = v.g; cfg.gamma = Counted(gam); cfg.scheme = v.scheme; cfg.recon = v.recon;
    cfg.riemann = v.riemann; cfg.limvar = v.limvar; cfg.min_dens = Counted(1e-10); cfg.min_pres = Counted(1e-10); cfg.emf_tie = Counted(1e-12); cfg.limiter = 0;
    cfg.minimal_ranges = mn; cfg.hcorr = 0;
    std::vector<Counted> U(5 * T * T * T), B(3 * T * T * (T + 1)), Uo(5 * N * N * N), Bo(3 * N * N * (N + 1)), fo(9 * 5 * N * N), eo(9 * 2 * (N + 1) * N);
    const real_t k = 2.0 * 3.14159265358979323846 / N;
    for (int kk = 0; kk < T; ++kk) for (int j = 0; j < T; ++j) for (int i = 0; i < T; ++i) {
      const size_t q = ((size_t)kk * T + j) * T + i, T3 = (size_t)T * T * T;
      const real_t rho = 1.0 + 0.2 * std::sin(k * i) * std::cos(k * j), vx = 0.2 * std::sin(k * j), vy = 0.1 * std::cos(k * kk), vz = 0.15 * std::sin(k * i);
      U[q] = Counted(rho); U[T3 + q] = Counted(rho * vx); U[2 * T3 + q] = Counted(rho * vy); U[3 * T3 + q] = Counted(rho * vz);
      U[4 * T3 + q] = Counted(1.0 / (gam - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (0.36 + 0.25 + 0.16));
    }
    const size_t nf = (size_t)T * T * (T + 1);
    for (size_t q = 0; q < nf; ++q) { B[q] = Counted(0.6); B[nf + q] = Counted(0.5); B[2 * nf + q] = Counted(-0.4); }
    unsigned long long st[3] = { 0, 0, 0 };
    Tally t0 = g_t;
    mhdref_advance(&cfg, U.data(), B.data(), Uo.data(), Bo.data(), fo.data(), eo.data(), 1, Counted(0.01), Counted(1.0 / N), st, 0);
    char buf[96]; std::snprintf(buf, sizeof buf, "%s, %s ranges, per cell-update", v.name, mn ? "minimal" : "maximal");
    show(buf, diff(g_t, t0), (double)N * N * N);
    for (int n = 1; n < 8; ++n) {
      const Tally d = diff(marks[n], marks[n - 1]);
      std::printf("    step %d %-40s flops per group %12llu\n", n, steps[n], d.add + d.mul + d.div + d.sqrt);
    }
  }
  return 0;
}

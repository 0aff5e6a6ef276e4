// mhd_oracle_f32.cpp -- TEST INFRASTRUCTURE ONLY.  The oracle (mhd_oracle.cpp, unchanged, included below) instantiated
// in single precision: `double` is replaced by a scalar that holds a float and rounds EVERY operation to float (IEEE
// round-to-nearest add, subtract, multiply, divide, square root; literals are rounded to float first).  Same trick as
// count_ops.cpp.  It is the control experiment of DESIGN.md section 9: oracle-FP32 against oracle-FP64 is the error that
// the plain algorithm itself has in single precision (single precision is the paper's headline mode),
// which is what the FP32 parity gates of the CUDA path are measured against.  The FP64 library stays the checker.
//
// Build: g++ -O2 -fno-fast-math -ffp-contract=off -fopenmp -shared -fPIC -o libmhdref_f32.so mhd_oracle_f32.cpp
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstring>
#include <limits>
#include <vector>

struct F32 {
  float v;
  F32() : v(0.0f) {}
  F32(double x) : v((float)x) {}
  F32(float x) : v(x) {}
  F32(int x) : v((float)x) {}
  explicit operator float() const { return v; }
};
#define F32_BINOP(op)                                                              \
  inline F32 operator op(F32 a, F32 b) { return F32(a.v op b.v); }                 \
  inline F32 operator op(F32 a, double b) { return F32(a.v op (float)b); }         \
  inline F32 operator op(double a, F32 b) { return F32((float)a op b.v); }
F32_BINOP(+) F32_BINOP(-) F32_BINOP(*) F32_BINOP(/)
#define F32_CMPOP(op)                                                              \
  inline bool operator op(F32 a, F32 b) { return a.v op b.v; }                     \
  inline bool operator op(F32 a, double b) { return a.v op (float)b; }             \
  inline bool operator op(double a, F32 b) { return (float)a op b.v; }
F32_CMPOP(<) F32_CMPOP(>) F32_CMPOP(<=) F32_CMPOP(>=) F32_CMPOP(==) F32_CMPOP(!=)
inline F32 operator-(F32 a) { return F32(-a.v); }
inline F32& operator+=(F32& a, F32 b) { a.v = a.v + b.v; return a; }
inline F32& operator-=(F32& a, F32 b) { a.v = a.v - b.v; return a; }
inline F32& operator*=(F32& a, F32 b) { a.v = a.v * b.v; return a; }
namespace std {
inline F32 sqrt(F32 a) { return F32(sqrtf(a.v)); }
inline F32 fabs(F32 a) { return F32(fabsf(a.v)); }
inline F32 min(double a, F32 b) { return F32((float)a < b.v ? (float)a : b.v); }
inline F32 min(F32 a, double b) { return F32((float)b < a.v ? (float)b : a.v); }
inline F32 max(double a, F32 b) { return F32((float)a < b.v ? b.v : (float)a); }
inline F32 max(F32 a, double b) { return F32(a.v < (float)b ? (float)b : a.v); }
template <> struct numeric_limits<F32> { static F32 quiet_NaN() { return F32(numeric_limits<float>::quiet_NaN()); } };
}  // namespace std

#define double F32
#include "mhd_oracle.cpp"
#undef double

// plain-C entry points (float arrays, double scalars) so that the binding does not depend on how F32 is passed by value
extern "C" {
typedef struct {
  int ps2, nghost; double gamma; int scheme, recon, riemann, limvar; double min_dens, min_pres, emf_tie; int limiter, minimal_ranges, hcorr;
} mhdref32_config;

static mhdref_config to_f32_cfg(const mhdref32_config* c) {
  mhdref_config k;
  k.ps2 = c->ps2; k.nghost = c->nghost; k.gamma = F32(c->gamma); k.scheme = c->scheme; k.recon = c->recon; k.riemann = c->riemann;
  k.limvar = c->limvar; k.min_dens = F32(c->min_dens); k.min_pres = F32(c->min_pres); k.emf_tie = F32(c->emf_tie); k.limiter = c->limiter; k.minimal_ranges = c->minimal_ranges; k.hcorr = c->hcorr;
  return k;
}
int mhdref32_advance(const mhdref32_config* cfg, const float* U_in, const float* B_in, float* U_out, float* B_out, float* flux_out,
                     float* emf_out, int ngroups, double dt, double dh, unsigned long long* stats, int force_ghost_ok) {
  static_assert(sizeof(F32) == sizeof(float), "F32 must be layout-compatible with float");
  if (!cfg) return -1;
  const mhdref_config k = to_f32_cfg(cfg);
  return mhdref_advance(&k, reinterpret_cast<const F32*>(U_in), reinterpret_cast<const F32*>(B_in), reinterpret_cast<F32*>(U_out),
                        reinterpret_cast<F32*>(B_out), reinterpret_cast<F32*>(flux_out), reinterpret_cast<F32*>(emf_out), ngroups,
                        F32(dt), F32(dh), stats, force_ghost_ok);
}
int mhdref32_dt(const mhdref32_config* cfg, const float* U, const float* B, int ngroups, int ng, double dh, double cfl, double* dt_out,
                double* maxspeed_out) {
  if (!cfg || !dt_out) return -1;
  const mhdref_config k = to_f32_cfg(cfg);
  F32 dt, sm;
  const int rc = mhdref_dt(&k, reinterpret_cast<const F32*>(U), reinterpret_cast<const F32*>(B), ngroups, ng, F32(dh), F32(cfl), &dt, &sm);
  *dt_out = dt.v;
  if (maxspeed_out) *maxspeed_out = sm.v;
  return rc;
}
}

// sanitize_main.cpp -- TEST INFRASTRUCTURE ONLY.  The oracle (mhd_oracle.cpp, unchanged, included below) under the address and
// undefined-behaviour sanitizers: every scheme / reconstruction / solver combination on two patch groups of
// a smooth seeded state with a shock-like jump, plus mhdref_dt.  Exit code 0 and no sanitizer report = clean.
//
//   g++ -std=c++17 -O1 -g -fsanitize=address,undefined -fno-sanitize-recover=all -o /tmp/oracle_san oracle/sanitize_main.cpp && /tmp/oracle_san
#include <cstdio>
#include "mhd_oracle.cpp"

int main() {
  const double gam = 5.0 / 3.0;
  int runs = 0;
  for (int scheme = 0; scheme < 2; ++scheme) for (int recon = 0; recon < 2; ++recon) for (int riemann = 0; riemann < 3; ++riemann)
    for (int limvar = 0; limvar < 2; ++limvar) for (int mn = 0; mn < 2; ++mn) {
      const int N = 8, g = recon ? 4 : 3, T = N + 2 * g, G = 2;
      mhdref_config cfg; cfg.ps2 = N; cfg.nghost = g; cfg.gamma = gam; cfg.scheme = scheme; cfg.recon = recon; cfg.riemann = riemann;
      cfg.limvar = limvar; cfg.min_dens = 1e-10; cfg.min_pres = 1e-10; cfg.emf_tie = (riemann == 1 ? 1e-5 : 1e-12); cfg.limiter = (riemann + recon) % 3;
      cfg.minimal_ranges = mn; cfg.hcorr = 0;
      const size_t T3 = (size_t)T * T * T, nf = (size_t)T * T * (T + 1);
      std::vector<double> U(G * 5 * T3), B(G * 3 * nf), Uo(G * 5 * N * N * N), Bo(G * 3 * N * N * (N + 1)), fo(G * 9 * 5 * N * N), eo(G * 9 * 2 * (N + 1) * N);
      const double k = 2.0 * 3.14159265358979323846 / N;
      for (int gi = 0; gi < G; ++gi) {
        for (int kk = 0; kk < T; ++kk) for (int j = 0; j < T; ++j) for (int i = 0; i < T; ++i) {
          const size_t q = ((size_t)kk * T + j) * T + i;
          const double jump = (i + gi > T / 2) ? 3.0 : 1.0;             // a pressure jump: exercises the limiters and solver branches
          const double rho = 1.0 + 0.3 * std::sin(k * i) * std::cos(k * j), vx = 0.4 * std::sin(k * j), vy = -0.2 * std::cos(k * kk), vz = 0.3 * std::sin(k * i);
          double* u = &U[gi * 5 * T3];
          u[q] = rho; u[T3 + q] = rho * vx; u[2 * T3 + q] = rho * vy; u[3 * T3 + q] = rho * vz;
          u[4 * T3 + q] = jump / (gam - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (0.36 + 0.25 + 0.16);
        }
        for (size_t q = 0; q < nf; ++q) { B[gi * 3 * nf + q] = 0.6; B[gi * 3 * nf + nf + q] = 0.5; B[gi * 3 * nf + 2 * nf + q] = -0.4; }
      }
      unsigned long long st[3] = { 0, 0, 0 };
      double dt = 0, sm = 0;
      if (mhdref_dt(&cfg, U.data(), B.data(), G, g, 1.0 / N, 0.3, &dt, &sm)) return 2;
      if (mhdref_advance(&cfg, U.data(), B.data(), Uo.data(), Bo.data(), fo.data(), eo.data(), G, dt, 1.0 / N, st, 0)) return 3;
      for (double x : Uo) if (!(x == x)) return 4;
      for (double x : eo) if (!(x == x)) return 5;
      ++runs;
    }
  std::printf("oracle under -fsanitize=address,undefined: %d runs clean\n", runs);
  return 0;
}

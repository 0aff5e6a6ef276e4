// mhd_amr.cuh -- the AMR correction operation on a static two-level mesh:
//   * restriction: coarse cells / faces covered by fine patch groups <- volume / area average of the fine data;
//   * flux fix-up: a leaf coarse cell next to the coarse-fine interface trades the coarse flux it was updated with
//     for the area average of the fine fluxes on that face;
//   * EMF fix-up: a leaf coarse face touching a coarse-fine inter-edge trades the coarse edge EMF for the mean of the two
//     fine edge EMFs, so that the discrete divergence (Eq. 16) of the corrected coarse grid stays at round-off.
// The consumers of flux_out / emf_out (include/mhd.h).  One refined box per call: coarse cells lo..hi-1 per axis,
// multiples of ps2/2, strictly inside the periodic domain; fine groups ordered z outermost, x fastest.
#pragma once
#include "mhd_kernels.cuh"

namespace mhd {

// three integers selected by axis with compares (no dynamically indexed local arrays: everything stays in registers)
struct I3 {
  int x, y, z;
  __host__ __device__ __forceinline__ int operator[](int d) const { return d == 0 ? x : (d == 1 ? y : z); }
  __host__ __device__ __forceinline__ void set(int d, int v) { if (d == 0) x = v; else if (d == 1) y = v; else z = v; }
};

struct Amr {
  I3 n;            // coarse grid cells per axis (x, y, z)
  I3 mg;           // coarse patch groups per axis
  I3 lo, hi;
  I3 mf;           // fine patch groups per axis of the box
  int N, h;        // ps2 and ps2 / 2 (coarse cells covered by one fine group per axis)
};

// group, plane slot and in-group position of a point on the coarse plane with normal d through coarse index pos[d]
__host__ __device__ __forceinline__ void coarse_plane(const Amr& a, const I3& pos, int d, int& grp, int& slot, I3& loc) {
  const I3 g = { pos.x / a.N, pos.y / a.N, pos.z / a.N };
  loc = { pos.x - g.x * a.N, pos.y - g.y * a.N, pos.z - g.z * a.N };
  slot = 3 * d + (loc[d] == 0 ? 0 : 1);              // the plane is a group boundary (0) or its mid plane (ps2/2)
  grp = (g.z * a.mg.y + g.y) * a.mg.x + g.x;
}
// fine group on the box surface (normal d; side 0 = lower, 1 = upper), its plane slot and the fine in-group position of
// coarse position pos (cells along an axis map to their first fine cell, the far rim to fine index ps2)
__host__ __device__ __forceinline__ void fine_plane(const Amr& a, const I3& pos, int d, int side, int& grp, int& slot, I3& f) {
  I3 g;
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    int gg, ff;
    if (ax == d) { gg = side ? a.mf[ax] - 1 : 0; ff = 0; }
    else {
      const int rel = pos[ax] - a.lo[ax], nb = a.hi[ax] - a.lo[ax];
      const int rc = rel < 0 ? 0 : (rel > nb - 1 ? nb - 1 : rel);
      gg = rc / a.h;
      ff = 2 * (rel - gg * a.h);
    }
    g.set(ax, gg); f.set(ax, ff);
  }
  slot = 3 * d + (side ? 2 : 0);
  grp = (g.z * a.mf.y + g.y) * a.mf.x + g.x;
}

// ---- restriction: one thread per point of the (nb+1)^3 lattice of the box (cell + its three lower faces) ----------
template <class R>
__global__ void __launch_bounds__(256) k_amr_restrict(const R* __restrict__ Uf, const R* __restrict__ Bf, Amr a,
                                                      R* __restrict__ Uc, R* __restrict__ bxc, R* __restrict__ byc, R* __restrict__ bzc) {
  const int nbx = a.hi.x - a.lo.x, nby = a.hi.y - a.lo.y, nbz = a.hi.z - a.lo.z;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (nbx + 1) * (nby + 1) * (nbz + 1)) return;
  const int i = t % (nbx + 1), j = (t / (nbx + 1)) % (nby + 1), k = t / ((nbx + 1) * (nby + 1));
  const int N = a.N, h = a.h;
  // fine group holding the point (the far rim belongs to the last group) and fine in-group index of the point
  const int gx = i / h < a.mf.x ? i / h : a.mf.x - 1, gy = j / h < a.mf.y ? j / h : a.mf.y - 1, gz = k / h < a.mf.z ? k / h : a.mf.z - 1;
  const int fi = 2 * (i - gx * h), fj = 2 * (j - gy * h), fk = 2 * (k - gz * h);
  const size_t grp = ((size_t)gz * a.mf.y + gy) * a.mf.x + gx;
  const size_t N3 = (size_t)N * N * N, nf = (size_t)N * N * (N + 1);
  const R* U = Uf + grp * 5 * N3;
  const R* Bx = Bf + grp * 3 * nf;
  const R* By = Bx + nf;
  const R* Bz = By + nf;
  const int X = a.lo.x + i, Y = a.lo.y + j, Z = a.lo.z + k;
  const size_t n3 = (size_t)a.n.x * a.n.y * a.n.z;
  if (i < nbx && j < nby && k < nbz) {
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      R sum = R(0);
#pragma unroll
      for (int c = 0; c < 8; ++c) sum += U[v * N3 + ((size_t)(fk + (c >> 2)) * N + fj + ((c >> 1) & 1)) * N + fi + (c & 1)];
      Uc[v * n3 + ((size_t)Z * a.n.y + Y) * a.n.x + X] = R(0.125) * sum;
    }
  }
  if (j < nby && k < nbz) {
    R sum = R(0);
#pragma unroll
    for (int c = 0; c < 4; ++c) sum += Bx[((size_t)(fk + (c >> 1)) * N + fj + (c & 1)) * (N + 1) + fi];
    bxc[((size_t)Z * a.n.y + Y) * (a.n.x + 1) + X] = R(0.25) * sum;
  }
  if (i < nbx && k < nbz) {
    R sum = R(0);
#pragma unroll
    for (int c = 0; c < 4; ++c) sum += By[((size_t)(fk + (c >> 1)) * (N + 1) + fj) * N + fi + (c & 1)];
    byc[((size_t)Z * (a.n.y + 1) + Y) * a.n.x + X] = R(0.25) * sum;
  }
  if (i < nbx && j < nby) {
    R sum = R(0);
#pragma unroll
    for (int c = 0; c < 4; ++c) sum += Bz[((size_t)fk * N + fj + (c >> 1)) * N + fi + (c & 1)];
    bzc[((size_t)Z * a.n.y + Y) * a.n.x + X] = R(0.25) * sum;
  }
}

// ---- flux fix-up: one thread per coarse face of the box surface ------------------------------------------------------
template <class R>
__global__ void __launch_bounds__(256) k_amr_flux_fixup(const R* __restrict__ flux_c, const R* __restrict__ flux_f, Amr a, R q, R wc, R wf,
                                                        R* __restrict__ Uc) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  const I3 nb = { a.hi.x - a.lo.x, a.hi.y - a.lo.y, a.hi.z - a.lo.z };
  int d = 0;
  for (; d < 3; ++d) {
    const int cnt = 2 * nb[(d + 1) % 3] * nb[(d + 2) % 3];
    if (t < cnt) break;
    t -= cnt;
  }
  if (d == 3) return;
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  const int side = t / (nb[t1] * nb[t2]), r = t - side * nb[t1] * nb[t2];
  I3 pos;
  pos.set(d, side ? a.hi[d] : a.lo[d]);
  pos.set(t1, a.lo[t1] + r % nb[t1]);
  pos.set(t2, a.lo[t2] + r / nb[t1]);
  const int N = a.N;
  int gc, sc, gf, sf;
  I3 loc, f;
  coarse_plane(a, pos, d, gc, sc, loc);
  fine_plane(a, pos, d, side, gf, sf, f);
  const size_t NN = (size_t)N * N;
  const R* Fc = flux_c + ((size_t)gc * 9 + sc) * 5 * NN + (size_t)loc[t2] * N + loc[t1];
  const R* Ff = flux_f + ((size_t)gf * 9 + sf) * 5 * NN + (size_t)f[t2] * N + f[t1];
  I3 cell = pos;
  if (side == 0) cell.set(d, pos[d] - 1);          // the leaf cell outside the box
  // lower side: the face is the leaf cell's UPPER face (it entered Eq. 10 with -q F); upper side: its LOWER face (+q F)
  const R sgn = side ? R(1) : R(-1);
  const size_t n3 = (size_t)a.n.x * a.n.y * a.n.z, ci = ((size_t)cell.z * a.n.y + cell.y) * a.n.x + cell.x;
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    const R fine = R(0.25) * (Ff[v * NN] + Ff[v * NN + 1] + Ff[v * NN + N] + Ff[v * NN + N + 1]);
    Uc[v * n3 + ci] += sgn * q * (wf * fine - wc * Fc[v * NN]);
  }
}

// ---- EMF fix-up: one thread per coarse face within one cell of the box; leaf faces touching the surface get corrected --
// w_f <fine EMF> - w_c (coarse EMF) of the coarse edge along c whose lower end is the lattice point e; 0 off the surface
template <class R>
__host__ __device__ __forceinline__ R emf_jump(const R* __restrict__ emf_c, const R* __restrict__ emf_f, const Amr& a, int c, const I3& e, R wc, R wf) {
  const int A = (c + 1) % 3, B = (c + 2) % 3;
  const int ec = e[c], eA = e[A], eB = e[B];
  if (ec < a.lo[c] || ec >= a.hi[c]) return R(0);
  int dn = -1;
  if ((eA == a.lo[A] || eA == a.hi[A]) && eB >= a.lo[B] && eB <= a.hi[B]) dn = A;
  else if ((eB == a.lo[B] || eB == a.hi[B]) && eA >= a.lo[A] && eA <= a.hi[A]) dn = B;
  if (dn < 0) return R(0);                          // not an edge of the box surface
  const int side = e[dn] == a.lo[dn] ? 0 : 1, t1 = (dn + 1) % 3, t2 = (dn + 2) % 3, N = a.N, M = N + 1;
  int gc, sc, gf, sf;
  I3 loc, f;
  coarse_plane(a, e, dn, gc, sc, loc);
  fine_plane(a, e, dn, side, gf, sf, f);
  const R* Ec = emf_c + ((size_t)gc * 9 + sc) * 2 * M * N;
  const R* Ef = emf_f + ((size_t)gf * 9 + sf) * 2 * M * N;
  const int l1 = loc[t1], l2 = loc[t2], f1 = f[t1], f2 = f[t2];
  R coarse, fine;
  if (c == t1) {       // edge along t1 at t2 - 1/2: component 0, [t2 edge][t1 cell]
    coarse = Ec[(size_t)l2 * N + l1];
    fine = R(0.5) * (Ef[(size_t)f2 * N + f1] + Ef[(size_t)f2 * N + f1 + 1]);
  } else {             // edge along t2 at t1 - 1/2: component 1, [t2 cell][t1 edge]
    Ec += (size_t)M * N; Ef += (size_t)M * N;
    coarse = Ec[(size_t)l2 * M + l1];
    fine = R(0.5) * (Ef[(size_t)f2 * M + f1] + Ef[(size_t)(f2 + 1) * M + f1]);
  }
  return wf * fine - wc * coarse;
}

template <class R>
__global__ void __launch_bounds__(256) k_amr_emf_fixup(const R* __restrict__ emf_c, const R* __restrict__ emf_f, Amr a, R q, R wc, R wf,
                                                       R* __restrict__ bxc, R* __restrict__ byc, R* __restrict__ bzc) {
  const int ex = a.hi.x - a.lo.x + 3, ey = a.hi.y - a.lo.y + 3, ez = a.hi.z - a.lo.z + 3;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ex * ey * ez) return;
  const int D = blockIdx.y;                          // direction of the face
  const I3 pos = { a.lo.x - 1 + t % ex, a.lo.y - 1 + (t / ex) % ey, a.lo.z - 1 + t / (ex * ey) };
  bool closure = true;                                // faces inside the box or on its surface are owned by the restriction
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) closure = closure && pos[ax] >= a.lo[ax] && (ax == D ? pos[ax] <= a.hi[ax] : pos[ax] < a.hi[ax]);
  if (closure) return;
  const int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  // Eq. 13 for the lower D-face of cell pos:  b -= q [ (E_T2(T1+) - E_T2(T1-)) - (E_T1(T2+) - E_T1(T2-)) ]
  R corr = R(0);
  {
    I3 e = pos;
    corr -= emf_jump(emf_c, emf_f, a, T2, e, wc, wf);
    e.set(T1, pos[T1] + 1);
    corr += emf_jump(emf_c, emf_f, a, T2, e, wc, wf);
  }
  {
    I3 e = pos;
    corr += emf_jump(emf_c, emf_f, a, T1, e, wc, wf);
    e.set(T2, pos[T2] + 1);
    corr -= emf_jump(emf_c, emf_f, a, T1, e, wc, wf);
  }
  if (corr == R(0)) return;
  R* b = D == 0 ? bxc : (D == 1 ? byc : bzc);
  const size_t idx = D == 0 ? ((size_t)pos.z * a.n.y + pos.y) * (a.n.x + 1) + pos.x
                   : D == 1 ? ((size_t)pos.z * (a.n.y + 1) + pos.y) * a.n.x + pos.x
                            : ((size_t)pos.z * a.n.y + pos.y) * a.n.x + pos.x;
  b[idx] -= q * corr;
}

}  // namespace mhd

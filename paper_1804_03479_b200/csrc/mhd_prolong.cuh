// mhd_prolong.cuh -- creating new fine grids: conservative interpolation of the
// cell-centred conserved variables and the divergence-free interpolation of Balsara (2001) for the face-centred field,
// the paper's 2-D example (Eq. 17: 10 coefficients, 11 conditions) carried to 3-D.
//
// Per coarse cell, in units of its size and centred on it, the field is the polynomial (one more axis)
//     Bx = a0 + ax x + ay y + az z + axx x^2 + axy x y + axz x z      (By, Bz: cyclic)
// The paper solves for the coefficients from the interface conditions and the divergence conditions.  In closed form
// (face values b(d, -+) on the lower / upper d-face, their limited in-face slopes s_t(d, -+) along t):
//     interface conditions (the profile on a coarse face is linear):
//         ax = b(x,+) - b(x,-),  ay = (s_y(x,+) + s_y(x,-))/2,  axy = s_y(x,+) - s_y(x,-),  az, axz alike,
//         a0 + axx/4 = (b(x,+) + b(x,-))/2
//     divergence conditions (the constant one, ax + by + cz = 0, holds because the coarse field is
//     divergence-free):  2 axx + bxy + cxz = 0  (coefficient of x), cyclic
// The second-set fine faces (the interior ones) lie on x = 0: the area average of a0 + ay y + az z over a
// fine face is its value at the face centre (y, z) = (-+1/4, -+1/4).  The first-set fine faces (on the coarse faces) are
// the linear profile at their centres.  Slopes: the MC limiter of the solver (R5), neighbours periodic.
#pragma once
#include "mhd_amr.cuh"
#include "mhd_grid.cuh"   // wrap()

namespace mhd {

template <class R> __device__ __forceinline__ R mc_slope(R dl, R dr) {     // MC(a, b) of DESIGN.md R5 (a = left difference)
  if (dl * dr <= R(0)) return R(0);
  const R s = dl + dr, a = Num<R>::abs(s) * R(0.5), b = R(2) * Num<R>::abs(dl), c = R(2) * Num<R>::abs(dr);
  const R m = a < b ? (a < c ? a : c) : (b < c ? b : c);
  return s > R(0) ? m : -m;
}

struct ProlongGeom {
  I3 n;        // coarse grid cells per axis
  I3 lo, hi;   // refined box of coarse cells lo..hi-1
};

// value and the two limited in-face slopes of the coarse D-face at lattice position (X, Y, Z) (periodic)
template <class R, int D>
__device__ __forceinline__ void coarse_face(const R* __restrict__ b, const ProlongGeom& g, int X, int Y, int Z, R& val, R& s1, R& s2) {
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  const int nx = g.n.x + (D == 0), ny = g.n.y + (D == 1);
  // the face array holds n+1 faces along its own normal (last = first); cells wrap along the in-face axes
  auto at = [&](int x, int y, int z) {
    x = D == 0 ? x : wrap(x, g.n.x); y = D == 1 ? y : wrap(y, g.n.y); z = D == 2 ? z : wrap(z, g.n.z);
    return b[((size_t)z * ny + y) * nx + x];
  };
  int p[3] = { X, Y, Z };
  val = at(p[0], p[1], p[2]);
  int q[3] = { X, Y, Z };
  q[T1] = p[T1] + 1; const R u1 = at(q[0], q[1], q[2]);
  q[T1] = p[T1] - 1; const R d1 = at(q[0], q[1], q[2]);
  q[T1] = p[T1];
  q[T2] = p[T2] + 1; const R u2 = at(q[0], q[1], q[2]);
  q[T2] = p[T2] - 1; const R d2 = at(q[0], q[1], q[2]);
  s1 = mc_slope(val - d1, u1 - val);
  s2 = mc_slope(val - d2, u2 - val);
}

// one thread per point of the (nb+1)^3 lattice of the box: the coarse cell (if inside) and its three lower faces
template <class R>
__global__ void __launch_bounds__(128) k_amr_prolong(const R* __restrict__ Uc, const R* __restrict__ bxc, const R* __restrict__ byc,
                                                     const R* __restrict__ bzc, ProlongGeom g, R* __restrict__ Uf, R* __restrict__ bxf,
                                                     R* __restrict__ byf, R* __restrict__ bzf) {
  const int nbx = g.hi.x - g.lo.x, nby = g.hi.y - g.lo.y, nbz = g.hi.z - g.lo.z;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (nbx + 1) * (nby + 1) * (nbz + 1)) return;
  const int i = t % (nbx + 1), j = (t / (nbx + 1)) % (nby + 1), k = t / ((nbx + 1) * (nby + 1));
  const int X = g.lo.x + i, Y = g.lo.y + j, Z = g.lo.z + k;
  const int fx = 2 * nbx, fy = 2 * nby, fz = 2 * nbz;            // fine cells per axis
  const bool cell = i < nbx && j < nby && k < nbz;
  const R q = R(0.25);
  // lower faces: value, slopes; first-set fine faces
  R vx0 = R(0), sxy0 = R(0), sxz0 = R(0), vy0 = R(0), syz0 = R(0), syx0 = R(0), vz0 = R(0), szx0 = R(0), szy0 = R(0);
  if (j < nby && k < nbz) {
    coarse_face<R, 0>(bxc, g, X, Y, Z, vx0, sxy0, sxz0);           // slopes along y, z
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int oy = c & 1, oz = c >> 1;
      bxf[((size_t)(2 * k + oz) * fy + 2 * j + oy) * (fx + 1) + 2 * i] = vx0 + (oy ? q : -q) * sxy0 + (oz ? q : -q) * sxz0;
    }
  }
  if (i < nbx && k < nbz) {
    coarse_face<R, 1>(byc, g, X, Y, Z, vy0, syz0, syx0);           // slopes along z, x
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int oz = c & 1, ox = c >> 1;
      byf[((size_t)(2 * k + oz) * (fy + 1) + 2 * j) * fx + 2 * i + ox] = vy0 + (oz ? q : -q) * syz0 + (ox ? q : -q) * syx0;
    }
  }
  if (i < nbx && j < nby) {
    coarse_face<R, 2>(bzc, g, X, Y, Z, vz0, szx0, szy0);           // slopes along x, y
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int ox = c & 1, oy = c >> 1;
      bzf[((size_t)(2 * k) * fy + 2 * j + oy) * fx + 2 * i + ox] = vz0 + (ox ? q : -q) * szx0 + (oy ? q : -q) * szy0;
    }
  }
  if (!cell) return;
  // upper faces of the cell
  R vx1, sxy1, sxz1, vy1, syz1, syx1, vz1, szx1, szy1;
  coarse_face<R, 0>(bxc, g, X + 1, Y, Z, vx1, sxy1, sxz1);
  coarse_face<R, 1>(byc, g, X, Y + 1, Z, vy1, syz1, syx1);
  coarse_face<R, 2>(bzc, g, X, Y, Z + 1, vz1, szx1, szy1);
  // interface conditions
  const R ay = R(0.5) * (sxy1 + sxy0), axy = sxy1 - sxy0, az = R(0.5) * (sxz1 + sxz0), axz = sxz1 - sxz0;
  const R bz = R(0.5) * (syz1 + syz0), byz = syz1 - syz0, bx = R(0.5) * (syx1 + syx0), bxy = syx1 - syx0;
  const R cx = R(0.5) * (szx1 + szx0), cxz = szx1 - szx0, cy = R(0.5) * (szy1 + szy0), cyz = szy1 - szy0;
  // divergence conditions
  const R axx = -R(0.5) * (bxy + cxz), byy = -R(0.5) * (axy + cyz), czz = -R(0.5) * (axz + byz);
  const R a0 = R(0.5) * (vx1 + vx0) - q * axx, b0 = R(0.5) * (vy1 + vy0) - q * byy, c0 = R(0.5) * (vz1 + vz0) - q * czz;
  // second set: the interior fine faces
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const int o1 = c & 1, o2 = c >> 1;
    const R p1 = o1 ? q : -q, p2 = o2 ? q : -q;
    bxf[((size_t)(2 * k + o2) * fy + 2 * j + o1) * (fx + 1) + 2 * i + 1] = a0 + ay * p1 + az * p2;        // (y, z) = (p1, p2)
    byf[((size_t)(2 * k + o1) * (fy + 1) + 2 * j + 1) * fx + 2 * i + o2] = b0 + bz * p1 + bx * p2;        // (z, x) = (p1, p2)
    bzf[((size_t)(2 * k + 1) * fy + 2 * j + o2) * fx + 2 * i + o1] = c0 + cx * p1 + cy * p2;              // (x, y) = (p1, p2)
  }
  // conserved variables: conservative piecewise-linear interpolation
  const size_t n3 = (size_t)g.n.x * g.n.y * g.n.z, f3 = (size_t)fx * fy * fz;
  const int xm = wrap(X - 1, g.n.x), xp = wrap(X + 1, g.n.x), ym = wrap(Y - 1, g.n.y), yp = wrap(Y + 1, g.n.y),
            zm = wrap(Z - 1, g.n.z), zp = wrap(Z + 1, g.n.z);
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    const R* u = Uc + v * n3;
    auto at = [&](int x, int y, int z) { return u[((size_t)z * g.n.y + y) * g.n.x + x]; };
    const R c0v = at(X, Y, Z);
    const R sx = mc_slope(c0v - at(xm, Y, Z), at(xp, Y, Z) - c0v), sy = mc_slope(c0v - at(X, ym, Z), at(X, yp, Z) - c0v),
            sz = mc_slope(c0v - at(X, Y, zm), at(X, Y, zp) - c0v);
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const int ox = c & 1, oy = (c >> 1) & 1, oz = c >> 2;
      Uf[v * f3 + ((size_t)(2 * k + oz) * fy + 2 * j + oy) * fx + 2 * i + ox] = c0v + (ox ? q : -q) * sx + (oy ? q : -q) * sy + (oz ? q : -q) * sz;
    }
  }
}

}  // namespace mhd

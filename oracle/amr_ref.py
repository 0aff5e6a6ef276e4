"""CPU oracle of the AMR correction operation on a static two-level mesh.  TEST INFRASTRUCTURE ONLY.

Plain numpy / Python loops written from the paper's statement:
  (1) a coarse grid overlapping fine grids is replaced by the volume average (conserved variables) and the area
      average (face magnetic field) of the fine data;
  (2) a leaf coarse cell adjacent to a coarse-fine interface is corrected by the flux difference between the coarse and
      the fine grids on the interface, and the magnetic field of leaf coarse faces touching a coarse-fine inter-edge by
      the electric-field difference on that edge.
Readings: one refined box per call, aligned to patches (multiples of ps2/2 coarse cells), away from
the periodic boundary; both levels advanced with the same dt (w_c = w_f = 1); with sub-cycling the fine fluxes / EMFs
enter with weight 1/nsub per fine step.

Layouts: coarse grid as paper_1804_03479_b200.inputs (U[5][nz][ny][nx], bx[nz][ny][nx+1], ...); fine data as the solver's
U_out / B_out / flux_out / emf_out of the fine patch groups covering the box, ordered z outermost, x fastest; coarse
flux_out / emf_out of ALL coarse groups in grid order.  N = ps2.
"""
from __future__ import annotations

import numpy as np


def _split_B(Bflat, N):
    s = N * N * (N + 1)
    return (Bflat[0:s].reshape(N, N, N + 1), Bflat[s:2 * s].reshape(N, N + 1, N), Bflat[2 * s:3 * s].reshape(N + 1, N, N))


def restrict(U_f, B_f, lo, hi, N, Uc, bxc, byc, bzc):
    """(1): overwrite coarse cells lo..hi-1 and all their faces (including those on the box surface) in place."""
    h = N // 2
    m = [(hi[d] - lo[d]) // h for d in range(3)]          # fine groups per axis
    gi = 0
    for gz in range(m[2]):
        for gy in range(m[1]):
            for gx in range(m[0]):
                Ug = U_f[gi].reshape(5, N, N, N)
                bxg, byg, bzg = _split_B(B_f[gi], N)
                x0, y0, z0 = lo[0] + gx * h, lo[1] + gy * h, lo[2] + gz * h
                for k in range(h):
                    for j in range(h):
                        for i in range(h):
                            Uc[:, z0 + k, y0 + j, x0 + i] = Ug[:, 2 * k:2 * k + 2, 2 * j:2 * j + 2, 2 * i:2 * i + 2].reshape(5, 8).mean(axis=1)
                for k in range(h):
                    for j in range(h):
                        for i in range(h + 1):
                            bxc[z0 + k, y0 + j, x0 + i] = bxg[2 * k:2 * k + 2, 2 * j:2 * j + 2, 2 * i].mean()
                for k in range(h):
                    for j in range(h + 1):
                        for i in range(h):
                            byc[z0 + k, y0 + j, x0 + i] = byg[2 * k:2 * k + 2, 2 * j, 2 * i:2 * i + 2].mean()
                for k in range(h + 1):
                    for j in range(h):
                        for i in range(h):
                            bzc[z0 + k, y0 + j, x0 + i] = bzg[2 * k, 2 * j:2 * j + 2, 2 * i:2 * i + 2].mean()
                gi += 1


class _Planes:
    """access to flux_out[G][9][5][N][N] and emf_out[G][9][2][(N+1)N] by global position"""

    def __init__(self, flux, emf, N):
        self.N = N
        self.flux = np.asarray(flux).reshape(-1, 9, 5, N, N)
        e = np.asarray(emf).reshape(-1, 9, 2, (N + 1) * N)
        self.e0 = e[:, :, 0].reshape(-1, 9, N + 1, N)      # E_t1 [t2 edge pos][t1 cell]
        self.e1 = e[:, :, 1].reshape(-1, 9, N, N + 1)      # E_t2 [t2 cell][t1 edge pos]


def _coarse_group(pos, d, N, mg):
    """coarse group and plane slot holding the d-face plane at coarse index pos[d]; local indices of the other axes"""
    g = [p // N for p in pos]
    loc = [p - gg * N for p, gg in zip(pos, g)]
    s = {0: 0, N // 2: 1}[loc[d]]
    return (g[2] * mg[1] + g[1]) * mg[0] + g[0], 3 * d + s, loc


def fixup(flux_c, emf_c, flux_f, emf_f, lo, hi, N, dt, dh_c, Uc, bxc, byc, bzc, w_c=1.0, w_f=1.0):
    """(2): flux fix-up of leaf coarse cells next to the box and EMF fix-up of leaf coarse faces touching its surface."""
    nz, ny, nx = Uc.shape[1:]
    mg = (nx // N, ny // N, nz // N)
    h = N // 2
    mf = [(hi[d] - lo[d]) // h for d in range(3)]
    C, F = _Planes(flux_c, emf_c, N), _Planes(flux_f, emf_f, N)
    q = dt / dh_c
    b = (bxc, byc, bzc)

    def fine_group(cpos, d, side):
        """fine group touching the box surface (normal d, side 0 lower / 1 upper) that contains coarse position cpos
        (cell indices along the in-plane axes); returns (group, plane slot, fine local origin of the coarse cell)"""
        g, f0 = [0, 0, 0], [0, 0, 0]
        for a in range(3):
            if a == d:
                g[a] = 0 if side == 0 else mf[a] - 1
            else:
                rel = min(max(cpos[a] - lo[a], 0), hi[a] - lo[a] - 1)
                g[a] = rel // h
                f0[a] = 2 * (cpos[a] - lo[a] - g[a] * h)
        return (g[2] * mf[1] + g[1]) * mf[0] + g[0], 3 * d + (0 if side == 0 else 2), f0

    # ---- fluxes: the six faces of the box ----
    for d in range(3):
        t1, t2 = (d + 1) % 3, (d + 2) % 3
        for side in (0, 1):
            X = lo[d] if side == 0 else hi[d]
            for c2 in range(lo[t2], hi[t2]):
                for c1 in range(lo[t1], hi[t1]):
                    pos = [0, 0, 0]; pos[d] = X; pos[t1] = c1; pos[t2] = c2
                    gc, pc, loc = _coarse_group(pos, d, N, mg)
                    Fc = C.flux[gc, pc, :, loc[t2], loc[t1]]
                    gf, pf, f0 = fine_group(pos, d, side)
                    Ff = F.flux[gf, pf, :, f0[t2]:f0[t2] + 2, f0[t1]:f0[t1] + 2].reshape(5, 4).mean(axis=1)
                    cell = list(pos); cell[d] = X - 1 if side == 0 else X       # the leaf cell outside the box
                    # lower side: the face is the cell's UPPER face (dU = -q F); upper side: its LOWER face (dU = +q F)
                    sgn = -1.0 if side == 0 else 1.0
                    Uc[:, cell[2], cell[1], cell[0]] += sgn * q * (w_f * Ff - w_c * Fc)

    # ---- EMFs: every leaf coarse face that touches an edge of the box surface ----
    def on_surface_edge(c, pa, pb, pc):
        a, bb = (c + 1) % 3, (c + 2) % 3
        if not (lo[c] <= pc < hi[c]):
            return None
        if pa in (lo[a], hi[a]) and lo[bb] <= pb <= hi[bb]:
            return a
        if pb in (lo[bb], hi[bb]) and lo[a] <= pa <= hi[a]:
            return bb
        return None

    def edge_emfs(c, pa, pb, pc, dnorm):
        """coarse EMF and mean fine EMF of the coarse edge along c at (pa, pb), cell pc, read from the plane with normal dnorm"""
        a, bb = (c + 1) % 3, (c + 2) % 3
        pos = [0, 0, 0]; pos[a] = pa; pos[bb] = pb; pos[c] = pc
        side = 0 if pos[dnorm] == lo[dnorm] else 1
        t1, t2 = (dnorm + 1) % 3, (dnorm + 2) % 3
        # coarse: the plane may be indexed at the upper end of a group in an in-plane axis (local index N): use the next group
        gc, pcs, loc = _coarse_group(pos, dnorm, N, mg)
        gf, pfs, f0 = fine_group(pos, dnorm, side)
        # fine local position in the plane: along the edge = first fine cell of the coarse cell; across = fine edge index
        # relative to the fine group that holds it (2h = N at the far rim)
        fl = {}
        for ax in (t1, t2):
            if ax == c:
                fl[ax] = f0[ax]
            else:                                           # edge position across: relative to the fine group that holds it
                rel = pos[ax] - lo[ax]
                gidx = min(rel // h, mf[ax] - 1)
                fl[ax] = 2 * (rel - gidx * h)
        if c == t1:      # edge along t1, located at t2 - 1/2: component 0, [t2 edge][t1 cell]
            Ec = C.e0[gc, pcs, loc[t2], loc[t1]]
            Ef = 0.5 * (F.e0[gf, pfs, fl[t2], fl[t1]] + F.e0[gf, pfs, fl[t2], fl[t1] + 1])
        else:            # edge along t2, located at t1 - 1/2: component 1, [t2 cell][t1 edge]
            Ec = C.e1[gc, pcs, loc[t2], loc[t1]]
            Ef = 0.5 * (F.e1[gf, pfs, fl[t2], fl[t1]] + F.e1[gf, pfs, fl[t2] + 1, fl[t1]])
        return Ec, Ef

    def inside_closure(dface, pos):
        """is the coarse dface-face at pos (lower face of cell pos) inside the box or on its surface?"""
        for a in range(3):
            if a == dface:
                if not (lo[a] <= pos[a] <= hi[a]):
                    return False
            elif not (lo[a] <= pos[a] < hi[a]):
                return False
        return True

    for dface in range(3):
        t1, t2 = (dface + 1) % 3, (dface + 2) % 3
        rng = [range(lo[a] - 1, hi[a] + 2) for a in range(3)]
        for pz in rng[2]:
            for py in rng[1]:
                for px in rng[0]:
                    pos = [px, py, pz]
                    if inside_closure(dface, pos):
                        continue
                    # Eq. 13 for the lower dface-face of cell pos:  b -= q [ (E_t2(t1+) - E_t2(t1-)) - (E_t1(t2+) - E_t1(t2-)) ]
                    corr = 0.0
                    for (c, across, sign_) in ((t2, t1, +1.0), (t1, t2, -1.0)):
                        for up in (0, 1):
                            e = list(pos); e[across] += up
                            a_, b_ = (c + 1) % 3, (c + 2) % 3
                            dn = on_surface_edge(c, e[a_], e[b_], e[c])
                            if dn is None:
                                continue
                            Ec, Ef = edge_emfs(c, e[a_], e[b_], e[c], dn)
                            corr += sign_ * (1.0 if up else -1.0) * (w_f * Ef - w_c * Ec)
                    if corr != 0.0:
                        b[dface][pos[2], pos[1], pos[0]] -= q * corr


def inject(Uc, bxc, byc, bzc):
    """divergence-free piecewise-constant prolongation of a periodic coarse grid to twice the resolution (harness helper:
    fine faces lying on coarse faces take the coarse value, the faces in between the mean of the two)."""
    U = np.repeat(np.repeat(np.repeat(Uc, 2, axis=1), 2, axis=2), 2, axis=3)
    nz, ny, nx = Uc.shape[1:]
    def up(bc, axis):
        f = np.repeat(np.repeat(bc, 2, axis=(axis + 1) % 3), 2, axis=(axis + 2) % 3)      # transverse replication
        n = bc.shape[axis] - 1
        out_shape = list(f.shape); out_shape[axis] = 2 * n + 1
        out = np.empty(out_shape)
        sl = [slice(None)] * 3
        sl[axis] = slice(0, None, 2); out[tuple(sl)] = f
        lo_ = [slice(None)] * 3; hi_ = [slice(None)] * 3
        lo_[axis] = slice(0, n); hi_[axis] = slice(1, n + 1)
        sl[axis] = slice(1, None, 2); out[tuple(sl)] = 0.5 * (f[tuple(lo_)] + f[tuple(hi_)])
        return out
    return U, up(bxc, 2), up(byc, 1), up(bzc, 0)


# ------------------------------------------------------------------------------------------------------------------
# NEXT-3: creating new fine grids: conservative interpolation of the conserved variables and the
# divergence-free interpolation of Balsara (2001) for the face field, written as the paper words it and generalised
# from its 2-D example (Eq. 17, 10 coefficients) to 3-D (21 coefficients).  Readings: MC-limited
# slopes (the limiter of the solver); periodic coarse neighbours; the refined box is surrounded by coarse
# cells (no copy from pre-existing fine neighbours).
#
# Step by step for every coarse cell (unit cube, centre at the origin, x, y, z in units of the coarse cell size):
#   first set  -- the 24 fine faces lying on the six coarse faces: piecewise-linear interpolation of the coarse face
#                 value within the face, slopes from the neighbouring coarse faces of the same orientation;
#   second set -- the 12 interior fine faces: the polynomial
#                     Bx = a0 + ax x + ay y + az z + axx x^2 + axy xy + axz xz          (and cyclic for By, Bz)
#                 whose 21 coefficients are fixed by (i) matching the linear profile on each of the six coarse faces
#                 (18 equations, 17 independent when the coarse field is divergence-free) and (ii) div B = 0
#                 identically (4 equations); the linear system is SOLVED NUMERICALLY here (no closed form), and the
#                 interior fine-face values are the area averages of the polynomial (2-point Gauss, exact for degree 2).
# ------------------------------------------------------------------------------------------------------------------
def mc(a, b):
    """MC limiter: 0 if ab <= 0, else sign(a+b) min(|a+b|/2, 2|a|, 2|b|)"""
    if a * b <= 0.0:
        return 0.0
    return np.sign(a + b) * min(0.5 * abs(a + b), 2.0 * abs(a), 2.0 * abs(b))


# monomials of the three components: exponents (px, py, pz) in the order of the comment above
_MONO = (
    ((0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 0, 0), (1, 1, 0), (1, 0, 1)),      # Bx
    ((0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (0, 2, 0), (1, 1, 0), (0, 1, 1)),      # By
    ((0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (0, 0, 2), (1, 0, 1), (0, 1, 1)),      # Bz
)


def _poly(coef, comp, x, y, z):
    return sum(c * x ** p[0] * y ** p[1] * z ** p[2] for c, p in zip(coef[7 * comp:7 * comp + 7], _MONO[comp]))


def _dmono(p, axis):
    """d/d(axis) of the monomial with exponents p: (factor, exponents)"""
    if p[axis] == 0:
        return 0.0, p
    q = list(p); q[axis] -= 1
    return float(p[axis]), tuple(q)


def balsara_coefficients(face_val, face_slope):
    """face_val[d][s]: coarse face value of component d on side s (0 lower, 1 upper); face_slope[d][s][t]: its slope
    along axis t (t != d) per coarse cell.  Returns the 21 coefficients solving the matching + divergence-free system."""
    rows, rhs = [], []
    for d in range(3):
        for s in (0, 1):
            pos = [0.0, 0.0, 0.0]; pos[d] = -0.5 if s == 0 else 0.5
            # value at the face centre
            r = np.zeros(21)
            for m, p in enumerate(_MONO[d]):
                r[7 * d + m] = pos[0] ** p[0] * pos[1] ** p[1] * pos[2] ** p[2]
            rows.append(r); rhs.append(face_val[d][s])
            # in-face slopes at the face centre (the profile on the face is linear in the in-face coordinates)
            for t in range(3):
                if t == d:
                    continue
                r = np.zeros(21)
                for m, p in enumerate(_MONO[d]):
                    f, q = _dmono(p, t)
                    r[7 * d + m] = f * pos[0] ** q[0] * pos[1] ** q[1] * pos[2] ** q[2]
                rows.append(r); rhs.append(face_slope[d][s][t])
    # div B = 0 identically: the coefficient of every monomial of d(Bx)/dx + d(By)/dy + d(Bz)/dz vanishes
    div = {}
    for d in range(3):
        for m, p in enumerate(_MONO[d]):
            f, q = _dmono(p, d)
            if f != 0.0:
                div.setdefault(q, np.zeros(21))[7 * d + m] += f
    for q, r in sorted(div.items()):
        rows.append(r); rhs.append(0.0)
    A, b = np.array(rows), np.array(rhs)
    coef, res, rank, _ = np.linalg.lstsq(A, b, rcond=None)
    assert rank == 21
    return coef, float(np.abs(A @ coef - b).max())


_GAUSS = (-0.5 / np.sqrt(3.0), 0.5 / np.sqrt(3.0))      # 2-point Gauss nodes on [-1/2, 1/2] (scaled by the interval length)


def _face_average(coef, comp, centre, size):
    """area average of component comp over the square fine face centred at `centre` (normal = comp), edge `size`"""
    t1, t2 = (comp + 1) % 3, (comp + 2) % 3
    acc = 0.0
    for g1 in _GAUSS:
        for g2 in _GAUSS:
            p = list(centre); p[t1] += g1 * size; p[t2] += g2 * size
            acc += 0.25 * _poly(coef, comp, *p)
    return acc


def prolong(Uc, bxc, byc, bzc, lo, hi):
    """new fine grids covering coarse cells lo..hi-1 of a periodic coarse grid.  Returns U_f[5][2nbz][2nby][2nbx],
    bx_f[2nbz][2nby][2nbx+1], by_f[2nbz][2nby+1][2nbx], bz_f[2nbz+1][2nby][2nbx] and the largest residual of the linear
    systems (round-off when the coarse field is divergence-free)."""
    nz, ny, nx = Uc.shape[1:]
    n = (nx, ny, nz)
    nb = [hi[d] - lo[d] for d in range(3)]
    b = (bxc, byc, bzc)

    def face(d, pos):
        """coarse face value of component d at lattice position pos (periodic)"""
        q = [pos[a] % n[a] for a in range(3)]
        return b[d][q[2], q[1], q[0]]

    def slope(d, pos, t):
        up = list(pos); up[t] += 1
        dn = list(pos); dn[t] -= 1
        c = face(d, pos)
        return mc(face(d, up) - c, c - face(d, dn))

    U_f = np.empty((5, 2 * nb[2], 2 * nb[1], 2 * nb[0]))
    out = [np.full((2 * nb[2], 2 * nb[1], 2 * nb[0] + 1), np.nan), np.full((2 * nb[2], 2 * nb[1] + 1, 2 * nb[0]), np.nan),
           np.full((2 * nb[2] + 1, 2 * nb[1], 2 * nb[0]), np.nan)]
    worst = 0.0
    for k in range(nb[2]):
        for j in range(nb[1]):
            for i in range(nb[0]):
                cell = (lo[0] + i, lo[1] + j, lo[2] + k)
                rel = (i, j, k)
                # ---- conserved variables: conservative piecewise-linear interpolation ----
                for v in range(5):
                    c = Uc[v, cell[2], cell[1], cell[0]]
                    s = []
                    for t in range(3):
                        up = list(cell); up[t] = (up[t] + 1) % n[t]
                        dn = list(cell); dn[t] = (dn[t] - 1) % n[t]
                        s.append(mc(Uc[v, up[2], up[1], up[0]] - c, c - Uc[v, dn[2], dn[1], dn[0]]))
                    for dz in (0, 1):
                        for dy in (0, 1):
                            for dx in (0, 1):
                                U_f[v, 2 * k + dz, 2 * j + dy, 2 * i + dx] = c + (dx - 0.5) * 0.5 * s[0] + (dy - 0.5) * 0.5 * s[1] + (dz - 0.5) * 0.5 * s[2]
                # ---- face field ----
                fv = [[0.0, 0.0] for _ in range(3)]
                fs = [[[0.0] * 3, [0.0] * 3] for _ in range(3)]
                for d in range(3):
                    t1, t2 = (d + 1) % 3, (d + 2) % 3
                    for s_ in (0, 1):
                        pos = list(cell); pos[d] += s_
                        fv[d][s_] = face(d, pos)
                        fs[d][s_][t1] = slope(d, pos, t1)
                        fs[d][s_][t2] = slope(d, pos, t2)
                        # first set: the four fine faces on this coarse face
                        for o2 in (0, 1):
                            for o1 in (0, 1):
                                val = fv[d][s_] + (o1 - 0.5) * 0.5 * fs[d][s_][t1] + (o2 - 0.5) * 0.5 * fs[d][s_][t2]
                                idx = [0, 0, 0]
                                idx[d] = 2 * rel[d] + 2 * s_
                                idx[t1] = 2 * rel[t1] + o1
                                idx[t2] = 2 * rel[t2] + o2
                                out[d][idx[2], idx[1], idx[0]] = val
                coef, res = balsara_coefficients(fv, fs)
                worst = max(worst, res)
                # second set: the four interior fine faces per direction (normal coordinate 0)
                for d in range(3):
                    t1, t2 = (d + 1) % 3, (d + 2) % 3
                    for o2 in (0, 1):
                        for o1 in (0, 1):
                            centre = [0.0, 0.0, 0.0]; centre[t1] = (o1 - 0.5) * 0.5; centre[t2] = (o2 - 0.5) * 0.5
                            idx = [0, 0, 0]
                            idx[d] = 2 * rel[d] + 1
                            idx[t1] = 2 * rel[t1] + o1
                            idx[t2] = 2 * rel[t2] + o2
                            out[d][idx[2], idx[1], idx[0]] = _face_average(coef, d, centre, 0.5)
    return U_f, out[0], out[1], out[2], worst

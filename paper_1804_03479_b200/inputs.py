"""Seeded synthetic inputs and array-layout helpers (numpy only).

This module serves BOTH the CPU oracle tests and the CUDA path (DESIGN.md §"Input recipe").
It holds none of the solver's arithmetic: it builds initial states (which needs the
definition of the total energy, Eq. 5) and moves data between a periodic
uniform grid and ghost-zoned patch groups (the "preparation" and
"closing" steps, here reduced to periodic copies).

Layouts; index order [k][j][i], x fastest:
  grid   : U[5][n][n][n], bx[n][n][n+1], by[n][n+1][n], bz[n+1][n][n]  (periodic: last face == first)
  groups : U_in [G][5][T][T][T];  B_in [G][ Bx[T][T][T+1] | By[T][T+1][T] | Bz[T+1][T][T] ]  (flat)
           U_out[G][5][N][N][N];  B_out[G][ Bx[N][N][N+1] | By[N][N+1][N] | Bz[N+1][N][N] ]  (flat)
"""
from __future__ import annotations

import numpy as np

GAMMA = 5.0 / 3.0


# ----------------------------------------------------------------------------------------
# sizes
# ----------------------------------------------------------------------------------------
def sizes(N: int, g: int) -> dict:
    """Element counts per patch group."""
    T = N + 2 * g
    return dict(
        T=T,
        n_U_in=5 * T ** 3,
        n_B_in=3 * T * T * (T + 1),
        n_U_out=5 * N ** 3,
        n_B_out=3 * N * N * (N + 1),
        n_flux=9 * 5 * N * N,
        n_emf=9 * 2 * (N + 1) * N,
    )


def split_B(Bflat: np.ndarray, M: int):
    """Views (bx[M][M][M+1], by[M][M+1][M], bz[M+1][M][M]) of one group's flat B array."""
    s = M * M * (M + 1)
    bx = Bflat[..., 0:s].reshape(Bflat.shape[:-1] + (M, M, M + 1))
    by = Bflat[..., s:2 * s].reshape(Bflat.shape[:-1] + (M, M + 1, M))
    bz = Bflat[..., 2 * s:3 * s].reshape(Bflat.shape[:-1] + (M + 1, M, M))
    return bx, by, bz


def join_B(bx, by, bz) -> np.ndarray:
    lead = bx.shape[:-3]
    return np.concatenate(
        [bx.reshape(lead + (-1,)), by.reshape(lead + (-1,)), bz.reshape(lead + (-1,))], axis=-1
    )


# ----------------------------------------------------------------------------------------
# initial-state helpers
# ----------------------------------------------------------------------------------------
def faces_from_potential(Ax, Ay, Az, dh):
    """Discrete curl of an edge-centred vector potential -> face-centred B with div B = 0.

    Ax[k][j][i] sits at (x_i, y_{j-1/2}, z_{k-1/2})  shape [n+1][n+1][n]
    Ay[k][j][i] sits at (x_{i-1/2}, y_j, z_{k-1/2})  shape [n+1][n][n+1]
    Az[k][j][i] sits at (x_{i-1/2}, y_{j-1/2}, z_k)  shape [n][n+1][n+1]
    """
    bx = (Az[:, 1:, :] - Az[:, :-1, :]) / dh - (Ay[1:, :, :] - Ay[:-1, :, :]) / dh
    by = (Ax[1:, :, :] - Ax[:-1, :, :]) / dh - (Az[:, :, 1:] - Az[:, :, :-1]) / dh
    bz = (Ay[:, :, 1:] - Ay[:, :, :-1]) / dh - (Ax[:, 1:, :] - Ax[:, :-1, :]) / dh
    return bx, by, bz


def cell_centred_B(bx, by, bz):
    return (0.5 * (bx[..., :, :, :-1] + bx[..., :, :, 1:]),
            0.5 * (by[..., :, :-1, :] + by[..., :, 1:, :]),
            0.5 * (bz[..., :-1, :, :] + bz[..., 1:, :, :]))


def conserved(rho, vx, vy, vz, p, bx, by, bz, gamma=GAMMA):
    """U[5] from primitives and FACE fields; e includes 1/2 Bc^2 (Eq. 5)."""
    bcx, bcy, bcz = cell_centred_B(bx, by, bz)
    e = p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (bcx * bcx + bcy * bcy + bcz * bcz)
    return np.stack([rho, rho * vx, rho * vy, rho * vz, e])


def _edge_coords(n, dh, x0=0.0):
    c = x0 + (np.arange(n) + 0.5) * dh       # centres
    f = x0 + np.arange(n + 1) * dh           # faces
    return c, f


def abc_potential(n, dh, A=1.0, B=1.0, C=1.0, kwave=2.0 * np.pi, x0=0.0):
    """Edge potential of the ABC field, Eq. 20; curl(B_abc) = k B_abc so A_pot = B_abc/k."""
    c, f = _edge_coords(n, dh, x0)
    k = kwave

    def bxf(x, y, z): return A * np.sin(k * z) + C * np.cos(k * y) + 0 * x
    def byf(x, y, z): return B * np.sin(k * x) + A * np.cos(k * z) + 0 * y
    def bzf(x, y, z): return C * np.sin(k * y) + B * np.cos(k * x) + 0 * z

    Z, Y, X = np.meshgrid(f, f, c, indexing="ij"); Ax = bxf(X, Y, Z) / k
    Z, Y, X = np.meshgrid(f, c, f, indexing="ij"); Ay = byf(X, Y, Z) / k
    Z, Y, X = np.meshgrid(c, f, f, indexing="ij"); Az = bzf(X, Y, Z) / k
    return Ax, Ay, Az


def abc_grid(n, seed, p0=1.0, vamp=1e-3, gamma=GAMMA):
    """Configs 1/3/5 (BASELINE.json): rho=1, uniform p, ABC field A=B=C=1 at k=2*pi on [0,1)^3,
    v_d ~ U(-vamp, vamp) per cell."""
    dh = 1.0 / n
    rng = np.random.Generator(np.random.PCG64(seed))
    bx, by, bz = faces_from_potential(*abc_potential(n, dh), dh)
    rho = np.ones((n, n, n))
    v = rng.uniform(-vamp, vamp, size=(3, n, n, n)) if vamp > 0 else np.zeros((3, n, n, n))
    p = np.full((n, n, n), p0)
    return conserved(rho, v[0], v[1], v[2], p, bx, by, bz, gamma), bx, by, bz, dh


def blast_grid(n, gamma=GAMMA, p_in=10.0, p_out=0.1, r0=0.1):
    """Config 4: rho=1, p=10 for r<0.1 else 0.1, v=0, B=(1,1,1)/sqrt(2), box [-0.5,0.5)^3."""
    dh = 1.0 / n
    c = -0.5 + (np.arange(n) + 0.5) * dh
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    p = np.where(X * X + Y * Y + Z * Z < r0 * r0, p_in, p_out)
    b0 = 1.0 / np.sqrt(2.0)
    bx = np.full((n, n, n + 1), b0); by = np.full((n, n + 1, n), b0); bz = np.full((n + 1, n, n), b0)
    z = np.zeros((n, n, n))
    return conserved(np.ones((n, n, n)), z, z, z, p, bx, by, bz, gamma), bx, by, bz, dh


class _Fourier:
    """Sum of nm random Fourier modes with integer |k_d| <= kmax, unit one-point variance."""

    def __init__(self, rng, nm=8, kmax=2):
        k = np.zeros((nm, 3))
        for m in range(nm):
            while True:
                kk = rng.integers(-kmax, kmax + 1, size=3)
                if np.any(kk != 0):
                    break
            k[m] = kk
        self.k = 2.0 * np.pi * k
        self.phi = rng.uniform(0.0, 2.0 * np.pi, size=nm)
        self.a = rng.normal(size=nm)
        self.a *= np.sqrt(2.0 / np.sum(self.a ** 2))

    def __call__(self, X, Y, Z):
        out = np.zeros(np.broadcast(X, Y, Z).shape)
        for (kx, ky, kz), ph, a in zip(self.k, self.phi, self.a):
            out += a * np.cos(kx * X + ky * Y + kz * Z + ph)
        return out


def random_group_grid(n, seed, gamma=GAMMA, beta=1.0):
    """Config 2, one group = its own periodic n^3 box on [0,1)^3: rho lognormal(0,0.5), p lognormal(0,0.5),
    v ~ N(0,0.3^2) (one-point), face B = curl of an 8-mode random vector potential scaled to plasma beta."""
    dh = 1.0 / n
    rng = np.random.Generator(np.random.PCG64(seed))
    c, f = _edge_coords(n, dh)
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    rho = np.exp(0.5 * _Fourier(rng)(X, Y, Z))
    p = np.exp(0.5 * _Fourier(rng)(X, Y, Z))
    v = [0.3 * _Fourier(rng)(X, Y, Z) for _ in range(3)]
    fa = [_Fourier(rng) for _ in range(3)]
    Zc, Yc, Xc = np.meshgrid(f, f, c, indexing="ij"); Ax = fa[0](Xc, Yc, Zc)
    Zc, Yc, Xc = np.meshgrid(f, c, f, indexing="ij"); Ay = fa[1](Xc, Yc, Zc)
    Zc, Yc, Xc = np.meshgrid(c, f, f, indexing="ij"); Az = fa[2](Xc, Yc, Zc)
    bx, by, bz = faces_from_potential(Ax, Ay, Az, dh)
    bcx, bcy, bcz = cell_centred_B(bx, by, bz)
    b2 = np.mean(bcx ** 2 + bcy ** 2 + bcz ** 2)
    s = np.sqrt(2.0 * np.mean(p) / (beta * b2))
    bx, by, bz = s * bx, s * by, s * bz
    return conserved(rho, v[0], v[1], v[2], p, bx, by, bz, gamma), bx, by, bz, dh


# ----------------------------------------------------------------------------------------
# periodic grid <-> ghost-zoned patch groups (pure data movement)
# ----------------------------------------------------------------------------------------
def pack_groups(U, bx, by, bz, N, g, dtype=np.float64):
    """Cut a periodic (nz,ny,nx) grid into groups of N^3 cells with g ghost cells per side.
    Group order: gz outermost, gx fastest.  Returns (U_in[G][5*T^3], B_in[G][3*T*T*(T+1)])."""
    nz, ny, nx = U.shape[-3:]
    assert nx % N == 0 and ny % N == 0 and nz % N == 0
    mz, my, mx = nz // N, ny // N, nx // N
    T = N + 2 * g
    G = mx * my * mz
    Uo = np.empty((G, 5, T, T, T), dtype=dtype)
    Bo = np.empty((G, 3 * T * T * (T + 1)), dtype=dtype)
    bxo, byo, bzo = split_B(Bo, T)
    gi = 0
    for gz in range(mz):
        kc = (np.arange(-g, N + g) + gz * N) % nz
        kf = (np.arange(-g, N + g + 1) + gz * N) % nz
        for gy in range(my):
            jc = (np.arange(-g, N + g) + gy * N) % ny
            jf = (np.arange(-g, N + g + 1) + gy * N) % ny
            for gx in range(mx):
                ic = (np.arange(-g, N + g) + gx * N) % nx
                if_ = (np.arange(-g, N + g + 1) + gx * N) % nx
                Uo[gi] = U[np.ix_(np.arange(5), kc, jc, ic)]
                bxo[gi] = bx[np.ix_(kc, jc, if_)]
                byo[gi] = by[np.ix_(kc, jf, ic)]
                bzo[gi] = bz[np.ix_(kf, jc, ic)]
                gi += 1
    return Uo.reshape(G, -1), Bo


def unpack_groups(U_out, B_out, shape, N):
    """Inverse of pack_groups for solver OUTPUT (no ghosts); shape = n or (nz,ny,nx).  Periodic face arrays get
    face n := face 0.  Faces shared by two groups are taken from the group that owns them as LOWER faces; the
    largest |difference| to the upper copies is returned so that tests can check they agree bitwise (P4)."""
    nz, ny, nx = (shape, shape, shape) if np.isscalar(shape) else shape
    mz, my, mx = nz // N, ny // N, nx // N
    U = np.empty((5, nz, ny, nx), dtype=U_out.dtype)
    bx = np.empty((nz, ny, nx + 1), dtype=U_out.dtype)
    by = np.empty((nz, ny + 1, nx), dtype=U_out.dtype)
    bz = np.empty((nz + 1, ny, nx), dtype=U_out.dtype)
    Ug = U_out.reshape(-1, 5, N, N, N)
    bxg, byg, bzg = split_B(B_out, N)
    gi = 0
    for gz in range(mz):
        for gy in range(my):
            for gx in range(mx):
                ks, js, is_ = gz * N, gy * N, gx * N
                U[:, ks:ks + N, js:js + N, is_:is_ + N] = Ug[gi]
                bx[ks:ks + N, js:js + N, is_:is_ + N] = bxg[gi][:, :, :N]
                by[ks:ks + N, js:js + N, is_:is_ + N] = byg[gi][:, :N, :]
                bz[ks:ks + N, js:js + N, is_:is_ + N] = bzg[gi][:N, :, :]
                gi += 1
    mism = 0.0
    gi = 0
    for gz in range(mz):
        for gy in range(my):
            for gx in range(mx):
                ks, js, is_ = gz * N, gy * N, gx * N
                mism = max(mism, np.max(np.abs(bxg[gi][:, :, N] - bx[ks:ks + N, js:js + N, (is_ + N) % nx])))
                mism = max(mism, np.max(np.abs(byg[gi][:, N, :] - by[ks:ks + N, (js + N) % ny, is_:is_ + N])))
                mism = max(mism, np.max(np.abs(bzg[gi][N, :, :] - bz[(ks + N) % nz, js:js + N, is_:is_ + N])))
                gi += 1
    bx[:, :, nx] = bx[:, :, 0]
    by[:, ny, :] = by[:, 0, :]
    bz[nz, :, :] = bz[0, :, :]
    return U, bx, by, bz, float(mism)


def div_b(bx, by, bz, dh):
    """Discrete divergence, Eq. 16."""
    return ((bx[..., :, :, 1:] - bx[..., :, :, :-1]) + (by[..., :, 1:, :] - by[..., :, :-1, :])
            + (bz[..., 1:, :, :] - bz[..., :-1, :, :])) / dh


# ----------------------------------------------------------------------------------------
# the five BASELINE.json configs as packed group batches
# ----------------------------------------------------------------------------------------
def config2_batch(G, N=16, g=3, seed=3479, first=0, dtype=np.float64, gamma=GAMMA):
    """G independent periodic N^3 boxes, each packed as one ghost-zoned group (seed + group id)."""
    sz = sizes(N, g)
    U_in = np.empty((G, sz["n_U_in"]), dtype=dtype)
    B_in = np.empty((G, sz["n_B_in"]), dtype=dtype)
    for q in range(G):
        U, bx, by, bz, _ = random_group_grid(N, seed + first + q, gamma)
        u, b = pack_groups(U, bx, by, bz, N, g, dtype)
        U_in[q], B_in[q] = u[0], b[0]
    return U_in, B_in, 1.0 / N


def _hash_uniform(idx, seed):
    """Counter-based uniform [0,1) from an integer array (splitmix64 finaliser): the value of a cell depends only on its
    global index, so ghost cells of one group equal the interior cells of its neighbour without building the grid."""
    with np.errstate(over="ignore"):
        z = idx.astype(np.uint64) + np.uint64(seed) * np.uint64(0x9E3779B97F4A7C15) + np.uint64(0x632BE59BD9B4E019)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def abc_groups(n, first, G, N=16, g=3, seed=1805, p0=0.15, vamp=1e-2, dtype=np.float64, gamma=GAMMA):
    """Config 5 (BASELINE.json): G consecutive patch groups (group order of pack_groups: gz outermost, gx fastest), starting
    at group `first`, of the periodic n^3 ABC state of config 3 (rho = 1, p = p0, A=B=C=1, k = 2 pi, v_d ~ U(-vamp, vamp)),
    generated group by group WITHOUT building the grid (1024^3 does not fit): the face field is the discrete curl of the
    analytic edge potential on the ghost-zoned tile, the velocity of a cell a counter-based hash of its global index."""
    dh = 1.0 / n
    m = n // N
    T = N + 2 * g
    k = 2.0 * np.pi
    U_in = np.empty((G, 5, T, T, T), dtype=dtype)
    B_in = np.empty((G, 3 * T * T * (T + 1)), dtype=dtype)
    bxo, byo, bzo = split_B(B_in, T)
    for q in range(G):
        gi = first + q
        gx, gy, gz = gi % m, (gi // m) % m, gi // (m * m)
        ci = [np.arange(-g, N + g) + o * N for o in (gx, gy, gz)]            # global (unwrapped) cell indices per axis
        c = [(a + 0.5) * dh for a in ci]
        f = [np.arange(-g, N + g + 1) * dh + o * N * dh for o in (gx, gy, gz)]
        Z, Y, X = np.meshgrid(f[2], f[1], c[0], indexing="ij"); Ax = (np.sin(k * Z) + np.cos(k * Y) + 0 * X) / k
        Z, Y, X = np.meshgrid(f[2], c[1], f[0], indexing="ij"); Ay = (np.sin(k * X) + np.cos(k * Z) + 0 * Y) / k
        Z, Y, X = np.meshgrid(c[2], f[1], f[0], indexing="ij"); Az = (np.sin(k * Y) + np.cos(k * X) + 0 * Z) / k
        bx, by, bz = faces_from_potential(Ax, Ay, Az, dh)
        K, J, I = np.meshgrid(ci[2] % n, ci[1] % n, ci[0] % n, indexing="ij")
        lin = (K.astype(np.int64) * n + J) * n + I
        v = [vamp * (2.0 * _hash_uniform(3 * lin + d, seed) - 1.0) for d in range(3)]
        o = np.ones((T, T, T))
        U_in[q] = conserved(o, v[0], v[1], v[2], p0 * o, bx, by, bz, gamma)
        bxo[q], byo[q], bzo[q] = bx, by, bz
    return U_in.reshape(G, -1), B_in, dh


# ----------------------------------------------------------------------------------------
# SURVEY 8(f) NEXT-4 second workload: the paper's 1-D Riemann problems (Table 1)
# ----------------------------------------------------------------------------------------
# (rho, vn, vt1, vt2, P, Bt1, Bt2) left / right and the longitudinal field Bn, as printed in Table 1 and PAPER.md:270
RIEMANN_PROBLEMS = {
    "rj2a": dict(L=(1.08, 1.2, 0.01, 0.5, 0.95, 3.6 / np.sqrt(4 * np.pi), 2.0 / np.sqrt(4 * np.pi)),
                 R=(1.0, 0.0, 0.0, 0.0, 1.0, 4.0 / np.sqrt(4 * np.pi), 2.0 / np.sqrt(4 * np.pi)), Bn=2.0 / np.sqrt(4 * np.pi), t_end=0.2),
    "torrilhon": dict(L=(1.0, 0.0, 0.0, 0.0, 1.0, 1.0, 0.0), R=(0.2, 0.0, 0.0, 0.0, 0.2, np.cos(3.0), np.sin(3.0)), Bn=1.0, t_end=0.08),
}


def shock_tube(name, n, axis=0, nt=8, gamma=GAMMA):
    """Two copies of the tube back to back on a PERIODIC domain of length 2 along `axis` (2n cells, nt cells across):
    left state on [0, 0.5) and [1.5, 2), right state on [0.5, 1.5), so that the paper's Dirichlet tube of length 1
     is the part [0, 1) until the waves of the second interface arrive.  Returns U, bx, by, bz, dh."""
    pr = RIEMANN_PROBLEMS[name]
    nn = 2 * n
    dh = 1.0 / n
    xc = (np.arange(nn) + 0.5) * dh
    left = (xc < 0.5) | (xc >= 1.5)
    n_, t1, t2 = axis, (axis + 1) % 3, (axis + 2) % 3
    shape = [nt, nt, nt]; shape[2 - axis] = nn
    nz, ny, nx = shape
    bshape = [1, 1, 1]; bshape[2 - axis] = nn
    prof = [np.where(left, pr["L"][v], pr["R"][v]).reshape(bshape) for v in range(7)]
    fs = [(nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)]
    b = [None, None, None]
    b[n_] = np.full(fs[n_], pr["Bn"])
    b[t1] = prof[5] + np.zeros(fs[t1])
    b[t2] = prof[6] + np.zeros(fs[t2])
    o = np.zeros((nz, ny, nx))
    v = [None, None, None]
    v[n_], v[t1], v[t2] = prof[1] + o, prof[2] + o, prof[3] + o
    U = conserved(prof[0] + o, v[0], v[1], v[2], prof[4] + o, b[0], b[1], b[2], gamma)
    return U, b[0], b[1], b[2], dh
